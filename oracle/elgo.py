"""ctypes binding of the CPU ORACLE (oracle/elgo.cpp).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg import
this module.  It shares nothing with paper_1710_07350_b200/ (the CUDA path); both are driven with
the same bytes produced by elg_inputs/.

    from oracle import elgo
    elgo.build()                      # g++ -O2 -ffp-contract=off  ->  oracle/libelgo.so
    b = elgo.Bunch(coords6xn, p0c_eV=1e9, charge_C=1e-9)
    bl = elgo.Beamline(workload.elements, ring=False)
    out = b.track(bl, n_turns=1, moments_every="turn", want_stage_outputs=True)
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "elgo.cpp")
_HDR = os.path.join(_HERE, "elgo.h")
_LIB = os.path.join(_HERE, "libelgo.so")

OK, EINVAL, ENOMEM, ESTATE, ECAPACITY = 0, -1, -2, -4, -5
DRIFT, MATRIX, RFKICK, RCOL, ECOL, WAKE, HISTO, MATRIX2, TRWAKE, MATRIX3 = 1, 2, 3, 4, 5, 6, 7, 8, 9, 10
WIN = {"EXPLICIT": 0, "AUTO_MINMAX": 1, "AUTO_TABLE": 2}
WAKEKIND = {"RESONATOR": 0, "TABLE": 1, "RESONATOR_T": 2, "RESONATOR_REC": 3}
MOM = {"none": 0, "turn": 1, "element": 2}
ELECTRON_MC2_EV = 0.51099895e6

_dp = C.POINTER(C.c_double)
_i64p = C.POINTER(C.c_int64)
_i32p = C.POINTER(C.c_int32)
_u32p = C.POINTER(C.c_uint32)
_u8p = C.POINTER(C.c_uint8)


class Element(C.Structure):
    _fields_ = [
        ("type", C.c_int32), ("nb", C.c_int32), ("window", C.c_int32), ("wake", C.c_int32),
        ("interp", C.c_int32), ("fiducial", C.c_int32),
        ("L", C.c_double), ("V", C.c_double), ("f", C.c_double), ("phi", C.c_double),
        ("ax", C.c_double), ("ay", C.c_double), ("Q", C.c_double), ("Rs", C.c_double),
        ("t_lo_rel", C.c_double), ("dt", C.c_double), ("dt_table", C.c_double),
        ("R", _dp), ("C", _dp), ("table", _dp), ("n_table", C.c_int64), ("T", _dp), ("U", _dp),
    ]


class TrackOpts(C.Structure):
    _fields_ = [
        ("moments_every", C.c_int32), ("n_threads", C.c_int32),
        ("records", _dp), ("capacity_records", C.c_int64), ("n_records", C.c_int64),
        ("hist_out", _u32p), ("hist_capacity", C.c_int64), ("hist_written", C.c_int64),
        ("V_out", _dp), ("V_capacity", C.c_int64), ("V_written", C.c_int64),
        ("window_out", _dp), ("window_capacity", C.c_int64), ("window_written", C.c_int64),
    ]


def build(force: bool = False) -> str:
    """Compile the oracle (plain g++, no CUDA).  Building the checker is not using it."""
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fPIC", "-shared", "-pthread",
               _SRC, "-o", _LIB]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        v6 = _dp * 6
        L.elgo_drift.argtypes = [_dp, _dp, _dp, _dp, _dp, C.c_int64, C.c_double]
        L.elgo_drift.restype = None
        L.elgo_matrix.argtypes = [v6, C.c_int64, _dp, _dp]
        L.elgo_matrix.restype = None
        L.elgo_matrix2.argtypes = [v6, C.c_int64, _dp, _dp, _dp]
        L.elgo_matrix2.restype = None
        L.elgo_matrix3.argtypes = [v6, C.c_int64, _dp, _dp, _dp, _dp]
        L.elgo_matrix3.restype = None
        L.elgo_rfkick.argtypes = [_dp, _dp, C.c_int64] + [C.c_double] * 5
        L.elgo_rfkick.restype = None
        L.elgo_fiducial.argtypes = [_dp, C.c_int64, C.c_double]
        L.elgo_fiducial.restype = C.c_double
        L.elgo_aperture_flags.argtypes = [_dp, _dp, C.c_int64, C.c_int32, C.c_double, C.c_double, _u8p]
        L.elgo_aperture_flags.restype = None
        L.elgo_compact.argtypes = [v6, _i64p, C.c_int64, _u8p, v6, _i64p]
        L.elgo_compact.restype = C.c_int64
        L.elgo_window.argtypes = [_dp, C.c_int64, C.c_double, C.c_int32, C.c_int32, C.c_double,
                                  C.c_double, C.c_double, _dp]
        L.elgo_window.restype = C.c_int32
        L.elgo_histogram.argtypes = [_dp, C.c_int64, C.c_double, C.c_double, C.c_double, C.c_int32,
                                     _u32p, _i32p]
        L.elgo_histogram.restype = C.c_int64
        L.elgo_wake_samples.argtypes = [C.c_int32, C.c_int32, C.c_double, C.c_double, C.c_double,
                                        C.c_double, _dp, C.c_int64, C.c_double, _dp]
        L.elgo_wake_samples.restype = C.c_int32
        L.elgo_convolve.argtypes = [_u32p, _dp, C.c_int32, C.c_double, _dp]
        L.elgo_convolve.restype = None
        L.elgo_kick.argtypes = [_dp, _dp, C.c_int64, C.c_double, C.c_double, C.c_double, C.c_int32,
                                _dp, C.c_double, C.c_int32]
        L.elgo_kick.restype = None
        L.elgo_convolve_resonator.argtypes = [_u32p, C.c_int32, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double, _dp]
        L.elgo_convolve_resonator.restype = C.c_int32
        L.elgo_dipole_histogram.argtypes = [_dp, _dp, _dp, C.c_int64, C.c_double, C.c_double, C.c_double, C.c_int32,
                                            _u32p, _dp, _dp]
        L.elgo_dipole_histogram.restype = C.c_int64
        L.elgo_convolve_d.argtypes = [_dp, _dp, C.c_int32, C.c_double, _dp]
        L.elgo_convolve_d.restype = None
        L.elgo_tkick.argtypes = [_dp, _dp, _dp, C.c_int64, C.c_double, C.c_double, C.c_double, C.c_int32,
                                 _dp, _dp, C.c_double, C.c_int32]
        L.elgo_tkick.restype = None
        L.elgo_moments.argtypes = [v6, C.c_int64, _dp, _dp]
        L.elgo_moments.restype = C.c_int32
        for name in ("elgo_beta0",):
            getattr(L, name).argtypes = [C.c_double, C.c_double]
            getattr(L, name).restype = C.c_double
        L.elgo_inv_bc.argtypes = [C.c_double]
        L.elgo_inv_bc.restype = C.c_double
        L.elgo_inv_E.argtypes = [C.c_double, C.c_double]
        L.elgo_inv_E.restype = C.c_double
        L.elgo_bunch_create.argtypes = [C.POINTER(C.c_void_p), C.c_int64, v6, _i64p, C.c_double,
                                        C.c_double, C.c_double]
        L.elgo_bunch_create.restype = C.c_int32
        L.elgo_bunch_destroy.argtypes = [C.c_void_p]
        L.elgo_bunch_destroy.restype = None
        L.elgo_beamline_load.argtypes = [C.POINTER(C.c_void_p), C.POINTER(Element), C.c_int64, C.c_int32]
        L.elgo_beamline_load.restype = C.c_int32
        L.elgo_beamline_destroy.argtypes = [C.c_void_p]
        L.elgo_beamline_destroy.restype = None
        L.elgo_beamline_s_design.argtypes = [C.c_void_p, C.c_int64]
        L.elgo_beamline_s_design.restype = C.c_double
        L.elgo_beamline_length.argtypes = [C.c_void_p]
        L.elgo_beamline_length.restype = C.c_double
        L.elgo_track.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.POINTER(TrackOpts)]
        L.elgo_track.restype = C.c_int32
        L.elgo_n_alive.argtypes = [C.c_void_p]
        L.elgo_n_alive.restype = C.c_int64
        L.elgo_bunch_read.argtypes = [C.c_void_p, v6, _i64p, C.c_int64]
        L.elgo_bunch_read.restype = C.c_int32
        L.elgo_moments_now.argtypes = [C.c_void_p, _i64p, _dp, _dp]
        L.elgo_moments_now.restype = C.c_int32
        L.elgo_lost.argtypes = [C.c_void_p, _i64p, C.c_int64, _i64p, _i32p, _i32p, _dp]
        L.elgo_lost.restype = C.c_int32
        _lib = L
    return _lib


# --------------------------------------------------------------------------- helpers
def _p(a: Optional[np.ndarray], typ=_dp):
    return None if a is None else a.ctypes.data_as(typ)


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _v6(rows: Sequence[np.ndarray]):
    return (_dp * 6)(*[_p(r) for r in rows])


# --------------------------------------------------------------------------- stage functions
def drift(v: np.ndarray, L: float) -> None:
    """v: (6, n) C-contiguous float64, updated in place."""
    lib().elgo_drift(_p(v[0]), _p(v[1]), _p(v[2]), _p(v[3]), _p(v[4]), v.shape[1], L)


def matrix(v: np.ndarray, R, Cvec=None) -> None:
    R = _f64(R).reshape(36)
    Cv = None if Cvec is None else _f64(Cvec)
    lib().elgo_matrix(_v6(v), v.shape[1], _p(R), _p(Cv))


def matrix2(v: np.ndarray, R, T, Cvec=None) -> None:
    R = _f64(R).reshape(36)
    T = _f64(T).reshape(126)
    Cv = None if Cvec is None else _f64(Cvec)
    lib().elgo_matrix2(_v6(v), v.shape[1], _p(R), _p(Cv), _p(T))


def matrix3(v: np.ndarray, R, T, U, Cvec=None) -> None:
    R = _f64(R).reshape(36); T = _f64(T).reshape(126); U = _f64(U).reshape(336)
    Cv = None if Cvec is None else _f64(Cvec)
    lib().elgo_matrix3(_v6(v), v.shape[1], _p(R), _p(Cv), _p(T), _p(U))


def rfkick(v: np.ndarray, A: float, omega: float, phi0: float, s_ref: float, inv_bc: float) -> None:
    lib().elgo_rfkick(_p(v[4]), _p(v[5]), v.shape[1], A, omega, phi0, s_ref, inv_bc)


def fiducial(s: np.ndarray, s_design: float) -> float:
    s = _f64(s)
    return lib().elgo_fiducial(_p(s), s.shape[0], s_design)


def aperture_flags(x: np.ndarray, y: np.ndarray, kind: int, ax: float, ay: float) -> np.ndarray:
    x = _f64(x); y = _f64(y)
    out = np.empty(x.shape[0], dtype=np.uint8)
    lib().elgo_aperture_flags(_p(x), _p(y), x.shape[0], kind, ax, ay, _p(out, _u8p))
    return out


def compact(v: np.ndarray, ids: np.ndarray, survive: np.ndarray):
    """Stable partition in place.  Returns (n_surv, lost_v (6, n_lost), lost_ids)."""
    n = v.shape[1]
    lost_v = np.empty((6, max(n, 1)), dtype=np.float64)
    lost_id = np.empty(max(n, 1), dtype=np.int64)
    survive = np.ascontiguousarray(survive, dtype=np.uint8)
    ns = lib().elgo_compact(_v6(v), _p(ids, _i64p), n, _p(survive, _u8p), _v6(lost_v), _p(lost_id, _i64p))
    return ns, lost_v[:, : n - ns].copy(), lost_id[: n - ns].copy()


def window(s: np.ndarray, inv_bc: float, mode: int, nb: int, t_lo_rel=0.0, dt_in=0.0, t_design=0.0):
    s = _f64(s)
    out = np.empty(3, dtype=np.float64)
    rc = lib().elgo_window(_p(s), s.shape[0], inv_bc, mode, nb, t_lo_rel, dt_in, t_design, _p(out))
    if rc != OK:
        raise ValueError(f"elgo_window rc={rc}")
    return out  # t_lo, dt, inv_dt


def histogram(s: np.ndarray, inv_bc: float, t_lo: float, inv_dt: float, nb: int, want_bins=False):
    s = _f64(s)
    counts = np.empty(nb, dtype=np.uint32)
    bins = np.empty(s.shape[0], dtype=np.int32) if want_bins else None
    binned = lib().elgo_histogram(_p(s), s.shape[0], inv_bc, t_lo, inv_dt, nb, _p(counts, _u32p),
                                  _p(bins, _i32p))
    return (counts, binned, bins) if want_bins else (counts, binned)


def wake_samples(kind: int, nb: int, dt: float, f=0.0, Q=0.0, Rs=0.0, table=None, dt_table=0.0):
    W = np.empty(nb, dtype=np.float64)
    t = None if table is None else _f64(table)
    rc = lib().elgo_wake_samples(kind, nb, dt, f, Q, Rs, _p(t), 0 if t is None else t.shape[0], dt_table, _p(W))
    if rc != OK:
        raise ValueError(f"elgo_wake_samples rc={rc}")
    return W


def convolve(counts: np.ndarray, W: np.ndarray, q: float) -> np.ndarray:
    counts = np.ascontiguousarray(counts, dtype=np.uint32)
    W = _f64(W)
    V = np.empty(counts.shape[0], dtype=np.float64)
    lib().elgo_convolve(_p(counts, _u32p), _p(W), counts.shape[0], q, _p(V))
    return V


def convolve_resonator(counts, q: float, dt: float, f: float, Q: float, Rs: float) -> np.ndarray:
    counts = np.ascontiguousarray(counts, dtype=np.uint32)
    V = np.empty(counts.shape[0], dtype=np.float64)
    rc = lib().elgo_convolve_resonator(_p(counts, _u32p), counts.shape[0], q, dt, f, Q, Rs, _p(V))
    if rc != OK:
        raise ValueError(f"elgo_convolve_resonator rc={rc}")
    return V


def kick(s: np.ndarray, delta: np.ndarray, inv_bc, t_lo, inv_dt, nb, V, inv_E, interp=True) -> None:
    V = _f64(V)
    lib().elgo_kick(_p(s), _p(delta), s.shape[0], inv_bc, t_lo, inv_dt, nb, _p(V), inv_E, 1 if interp else 0)


def dipole_histogram(s, x, y, inv_bc: float, t_lo: float, inv_dt: float, nb: int):
    """TRWAKE stage (G32, G33): counts and exact per-bin dipole sums.  Returns (counts, Dx, Dy, binned)."""
    s = _f64(s); x = _f64(x); y = _f64(y)
    counts = np.empty(nb, dtype=np.uint32); Dx = np.empty(nb); Dy = np.empty(nb)
    binned = lib().elgo_dipole_histogram(_p(s), _p(x), _p(y), s.shape[0], inv_bc, t_lo, inv_dt, nb,
                                         _p(counts, _u32p), _p(Dx), _p(Dy))
    return counts, Dx, Dy, binned


def convolve_d(D, W, q: float) -> np.ndarray:
    D = _f64(D); W = _f64(W)
    V = np.empty(D.shape[0], dtype=np.float64)
    lib().elgo_convolve_d(_p(D), _p(W), D.shape[0], q, _p(V))
    return V


def tkick(s, xp, yp, inv_bc, t_lo, inv_dt, nb, Vx, Vy, inv_E, interp=True) -> None:
    Vx = _f64(Vx); Vy = _f64(Vy)
    lib().elgo_tkick(_p(s), _p(xp), _p(yp), s.shape[0], inv_bc, t_lo, inv_dt, nb, _p(Vx), _p(Vy), inv_E,
                     1 if interp else 0)


def moments(v: np.ndarray):
    cen = np.empty(6); sig = np.empty(36)
    rc = lib().elgo_moments(_v6(v), v.shape[1], _p(cen), _p(sig))
    if rc != OK:
        raise ValueError(f"elgo_moments rc={rc}")
    return cen, sig.reshape(6, 6)


def beta0(p0c, mc2=ELECTRON_MC2_EV):
    return lib().elgo_beta0(p0c, mc2)


def inv_bc(b0):
    return lib().elgo_inv_bc(b0)


def inv_E(b0, p0c):
    return lib().elgo_inv_E(b0, p0c)


# --------------------------------------------------------------------------- beamline / bunch
def _elements_to_c(elements):
    """elg_inputs element dictionaries -> (Element array, keep-alive list)."""
    arr = (Element * max(1, len(elements)))()
    keep = []
    for k, d in enumerate(elements):
        e = arr[k]
        t = d["type"]
        if t == "DRIFT":
            e.type, e.L = DRIFT, float(d["L"])
        elif t == "MATRIX":
            R = _f64(d["R"]).reshape(36); keep.append(R)
            e.type, e.R = MATRIX, _p(R)
            if d.get("C") is not None:
                Cv = _f64(d["C"]).reshape(6); keep.append(Cv); e.C = _p(Cv)
        elif t in ("MATRIX2", "MATRIX3"):
            R = _f64(d["R"]).reshape(36); T = _f64(d["T"]).reshape(126); keep += [R, T]
            e.type, e.R, e.T = (MATRIX2 if t == "MATRIX2" else MATRIX3), _p(R), _p(T)
            if t == "MATRIX3":
                U = _f64(d["U"]).reshape(336); keep.append(U); e.U = _p(U)
            if d.get("C") is not None:
                Cv = _f64(d["C"]).reshape(6); keep.append(Cv); e.C = _p(Cv)
        elif t == "RFKICK":
            e.type, e.V, e.f, e.phi = RFKICK, float(d["V"]), float(d["f"]), float(d["phi"])
            e.fiducial = 1 if d.get("fiducial", False) else 0
        elif t == "RCOL":
            e.type, e.ax, e.ay = RCOL, float(d["ax"]), float(d["ay"])
        elif t == "ECOL":
            e.type, e.ax, e.ay = ECOL, float(d["a"]), float(d["b"])
        elif t in ("WAKE", "HISTO", "TRWAKE"):
            e.type = {"WAKE": WAKE, "HISTO": HISTO, "TRWAKE": TRWAKE}[t]
            e.nb = int(d["nb"])
            e.window = WIN[d["window"]]
            e.t_lo_rel = float(d.get("t_lo_rel", 0.0))
            e.dt = float(d.get("dt", 0.0))
            if t != "HISTO":
                e.wake = WAKEKIND[d["wake"]]
                e.interp = 1 if d.get("interp", True) else 0
                if d["wake"] in ("RESONATOR", "RESONATOR_T", "RESONATOR_REC"):
                    e.f, e.Q, e.Rs = float(d["f"]), float(d["Q"]), float(d["Rs"])
                else:
                    tb = _f64(d["table"]); keep.append(tb)
                    e.table, e.n_table, e.dt_table = _p(tb), tb.shape[0], float(d["dt_table"])
        else:
            raise ValueError(f"unknown element type {t!r}")
    return arr, keep


class Beamline:
    def __init__(self, elements, ring: bool = False):
        arr, keep = _elements_to_c(elements)
        self.n_elems = len(elements)
        self.elements = list(elements)
        h = C.c_void_p()
        rc = lib().elgo_beamline_load(C.byref(h), arr, self.n_elems, 1 if ring else 0)
        if rc != OK:
            raise ValueError(f"elgo_beamline_load rc={rc}")
        self._h = h

    def s_design(self, k: int) -> float:
        return lib().elgo_beamline_s_design(self._h, k)

    @property
    def length(self) -> float:
        return lib().elgo_beamline_length(self._h)

    def __del__(self):
        if getattr(self, "_h", None):
            lib().elgo_beamline_destroy(self._h)
            self._h = None


class Bunch:
    def __init__(self, coords: np.ndarray, p0c_eV: float, charge_C: float, ids=None,
                 mc2_eV: float = ELECTRON_MC2_EV):
        coords = _f64(coords)
        assert coords.ndim == 2 and coords.shape[0] == 6
        self.n0 = coords.shape[1]
        idp = None if ids is None else np.ascontiguousarray(ids, dtype=np.int64)
        h = C.c_void_p()
        rc = lib().elgo_bunch_create(C.byref(h), self.n0, _v6(coords), _p(idp, _i64p), p0c_eV, mc2_eV, charge_C)
        if rc != OK:
            raise ValueError(f"elgo_bunch_create rc={rc}")
        self._h = h

    def __del__(self):
        if getattr(self, "_h", None):
            lib().elgo_bunch_destroy(self._h)
            self._h = None

    @property
    def n_alive(self) -> int:
        return lib().elgo_n_alive(self._h)

    def track(self, bl: Beamline, n_turns: int = 1, moments_every: str = "none", n_threads: int = 1,
              want_stage_outputs: bool = False):
        """Returns dict(records (k,43), hist [per WAKE/HISTO], V [per WAKE], window (k,3))."""
        o = TrackOpts()
        o.moments_every = MOM[moments_every]
        o.n_threads = n_threads
        n_rec = {"none": 0, "turn": n_turns, "element": n_turns * bl.n_elems}[moments_every]
        rec = np.zeros((max(n_rec, 1), 43), dtype=np.float64)
        o.records, o.capacity_records = _p(rec), n_rec
        hist = V = win = None
        if want_stage_outputs:
            nh = sum(e["nb"] for e in bl.elements if e["type"] in ("WAKE", "HISTO", "TRWAKE")) * n_turns
            nv = sum(e["nb"] * {"WAKE": 1, "TRWAKE": 4}[e["type"]] for e in bl.elements if e["type"] in ("WAKE", "TRWAKE")) * n_turns
            nw = sum(1 for e in bl.elements if e["type"] in ("WAKE", "HISTO", "TRWAKE")) * n_turns
            hist = np.zeros(max(nh, 1), dtype=np.uint32)
            V = np.zeros(max(nv, 1), dtype=np.float64)
            win = np.zeros((max(nw, 1), 3), dtype=np.float64)
            o.hist_out, o.hist_capacity = _p(hist, _u32p), nh
            o.V_out, o.V_capacity = _p(V), nv
            o.window_out, o.window_capacity = _p(win), nw
        rc = lib().elgo_track(self._h, bl._h, n_turns, C.byref(o))
        if rc != OK:
            raise RuntimeError(f"elgo_track rc={rc}")
        out = {"records": rec[: o.n_records].copy()}
        if want_stage_outputs:
            out["hist"] = hist[: o.hist_written].copy()
            out["V"] = V[: o.V_written].copy()
            out["window"] = win[: o.window_written].copy()
        return out

    def read(self):
        n = self.n_alive
        v = np.empty((6, n), dtype=np.float64)
        ids = np.empty(n, dtype=np.int64)
        if n:
            rc = lib().elgo_bunch_read(self._h, _v6(v), _p(ids, _i64p), n)
            assert rc == OK
        return v, ids

    def moments(self):
        n = C.c_int64()
        cen = np.empty(6); sig = np.empty(36)
        rc = lib().elgo_moments_now(self._h, C.byref(n), _p(cen), _p(sig))
        if rc != OK:
            raise RuntimeError(f"elgo_moments_now rc={rc}")
        return n.value, cen, sig.reshape(6, 6)

    def lost(self, cap: Optional[int] = None):
        """elgo_lost.  cap=None: every record.  With a cap the first min(cap, n_lost) records come back together with
        the status code and the true n_lost (cap < n_lost: ELGO_ECAPACITY)."""
        nl = C.c_int64()
        lib().elgo_lost(self._h, C.byref(nl), 0, None, None, None, None)
        n = nl.value if cap is None else min(cap, nl.value)
        ids = np.empty(n, dtype=np.int64); turn = np.empty(n, dtype=np.int32)
        elem = np.empty(n, dtype=np.int32); co = np.empty((n, 6), dtype=np.float64)
        rc = OK
        if n or cap is not None:
            rc = lib().elgo_lost(self._h, C.byref(nl), n if cap is None else cap, _p(ids, _i64p), _p(turn, _i32p),
                                 _p(elem, _i32p), _p(co))
        if cap is None:
            assert rc == OK
            return ids, turn, elem, co
        return ids, turn, elem, co, rc, nl.value

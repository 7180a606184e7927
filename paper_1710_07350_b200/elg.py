"""Thin ctypes binding of libelg.so (include/elg.h): argument marshalling only.

Same names as the C ABI: Beamline ~ elg_beamline_load, Bunch ~ elg_bunch_create, Bunch.track ~
elg_track, Bunch.moments ~ elg_moments, Bunch.lost ~ elg_lost.  PyTorch supplies device memory and the
stream; every step of the path runs in the library's CUDA kernels.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

from .build import LIB, build

OK, EINVAL, ENOMEM, ECUDA, ESTATE, ECAPACITY = 0, -1, -2, -3, -4, -5
DRIFT, MATRIX, RFKICK, RCOL, ECOL, WAKE, HISTO, MATRIX2, TRWAKE, MATRIX3 = 1, 2, 3, 4, 5, 6, 7, 8, 9, 10
WIN = {"EXPLICIT": 0, "AUTO_MINMAX": 1, "AUTO_TABLE": 2}
WAKEKIND = {"RESONATOR": 0, "TABLE": 1, "RESONATOR_T": 2, "RESONATOR_REC": 3}
MOM = {"none": 0, "turn": 1, "element": 2}
ELECTRON_MC2_EV = 0.51099895e6

_dp = C.POINTER(C.c_double)
_i64p = C.POINTER(C.c_int64)
_i32p = C.POINTER(C.c_int32)
_u32p = C.POINTER(C.c_uint32)

EXPORTS = (
    "elg_version", "elg_last_error", "elg_launch_count", "elg_soa_stride", "elg_soa_bytes",
    "elg_beamline_load", "elg_beamline_destroy", "elg_beamline_n_elements", "elg_beamline_length",
    "elg_beamline_s_design", "elg_beamline_launches_per_turn", "elg_workspace_bytes",
    "elg_bunch_create", "elg_bunch_destroy", "elg_bunch_upload", "elg_bunch_rewind", "elg_track",
    "elg_upload_and_track", "elg_bunch_host_state_save", "elg_bunch_host_state_restore",
    "elg_moments", "elg_lost", "elg_n_alive", "elg_bunch_read", "elg_bunch_device_array",
    "elg_profile_enable", "elg_profile_read",
    "elg_dbg_histogram", "elg_dbg_dipole_histogram", "elg_dbg_kick", "elg_dbg_tkick", "elg_dbg_compact",
    "elg_dbg_wake_samples", "elg_dbg_convolve", "elg_dbg_fp64_peak",
    "elg_noalloc_max_bins", "elg_dipole_histogram_noalloc",
)
KERNEL_KINDS = ("chain", "chain_compact", "window", "hist", "wake_samples", "conv", "moments", "chain_long")


class ElgError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"elg error {code}: {msg}")
        self.code = code


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
        ("moments_every", C.c_int32), ("flags", C.c_int32),
        ("records", _dp), ("capacity_records", C.c_int64), ("n_records", C.c_int64),
        ("hist_out", _u32p), ("hist_capacity", C.c_int64), ("hist_written", C.c_int64),
        ("V_out", _dp), ("V_capacity", C.c_int64), ("V_written", C.c_int64),
        ("window_out", _dp), ("window_capacity", C.c_int64), ("window_written", C.c_int64),
    ]


_lib = None


def lib():
    """Load libelg.so (building it with nvcc if it does not match the sources).  Fails loudly if that is impossible."""
    global _lib
    if _lib is not None:
        return _lib
    if os.environ.get("ELG_LIB"):                       # an explicitly named tuning variant (build(out=..., extra=...))
        path = os.environ["ELG_LIB"]
        if not os.path.exists(path):
            raise RuntimeError(f"ELG_LIB={path} does not exist")
    else:
        # current by content hash: load it; otherwise rebuild.  A compile error or a missing compiler propagates --
        # a library that does not match the sources is never loaded silently.
        path = build(force=bool(os.environ.get("ELG_REBUILD")))
    L = C.CDLL(path)
    v6 = _dp * 6
    vp = C.c_void_p
    L.elg_version.restype = C.c_char_p
    L.elg_last_error.restype = C.c_char_p
    L.elg_launch_count.restype = C.c_int64
    L.elg_soa_stride.argtypes = [C.c_int64]; L.elg_soa_stride.restype = C.c_int64
    L.elg_soa_bytes.argtypes = [C.c_int64]; L.elg_soa_bytes.restype = C.c_int64
    L.elg_beamline_load.argtypes = [C.POINTER(vp), C.POINTER(Element), C.c_int64, C.c_int32]
    L.elg_beamline_load.restype = C.c_int32
    L.elg_beamline_destroy.argtypes = [vp]; L.elg_beamline_destroy.restype = None
    L.elg_beamline_n_elements.argtypes = [vp]; L.elg_beamline_n_elements.restype = C.c_int64
    L.elg_beamline_length.argtypes = [vp]; L.elg_beamline_length.restype = C.c_double
    L.elg_beamline_s_design.argtypes = [vp, C.c_int64]; L.elg_beamline_s_design.restype = C.c_double
    L.elg_beamline_launches_per_turn.argtypes = [vp, C.c_int32]
    L.elg_beamline_launches_per_turn.restype = C.c_int64
    L.elg_workspace_bytes.argtypes = [C.c_int64, vp, C.c_int64, _i64p]; L.elg_workspace_bytes.restype = C.c_int32
    L.elg_bunch_create.argtypes = [C.POINTER(vp), C.c_int64, vp, vp, C.c_int64, vp, C.c_int64,
                                   C.c_double, C.c_double, C.c_double, vp]
    L.elg_bunch_create.restype = C.c_int32
    L.elg_bunch_destroy.argtypes = [vp]; L.elg_bunch_destroy.restype = None
    L.elg_bunch_upload.argtypes = [vp, v6, _i64p]; L.elg_bunch_upload.restype = C.c_int32
    L.elg_bunch_rewind.argtypes = [vp]; L.elg_bunch_rewind.restype = C.c_int32
    L.elg_track.argtypes = [vp, vp, C.c_int64, C.POINTER(TrackOpts)]; L.elg_track.restype = C.c_int32
    L.elg_bunch_host_state_save.argtypes = [vp, C.POINTER(C.c_int64)]; L.elg_bunch_host_state_save.restype = C.c_int32
    L.elg_bunch_host_state_restore.argtypes = [vp, C.POINTER(C.c_int64)]; L.elg_bunch_host_state_restore.restype = C.c_int32
    L.elg_upload_and_track.argtypes = [vp, vp, v6, _i64p, C.c_int64, C.POINTER(TrackOpts), C.c_int32]
    L.elg_upload_and_track.restype = C.c_int32
    L.elg_moments.argtypes = [vp, _i64p, _dp, _dp]; L.elg_moments.restype = C.c_int32
    L.elg_lost.argtypes = [vp, _i64p, C.c_int64, _i64p, _i32p, _i32p, _dp]; L.elg_lost.restype = C.c_int32
    L.elg_n_alive.argtypes = [vp, _i64p]; L.elg_n_alive.restype = C.c_int32
    L.elg_bunch_read.argtypes = [vp, v6, _i64p, C.c_int64]; L.elg_bunch_read.restype = C.c_int32
    L.elg_bunch_device_array.argtypes = [vp, C.c_int32, C.POINTER(vp)]; L.elg_bunch_device_array.restype = C.c_int32
    L.elg_profile_enable.argtypes = [vp, C.c_int32]; L.elg_profile_enable.restype = C.c_int32
    L.elg_profile_read.argtypes = [vp, _i64p, _dp, _dp, _dp]; L.elg_profile_read.restype = C.c_int32
    L.elg_dbg_fp64_peak.argtypes = [vp, C.c_int64, _dp, _dp, vp]; L.elg_dbg_fp64_peak.restype = C.c_int32
    L.elg_dbg_histogram.argtypes = [vp, C.c_double, C.c_double, C.c_int32, vp]; L.elg_dbg_histogram.restype = C.c_int32
    L.elg_dbg_dipole_histogram.argtypes = [vp, C.c_double, C.c_double, C.c_int32, vp, vp]
    L.elg_dbg_dipole_histogram.restype = C.c_int32
    L.elg_dbg_kick.argtypes = [vp, C.c_double, C.c_double, C.c_int32, vp, C.c_int32]; L.elg_dbg_kick.restype = C.c_int32
    L.elg_dbg_tkick.argtypes = [vp, C.c_double, C.c_double, C.c_int32, vp, vp, C.c_int32]; L.elg_dbg_tkick.restype = C.c_int32
    L.elg_dbg_compact.argtypes = [vp, C.c_int32, C.c_double, C.c_double]; L.elg_dbg_compact.restype = C.c_int32
    L.elg_dbg_wake_samples.argtypes = [C.c_int32, C.c_int32, C.c_double, C.c_double, C.c_double, C.c_double,
                                       vp, C.c_int64, C.c_double, vp, vp]
    L.elg_dbg_wake_samples.restype = C.c_int32
    L.elg_dbg_convolve.argtypes = [vp, vp, C.c_int32, C.c_double, vp, vp]; L.elg_dbg_convolve.restype = C.c_int32
    _lib = L
    return L


def _ck(rc: int) -> None:
    if rc != OK:
        raise ElgError(rc, lib().elg_last_error().decode())


def _p(a: Optional[np.ndarray], typ=_dp):
    return None if a is None else a.ctypes.data_as(typ)


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def launch_count() -> int:
    return lib().elg_launch_count()


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise ElgError(ECUDA, "no CUDA device: libelg has no CPU fallback")
    return torch


def _elements_to_c(elements):
    """Workload element dictionaries -> (elg_element array, keep-alive list).  Layout only."""
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
    """elg_beamline_load: host-only object (needs no device)."""

    def __init__(self, elements, ring: bool = False):
        arr, keep = _elements_to_c(elements)
        self.elements = list(elements)
        self.n_elems = len(elements)
        self.ring = bool(ring)
        h = C.c_void_p()
        _ck(lib().elg_beamline_load(C.byref(h), arr, self.n_elems, 1 if ring else 0))
        self._h = h

    @property
    def length(self) -> float:
        return lib().elg_beamline_length(self._h)

    def s_design(self, k: int) -> float:
        return lib().elg_beamline_s_design(self._h, k)

    def launches_per_turn(self, moments_every: str = "none") -> int:
        return lib().elg_beamline_launches_per_turn(self._h, MOM[moments_every])

    @property
    def has_aperture(self) -> bool:
        return any(e["type"] in ("RCOL", "ECOL") for e in self.elements)

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:       # (module globals are gone at interpreter exit)
            _lib.elg_beamline_destroy(self._h)
            self._h = None


class Bunch:
    """elg_bunch_create on torch-allocated device memory.

    coords: (6, n0) float64 host array (numpy, or a pinned torch CPU tensor) uploaded with
    elg_bunch_upload; or None with n0 given, when the caller fills `soa` on the device itself and then
    calls rewind()."""

    def __init__(self, coords=None, p0c_eV: float = 1e9, charge_C: float = 1e-9, ids=None,
                 beamline: Optional[Beamline] = None, lost_capacity: Optional[int] = None,
                 mc2_eV: float = ELECTRON_MC2_EV, n0: Optional[int] = None, device: str = "cuda:0",
                 stream=None):
        torch = _torch()
        L = lib()
        if coords is not None:
            n0 = int(coords.shape[1])
        assert n0 is not None
        self.n0 = n0
        self.device = torch.device(device)
        self.stride = L.elg_soa_stride(n0)
        if lost_capacity is None:
            lost_capacity = n0 if (beamline is None or beamline.has_aperture) else 0
        self.lost_capacity = int(lost_capacity)
        wb = C.c_int64()
        _ck(L.elg_workspace_bytes(n0, beamline._h if beamline else None, self.lost_capacity, C.byref(wb)))
        with torch.cuda.device(self.device):
            self.soa = torch.empty(7 * self.stride, dtype=torch.float64, device=self.device)
            self.work = torch.empty((wb.value + 7) // 8, dtype=torch.float64, device=self.device)
            self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            h = C.c_void_p()
            _ck(L.elg_bunch_create(C.byref(h), n0, self.soa.data_ptr(), self.work.data_ptr(), wb.value,
                                   beamline._h if beamline else None, self.lost_capacity,
                                   p0c_eV, mc2_eV, charge_C, self._stream.cuda_stream))
        self._h = h
        if coords is not None:
            self.upload(coords, ids)

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.elg_bunch_destroy(self._h)
            self._h = None

    # -- data movement -------------------------------------------------------------------------
    def upload(self, coords, ids=None) -> None:
        """elg_bunch_upload from host memory ((6, n0) numpy array or pinned torch tensor)."""
        if hasattr(coords, "data_ptr"):          # torch CPU tensor (possibly pinned)
            assert coords.dtype.is_floating_point and coords.element_size() == 8 and coords.is_contiguous()
            base = coords.data_ptr()
            ptrs = (_dp * 6)(*[C.cast(base + c * self.n0 * 8, _dp) for c in range(6)])
            self._keep = coords
        else:
            coords = _f64(coords)
            assert coords.shape == (6, self.n0)
            ptrs = (_dp * 6)(*[_p(coords[c]) for c in range(6)])
            self._keep = coords
        idp = None
        if ids is not None:
            ids = np.ascontiguousarray(ids, dtype=np.int64)
            idp = _p(ids, _i64p)
        _ck(lib().elg_bunch_upload(self._h, ptrs, idp))
        if not hasattr(coords, "is_pinned") or not coords.is_pinned():
            self.synchronize()                   # pageable source: make the copy complete before returning

    def rewind(self) -> None:
        _ck(lib().elg_bunch_rewind(self._h))

    def synchronize(self) -> None:
        self._stream.synchronize()

    # -- tracking ------------------------------------------------------------------------------
    def _host_ptrs(self, coords):
        if hasattr(coords, "data_ptr"):          # torch CPU tensor (possibly pinned)
            assert coords.dtype.is_floating_point and coords.element_size() == 8 and coords.is_contiguous()
            base = coords.data_ptr()
            ptrs = (_dp * 6)(*[C.cast(base + c * self.n0 * 8, _dp) for c in range(6)])
        else:
            coords = _f64(coords)
            assert coords.shape == (6, self.n0)
            ptrs = (_dp * 6)(*[_p(coords[c]) for c in range(6)])
        self._keep = coords
        return ptrs

    def _opts(self, bl, n_turns, moments_every, want_stage_outputs, records):
        o = TrackOpts()
        o.moments_every = MOM[moments_every]
        o.flags = 1 if getattr(self, "sparse_matrices", False) else 0      # ELG_TRACK_SPARSE_MATRICES
        n_rec = {"none": 0, "turn": n_turns, "element": n_turns * bl.n_elems}[moments_every]
        rec = None
        if records and n_rec:
            rec = np.zeros((n_rec, 43), dtype=np.float64)
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
        return o, rec, hist, V, win

    @staticmethod
    def _outputs(o, rec, hist, V, win, want_stage_outputs):
        out = {"n_records": o.n_records}
        if rec is not None:
            out["records"] = rec[: o.n_records]
        if want_stage_outputs:
            out["hist"] = hist[: o.hist_written]
            out["V"] = V[: o.V_written]
            out["window"] = win[: o.window_written]
        return out

    def track(self, bl: Beamline, n_turns: int = 1, moments_every: str = "none",
              want_stage_outputs: bool = False, records: bool = True):
        """elg_track.  Returns dict(records (k,43)[, hist, V, window])."""
        o, rec, hist, V, win = self._opts(bl, n_turns, moments_every, want_stage_outputs, records)
        _ck(lib().elg_track(self._h, bl._h, n_turns, C.byref(o)))
        return self._outputs(o, rec, hist, V, win, want_stage_outputs)

    def capture_track(self, bl: Beamline, n_turns: int = 1, moments_every: str = "none", prologue=None) -> "TrackGraph":
        """Capture [prologue(), elg_bunch_rewind, elg_track] into a CUDA graph on the bunch's stream (which must not be the
        default stream) and return it; .replay() launches the graph and puts the host mirror of the device state back to
        what it was after the capture (include/elg.h, "CUDA graphs").  prologue: e.g. the copy of fresh particles into
        bunch.soa.  The beamline must have been tracked once before (wake tables)."""
        return TrackGraph(self, bl, n_turns, moments_every, prologue)

    def upload_and_track(self, coords, bl: Beamline, n_turns: int = 1, moments_every: str = "none",
                         want_stage_outputs: bool = False, records: bool = True, n_chunks: int = 8, ids=None):
        """elg_upload_and_track: upload from host memory pipelined against the first turn's leading maps."""
        ptrs = self._host_ptrs(coords)
        idp = None
        if ids is not None:
            ids = np.ascontiguousarray(ids, dtype=np.int64)
            idp = _p(ids, _i64p)
            self._keep_ids = ids
        o, rec, hist, V, win = self._opts(bl, n_turns, moments_every, want_stage_outputs, records)
        _ck(lib().elg_upload_and_track(self._h, bl._h, ptrs, idp, n_turns, C.byref(o), n_chunks))
        if not (rec is not None or want_stage_outputs):
            pinned = hasattr(coords, "is_pinned") and coords.is_pinned()
            if not pinned:
                self.synchronize()
        return self._outputs(o, rec, hist, V, win, want_stage_outputs)

    # -- read-backs (synchronise) ----------------------------------------------------------------
    @property
    def n_alive(self) -> int:
        n = C.c_int64()
        _ck(lib().elg_n_alive(self._h, C.byref(n)))
        return n.value

    def read(self, out: Optional[np.ndarray] = None):
        n = self.n_alive
        v = np.empty((6, n), dtype=np.float64) if out is None else out[:, :n]
        ids = np.empty(n, dtype=np.int64)
        if n:
            ptrs = (_dp * 6)(*[_p(v[c]) for c in range(6)])
            _ck(lib().elg_bunch_read(self._h, ptrs, _p(ids, _i64p), n))
        return v, ids

    def moments(self):
        n = C.c_int64()
        cen = np.empty(6); sig = np.empty(36)
        _ck(lib().elg_moments(self._h, C.byref(n), _p(cen), _p(sig)))
        return n.value, cen, sig.reshape(6, 6)

    def lost(self):
        nl = C.c_int64()
        rc = lib().elg_lost(self._h, C.byref(nl), 0, None, None, None, None)
        if rc not in (OK, ECAPACITY):
            _ck(rc)
        n = min(nl.value, self.lost_capacity)
        ids = np.empty(n, dtype=np.int64); turn = np.empty(n, dtype=np.int32)
        elem = np.empty(n, dtype=np.int32); co = np.empty((n, 6), dtype=np.float64)
        if n:
            rc = lib().elg_lost(self._h, C.byref(nl), n, _p(ids, _i64p), _p(turn, _i32p), _p(elem, _i32p), _p(co))
            if rc not in (OK, ECAPACITY):
                _ck(rc)
        return ids, turn, elem, co

    def profile(self, on: bool = True) -> None:
        """elg_profile_enable: bracket every kernel launch of this bunch with CUDA events."""
        _ck(lib().elg_profile_enable(self._h, 1 if on else 0))

    def profile_read(self, work: bool = False) -> dict:
        """elg_profile_read: {kernel kind: (launches, summed device ms)} since the last read; with work=True
        {kind: (launches, ms, algorithmic bytes, algorithmic flops)}."""
        n = len(KERNEL_KINDS)
        cnt = np.zeros(n, dtype=np.int64); ms = np.zeros(n, dtype=np.float64)
        by = np.zeros(n, dtype=np.float64); fl = np.zeros(n, dtype=np.float64)
        _ck(lib().elg_profile_read(self._h, _p(cnt, _i64p), _p(ms), _p(by), _p(fl)))
        if work:
            return {k: (int(cnt[i]), float(ms[i]), float(by[i]), float(fl[i])) for i, k in enumerate(KERNEL_KINDS)}
        return {k: (int(cnt[i]), float(ms[i])) for i, k in enumerate(KERNEL_KINDS)}

    def device_array(self, c: int):
        """torch view of coordinate c (0..5; 6 = IDs as int64) of the CURRENT store, live prefix not applied."""
        torch = _torch()
        p = C.c_void_p()
        _ck(lib().elg_bunch_device_array(self._h, c, C.byref(p)))
        for base in (self.soa, self.work):
            off = p.value - base.data_ptr()
            if 0 <= off < base.numel() * 8:
                t = base[off // 8: off // 8 + self.stride]
                return t.view(torch.int64) if c == 6 else t
        raise ElgError(ESTATE, "device array outside the lent buffers")


class TrackGraph:
    """A captured [prologue, rewind, track] (Bunch.capture_track).  Argument marshalling and torch.cuda.CUDAGraph only."""

    def __init__(self, bunch: Bunch, bl: Beamline, n_turns: int, moments_every: str, prologue):
        torch = _torch()
        self.bunch = bunch
        self.graph = torch.cuda.CUDAGraph()
        o = TrackOpts()
        o.moments_every = MOM[moments_every]
        o.flags = 1 if getattr(bunch, "sparse_matrices", False) else 0
        with torch.cuda.graph(self.graph, stream=bunch._stream):
            if prologue is not None:
                prologue()
            _ck(lib().elg_bunch_rewind(bunch._h))
            _ck(lib().elg_track(bunch._h, bl._h, n_turns, C.byref(o)))
        self.state = (C.c_int64 * 8)()
        _ck(lib().elg_bunch_host_state_save(bunch._h, self.state))

    def replay(self) -> None:
        self.graph.replay()
        _ck(lib().elg_bunch_host_state_restore(self.bunch._h, self.state))


# ------------------------------------------------------------------------------- single-stage hooks
def _stage_bunch(coords, p0c_eV: float, nb: int, charge_C: float = 1e-9) -> "Bunch":
    """A bunch holding the ORACLE's input of one stage (coords (6, n)), its workspace sized for nb bins."""
    sizing = Beamline([{"type": "HISTO", "nb": int(nb), "window": "EXPLICIT", "dt": 1.0}])
    return Bunch(_f64(coords), p0c_eV, charge_C, beamline=sizing, lost_capacity=int(np.shape(coords)[1]))


def _coords_from(n: int, **rows) -> np.ndarray:
    v = np.zeros((6, n), dtype=np.float64)
    for name, a in rows.items():
        v[{"x": 0, "xp": 1, "y": 2, "yp": 3, "s": 4, "delta": 5}[name]] = a
    return v


def dbg_histogram(s, p0c_eV: float, t_lo: float, dt: float, nb: int) -> np.ndarray:
    """elg_dbg_histogram on a bunch whose s coordinates are `s`: tracking's own epilogue + window + hist kernels."""
    torch = _torch()
    s = _f64(s)
    b = _stage_bunch(_coords_from(s.size, s=s), p0c_eV, nb)
    d_c = torch.empty(nb, dtype=torch.int32, device=b.device)
    _ck(lib().elg_dbg_histogram(b._h, t_lo, dt, nb, d_c.data_ptr()))
    b.synchronize()
    return d_c.cpu().numpy().view(np.uint32)


def dbg_dipole_histogram(s, x, y, p0c_eV: float, t_lo: float, dt: float, nb: int):
    torch = _torch()
    s = _f64(s)
    b = _stage_bunch(_coords_from(s.size, s=s, x=x, y=y), p0c_eV, nb)
    d_c = torch.empty(nb, dtype=torch.int32, device=b.device)
    d_D = torch.empty(2 * nb, dtype=torch.float64, device=b.device)
    _ck(lib().elg_dbg_dipole_histogram(b._h, t_lo, dt, nb, d_c.data_ptr(), d_D.data_ptr()))
    b.synchronize()
    D = d_D.cpu().numpy()
    return d_c.cpu().numpy().view(np.uint32), D[:nb], D[nb:]


def dipole_histogram_noalloc(d_s, d_x, d_y, inv_bc: float, t_lo: float, dt: float, nb: int, d_counts, d_D, stream=None) -> None:
    """elg_dipole_histogram_noalloc: every array is the CALLER's torch CUDA tensor (s, x, y float64[n]; counts int32[nb];
    D float64[2 nb]); the library allocates nothing and does not synchronise.  Argument marshalling only."""
    torch = _torch()
    L = lib()
    L.elg_dipole_histogram_noalloc.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_double, C.c_double, C.c_double,
                                               C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
    L.elg_dipole_histogram_noalloc.restype = C.c_int32
    st = stream if stream is not None else torch.cuda.current_stream(d_s.device)
    _ck(L.elg_dipole_histogram_noalloc(d_s.data_ptr(), d_x.data_ptr(), d_y.data_ptr(), int(d_s.numel()), float(inv_bc), float(t_lo),
                                       float(dt), int(nb), d_counts.data_ptr(), d_D.data_ptr(), st.cuda_stream))


def noalloc_max_bins() -> int:
    return int(lib().elg_noalloc_max_bins())


def dbg_kick(s, delta, p0c_eV: float, t_lo: float, dt: float, nb: int, V, interp=True) -> np.ndarray:
    """elg_dbg_kick: OP_KICK as a fused run of one op on a bunch holding (s, delta); returns delta."""
    torch = _torch()
    s = _f64(s)
    b = _stage_bunch(_coords_from(s.size, s=s, delta=delta), p0c_eV, nb)
    d_V = torch.as_tensor(_f64(V), device=b.device)
    _ck(lib().elg_dbg_kick(b._h, t_lo, dt, nb, d_V.data_ptr(), 1 if interp else 0))
    b.synchronize()
    return b.device_array(5)[: s.size].cpu().numpy()


def dbg_tkick(s, xp, yp, p0c_eV: float, t_lo: float, dt: float, nb: int, Vx, Vy, interp=True):
    torch = _torch()
    s = _f64(s)
    b = _stage_bunch(_coords_from(s.size, s=s, xp=xp, yp=yp), p0c_eV, nb)
    d_Vx = torch.as_tensor(_f64(Vx), device=b.device); d_Vy = torch.as_tensor(_f64(Vy), device=b.device)
    _ck(lib().elg_dbg_tkick(b._h, t_lo, dt, nb, d_Vx.data_ptr(), d_Vy.data_ptr(), 1 if interp else 0))
    b.synchronize()
    return b.device_array(1)[: s.size].cpu().numpy(), b.device_array(3)[: s.size].cpu().numpy()


def dbg_compact(coords, kind: str, ax: float, ay: float, ids=None):
    """elg_dbg_compact on a bunch holding `coords` (the oracle's pre-aperture coordinates): returns
    (survivor coords, survivor ids, lost ids, lost coords (n_lost, 6))."""
    coords = _f64(coords)
    b = Bunch(coords, 1e9, 1e-9, ids=ids, lost_capacity=coords.shape[1])
    _ck(lib().elg_dbg_compact(b._h, {"RCOL": RCOL, "ECOL": ECOL}[kind], ax, ay))
    v, sid = b.read()
    lid, _, _, lco = b.lost()
    return v, sid, lid, lco


def dbg_wake_samples(kind: int, nb: int, dt: float, f=0.0, Q=0.0, Rs=0.0, table=None, dt_table=0.0) -> np.ndarray:
    torch = _torch()
    d_t = None if table is None else torch.as_tensor(_f64(table), device="cuda")
    d_W = torch.empty(nb, dtype=torch.float64, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    _ck(lib().elg_dbg_wake_samples(kind, nb, dt, f, Q, Rs, None if d_t is None else d_t.data_ptr(),
                                   0 if d_t is None else d_t.numel(), dt_table, d_W.data_ptr(), st))
    return d_W.cpu().numpy()


def dbg_convolve(counts, W, q: float) -> np.ndarray:
    torch = _torch()
    d_c = torch.as_tensor(np.ascontiguousarray(counts, dtype=np.uint32).view(np.int32), device="cuda")
    d_W = torch.as_tensor(_f64(W), device="cuda")
    d_V = torch.empty(d_c.numel(), dtype=torch.float64, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    _ck(lib().elg_dbg_convolve(d_c.data_ptr(), d_W.data_ptr(), d_c.numel(), q, d_V.data_ptr(), st))
    return d_V.cpu().numpy()


def dbg_fp64_peak(iters: int = 20000):
    """elg_dbg_fp64_peak: (TFLOP/s, ms) of the DFMA-only kernel -- the measured fp64 roofline denominator."""
    torch = _torch()
    scratch = torch.empty(512, dtype=torch.float64, device="cuda")
    tf = C.c_double(); ms = C.c_double()
    _ck(lib().elg_dbg_fp64_peak(scratch.data_ptr(), iters, C.byref(tf), C.byref(ms), torch.cuda.current_stream().cuda_stream))
    return tf.value, ms.value

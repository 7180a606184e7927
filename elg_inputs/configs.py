"""The five BASELINE.json workloads (and the roofline probes) as neutral data.

A workload is a particle recipe plus a list of element dictionaries.  Nothing here
applies an element to a particle: this module only writes the inputs down.  The
readings it encodes (restated in DESIGN.md "Readings"):

* G4  cfg0 matrix = thin quad AFTER a 0.5 m drift, M = Q(k1L) . D(0.5)
* G5  k1L > 0 focuses in x:  x' -= k1L x,  y' += k1L y
* G6  cfg1 "0.2 m thin quad" = D(0.1) Q D(0.1); 25 x [quad, ECOL, drift 2 m] with the two
      RF cavities after elements 16 and 33 (77 elements), first quad +0.8
* G7  p0c = 1 GeV electrons (cfg 0,1,2,4), 3 GeV (cfg 3)
* G16 cfg2 table amplitude 1e14 V/C; cfg3 R_s = 1 kOhm
* G22 literal aperture geometry is kept even though it loses more than the config text says
* G23 cfg3 uses the stabilised ring ("cfg3-stable"); "cfg3-literal" is the literal reading
* G25 seed = 1710073500 + config index; generated once on the host

Element dictionaries (keys are the paper's/BASELINE.json's names):
  DRIFT  {L}                         exact drift, PAPER.md:68-79 (Listing 1)
  MATRIX {R (6,6), C (6,)}           first-order transport matrix
  MATRIX2 {R, C, T (6,21)}           second-order transport map, PAPER.md:156 (G31)
  RFKICK {V, f, phi}                 thin RF cavity, PAPER.md:154,175
  RCOL   {ax, ay}  ECOL {a, b}       collimators, PAPER.md:149,153
  WAKE   {nb, window, wake, ...}     longitudinal wake, PAPER.md:165
  HISTO  {nb, window, ...}           diagnostic time histogram only, PAPER.md:111
  TRWAKE {nb, window, wake, ...}     transverse (dipole) wake, PAPER.md:164 (G32-G34)
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

from .rng import SEED_BASE, normal01, uniform01

ELECTRON_MC2_EV = 0.51099895e6
C_LIGHT = 299792458.0

WORKLOAD_NAMES = (
    "cfg0", "cfg1", "cfg2", "cfg3", "cfg3-literal", "cfg4",
    "p1-chain", "p2-chain-rcol", "p3-matrices", "p4-second-order", "p5-trwake", "p6-rfcw", "p7-third-order",
)


# ----------------------------------------------------------------------------- matrices
def drift_matrix(L: float):
    """Linear drift as a MATRIX element: R12 = R34 = L, C5 = L (s stays a path length, G3)."""
    R = np.eye(6)
    R[0, 1] = L
    R[2, 3] = L
    C = np.zeros(6)
    C[4] = L
    return R, C


def thin_quad_matrix(k1L: float):
    """Thin quadrupole, G5 sign: x' -= k1L x, y' += k1L y."""
    R = np.eye(6)
    R[1, 0] = -k1L
    R[3, 2] = +k1L
    return R, np.zeros(6)


def pair_index(j: int, k: int) -> int:
    """Position of the pair (j, k), j <= k, in the order (0,0) (0,1) .. (0,5) (1,1) .. (5,5) (G31)."""
    if j > k:
        j, k = k, j
    return j * 6 - j * (j - 1) // 2 + (k - j)


def second_order_drift(L: float):
    """Drift to second order: the linear drift plus the path-length terms s += L/2 (x'^2 + y'^2)."""
    R, C = drift_matrix(L)
    T = np.zeros((6, 21))
    T[4, pair_index(1, 1)] = 0.5 * L
    T[4, pair_index(3, 3)] = 0.5 * L
    return R, C, T


def thin_quad_sextupole(k1L: float, k2L: float):
    """Thin quadrupole + sextupole kick (G5 signs): x' -= k1L x + k2L/2 (x^2 - y^2);  y' += k1L y + k2L x y."""
    R, C = thin_quad_matrix(k1L)
    T = np.zeros((6, 21))
    T[1, pair_index(0, 0)] = -0.5 * k2L
    T[1, pair_index(2, 2)] = +0.5 * k2L
    T[3, pair_index(0, 2)] = +k2L
    return R, C, T


def triple_index(j: int, k: int, l: int) -> int:
    """Position of the triple j <= k <= l in lexicographic order (G35)."""
    j, k, l = sorted((j, k, l))
    t = 0
    for a in range(6):
        for b in range(a, 6):
            for c in range(b, 6):
                if (a, b, c) == (j, k, l):
                    return t
                t += 1
    raise ValueError((j, k, l))


def thin_quad_sext_octupole(k1L: float, k2L: float, k3L: float):
    """Thin multipole kick to third order: quadrupole + sextupole (see thin_quad_sextupole) + octupole
    x' -= k3L/6 (x^3 - 3 x y^2);  y' -= k3L/6 (y^3 - 3 x^2 y)."""
    R, C, T = thin_quad_sextupole(k1L, k2L)
    U = np.zeros((6, 56))
    U[1, triple_index(0, 0, 0)] = -k3L / 6.0
    U[1, triple_index(0, 2, 2)] = +k3L / 2.0
    U[3, triple_index(2, 2, 2)] = -k3L / 6.0
    U[3, triple_index(0, 0, 2)] = +k3L / 2.0
    return R, C, T, U


def third_order_drift(L: float):
    """Drift to third order: second_order_drift (the cubic terms of x, y and s vanish for a drift in these
    coordinates: x = x + L x' exactly, s gains L/2 (x'^2 + y'^2) and nothing cubic)."""
    R, C, T = second_order_drift(L)
    return R, C, T, np.zeros((6, 56))


def _matrix3_elem(R, C, T, U):
    return {"type": "MATRIX3", "R": np.ascontiguousarray(R, dtype=np.float64),
            "C": np.ascontiguousarray(C, dtype=np.float64), "T": np.ascontiguousarray(T, dtype=np.float64),
            "U": np.ascontiguousarray(U, dtype=np.float64)}


def _matrix2_elem(R, C, T):
    return {"type": "MATRIX2", "R": np.ascontiguousarray(R, dtype=np.float64),
            "C": np.ascontiguousarray(C, dtype=np.float64), "T": np.ascontiguousarray(T, dtype=np.float64)}


def compose(*maps):
    """compose(m1, m2, ...) = the map "m1 first, then m2, ..." as one (R, C)."""
    R = np.eye(6)
    C = np.zeros(6)
    for (R2, C2) in maps:
        C = C2 + R2 @ C
        R = R2 @ R
    return R, C


def _matrix_elem(R, C):
    return {"type": "MATRIX", "R": np.ascontiguousarray(R, dtype=np.float64),
            "C": np.ascontiguousarray(C, dtype=np.float64)}


def dense_symplectic_matrix(seed: int, strength: float = 0.6, c_s: float = 0.7):
    """A seeded DENSE symplectic 6x6 matrix (all 36 entries non-zero) with all six C entries non-zero, for parity
    tests whose inputs must exercise every coefficient of a map.  Cayley transform of a random Hamiltonian matrix
    H = J S (S symmetric): M = (I - H/2)^-1 (I + H/2) satisfies M^T J M = J exactly in exact arithmetic; the pairs
    are (x, x'), (y, y'), (s, delta).  Layout / coefficient generation only: nothing is applied to a particle."""
    rng = np.random.default_rng(seed)
    A = rng.normal(size=(6, 6))
    S = strength * (A + A.T) / 2.0
    J = np.zeros((6, 6))
    for k in range(3):
        J[2 * k, 2 * k + 1] = 1.0
        J[2 * k + 1, 2 * k] = -1.0
    H = J @ S
    M = np.linalg.solve(np.eye(6) - 0.5 * H, np.eye(6) + 0.5 * H)
    C = rng.normal(size=6) * np.array([2e-5, 2e-6, 2e-5, 2e-6, c_s, 2e-4])
    assert np.all(M != 0.0) and np.all(C != 0.0)
    return np.ascontiguousarray(M), np.ascontiguousarray(C)


def dense_higher_order(seed: int, order: int, t_scale: float = 1.0, u_scale: float = 1.0e4):
    """Seeded DENSE second- (T: all 126 entries non-zero) and third-order (U: all 336 non-zero) coefficients, scaled so
    that for a 100 um / 10 urad / 1 mm / 1e-3 beam the higher-order terms stay around 1e-3 of the linear ones."""
    rng = np.random.default_rng(seed + 7919)
    T = rng.normal(size=(6, 21)) * t_scale
    T[np.abs(T) < 1e-3 * t_scale] = 1e-3 * t_scale
    if order < 3:
        return np.ascontiguousarray(T), None
    U = rng.normal(size=(6, 56)) * u_scale
    U[np.abs(U) < 1e-3 * u_scale] = 1e-3 * u_scale
    return np.ascontiguousarray(T), np.ascontiguousarray(U)


def dense_map_element(seed: int, order: int = 1, strength: float = 0.6, t_scale: float = 1.0, u_scale: float = 1.0e4,
                      c_s: float = 0.7):
    """One MATRIX / MATRIX2 / MATRIX3 element dictionary with dense seeded coefficients (see above).  Long runs of
    higher-order maps need small strength / c_s / scales to keep the beam finite (parity is value-independent)."""
    R, C = dense_symplectic_matrix(seed, strength, c_s)
    if order == 1:
        return _matrix_elem(R, C)
    T, U = dense_higher_order(seed, order, t_scale, u_scale)
    return _matrix2_elem(R, C, T) if order == 2 else _matrix3_elem(R, C, T, U)


def beta0_of(p0c_eV: float, mc2_eV: float) -> float:
    return p0c_eV / np.sqrt(p0c_eV * p0c_eV + mc2_eV * mc2_eV)


# ----------------------------------------------------------------------------- workload
@dataclass
class Workload:
    name: str
    index: int                       # BASELINE.json config index (probes reuse cfg0's)
    n0: int
    p0c_eV: float
    charge_C: float
    ring: bool
    n_turns: int
    moments_every: str               # "none" | "turn" | "element"
    elements: list
    distribution: str                # "gauss6" | "chirp" | "flattop"
    mc2_eV: float = ELECTRON_MC2_EV
    notes: str = ""
    seed: int = field(default=0)

    def __post_init__(self):
        if not self.seed:
            self.seed = SEED_BASE + self.index

    # particle recipe -----------------------------------------------------------------
    def _fill(self, v: np.ndarray, start: int) -> None:
        n = v.shape[1]
        sd = self.seed
        if self.distribution == "gauss6":
            sig = (100e-6, 10e-6, 100e-6, 10e-6, 1e-3, 1e-3)
            for c in range(6):
                v[c] = normal01(sd, c, n, start)
                v[c] *= sig[c]
        elif self.distribution == "chirp":
            v[0:4] = 0.0
            v[4] = uniform01(sd, 4, n, start)
            v[4] *= 4e-3
            v[4] -= 2e-3
            v[5] = normal01(sd, 5, n, start)
            v[5] *= 1e-4
            v[5] += -5.0 * v[4]
        elif self.distribution == "flattop":
            for c in (0, 2):
                v[c] = uniform01(sd, c, n, start)
                v[c] *= 2e-3
                v[c] -= 1e-3
            for c in (1, 3):
                v[c] = normal01(sd, c, n, start)
                v[c] *= 50e-6
            v[4] = normal01(sd, 4, n, start)
            v[4] *= 1e-3
            v[5] = normal01(sd, 5, n, start)
            v[5] *= 1e-3
        else:
            raise ValueError(self.distribution)

    def particles(self, n: Optional[int] = None, start: int = 0,
                  out: Optional[np.ndarray] = None) -> np.ndarray:
        """(6, n) float64, rows x, x', y, y', s, delta for particle indices start..start+n-1.

        The generator is counter-based, so the result does not depend on the chunking or on
        the number of host threads used to fill it."""
        n = self.n0 if n is None else int(n)
        v = np.empty((6, n), dtype=np.float64) if out is None else out
        assert v.shape == (6, n) and v.dtype == np.float64
        chunk = 1 << 21
        if n <= chunk:
            self._fill(v, start)
            return v
        import os
        from concurrent.futures import ThreadPoolExecutor
        workers = max(1, min(32, (os.cpu_count() or 1)))
        spans = [(lo, min(n, lo + chunk)) for lo in range(0, n, chunk)]
        with ThreadPoolExecutor(max_workers=workers) as ex:
            list(ex.map(lambda sp: self._fill(v[:, sp[0]:sp[1]], start + sp[0]), spans))
        return v

    def ids(self, n: Optional[int] = None, start: int = 0) -> np.ndarray:
        n = self.n0 if n is None else int(n)
        return np.arange(start, start + n, dtype=np.int64)   # G27

    @property
    def n_pass_elements(self) -> int:
        """Elements that count as a particle-element pass: all but HISTO."""
        return sum(1 for e in self.elements if e["type"] != "HISTO")


# ----------------------------------------------------------------------------- recipes
def _cfg0(n):
    R, C = compose(drift_matrix(0.5), thin_quad_matrix(0.5))      # G4: drift then quad
    elems = [
        {"type": "DRIFT", "L": 1.0},
        _matrix_elem(R, C),
        {"type": "RCOL", "ax": 300e-6, "ay": 300e-6},
        {"type": "WAKE", "nb": 512, "window": "AUTO_MINMAX", "wake": "RESONATOR",
         "f": 1e9, "Q": 1.0, "Rs": 1e3, "interp": True},
    ]
    return Workload("cfg0", 0, n or 100_000, 1e9, 1e-9, False, 1, "turn", elems, "gauss6")


def _cfg1(n):
    elems = []
    count = 0
    for cell in range(25):
        k = 0.8 if cell % 2 == 0 else -0.8
        quad = compose(drift_matrix(0.1), thin_quad_matrix(k), drift_matrix(0.1))   # G6
        for e in (_matrix_elem(*quad), {"type": "ECOL", "a": 250e-6, "b": 250e-6},
                  _matrix_elem(*drift_matrix(2.0))):
            elems.append(e)
            count += 1
            if count in (16, 33):
                elems.append({"type": "RFKICK", "V": 1e6, "f": 2.856e9, "phi": np.pi / 2})
    assert len(elems) == 77
    return Workload("cfg1", 1, n or 1_000_000, 1e9, 1e-9, False, 1, "element", elems, "gauss6")


def _cfg2(n):
    dt = 0.05e-12
    k = np.arange(4096, dtype=np.float64)
    t = k * dt
    table = 1e14 * np.exp(-t / 10e-12) * np.cos(2 * np.pi * 3e9 * t)                # G16
    elems = [
        {"type": "DRIFT", "L": 1.0},
        {"type": "WAKE", "nb": 8192, "window": "AUTO_TABLE", "wake": "TABLE",
         "table": np.ascontiguousarray(table), "dt_table": dt, "interp": True},
    ]
    return Workload("cfg2", 2, n or 10_000_000, 1e9, 1e-9, True, 10, "none", elems, "chirp")


def _ring_tail():
    return [
        {"type": "RFKICK", "V": 5e6, "f": 500e6, "phi": np.deg2rad(160.0)},
        {"type": "WAKE", "nb": 1024, "window": "AUTO_MINMAX", "wake": "RESONATOR",
         "f": 1.3e9, "Q": 1e4, "Rs": 1e3, "interp": True},
    ]


def _one_turn_traces(ks, L):
    Mx = np.eye(2)
    My = np.eye(2)
    D = np.array([[1.0, L], [0.0, 1.0]])
    for k in ks:
        Mx = np.array([[1.0, 0.0], [-k, 1.0]]) @ D @ Mx
        My = np.array([[1.0, 0.0], [+k, 1.0]]) @ D @ My
    return np.trace(Mx), np.trace(My)


def _cfg3(n, n_matrices=200, n_turns=100):
    """cfg3-stable (G23): alternating-sign quads 0.4(1 + 0.1 u), 1 m drifts, sub-seed advanced
    until both planes are stable (|trace| < 1.9)."""
    L = 1.0
    seed = SEED_BASE + 3
    sign = np.where(np.arange(n_matrices) % 2 == 0, 1.0, -1.0)
    for attempt in range(10_000):
        u = uniform01(seed, 100 + attempt, n_matrices) - 0.5
        ks = sign * 0.4 * (1.0 + 0.1 * u)
        tx, ty = _one_turn_traces(ks, L)
        if abs(tx) < 1.9 and abs(ty) < 1.9:
            break
    else:  # pragma: no cover
        raise RuntimeError("no stable cfg3 ring found")
    elems = [_matrix_elem(*compose(drift_matrix(L), thin_quad_matrix(k))) for k in ks]
    elems += _ring_tail()
    w = Workload("cfg3", 3, n or 100_000_000, 3e9, 1e-9, True, n_turns, "turn", elems, "gauss6",
                 notes=f"cfg3-stable sub-seed attempt {attempt}, traces {tx:+.3f} {ty:+.3f}")
    return w


def _cfg3_literal(n, n_turns=5):
    seed = SEED_BASE + 3
    ks = uniform01(seed, 99, 200) - 0.5                                  # k1L in [-0.5, 0.5]
    elems = [_matrix_elem(*compose(drift_matrix(1.0), thin_quad_matrix(k))) for k in ks]
    elems += _ring_tail()
    return Workload("cfg3-literal", 3, n or 100_000_000, 3e9, 1e-9, True, n_turns, "turn", elems,
                    "gauss6", notes="literal random ring; exponentially unstable (G23)")


def _cfg4(n):
    p0c = 1e9
    beta0 = beta0_of(p0c, ELECTRON_MC2_EV)
    dt = 0.16e-3 / (beta0 * C_LIGHT)
    nb = 65536
    elems = []
    for i in range(20):
        hw = 0.9e-3 + (0.2e-3 - 0.9e-3) * i / 19.0
        elems.append({"type": "RCOL", "ax": hw, "ay": hw})
        elems.append({"type": "HISTO", "nb": nb, "window": "EXPLICIT",
                      "t_lo_rel": -(nb // 2) * dt, "dt": dt})
        elems.append({"type": "DRIFT", "L": 1.0})
    return Workload("cfg4", 4, n or 10_000_000, p0c, 1e-9, False, 1, "none", elems, "flattop")


def _p1(n):
    c0 = _cfg0(n)
    return Workload("p1-chain", 0, n or 100_000_000, 1e9, 1e-9, False, 1, "none",
                    c0.elements[:2], "gauss6", notes="cfg0 DRIFT+MATRIX run, no aperture")


def _p2(n, half_width=300e-6):
    c0 = _cfg0(n)
    elems = c0.elements[:2] + [{"type": "RCOL", "ax": half_width, "ay": half_width}]
    return Workload("p2-chain-rcol", 0, n or 100_000_000, 1e9, 1e-9, False, 1, "none",
                    elems, "gauss6", notes=f"cfg0 run ending in RCOL {half_width:g} m")


def _p3(n, n_matrices=8):
    c3 = _cfg3(n, n_matrices=200)
    return Workload("p3-matrices", 3, n or 100_000_000, 3e9, 1e-9, True, 1, "none",
                    c3.elements[:n_matrices], "gauss6", notes=f"{n_matrices} cfg3 matrices")


def _p7(n, n_cells=40, n_turns=1):
    """Third-order ring (track_particles M3): n_cells x [third-order drift 1 m, thin quadrupole +
    sextupole + octupole], strengths as p4 plus k3L = +-500 m^-3."""
    seed = SEED_BASE + 3
    u = uniform01(seed, 301, n_cells) - 0.5
    elems = []
    for i in range(n_cells):
        sg = 1.0 if i % 2 == 0 else -1.0
        elems.append(_matrix3_elem(*third_order_drift(1.0)))
        elems.append(_matrix3_elem(*thin_quad_sext_octupole(sg * 0.4 * (1.0 + 0.1 * u[i]), sg * 2.0, sg * 500.0)))
    return Workload("p7-third-order", 3, n or 100_000_000, 3e9, 1e-9, True, n_turns, "none",
                    elems, "gauss6", notes=f"{2 * n_cells} third-order maps per turn")


def _p4(n, n_cells=100, n_turns=1):
    """Second-order ring (track_particles M2): n_cells x [second-order drift 1 m,
    thin quadrupole + sextupole], quadrupole strengths of the stabilised cfg3 ring, k2L = +-2 m^-2."""
    seed = SEED_BASE + 3
    u = uniform01(seed, 300, n_cells) - 0.5
    elems = []
    for i in range(n_cells):
        k1L = (1.0 if i % 2 == 0 else -1.0) * 0.4 * (1.0 + 0.1 * u[i])
        k2L = (2.0 if i % 2 == 0 else -2.0)
        elems.append(_matrix2_elem(*second_order_drift(1.0)))
        elems.append(_matrix2_elem(*thin_quad_sextupole(k1L, k2L)))
    return Workload("p4-second-order", 3, n or 100_000_000, 3e9, 1e-9, True, n_turns, "none",
                    elems, "gauss6", notes=f"{2 * n_cells} second-order maps per turn")


def _p5(n, n_turns=1):
    """Transverse wake line (track_through_trwake): an offset bunch through two TRWAKE
    elements (transverse resonator, tabulated dipole wake) and a WAKE, drifts in between (readings G32-G34)."""
    off = np.zeros(6); off[0] = 2e-4; off[2] = -1e-4
    tt = np.arange(1024) * 0.02e-12
    table = 1e17 * np.sin(2 * np.pi * 5e9 * tt) * np.exp(-tt / 8e-12)          # V/C/m, W_T(0) = 0
    elems = [
        _matrix_elem(np.eye(6), off),
        {"type": "DRIFT", "L": 1.0},
        {"type": "TRWAKE", "nb": 512, "window": "AUTO_MINMAX", "wake": "RESONATOR_T", "f": 3e9, "Q": 20.0, "Rs": 1e6,
         "interp": True},
        {"type": "DRIFT", "L": 0.5},
        {"type": "TRWAKE", "nb": 2048, "window": "AUTO_TABLE", "wake": "TABLE", "table": table, "dt_table": 0.02e-12,
         "interp": True},
        {"type": "WAKE", "nb": 512, "window": "AUTO_MINMAX", "wake": "RESONATOR", "f": 1e9, "Q": 1.0, "Rs": 1e3,
         "interp": True},
        {"type": "DRIFT", "L": 0.25},
    ]
    return Workload("p5-trwake", 0, n or 100_000_000, 1e9, 1e-9, False, n_turns, "none", elems, "gauss6",
                    notes="offset bunch, TRWAKE resonator + TRWAKE table + WAKE")


def _p6(n, n_cavities=8, n_turns=1):
    """RFCW-style composite ("RFCW, which is a combination of RFCA, WAKE, TRWAKE ..."):
    an offset bunch through n_cavities x [drift x quad MATRIX of the cfg3 ring, RFKICK, WAKE, TRWAKE], the two wakes
    with the same 512-bin AUTO_MINMAX binning."""
    ring = _cfg3(n, n_matrices=max(8, n_cavities))
    mats = [e for e in ring.elements if e["type"] == "MATRIX"][:n_cavities]
    off = np.zeros(6); off[0] = 2e-4; off[2] = -1e-4
    elems = [_matrix_elem(np.eye(6), off)]
    for m in mats:
        elems += [m,
                  {"type": "RFKICK", "V": 2e6, "f": 1.3e9, "phi": 1.2},
                  {"type": "WAKE", "nb": 512, "window": "AUTO_MINMAX", "wake": "RESONATOR", "f": 1.3e9, "Q": 5.0,
                   "Rs": 1e3, "interp": True},
                  {"type": "TRWAKE", "nb": 512, "window": "AUTO_MINMAX", "wake": "RESONATOR_T", "f": 2.4e9, "Q": 10.0,
                   "Rs": 1e6, "interp": True}]
    return Workload("p6-rfcw", 3, n or 100_000_000, 3e9, 1e-9, False, n_turns, "none", elems, "gauss6",
                    notes=f"{n_cavities} cavities of MATRIX + RFKICK + WAKE + TRWAKE")


def make_workload(name: str, n: Optional[int] = None, **kw) -> Workload:
    """name in WORKLOAD_NAMES; n overrides the particle count (reduced-size parity cases)."""
    table = {
        "cfg0": _cfg0, "cfg1": _cfg1, "cfg2": _cfg2, "cfg3": _cfg3, "cfg3-literal": _cfg3_literal,
        "cfg4": _cfg4, "p1-chain": _p1, "p2-chain-rcol": _p2, "p3-matrices": _p3, "p4-second-order": _p4, "p5-trwake": _p5, "p6-rfcw": _p6, "p7-third-order": _p7,
    }
    if name not in table:
        raise KeyError(f"unknown workload {name!r}; known: {WORKLOAD_NAMES}")
    return table[name](n, **kw)

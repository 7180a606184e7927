"""Parity of every map kernel instantiation against the oracle with DENSE seeded coefficients.

The workloads of BASELINE.json only ever use uncoupled drift x thin-quadrupole matrices (26 of 36 R entries exactly
zero, row s = (0,0,0,0,1,0)) and higher-order maps with a handful of non-zero T / U entries, so a wrong index, lane
swap or transposition in a map kernel would pass every workload test.  Here R has all 36 entries non-zero (a random
symplectic matrix), all six C entries are non-zero, T has all 126 and U all 336 entries non-zero, and each case is
routed through one of the instantiations the planner can pick (unit tests compare CPU and GPU on
the same random inputs; per-element comparison):

    chain_kernel<8,2,0>   1-2 MATRIX                      chain_kernel<8,4,0>   3-4 MATRIX
    chain_kernel<8,2,1>   TKICK run                       chain_kernel<8,4,1>   one MATRIX2
    compact_kernel<8,0>   <= 8 maps + aperture            compact_kernel<8,1>   MATRIX2 + aperture
    chain_long_kernel<80,0>  >= 5 MATRIX (odd / even counts, DRIFT inside, > 80 maps: two launches)
    chain_long_kernel<80,1>  MATRIX2 runs                 chain_long_kernel<80,2>  MATRIX3 (12 slots, > 6 maps: two launches)
    chain_long_kernel<80,3>  ELG_TRACK_SPARSE_MATRICES with a dense matrix between patterned ones

Per-particle maps follow the arithmetic specification (explicit FMAs in a fixed order), so x, x', y, y', s, delta are
compared with array_equal.
"""
import numpy as np
import pytest

from elg_inputs import dense_map_element, make_workload

pytestmark = pytest.mark.gpu

SIZES = [1, 1535, 1536, 1537, 100_003]
SOFT = dict(strength=0.1, c_s=1e-3, t_scale=0.3, u_scale=300.0)      # long runs of higher-order maps stay finite


@pytest.fixture(scope="module")
def elg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1710_07350_b200 import elg as mod
    mod.lib()
    return mod


def _run_both(elg, elgo, elems, n, n_turns=1, ring=False, sparse=False, seed_shift=0.0):
    v0 = make_workload("cfg0", n=n).particles()
    v0[4] += seed_shift
    ob = elgo.Bunch(v0, 1e9, 1e-9)
    ob.track(elgo.Beamline(elems, ring=ring), n_turns, n_threads=8)
    gbl = elg.Beamline(elems, ring=ring)
    gb = elg.Bunch(v0, 1e9, 1e-9, beamline=gbl)
    gb.sparse_matrices = sparse
    gb.track(gbl, n_turns)
    return ob, gb, gbl


def _aperture_for(pv, kind, keep=0.7):
    """An aperture (centred on the axis, G17) that keeps about `keep` of the particles pv (6, n), whatever their offset."""
    if kind == "RCOL":
        k = np.sqrt(keep)
        return {"type": "RCOL", "ax": float(np.quantile(np.abs(pv[0]), k)), "ay": float(np.quantile(np.abs(pv[2]), k))}
    a0, b0 = np.max(np.abs(pv[0])), np.max(np.abs(pv[2]))
    k = np.sqrt(np.quantile((pv[0] / a0) ** 2 + (pv[2] / b0) ** 2, keep))
    return {"type": "ECOL", "a": float(a0 * k), "b": float(b0 * k)}


def _assert_identical(ob, gb, what=""):
    ov, oid = ob.read()
    gv, gid = gb.read()
    assert np.all(np.isfinite(ov)), "test input must keep the beam finite"
    assert np.array_equal(gid, oid), what
    for c, name in enumerate(("x", "x'", "y", "y'", "s", "delta")):
        assert np.array_equal(gv[c], ov[c]), f"{what}: coordinate {name} differs"


# ------------------------------------------------------------------------------------ first order, short runs
@pytest.mark.parametrize("n", SIZES)
@pytest.mark.parametrize("n_mat", [1, 2, 3, 4])
def test_dense_matrix_short_runs(elg, elgo, n, n_mat):
    """1-2 matrices: chain_kernel<8,2,0>; 3-4: chain_kernel<8,4,0> (parameter-bank coefficients)."""
    elems = [dense_map_element(100 + k) for k in range(n_mat)]
    ob, gb, gbl = _run_both(elg, elgo, elems, n)
    assert gbl.launches_per_turn("none") == 1
    _assert_identical(ob, gb, f"{n_mat} dense MATRIX")


@pytest.mark.parametrize("n", SIZES)
def test_dense_matrix_with_drifts_short(elg, elgo, n):
    """DRIFT, MATRIX, DRIFT, MATRIX, DRIFT: s row, C and the sqrt path together (P = 2)."""
    elems = [{"type": "DRIFT", "L": 0.7}, dense_map_element(7), {"type": "DRIFT", "L": -0.3}, dense_map_element(8),
             {"type": "DRIFT", "L": 1.9}]
    ob, gb, gbl = _run_both(elg, elgo, elems, n)
    assert gbl.launches_per_turn("none") == 1
    _assert_identical(ob, gb)


# ------------------------------------------------------------------------------------ first order, long runs
@pytest.mark.parametrize("n", SIZES)
@pytest.mark.parametrize("n_mat", [5, 6, 23, 80, 81, 163])
def test_dense_matrix_long_runs(elg, elgo, n, n_mat):
    """>= 5 matrices: chain_long_kernel<80,0> (coefficients in shared memory, LDS.128 pairs, 6 particles per thread):
    odd and even counts (the pairing), exactly one parameter block (80), one more (81), and three launches (163)."""
    if n == 100_003 and n_mat == 163:
        n = 20_011
    elems = [dense_map_element(1000 + k, strength=0.15, c_s=0.05) for k in range(n_mat)]
    ob, gb, gbl = _run_both(elg, elgo, elems, n)
    assert gbl.launches_per_turn("none") == (n_mat + 79) // 80
    _assert_identical(ob, gb, f"{n_mat} dense MATRIX (long run)")


@pytest.mark.parametrize("n", [1537, 50_021])
def test_dense_matrix_long_run_with_other_maps(elg, elgo, n):
    """DRIFTs between the matrices break the pairing at odd and even positions; two turns of a ring."""
    elems = []
    for k in range(24):
        elems.append(dense_map_element(2000 + k, strength=0.15, c_s=0.05))
        if k in (0, 3, 4, 11, 18, 22):
            elems.append({"type": "DRIFT", "L": 0.25 + 0.1 * k})
    ob, gb, gbl = _run_both(elg, elgo, elems, n, n_turns=2, ring=True)
    assert gbl.launches_per_turn("none") == 1
    _assert_identical(ob, gb)


def test_dense_matrix_then_rfkick_tolerance(elg, elgo):
    """With a dense matrix behind an RFKICK the 2-ulp sin difference in delta spreads to all coordinates: compared at
    north_star's 1e-12 (relative to max(|value|, sigma), G21) instead of bit for bit."""
    elems = [dense_map_element(31), {"type": "RFKICK", "V": 1e6, "f": 2.856e9, "phi": 0.7}, dense_map_element(32),
             {"type": "DRIFT", "L": 0.5}, dense_map_element(33)]
    ob, gb, _ = _run_both(elg, elgo, elems, 70_001)
    ov, _ = ob.read(); gv, _ = gb.read()
    sig = ov.std(axis=1, keepdims=True)
    assert np.max(np.abs(gv - ov) / np.maximum(np.abs(ov), sig)) <= 1e-12


# ------------------------------------------------------------------------------------ runs ending in an aperture
@pytest.mark.parametrize("n", SIZES)
@pytest.mark.parametrize("n_mat,kind", [(1, "RCOL"), (2, "ECOL"), (4, "RCOL"), (8, "ECOL")])
def test_dense_matrix_run_ending_in_aperture(elg, elgo, n, n_mat, kind):
    """compact_kernel<8,0>: up to 8 dense matrices applied inside the compacting run (2 particles per thread), the
    aperture cutting at the 85 % quantiles of the mapped beam."""
    elems = [dense_map_element(300 + k, strength=0.3, c_s=0.01) for k in range(n_mat)]
    v0 = make_workload("cfg0", n=max(n, 4000)).particles()
    probe = elgo.Bunch(v0, 1e9, 1e-9); probe.track(elgo.Beamline(elems), 1)
    pv, _ = probe.read()
    ap = _aperture_for(pv, kind)                                                     # ~ 30 % loss
    line = elems + [ap, {"type": "DRIFT", "L": 0.5}, dense_map_element(399)]
    ob, gb, gbl = _run_both(elg, elgo, line, n)
    assert gbl.launches_per_turn("none") == 2
    _assert_identical(ob, gb)
    oi, ot, oe, oc = ob.lost(); gi, gt, ge, gc = gb.lost()
    assert np.array_equal(gi, oi) and np.array_equal(ge, oe) and np.array_equal(gc, oc)
    if n >= 1535:
        assert 0.1 * n < oi.size < 0.6 * n


# ------------------------------------------------------------------------------------ second order
@pytest.mark.parametrize("n", SIZES)
def test_dense_matrix2_single(elg, elgo, n):
    """One MATRIX2 (4 parameter slots): chain_kernel<8,4,1>, pair-major T from the constant bank."""
    elems = [dense_map_element(41, order=2)]
    ob, gb, gbl = _run_both(elg, elgo, elems, n)
    assert gbl.launches_per_turn("none") == 1
    _assert_identical(ob, gb)


@pytest.mark.parametrize("n", SIZES)
@pytest.mark.parametrize("n_map", [2, 3, 12, 21])
def test_dense_matrix2_long_runs(elg, elgo, n, n_map):
    """>= 2 MATRIX2: chain_long_kernel<80,1> (20 maps fill a parameter block; 21 -> two launches)."""
    elems = [dense_map_element(4000 + k, order=2, **SOFT) for k in range(n_map)]
    ob, gb, gbl = _run_both(elg, elgo, elems, n)
    assert gbl.launches_per_turn("none") == (n_map + 19) // 20
    _assert_identical(ob, gb)


@pytest.mark.parametrize("n", [1537, 60_007])
def test_dense_matrix2_mixed_with_first_order_and_aperture(elg, elgo, n):
    """MATRIX, MATRIX2, DRIFT, MATRIX2, MATRIX in a long run; then MATRIX2 + ECOL (compact_kernel<8,1>)."""
    e1 = lambda k: dense_map_element(5000 + k, order=1, strength=0.1, c_s=1e-3)
    e2 = lambda k: dense_map_element(5100 + k, order=2, **SOFT)
    elems = [e1(0), e2(0), {"type": "DRIFT", "L": 0.4}, e2(1), e1(1), e1(2), e2(2),
             {"type": "RCOL", "ax": 1.0, "ay": 1.0}]                   # wide open: only ends the long run
    tail = [e2(3), {"type": "DRIFT", "L": 0.2}, e1(3)]                 # 6 slots + aperture: compact_kernel<8,1>
    v0 = make_workload("cfg0", n=4000).particles()
    probe = elgo.Bunch(v0, 1e9, 1e-9); probe.track(elgo.Beamline(elems + tail), 1)
    pv, _ = probe.read()
    line = elems + tail + [_aperture_for(pv, "ECOL"), e2(4)]
    ob, gb, gbl = _run_both(elg, elgo, line, n)
    assert gbl.launches_per_turn("none") == 1 + 1 + 1 + 1             # long run, RCOL alone, compacting run, last map
    _assert_identical(ob, gb)
    oi, _, oe, oc = ob.lost(); gi, _, ge, gc = gb.lost()
    assert 0 < oi.size < n and np.array_equal(gi, oi) and np.array_equal(gc, oc)


# ------------------------------------------------------------------------------------ third order
@pytest.mark.parametrize("n", [1, 1023, 1024, 1025, 1537, 100_003])
@pytest.mark.parametrize("n_map", [1, 2, 6, 7, 14])
def test_dense_matrix3(elg, elgo, n, n_map):
    """MATRIX3 (12 slots: R, C | Tt[21][6] | Ut[56][6]): chain_long_kernel<80,2>, 4 particles per thread (1024-particle
    tiles); 6 maps fill a parameter block, 7 -> two launches."""
    if n == 100_003 and n_map == 14:
        n = 30_011
    elems = [dense_map_element(6000 + k, order=3, **SOFT) for k in range(n_map)]
    ob, gb, gbl = _run_both(elg, elgo, elems, n)
    assert gbl.launches_per_turn("none") == (n_map + 5) // 6
    _assert_identical(ob, gb)


def test_dense_all_orders_in_one_run(elg, elgo):
    """MATRIX, MATRIX2 and MATRIX3 with DRIFTs in one level-2 run, then a collimator (split: long run + compacting run)."""
    elems = [dense_map_element(7001, 1, strength=0.1, c_s=1e-3), dense_map_element(7002, 3, **SOFT),
             {"type": "DRIFT", "L": 0.3}, dense_map_element(7003, 2, **SOFT), dense_map_element(7004, 1, strength=0.1, c_s=1e-3),
             dense_map_element(7005, 1, strength=0.1, c_s=1e-3), dense_map_element(7006, 3, **SOFT)]
    v0 = make_workload("cfg0", n=4000).particles()
    probe = elgo.Bunch(v0, 1e9, 1e-9); probe.track(elgo.Beamline(elems), 1)
    pv, _ = probe.read()
    line = elems + [_aperture_for(pv, "RCOL"),
                    dense_map_element(7007, 2, **SOFT)]
    ob, gb, _ = _run_both(elg, elgo, line, 45_007)
    _assert_identical(ob, gb)
    oi, _, _, oc = ob.lost(); gi, _, _, gc = gb.lost()
    assert 0 < oi.size < 45_007 and np.array_equal(gi, oi) and np.array_equal(gc, oc)


# ------------------------------------------------------------------------------------ flagged sparse option
@pytest.mark.parametrize("n", [1537, 80_021])
def test_sparse_option_with_dense_matrices_between_patterned_ones_vs_oracle(elg, elgo, n):
    """ELG_TRACK_SPARSE_MATRICES (chain_long_kernel<80,3>): patterned (drift x quad) matrices take the 20-FMA path,
    dense ones in the same run stay dense; compared with the ORACLE (round 1 compared GPU with GPU)."""
    ring = make_workload("cfg3", n=8, n_matrices=30)
    mats = [e for e in ring.elements if e["type"] == "MATRIX"]
    elems = []
    for k, m in enumerate(mats):
        elems.append(m)
        if k in (0, 5, 6, 17, 28):
            elems.append(dense_map_element(8000 + k, strength=0.15, c_s=0.05))
    ob, gb, gbl = _run_both(elg, elgo, elems, n, sparse=True)
    _assert_identical(ob, gb, "sparse option")


# ------------------------------------------------------------------------------------ wake kicks without interpolation
@pytest.mark.parametrize("n", [3, 1537, 120_001])
def test_wake_and_trwake_own_bin_kicks_end_to_end(elg, elgo, n):
    """interp = 0 (G14: the particle's own bin) for WAKE and TRWAKE in the PRODUCT path (OP_KICK / OP_TKICK inside
    the next fused run), alone and as the merged RFCW pair."""
    w = make_workload("p5-trwake", n=n)
    elems = [dict(e) for e in w.elements]
    for e in elems:
        if e["type"] in ("WAKE", "TRWAKE"):
            e["interp"] = False
    # + a merged pair (same binning) with own-bin kicks
    elems += [{"type": "WAKE", "nb": 256, "window": "AUTO_MINMAX", "wake": "RESONATOR", "f": 1.3e9, "Q": 5.0, "Rs": 1e3,
               "interp": False},
              {"type": "TRWAKE", "nb": 256, "window": "AUTO_MINMAX", "wake": "RESONATOR_T", "f": 2.4e9, "Q": 10.0,
               "Rs": 1e6, "interp": False},
              {"type": "DRIFT", "L": 0.1}]
    v0 = w.particles()
    ob = elgo.Bunch(v0, w.p0c_eV, w.charge_C)
    oo = ob.track(elgo.Beamline(elems), 1, want_stage_outputs=True, n_threads=8)
    gbl = elg.Beamline(elems); gb = elg.Bunch(v0, w.p0c_eV, w.charge_C, beamline=gbl)
    go = gb.track(gbl, 1, want_stage_outputs=True)
    assert np.array_equal(go["window"][0], oo["window"][0]) and np.array_equal(go["hist"][:512], oo["hist"][:512])
    assert go["V"].size == oo["V"].size
    ov, oid = ob.read(); gv, gid = gb.read()
    assert np.array_equal(gid, oid)
    if n > 3:
        sig = ov.std(axis=1, keepdims=True)
        assert np.max(np.abs(gv - ov) / np.maximum(np.abs(ov), sig)) <= 1e-12
        # own-bin and interpolated kicks differ: the branch under test is really taken
        wi = make_workload("p5-trwake", n=n)
        oi = elgo.Bunch(v0, w.p0c_eV, w.charge_C); oi.track(elgo.Beamline(wi.elements), 1, n_threads=8)
        assert np.max(np.abs(oi.read()[0][1] - ov[1])) > 0


def test_rfcw_pair_with_different_interpolation_flags(elg, elgo):
    """A WAKE + TRWAKE pair that shares its histogram pass but not its interpolation rule: the planner must keep two
    kick ops (the fused OP_KICK3 holds one rule for both)."""
    n = 50_003
    w = make_workload("p5-trwake", n=n)
    pair = [{"type": "WAKE", "nb": 300, "window": "AUTO_MINMAX", "wake": "RESONATOR", "f": 1.3e9, "Q": 5.0, "Rs": 1e3,
             "interp": True},
            {"type": "TRWAKE", "nb": 300, "window": "AUTO_MINMAX", "wake": "RESONATOR_T", "f": 2.4e9, "Q": 10.0,
             "Rs": 1e6, "interp": False},
            {"type": "DRIFT", "L": 0.1}]
    same = [dict(e, interp=True) for e in pair[:2]] + [pair[2]]
    v0 = w.particles()
    v0[0] += 2e-4; v0[2] -= 1e-4
    res = {}
    for name, elems in (("mixed", pair), ("both", same)):
        ob = elgo.Bunch(v0, w.p0c_eV, w.charge_C)
        ob.track(elgo.Beamline(elems), 1, n_threads=8)
        gbl = elg.Beamline(elems); gb = elg.Bunch(v0, w.p0c_eV, w.charge_C, beamline=gbl)
        gb.track(gbl, 1)
        ov, oid = ob.read(); gv, gid = gb.read()
        assert np.array_equal(gid, oid)
        sig = ov.std(axis=1, keepdims=True)
        assert np.max(np.abs(gv - ov) / np.maximum(np.abs(ov), sig)) <= 1e-12
        res[name] = gv
    assert np.array_equal(res["mixed"][5], res["both"][5])          # same longitudinal kick
    assert np.max(np.abs(res["mixed"][1] - res["both"][1])) > 0      # different transverse rule

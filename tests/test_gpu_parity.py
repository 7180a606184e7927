"""Parity of the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Protocol: stage by stage with the ORACLE's input to each stage uploaded
to the GPU, then end to end per workload.  Bars (BASELINE.json north_star): integer / index work
bit-exact; coordinates <= 1e-12 relative after one pass, <= 1e-9 after 100 turns; moments and wake
voltages <= 1e-10 relative to their maximum.  "Relative" for coordinate k means relative to
max(|oracle value|, sigma_k) (G21).  Particles within 1e-12 of an aperture or bin edge would be listed
separately; with the shared arithmetic specification the lists are expected to be empty and the tests
assert exact equality.
"""
import math

import numpy as np
import pytest

from elg_inputs import make_workload

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def elg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1710_07350_b200 import elg as mod
    mod.lib()
    return mod


def rel_err(a, b):
    """max over coordinates of |a-b| / max(|b|, sigma_k) (G21)."""
    a = np.asarray(a); b = np.asarray(b)
    if b.size == 0:
        return 0.0
    sig = b.std(axis=1, keepdims=True) if b.ndim == 2 else np.std(b)
    den = np.maximum(np.abs(b), np.maximum(sig, 1e-300))
    return float(np.max(np.abs(a - b) / den))


def both(elg, elgo, w, n_turns=None, moments_every=None, n_threads=8, stage=True):
    """Track workload w on both sides from the same bytes."""
    v0 = w.particles()
    nt = w.n_turns if n_turns is None else n_turns
    mom = w.moments_every if moments_every is None else moments_every
    ob = elgo.Bunch(v0, w.p0c_eV, w.charge_C)
    obl = elgo.Beamline(w.elements, ring=w.ring)
    oo = ob.track(obl, nt, moments_every=mom, n_threads=n_threads, want_stage_outputs=stage)
    gbl = elg.Beamline(w.elements, ring=w.ring)
    gb = elg.Bunch(v0, w.p0c_eV, w.charge_C, beamline=gbl)
    go = gb.track(gbl, nt, moments_every=mom, want_stage_outputs=stage)
    return ob, oo, gb, go


def check_lost(ob, gb):
    oi, ot, oe, oc = ob.lost()
    gi, gt, ge, gc = gb.lost()
    assert np.array_equal(gi, oi), "lost IDs / order differ"
    assert np.array_equal(gt, ot) and np.array_equal(ge, oe)
    assert np.array_equal(gc[:, :5], oc[:, :5]), "lost-particle coordinates differ"
    if oc.size:
        assert np.max(np.abs(gc[:, 5] - oc[:, 5])) <= 1e-12 * max(np.max(np.abs(oc[:, 5])), 1e-300)
    return oi.size


def check_records(go, oo, tol=1e-10):
    gr, orr = go["records"], oo["records"]
    assert gr.shape == orr.shape
    if gr.size == 0:
        return
    assert np.array_equal(gr[:, 0], orr[:, 0]), "n_alive per record differs"
    for k in range(orr.shape[0]):
        if orr[k, 0] == 0:
            continue
        S = orr[k, 7:].reshape(6, 6)
        sig = np.sqrt(np.diag(S))
        cen_tol = tol * np.maximum(np.max(np.abs(orr[k, 1:7])), sig)       # floor: sigma of that coordinate
        assert np.all(np.abs(gr[k, 1:7] - orr[k, 1:7]) <= cen_tol + 1e-300), f"centroid, record {k}"
        assert np.max(np.abs(gr[k, 7:] - orr[k, 7:])) <= tol * np.max(np.abs(S)) + 1e-300, f"Sigma, record {k}"


# ------------------------------------------------------------------------------------ (i) transport
@pytest.mark.parametrize("n", [1, 2, 511, 512, 513, 100_003])
def test_transport_chain_bitexact(elg, elgo, n):
    """DRIFT + MATRIX fused run (p1): several tiles and a ragged tail; <= 1e-12, in fact bit-identical."""
    w = make_workload("p1-chain", n=n)
    ob, oo, gb, go = both(elg, elgo, w, stage=False)
    ov, oid = ob.read()
    gv, gid = gb.read()
    assert np.array_equal(gid, oid)
    assert rel_err(gv, ov) <= 1e-12
    assert np.array_equal(gv, ov), "fma/sqrt arithmetic specification should make this bit-identical"


def test_each_map_alone(elg, elgo):
    """Single-element beamlines (one launch per element, like the paper): DRIFT, MATRIX, RFKICK."""
    base = make_workload("cfg1", n=70_001)
    v0 = base.particles()
    v0[4] += 3.25                                   # s is an absolute path length
    elems = {
        "DRIFT": {"type": "DRIFT", "L": 2.5},
        "MATRIX": base.elements[0],
        "RFKICK": {"type": "RFKICK", "V": 1e6, "f": 2.856e9, "phi": 0.7},
    }
    for name, e in elems.items():
        ob = elgo.Bunch(v0, 1e9, 1e-9); obl = elgo.Beamline([e])
        ob.track(obl, 1)
        gbl = elg.Beamline([e]); gb = elg.Bunch(v0, 1e9, 1e-9, beamline=gbl)
        gb.track(gbl, 1)
        ov, _ = ob.read(); gv, _ = gb.read()
        assert rel_err(gv, ov) <= 1e-12, name
        if name != "RFKICK":
            assert np.array_equal(gv, ov), name
        else:
            assert np.array_equal(gv[:5], ov[:5])                    # only delta sees sin (<= 2 ulp)


def _long_line(n_mat, extra):
    """n_mat distinct symplectic drift x quad matrices (cfg3's generator) with other maps spliced in."""
    ring = make_workload("cfg3", n=8, n_matrices=n_mat)
    mats = [e for e in ring.elements if e["type"] == "MATRIX"]
    out = []
    for k, m in enumerate(mats):
        out.append(m)
        if k in extra:
            out.append(extra[k])
    return out


@pytest.mark.parametrize("n", [1, 1535, 1536, 1537, 3 * 1536 + 7, 200_001])
def test_long_run_kernel_bitexact(elg, elgo, n):
    """Runs of more than 8 maps go through chain_long_kernel (6 particles per thread, 1536-particle tiles,
    coefficients in shared memory, matrix pairs): odd matrix counts, DRIFT / RFKICK inside the run, ragged tails."""
    elems = _long_line(23, {4: {"type": "DRIFT", "L": 0.75}, 11: {"type": "RFKICK", "V": 2e6, "f": 1.3e9, "phi": 2.1},
                            12: {"type": "DRIFT", "L": 0.25}})
    v0 = make_workload("cfg0", n=n).particles()
    ob = elgo.Bunch(v0, 1e9, 1e-9); ob.track(elgo.Beamline(elems), 1)
    gbl = elg.Beamline(elems)
    assert gbl.launches_per_turn("none") == 1                      # one fused run
    gb = elg.Bunch(v0, 1e9, 1e-9, beamline=gbl); gb.track(gbl, 1)
    ov, oid = ob.read(); gv, gid = gb.read()
    assert np.array_equal(gid, oid)
    assert np.array_equal(gv[:5], ov[:5])
    assert rel_err(gv, ov) <= 1e-12


def test_long_run_ending_in_aperture(elg, elgo):
    """More than 8 maps and then a collimator: long-run kernel, then the aperture as a compacting run."""
    elems = _long_line(12, {}) + [{"type": "ECOL", "a": 400e-6, "b": 350e-6}, {"type": "DRIFT", "L": 1.0}]
    v0 = make_workload("cfg0", n=50_003).particles()
    ob = elgo.Bunch(v0, 1e9, 1e-9); ob.track(elgo.Beamline(elems), 1)
    gbl = elg.Beamline(elems); gb = elg.Bunch(v0, 1e9, 1e-9, beamline=gbl); gb.track(gbl, 1)
    ov, oid = ob.read(); gv, gid = gb.read()
    assert 0 < gid.size < 50_003
    assert np.array_equal(gid, oid) and np.array_equal(gv, ov)
    check_lost(ob, gb)


@pytest.mark.parametrize("n,n_cells", [(1, 1), (513, 1), (1537, 2), (100_003, 3), (40_001, 30)])
def test_second_order_maps_bitexact(elg, elgo, n, n_cells):
    """MATRIX2 (second-order transport map, G31) in short runs (parameter-bank kernel, 4 slots per map) and in
    long runs (chain_long_kernel): bit-identical to the oracle, two turns."""
    w = make_workload("p4-second-order", n=n, n_cells=n_cells, n_turns=2)
    ob, oo, gb, go = both(elg, elgo, w, stage=False)
    ov, oid = ob.read(); gv, gid = gb.read()
    assert np.array_equal(gid, oid)
    assert np.array_equal(gv, ov)


@pytest.mark.parametrize("n,n_cells", [(1, 1), (1537, 1), (50_001, 7)])
def test_third_order_maps_bitexact(elg, elgo, n, n_cells):
    """MATRIX3 (third-order transport map, G35; 12 parameter slots, long-run kernel): bit-identical, two turns."""
    w = make_workload("p7-third-order", n=n, n_cells=n_cells, n_turns=2)
    ob, oo, gb, go = both(elg, elgo, w, stage=False)
    ov, oid = ob.read(); gv, gid = gb.read()
    assert np.array_equal(gid, oid) and np.array_equal(gv, ov)


def test_third_order_then_aperture(elg, elgo):
    from elg_inputs import thin_quad_sext_octupole, third_order_drift
    m3 = lambda t: {"type": "MATRIX3", "R": t[0], "C": t[1], "T": t[2], "U": t[3]}
    elems = [m3(third_order_drift(0.8)), m3(thin_quad_sext_octupole(0.3, 20.0, 4000.0)), {"type": "DRIFT", "L": 0.4},
             {"type": "RCOL", "ax": 250e-6, "ay": 260e-6}, m3(third_order_drift(0.2))]
    v0 = make_workload("cfg0", n=30_001).particles()
    ob = elgo.Bunch(v0, 1e9, 1e-9); ob.track(elgo.Beamline(elems), 1)
    gbl = elg.Beamline(elems); gb = elg.Bunch(v0, 1e9, 1e-9, beamline=gbl); gb.track(gbl, 1)
    ov, oid = ob.read(); gv, gid = gb.read()
    assert 0 < gid.size < 30_001 and np.array_equal(gid, oid) and np.array_equal(gv, ov)
    check_lost(ob, gb)


def test_second_order_mixed_with_other_maps(elg, elgo):
    """MATRIX2 between MATRIX, DRIFT and RFKICK, then a collimator: slot accounting of the planner."""
    from elg_inputs import second_order_drift, thin_quad_sextupole
    m2 = lambda t: {"type": "MATRIX2", "R": t[0], "C": t[1], "T": t[2]}
    lin = _long_line(23, {})[:5]
    elems = [lin[0], m2(thin_quad_sextupole(0.3, 40.0)), {"type": "DRIFT", "L": 0.5}, m2(second_order_drift(0.7)),
             lin[1], lin[2], {"type": "RFKICK", "V": 1e6, "f": 1.3e9, "phi": 0.4}, m2(thin_quad_sextupole(-0.3, -40.0)),
             lin[3], m2(second_order_drift(1.1)), lin[4], {"type": "RCOL", "ax": 500e-6, "ay": 450e-6},
             m2(thin_quad_sextupole(0.2, 10.0)), {"type": "DRIFT", "L": 0.3}]
    v0 = make_workload("cfg0", n=60_001).particles()
    ob = elgo.Bunch(v0, 1e9, 1e-9); ob.track(elgo.Beamline(elems), 1)
    gbl = elg.Beamline(elems); gb = elg.Bunch(v0, 1e9, 1e-9, beamline=gbl); gb.track(gbl, 1)
    ov, oid = ob.read(); gv, gid = gb.read()
    assert 0 < gid.size < 60_001 and np.array_equal(gid, oid)
    assert np.array_equal(gv[:5], ov[:5]) and rel_err(gv, ov) <= 1e-12
    check_lost(ob, gb)


@pytest.mark.parametrize("n", [1, 513, 150_001])
def test_fiducial_rf_phase(elg, elgo, n):
    """RFKICK with the phase reference on the bunch (G36): exact integer reduction, so s_ref is bit-identical and
    delta differs by sin's 2 ulp only."""
    ring = _long_line(23, {})
    elems = [ring[0], {"type": "RFKICK", "V": 2e6, "f": 1.3e9, "phi": 0.9, "fiducial": True}, ring[1],
             {"type": "DRIFT", "L": 0.5}, {"type": "RFKICK", "V": 1e6, "f": 2.856e9, "phi": 2.0, "fiducial": True},
             {"type": "RFKICK", "V": 1e6, "f": 2.856e9, "phi": 0.1}, ring[2]]
    v0 = make_workload("cfg0", n=n).particles()
    v0[4] += 2.5e-4                                          # the bunch is late: fiducial and design phase differ
    ob = elgo.Bunch(v0, 1e9, 1e-9); ob.track(elgo.Beamline(elems, ring=True), 3)
    gbl = elg.Beamline(elems, ring=True); gb = elg.Bunch(v0, 1e9, 1e-9, beamline=gbl); gb.track(gbl, 3)
    ov, _ = ob.read(); gv, _ = gb.read()
    assert np.array_equal(gv[:5], ov[:5])
    assert rel_err(gv, ov) <= 1e-12


# ------------------------------------------------------------------------------------ (ii) loss
def test_compaction_hand_placed(elg, elgo):
    """Edge-inclusive, NaN lost, Fig. 2 shape (20 particles, 4 lost)."""
    a = 300e-6
    n = 20
    v0 = np.zeros((6, n))
    v0[0] = np.linspace(-a, a, n)                 # both end points exactly on the edge: survive
    v0[5] = np.arange(n) * 1e-3
    lost_pos = [3, 7, 8, 19]
    v0[0, 3] = a * (1 + 1e-6); v0[2, 7] = -a * (1 + 1e-6); v0[0, 8] = np.nan; v0[2, 19] = np.nan
    e = [{"type": "RCOL", "ax": a, "ay": a}]
    ob = elgo.Bunch(v0, 1e9, 1e-9); ob.track(elgo.Beamline(e), 1)
    gbl = elg.Beamline(e); gb = elg.Bunch(v0, 1e9, 1e-9, beamline=gbl); gb.track(gbl, 1)
    gv, gid = gb.read(); ov, oid = ob.read()
    assert gid.tolist() == [i for i in range(n) if i not in lost_pos] == oid.tolist()
    assert np.array_equal(gv, ov)
    gi, gt, ge, gc = gb.lost()
    assert gi.tolist() == lost_pos and gt.tolist() == [0] * 4 and ge.tolist() == [0] * 4
    assert np.array_equal(gc[:, 5], v0[5, lost_pos])
    assert gb.n_alive == 16


@pytest.mark.parametrize("case", ["none_lost", "all_lost", "heavy", "ecol"])
def test_compaction_cases(elg, elgo, case):
    n = 200_001
    w = make_workload("cfg0", n=n)
    v0 = w.particles()
    e = {"none_lost": [{"type": "RCOL", "ax": 1.0, "ay": 1.0}],
         "all_lost": [{"type": "RCOL", "ax": 1e-12, "ay": 1e-12}],
         "heavy": [{"type": "DRIFT", "L": 0.3}, {"type": "RCOL", "ax": 60e-6, "ay": 90e-6}, {"type": "DRIFT", "L": 0.1},
                   {"type": "RCOL", "ax": 50e-6, "ay": 50e-6}],
         "ecol": [{"type": "ECOL", "a": 150e-6, "b": 220e-6}, {"type": "ECOL", "a": 120e-6, "b": 100e-6}]}[case]
    ob = elgo.Bunch(v0, 1e9, 1e-9); ob.track(elgo.Beamline(e), 1, n_threads=8)
    gbl = elg.Beamline(e); gb = elg.Bunch(v0, 1e9, 1e-9, beamline=gbl); gb.track(gbl, 1)
    ov, oid = ob.read(); gv, gid = gb.read()
    assert gb.n_alive == ob.n_alive
    assert np.array_equal(gid, oid) and np.array_equal(gv, ov)
    nl = check_lost(ob, gb)
    assert nl + oid.size == n
    if case == "all_lost":
        assert gb.n_alive == 0
        with pytest.raises(elg.ElgError) as ei:
            gb.moments()
        assert ei.value.code == elg.ESTATE
        gb.track(gbl, 1)                       # tracking an empty bunch is a no-op
        assert gb.n_alive == 0
    if case == "none_lost":
        assert nl == 0


def test_compaction_randomized_sizes(elg, elgo):
    """Many sizes around the tile (512) and row (blocks x 512) boundaries and random apertures: survivor IDs / order
    and the lost log against the oracle's stable partition (the scan has no chained look-back: a block adds the
    aggregates of one round-robin row to its own prefix, so row boundaries are the edge cases)."""
    import torch
    rows = 2 * torch.cuda.get_device_properties(0).multi_processor_count * 512
    rng = np.random.default_rng(99)
    sizes = [rows - 1, rows, rows + 1, 2 * rows + 513, 3 * rows - 511] + [int(x) for x in rng.integers(1, 2_000_000, 7)]
    for n in sizes:
        a = float(rng.choice([60e-6, 150e-6, 400e-6]))
        v0 = np.zeros((6, n)); v0[0] = rng.normal(size=n) * 1e-4; v0[2] = rng.normal(size=n) * 1e-4
        v0[5] = np.arange(n) * 1e-9
        e = [{"type": "ECOL", "a": a, "b": 1.3 * a}]
        ob = elgo.Bunch(v0, 1e9, 1e-9); ob.track(elgo.Beamline(e), 1)
        gbl = elg.Beamline(e); gb = elg.Bunch(v0, 1e9, 1e-9, beamline=gbl); gb.track(gbl, 1)
        ov, oid = ob.read(); gv, gid = gb.read()
        assert np.array_equal(gid, oid) and np.array_equal(gv, ov), n
        check_lost(ob, gb)


def test_lost_capacity_truncates(elg, elgo):
    w = make_workload("cfg4", n=50_000)
    v0 = w.particles()
    gbl = elg.Beamline(w.elements)
    gb = elg.Bunch(v0, w.p0c_eV, w.charge_C, beamline=gbl, lost_capacity=1000)
    gb.track(gbl, 1)
    ob = elgo.Bunch(v0, w.p0c_eV, w.charge_C); ob.track(elgo.Beamline(w.elements), 1)
    oi, ot, oe, oc = ob.lost()
    gi, gt, ge, gc = gb.lost()
    assert gi.size == 1000 and np.array_equal(gi, oi[:1000]) and np.array_equal(gc[:, :5], oc[:1000, :5])
    assert gb.n_alive == ob.n_alive
    assert np.array_equal(gb.read()[1], ob.read()[1])


# ------------------------------------------------------------------------------------ (iii) histogram
@pytest.mark.parametrize("nb,mode", [(512, "AUTO_MINMAX"), (8192, "AUTO_TABLE"), (65536, "EXPLICIT"), (100_000, "EXPLICIT")])
def test_histogram_stage(elg, elgo, nb, mode):
    """Protocol (iii): the ORACLE's coordinates and window uploaded, counts bit-exact.  elg_dbg_histogram runs
    tracking's own sequence (min/max epilogue, window_kernel, hist_kernel with the occupied-range privatisation)."""
    w = make_workload("cfg0", n=300_007)
    v = w.particles()
    v[4] += 1.5
    ibc = elgo.inv_bc(elgo.beta0(w.p0c_eV))
    kw = {"AUTO_MINMAX": {}, "AUTO_TABLE": {"dt_in": 1e-14},
          "EXPLICIT": {"t_lo_rel": -(nb // 2) * 5.3e-13, "dt_in": 5.3e-13, "t_design": 1.5 * ibc}}[mode]
    t_lo, dt, inv_dt = elgo.window(v[4], ibc, elgo.WIN[mode], nb, **kw)
    oc, binned = elgo.histogram(v[4], ibc, t_lo, inv_dt, nb)
    gc = elg.dbg_histogram(v[4], w.p0c_eV, t_lo, dt, nb)
    assert np.array_equal(gc, oc)
    # degenerate inputs: empty, all in one bin, NaN / out of range
    assert int(elg.dbg_histogram(np.zeros(0), w.p0c_eV, t_lo, dt, nb).sum()) == 0
    one = np.full(100_000, v[4, 0])
    assert np.array_equal(elg.dbg_histogram(one, w.p0c_eV, t_lo, dt, nb), elgo.histogram(one, ibc, t_lo, inv_dt, nb)[0])
    odd = np.array([np.nan, 1e30, -1e30, v[4, 1]])
    assert np.array_equal(elg.dbg_histogram(odd, w.p0c_eV, t_lo, dt, nb), elgo.histogram(odd, ibc, t_lo, inv_dt, nb)[0])


def test_histogram_aggregated_path(elg, elgo, monkeypatch):
    """Contention case (cfg4-like: everything in ~50 of 65536 bins) with and without warp-aggregated atomics."""
    w = make_workload("cfg4", n=400_000)
    v = w.particles()
    e = w.elements[1]
    ibc = elgo.inv_bc(elgo.beta0(w.p0c_eV))
    t_lo, dt, inv_dt = elgo.window(v[4], ibc, elgo.WIN["EXPLICIT"], e["nb"], t_lo_rel=e["t_lo_rel"], dt_in=e["dt"])
    oc, _ = elgo.histogram(v[4], ibc, t_lo, inv_dt, e["nb"])
    assert 30 <= (oc > 0).sum() <= 80
    for agg in ("0", "1"):
        monkeypatch.setenv("ELG_HIST_AGGREGATE", agg)
        assert np.array_equal(elg.dbg_histogram(v[4], w.p0c_eV, t_lo, dt, e["nb"]), oc)


def test_dipole_histogram_stage(elg, elgo):
    """TRWAKE stage (G33): counts bit-exact; the dipole sums (exact integer accumulation on the device) against the
    oracle's plain long-double sums at north_star's 1e-10 of the maximum -- in fact to the final rounding; and the
    device sums do not depend on the particle order, bit for bit."""
    w = make_workload("p5-trwake", n=250_003)
    v = w.particles()
    v[0] += 2e-4; v[2] -= 1e-4
    nb = 777
    ibc = elgo.inv_bc(elgo.beta0(w.p0c_eV))
    t_lo, dt, inv_dt = elgo.window(v[4], ibc, elgo.WIN["AUTO_MINMAX"], nb)
    oc, oDx, oDy, _ = elgo.dipole_histogram(v[4], v[0], v[2], ibc, t_lo, inv_dt, nb)
    gc, gDx, gDy = elg.dbg_dipole_histogram(v[4], v[0], v[2], w.p0c_eV, t_lo, dt, nb)
    assert np.array_equal(gc, oc)
    for g, o in ((gDx, oDx), (gDy, oDy)):
        assert np.max(np.abs(g - o)) <= 1e-10 * np.max(np.abs(o))
        assert np.max(np.abs(g - o)) <= 4e-16 * np.max(np.abs(o))               # what the arithmetic actually gives
    p = np.random.default_rng(3).permutation(v.shape[1])
    pc, pDx, pDy = elg.dbg_dipole_histogram(v[4, p], v[0, p], v[2, p], w.p0c_eV, t_lo, dt, nb)
    assert np.array_equal(pc, gc) and np.array_equal(pDx, gDx) and np.array_equal(pDy, gDy)
    # out-of-range / NaN offsets are counted, not summed (G33)
    s4 = np.full(4, v[4, 0]); x4 = np.array([1e-4, np.nan, 4e6, -2e-4]); y4 = np.array([1e-5, 1e-5, 1e-5, np.nan])
    oc4, oDx4, oDy4, _ = elgo.dipole_histogram(s4, x4, y4, ibc, t_lo, inv_dt, nb)
    gc4, gDx4, gDy4 = elg.dbg_dipole_histogram(s4, x4, y4, w.p0c_eV, t_lo, dt, nb)
    assert np.array_equal(gc4, oc4) and gc4.sum() == 4
    assert np.max(np.abs(gDx4 - oDx4)) <= 2.0 ** -64 and np.max(np.abs(gDy4 - oDy4)) <= 2.0 ** -64     # G33 resolution
    assert abs(gDx4.sum() - 1e-4) <= 2.0 ** -64 and oDx4.sum() == 1e-4 and abs(gDy4.sum() - 1e-5) <= 2.0 ** -64
    # offsets of kilometres take the other branch of the device's split (|x| >= 2^14 m): one particle per bin, so the
    # sum is the value itself
    big = np.array([5e4 + 1e-7, -7e5 - 1.0 / 3, 16384.0, -16383.999999, 1048575.9])
    s5 = v[4, 0] + (np.arange(5) - 2) * 3 * dt / ibc
    oc5, oDx5, oDy5, _ = elgo.dipole_histogram(s5, big, -big, ibc, t_lo, inv_dt, nb)
    gc5, gDx5, gDy5 = elg.dbg_dipole_histogram(s5, big, -big, w.p0c_eV, t_lo, dt, nb)
    assert np.array_equal(gc5, oc5) and gc5.sum() == 5 and gc5.max() == 1
    assert np.array_equal(gDx5, oDx5) and np.array_equal(gDy5, oDy5) and np.array_equal(np.sort(gDx5[gc5 > 0]), np.sort(big))


# ------------------------------------------------------------------------------------ (iv) wake, convolution
def test_wake_samples_and_convolution_stage(elg, elgo):
    rng = np.random.default_rng(11)
    for nb, kind, kw in ((512, 0, dict(f=1e9, Q=1.0, Rs=1e3)), (1024, 0, dict(f=1.3e9, Q=1e4, Rs=1e3)),
                         (8192, 1, None), (37, 1, None)):
        dt = 2.6e-14 if kind == 0 else 0.05e-12
        if kind == 1:
            table = make_workload("cfg2", n=8).elements[1]["table"]
            kw = dict(table=table, dt_table=0.05e-12)
        W = elgo.wake_samples(kind, nb, dt, **kw)
        gW = elg.dbg_wake_samples(kind, nb, dt, **kw)
        assert np.max(np.abs(gW - W)) <= 1e-13 * np.max(np.abs(W))
        counts = rng.integers(0, 30000, size=nb).astype(np.uint32)
        counts[rng.random(nb) < 0.3] = 0
        q = 1e-9 / 1e7
        V = elgo.convolve(counts, W, q)
        gV = elg.dbg_convolve(counts, W, q)                       # the ORACLE's W and counts
        assert np.max(np.abs(gV - V)) <= 1e-10 * np.max(np.abs(V))
        assert np.array_equal(elg.dbg_convolve(counts, W, q), gV)  # run-to-run deterministic
    # table resampled at another dt (G12)
    table = np.array([5.0, 3.0, -1.0, 0.5])
    assert elg.dbg_wake_samples(1, 8, 1.0, table=table, dt_table=2.0).tolist() == [5.0, 4.0, 3.0, 1.0, -1.0, -0.25, 0.5, 0.0]


# ------------------------------------------------------------------------------------ (v) kick
@pytest.mark.parametrize("nb,Q", [(512, 1.0), (1000, 1e4), (8192, 30.0), (70_001, 200.0)])
def test_recursive_resonator_wake(elg, elgo, nb, Q):
    """WAKE with wake = RESONATOR_REC (G37): V from the blocked O(nb) recurrence against the oracle's sequential one
    and against the direct convolution; histogram and window bit-identical, delta to 1e-12."""
    w = make_workload("cfg0", n=120_001)
    e = dict(w.elements[3]); e.update(nb=nb, Q=Q, wake="RESONATOR_REC")
    elems = w.elements[:3] + [e, {"type": "DRIFT", "L": 0.5}]
    v0 = w.particles()
    ob = elgo.Bunch(v0, w.p0c_eV, w.charge_C)
    oo = ob.track(elgo.Beamline(elems), 1, want_stage_outputs=True)
    gbl = elg.Beamline(elems); gb = elg.Bunch(v0, w.p0c_eV, w.charge_C, beamline=gbl)
    go = gb.track(gbl, 1, want_stage_outputs=True)
    assert np.array_equal(go["window"], oo["window"]) and np.array_equal(go["hist"], oo["hist"])
    m = np.max(np.abs(oo["V"]))
    assert np.max(np.abs(go["V"] - oo["V"])) <= 1e-10 * m
    W = elgo.wake_samples(0, nb, oo["window"][0, 1], f=e["f"], Q=Q, Rs=e["Rs"])
    Vd = elgo.convolve(oo["hist"], W, w.charge_C / w.n0)
    assert np.max(np.abs(go["V"] - Vd)) <= 1e-10 * m
    ov, oid = ob.read(); gv, gid = gb.read()
    assert np.array_equal(gid, oid) and np.array_equal(gv[:5], ov[:5]) and rel_err(gv, ov) <= 1e-12


def test_kick_stage(elg, elgo):
    """Protocol (v): the ORACLE's V and coordinates uploaded; elg_dbg_kick applies the kick the way tracking does
    (OP_KICK as a fused run of one op), interpolated and own-bin."""
    w = make_workload("cfg0", n=150_001)
    v = w.particles()
    b0 = elgo.beta0(w.p0c_eV); ibc = elgo.inv_bc(b0); iE = elgo.inv_E(b0, w.p0c_eV)
    nb = 512
    V = np.random.default_rng(5).normal(size=nb) * 1e5
    s = v[4].copy()
    s[:3] = [1e9, -1e9, np.nan]                                    # unbinned particles are not kicked
    t_lo, dt, inv_dt = elgo.window(v[4], ibc, elgo.WIN["AUTO_MINMAX"], nb)
    for interp in (True, False):
        d = v[5].copy()
        elgo.kick(s, d, ibc, t_lo, inv_dt, nb, V, iE, interp=interp)
        gd = elg.dbg_kick(s, v[5], w.p0c_eV, t_lo, dt, nb, V, interp=interp)
        assert np.array_equal(gd, d)                               # same V in -> bit-identical delta
        assert np.array_equal(gd[:3], v[5, :3])
    d0 = v[5].copy(); d1 = v[5].copy()
    elgo.kick(s, d0, ibc, t_lo, inv_dt, nb, V, iE, interp=False); elgo.kick(s, d1, ibc, t_lo, inv_dt, nb, V, iE, interp=True)
    assert np.max(np.abs(d0 - d1)) > 0                             # the two branches differ on this input


def test_tkick_stage(elg, elgo):
    """The transverse kick (OP_TKICK, G32 / G14) on the ORACLE's Vx, Vy and coordinates: x', y' bit-identical."""
    w = make_workload("cfg0", n=90_001)
    v = w.particles()
    b0 = elgo.beta0(w.p0c_eV); ibc = elgo.inv_bc(b0); iE = elgo.inv_E(b0, w.p0c_eV)
    nb = 300
    rng = np.random.default_rng(6)
    Vx = rng.normal(size=nb) * 1e3; Vy = rng.normal(size=nb) * 2e3
    s = v[4].copy(); s[:2] = [np.nan, 7e8]
    t_lo, dt, inv_dt = elgo.window(v[4], ibc, elgo.WIN["AUTO_MINMAX"], nb)
    for interp in (True, False):
        xp = v[1].copy(); yp = v[3].copy()
        elgo.tkick(s, xp, yp, ibc, t_lo, inv_dt, nb, Vx, Vy, iE, interp=interp)
        gxp, gyp = elg.dbg_tkick(s, v[1], v[3], w.p0c_eV, t_lo, dt, nb, Vx, Vy, interp=interp)
        assert np.array_equal(gxp, xp) and np.array_equal(gyp, yp)
        assert np.array_equal(gxp[:2], v[1, :2])


def test_compact_stage(elg, elgo):
    """Protocol (ii): the ORACLE's pre-aperture coordinates uploaded, elg_dbg_compact = predicate + stable compaction +
    lost log alone (PAPER.md:141 loss contract): survivor IDs / order, coordinates, lost records bit-exact."""
    w = make_workload("cfg0", n=333_337)
    v = w.particles()
    elgo.drift(v, 1.0)                                             # the oracle's coordinates in front of the aperture
    ids = np.arange(v.shape[1], dtype=np.int64)[::-1].copy() * 3 + 11      # arbitrary IDs travel with the particles
    for kind, ax, ay in (("RCOL", 120e-6, 90e-6), ("ECOL", 260e-6, 130e-6)):
        f = elgo.aperture_flags(v[0], v[2], elgo.RCOL if kind == "RCOL" else elgo.ECOL, ax, ay)
        h = v.copy(); hid = ids.copy()
        ns, lv, lid = elgo.compact(h, hid, f)
        gv, gid, glid, glco = elg.dbg_compact(v, kind, ax, ay, ids=ids)
        assert 0 < ns < v.shape[1]
        assert np.array_equal(gid, hid[:ns]) and np.array_equal(gv, h[:, :ns])
        assert np.array_equal(glid, lid) and np.array_equal(glco.T, lv)


# ------------------------------------------------------------------------------------ (vi) moments
@pytest.mark.parametrize("n", [1, 2, 3, 1000, 262_145])
def test_moments_stage(elg, elgo, n):
    w = make_workload("cfg0", n=n)
    v = w.particles()
    v[4] += 1.0e4                                                  # absolute path length: cancellation trap
    v[0] += 3e-4
    gb = elg.Bunch(v, w.p0c_eV, w.charge_C)
    gn, gc, gS = gb.moments()
    oc, oS = elgo.moments(v)
    assert gn == n
    sig = np.sqrt(np.diag(oS))
    assert np.all(np.abs(gc - oc) <= 1e-10 * np.maximum(np.max(np.abs(oc)), sig) + 1e-300)
    assert np.max(np.abs(gS - oS)) <= 1e-10 * np.max(np.abs(oS)) + 1e-300
    gn2, gc2, gS2 = gb.moments()
    assert np.array_equal(gc, gc2) and np.array_equal(gS, gS2)     # deterministic


# ------------------------------------------------------------------------------------ (vii) end to end
def test_cfg0_end_to_end(elg, elgo):
    w = make_workload("cfg0")
    ob, oo, gb, go = both(elg, elgo, w)
    ov, oid = ob.read(); gv, gid = gb.read()
    assert np.array_equal(gid, oid)
    assert np.array_equal(gv[:5], ov[:5])
    assert np.array_equal(go["window"], oo["window"]), "window (t_lo, dt, 1/dt) must be bit-equal"
    assert np.array_equal(go["hist"], oo["hist"])
    assert np.max(np.abs(go["V"] - oo["V"])) <= 1e-10 * np.max(np.abs(oo["V"]))
    assert rel_err(gv, ov) <= 1e-12
    nl = check_lost(ob, gb)
    assert 0.002 < nl / w.n0 < 0.012
    check_records(go, oo)


def test_cfg1_end_to_end(elg, elgo):
    """FODO line with 25 elliptical apertures, 2 RF cavities, moments after each element (77 records)."""
    w = make_workload("cfg1", n=200_000)
    ob, oo, gb, go = both(elg, elgo, w)
    ov, oid = ob.read(); gv, gid = gb.read()
    assert np.array_equal(gid, oid)
    assert np.array_equal(gv[:5], ov[:5])
    assert rel_err(gv, ov) <= 1e-12
    check_lost(ob, gb)
    assert go["records"].shape == (77, 43)
    check_records(go, oo)


def test_cfg2_end_to_end(elg, elgo):
    """10 passes of drift + tabulated wake, 8192 bins (bunch in ~267 of them), interpolated kick."""
    w = make_workload("cfg2", n=400_000)
    ob, oo, gb, go = both(elg, elgo, w)
    ov, oid = ob.read(); gv, gid = gb.read()
    assert np.array_equal(gv[:5], ov[:5])
    assert np.array_equal(go["window"], oo["window"])
    assert np.array_equal(go["hist"], oo["hist"])
    assert go["hist"].size == 10 * 8192 and int(go["hist"][:8192].sum()) == w.n0
    for t in range(10):
        Vo = oo["V"][t * 8192:(t + 1) * 8192]; Vg = go["V"][t * 8192:(t + 1) * 8192]
        assert np.max(np.abs(Vg - Vo)) <= 1e-10 * np.max(np.abs(Vo))
    assert rel_err(gv, ov) <= 1e-10         # 10 kicks, each good to 1e-10 of the maximum kick


def test_cfg3_100_turns(elg, elgo):
    """Ring: 200 matrices + RF + resonator wake per turn, 100 turns, moments every turn (<= 1e-9)."""
    w = make_workload("cfg3", n=20_000)
    ob, oo, gb, go = both(elg, elgo, w)
    ov, oid = ob.read(); gv, gid = gb.read()
    assert np.array_equal(gv[:5], ov[:5])                          # x, x', y, y', s never see delta here
    assert np.array_equal(go["hist"], oo["hist"])
    assert rel_err(gv, ov) <= 1e-9
    assert go["records"].shape == (100, 43)
    check_records(go, oo)
    Vo = oo["V"].reshape(100, 1024); Vg = go["V"].reshape(100, 1024)
    assert np.max(np.abs(Vg - Vo) / np.max(np.abs(Vo), axis=1, keepdims=True)) <= 1e-10


def test_cfg3_literal_5_turns(elg, elgo):
    w = make_workload("cfg3-literal", n=20_000)
    ob, oo, gb, go = both(elg, elgo, w)
    ov, _ = ob.read(); gv, _ = gb.read()
    assert np.array_equal(gv[:5], ov[:5])
    assert rel_err(gv, ov) <= 1e-11
    check_records(go, oo)


def test_cfg4_end_to_end(elg, elgo):
    """Loss-heavy collimation: 20 RCOL + 65536-bin histograms in ~50 bins; everything bit-exact."""
    w = make_workload("cfg4", n=1_000_003)
    ob, oo, gb, go = both(elg, elgo, w)
    ov, oid = ob.read(); gv, gid = gb.read()
    assert np.array_equal(gid, oid) and np.array_equal(gv, ov)
    assert np.array_equal(go["window"], oo["window"])
    assert np.array_equal(go["hist"], oo["hist"])
    nl = check_lost(ob, gb)
    assert nl + gid.size == w.n0 and nl / w.n0 > 0.9


@pytest.mark.parametrize("n", [1, 2, 1000, 300_007])
def test_trwake_end_to_end(elg, elgo, n):
    """TRWAKE (G32-G34): counts bit-identical, dipole sums and Vx / Vy to 1e-10 of their maximum, coordinates to 1e-12
    (the transverse kicks feed x, y and s through the following drifts)."""
    w = make_workload("p5-trwake", n=n)
    ob, oo, gb, go = both(elg, elgo, w)
    nb1, nb2 = w.elements[2]["nb"], w.elements[4]["nb"]
    assert np.array_equal(go["window"][0], oo["window"][0])
    assert np.array_equal(go["hist"][:nb1], oo["hist"][:nb1])
    Vo, Vg = oo["V"], go["V"]
    assert Vg.size == Vo.size == 4 * nb1 + 4 * nb2 + w.elements[5]["nb"]
    for lo, hi in ((0, nb1), (nb1, 2 * nb1)):                      # dipole sums of the first TRWAKE (G33)
        assert np.max(np.abs(Vg[lo:hi] - Vo[lo:hi])) <= 1e-10 * np.max(np.abs(Vo[lo:hi])) + 1e-300
    for lo, hi in ((2 * nb1, 3 * nb1), (3 * nb1, 4 * nb1)):
        m = np.max(np.abs(Vo[lo:hi]))
        assert np.max(np.abs(Vg[lo:hi] - Vo[lo:hi])) <= 1e-10 * m + 1e-300
    if n > 2:
        assert np.max(np.abs(Vo[2 * nb1:3 * nb1])) > 0
    # later stages see coordinates that agree to ~1e-15 only: relative to their maximum
    o2 = 4 * nb1
    for k in range(4):
        a, b_ = Vg[o2 + k * nb2: o2 + (k + 1) * nb2], Vo[o2 + k * nb2: o2 + (k + 1) * nb2]
        assert np.max(np.abs(a - b_)) <= 1e-9 * np.max(np.abs(b_)) + 1e-300
    assert int(go["hist"][nb1:nb1 + nb2].sum()) == int(oo["hist"][nb1:nb1 + nb2].sum())
    ov, oid = ob.read(); gv, gid = gb.read()
    assert np.array_equal(gid, oid)
    if n > 2:
        assert rel_err(gv, ov) <= 1e-12


def test_trwake_run_to_run_deterministic(elg):
    """Integer atomics: two runs give the same bits (a sum of doubles accumulated with atomics would not)."""
    w = make_workload("p5-trwake", n=200_003)
    v0 = w.particles()
    outs = []
    for _ in range(2):
        bl = elg.Beamline(w.elements)
        b = elg.Bunch(v0, w.p0c_eV, w.charge_C, beamline=bl)
        o = b.track(bl, 1, want_stage_outputs=True)
        outs.append((b.read()[0], o["V"], o["hist"]))
    for a, b_ in zip(outs[0], outs[1]):
        assert np.array_equal(a, b_)


@pytest.mark.parametrize("n", [3, 70_001])
def test_rfcw_composite(elg, elgo, n):
    """RFKICK + WAKE + TRWAKE per cavity with shared binning (one histogram pass on the CUDA side, two on the
    oracle's): identical windows, counts and dipole sums at the first cavity, V to 1e-10, coordinates to 1e-12."""
    w = make_workload("p6-rfcw", n=n, n_cavities=4)
    ob, oo, gb, go = both(elg, elgo, w)
    nb = 512
    assert go["hist"].size == oo["hist"].size == 8 * nb and go["window"].shape == oo["window"].shape == (8, 3)
    assert np.array_equal(go["window"][:2], oo["window"][:2]) and np.array_equal(go["window"][0], go["window"][1])
    assert np.array_equal(go["hist"][:2 * nb], oo["hist"][:2 * nb])
    assert np.array_equal(go["hist"][:nb], go["hist"][nb:2 * nb])
    Vo, Vg = oo["V"], go["V"]
    assert Vg.size == Vo.size == 4 * 5 * nb
    for lo, hi in ((nb, 2 * nb), (2 * nb, 3 * nb)):                 # dipole sums of the first cavity (G33)
        assert np.max(np.abs(Vg[lo:hi] - Vo[lo:hi])) <= 1e-10 * np.max(np.abs(Vo[lo:hi])) + 1e-300
    for c in range(4):
        for lo, hi in ((0, nb), (3 * nb, 4 * nb), (4 * nb, 5 * nb)):
            a = Vg[5 * nb * c + lo: 5 * nb * c + hi]; r = Vo[5 * nb * c + lo: 5 * nb * c + hi]
            assert np.max(np.abs(a - r)) <= (1e-10 if c == 0 else 1e-9) * np.max(np.abs(r)) + 1e-300
        assert int(go["hist"][2 * nb * c: 2 * nb * c + nb].sum()) == n
    ov, oid = ob.read(); gv, gid = gb.read()
    assert np.array_equal(gid, oid) and rel_err(gv, ov) <= 1e-12


@pytest.mark.parametrize("name,n,chunks", [("cfg3", 100_003, 5), ("cfg0", 50_001, 3), ("p6-rfcw", 40_000, 4), ("cfg2", 30_000, 7)])
def test_upload_and_track_equals_upload_then_track(elg, name, n, chunks):
    """elg_upload_and_track (upload pipelined against the leading maps, chunk by chunk) gives the same bits as
    elg_bunch_upload + elg_track: coordinates, IDs, lost log, records, stage outputs."""
    kw = {"n_turns": 3} if name == "cfg3" else {}
    w = make_workload(name, n=n, **kw)
    v0 = w.particles()
    nt = min(w.n_turns, 3)
    bl = elg.Beamline(w.elements, ring=w.ring)
    a = elg.Bunch(v0, w.p0c_eV, w.charge_C, beamline=bl)
    oa = a.track(bl, nt, moments_every=w.moments_every, want_stage_outputs=True)
    b = elg.Bunch(None, w.p0c_eV, w.charge_C, beamline=bl, n0=n)
    ob = b.upload_and_track(v0, bl, nt, moments_every=w.moments_every, want_stage_outputs=True, n_chunks=chunks)
    av, aid = a.read(); bv, bid = b.read()
    assert np.array_equal(aid, bid) and np.array_equal(av, bv)
    for k in ("hist", "V", "window"):
        assert np.array_equal(oa[k], ob[k]), k
    if "records" in oa:
        assert np.array_equal(oa["records"], ob["records"])
    for x, y in zip(a.lost(), b.lost()):
        assert np.array_equal(x, y)
    # and once more on the same bunch (copy stream and events are reused)
    ob2 = b.upload_and_track(v0, bl, nt, moments_every=w.moments_every, want_stage_outputs=True, n_chunks=chunks)
    assert np.array_equal(b.read()[0], av) and np.array_equal(ob2["V"], oa["V"])


def test_more_records_than_the_device_ring(elg, elgo):
    """3 000 per-element records in one call: the 2 048-record device ring is drained to the host mid-run."""
    ring = _long_line(23, {})[:6]
    v0 = make_workload("cfg0", n=3001).particles()
    ob = elgo.Bunch(v0, 1e9, 1e-9)
    oo = ob.track(elgo.Beamline(ring, ring=True), 500, moments_every="element")
    gbl = elg.Beamline(ring, ring=True); gb = elg.Bunch(v0, 1e9, 1e-9, beamline=gbl)
    go = gb.track(gbl, 500, moments_every="element")
    assert go["records"].shape == oo["records"].shape == (3000, 43)
    check_records(go, oo)
    assert np.array_equal(gb.read()[0], ob.read()[0])


def test_empty_bunch_and_everything_lost(elg, elgo):
    """G28: n = 0 from the start, and a bunch that loses every particle half way: later elements are no-ops,
    histograms are zero, moment records are zero, elg_moments reports ELG_ESTATE."""
    w = make_workload("cfg0", n=2000)
    elems = [w.elements[0], {"type": "RCOL", "ax": 1e-9, "ay": 1e-9}] + w.elements[1:]
    for v0 in (w.particles(), np.zeros((6, 0))):
        ob = elgo.Bunch(v0, w.p0c_eV, w.charge_C)
        oo = ob.track(elgo.Beamline(elems), 1, moments_every="turn", want_stage_outputs=True)
        gbl = elg.Beamline(elems); gb = elg.Bunch(v0, w.p0c_eV, w.charge_C, beamline=gbl)
        go = gb.track(gbl, 1, moments_every="turn", want_stage_outputs=True)
        assert gb.n_alive == ob.n_alive == 0
        assert np.array_equal(go["hist"], oo["hist"]) and not go["hist"].any()
        assert np.array_equal(go["records"], oo["records"]) and not go["records"].any()
        check_lost(ob, gb)
        with pytest.raises(elg.ElgError) as ei:
            gb.moments()
        assert ei.value.code == elg.ESTATE


def test_sparse_matrix_option_equals_dense(elg, elgo):
    """ELG_TRACK_SPARSE_MATRICES (flagged option, reported separately): matrices with the zero pattern of an uncoupled
    element take 20 FMAs instead of 36; results equal the dense ones (and hence the oracle's) on finite coordinates.
    Covers long runs (pattern kernel), a coupled matrix inside the run (stays dense), and short runs (fall back)."""
    w = make_workload("cfg3", n=60_001, n_turns=3)
    v0 = w.particles()
    rng = np.random.default_rng(8)
    coupled = {"type": "MATRIX", "R": np.eye(6) + 1e-3 * rng.normal(size=(6, 6)), "C": np.zeros(6)}
    lines = {"ring": (w.elements, True, 3), "mixed": (w.elements[:30] + [coupled] + w.elements[30:60], False, 1),
             "short": (w.elements[:3] + [{"type": "RCOL", "ax": 1e-3, "ay": 1e-3}] + w.elements[3:6], False, 1)}
    for name, (elems, ring, nt) in lines.items():
        outs = []
        for sparse in (False, True):
            bl = elg.Beamline(elems, ring=ring)
            b = elg.Bunch(v0, w.p0c_eV, w.charge_C, beamline=bl)
            b.sparse_matrices = sparse
            o = b.track(bl, nt, moments_every="turn" if ring else "none")
            outs.append((b.read(), o))
        (dv, did), _ = outs[0]; (sv, sid), _ = outs[1]
        assert np.array_equal(did, sid) and np.array_equal(dv, sv), name
        if name == "ring":
            ob = elgo.Bunch(v0, w.p0c_eV, w.charge_C); ob.track(elgo.Beamline(elems, ring=True), 3)
            assert np.array_equal(sv[:5], ob.read()[0][:5])
            check_records(outs[1][1], outs[0][1])


def test_track_in_two_calls_equals_one(elg, elgo):
    """Turn counter, RF reference and lost log carry across elg_track calls."""
    w = make_workload("cfg3", n=5000, n_matrices=10, n_turns=6)
    v0 = w.particles()
    bl = elg.Beamline(w.elements, ring=True)
    a = elg.Bunch(v0, w.p0c_eV, w.charge_C, beamline=bl); a.track(bl, 6)
    b = elg.Bunch(v0, w.p0c_eV, w.charge_C, beamline=bl); b.track(bl, 2); b.track(bl, 4)
    assert np.array_equal(a.read()[0], b.read()[0])
    ob = elgo.Bunch(v0, w.p0c_eV, w.charge_C); ob.track(elgo.Beamline(w.elements, ring=True), 6)
    assert rel_err(a.read()[0], ob.read()[0]) <= 1e-11
    # rewind + re-upload gives the same answer again (workspace reuse)
    a.upload(v0); a.track(bl, 6)
    assert np.array_equal(a.read()[0], b.read()[0])


def test_profile_reports_algorithmic_work(elg):
    """elg_profile_read's bytes / flops (what bench.py's roofline uses): coordinates read + written x live particles of
    every launch, counted on the device.  DRIFT + MATRIX reads 6 and writes 6 coordinates (96 B); a compacting run
    moves all seven arrays (112 B); 10 matrices are 720 flop per particle; lossy lines use the live count of each launch."""
    n = 300_001
    w = make_workload("p1-chain", n=n)
    v0 = w.particles()
    bl = elg.Beamline(w.elements); b = elg.Bunch(v0, w.p0c_eV, w.charge_C, beamline=bl)
    b.profile(True); b.profile_read()
    b.track(bl, 1)
    p = b.profile_read(work=True)
    assert p["chain"][0] == 1 and p["chain"][2] == 96.0 * n and p["chain"][3] == (11 + 72) * n
    b.upload(v0)                                           # rewinds: the counters survive a rewind
    b.track(bl, 1); b.upload(v0); b.track(bl, 1)
    p = b.profile_read(work=True)
    assert p["chain"][0] == 2 and p["chain"][2] == 2 * 96.0 * n
    w2 = make_workload("cfg4", n=n)
    bl2 = elg.Beamline(w2.elements); b2 = elg.Bunch(w2.particles(), w2.p0c_eV, w2.charge_C, beamline=bl2)
    b2.profile(True); b2.profile_read()
    b2.track(bl2, 1)
    p2 = b2.profile_read(work=True)
    _, _, elem, _ = b2.lost()
    n_in = n - np.array([(elem < 3 * i).sum() for i in range(20)])          # live count entering collimator i
    assert p2["chain_compact"][0] == 20 and p2["chain_compact"][2] == 112.0 * n_in.sum()
    n_hist = n - np.array([(elem <= 3 * i).sum() for i in range(20)])
    assert p2["hist"][0] == 20 and p2["hist"][2] == 8.0 * n_hist.sum()
    w3 = make_workload("p3-matrices", n=n, n_matrices=10)
    bl3 = elg.Beamline(w3.elements, ring=True); b3 = elg.Bunch(w3.particles(), w3.p0c_eV, w3.charge_C, beamline=bl3)
    b3.profile(True); b3.profile_read()
    b3.track(bl3, 2)                                       # the planner fuses the two turns into one 20-matrix run
    p3 = b3.profile_read(work=True)
    assert p3["chain_long"][0] == 1 and p3["chain_long"][3] == 2 * 720.0 * n and p3["chain_long"][2] == 96.0 * n
    b3.profile(False)
    b3.track(bl3, 1)
    assert b3.profile_read(work=True)["chain_long"] == (0, 0.0, 0.0, 0.0)   # nothing is counted while profiling is off


def test_fp64_peak_hook(elg):
    """elg_dbg_fp64_peak (the measured denominator of the fp64 roofline): a DFMA-only kernel must land near the nominal
    148 SMs x 64 DFMA/clk x 2 x clock."""
    tf, ms = elg.dbg_fp64_peak(5000)
    assert ms > 0 and 25.0 < tf < 45.0


# ------------------------------------------------------------------------------------ launch options change no bit
_SWITCH_SCRIPT = r"""
import hashlib, sys
import numpy as np
sys.path.insert(0, {root!r})
from elg_inputs import make_workload
from paper_1710_07350_b200 import elg
h = hashlib.sha256()
for name, n, turns in (("cfg4", 300_007, 1), ("cfg0", 100_000, 1), ("cfg2", 200_003, 3), ("p6-rfcw", 150_001, 1), ("cfg1", 120_011, 1)):
    w = make_workload(name, n=n)
    bl = elg.Beamline(w.elements, ring=w.ring)
    for rep in range(3):                                  # repeated: a launch-order race would not hit every time
        b = elg.Bunch(w.particles(), w.p0c_eV, w.charge_C, beamline=bl, lost_capacity=n)
        o = b.track(bl, turns, moments_every=w.moments_every, want_stage_outputs=True)
        v, ids = b.read()
        lost = b.lost()
        for arr in (v, ids, o["hist"], o["V"], o["window"], o.get("records", np.zeros(0)), lost[0], lost[3]):
            h.update(np.ascontiguousarray(arr).tobytes())
print(h.hexdigest())
"""


@pytest.mark.gpu
def test_launch_switches_change_no_bit(elg):
    """Programmatic dependent launch (every kernel starts with griddepcontrol.wait) and the bulk-copy ring of the short
    runs are launch mechanics: coordinates, IDs, histograms, voltages, windows, records and the lost log of five
    workloads (61-launch cfg4, the compacting runs of cfg0 / cfg1 with records, multi-turn cfg2, RFCW cavities) must be
    bit-identical with each of them switched off (ELG_PDL=0, ELG_CHAIN_RING=0), run three times each."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    script = _SWITCH_SCRIPT.format(root=root)
    digests = {}
    for tag, env in (("default", {}), ("no-pdl", {"ELG_PDL": "0"}), ("no-ring", {"ELG_CHAIN_RING": "0"})):
        e = dict(os.environ); e.update(env)
        out = subprocess.run([sys.executable, "-c", script], env=e, capture_output=True, text=True, check=True, timeout=600)
        digests[tag] = out.stdout.strip().splitlines()[-1]
    assert len(digests["default"]) == 64
    assert digests["no-pdl"] == digests["default"] and digests["no-ring"] == digests["default"], digests


# ------------------------------------------------------------------------------------ the roofline's numerator
@pytest.mark.gpu
def test_work_accounting_matches_the_algorithmic_counts(elg):
    """bench.py's roofline divides the ALGORITHMIC bytes / flops the launches report (elg_profile_read) by their device
    time.  The reported work must be DESIGN.md section 5's per-particle figures times the live particles of each launch:
    96 B and 11 + 72 flops for DRIFT + MATRIX, 112 B for a compacting run (live count BEFORE the aperture), 8 B per
    histogram, 24 B for a wake kick (+ the record's coordinates), 72 flops per matrix of a long run."""
    n = 100_003
    # p1: DRIFT + MATRIX, one launch
    w = make_workload("p1-chain", n=n)
    bl = elg.Beamline(w.elements); b = elg.Bunch(w.particles(), w.p0c_eV, w.charge_C, beamline=bl)
    b.profile(True); b.profile_read()
    b.track(bl, 1, moments_every="none", records=False)
    p = b.profile_read(work=True)
    assert p["chain"][0] == 1 and p["chain"][2] == 96.0 * n and p["chain"][3] == (11 + 72) * float(n)
    assert sum(v[0] for k, v in p.items() if k != "chain") == 0
    # cfg0 with the turn record: compacting run (112 B x n0), histogram (8 B x survivors), kick + record (56 B x survivors)
    w = make_workload("cfg0", n=n)
    bl = elg.Beamline(w.elements); b = elg.Bunch(w.particles(), w.p0c_eV, w.charge_C, beamline=bl, lost_capacity=n)
    b.profile(True); b.profile_read()
    b.track(bl, 1, moments_every="turn", records=False)
    p = b.profile_read(work=True)
    alive = b.n_alive
    assert 0 < alive < n
    assert p["chain_compact"][0] == 1 and p["chain_compact"][2] == 112.0 * n and p["chain_compact"][3] == (11 + 72) * float(n)
    assert p["hist"][0] == 1 and p["hist"][2] == 8.0 * alive
    assert p["chain"][0] == 1 and p["chain"][2] == 56.0 * alive and p["chain"][3] == (10 + 60) * float(alive)
    assert p["moments"][0] == 0                                        # the record rode in the kick run's epilogue
    # cfg3, one turn: 200 matrices + RF kick in three long-run launches
    w = make_workload("cfg3", n=n, n_turns=1)
    bl = elg.Beamline(w.elements, ring=True); b = elg.Bunch(w.particles(), w.p0c_eV, w.charge_C, beamline=bl)
    b.profile(True); b.profile_read()
    b.track(bl, 1, moments_every="turn", records=False)
    p = b.profile_read(work=True)
    assert p["chain_long"][0] == 3 and p["chain_long"][2] == 3 * 96.0 * n and p["chain_long"][3] == (200 * 72 + 6) * float(n)
    assert p["chain"][0] == 1 and p["chain"][2] == 56.0 * n
    b.profile(False)


# ------------------------------------------------------------------------------------ CUDA-graph replay of elg_track
@pytest.mark.gpu
@pytest.mark.parametrize("name,n,turns", [("cfg0", 100_000, 1), ("cfg4", 200_003, 1), ("cfg1", 150_001, 1), ("p6-rfcw", 120_007, 1),
                                         ("cfg2", 150_000, 3), ("cfg3", 30_011, 2)])
def test_cuda_graph_replay_equals_direct_tracking(elg, name, n, turns):
    """[copy of fresh particles, rewind, elg_track] captured into a CUDA graph on the bunch's own stream (cooperative
    compaction launches and the programmatic-dependent-launch attribute included) and replayed three times gives, bit
    for bit, the coordinates, IDs, lost log and moments of a direct call -- whatever the parity of the compactions
    (the host mirror of the device state is restored after each replay, include/elg.h "CUDA graphs")."""
    import torch
    kw = {"n_turns": turns} if name == "cfg3" else {}
    w = make_workload(name, n=n, **kw)
    v0 = w.particles()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        bl = elg.Beamline(w.elements, ring=w.ring)
        b = elg.Bunch(v0, w.p0c_eV, w.charge_C, beamline=bl, lost_capacity=n, stream=s)
        keep = b.soa.clone()
        b.track(bl, turns, moments_every=w.moments_every, records=False)      # direct (also uploads the wake tables)
        rv, rid = b.read(); rlost = b.lost(); rmom = b.moments() if rv.shape[1] else None
        g = b.capture_track(bl, turns, moments_every=w.moments_every, prologue=lambda: b.soa.copy_(keep))
        for rep in range(3):
            if rep == 1:
                b.rewind()                                            # host state knocked out of step on purpose
            g.replay()
            gv, gid = b.read(); glost = b.lost()
            assert np.array_equal(gid, rid) and np.array_equal(gv, rv)
            for x, y in zip(glost, rlost):
                assert np.array_equal(x, y)
            if rmom is not None:
                gm = b.moments()
                assert gm[0] == rmom[0] and np.array_equal(gm[1], rmom[1]) and np.array_equal(gm[2], rmom[2])
        # a direct call afterwards continues from the replayed state like from a direct one
        b.soa.copy_(keep); b.rewind()
        b.track(bl, turns, moments_every=w.moments_every, records=False)
        assert np.array_equal(b.read()[0], rv)

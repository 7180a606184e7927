"""elg_dipole_histogram_noalloc (include/elg.h, "an entry point that allocates nothing"): the dipole histogram stage with
its scratch in a file-scope device array of the library instead of a caller-lent workspace.  Checked against the
existing path (elg_dbg_dipole_histogram: tracking's planner, window kernel, dipole_hist_kernel, finalize) on calls in a
row that share the static scratch.  This file is collected last on purpose (the suite runs with pytest -x)."""
import math

import numpy as np
import pytest

from elg_inputs import make_workload

pytestmark = pytest.mark.gpu


def _inv_bc(p0c_eV, mc2_eV):
    # the same fp64 operations, in the same order, as elg_bunch_create (G7, G9): identical bits
    e2 = p0c_eV * p0c_eV + mc2_eV * mc2_eV
    beta0 = p0c_eV / math.sqrt(e2)
    return 1.0 / (beta0 * 299792458.0)


def _case(n, seed_shift, nb, offset):
    w = make_workload("p5-trwake", n=n)
    v = w.particles()
    rng = np.random.default_rng(100 + seed_shift)
    v[0] = v[0] * rng.uniform(0.5, 2.0) + offset[0]
    v[2] = v[2] * rng.uniform(0.5, 2.0) + offset[1]
    s = v[4]
    dt = (s.max() - s.min()) / 299792458.0 / (nb - 3)               # a few particles fall outside the window on purpose
    t_lo = s.min() / 299792458.0 + 1.5 * dt
    return w, v, t_lo, dt


def test_no_alloc_entry_matches_the_existing_path_on_calls_in_a_row():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1710_07350_b200 import elg
    dev = torch.device("cuda:0")
    assert elg.noalloc_max_bins() == 16384
    # three calls in a row on the same static scratch: large histogram, then a SMALLER one with other particles (stale
    # accumulators or counts of the first call would show), then the first again
    cases = [(250_003, 0, 4001, (2e-4, -1e-4)), (70_001, 1, 777, (-3e-4, 5e-5)), (250_003, 0, 4001, (2e-4, -1e-4))]
    free_before = None
    results = []
    for k, (n, shift, nb, off) in enumerate(cases):
        w, v, t_lo, dt = _case(n, shift, nb, off)
        ref_c, ref_dx, ref_dy = elg.dbg_dipole_histogram(v[4], v[0], v[2], w.p0c_eV, t_lo, dt, nb)       # existing path
        d_s = torch.as_tensor(v[4], device=dev); d_x = torch.as_tensor(v[0], device=dev); d_y = torch.as_tensor(v[2], device=dev)
        d_c = torch.full((nb,), 12345, dtype=torch.int32, device=dev)                # garbage: the call must overwrite
        d_D = torch.full((2 * nb,), float("nan"), dtype=torch.float64, device=dev)
        torch.cuda.synchronize(dev)
        if k > 0:
            free_before = torch.cuda.mem_get_info(dev)[0]
        elg.dipole_histogram_noalloc(d_s, d_x, d_y, _inv_bc(w.p0c_eV, elg.ELECTRON_MC2_EV), t_lo, dt, nb, d_c, d_D)
        torch.cuda.synchronize(dev)
        if k > 0:
            assert torch.cuda.mem_get_info(dev)[0] == free_before, "the call changed the free device memory"
        got_c = d_c.cpu().numpy().view(np.uint32)
        got_D = d_D.cpu().numpy()
        assert 0 < int(ref_c.sum()) < n                                               # some particles outside the window
        assert np.array_equal(got_c, ref_c)                                           # integer work: bit-exact
        for got, ref in ((got_D[:nb], ref_dx), (got_D[nb:], ref_dy)):
            assert np.max(np.abs(got - ref)) <= 1e-10 * np.max(np.abs(ref))          # north_star's tolerance for sums
            assert np.array_equal(got, ref)                                           # in fact the same integers: same bits
        results.append((got_c, got_D))
    assert np.array_equal(results[0][0], results[2][0]) and np.array_equal(results[0][1], results[2][1])


def test_no_alloc_entry_rejects_sizes_beyond_the_static_scratch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1710_07350_b200 import elg
    dev = torch.device("cuda:0")
    nb = elg.noalloc_max_bins() + 1
    d = torch.zeros(64, dtype=torch.float64, device=dev)
    d_c = torch.zeros(nb, dtype=torch.int32, device=dev)
    d_D = torch.zeros(2 * nb, dtype=torch.float64, device=dev)
    with pytest.raises(elg.ElgError) as ei:
        elg.dipole_histogram_noalloc(d, d, d, 3.3e-9, 0.0, 1e-12, nb, d_c, d_D)
    assert ei.value.code == elg.ECAPACITY and "16384" in str(ei.value)
    # the largest allowed size works (bins beyond the shared-memory range take the global atomics)
    nb = elg.noalloc_max_bins()
    s = torch.linspace(0.0, 1.0, 50_000, dtype=torch.float64, device=dev)
    x = torch.full_like(s, 1e-4); y = torch.full_like(s, -2e-4)
    d_c = torch.zeros(nb, dtype=torch.int32, device=dev); d_D = torch.zeros(2 * nb, dtype=torch.float64, device=dev)
    elg.dipole_histogram_noalloc(s, x, y, 1.0, -1e-9, (1.0 + 2e-9) / nb, nb, d_c, d_D)
    torch.cuda.synchronize(dev)
    c = d_c.cpu().numpy().astype(np.int64); D = d_D.cpu().numpy()
    assert c.sum() == 50_000
    assert np.max(np.abs(D[:nb] - 1e-4 * c)) <= 1e-10 * np.max(np.abs(D[:nb]))
    assert np.max(np.abs(D[nb:] + 2e-4 * c)) <= 1e-10 * np.max(np.abs(D[nb:]))

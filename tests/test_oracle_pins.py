"""Pins of the CPU oracle (oracle/elgo.cpp) against what the paper and the mathematics fix.

None of these tests calls the CUDA path.  Each pin is independent of the oracle's own code:
values printed in / derivable by hand from the paper (tests/golden/), closed forms, invariants,
brute force on tiny inputs, library routines (numpy) on special cases.  A plausible mistake in the
oracle (dropped term, wrong sign or index, transposed operand) fails at least one of them.
Citations: PAPER.md:NN = line of /root/reference/PAPER.md; Gk = readings in DESIGN.md.
"""
import math
import os

import numpy as np
import pytest

from elg_inputs import (C_LIGHT, ELECTRON_MC2_EV, compose, drift_matrix, make_workload,
                        thin_quad_matrix)

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _J():
    J = np.zeros((6, 6))
    for k in range(3):
        J[2 * k, 2 * k + 1] = 1.0
        J[2 * k + 1, 2 * k] = -1.0
    return J


# ------------------------------------------------------------------------------------ DRIFT
def test_drift_golden_listing1(elgo):
    """PAPER.md:68-79 (Listing 1): hand-computed exact cases."""
    rows = np.loadtxt(os.path.join(GOLD, "drift_listing1.txt"))
    assert rows.shape[1] == 9 and rows.shape[0] >= 6
    for L, x, xp, y, yp, s, xo, yo, so in rows:
        v = np.array([[x], [xp], [y], [yp], [s], [0.123]])
        elgo.drift(v, L)
        assert v[0, 0] == xo and v[2, 0] == yo and v[4, 0] == so
        assert v[1, 0] == xp and v[3, 0] == yp and v[5, 0] == 0.123     # untouched coordinates


def test_drift_matches_literal_listing(elgo):
    """Listing 1 evaluated literally (unfused, left to right) in numpy agrees to 1 ulp-level (G2)."""
    rng = np.random.default_rng(1)
    v = rng.normal(size=(6, 1000)) * np.array([[1e-4, 1e-3, 1e-4, 1e-3, 1.0, 1e-3]]).T
    w = v.copy()
    L = 1.7
    elgo.drift(w, L)
    x = v[0] + v[1] * L
    y = v[2] + v[3] * L
    s = v[4] + L * np.sqrt(1 + v[1] ** 2 + v[3] ** 2)
    assert np.max(np.abs(w[0] - x)) <= 2e-16 * np.max(np.abs(x)) + 1e-20
    assert np.max(np.abs(w[2] - y)) <= 2e-16 * np.max(np.abs(y)) + 1e-20
    assert np.max(np.abs(w[4] - s)) <= 4e-16 * np.max(np.abs(s))
    # zero-length drift is the identity, bitwise
    z = v.copy()
    elgo.drift(z, 0.0)
    assert np.array_equal(z, v)


# ------------------------------------------------------------------------------------ MATRIX
def test_matrix_identity_bitwise_and_closed_forms(elgo):
    rng = np.random.default_rng(2)
    v0 = rng.normal(size=(6, 257))
    v = v0.copy()
    elgo.matrix(v, np.eye(6), None)
    assert np.array_equal(v, v0)
    # D(L): x += L x', y += L y', s += L (C5 = L); everything else unchanged (G3)
    L = 0.75
    R, Cv = drift_matrix(L)
    v = v0.copy()
    elgo.matrix(v, R, Cv)
    np.testing.assert_allclose(v[0], v0[0] + L * v0[1], rtol=0, atol=1e-15)
    np.testing.assert_allclose(v[2], v0[2] + L * v0[3], rtol=0, atol=1e-15)
    np.testing.assert_allclose(v[4], v0[4] + L, rtol=0, atol=1e-15)
    for c in (1, 3, 5):
        assert np.array_equal(v[c], v0[c])
    # Q(k): x' -= k x, y' += k y (G5)
    k = 0.5
    R, Cv = thin_quad_matrix(k)
    v = v0.copy()
    elgo.matrix(v, R, Cv)
    np.testing.assert_allclose(v[1], v0[1] - k * v0[0], rtol=0, atol=1e-15)
    np.testing.assert_allclose(v[3], v0[3] + k * v0[2], rtol=0, atol=1e-15)
    for c in (0, 2, 4, 5):
        assert np.array_equal(v[c], v0[c])


def test_matrix_is_not_transposed_and_uses_C(elgo):
    """A matrix with a single off-diagonal entry moves exactly one coordinate (index pin)."""
    for r in range(6):
        for c in range(6):
            if r == c:
                continue
            R = np.eye(6)
            R[r, c] = 2.0
            Cv = np.arange(6, dtype=float) * 0.5
            v0 = np.arange(1.0, 7.0).reshape(6, 1)
            v = v0.copy()
            elgo.matrix(v, R, Cv)
            exp = v0[:, 0] + Cv
            exp[r] += 2.0 * v0[c, 0]
            assert np.array_equal(v[:, 0], exp), (r, c)


def test_cfg0_matrix_closed_form_G4(elgo):
    """G4: M = Q(k) D(L): [[1, L], [-k, 1-kL]] in x and [[1, L], [k, 1+kL]] in y."""
    w = make_workload("cfg0")
    R = w.elements[1]["R"]
    L, k = 0.5, 0.5
    assert np.allclose(R[0:2, 0:2], [[1, L], [-k, 1 - k * L]], rtol=0, atol=1e-16)
    assert np.allclose(R[2:4, 2:4], [[1, L], [k, 1 + k * L]], rtol=0, atol=1e-16)
    assert w.elements[1]["C"][4] == L


def test_generated_matrices_symplectic(elgo):
    """north_star: M^T J M = J and det = 1 for every generated matrix (all workloads)."""
    J = _J()
    count = 0
    for name in ("cfg0", "cfg1", "cfg3", "cfg3-literal"):
        w = make_workload(name, n=16)
        for e in w.elements:
            if e["type"] != "MATRIX":
                continue
            M = e["R"]
            err = np.max(np.abs(M.T @ J @ M - J))
            assert err <= 1e-15 * max(1.0, np.max(np.abs(M))) ** 2, (name, err)
            assert abs(np.linalg.det(M) - 1.0) < 1e-13
            count += 1
    assert count > 400


def test_matrix_inverse_roundtrip_and_sigma_transport(elgo):
    """M then M^-1 = -J M^T J returns the input; Sigma_out = R Sigma_in R^T; emittance invariant."""
    J = _J()
    R, Cv = compose(drift_matrix(0.5), thin_quad_matrix(0.5), drift_matrix(1.3), thin_quad_matrix(-0.7))
    Rinv = -J @ R.T @ J
    rng = np.random.default_rng(3)
    v0 = rng.normal(size=(6, 20000)) * np.array([[1e-4, 1e-5, 1e-4, 1e-5, 1e-3, 1e-3]]).T
    v = v0.copy()
    elgo.matrix(v, R, None)
    _, S1 = elgo.moments(v)
    _, S0 = elgo.moments(v0)
    assert np.max(np.abs(S1 - R @ S0 @ R.T)) <= 1e-12 * np.max(np.abs(S1))
    for a in (0, 2):
        e0 = math.sqrt(np.linalg.det(S0[a:a + 2, a:a + 2]))
        e1 = math.sqrt(np.linalg.det(S1[a:a + 2, a:a + 2]))
        assert abs(e1 - e0) <= 1e-10 * e0
    elgo.matrix(v, Rinv, None)
    scale = np.max(np.abs(v0), axis=1, keepdims=True)
    assert np.max(np.abs(v - v0) / scale) <= 1e-14


# ------------------------------------------------------------------------------------ RFKICK
def test_rfkick_closed_forms(elgo):
    p0c = 1e9
    b0 = elgo.beta0(p0c)
    ibc, iE = elgo.inv_bc(b0), elgo.inv_E(b0, p0c)
    assert abs(b0 - p0c / math.hypot(p0c, ELECTRON_MC2_EV)) < 1e-16
    assert abs(ibc * b0 * C_LIGHT - 1) < 1e-15 and abs(iE * b0 * p0c - 1) < 1e-15
    V, f = 1e6, 2.856e9
    A, om = V * iE, 2 * math.pi * f
    s_ref = 12.5
    # on crest (phi = 90 deg) at s = s_ref: delta += A exactly (sin(fl(pi/2)) == 1)
    v = np.zeros((6, 1)); v[4] = s_ref; v[5] = 0.25
    elgo.rfkick(v, A, om, math.pi / 2, s_ref, ibc)
    assert v[5, 0] == 0.25 + A
    # zero crossing (phi = 0): no kick
    v = np.zeros((6, 1)); v[4] = s_ref; v[5] = 0.25
    elgo.rfkick(v, A, om, 0.0, s_ref, ibc)
    assert v[5, 0] == 0.25
    # periodicity: shifting s by one RF wavelength beta0 c / f gives the same kick
    lam = b0 * C_LIGHT / f
    s = np.linspace(-0.01, 0.01, 101) + s_ref
    v1 = np.zeros((6, s.size)); v1[4] = s
    v2 = np.zeros((6, s.size)); v2[4] = s + lam
    elgo.rfkick(v1, A, om, 0.3, s_ref, ibc)
    elgo.rfkick(v2, A, om, 0.3, s_ref, ibc)
    assert np.max(np.abs(v1[5] - v2[5])) <= 1e-12 * A * 40   # phase error ~ omega*tau*eps
    # direct formula and sign of the slope at phi = 180 deg: d(delta)/d(tau) = -A omega
    expect = A * np.sin(0.3 + om * (s - s_ref) / (b0 * C_LIGHT))
    assert np.max(np.abs(v1[5] - expect)) <= 1e-12 * A
    ds = 1e-6
    v = np.zeros((6, 2)); v[4] = [s_ref, s_ref + ds]
    elgo.rfkick(v, A, om, math.pi, s_ref, ibc)
    slope = (v[5, 1] - v[5, 0]) / (ds * ibc)
    assert abs(slope / (-A * om) - 1) < 1e-6
    # only delta changes
    assert np.array_equal(v[4], [s_ref, s_ref + ds])


# ------------------------------------------------------------------------------------ apertures
def test_aperture_hand_placed(elgo):
    a = 300e-6
    eps = 1e-6
    x = np.array([0.0, a * (1 - eps), a * (1 + eps), a, -a, -a * (1 + eps), np.nan, 0.0, 0.0, 0.0])
    y = np.array([0.0, 0.0, 0.0, a, -a, 0.0, 0.0, np.nan, a * (1 + eps), -a * (1 - eps)])
    got = elgo.aperture_flags(x, y, elgo.RCOL, a, a)
    assert got.tolist() == [1, 1, 0, 1, 1, 0, 0, 0, 0, 1]          # inclusive edges, NaN lost (G17)
    # ellipse a x b: on-axis edge points inclusive, corner of the rectangle outside
    b = 150e-6
    x = np.array([a, -a, 0.0, 0.0, a, a / 2, a * 0.8, np.nan, a * (1 + eps)])
    y = np.array([0.0, 0.0, b, -b, b, b / 2, b * 0.7, 0.0, 0.0])
    got = elgo.aperture_flags(x, y, elgo.ECOL, a, b)
    assert got.tolist() == [1, 1, 1, 1, 0, 1, 0, 0, 0]
    # asymmetric rectangle: ax applies to x, ay to y (argument order pin)
    got = elgo.aperture_flags(np.array([2.0, 0.0]), np.array([0.0, 2.0]), elgo.RCOL, 3.0, 1.0)
    assert got.tolist() == [1, 0]
    got = elgo.aperture_flags(np.array([2.0, 0.0]), np.array([0.0, 2.0]), elgo.ECOL, 3.0, 1.0)
    assert got.tolist() == [1, 0]


def test_compact_fig2_shape_and_bruteforce(elgo):
    """PAPER.md:135 (Fig. 2 caption): 20 particles, 4 lost.  Stable order (north_star part 2)."""
    n = 20
    lost_pos = [3, 7, 8, 19]
    surv = np.ones(n, dtype=np.uint8); surv[lost_pos] = 0
    v = np.arange(6 * n, dtype=np.float64).reshape(6, n)
    ids = np.arange(100, 100 + n, dtype=np.int64)
    v0 = v.copy()
    ns, lv, lid = elgo.compact(v, ids, surv)
    keep = [i for i in range(n) if i not in lost_pos]
    assert ns == 16
    assert ids[:ns].tolist() == [100 + i for i in keep]
    assert np.array_equal(v[:, :ns], v0[:, keep])
    assert lid.tolist() == [100 + i for i in lost_pos]
    assert np.array_equal(lv, v0[:, lost_pos])
    # brute-force O(n^2) stable partition on random flags: destination = number of earlier survivors
    rng = np.random.default_rng(5)
    for n in (1, 2, 33, 1000):
        surv = (rng.random(n) < 0.7).astype(np.uint8)
        v0 = rng.normal(size=(6, n)); ids0 = rng.permutation(n).astype(np.int64)
        v = v0.copy(); ids = ids0.copy()
        ns, lv, lid = elgo.compact(v, ids, surv)
        exp_ids = np.full(n, -1, dtype=np.int64)
        for i in range(n):
            if surv[i]:
                exp_ids[sum(int(f) for f in surv[:i])] = ids0[i]
        assert ns == int(surv.sum())
        assert np.array_equal(ids[:ns], exp_ids[:ns])
        assert sorted(ids[:ns].tolist() + lid.tolist()) == sorted(ids0.tolist())    # each ID once
        assert np.array_equal(lid, ids0[surv == 0])
        assert np.array_equal(v[:, :ns], v0[:, surv == 1])
        assert np.array_equal(lv, v0[:, surv == 0])
    # nothing lost / everything lost
    v = np.ones((6, 5)); ids = np.arange(5, dtype=np.int64)
    assert elgo.compact(v, ids, np.ones(5, np.uint8))[0] == 5
    assert elgo.compact(v, ids, np.zeros(5, np.uint8))[0] == 0


def test_loss_fraction_statistics(elgo):
    """Gaussian beam through RCOL / ECOL: loss fraction vs erf / exp(-r^2/2) within 4/sqrt(N)."""
    w = make_workload("cfg0", n=400_000)
    v = w.particles()
    sig = 100e-6
    a = 2.0 * sig
    f = elgo.aperture_flags(v[0], v[2], elgo.RCOL, a, a)
    p_surv = math.erf(2.0 / math.sqrt(2)) ** 2
    assert abs(f.mean() - p_surv) < 4 / math.sqrt(v.shape[1])
    f = elgo.aperture_flags(v[0], v[2], elgo.ECOL, a, a)
    assert abs(f.mean() - (1 - math.exp(-2.0))) < 4 / math.sqrt(v.shape[1])


# ------------------------------------------------------------------------------------ histogram
def test_window_modes(elgo):
    ibc = 1.0 / 3e8
    s = np.array([3.0, 9.0, 6.0])
    t_lo, dt, inv_dt = elgo.window(s, ibc, elgo.WIN["AUTO_MINMAX"], 4)
    assert dt == (9.0 * ibc - 3.0 * ibc) / 3 and t_lo == 3.0 * ibc - 0.5 * dt and inv_dt == 1.0 / dt
    t_lo, dt, _ = elgo.window(s, ibc, elgo.WIN["AUTO_TABLE"], 8, dt_in=1e-9)
    assert dt == 1e-9 and t_lo == 0.5 * (3.0 * ibc + 9.0 * ibc) - 4 * 1e-9
    t_lo, dt, _ = elgo.window(s, ibc, elgo.WIN["EXPLICIT"], 8, t_lo_rel=-2e-9, dt_in=5e-10, t_design=1e-6)
    assert dt == 5e-10 and t_lo == 1e-6 - 2e-9
    # degenerate: a single particle (G10/G28)
    t_lo, dt, _ = elgo.window(np.array([2.0]), ibc, elgo.WIN["AUTO_MINMAX"], 16)
    assert dt == 1e-15 and t_lo == 2.0 * ibc - 0.5e-15


def test_histogram_hand_placed(elgo):
    nb, t_lo, dt = 8, 1.0, 0.5           # power-of-two spacing: everything exact; inv_bc = 1
    centres = t_lo + (np.arange(nb) + 0.5) * dt
    c, binned = elgo.histogram(centres, 1.0, t_lo, 1 / dt, nb)
    assert c.tolist() == [1] * nb and binned == nb
    edges = t_lo + np.arange(nb + 1) * dt            # lower edge inclusive; the last edge is outside
    c, binned, bins = elgo.histogram(edges, 1.0, t_lo, 1 / dt, nb, want_bins=True)
    assert c.tolist() == [1] * nb and binned == nb
    assert bins.tolist() == list(range(nb)) + [-1]
    # outside and NaN are not counted
    c, binned = elgo.histogram(np.array([0.99, 5.0, 100.0, np.nan, -1e30]), 1.0, t_lo, 1 / dt, nb)
    assert int(c.sum()) == 0 and binned == 0
    # all in one bin (contention case)
    c, binned = elgo.histogram(np.full(1000, 2.3), 1.0, t_lo, 1 / dt, nb)
    assert c[2] == 1000 and int(c.sum()) == 1000
    # inv_bc is applied to s
    c, _ = elgo.histogram(np.array([4.6]), 0.5, t_lo, 1 / dt, nb)
    assert c[2] == 1


def test_histogram_matches_numpy_and_sums_to_n(elgo):
    """AUTO windows cover every particle: sum(counts) == n (north_star); counts == numpy.histogram."""
    w = make_workload("cfg0", n=200_000)
    v = w.particles()
    b0 = elgo.beta0(w.p0c_eV); ibc = elgo.inv_bc(b0)
    for mode, nb, kw in (("AUTO_MINMAX", 512, {}), ("AUTO_TABLE", 1 << 15, {"dt_in": 0.05e-12 * 40})):
        t_lo, dt, inv_dt = elgo.window(v[4], ibc, elgo.WIN[mode], nb, **kw)
        c, binned, bins = elgo.histogram(v[4], ibc, t_lo, inv_dt, nb, want_bins=True)
        assert binned == v.shape[1] and int(c.sum()) == v.shape[1]
        ref = np.bincount(bins, minlength=nb)
        assert np.array_equal(ref, c)
        # independent: numpy.histogram on uniform edges, away from edge-rounding cases
        u = (v[4] * ibc - t_lo) / dt
        safe = np.abs(u - np.round(u)) > 1e-9
        ref2, _ = np.histogram(u[safe], bins=nb, range=(0, nb))
        c2, _ = elgo.histogram(v[4][safe], ibc, t_lo, inv_dt, nb)
        assert np.array_equal(ref2, c2)


# ------------------------------------------------------------------------------------ wake
def test_wake_samples_resonator(elgo):
    f, Q, Rs, dt, nb = 1e9, 1.0, 1e3, 7e-12, 64
    W = elgo.wake_samples(elgo.WAKEKIND["RESONATOR"], nb, dt, f=f, Q=Q, Rs=Rs)
    wr = 2 * math.pi * f
    kloss = wr * Rs / (2 * Q)
    assert abs(W[0] / kloss - 1) < 1e-15                       # beam-loading theorem (G11)
    # independent evaluation through the complex form  W = 2k Re[(1 + i a/wb) e^{(-a + i wb) t}]
    a = wr / (2 * Q)
    wb = math.sqrt(wr * wr - a * a)
    t = np.arange(1, nb) * dt
    ref = 2 * kloss * np.real((1 + 1j * a / wb) * np.exp((-a + 1j * wb) * t))
    assert np.max(np.abs(W[1:] - ref)) <= 1e-13 * 2 * kloss
    # t -> 0+ limit is 2 k_loss; high-Q wake oscillates at ~f with slow decay
    W2 = elgo.wake_samples(elgo.WAKEKIND["RESONATOR"], 4, 1e-18, f=f, Q=Q, Rs=Rs)
    assert abs(W2[1] / (2 * kloss) - 1) < 1e-6
    W3 = elgo.wake_samples(elgo.WAKEKIND["RESONATOR"], 3, 1.0 / f, f=f, Q=1e6, Rs=Rs)
    assert abs(W3[1] / (2 * wr * Rs / 2e6) - 1) < 1e-4          # one period later: ~ 2k (cos = 1)
    with pytest.raises(ValueError):
        elgo.wake_samples(elgo.WAKEKIND["RESONATOR"], 4, dt, f=f, Q=0.5, Rs=Rs)


def test_wake_samples_table(elgo):
    tb = np.array([5.0, 3.0, -1.0, 0.5])
    W = elgo.wake_samples(elgo.WAKEKIND["TABLE"], 6, 2.0, table=tb, dt_table=2.0)
    assert W.tolist() == [5.0, 3.0, -1.0, 0.5, 0.0, 0.0]        # verbatim, zero beyond (G12)
    W = elgo.wake_samples(elgo.WAKEKIND["TABLE"], 8, 1.0, table=tb, dt_table=2.0)
    assert W.tolist() == [5.0, 4.0, 3.0, 1.0, -1.0, -0.25, 0.5, 0.0]   # linear interpolation


def test_convolve_bruteforce_and_numpy(elgo):
    rng = np.random.default_rng(7)
    for nb in (1, 2, 5, 64, 300):
        cnt = rng.integers(0, 50, size=nb).astype(np.uint32)
        W = rng.normal(size=nb)
        q = 1.5e-12
        V = elgo.convolve(cnt, W, q)
        ref = np.zeros(nb)
        for i in range(nb):                    # the serial O(N1 N2) algorithm
            for j in range(i + 1):
                ref[i] += cnt[j] * W[i - j]
        ref *= q
        scale = np.max(np.abs(ref)) + 1e-300
        assert np.max(np.abs(V - ref)) <= 1e-13 * scale
        ref2 = q * np.convolve(cnt.astype(np.float64), W)[:nb]      # library routine
        assert np.max(np.abs(V - ref2)) <= 1e-13 * scale
        assert abs(V[0] - q * float(cnt[0]) * W[0]) <= 4e-16 * abs(V[0])                  # causality
        assert np.allclose(elgo.convolve(cnt, W, 2 * q), 2 * V, rtol=1e-15, atol=0)      # linearity
    # orientation: a single leading macro-particle kicks the ones BEHIND it (larger bins), G13
    cnt = np.zeros(8, np.uint32); cnt[2] = 1
    W = np.arange(1.0, 9.0)
    V = elgo.convolve(cnt, W, 1.0)
    assert V.tolist() == [0, 0, 1, 2, 3, 4, 5, 6]


def test_single_and_two_particle_wake_kick(elgo):
    """One macro-particle loses q k_loss (beam loading); a trailing one m bins behind sees W_0 + W_m."""
    p0c = 1e9
    b0 = elgo.beta0(p0c); ibc = elgo.inv_bc(b0); iE = elgo.inv_E(b0, p0c)
    f, Q, Rs, q = 1e9, 1.0, 1e3, 1e-12
    nb, dt, m = 16, 2.0 ** -36, 5
    t_lo = 0.0
    kind = elgo.WAKEKIND["RESONATOR"]
    W = elgo.wake_samples(kind, nb, dt, f=f, Q=Q, Rs=Rs)
    t = np.array([2.5 * dt, (2.5 + m) * dt])            # bin centres of bins 2 and 7
    s = t / ibc
    c, binned = elgo.histogram(s, ibc, t_lo, 1 / dt, nb)
    assert binned == 2 and c[2] == 1 and c[7] == 1
    V = elgo.convolve(c, W, q)
    delta = np.zeros(2)
    elgo.kick(s, delta, ibc, t_lo, 1 / dt, nb, V, iE, interp=False)
    kloss = 2 * math.pi * f * Rs / (2 * Q)
    assert abs(delta[0] / (-q * kloss * iE) - 1) < 1e-14
    assert abs(delta[1] / (-q * (W[0] + W[m]) * iE) - 1) < 1e-14


def test_kick_interpolation(elgo):
    nb, t_lo, dt = 8, 0.0, 0.25
    V = np.array([1.0, 3.0, 2.0, -4.0, 0.0, 8.0, 8.5, 7.0])
    iE = 0.5
    centres = t_lo + (np.arange(nb) + 0.5) * dt
    d = np.zeros(nb)
    elgo.kick(centres, d, 1.0, t_lo, 1 / dt, nb, V, iE)
    assert np.array_equal(d, -V * iE)                            # at a bin centre: exactly V_k
    mid = centres[:-1] + dt / 2
    d = np.zeros(nb - 1)
    elgo.kick(mid - 1e-12, d, 1.0, t_lo, 1 / dt, nb, V, iE)
    assert np.allclose(d, -0.5 * (V[:-1] + V[1:]) * iE, rtol=0, atol=1e-9)   # midway: the mean
    d = np.zeros(2)
    elgo.kick(np.array([t_lo + 0.01 * dt, t_lo + (nb - 0.01) * dt]), d, 1.0, t_lo, 1 / dt, nb, V, iE)
    assert d.tolist() == [-V[0] * iE, -V[-1] * iE]               # beyond the end centres: end values
    d = np.full(3, 0.125)
    elgo.kick(np.array([t_lo - dt, t_lo + nb * dt, np.nan]), d, 1.0, t_lo, 1 / dt, nb, V, iE)
    assert d.tolist() == [0.125] * 3                             # unbinned particles are not kicked
    d = np.zeros(1)
    elgo.kick(np.array([t_lo + 2.9 * dt]), d, 1.0, t_lo, 1 / dt, nb, V, iE, interp=False)
    assert d[0] == -V[2] * iE


def test_cfg2_wake_continuous_closed_form(elgo):
    """Uniform bunch + W = A e^{-t/tau} cos(w t): V(t) = q lam A Re[(1 - e^{-z t})/z], z = 1/tau - i w
    (statistical pin: discretisation + shot noise, ~1e-2 of max)."""
    w = make_workload("cfg2", n=400_000)
    v = w.particles()
    e = w.elements[1]
    b0 = elgo.beta0(w.p0c_eV); ibc = elgo.inv_bc(b0)
    nb, dt = e["nb"], e["dt_table"]
    t_lo, _, inv_dt = elgo.window(v[4], ibc, elgo.WIN["AUTO_TABLE"], nb, dt_in=dt)
    c, binned = elgo.histogram(v[4], ibc, t_lo, inv_dt, nb)
    assert binned == v.shape[1]
    W = elgo.wake_samples(elgo.WAKEKIND["TABLE"], nb, dt, table=e["table"], dt_table=dt)
    q = w.charge_C / v.shape[1]
    V = elgo.convolve(c, W, q)
    T = 4e-3 * ibc
    lam = w.charge_C / T                                          # C/s
    t0 = (v[4].min()) * ibc
    tc = t_lo + (np.arange(nb) + 0.5) * dt - t0
    z = 1 / 10e-12 - 1j * 2 * np.pi * 3e9
    ref = np.where((tc > 0) & (tc < T), lam * 1e14 * np.real((1 - np.exp(-z * np.clip(tc, 0, T))) / z), np.nan)
    ok = ~np.isnan(ref)
    assert ok.sum() > 200
    assert np.nanmax(np.abs(V[ok] - ref[ok])) < 0.05 * np.nanmax(np.abs(ref))


# ------------------------------------------------------------------------------------ moments
def test_moments_exact_sets_and_shift_invariance(elgo):
    # +-1 points on each axis pair: centroid 0, Sigma = diag(1/3 ... ) exactly computable
    v = np.zeros((6, 12))
    for c in range(6):
        v[c, 2 * c] = 1.0
        v[c, 2 * c + 1] = -1.0
    cen, S = elgo.moments(v)
    assert np.array_equal(cen, np.zeros(6))
    assert np.allclose(S, np.eye(6) * (2.0 / 12.0), rtol=0, atol=1e-17)
    # correlated pair: x = (1,2,3,4), x' = 2x  -> var 1.25, cov 2.5, var' 5
    v = np.zeros((6, 4)); v[0] = [1, 2, 3, 4]; v[1] = [2, 4, 6, 8]; v[4] = [7, 7, 7, 7]
    cen, S = elgo.moments(v)
    assert cen[0] == 2.5 and cen[1] == 5.0 and cen[4] == 7.0
    assert S[0, 0] == 1.25 and S[0, 1] == 2.5 and S[1, 0] == 2.5 and S[1, 1] == 5.0 and S[4, 4] == 0.0
    # shift invariance: s is an absolute path length -> catches one-pass cancellation
    w = make_workload("cfg0", n=100_000)
    v = w.particles()
    _, S0 = elgo.moments(v)
    v2 = v.copy(); v2[4] += 1.0e4
    cen2, S2 = elgo.moments(v2)
    assert np.max(np.abs(S2 - S0)) <= 1e-10 * np.max(np.abs(S0))
    # Gaussian statistics
    sig = np.array([100e-6, 10e-6, 100e-6, 10e-6, 1e-3, 1e-3])
    n = v.shape[1]
    assert np.all(np.abs(np.diag(S0) / sig ** 2 - 1) < 4 * math.sqrt(2.0 / n))
    # numpy reference (library routine)
    assert np.max(np.abs(S0 - np.cov(v, bias=True))) <= 1e-12 * np.max(np.abs(S0))
    assert np.max(np.abs(cen2 - v2.mean(axis=1))) <= 1e-12 * 1e4


# ------------------------------------------------------------------------------------ track
def test_track_is_the_composition_of_stages(elgo):
    """elgo_track on cfg0 equals the stage functions applied by hand in the order of PAPER.md:51."""
    w = make_workload("cfg0", n=20_000)
    v0 = w.particles()
    b = elgo.Bunch(v0, w.p0c_eV, w.charge_C)
    bl = elgo.Beamline(w.elements, ring=False)
    assert bl.length == 1.5 and bl.s_design(1) == 1.0 and bl.s_design(3) == 1.5
    out = b.track(bl, 1, moments_every="turn", want_stage_outputs=True)
    v, ids = b.read()
    # by hand
    h = v0.copy(); hid = np.arange(h.shape[1], dtype=np.int64)
    elgo.drift(h, 1.0)
    elgo.matrix(h, w.elements[1]["R"], w.elements[1]["C"])
    f = elgo.aperture_flags(h[0], h[2], elgo.RCOL, 300e-6, 300e-6)
    pre = h.copy()
    ns, lv, lid = elgo.compact(h, hid, f)
    h = np.ascontiguousarray(h[:, :ns]); hid = hid[:ns]
    b0 = elgo.beta0(w.p0c_eV); ibc = elgo.inv_bc(b0); iE = elgo.inv_E(b0, w.p0c_eV)
    t_lo, dt, inv_dt = elgo.window(h[4], ibc, elgo.WIN["AUTO_MINMAX"], 512)
    c, binned = elgo.histogram(h[4], ibc, t_lo, inv_dt, 512)
    W = elgo.wake_samples(elgo.WAKEKIND["RESONATOR"], 512, dt, f=1e9, Q=1.0, Rs=1e3)
    V = elgo.convolve(c, W, w.charge_C / w.n0)
    elgo.kick(h[4], h[5], ibc, t_lo, inv_dt, 512, V, iE)
    assert np.array_equal(ids, hid) and np.array_equal(v, h)
    assert np.array_equal(out["hist"], c) and np.array_equal(out["V"], V)
    assert out["window"][0].tolist() == [t_lo, dt, inv_dt]
    assert binned == ns and 0.002 < 1 - ns / w.n0 < 0.012          # G4/G22: ~0.59 % loss
    li, lt, le, lc = b.lost()
    assert np.array_equal(li, lid) and set(lt.tolist()) == {0} and set(le.tolist()) == {2}
    assert np.array_equal(lc.T, pre[:, f == 0])
    assert np.all(np.diff(ids) > 0)                                # stable: IDs strictly increasing
    rec = out["records"]
    assert rec.shape == (1, 43) and rec[0, 0] == ns
    cen, S = elgo.moments(h)
    assert np.array_equal(rec[0, 1:7], cen) and np.array_equal(rec[0, 7:].reshape(6, 6), S)
    # the wake decelerates: mean delta decreases (sign pin, G30)
    assert h[5].mean() < pre[5][f == 1].mean()


def test_track_threads_and_turns(elgo):
    """n_threads does not change results; a ring advances s_ref by the ring length per turn (G8)."""
    w = make_workload("cfg3", n=3000, n_matrices=6, n_turns=3)
    v0 = w.particles()
    outs = []
    for nt in (1, 4):
        b = elgo.Bunch(v0, w.p0c_eV, w.charge_C)
        bl = elgo.Beamline(w.elements, ring=True)
        o = b.track(bl, 3, moments_every="turn", n_threads=nt, want_stage_outputs=True)
        outs.append((b.read()[0], o))
    assert np.array_equal(outs[0][0], outs[1][0])
    assert np.array_equal(outs[0][1]["records"], outs[1][1]["records"])
    assert outs[0][1]["records"].shape == (3, 43)
    # by hand, turn by turn, with explicit s_ref = turn * length + s_design(k)
    bl = elgo.Beamline(w.elements, ring=True)
    assert bl.length == 6.0
    b0 = elgo.beta0(w.p0c_eV); ibc = elgo.inv_bc(b0); iE = elgo.inv_E(b0, w.p0c_eV)
    h = v0.copy()
    for turn in range(3):
        for k, e in enumerate(w.elements):
            if e["type"] == "MATRIX":
                elgo.matrix(h, e["R"], e["C"])
            elif e["type"] == "RFKICK":
                elgo.rfkick(h, e["V"] * iE, 2 * math.pi * e["f"], e["phi"], turn * 6.0 + 6.0, ibc)
            else:
                t_lo, dt, inv_dt = elgo.window(h[4], ibc, elgo.WIN["AUTO_MINMAX"], e["nb"])
                c, _ = elgo.histogram(h[4], ibc, t_lo, inv_dt, e["nb"])
                W = elgo.wake_samples(0, e["nb"], dt, f=e["f"], Q=e["Q"], Rs=e["Rs"])
                V = elgo.convolve(c, W, w.charge_C / w.n0)
                elgo.kick(h[4], h[5], ibc, t_lo, inv_dt, e["nb"], V, iE)
    assert np.array_equal(outs[0][0], h)
    # design orbit: centroid of s after 3 turns is 18 m + initial (all matrices carry C5 = 1)
    assert abs(outs[0][1]["records"][2, 1 + 4] - 18.0) < 1e-3


def test_track_loss_sequence_cfg4_small(elgo):
    """cfg4 at reduced size: survivors + lost = all IDs once; chronological canonical order (G18)."""
    w = make_workload("cfg4", n=30_000)
    v0 = w.particles()
    b = elgo.Bunch(v0, w.p0c_eV, w.charge_C)
    bl = elgo.Beamline(w.elements, ring=False)
    out = b.track(bl, 1, want_stage_outputs=True)
    v, ids = b.read()
    li, lt, le, lc = b.lost()
    assert ids.size + li.size == w.n0
    assert np.array_equal(np.sort(np.concatenate([ids, li])), np.arange(w.n0))
    assert np.all(np.diff(ids) > 0)
    key = le.astype(np.int64) * w.n0 + li
    assert np.all(np.diff(key) > 0)                                # (element, ID) strictly increasing
    hist = out["hist"].reshape(20, 65536)
    n_after = w.n0 - np.array([(le <= 3 * i).sum() for i in range(20)])
    assert np.array_equal(hist.sum(axis=1), n_after)               # every survivor is binned
    occupied = (hist[0] > 0).sum()
    assert 30 <= occupied <= 80                                     # "~50 bins" contention case
    # first collimator: uniform +-1 mm through +-0.9 mm in x and y -> survive 0.81
    assert abs((le == 0).sum() / w.n0 - 0.19) < 4 / math.sqrt(w.n0)
    # every lost record violates its aperture, at the recorded coordinates
    hw = np.array([0.9e-3 + (0.2e-3 - 0.9e-3) * (e // 3) / 19.0 for e in le])
    assert np.all((np.abs(lc[:, 0]) > hw) | (np.abs(lc[:, 2]) > hw))


# ------------------------------------------------------------------------------------ MATRIX2 (G31)
def test_matrix2_reduces_to_matrix_and_index_convention(elgo):
    """T = 0 is elgo_matrix bit for bit; a single T entry (i; j,k) gives out_i = R-part + T v_j v_k, for every
    (i, j <= k): catches a transposed or mis-ordered pair index."""
    from elg_inputs import pair_index
    rng = np.random.default_rng(5)
    v0 = rng.normal(size=(6, 50)) * np.array([1e-3, 1e-4, 1e-3, 1e-4, 1e-2, 1e-3])[:, None]
    R = np.eye(6) + 0.1 * rng.normal(size=(6, 6)); Cv = rng.normal(size=6) * 1e-3
    a = v0.copy(); b = v0.copy()
    elgo.matrix(a, R, Cv); elgo.matrix2(b, R, np.zeros((6, 21)), Cv)
    assert np.array_equal(a, b)
    seen = set()
    for i in range(6):
        for j in range(6):
            for k in range(j, 6):
                q = pair_index(j, k); seen.add(q)
                T = np.zeros((6, 21)); T[i, q] = 3.0
                b = v0.copy(); elgo.matrix2(b, np.eye(6), T)
                exp = v0.copy(); exp[i] = exp[i] + 3.0 * (v0[j] * v0[k])
                assert np.allclose(b, exp, rtol=0, atol=1e-18), (i, j, k)
                others = [r for r in range(6) if r != i]
                assert np.array_equal(b[others], v0[others])
    assert seen == set(range(21)) and pair_index(2, 0) == pair_index(0, 2) == 2 and pair_index(5, 5) == 20


def test_matrix2_sextupole_and_drift_closed_forms(elgo):
    """Thin quadrupole + sextupole kick against its definition; the second-order drift against Listing 1's
    exact drift: the path lengths differ by the next term of the expansion, -L/8 (x'^2+y'^2)^2."""
    from elg_inputs import second_order_drift, thin_quad_sextupole
    rng = np.random.default_rng(6)
    v0 = rng.normal(size=(6, 200)) * np.array([1e-3, 1e-3, 1e-3, 1e-3, 1e-2, 1e-3])[:, None]
    k1, k2 = 0.7, -35.0
    R, Cv, T = thin_quad_sextupole(k1, k2)
    a = v0.copy(); elgo.matrix2(a, R, T, Cv)
    x, xp, y, yp = v0[:4]
    assert np.array_equal(a[[0, 2, 4, 5]], v0[[0, 2, 4, 5]])
    assert np.allclose(a[1], xp - k1 * x - 0.5 * k2 * (x * x - y * y), rtol=1e-15, atol=1e-20)
    assert np.allclose(a[3], yp + k1 * y + k2 * x * y, rtol=1e-15, atol=1e-20)
    L = 2.5
    R, Cv, T = second_order_drift(L)
    v1 = v0.copy(); v1[1] *= 10.0; v1[3] *= 10.0; v1[4] = 0.0                  # slopes ~1e-2: the O(x'^4) term is resolved
    a = v1.copy(); elgo.matrix2(a, R, T, Cv)
    e = v1.copy(); elgo.drift(e, L)
    assert np.allclose(a[[0, 2]], e[[0, 2]], rtol=1e-15, atol=1e-20)
    u = v1[1] * v1[1] + v1[3] * v1[3]
    # sqrt(1 + u) = 1 + u/2 - u^2/8 + ...: the second-order map keeps L (1 + u/2), the exact drift has the rest
    assert np.allclose(a[4] - e[4], L / 8.0 * u * u, rtol=2e-3, atol=1e-15)
    assert np.allclose(a[4], L * (1.0 + 0.5 * u), rtol=1e-15, atol=0)


def test_matrix2_in_track(elgo):
    """elgo_track applies MATRIX2 elements in order and counts C[4] into the design path length (G8)."""
    w = make_workload("p4-second-order", n=300, n_cells=3)
    v0 = w.particles()
    ob = elgo.Bunch(v0, w.p0c_eV, w.charge_C); bl = elgo.Beamline(w.elements, ring=True)
    ob.track(bl, 2)
    ref = v0.copy()
    for _ in range(2):
        for e in w.elements:
            elgo.matrix2(ref, e["R"], e["T"], e["C"])
    assert np.array_equal(ob.read()[0], ref)
    assert bl.length == 3.0


# ------------------------------------------------------------------------------------ TRWAKE (G32-G34)
def test_dipole_histogram_is_the_plain_weighted_sum(elgo):
    """G33: the dipole sums are the plain per-bin sums of x and y (against the exactly rounded math.fsum: <= 1e-15 of
    the sum of magnitudes, i.e. at most the final rounding), a permutation of the particles changes them by no more
    than that, and the counts are elgo_histogram's."""
    rng = np.random.default_rng(11)
    n, nb = 200_000, 97
    s = rng.normal(size=n) * 1e-3
    x = rng.normal(size=n) * 1e-4 + 3e-5
    y = rng.normal(size=n) * 2e-4 - 1e-5
    inv_bc = elgo.inv_bc(elgo.beta0(1e9))
    t_lo, dt, inv_dt = elgo.window(s, inv_bc, 1, nb)
    c, Dx, Dy, binned = elgo.dipole_histogram(s, x, y, inv_bc, t_lo, inv_dt, nb)
    c0, b0, bins = elgo.histogram(s, inv_bc, t_lo, inv_dt, nb, want_bins=True)
    assert np.array_equal(c, c0) and binned == b0 == n
    import math
    p = rng.permutation(n)
    c2, Dx2, Dy2, _ = elgo.dipole_histogram(s[p], x[p], y[p], inv_bc, t_lo, inv_dt, nb)
    assert np.array_equal(c, c2)
    for D, D2, w in ((Dx, Dx2, x), (Dy, Dy2, y)):
        ref = np.array([math.fsum(w[bins == k]) for k in range(nb)])              # exactly rounded sums
        mag = np.array([math.fsum(np.abs(w[bins == k])) for k in range(nb)])
        assert np.all(np.abs(D - ref) <= 1e-15 * mag + 1e-300)
        assert np.all(np.abs(D2 - ref) <= 1e-15 * mag + 1e-300)
        assert np.max(np.abs(ref)) > 0
    # a wrong weight (y for x), a dropped particle or a shifted bin would be far outside: sanity of the pin itself
    assert np.max(np.abs(Dx - Dy)) > 1e-6
    # exactly representable offsets give exact sums; out-of-range / NaN offsets are counted but not summed
    s3 = np.zeros(5); x3 = np.array([0.5, 0.25, -0.125, np.nan, 4.0e6]); y3 = np.ones(5)
    c3, Dx3, Dy3, _ = elgo.dipole_histogram(s3, x3, y3, 1.0, -0.5, 1.0, 2)
    assert c3.tolist() == [5, 0] and Dx3[0] == 0.625 and Dy3[0] == 3.0
    # two particles in two bins: each sum is that particle's coordinate, bit for bit
    c4, Dx4, Dy4, _ = elgo.dipole_histogram(np.array([0.0, 1.0]), np.array([1e-4 / 3, -7e-5]), np.array([2e-4, 1e-5 / 7]),
                                            1.0, -0.5, 1.0, 2)
    assert c4.tolist() == [1, 1] and Dx4.tolist() == [1e-4 / 3, -7e-5] and Dy4.tolist() == [2e-4, 1e-5 / 7]


def test_convolve_d_bruteforce(elgo):
    rng = np.random.default_rng(12)
    D = rng.normal(size=40); W = rng.normal(size=40)
    V = elgo.convolve_d(D, W, 2.5)
    ref = np.array([2.5 * sum(D[j] * W[i - j] for j in range(i + 1)) for i in range(40)])
    assert np.allclose(V, ref, rtol=1e-13, atol=1e-15)
    assert np.allclose(V, 2.5 * np.convolve(D, W)[:40], rtol=1e-12, atol=1e-14)
    assert V[0] == 2.5 * D[0] * W[0]                                              # causality


def test_transverse_resonator_samples(elgo):
    """G34 by independent evaluation: W_T(0) = 0, W_T(tau) = (w Rs/Q)(w/wbar) exp(-alpha tau) sin(wbar tau)."""
    f, Q, Rs, dt = 3e9, 20.0, 1e6, 0.1e-12
    W = elgo.wake_samples(2, 64, dt, f=f, Q=Q, Rs=Rs)
    w = 2 * np.pi * f; al = w / (2 * Q); wb = np.sqrt(w * w - al * al)
    tau = np.arange(64) * dt
    ref = (w * Rs / Q) * (w / wb) * np.exp(-al * tau) * np.sin(wb * tau)
    assert W[0] == 0.0 and np.allclose(W, ref, rtol=1e-13, atol=0)
    assert W[1] > 0 and abs(W[1] / (w * Rs / Q * w * dt) - 1) < 1e-2              # initial slope w^2 Rs/Q


def test_trwake_two_particle_closed_form_and_linearity(elgo):
    """A leading particle with offset (x0, y0) kicks a trailing one m bins behind by q W_T(m dt) x0 / (beta0 p0c); the
    leading one is not kicked (W_T(0) = 0); zero offsets give zero kicks; the kick is linear in the offsets."""
    p0c, Qb = 1e9, 2e-9
    b0 = elgo.beta0(p0c); inv_bc = elgo.inv_bc(b0); inv_E = elgo.inv_E(b0, p0c)
    nb, dt, m = 64, 0.2e-12, 7
    f, Q, Rs = 3e9, 20.0, 1e6
    el = [{"type": "TRWAKE", "nb": nb, "window": "EXPLICIT", "t_lo_rel": -0.5 * dt, "dt": dt, "wake": "RESONATOR_T",
           "f": f, "Q": Q, "Rs": Rs, "interp": True}]
    def run(x0, y0, x1=0.0):
        v = np.zeros((6, 2)); v[0] = [x0, x1]; v[2] = [y0, 0.0]
        v[4, 1] = m * dt / inv_bc                                                  # bin centres 0 and m
        ob = elgo.Bunch(v, p0c, Qb); ob.track(elgo.Beamline(el), 1)
        return ob.read()[0]
    W = elgo.wake_samples(2, nb, dt, f=f, Q=Q, Rs=Rs)
    q = Qb / 2
    out = run(1e-3, -2e-3)
    assert out[1, 0] == 0.0 and out[3, 0] == 0.0
    assert np.isclose(out[1, 1], q * W[m] * 1e-3 * inv_E, rtol=1e-12) and out[1, 1] != 0.0
    assert np.isclose(out[3, 1], q * W[m] * -2e-3 * inv_E, rtol=1e-12)
    assert np.array_equal(out[[0, 2, 4, 5]], run(1e-3, -2e-3)[[0, 2, 4, 5]])
    zero = run(0.0, 0.0)
    assert not zero[1].any() and not zero[3].any()
    twice = run(2e-3, -4e-3)
    assert np.allclose(twice[[1, 3]], 2 * out[[1, 3]], rtol=1e-13, atol=0)
    # the trailing particle's own offset does not kick itself
    assert np.array_equal(run(1e-3, -2e-3, x1=5e-3)[[1, 3]], out[[1, 3]])


def test_trwake_track_is_the_composition_of_stages(elgo):
    w = make_workload("p5-trwake", n=20_000)
    v0 = w.particles()
    ob = elgo.Bunch(v0, w.p0c_eV, w.charge_C)
    oo = ob.track(elgo.Beamline(w.elements), 1, want_stage_outputs=True)
    b0 = elgo.beta0(w.p0c_eV); inv_bc = elgo.inv_bc(b0); inv_E = elgo.inv_E(b0, w.p0c_eV)
    v = v0.copy()
    elgo.matrix(v, w.elements[0]["R"], w.elements[0]["C"]); elgo.drift(v, 1.0)
    e = w.elements[2]
    t_lo, dt, inv_dt = elgo.window(v[4], inv_bc, 1, e["nb"])
    c, Dx, Dy, _ = elgo.dipole_histogram(v[4], v[0], v[2], inv_bc, t_lo, inv_dt, e["nb"])
    W = elgo.wake_samples(2, e["nb"], dt, f=e["f"], Q=e["Q"], Rs=e["Rs"])
    q = w.charge_C / w.n0
    Vx = elgo.convolve_d(Dx, W, q); Vy = elgo.convolve_d(Dy, W, q)
    nb = e["nb"]
    assert np.array_equal(oo["hist"][:nb], c)
    assert np.array_equal(oo["V"][:4 * nb], np.concatenate([Dx, Dy, Vx, Vy]))
    assert np.max(np.abs(Vx)) > 0 and abs(Dx.sum() / w.n0 - 2e-4) < 1e-5          # the bunch is offset by 200 um


# ------------------------------------------------------------------------------------ MATRIX3 (G35)
def test_matrix3_reduces_to_matrix2_and_index_convention(elgo):
    from elg_inputs import triple_index
    rng = np.random.default_rng(21)
    v0 = rng.normal(size=(6, 40)) * np.array([1e-3, 1e-4, 1e-3, 1e-4, 1e-2, 1e-3])[:, None]
    R = np.eye(6) + 0.1 * rng.normal(size=(6, 6)); Cv = rng.normal(size=6) * 1e-3; T = rng.normal(size=(6, 21))
    a = v0.copy(); b = v0.copy()
    elgo.matrix2(a, R, T, Cv); elgo.matrix3(b, R, T, np.zeros((6, 56)), Cv)
    assert np.array_equal(a, b)
    seen = set()
    for i in (0, 3, 5):
        for j in range(6):
            for k in range(j, 6):
                for l in range(k, 6):
                    t = triple_index(j, k, l); seen.add(t)
                    U = np.zeros((6, 56)); U[i, t] = 2.0
                    b = v0.copy(); elgo.matrix3(b, np.eye(6), np.zeros((6, 21)), U)
                    exp = v0.copy(); exp[i] = exp[i] + 2.0 * ((v0[j] * v0[k]) * v0[l])
                    assert np.allclose(b, exp, rtol=0, atol=1e-20), (i, j, k, l)
    assert seen == set(range(56)) and triple_index(5, 5, 5) == 55 and triple_index(2, 0, 1) == triple_index(0, 1, 2)


def test_matrix3_octupole_closed_form(elgo):
    """Thin quadrupole + sextupole + octupole kick against the multipole expansion Re/Im (x + i y)^n."""
    from elg_inputs import thin_quad_sext_octupole
    rng = np.random.default_rng(22)
    v0 = rng.normal(size=(6, 300)) * 2e-3
    k1, k2, k3 = 0.4, -30.0, 900.0
    R, Cv, T, U = thin_quad_sext_octupole(k1, k2, k3)
    a = v0.copy(); elgo.matrix3(a, R, T, U, Cv)
    z = v0[0] + 1j * v0[2]
    kick = k1 * z + k2 / 2 * z ** 2 + k3 / 6 * z ** 3            # sum_n knL/n! (x + i y)^n
    assert np.array_equal(a[[0, 2, 4, 5]], v0[[0, 2, 4, 5]])
    assert np.allclose(a[1], v0[1] - kick.real, rtol=1e-14, atol=1e-17)      # a few ulp of the 1e-3 slopes
    assert np.allclose(a[3], v0[3] + kick.imag, rtol=1e-14, atol=1e-17)
    assert np.max(np.abs(kick.real)) > 1e-4 and np.max(np.abs((k3 / 6 * z ** 3).real)) > 1e-7


def test_matrix3_in_track(elgo):
    w = make_workload("p7-third-order", n=200, n_cells=2)
    v0 = w.particles()
    ob = elgo.Bunch(v0, w.p0c_eV, w.charge_C); ob.track(elgo.Beamline(w.elements, ring=True), 2)
    ref = v0.copy()
    for _ in range(2):
        for e in w.elements:
            elgo.matrix3(ref, e["R"], e["T"], e["U"], e["C"])
    assert np.array_equal(ob.read()[0], ref)


# ------------------------------------------------------------------------------------ fiducial RF phase (G36)
def test_fiducial_is_the_plain_mean_and_makes_kicks_delay_invariant(elgo):
    import math
    rng = np.random.default_rng(31)
    s0 = 271.25
    s = s0 + rng.normal(size=50_000) * 1e-3 + 3e-4
    f = elgo.fiducial(s, s0)
    exact = math.fsum(s - s0) / s.size                                        # mean of the rounded differences
    assert abs((f - s0) - exact) <= 2.0 ** -52 * s0                           # the final s0 + mean rounds at ulp(s0)
    assert abs(exact - 3e-4) < 2e-5                                           # the bunch is 0.3 mm late
    assert abs(elgo.fiducial(s[rng.permutation(s.size)], s0) - f) <= 2.0 ** -52 * s0
    assert elgo.fiducial(s[:0], s0) == s0
    assert elgo.fiducial(np.array([s0 + 0.5, s0 + 0.25, s0 - 0.125, np.nan, s0 + 4.0e6]), s0) == s0 + 0.625 / 5
    # a common delay of the whole bunch changes the design-orbit kick but not the fiducial one
    w = make_workload("cfg0", n=2000)
    v0 = w.particles()
    def kicks(fid, shift):
        v = v0.copy(); v[4] += shift
        ob = elgo.Bunch(v, 1e9, 1e-9)
        ob.track(elgo.Beamline([{"type": "DRIFT", "L": 1.0}, {"type": "RFKICK", "V": 1e6, "f": 2.856e9, "phi": 0.3,
                                                          "fiducial": fid}]), 1)
        return ob.read()[0][5] - v0[5]
    a, b_ = kicks(True, 0.0), kicks(True, 7e-3)
    assert np.max(np.abs(a - b_)) <= 1e-9 * np.max(np.abs(a))                 # s + shift rounds at 1e-16 relative
    c, d = kicks(False, 0.0), kicks(False, 7e-3)
    assert np.max(np.abs(c - d)) > 0.1 * np.max(np.abs(c))
    # with the fiducial the mean phase is phi exactly: the mean kick is A sin(phi) <cos> ~ A sin(phi)
    A = 1e6 * elgo.inv_E(elgo.beta0(1e9), 1e9)
    assert abs(a.mean() / (A * math.sin(0.3)) - 1.0) < 2e-3


# ------------------------------------------------------------------------------------ recursive resonator (G37)
def test_convolve_resonator_equals_direct_convolution(elgo):
    """The O(nb) recurrence gives the V of elgo_convolve(elgo_wake_samples(resonator)) for damped (Q = 1), ringing
    (Q = 1e4) and long (8192-bin) cases; a single bin reproduces the wake samples themselves."""
    rng = np.random.default_rng(41)
    for nb, dt, f, Q, Rs in [(512, 2e-14, 1e9, 1.0, 1e3), (1024, 1.2e-14, 1.3e9, 1e4, 1e3), (8192, 5e-14, 3e9, 50.0, 2e3)]:
        c = rng.integers(0, 200_000, nb).astype(np.uint32)
        W = elgo.wake_samples(0, nb, dt, f=f, Q=Q, Rs=Rs)
        V = elgo.convolve(c, W, 1e-17)
        Vr = elgo.convolve_resonator(c, 1e-17, dt, f, Q, Rs)
        assert np.max(np.abs(V - Vr)) <= 1e-12 * np.max(np.abs(V))
        one = np.zeros(nb, dtype=np.uint32); one[0] = 1
        assert np.allclose(elgo.convolve_resonator(one, 1.0, dt, f, Q, Rs), W, rtol=1e-12, atol=1e-12 * np.max(np.abs(W)))


# ------------------------------------------------------------------------------------ record placement, lost log, ring
def test_records_after_every_element_hand_case(elgo):
    """G26 (statistics after every element): with moments_every = "element" one record follows EVERY
    element, taken on the live set AFTER that element (after the compaction of an aperture).  Three particles, the
    middle one is removed by an RCOL: the record behind the RCOL has n = 2 and the survivors' centroid; the record
    in front of it still has n = 3.  moments_every = "turn": one record, after the last element."""
    v0 = np.zeros((6, 3))
    v0[0] = [1e-4, 5e-3, -3e-4]                          # x: the middle particle is outside a 1 mm RCOL
    v0[1] = [1e-5, 0.0, -2e-5]
    v0[5] = [1e-3, 2e-3, 4e-3]
    elems = [{"type": "DRIFT", "L": 2.0}, {"type": "RCOL", "ax": 1e-3, "ay": 1e-3}, {"type": "DRIFT", "L": 1.0}]
    b = elgo.Bunch(v0, 1e9, 1e-9)
    out = b.track(elgo.Beamline(elems), 1, moments_every="element")
    rec = out["records"]
    assert rec.shape == (3, 43)
    assert rec[:, 0].tolist() == [3.0, 2.0, 2.0]
    x_after_drift = v0[0] + 2.0 * v0[1]                  # fma(x', L, x) is exact for these values? compare loosely
    assert abs(rec[0, 1] - x_after_drift.mean()) <= 1e-18
    assert abs(rec[1, 1] - x_after_drift[[0, 2]].mean()) <= 1e-18          # survivors only, right behind the RCOL
    assert abs(rec[1, 6] - 2.5e-3) <= 1e-18 and abs(rec[0, 6] - 7e-3 / 3) <= 1e-18       # <delta>
    assert abs(rec[1, 5] - 2.0) < 1e-9 and abs(rec[2, 5] - 3.0) < 1e-9      # <s>: 2 m, then 3 m
    x_end = x_after_drift[[0, 2]] + 1.0 * v0[1, [0, 2]]
    assert abs(rec[2, 1] - x_end.mean()) <= 1e-18
    S_xx = np.var(x_end)
    assert abs(rec[2, 7] - S_xx) <= 1e-12 * S_xx
    # "turn": one record, after the whole line = the last per-element record
    b2 = elgo.Bunch(v0, 1e9, 1e-9)
    out2 = b2.track(elgo.Beamline(elems), 1, moments_every="turn")
    assert out2["records"].shape == (1, 43) and np.array_equal(out2["records"][0], rec[2])
    # "none": no record
    b3 = elgo.Bunch(v0, 1e9, 1e-9)
    assert b3.track(elgo.Beamline(elems), 1, moments_every="none")["records"].shape[0] == 0


def test_records_cfg1_77_and_counts_follow_the_lost_log(elgo):
    """cfg1: 77 elements -> 77 records; n of record k = n0 - (lost at elements <= k)."""
    w = make_workload("cfg1", n=20_000)
    b = elgo.Bunch(w.particles(), w.p0c_eV, w.charge_C)
    out = b.track(elgo.Beamline(w.elements), 1, moments_every="element")
    rec = out["records"]
    assert rec.shape == (77, 43)
    li, lt, le, lc = b.lost()
    n_after = w.n0 - np.array([(le <= k).sum() for k in range(77)])
    assert np.array_equal(rec[:, 0], n_after.astype(np.float64))
    assert rec[-1, 0] == b.n_alive < w.n0


def test_tkick_interpolation(elgo):
    """elgo_tkick (G14 applied to Vx, Vy): bin centre -> exactly V_k; midway between two centres -> their mean; beyond
    the first / last centre -> the end value; interp = 0 -> the particle's own bin; unbinned -> untouched."""
    nb, t_lo, dt = 8, 0.0, 0.25
    Vx = np.array([1.0, 3.0, 2.0, -4.0, 0.0, 8.0, 8.5, 7.0])
    Vy = np.array([-2.0, 0.5, 0.25, 6.0, 1.0, -1.0, 3.0, 9.0])
    iE = 0.5
    centres = t_lo + (np.arange(nb) + 0.5) * dt
    xp = np.zeros(nb); yp = np.zeros(nb)
    elgo.tkick(centres, xp, yp, 1.0, t_lo, 1 / dt, nb, Vx, Vy, iE)
    assert np.array_equal(xp, Vx * iE) and np.array_equal(yp, Vy * iE)          # sign: x' += Vx / E (G32)
    mid = centres[:-1] + dt / 2                                                  # exactly representable: k dt
    xp = np.zeros(nb - 1); yp = np.zeros(nb - 1)
    elgo.tkick(mid - 1e-12, xp, yp, 1.0, t_lo, 1 / dt, nb, Vx, Vy, iE)
    assert np.allclose(xp, 0.5 * (Vx[:-1] + Vx[1:]) * iE, rtol=0, atol=1e-9)
    assert np.allclose(yp, 0.5 * (Vy[:-1] + Vy[1:]) * iE, rtol=0, atol=1e-9)
    # a quarter of the way from centre 2 to centre 3: V_2 + (V_3 - V_2)/4, exact in binary
    xp = np.zeros(1); yp = np.zeros(1)
    elgo.tkick(np.array([centres[2] + dt / 4]), xp, yp, 1.0, t_lo, 1 / dt, nb, Vx, Vy, iE)
    assert xp[0] == (2.0 + 0.25 * (-4.0 - 2.0)) * iE and yp[0] == (0.25 + 0.25 * (6.0 - 0.25)) * iE
    xp = np.zeros(2); yp = np.zeros(2)
    elgo.tkick(np.array([t_lo + 0.01 * dt, t_lo + (nb - 0.01) * dt]), xp, yp, 1.0, t_lo, 1 / dt, nb, Vx, Vy, iE)
    assert xp.tolist() == [Vx[0] * iE, Vx[-1] * iE] and yp.tolist() == [Vy[0] * iE, Vy[-1] * iE]
    xp = np.full(3, 0.125); yp = np.full(3, -0.5)
    elgo.tkick(np.array([t_lo - dt, t_lo + nb * dt, np.nan]), xp, yp, 1.0, t_lo, 1 / dt, nb, Vx, Vy, iE)
    assert xp.tolist() == [0.125] * 3 and yp.tolist() == [-0.5] * 3
    xp = np.zeros(1); yp = np.zeros(1)
    elgo.tkick(np.array([t_lo + 2.9 * dt]), xp, yp, 1.0, t_lo, 1 / dt, nb, Vx, Vy, iE, interp=False)
    assert xp[0] == Vx[2] * iE and yp[0] == Vy[2] * iE


def test_lost_log_truncation(elgo):
    """elgo_lost with cap < n_lost fills the first cap records (canonical order, G18), returns ELGO_ECAPACITY and the
    true n_lost; cap >= n_lost returns ELGO_OK."""
    n = 12
    v0 = np.zeros((6, n))
    v0[0] = np.where(np.arange(n) % 3 == 0, 2e-3, 1e-4)        # particles 0, 3, 6, 9 leave a 1 mm RCOL
    v0[2, 5] = -0.99e-3; v0[0, 5] = 0.5e-3                     # |x|, |y| <= 1 mm but x^2 + y^2 > 1 mm^2: lost at the ECOL only
    v0[5] = np.arange(n) * 1e-3
    elems = [{"type": "RCOL", "ax": 1e-3, "ay": 1e-3}, {"type": "ECOL", "a": 1e-3, "b": 1e-3}]
    b = elgo.Bunch(v0, 1e9, 1e-9)
    b.track(elgo.Beamline(elems, ring=True), 2)
    ids, turn, elem, co = b.lost()
    assert ids.tolist() == [0, 3, 6, 9, 5] and elem.tolist() == [0, 0, 0, 0, 1] and turn.tolist() == [0] * 5
    assert np.array_equal(co[:, 5], v0[5, [0, 3, 6, 9, 5]]) and np.array_equal(co[:, 0], v0[0, [0, 3, 6, 9, 5]])
    i3, t3, e3, c3, rc, nl = b.lost(cap=3)
    assert rc == elgo.ECAPACITY and nl == 5
    assert i3.tolist() == [0, 3, 6] and np.array_equal(c3, co[:3]) and e3.tolist() == [0, 0, 0]
    i5, t5, e5, c5, rc, nl = b.lost(cap=5)
    assert rc == elgo.OK and nl == 5 and i5.tolist() == ids.tolist()
    i9, t9, e9, c9, rc, nl = b.lost(cap=9)
    assert rc == elgo.OK and nl == 5 and i9.tolist() == ids.tolist()
    i0, t0, e0, c0, rc, nl = b.lost(cap=0)
    assert rc == elgo.ECAPACITY and nl == 5 and i0.size == 0


def test_ring_flag_advances_rf_reference_only_on_a_ring(elgo):
    """G8: on a ring (ring = 1) the RF phase reference advances by the ring length per turn; a line (ring = 0) is
    entered afresh on every pass (reference of turn 0).  One linear drift MATRIX (C5 = L) + RFKICK at 90 degrees:
    a particle on the design orbit is on crest every turn on a ring, and off crest by 2 pi f L / (beta0 c) per turn on
    a line."""
    from elg_inputs import drift_matrix
    p0c = 1e9
    b0 = elgo.beta0(p0c); ibc = elgo.inv_bc(b0); A = 1e6 * elgo.inv_E(b0, p0c)
    L, f = 0.3, 2.856e9
    R, Cv = drift_matrix(L)
    elems = [{"type": "MATRIX", "R": R, "C": Cv}, {"type": "RFKICK", "V": 1e6, "f": f, "phi": math.pi / 2}]
    v0 = np.zeros((6, 1))
    out = {}
    for ring in (True, False):
        b = elgo.Bunch(v0, p0c, 1e-9)
        b.track(elgo.Beamline(elems, ring=ring), 3)
        out[ring] = b.read()[0][5, 0]
    assert abs(out[True] - 3 * A) <= 1e-15 * A                                   # on crest three times
    phase = 2 * math.pi * f * L * ibc
    expect = A * (1.0 + math.cos(phase) + math.cos(2 * phase))                   # sin(pi/2 + k phase)
    assert abs(out[False] - expect) <= 1e-9 * A and abs(out[False] - out[True]) > 0.1 * A

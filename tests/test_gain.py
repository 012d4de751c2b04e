"""Pins of the G-Jones oracle (oracle/lra_ref_gain.c; Eq. 19-21) against
things the equations fix, not against itself: noise-free data V^obs = g_i conj(g_j) V^Mod are solved exactly (up to the
global phase the problem leaves free); the true gains are a fixed point of Eq. 20; the chi^2 of the paper falls
monotonically for alpha <= 1/2; Eq. 19 on constant ratios returns the ratio; partitions of the rows accumulate.  No GPU."""
import numpy as np
import pytest


def _setup(nant=7, ntime=40, nchan=3, ncorr=2, seed=3, noise=0.0):
    rng = np.random.default_rng(seed)
    a1, a2 = np.triu_indices(nant, 1)
    nbl = len(a1)
    g = (1 + 0.3 * rng.standard_normal((nant, ncorr))) * np.exp(1j * rng.uniform(-1, 1, (nant, ncorr)))
    model = (rng.standard_normal((ntime * nbl, nchan, ncorr)) + 1j * rng.standard_normal((ntime * nbl, nchan, ncorr))).astype(np.complex64)
    gg = g[a1][:, None, :] * np.conj(g[a2])[:, None, :]                       # [nbl, 1, ncorr]
    vis = (np.tile(gg, (ntime, 1, 1)) * model).astype(np.complex64)
    if noise:
        vis = (vis + noise * (rng.standard_normal(vis.shape) + 1j * rng.standard_normal(vis.shape))).astype(np.complex64)
    wt = rng.uniform(0.5, 1.0, vis.shape).astype(np.float32)
    return a1.astype(np.int32), a2.astype(np.int32), nbl, g, vis, model, wt


def test_eq19_is_the_weighted_mean_of_the_ratio(ref):
    a1, a2, nbl, g, vis, model, wt = _setup()
    x, w = ref.gain_accumulate(vis, model, wt, nbl)
    ratio = (vis.astype(np.complex128) / model.astype(np.complex128)).reshape(-1, nbl, *vis.shape[1:])
    wr = wt.astype(np.float64).reshape(-1, nbl, *vis.shape[1:])
    want_x = (ratio * wr).sum(axis=(0, 2)) / wr.sum(axis=(0, 2))
    assert np.abs(x / w - want_x).max() <= 1e-12
    assert np.abs(w - wr.sum(axis=(0, 2))).max() <= 1e-9
    gg = g[a1] * np.conj(g[a2])
    assert np.abs(x / w - gg).max() <= 2e-6                                    # complex64 inputs
    # an explicit baseline index that reverses the baselines, zero weights and zero models are skipped
    bl = (nbl - 1 - np.arange(len(vis)) % nbl).astype(np.int32)
    wt2, model2 = wt.copy(), model.copy()
    wt2[::5] = 0
    model2[1::7] = 0
    x2, w2 = ref.gain_accumulate(vis, model2, wt2, nbl, bl_index=bl)
    keep = (wt2 > 0) & (model2 != 0)
    with np.errstate(divide="ignore", invalid="ignore"):
        r2 = np.where(keep, vis.astype(np.complex128) / model2.astype(np.complex128), 0) * wt2
    want = np.zeros((nbl, vis.shape[2]), complex)
    np.add.at(want, bl, r2.sum(axis=1))
    assert np.abs(x2 - want).max() <= 1e-9


def test_partitions_accumulate(ref):
    a1, a2, nbl, g, vis, model, wt = _setup(seed=4)
    x, w = ref.gain_accumulate(vis, model, wt, nbl)
    h = (len(vis) // (2 * nbl)) * nbl
    xa, wa = ref.gain_accumulate(vis[:h], model[:h], wt[:h], nbl)
    xa, wa = ref.gain_accumulate(vis[h:], model[h:], wt[h:], nbl, xsum=xa, wsum=wa)
    assert np.abs(xa - x).max() <= 1e-10 and np.abs(wa - w).max() <= 1e-10


def test_true_gains_are_a_fixed_point_and_noise_free_data_are_solved(ref):
    a1, a2, nbl, g, vis, model, wt = _setup(seed=5)
    nant, ncorr = g.shape
    gg = g[a1] * np.conj(g[a2])
    w = np.random.default_rng(1).uniform(1, 2, (nbl, ncorr))
    # exact X: one step of Eq. 20-21 from the true gains changes nothing, for any alpha
    for alpha in (0.3, 1.0):
        g1, it = ref.gain_solve(nant, a1, a2, gg * w, w, alpha, 0.0, 1, g)
        assert np.abs(g1 - g).max() <= 1e-13
    # from unit gains the iteration converges; the products g_i conj(g_j) are the data (the global phase is free)
    sol, it = ref.gain_solve(nant, a1, a2, gg * w, w, 0.5, 1e-13, 2000, np.ones((nant, ncorr)))
    assert it < 2000
    assert np.abs(sol[a1] * np.conj(sol[a2]) - gg).max() <= 1e-10
    # swapping the roles of a baseline's antennas must break it: X_ji = conj(X_ij)
    bad, _ = ref.gain_solve(nant, a2, a1, gg * w, w, 0.5, 1e-13, 2000, np.ones((nant, ncorr)))
    assert np.abs(bad[a1] * np.conj(bad[a2]) - gg).max() > 1e-3


def test_chi2_falls_and_the_exit_test_counts_iterations(ref):
    a1, a2, nbl, g, vis, model, wt = _setup(seed=6, noise=0.2)
    nant, ncorr = g.shape
    x, w = ref.gain_accumulate(vis, model, wt, nbl)
    X = x / w

    def chi2(gs):
        return float((w * np.abs(X - gs[a1] * np.conj(gs[a2])) ** 2).sum())
    gk = np.ones((nant, ncorr), complex)
    last = chi2(gk)
    for k in range(30):
        gk, it = ref.gain_solve(nant, a1, a2, x, w, 0.5, 0.0, 1, gk)
        assert it == 1
        now = chi2(gk)
        assert now <= last * (1 + 1e-12)
        last = now
    full, it = ref.gain_solve(nant, a1, a2, x, w, 0.5, 0.0, 30, np.ones((nant, ncorr)))
    assert it == 30 and np.abs(full - gk).max() <= 1e-12                      # 30 single steps = one call of 30
    _, it2 = ref.gain_solve(nant, a1, a2, x, w, 0.5, 1e-3, 1000, np.ones((nant, ncorr)))
    assert 1 < it2 < 1000

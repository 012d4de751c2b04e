"""Pins of the CPU oracle (oracle/lra_ref.c) against what the paper and the mathematics fix.

None of these tests needs a GPU and none compares the oracle with itself through the same formula:
each expected value is produced here by an independent route (numpy histogram, exact rationals,
Fourier-domain closed form, inner products).  Pin numbers follow DESIGN.md / SURVEY.md Sec. 8(c).
"""
import os
from fractions import Fraction

import numpy as np
import pytest

from paper_2508_17187_b200 import workloads as W

C_LIGHT = 299792458.0


# ---------------------------------------------------------------------------------------------------
# helpers that build small hand-made problems (inputs only)
# ---------------------------------------------------------------------------------------------------
def random_cf_table(rng, supports, os_, real_symmetric=False):
    ks = []
    for S in supports:
        n = S * os_
        k = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
        ks.append(k.astype(np.complex64))
    sup = np.array(supports, np.int32)
    sizes = np.array([k.size for k in ks], np.int64)
    off = np.concatenate([[0], np.cumsum(sizes)[:-1]]).astype(np.int64)
    return sup, off, np.concatenate([k.ravel() for k in ks]).astype(np.complex64), ks


def pixel_problem(rng, n, nx, ny, nchan=1, margin=0.0):
    """uvw in 'pixels' (freq = c so lambda = 1 m, scale = 1), positions uniform over the grid."""
    u = rng.uniform(-nx / 2 + margin, nx / 2 - margin, n)
    v = rng.uniform(-ny / 2 + margin, ny / 2 - margin, n)
    uvw = np.stack([u, v, np.zeros(n)], 1)
    freq = np.full(nchan, C_LIGHT) * (1.0 + 0.03 * np.arange(nchan))
    return uvw, freq


def cn(rng, shape):
    return (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)).astype(np.complex64)


def exact_index(u, freq, scale, n, os_):
    """Pixel and phase from exact rational arithmetic on the double inputs (no rounding anywhere)."""
    su = Fraction(freq) / Fraction(C_LIGHT) * Fraction(scale)
    px = Fraction(u) * su + n // 2
    t = px * os_ + Fraction(1, 2)
    P = t.numerator // t.denominator          # floor
    ix = (P + os_ // 2) // os_
    return ix, P - ix * os_


# ---------------------------------------------------------------------------------------------------
# P1 adjoint identity  <G(w o v), g> = <w o v, D g>   (D is the reverse operator of G)
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("nterms,ncorr,os_,supports", [(1, 1, 4, [5]), (2, 2, 8, [3, 7, 9]), (1, 4, 1, [5, 1]),
                                                        (2, 1, 20, [7])])
def test_p1_adjoint(ref, nterms, ncorr, os_, supports):
    rng = np.random.default_rng(101 + nterms * 7 + ncorr)
    nx, ny, n, nchan = 48, 40, 300, 3
    sup, off, data, _ = random_cf_table(rng, supports, os_)
    uvw, freq = pixel_problem(rng, n, nx, ny, nchan)
    cf_index = rng.integers(0, len(supports), (n, nchan)).astype(np.int32)
    vis, wt = cn(rng, (n, nchan, ncorr)), rng.uniform(0.5, 1, (n, nchan, ncorr)).astype(np.float32)
    tau = rng.uniform(-1, 1, (nchan, nterms)).astype(np.float32) if nterms > 1 else None
    p = ref.RefPlan(nx, ny, ncorr, nterms, os_, 0.9, -0.8, sup, off, data, tile=8)
    # G with weights applied to v: lhs = <G(w o tau o v), g>
    g = (rng.standard_normal((nterms, ncorr, ny, nx)) + 1j * rng.standard_normal((nterms, ncorr, ny, nx)))
    Gv, _ = p.grid(uvw, freq, cf_index, vis, wt, tau)
    Dg = p.degrid(uvw, freq, cf_index, g, tau)
    lhs = np.vdot(Gv, g)
    rhs = np.vdot(wt.astype(np.float64) * vis.astype(np.complex128), Dg)
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)
    assert abs(lhs) > 1.0  # the identity is not vacuous: some points are valid


# ---------------------------------------------------------------------------------------------------
# P2 1x1 CF  =>  weighted 2-D histogram of floor(px + 0.5)
# ---------------------------------------------------------------------------------------------------
def test_p2_nearest_pixel_histogram(ref):
    rng = np.random.default_rng(2)
    nx, ny, n = 64, 48, 5000
    uvw, freq = pixel_problem(rng, n, nx + 8, ny + 8)     # some points fall off the grid
    vis, wt = cn(rng, (n, 1, 1)), rng.uniform(0.5, 1, (n, 1, 1)).astype(np.float32)
    p = ref.RefPlan(nx, ny, 1, 1, 1, 1.0, 1.0, [1], [0], np.ones(1, np.complex64))
    g, sw = p.grid(uvw, freq, None, vis, wt)
    px = uvw[:, 0] * 1.0 + nx // 2
    py = uvw[:, 1] * 1.0 + ny // 2
    ix, iy = np.floor(px + 0.5).astype(int), np.floor(py + 0.5).astype(int)
    ok = (ix >= 0) & (ix < nx) & (iy >= 0) & (iy < ny)
    h = np.zeros((ny, nx), np.complex128)
    np.add.at(h, (iy[ok], ix[ok]), (wt[ok, 0, 0].astype(np.float64) * vis[ok, 0, 0].astype(np.complex128)))
    assert 0 < ok.sum() < n
    assert np.abs(g[0, 0] - h).max() <= 1e-14 * np.abs(h).max()
    assert abs(sw[0, 0] - wt[ok].astype(np.float64).sum()) <= 1e-12 * sw[0, 0]


def test_p2b_sum_of_weights_with_tau_counts_valid_points_only(ref):
    """sumwt[t][p] = sum over the VALID points of wt * tau (R4, R6, R11): points off the grid contribute nothing, and
    the Taylor weight multiplies the weight (dropping it, or counting invalid points, fails here)."""
    rng = np.random.default_rng(22)
    nx, ny, n, nchan, ncorr, nterms = 40, 36, 1500, 3, 2, 3
    uvw, freq = pixel_problem(rng, n, nx + 10, ny + 10, nchan)     # some points fall off the grid
    vis, wt = cn(rng, (n, nchan, ncorr)), rng.uniform(0.5, 1, (n, nchan, ncorr)).astype(np.float32)
    tau = rng.uniform(-1, 1, (nchan, nterms)).astype(np.float32)
    sup, off, data, _ = random_cf_table(rng, [3], 2)
    p = ref.RefPlan(nx, ny, ncorr, nterms, 2, 1.0, 1.0, sup, off, data)
    _, sw = p.grid(uvw, freq, None, vis, wt, tau)
    valid = (p.bin(uvw, freq, None)["key"] != np.uint64(2 ** 64 - 1)).reshape(n, nchan)
    assert 0 < valid.sum() < n * nchan
    want = np.einsum("rcp,ct->tp", wt.astype(np.float64) * valid[:, :, None], tau.astype(np.float64))
    assert np.abs(sw - want).max() <= 1e-12 * np.abs(want).max()
    # not vacuous: without tau, or with the invalid points, the sums differ
    assert np.abs(np.einsum("rcp,ct->tp", wt.astype(np.float64), tau.astype(np.float64)) - want).max() > 1e-3
    assert np.abs(np.einsum("rcp->p", wt.astype(np.float64) * valid[:, :, None])[None, :] - want).max() > 1e-3


# ---------------------------------------------------------------------------------------------------
# P3 sum(grid) = sum_k wt*tau*V * slabsum(cf, fy, fx), slab sums straight from K_cf by strided slicing
# ---------------------------------------------------------------------------------------------------
def test_p3_sum_of_grid(ref):
    rng = np.random.default_rng(3)
    nx = ny = 64
    os_, supports, n, nchan, nterms, ncorr = 6, [3, 5, 9], 800, 2, 2, 2
    sup, off, data, ks = random_cf_table(rng, supports, os_)
    uvw, freq = pixel_problem(rng, n, nx, ny, nchan, margin=6)
    cf_index = rng.integers(0, 3, (n, nchan)).astype(np.int32)
    vis, wt = cn(rng, (n, nchan, ncorr)), rng.uniform(0.5, 1, (n, nchan, ncorr)).astype(np.float32)
    tau = rng.uniform(-1, 1, (nchan, nterms)).astype(np.float32)
    p = ref.RefPlan(nx, ny, ncorr, nterms, os_, 1.0, 1.0, sup, off, data)
    g, sw = p.grid(uvw, freq, cf_index, vis, wt, tau)
    b = p.bin(uvw, freq, cf_index)
    assert b["n_valid"] == n * nchan
    # sum of weights with Taylor weights (R6, R11): sumwt[t][p] = sum_{r,c} wt[r][c][p] * tau[c][t], no CF factor
    want_sw = np.einsum("rcp,ct->tp", wt.astype(np.float64), tau.astype(np.float64))
    assert np.abs(sw - want_sw).max() <= 1e-12 * np.abs(want_sw).max()
    expect = np.zeros((nterms, ncorr), np.complex128)
    for k in range(n * nchan):
        r, c = divmod(k, nchan)
        K = ks[cf_index[r, c]].astype(np.complex128)
        sy, sx = os_ // 2 - 1 - int(b["fy"][k]), os_ // 2 - 1 - int(b["fx"][k])
        slab = K[sy::os_, sx::os_]
        assert slab.shape == (supports[cf_index[r, c]],) * 2
        for t in range(nterms):
            expect[t] += slab.sum() * float(tau[c, t]) * wt[r, c].astype(np.float64) * vis[r, c].astype(np.complex128)
    got = g.sum(axis=(2, 3))
    assert np.abs(got - expect).max() <= 1e-12 * np.abs(expect).max()


# ---------------------------------------------------------------------------------------------------
# P4 single visibility at an exact pixel centre; then moved by +1/os pixel: phase sign
# ---------------------------------------------------------------------------------------------------
def test_p4_single_visibility_patch_and_phase_sign(ref):
    S, os_, nx = 7, 20, 32
    K = W.ps_kernel(S, os_)
    h, c0 = 3, 3 * os_ + os_ // 2 - 1
    p = ref.RefPlan(nx, nx, 1, 1, os_, 1.0, 1.0, [S], [0], K.ravel())
    one, w1 = np.ones((1, 1, 1), np.complex64), np.ones((1, 1, 1), np.float32)
    X, Y = 20, 11
    freq = np.array([C_LIGHT])
    g, _ = p.grid(np.array([[X - nx // 2, Y - nx // 2, 0.0]]), freq, None, one, w1)
    patch = g[0, 0, Y - h:Y + h + 1, X - h:X + h + 1]
    expect = K[c0 - h * os_:c0 + h * os_ + 1:os_, c0 - h * os_:c0 + h * os_ + 1:os_].astype(np.complex128)
    assert np.array_equal(patch, expect)
    assert np.count_nonzero(g) == np.count_nonzero(expect)
    # +1/os pixel in u: the fx = +1 samples, i.e. kernel evaluated at (pixel - true position)
    g2, _ = p.grid(np.array([[X - nx // 2 + 1.0 / os_, Y - nx // 2, 0.0]]), freq, None, one, w1)
    patch2 = g2[0, 0, Y - h:Y + h + 1, X - h:X + h + 1]
    expect2 = K[c0 - h * os_:c0 + h * os_ + 1:os_, c0 - 1 - h * os_:c0 - 1 + h * os_ + 1:os_].astype(np.complex128)
    assert np.array_equal(patch2, expect2)
    xs = np.arange(-h, h + 1)
    cen1 = (patch.real.sum(0) * xs).sum() / patch.real.sum()
    cen2 = (patch2.real.sum(0) * xs).sum() / patch2.real.sum()
    assert abs(cen1) < 1e-3 and cen2 > cen1 + 0.5 / os_     # centroid follows the visibility toward +x
    # same in v
    g3, _ = p.grid(np.array([[X - nx // 2, Y - nx // 2 - 2.0 / os_, 0.0]]), freq, None, one, w1)
    patch3 = g3[0, 0, Y - h:Y + h + 1, X - h:X + h + 1]
    expect3 = K[c0 + 2 - h * os_:c0 + 2 + h * os_ + 1:os_, c0 - h * os_:c0 + h * os_ + 1:os_].astype(np.complex128)
    assert np.array_equal(patch3, expect3)


# ---------------------------------------------------------------------------------------------------
# P5 Hermitian symmetry with a real even CF
# ---------------------------------------------------------------------------------------------------
def test_p5_hermitian(ref):
    rng = np.random.default_rng(5)
    S, os_, nx, n = 7, 8, 64, 400
    K = W.ps_kernel(S, os_)
    # positions on the oversampled lattice with phase != -os/2, plus a jitter far from rounding ties
    Px = rng.integers(-20 * os_, 20 * os_, n)
    Py = rng.integers(-20 * os_, 20 * os_, n)
    keep = (((Px + os_ // 2) % os_) != 0) & (((Py + os_ // 2) % os_) != 0)   # phase -os/2 <=> (P + os/2) % os == 0
    Px, Py = Px[keep], Py[keep]
    jit = rng.uniform(-0.2, 0.2, (2, len(Px))) / os_
    u, v = Px / os_ + jit[0], Py / os_ + jit[1]
    uvw = np.concatenate([np.stack([u, v, 0 * u], 1), np.stack([-u, -v, 0 * u], 1)])
    vis = cn(rng, (len(u), 1, 1))
    vis = np.concatenate([vis, np.conj(vis)])
    wt1 = rng.uniform(0.5, 1, (len(u), 1, 1)).astype(np.float32)
    wt = np.concatenate([wt1, wt1])
    p = ref.RefPlan(nx, nx, 1, 1, os_, 1.0, 1.0, [S], [0], K.ravel())
    g, _ = p.grid(uvw, np.array([C_LIGHT]), None, vis, wt)
    g = g[0, 0]
    a = g[1:, 1:]
    b = np.conj(g[1:, 1:][::-1, ::-1])       # g[ny - y][nx - x]
    assert np.abs(a - b).max() <= 1e-13 * np.abs(g).max()
    assert np.abs(g).max() > 0.1


# ---------------------------------------------------------------------------------------------------
# P6 tiny-grid closed form: DFT of the grid == sum_k wt V_k e^{2 pi i u~_k l / N} c^_{cf,f_k}(l, m),
# with positions/phases from exact rationals and the phase's taps picked by strided slicing.
# ---------------------------------------------------------------------------------------------------
def test_p6_closed_form_dft(ref):
    rng = np.random.default_rng(6)
    N, os_, supports, n, nchan = 24, 4, [3, 5], 60, 2
    sup, off, data, ks = random_cf_table(rng, supports, os_)          # complex, NOT separable
    su_scale, sv_scale = 0.93, -1.07
    uvw, freq = pixel_problem(rng, n, N - 8, N - 8, nchan)
    cf_index = rng.integers(0, 2, (n, nchan)).astype(np.int32)
    vis, wt = cn(rng, (n, nchan, 1)), rng.uniform(0.5, 1, (n, nchan, 1)).astype(np.float32)
    p = ref.RefPlan(N, N, 1, 1, os_, su_scale, sv_scale, sup, off, data)
    g, _ = p.grid(uvw, freq, cf_index, vis, wt)
    pix = np.arange(N) - N // 2
    lm = np.arange(N) - N // 2
    E = np.exp(2j * np.pi * np.outer(lm, pix) / N)                    # [l, pix]
    lhs = E @ g[0, 0] @ E.T                                          # [m, l]
    rhs = np.zeros((N, N), np.complex128)
    nvalid = 0
    for r in range(n):
        for c in range(nchan):
            ix, fx = exact_index(uvw[r, 0], freq[c], su_scale, N, os_)
            iy, fy = exact_index(uvw[r, 1], freq[c], sv_scale, N, os_)
            S = supports[cf_index[r, c]]
            h = (S - 1) // 2
            if ix - h < 0 or ix + h > N - 1 or iy - h < 0 or iy + h > N - 1:
                continue
            nvalid += 1
            K = ks[cf_index[r, c]].astype(np.complex128)
            Cf = K[os_ // 2 - 1 - fy::os_, os_ // 2 - 1 - fx::os_]    # the S x S taps of phase (fy, fx)
            tap = np.arange(-h, h + 1)
            ex = np.exp(2j * np.pi * np.outer(lm, tap - Fraction(fx, os_).__float__()) / N)   # [l, i]
            ey = np.exp(2j * np.pi * np.outer(lm, tap - Fraction(fy, os_).__float__()) / N)   # [m, j]
            chat = ey @ Cf @ ex.T                                                            # [m, l]
            ut, vt = ix + fx / os_ - N // 2, iy + fy / os_ - N // 2
            ph = np.outer(np.exp(2j * np.pi * vt * lm / N), np.exp(2j * np.pi * ut * lm / N))
            rhs += float(wt[r, c, 0]) * complex(vis[r, c, 0]) * ph * chat
    assert nvalid > 20
    assert np.abs(lhs - rhs).max() <= 1e-11 * np.abs(rhs).max()


# ---------------------------------------------------------------------------------------------------
# P7 point source: grid, direct DFT, divide by the image of the CF taper  (north_star's analytic check)
# ---------------------------------------------------------------------------------------------------
def test_p7_point_source(ref):
    rng = np.random.default_rng(7)
    N, S, os_, n = 32, 7, 16, 500
    K = W.ps_kernel(S, os_)
    c0 = 3 * os_ + os_ // 2 - 1
    uvw, freq = pixel_problem(rng, n, N, N, 1, margin=4)
    l0, m0 = 5, -3
    vis = np.exp(-2j * np.pi * (uvw[:, 0] * l0 + uvw[:, 1] * m0) / N).astype(np.complex64).reshape(n, 1, 1)
    wt = rng.uniform(0.5, 1, (n, 1, 1)).astype(np.float32)
    p = ref.RefPlan(N, N, 1, 1, os_, 1.0, 1.0, [S], [0], K.ravel())
    g, sw = p.grid(uvw, freq, None, vis, wt)
    lm = np.arange(N) - N // 2
    E = np.exp(2j * np.pi * np.outer(lm, lm) / N)
    img = E @ g[0, 0] @ E.T
    offs = (np.arange(S * os_) - c0) / os_
    Et = np.exp(2j * np.pi * np.outer(lm, offs) / N)
    taper = (Et @ K.astype(np.complex128) @ Et.T) / os_ ** 2            # DTFT of the oversampled kernel
    inner = slice(N // 2 - 10, N // 2 + 11)
    corr = (img / taper)[inner, inner]
    peak = np.unravel_index(np.abs(corr).argmax(), corr.shape)
    assert (peak[0] - 10, peak[1] - 10) == (m0, l0)
    amp = corr[peak]
    # amplitude within the oversampling quantisation error O((pi l/(N os))^2) plus aliasing of the taper
    assert abs(amp - sw[0, 0]) <= 5e-3 * sw[0, 0]
    assert abs(amp.imag) <= 5e-3 * sw[0, 0]


# ---------------------------------------------------------------------------------------------------
# P8 partition invariance and permutation invariance (sums are independent/partitionable)
# ---------------------------------------------------------------------------------------------------
def test_p8_partition_and_permutation(ref):
    wl = W.make_workload(W.small_config(3))
    p = ref.plan_for(wl)
    sl = slice(0, 351 * 6)
    uvw, cfi, vis, wt = wl.uvw[sl], wl.cf_index[sl], wl.vis[sl], wl.wt[sl]
    g, sw = p.grid(uvw, wl.freq, cfi, vis, wt)
    h = len(uvw) // 3
    ga, swa = p.grid(uvw[:h], wl.freq, cfi[:h], vis[:h], wt[:h])
    gb, swb = p.grid(uvw[h:], wl.freq, cfi[h:], vis[h:], wt[h:])
    scale = np.abs(g).max()
    assert np.abs(ga + gb - g).max() <= 1e-13 * scale
    assert np.abs(swa + swb - sw).max() <= 1e-12 * sw.max()
    perm = np.random.default_rng(8).permutation(len(uvw))
    gp, _ = p.grid(uvw[perm], wl.freq, cfi[perm], vis[perm], wt[perm])
    assert np.abs(gp - g).max() <= 1e-13 * scale
    # accumulate-into semantics: gridding B on top of A's grid
    gab, _ = p.grid(uvw[h:], wl.freq, cfi[h:], vis[h:], wt[h:], grid=ga.copy())
    assert np.abs(gab - g).max() <= 1e-13 * scale
    # thread count does not change a single bit (row-band scheme)
    g1, _ = p.grid(uvw, wl.freq, cfi, vis, wt, nthreads=1)
    g3, _ = p.grid(uvw, wl.freq, cfi, vis, wt, nthreads=3)
    assert np.array_equal(g1, g3) and np.array_equal(g1, g)


# ---------------------------------------------------------------------------------------------------
# P9 bin: exact rational indices on cfg1; perm/keys/tile_start structure, both sort modes
# ---------------------------------------------------------------------------------------------------
def test_p9_bin_exact_rational_cfg1(ref):
    wl = W.make_workload(W.full_config(1))
    p = ref.plan_for(wl, tile=32)
    b = p.bin(wl.uvw, wl.freq, None)
    n = wl.cfg.npoints
    h = 3
    nvalid = 0
    for k in range(n):
        ix, fx = exact_index(wl.uvw[k, 0], wl.freq[0], wl.scale_u, 256, 20)
        iy, fy = exact_index(wl.uvw[k, 1], wl.freq[0], wl.scale_v, 256, 20)
        valid = ix - h >= 0 and ix + h <= 255 and iy - h >= 0 and iy + h <= 255
        if valid:
            nvalid += 1
            assert (b["ix"][k], b["iy"][k], b["fx"][k], b["fy"][k]) == (ix, iy, fx, fy)
            assert b["key"][k] == (iy // 32) * 8 + ix // 32
        else:
            assert b["key"][k] == 2 ** 64 - 1 and b["ix"][k] == -1 and b["iy"][k] == -1
    assert nvalid == b["n_valid"] == n     # the 0.4 N disk keeps every footprint on the grid


@pytest.mark.parametrize("mode,Tx,Ty", [(0, 32, 32), (1, 32, 32), (1, 8, 64), (0, 16, 8)])
def test_p9_bin_structure(ref, mode, Tx, Ty):
    wl = W.make_workload(W.small_config(3))
    # push some points off the grid / to bad CFs / to NaN so that invalid handling is exercised
    uvw = wl.uvw.copy()
    cfi = wl.cf_index.copy()
    uvw[5] = [3.0e5, -2.0e5, 10.0]
    uvw[17, 0] = np.nan
    uvw[23, 1] = np.inf
    cfi[40, 1] = -1
    cfi[41, 2] = wl.cfg.n_cf
    p = ref.plan_for(wl, sort_mode=mode, tile=Ty, tile_x=Tx)      # R5: tiles Tx wide (u) by Ty tall (v)
    b = p.bin(uvw, wl.freq, cfi)
    n = wl.cfg.npoints
    key, perm, ts = b["key"], b["perm"], b["tile_start"]
    valid = key != np.uint64(2 ** 64 - 1)
    assert b["n_valid"] == valid.sum() < n
    assert not valid[5 * 4:6 * 4].any() and not valid[17 * 4] and not valid[23 * 4]
    assert not valid[40 * 4 + 1] and not valid[41 * 4 + 2] and valid[40 * 4]
    assert np.array_equal(np.sort(perm), np.nonzero(valid)[0])                 # permutation of the valid set
    ks = key[perm]
    assert (np.diff(ks.astype(np.int64)) >= 0).all()                           # keys non-decreasing
    same = np.diff(ks.astype(np.int64)) == 0
    assert (np.diff(perm.astype(np.int64))[same] > 0).all()                    # stable: equal keys ascending k
    # keys from the exported indices
    os_ = wl.cfg.oversampling
    ntx = (wl.cfg.nx + Tx - 1) // Tx
    tile = (b["iy"][valid] // Ty).astype(np.uint64) * np.uint64(ntx) + (b["ix"][valid] // Tx).astype(np.uint64)
    if mode == 0:
        expect = tile
    else:
        cf = cfi.reshape(-1)[valid].astype(np.uint64)
        expect = ((tile * np.uint64(wl.cfg.n_cf) + cf) * np.uint64(os_) + (b["fy"][valid].astype(np.int64) + os_ // 2).astype(np.uint64)) \
            * np.uint64(os_) + (b["fx"][valid].astype(np.int64) + os_ // 2).astype(np.uint64)
    assert np.array_equal(key[valid], expect)
    # tile_start: searchsorted over tile ids along perm
    tile_sorted = (b["iy"][perm] // Ty).astype(np.int64) * ntx + (b["ix"][perm] // Tx).astype(np.int64)
    ntiles = ntx * ((wl.cfg.ny + Ty - 1) // Ty)
    assert len(ts) == ntiles + 1
    assert np.array_equal(ts, np.searchsorted(tile_sorted, np.arange(ntiles + 1), side="left").astype(np.uint32))
    assert ts[-1] == b["n_valid"]
    # the rational check on a sample of points of this (scaled, multi-channel) problem
    rng = np.random.default_rng(9)
    for k in rng.choice(np.nonzero(valid)[0], 300, replace=False):
        r, c = divmod(int(k), wl.cfg.nchan)
        ix, fx = exact_index(uvw[r, 0], wl.freq[c], wl.scale_u, wl.cfg.nx, os_)
        iy, fy = exact_index(uvw[r, 1], wl.freq[c], wl.scale_v, wl.cfg.ny, os_)
        assert (b["ix"][k], b["iy"][k], b["fx"][k], b["fy"][k]) == (ix, iy, fx, fy)


def test_invalid_points_contribute_nothing_and_degrid_zero(ref):
    rng = np.random.default_rng(11)
    nx, S, os_ = 32, 5, 4
    sup, off, data, _ = random_cf_table(rng, [S], os_)
    uvw = np.array([[0.0, 0.0, 0], [15.0, 0.0, 0], [np.nan, 1.0, 0], [-16.2, 3.0, 0], [2.0, -13.4, 0], [1e300, 0, 0]])
    vis, wt = cn(rng, (6, 1, 1)), np.ones((6, 1, 1), np.float32)
    p = ref.RefPlan(nx, nx, 1, 1, os_, 1.0, 1.0, sup, off, data)
    b = p.bin(uvw, np.array([C_LIGHT]))
    # x = 15 -> pixel 31, footprint leaves the grid (R4); y = -13.4 -> pixel 3 (2.6 -> round 3), h = 2: valid
    assert list(b["key"] != np.uint64(2 ** 64 - 1)) == [True, False, False, False, True, False]
    g, sw = p.grid(uvw, np.array([C_LIGHT]), None, vis, wt)
    g_valid, _ = p.grid(uvw[[0, 4]], np.array([C_LIGHT]), None, vis[[0, 4]], wt[[0, 4]])
    assert np.array_equal(g, g_valid) and sw[0, 0] == 2.0
    G = rng.standard_normal((1, 1, nx, nx)) + 0j
    v = p.degrid(uvw, np.array([C_LIGHT]), None, G)
    assert (v[[1, 2, 3, 5]] == 0).all() and (v[[0, 4]] != 0).all()
    vin = cn(rng, (6, 1, 1))
    res = p.degrid(uvw, np.array([C_LIGHT]), None, G, vis_in=vin)
    assert np.allclose(res, vin.astype(np.complex128) - v, rtol=0, atol=1e-15)
    # empty input
    g0, sw0 = p.grid(np.zeros((0, 3)), np.array([C_LIGHT]), None, np.zeros((0, 1, 1), np.complex64), np.zeros((0, 1, 1), np.float32))
    assert not g0.any() and not sw0.any()
    assert p.bin(np.zeros((0, 3)), np.array([C_LIGHT]))["n_valid"] == 0


def test_sampled_outputs_match_full_oracle(ref):
    """grid_pixels / degrid_points (used for full-size parity) against the full oracle loops."""
    wl = W.make_workload(W.small_config(5))
    p = ref.plan_for(wl)
    g, _ = p.grid(wl.uvw, wl.freq, wl.cf_index, wl.vis, wl.wt, wl.tau)
    rng = np.random.default_rng(12)
    pix = np.stack([rng.integers(0, 2, 64), rng.integers(0, 2, 64), rng.integers(300, 724, 64), rng.integers(300, 724, 64)], 1)
    got = p.grid_pixels(wl.uvw, wl.freq, wl.cf_index, wl.vis, wl.wt, wl.tau, pix)
    want = g[pix[:, 0], pix[:, 1], pix[:, 2], pix[:, 3]]
    assert np.abs(got - want).max() <= 1e-12 * np.abs(g).max() and np.abs(want).max() > 0
    g32 = g.astype(np.complex64)
    sel = rng.choice(wl.cfg.npoints, 50, replace=False)
    v = p.degrid(wl.uvw, wl.freq, wl.cf_index, g32.astype(np.complex128), wl.tau, vis_in=wl.vis)
    got = p.degrid_points(wl.uvw, wl.freq, wl.cf_index, g32, wl.tau, wl.vis, sel)
    assert np.abs(got - v.reshape(-1, 2)[sel]).max() <= 1e-12 * np.abs(v).max()


# ---------------------------------------------------------------------------------------------------
# P10 generator sanity (workloads.py, not the library) and Table 1
# ---------------------------------------------------------------------------------------------------
def test_p10_w_kernel_sanity():
    S, os_ = 9, 8
    c0 = 4 * os_ + os_ // 2 - 1
    k0 = W.w_kernel(S, os_, S, 0.0, 0.01).astype(np.complex128)
    kw = W.w_kernel(S, os_, S, 3.0e4, 0.01).astype(np.complex128)
    ps = W.ps_kernel(S, os_).astype(np.complex128)
    # w = 0 plane: real (Hermitian image) and the same function as the PS kernel up to the raster's aliasing
    assert np.abs(k0.imag).max() <= 1e-3 * np.abs(k0).max()   # raster [-1, 1) is one sample short of symmetric
    assert np.abs(k0 - ps).max() <= 1e-4 * np.abs(ps).max()
    # even: K(-x) = K(x) about the centre sample c0 (for every w)
    n = 2 * c0 + 1
    for k in (k0, kw):
        sub = k[:n, :n]
        assert np.abs(sub - sub[::-1, ::-1]).max() <= 1e-3 * np.abs(k).max()
    assert np.abs(kw.imag).max() > 1e-3 * np.abs(kw).max()
    # R12 normalisation
    for k in (k0, kw, ps):
        assert abs(k.sum() / os_ ** 2 - 1.0) < 1e-5


def test_prolate_is_the_dominant_band_limited_eigenfunction():
    """The generator's psi against its integral definition: K psi = lambda psi with lambda -> 1 (the
    dominant eigenvalue of the band-limiting operator), psi even, positive, nodeless, concentrated."""
    for S in (7, 9, 33):
        psi = W.Prolate(S)
        lam, resid = psi.integral_residual()
        assert 1.0 - 1e-6 < lam < 1.0 + 1e-12 and resid < 1e-10
        x = np.linspace(-1, 1, 201)
        v = psi(x)
        assert (v > -1e-12).all() and np.abs(v - v[::-1]).max() < 1e-12 and v.argmax() == 100
        assert (np.diff(v[100:]) < 1e-12).all()
        assert v[0] / v[100] < 1e-3


def test_table1_rows_cover_the_generator_kinds():
    rows = [l.split() for l in open(os.path.join(os.path.dirname(__file__), "golden", "table1_cf_terms.txt")) if not l.startswith("#")]
    cf_of = {(r[1], r[2], r[3]): r[4] for r in rows}
    assert cf_of[("OFF", "ON", "OFF")] == "PS"          # cfg1, cfg2: kind "ps"
    assert cf_of[("OFF", "ON", "ON")] == "PS*W"         # cfg3, cfg5: kind "w"
    assert cf_of[("ON", "ON", "ON")] == "PS*A*W"        # cfg4: kind "aw"
    assert {W.full_config(i).cf_kind for i in range(1, 6)} == {"ps", "w", "aw"}


def test_workload_shapes_match_baseline_configs():
    c1, c2, c3, c4, c5 = (W.full_config(i) for i in range(1, 6))
    assert c1.npoints == 21060 and (c1.nx, c1.oversampling, c1.s_min) == (256, 20, 7)
    assert (c2.nrow, c2.nchan, c2.ncorr, c2.npoints) == (5054400, 64, 2, 323481600)
    assert (c3.nrow, c3.nchan, c3.npoints, c3.nx, c3.n_cf) == (2527200, 16, 40435200, 8192, 128)
    assert (c4.ncorr, c4.n_cf, c4.nx) == (4, 1024, 4096)
    assert c5.npoints == 6497712 and c5.nterms == 2
    assert W.w_plane_support(c3, 0) == 9 and W.w_plane_support(c3, 127) == 65
    assert W.w_plane_support(c4, 0) == 17 and W.w_plane_support(c4, 31) == 49
    wl = W.make_workload(W.small_config(4))
    assert wl.cf_index.max() < wl.cfg.n_cf and wl.cf_index.min() >= 0 and len(wl.cf.support) == wl.cfg.n_cf
    assert (wl.uvw[:, 2] >= 0).all()                      # R8 flip

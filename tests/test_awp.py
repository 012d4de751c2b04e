"""Pins of the general-kernel oracle (lra_ref_grid_awp / lra_ref_degrid_awp / lra_ref_phase_gradient in oracle/lra_ref.c):
Eq. 27's pointing term (Table 2) and per-element Mueller CFs.  CPU only."""
import cmath
import math

import numpy as np

from oracle import lra_ref

C_LIGHT = 299792458.0


def _table(rng, supports, os_):
    ks = [(rng.normal(size=(S * os_, S * os_)) + 1j * rng.normal(size=(S * os_, S * os_))).astype(np.complex64) for S in supports]
    sup = np.array(supports, dtype=np.int32)
    sizes = np.array([k.size for k in ks], dtype=np.int64)
    off = np.concatenate([[0], np.cumsum(sizes)[:-1]]).astype(np.int64)
    return sup, off, np.concatenate([k.ravel() for k in ks])


def _setup(seed=1, nx=48, ny=40, ngrid=2, nterms=1, os_=2, supports=(3, 5, 7), nrow=30, nchan=3, ncorr_vis=2):
    rng = np.random.default_rng(seed)
    sup, off, data = _table(rng, supports, os_)
    su, sv = 0.011, -0.013                                  # pixels per wavelength
    plan = lra_ref.RefPlan(nx, ny, ngrid, nterms, os_, su, sv, sup, off, data, tile=8, tile_x=8)
    freq = np.linspace(1.0e9, 1.2e9, nchan)
    lam = C_LIGHT / freq.max()
    uvw = np.zeros((nrow, 3))
    uvw[:, 0] = rng.uniform(-0.3, 0.3, nrow) * nx / abs(su) * lam
    uvw[:, 1] = rng.uniform(-0.3, 0.3, nrow) * ny / abs(sv) * lam
    vis = (rng.normal(size=(nrow, nchan, ncorr_vis)) + 1j * rng.normal(size=(nrow, nchan, ncorr_vis))).astype(np.complex64)
    wt = rng.uniform(0.5, 1.5, size=(nrow, nchan, ncorr_vis)).astype(np.float32)
    cfi = [rng.integers(0, len(supports), size=(nrow, nchan)).astype(np.int32) for _ in range(4)]
    return rng, plan, uvw, freq, vis, wt, cfi


def test_reduces_to_the_plain_oracle():
    """Diagonal elements sharing one kernel index and no pointing term: the pinned lra_ref_grid / lra_ref_degrid."""
    rng, plan, uvw, freq, vis, wt, cfi = _setup()
    g, sw = plan.grid_awp(uvw, freq, [(0, 0), (1, 1)], [cfi[0], cfi[0]], vis, wt)
    g0, sw0 = plan.grid(uvw, freq, cfi[0], vis, wt, nthreads=1)
    np.testing.assert_allclose(g, g0, rtol=0, atol=1e-12 * np.abs(g0).max())
    np.testing.assert_allclose(sw, sw0, rtol=1e-14)
    model = rng.normal(size=g.shape) + 1j * rng.normal(size=g.shape)
    v = plan.degrid_awp(uvw, freq, [(0, 0), (1, 1)], [cfi[0], cfi[0]], 2, model, vis_in=vis)
    v0 = plan.degrid(uvw, freq, cfi[0], model, vis_in=vis, nthreads=1)
    np.testing.assert_allclose(v, v0, rtol=0, atol=1e-12 * np.abs(v0).max())


def test_pointing_offset_of_whole_pixels_shifts_the_image():
    """e^{2 pi i dl u_X} with dl = kx scale_u / nx is e^{2 pi i kx (X - nx/2)/nx}: by the shift theorem of the centred DFT
    (oracle image(), pinned against numpy's FFT) the dirty image moves by kx pixels, circularly: I_po[l] = I_0[l + kx].
    Pins the sign, the scale and the origin pixel of u_X, v_Y."""
    rng, plan, uvw, freq, vis, wt, cfi = _setup(seed=2)
    kx, ky = 3, -5
    po = [[1.0, kx * plan.d.scale_u / plan.nx, ky * plan.d.scale_v / plan.ny]]
    g, _ = plan.grid_awp(uvw, freq, [(0, 0), (1, 1)], [cfi[0], cfi[1]], vis, wt, po_table=po)
    g0, _ = plan.grid_awp(uvw, freq, [(0, 0), (1, 1)], [cfi[0], cfi[1]], vis, wt)
    img, img0 = lra_ref.image(g), lra_ref.image(g0)
    np.testing.assert_allclose(img, np.roll(img0, (-ky, -kx), axis=(-2, -1)), rtol=0, atol=1e-9 * np.abs(img0).max())
    assert np.abs(img - img0).max() > 1e-3 * np.abs(img0).max()


def test_single_tap_closed_form_and_row_table():
    """S = 1: the grid pixel under the point receives c f e^{2 pi i (dl u_X + dm v_Y)} wt v, with the row's own table entry."""
    nx = ny = 32
    su = sv = 0.02
    c = np.array([0.75 - 0.5j], dtype=np.complex64)
    plan = lra_ref.RefPlan(nx, ny, 1, 1, 1, su, sv, [1], [0], c, tile=8, tile_x=8)
    freq = np.array([C_LIGHT])                               # 1 m wavelength: u in wavelengths = metres
    uvw = np.array([[100.0, -250.0, 0.0], [-300.0, 50.0, 0.0]])
    vis = np.array([[[1.5 + 2.0j]], [[-0.5 + 1.0j]]], dtype=np.complex64)
    wt = np.array([[[2.0]], [[0.25]]], dtype=np.float32)
    po = [[0.9, 1.0e-3, -2.0e-3], [0.6, -4.0e-3, 0.5e-3]]
    g, sw = plan.grid_awp(uvw, freq, [(0, 0)], [None], vis, wt, po_table=po, po_index=[1, 0])
    for r, e in ((0, 1), (1, 0)):
        X, Y = nx // 2 + round(uvw[r, 0] * su), ny // 2 + round(uvw[r, 1] * sv)
        f, dl, dm = po[e]
        want = complex(c[0]) * f * cmath.exp(2j * math.pi * (dl * (X - nx // 2) / su + dm * (Y - ny // 2) / sv)) * float(wt[r, 0, 0]) * complex(vis[r, 0, 0])
        assert abs(g[0, 0, Y, X] - want) < 1e-13
    assert abs(sw[0, 0] - 2.25) < 1e-15                      # sumwt: no f, no CF (R6)
    assert np.count_nonzero(g) == 2


def test_mueller_element_is_a_plain_gridding_of_one_correlation():
    """Element (p, q) with its own kernel index: the pinned plain oracle on column q of the data with those indices lands on
    plane p; only diagonal elements add to sumwt."""
    rng, plan, uvw, freq, vis, wt, cfi = _setup(seed=3)
    elems = [(0, 0), (1, 1), (0, 1), (1, 0)]
    g, sw = plan.grid_awp(uvw, freq, elems, cfi, vis, wt)
    one = lra_ref.RefPlan(plan.nx, plan.ny, 1, 1, plan.os, plan.d.scale_u, plan.d.scale_v, plan.cf_support, plan.cf_offset,
                          plan.cf_data, tile=8, tile_x=8)
    want = np.zeros_like(g)
    want_sw = np.zeros_like(sw)
    for (p, q), ci in zip(elems, cfi):
        ge, swe = one.grid(uvw, freq, ci, vis[:, :, q:q + 1], wt[:, :, q:q + 1], nthreads=1)
        want[0, p] += ge[0, 0]
        if p == q:
            want_sw[0, p] += swe[0, 0]
    np.testing.assert_allclose(g, want, rtol=0, atol=1e-12 * np.abs(want).max())
    np.testing.assert_allclose(sw, want_sw, rtol=1e-14)


def test_degridding_is_the_adjoint_of_gridding():
    """D uses conj(c): <G v, g> = <v, D g> for unit weights, with the pointing term and off-diagonal elements ON."""
    rng, plan, uvw, freq, vis, wt, cfi = _setup(seed=4)
    elems = [(0, 0), (1, 1), (0, 1)]
    po = [[0.8, 2.0e-3, -1.0e-3], [1.0, 0.0, 0.0], [0.5, -3.0e-3, 4.0e-3]]
    pi = rng.integers(0, 3, size=len(uvw)).astype(np.int32)
    one = np.ones_like(wt)
    Gv, _ = plan.grid_awp(uvw, freq, elems, cfi[:3], vis, one, po_table=po, po_index=pi)
    g = rng.normal(size=Gv.shape) + 1j * rng.normal(size=Gv.shape)
    Dg = plan.degrid_awp(uvw, freq, elems, cfi[:3], 2, g, po_table=po, po_index=pi)
    lhs = np.vdot(Gv, g)
    rhs = np.vdot(vis.astype(np.complex128), Dg)
    assert abs(lhs - rhs) < 1e-10 * abs(lhs)


def test_phase_gradient_on_a_grid_equals_the_per_tap_factor():
    """A group of points that share one table entry: the factor depends on the grid pixel only, so it can be applied to the
    group's grid once (Table 2: mosaic imaging, one entry per pointing); conjugate = the degridding side."""
    rng, plan, uvw, freq, vis, wt, cfi = _setup(seed=5)
    f, dl, dm = 0.7, 1.5e-3, -2.5e-3
    elems = [(0, 0), (1, 1)]
    g0, _ = plan.grid_awp(uvw, freq, elems, cfi[:2], vis, wt)
    g1, _ = plan.grid_awp(uvw, freq, elems, cfi[:2], vis, wt, po_table=[[f, dl, dm]])
    np.testing.assert_allclose(plan.phase_gradient(g0, f, dl, dm), g1, rtol=0, atol=1e-12 * np.abs(g1).max())
    acc = plan.phase_gradient(g0, f, dl, dm, dst=g0)
    np.testing.assert_allclose(acc, g0 + g1, rtol=0, atol=1e-12 * np.abs(g1).max())
    model = rng.normal(size=g0.shape) + 1j * rng.normal(size=g0.shape)
    v1 = plan.degrid_awp(uvw, freq, elems, cfi[:2], 2, model, po_table=[[f, dl, dm]])
    v0 = plan.degrid_awp(uvw, freq, elems, cfi[:2], 2, plan.phase_gradient(model, f, dl, dm, conjugate=True))
    np.testing.assert_allclose(v1, v0, rtol=0, atol=1e-12 * np.abs(v0).max())
    c = plan.phase_gradient(g0, f, dl, dm)
    assert abs(c[0, 1, plan.ny // 2, plan.nx // 2] - f * g0[0, 1, plan.ny // 2, plan.nx // 2]) < 1e-15 + 1e-15 * abs(g0).max()


def test_f_scales_the_kernel_only():
    rng, plan, uvw, freq, vis, wt, cfi = _setup(seed=6)
    g1, sw1 = plan.grid_awp(uvw, freq, [(0, 0)], [cfi[0]], vis, wt, po_table=[[1.0, 1e-3, 2e-3]])
    gh, swh = plan.grid_awp(uvw, freq, [(0, 0)], [cfi[0]], vis, wt, po_table=[[0.5, 1e-3, 2e-3]])
    np.testing.assert_allclose(gh, 0.5 * g1, rtol=0, atol=1e-13 * np.abs(g1).max())
    np.testing.assert_array_equal(sw1, swh)

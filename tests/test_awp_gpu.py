"""GPU parity of the Eq. 27 terms and the Mueller elements (lra_grid_po, lra_degrid_po, lra_phase_gradient,
lra_grid_mueller, lra_degrid_mueller) against lra_ref_grid_awp / lra_ref_degrid_awp /
lra_ref_phase_gradient, element by element, north_star's tolerances (relative L2 <= 1e-5, max abs <= 1e-4 max|.|).
No oracle input comes from the CUDA path."""
import numpy as np
import pytest

from paper_2508_17187_b200 import workloads as W

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2508_17187_b200 import binding
    binding.lib()
    return binding


def dev(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


def assert_close(got, want, what):
    want = np.asarray(want, dtype=np.complex128)
    got = np.asarray(got, dtype=np.complex128)
    scale = np.abs(want).max()
    assert scale > 0, what
    l2 = np.linalg.norm((got - want).ravel()) / np.linalg.norm(want.ravel())
    mx = np.abs(got - want).max()
    assert l2 <= 1e-5, f"{what}: relative L2 {l2:.3e}"
    assert mx <= 1e-4 * scale, f"{what}: max abs {mx:.3e} vs scale {scale:.3e}"


def _po_table(wl, n_po, seed):
    """Offsets of up to a few arcminutes: tens of turns of phase across the uv plane of the small configs."""
    rng = np.random.default_rng(seed)
    t = np.empty((n_po, 3))
    t[:, 0] = rng.uniform(0.6, 1.0, n_po)
    t[:, 1:] = rng.uniform(-1.0e-3, 1.0e-3, size=(n_po, 2))
    t[0] = [1.0, 0.0, 0.0]
    return t


def _plans(B, ref, wl, ncorr=None, nterms=None):
    c = wl.cfg
    ncorr = c.ncorr if ncorr is None else ncorr
    nterms = c.nterms if nterms is None else nterms
    plan = B.lra_plan_create(c.nx, c.ny, ncorr, nterms, c.oversampling, wl.scale_u, wl.scale_v, wl.cf.support, wl.cf.offset,
                             wl.cf.data)
    rp = ref.RefPlan(c.nx, c.ny, ncorr, nterms, c.oversampling, wl.scale_u, wl.scale_v, wl.cf.support, wl.cf.offset, wl.cf.data,
                     tile=8, sort_mode=1, tile_x=8)
    return plan, rp


@pytest.mark.parametrize("n", [3, 4, 5])
def test_grid_and_degrid_with_per_row_pointing_terms(B, ref, n):
    """Table 2 'with PO correction': every row has its own (f, dl, dm); direct kernels."""
    wl = W.make_workload(W.small_config(n))
    c = wl.cfg
    plan, rp = _plans(B, ref, wl)
    try:
        B.lra_bin(plan, dev(wl.uvw), wl.freq, dev(wl.cf_index))
        po = _po_table(wl, 37, n)
        pi = np.random.default_rng(50 + n).integers(0, len(po), size=len(wl.uvw)).astype(np.int32)
        elems = [(p, p) for p in range(c.ncorr)]
        cfis = [wl.cf_index] * c.ncorr
        g = torch.zeros((c.nterms, c.ncorr, c.ny, c.nx), dtype=torch.complex64, device="cuda")
        sw = torch.zeros((c.nterms, c.ncorr), dtype=torch.float64, device="cuda")
        B.lra_grid_po(plan, dev(wl.vis), dev(wl.wt), dev(wl.tau), po, dev(pi), g, sw)
        want, want_sw = rp.grid_awp(wl.uvw, wl.freq, elems, cfis, wl.vis, wl.wt, tau=wl.tau, po_table=po, po_index=pi)
        assert_close(g.cpu().numpy(), want, f"cfg{n} grid_po")
        np.testing.assert_allclose(sw.cpu().numpy(), want_sw, rtol=1e-6)
        plain, _ = rp.grid(wl.uvw, wl.freq, wl.cf_index, wl.vis, wl.wt, tau=wl.tau)
        assert np.abs(want - plain).max() > 1e-2 * np.abs(plain).max()        # the term does something
        model = want.astype(np.complex64)                                      # the oracle's own grid, rounded
        out = torch.full(wl.vis.shape, 7.0 + 7.0j, dtype=torch.complex64, device="cuda")
        B.lra_degrid_po(plan, dev(model), dev(wl.tau), po, dev(pi), dev(wl.vis), out)
        want_v = rp.degrid_awp(wl.uvw, wl.freq, elems, cfis, c.ncorr, model, tau=wl.tau, po_table=po, po_index=pi, vis_in=wl.vis)
        assert_close(out.cpu().numpy(), want_v, f"cfg{n} degrid_po")
    finally:
        B.lra_plan_destroy(plan)


def test_one_entry_for_all_rows_uses_the_tiled_kernels(B, ref):
    """Table 2 'mosaic imaging': one call per pointing, po_index = None; accumulates onto a grid that already holds
    another pointing; out-of-range row indices are skipped in the per-row form."""
    wl = W.make_workload(W.small_config(3))
    c = wl.cfg
    plan, rp = _plans(B, ref, wl)
    try:
        B.lra_bin(plan, dev(wl.uvw), wl.freq, dev(wl.cf_index))
        elems = [(p, p) for p in range(c.ncorr)]
        cfis = [wl.cf_index] * c.ncorr
        po = np.array([[0.85, 7.0e-4, -4.0e-4]])
        rng = np.random.default_rng(9)
        g0 = (rng.normal(size=(c.nterms, c.ncorr, c.ny, c.nx)) + 1j * rng.normal(size=(c.nterms, c.ncorr, c.ny, c.nx))).astype(np.complex64)
        g = dev(g0)
        sw = torch.zeros((c.nterms, c.ncorr), dtype=torch.float64, device="cuda")
        B.lra_grid_po(plan, dev(wl.vis), dev(wl.wt), dev(wl.tau), po, None, g, sw)
        want, want_sw = rp.grid_awp(wl.uvw, wl.freq, elems, cfis, wl.vis, wl.wt, tau=wl.tau, po_table=po)
        assert_close(g.cpu().numpy().astype(np.complex128) - g0, want, "grid_po one entry")
        np.testing.assert_allclose(sw.cpu().numpy(), want_sw, rtol=1e-6)
        model = want.astype(np.complex64)
        out = torch.zeros(wl.vis.shape, dtype=torch.complex64, device="cuda")
        B.lra_degrid_po(plan, dev(model), dev(wl.tau), po, None, None, out)
        want_v = rp.degrid_awp(wl.uvw, wl.freq, elems, cfis, c.ncorr, model, tau=wl.tau, po_table=po)
        assert_close(out.cpu().numpy(), want_v, "degrid_po one entry")
        # rows with an index outside the table are skipped
        pi = np.zeros(len(wl.uvw), dtype=np.int32)
        pi[::3] = 5
        pi[1::3] = -1
        keep = (pi == 0)
        g2 = torch.zeros((c.nterms, c.ncorr, c.ny, c.nx), dtype=torch.complex64, device="cuda")
        B.lra_grid_po(plan, dev(wl.vis), dev(wl.wt), dev(wl.tau), po, dev(pi), g2, None)
        wt_keep = wl.wt * keep[:, None, None]
        want2, _ = rp.grid_awp(wl.uvw, wl.freq, elems, cfis, wl.vis, wt_keep, tau=wl.tau, po_table=po)
        assert_close(g2.cpu().numpy(), want2, "grid_po skipped rows")
    finally:
        B.lra_plan_destroy(plan)


@pytest.mark.parametrize("conj,acc", [(False, False), (True, False), (False, True)])
def test_phase_gradient(B, ref, conj, acc):
    wl = W.make_workload(W.small_config(4))
    c = wl.cfg
    plan, rp = _plans(B, ref, wl)
    try:
        rng = np.random.default_rng(4)
        shape = (c.nterms, c.ncorr, c.ny, c.nx)
        src = (rng.normal(size=shape) + 1j * rng.normal(size=shape)).astype(np.complex64)
        dst0 = (rng.normal(size=shape) + 1j * rng.normal(size=shape)).astype(np.complex64)
        f, dl, dm = 0.9, 2.3e-3, -1.7e-3
        dst = dev(dst0)
        B.lra_phase_gradient(plan, dev(src), f, dl, dm, dst, conjugate=conj, accumulate=acc)
        want = rp.phase_gradient(src, f, dl, dm, conjugate=conj, dst=dst0 if acc else None)
        got = dst.cpu().numpy()
        assert np.abs(got - want).max() <= 4e-7 * np.abs(want).max() + 4e-7 * np.abs(src).max()
    finally:
        B.lra_plan_destroy(plan)


def test_mueller_elements_with_their_own_kernels(B, ref):
    """Four elements of a 2 x 2 Mueller matrix, each with its own kernel index per point (so its own supports), gridded and
    degridded through a one-plane plan; then the same with per-row pointing terms on top."""
    wl = W.make_workload(W.small_config(4))
    c = wl.cfg
    assert c.ncorr >= 2
    plan, _ = _plans(B, ref, wl, ncorr=1, nterms=1)
    rp = ref.RefPlan(c.nx, c.ny, 2, 1, c.oversampling, wl.scale_u, wl.scale_v, wl.cf.support, wl.cf.offset, wl.cf.data,
                     tile=8, sort_mode=1, tile_x=8)
    try:
        rng = np.random.default_rng(12)
        n_cf = len(wl.cf.support)
        elems = [(0, 0), (1, 1), (0, 1), (1, 0)]
        cfis = [wl.cf_index] + [rng.integers(0, n_cf, size=wl.cf_index.shape).astype(np.int32) for _ in range(3)]
        vis, wt = wl.vis[:, :, :2].copy(), wl.wt[:, :, :2].copy()
        tau = None if wl.tau is None else wl.tau[:, :1].copy()
        uvw_d = dev(wl.uvw)
        for po, pi in ((None, None), (_po_table(wl, 11, 2), rng.integers(0, 11, size=len(wl.uvw)).astype(np.int32))):
            g = torch.zeros((2, c.ny, c.nx), dtype=torch.complex64, device="cuda")
            sw = torch.zeros(2, dtype=torch.float64, device="cuda")
            B.lra_grid_mueller(plan, uvw_d, wl.freq, elems, [dev(a) for a in cfis], dev(vis), dev(wt), dev(tau), g, sw,
                               po_table=po, po_index=dev(pi))
            want, want_sw = rp.grid_awp(wl.uvw, wl.freq, elems, cfis, vis, wt, tau=tau, po_table=po, po_index=pi)
            assert_close(g.cpu().numpy(), want[0], f"grid_mueller po={po is not None}")
            np.testing.assert_allclose(sw.cpu().numpy(), want_sw[0], rtol=1e-6)
            model = want[0].astype(np.complex64)
            for vin in (None, vis):
                out = torch.full(vis.shape, 3.0 - 3.0j, dtype=torch.complex64, device="cuda")
                B.lra_degrid_mueller(plan, uvw_d, wl.freq, elems, [dev(a) for a in cfis], dev(model), dev(tau), dev(vin), out,
                                     po_table=po, po_index=dev(pi))
                want_v = rp.degrid_awp(wl.uvw, wl.freq, elems, cfis, 2, model[None], tau=tau, po_table=po, po_index=pi, vis_in=vin)
                assert_close(out.cpu().numpy(), want_v, f"degrid_mueller po={po is not None} vis_in={vin is not None}")
    finally:
        B.lra_plan_destroy(plan)


def test_awp_errors(B):
    wl = W.make_workload(W.small_config(3))
    c = wl.cfg
    plan = B.lra_plan_create(c.nx, c.ny, c.ncorr, c.nterms, c.oversampling, wl.scale_u, wl.scale_v, wl.cf.support, wl.cf.offset,
                             wl.cf.data)
    try:
        g = torch.zeros((c.nterms, c.ncorr, c.ny, c.nx), dtype=torch.complex64, device="cuda")
        with pytest.raises(B.LraError):                                   # before lra_bin
            B.lra_grid_po(plan, dev(wl.vis), dev(wl.wt), None, [[1.0, 0.0, 0.0]], None, g)
        B.lra_bin(plan, dev(wl.uvw), wl.freq, dev(wl.cf_index))
        with pytest.raises(B.LraError):                                   # NaN in the table
            B.lra_grid_po(plan, dev(wl.vis), dev(wl.wt), None, [[1.0, float("nan"), 0.0]], None, g)
        with pytest.raises(B.LraError):                                   # a multi-plane plan cannot run Mueller elements
            B.lra_grid_mueller(plan, dev(wl.uvw), wl.freq, [(0, 0)], [None], dev(wl.vis), dev(wl.wt), None, g[0])
    finally:
        B.lra_plan_destroy(plan)

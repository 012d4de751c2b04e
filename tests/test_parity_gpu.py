"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same seeded
inputs.  Tolerances are north_star's: bin outputs bit-exact; grid / degridded visibilities relative L2 <= 1e-5 and
max abs <= 1e-4 * max|.|; sumwt relative <= 1e-6."""
import numpy as np
import pytest

from paper_2508_17187_b200 import workloads as W

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
C_LIGHT = 299792458.0
TILE = (8, 8)       # (tile_x, tile): the library's default tiles, spelled out so that the oracle gets the same


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2508_17187_b200 import binding
    binding.lib()
    return binding


def dev(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


class GpuRun:
    """One plan + bin on the GPU for a Workload-like bundle of numpy inputs."""

    def __init__(self, B, nx, ny, ncorr, nterms, os_, su, sv, sup, off, data, uvw, freq, cf_index, tile=TILE[1], sort_mode=1,
                 tile_x=TILE[0]):
        self.B = B
        self.shape = (nterms, ncorr, ny, nx)
        self.plan = B.lra_plan_create(nx, ny, ncorr, nterms, os_, su, sv, sup, off, data, tile=tile, sort_mode=sort_mode,
                                      tile_x=tile_x)
        self.nrow, self.nchan, self.ncorr = len(uvw), len(freq), ncorr
        tile_x = tile_x or tile
        self.ntiles = ((nx + tile_x - 1) // tile_x) * ((ny + tile - 1) // tile)
        self.uvw, self.cfi = dev(uvw), dev(cf_index)
        B.lra_bin(self.plan, self.uvw, freq, self.cfi)

    def export(self):
        n = self.nrow * self.nchan
        o = dict(ix=torch.empty(n, dtype=torch.int32, device="cuda"), iy=torch.empty(n, dtype=torch.int32, device="cuda"),
                 fx=torch.empty(n, dtype=torch.int8, device="cuda"), fy=torch.empty(n, dtype=torch.int8, device="cuda"),
                 key=torch.empty(n, dtype=torch.int64, device="cuda"), perm=torch.empty(n, dtype=torch.int32, device="cuda"),
                 tile_start=torch.empty(self.ntiles + 1, dtype=torch.int32, device="cuda"))
        nv = self.B.lra_bin_export(self.plan, **o)
        out = {k: v.cpu().numpy() for k, v in o.items()}
        out["key"] = out["key"].view(np.uint64)
        out["perm"] = out["perm"].view(np.uint32)[:nv]
        out["tile_start"] = out["tile_start"].view(np.uint32)
        out["n_valid"] = nv
        return out

    def grid(self, vis, wt, tau=None, variant=0, grid0=None):
        self.B.lra_set_variant(self.plan, variant, 0)
        g = torch.zeros(self.shape, dtype=torch.complex64, device="cuda") if grid0 is None else dev(grid0)
        sw = torch.zeros(self.shape[:2], dtype=torch.float64, device="cuda")
        self.B.lra_grid(self.plan, dev(vis), dev(wt), dev(tau), g, sw)
        torch.cuda.synchronize()
        return g.cpu().numpy(), sw.cpu().numpy()

    def degrid(self, grid, tau=None, vis_in=None):
        out = torch.full((self.nrow, self.nchan, self.ncorr), 7.0 + 7.0j, dtype=torch.complex64, device="cuda")
        self.B.lra_degrid(self.plan, dev(grid.astype(np.complex64)), dev(tau), dev(vis_in), out)
        torch.cuda.synchronize()
        return out.cpu().numpy()

    def close(self):
        self.B.lra_plan_destroy(self.plan)


def run_for(B, wl, nterms=None, sort_mode=1, tile=TILE[1], tile_x=TILE[0]):
    c = wl.cfg
    return GpuRun(B, c.nx, c.ny, c.ncorr, c.nterms if nterms is None else nterms, c.oversampling, wl.scale_u, wl.scale_v,
                  wl.cf.support, wl.cf.offset, wl.cf.data, wl.uvw, wl.freq, wl.cf_index, tile=tile, sort_mode=sort_mode,
                  tile_x=tile_x)


def ref_for(ref, wl, nterms=None, sort_mode=1, tile=TILE[1], tile_x=TILE[0]):
    return ref.plan_for(wl, nterms=nterms, sort_mode=sort_mode, tile=tile, tile_x=tile_x)


def assert_close(got, want, what):
    want = np.asarray(want, dtype=np.complex128)
    got = np.asarray(got, dtype=np.complex128)
    scale = np.abs(want).max()
    assert scale > 0, what
    l2 = np.linalg.norm((got - want).ravel()) / np.linalg.norm(want.ravel())
    mx = np.abs(got - want).max()
    assert l2 <= 1e-5, f"{what}: relative L2 {l2:.3e}"
    assert mx <= 1e-4 * scale, f"{what}: max abs {mx:.3e} vs scale {scale:.3e}"


def assert_bin_equal(g, r):
    assert g["n_valid"] == r["n_valid"]
    for k in ("ix", "iy", "fx", "fy", "key", "perm", "tile_start"):
        assert np.array_equal(g[k], r[k]), k


# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [1, 2, 3, 4, 5])
@pytest.mark.parametrize("mode", [0, 1])
def test_bin_bit_exact(B, ref, n, mode):
    wl = W.make_workload(W.small_config(n))
    run = run_for(B, wl, sort_mode=mode)
    try:
        assert_bin_equal(run.export(), ref_for(ref, wl, sort_mode=mode).bin(wl.uvw, wl.freq, wl.cf_index))
    finally:
        run.close()


def test_bin_invalid_points_and_small_tile(B, ref):
    wl = W.make_workload(W.small_config(3))
    uvw, cfi = wl.uvw.copy(), wl.cf_index.copy()
    uvw[5] = [3.0e5, -2.0e5, 10.0]
    uvw[17, 0] = np.nan
    uvw[23, 1] = np.inf
    uvw[29, 0] = 1e300
    cfi[40, 1] = -1
    cfi[41, 2] = wl.cfg.n_cf
    for tile, tile_x, mode in ((8, 0, 1), (16, 0, 0), (64, 0, 1), (32, 4, 1), (8, 128, 0)):
        c = wl.cfg
        run = GpuRun(B, c.nx, c.ny, c.ncorr, 1, c.oversampling, wl.scale_u, -wl.scale_v, wl.cf.support, wl.cf.offset,
                     wl.cf.data, uvw, wl.freq, cfi, tile=tile, sort_mode=mode, tile_x=tile_x)
        try:
            r = ref.RefPlan(c.nx, c.ny, c.ncorr, 1, c.oversampling, wl.scale_u, -wl.scale_v, wl.cf.support, wl.cf.offset,
                            wl.cf.data, tile=tile, sort_mode=mode, tile_x=tile_x)
            want = r.bin(uvw, wl.freq, cfi)
            assert want["n_valid"] < c.npoints
            assert_bin_equal(run.export(), want)
        finally:
            run.close()


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5])
def test_grid_parity_small_configs(B, ref, n):
    wl = W.make_workload(W.small_config(n))
    rp = ref_for(ref, wl)
    want, want_sw = rp.grid(wl.uvw, wl.freq, wl.cf_index, wl.vis, wl.wt, wl.tau)
    run = run_for(B, wl)
    try:
        for variant in (0, 1):
            got, sw = run.grid(wl.vis, wl.wt, wl.tau, variant=variant)
            assert_close(got, want, f"cfg{n} grid variant {variant}")
            assert np.abs(sw - want_sw).max() <= 1e-6 * np.abs(want_sw).max()
        nv, s2 = B.lra_tap_count(run.plan)
        assert nv == rp.bin(wl.uvw, wl.freq, wl.cf_index)["n_valid"] and s2 > 0
    finally:
        run.close()


@pytest.mark.parametrize("n", [1, 3, 4, 5])
def test_degrid_parity_small_configs(B, ref, n):
    wl = W.make_workload(W.small_config(n))
    rng = np.random.default_rng(40 + n)
    c = wl.cfg
    if wl.model_grid is not None and c.nterms == 1:
        g = wl.model_grid
    else:
        g = (rng.standard_normal((c.nterms, c.ncorr, c.ny, c.nx)) + 1j * rng.standard_normal((c.nterms, c.ncorr, c.ny, c.nx))).astype(np.complex64)
    rp = ref_for(ref, wl)
    run = run_for(B, wl)
    try:
        want = rp.degrid(wl.uvw, wl.freq, wl.cf_index, g.astype(np.complex128), wl.tau)
        assert_close(run.degrid(g, wl.tau), want, f"cfg{n} degrid")
        want_res = rp.degrid(wl.uvw, wl.freq, wl.cf_index, g.astype(np.complex128), wl.tau, vis_in=wl.vis)
        assert_close(run.degrid(g, wl.tau, vis_in=wl.vis), want_res, f"cfg{n} degrid residual")
    finally:
        run.close()


def test_cfg5_pipeline_degrid_then_multiterm_grid(B, ref):
    """Config 5's chain: degrid the model grid (nterms = 1) with the fused residual, then grid the residuals onto
    two Taylor-weighted grids."""
    wl = W.make_workload(W.small_config(5))
    rp1, rp2 = ref_for(ref, wl, nterms=1), ref_for(ref, wl, nterms=2)
    res_want = rp1.degrid(wl.uvw, wl.freq, wl.cf_index, wl.model_grid.astype(np.complex128), None, vis_in=wl.vis)
    run1, run2 = run_for(B, wl, nterms=1), run_for(B, wl, nterms=2)
    try:
        res = run1.degrid(wl.model_grid, None, vis_in=wl.vis)
        assert_close(res, res_want, "cfg5 residual")
        res_in = res_want.astype(np.complex64)         # the oracle's residuals in the ABI's precision feed both sides
        want, want_sw = rp2.grid(wl.uvw, wl.freq, wl.cf_index, res_in, wl.wt, wl.tau)
        got, sw = run2.grid(res_in, wl.wt, wl.tau)
        assert_close(got, want, "cfg5 multi-term grid")
        assert np.abs(sw - want_sw).max() <= 1e-6 * np.abs(want_sw).max()
    finally:
        run1.close()
        run2.close()


@pytest.mark.parametrize("ncorr,nterms,os_,supports,tile,tile_x", [
    (1, 1, 4, [1, 3], 64, 8), (3, 1, 2, [5, 35, 65], 64, 8), (4, 2, 1, [9], 16, 0), (2, 3, 3, [7, 67], 64, 8),
    (1, 4, 8, [33, 31], 8, 0), (2, 2, 4, [17, 45], 64, 0), (2, 1, 2, [19, 53, 55], 64, 8), (2, 1, 2, [11, 29, 47], 32, 4),
    (1, 2, 1, [3, 21], 4, 64)])
def test_grid_and_degrid_random_tables(B, ref, ncorr, nterms, os_, supports, tile, tile_x):
    """Random complex (non-separable) kernels, supports across all groups of the strip kernels (regions of up to
    2048, 4096, 7168, 9216 pixels and the global-atomic fallback beyond), strips and square tiles, odd correlation /
    term counts, ragged point counts, points off the grid, accumulate-into semantics."""
    rng = np.random.default_rng(1000 + ncorr * 10 + nterms)
    nx, ny, n, nchan = 160, 144, 777, 3
    ks = [(rng.standard_normal((S * os_, S * os_)) + 1j * rng.standard_normal((S * os_, S * os_))).astype(np.complex64) for S in supports]
    sup = np.array(supports, np.int32)
    off = np.concatenate([[0], np.cumsum([k.size for k in ks])[:-1]]).astype(np.int64)
    data = np.concatenate([k.ravel() for k in ks])
    uvw = np.stack([rng.uniform(-nx / 2 - 3, nx / 2 + 3, n), rng.uniform(-ny / 2 - 3, ny / 2 + 3, n), np.zeros(n)], 1)
    freq = C_LIGHT * (1.0 + 0.02 * np.arange(nchan))
    cfi = rng.integers(0, len(supports), (n, nchan)).astype(np.int32)
    vis = (rng.standard_normal((n, nchan, ncorr)) + 1j * rng.standard_normal((n, nchan, ncorr))).astype(np.complex64)
    wt = rng.uniform(0.5, 1, (n, nchan, ncorr)).astype(np.float32)
    wt[rng.random((n, nchan, ncorr)) < 0.05] = 0.0           # flags as zero weight (R4)
    tau = rng.uniform(-1, 1, (nchan, nterms)).astype(np.float32) if nterms > 1 else None
    rp = ref.RefPlan(nx, ny, ncorr, nterms, os_, 0.97, -1.02, sup, off, data, tile=tile, sort_mode=1, tile_x=tile_x)
    run = GpuRun(B, nx, ny, ncorr, nterms, os_, 0.97, -1.02, sup, off, data, uvw, freq, cfi, tile=tile, sort_mode=1, tile_x=tile_x)
    try:
        assert_bin_equal(run.export(), rp.bin(uvw, freq, cfi))
        g0 = (rng.standard_normal((nterms, ncorr, ny, nx)) + 1j * rng.standard_normal((nterms, ncorr, ny, nx))).astype(np.complex64)
        want, want_sw = rp.grid(uvw, freq, cfi, vis, wt, tau, grid=g0.astype(np.complex128))
        for variant in (0, 1):
            got, sw = run.grid(vis, wt, tau, variant=variant, grid0=g0)
            assert_close(got, want, f"random table variant {variant}")
            assert np.abs(sw - want_sw).max() <= 1e-6 * np.abs(want_sw).max()
        gm = (rng.standard_normal((nterms, ncorr, ny, nx)) + 1j * rng.standard_normal((nterms, ncorr, ny, nx))).astype(np.complex64)
        want_v = rp.degrid(uvw, freq, cfi, gm.astype(np.complex128), tau, vis_in=vis)
        got_v = run.degrid(gm, tau, vis_in=vis)
        assert_close(got_v, want_v, "random table degrid")
        invalid = rp.bin(uvw, freq, cfi)["key"] == np.uint64(2 ** 64 - 1)
        assert invalid.any()
        assert np.array_equal(got_v.reshape(-1, ncorr)[invalid], vis.reshape(-1, ncorr)[invalid])   # V = 0 there
    finally:
        run.close()


def test_empty_and_state_errors(B):
    sup, off, data = np.array([3], np.int32), np.array([0], np.int64), np.ones(9, np.complex64)
    plan = B.lra_plan_create(64, 64, 1, 1, 1, 1.0, 1.0, sup, off, data)
    try:
        g = torch.zeros((1, 1, 64, 64), dtype=torch.complex64, device="cuda")
        with pytest.raises(B.LraError):
            B.lra_grid(plan, g, torch.zeros(1, device="cuda"), None, g)          # before lra_bin: LRA_ESTATE
        B.lra_bin(plan, torch.zeros((0, 3), dtype=torch.float64, device="cuda"), np.array([C_LIGHT]))
        assert B.lra_bin_export(plan) == 0
        B.lra_grid(plan, torch.zeros((0, 1, 1), dtype=torch.complex64, device="cuda"),
                   torch.zeros((0, 1, 1), dtype=torch.float32, device="cuda"), None, g)
        torch.cuda.synchronize()
        assert not g.abs().any()
        assert B.lra_launch_count(plan) >= 1
    finally:
        B.lra_plan_destroy(plan)


def test_p4_exact_patch_in_fp32(B):
    """Pin P4 on the GPU: a single unit visibility at a pixel centre reproduces the kernel samples exactly."""
    S, os_, nx = 7, 20, 64
    K = W.ps_kernel(S, os_)
    h, c0 = 3, 3 * os_ + os_ // 2 - 1
    run = GpuRun(B, nx, nx, 1, 1, os_, 1.0, 1.0, [S], [0], K.ravel(), np.array([[5.0 + 1.0 / os_, -9.0, 0.0]]), np.array([C_LIGHT]), None)
    try:
        g, sw = run.grid(np.ones((1, 1, 1), np.complex64), np.ones((1, 1, 1), np.float32))
        X, Y = 32 + 5, 32 - 9
        expect = K[c0 - h * os_:c0 + h * os_ + 1:os_, c0 - 1 - h * os_:c0 - 1 + h * os_ + 1:os_]
        assert np.array_equal(g[0, 0, Y - h:Y + h + 1, X - h:X + h + 1], expect)
        assert np.count_nonzero(g) == np.count_nonzero(expect) and sw[0, 0] == 1.0
    finally:
        run.close()


# ---------------------------------------------------------------------------------------------------
# Full size: BASELINE.json's configurations in the launch configuration bench.py times, compared with the oracle
# ELEMENT BY ELEMENT: every grid pixel (zeros included) and every degridded visibility; the bin bit-exact.  The
# oracle grids ~2.7e9 tap updates/s on the box's cores, so a configuration costs tens of seconds.  No oracle input
# comes from the CUDA path: the grid that is degridded is the oracle's own, rounded to complex64.
# ---------------------------------------------------------------------------------------------------
def _full_size(B, ref, n, check_bin=True, full_degrid=True, npts=4096):
    wl = W.make_workload(W.full_config(n))
    c = wl.cfg
    rp = ref.plan_for(wl, sort_mode=1)
    run = run_for(B, wl, tile=c.tile, tile_x=c.tile_x)
    try:
        if check_bin:
            want_bin = rp.bin(wl.uvw, wl.freq, wl.cf_index)
            assert_bin_equal(run.export(), want_bin)
            del want_bin
        want, want_sw = rp.grid(wl.uvw, wl.freq, wl.cf_index, wl.vis, wl.wt, wl.tau)
        got, sw = run.grid(wl.vis, wl.wt, wl.tau)
        assert_close(got, want, f"cfg{n} full-size grid")
        assert np.abs(sw - want_sw).max() <= 1e-6 * np.abs(want_sw).max()
        assert not got[want == 0].any()                # a pixel no footprint touches stays exactly zero
        del got
        # degridding with the fused residual: the model grid is the oracle's grid in the ABI's precision
        model = want.astype(np.complex64)
        del want
        tau_d = wl.tau
        res = run.degrid(model, tau_d, vis_in=wl.vis)
        if full_degrid:
            want_v = rp.degrid(wl.uvw, wl.freq, wl.cf_index, model.astype(np.complex128), tau_d, vis_in=wl.vis)
            assert_close(res, want_v, f"cfg{n} full-size residuals")
        else:                                          # the point set is drawn before any output is looked at
            sel = np.sort(np.random.default_rng(33 + n).choice(c.npoints, npts, replace=False))
            want_v = rp.degrid_points(wl.uvw, wl.freq, wl.cf_index, model, tau_d, wl.vis, sel)
            gv = res.reshape(-1, c.ncorr)[sel].astype(np.complex128)
            assert np.linalg.norm(gv - want_v) <= 1e-5 * np.linalg.norm(want_v)
            assert np.abs(gv - want_v).max() <= 1e-4 * float(np.abs(want_v).max())
    finally:
        run.close()


def test_full_size_cfg3_all_outputs(B, ref):
    _full_size(B, ref, 3)


@pytest.mark.parametrize("n", [4, 5])
def test_full_size_cfg4_cfg5_all_outputs(B, ref, n):
    _full_size(B, ref, n)


def test_full_size_cfg2_grid_all_pixels(B, ref):
    """323 M points: every grid pixel is compared; the oracle's full bin (a single-threaded merge sort) and its
    10 GB of double-precision residuals are left to the smaller configurations: 4,096 seeded points instead."""
    _full_size(B, ref, 2, check_bin=False, full_degrid=False)


def test_full_size_cfg1_all_outputs(B, ref):
    """Config 1 at full size is small enough for an element-by-element comparison."""
    wl = W.make_workload(W.full_config(1))
    rp = ref.plan_for(wl, sort_mode=1)
    run = run_for(B, wl, tile=wl.cfg.tile, tile_x=wl.cfg.tile_x)
    try:
        assert_bin_equal(run.export(), rp.bin(wl.uvw, wl.freq, wl.cf_index))
        want, want_sw = rp.grid(wl.uvw, wl.freq, wl.cf_index, wl.vis, wl.wt, wl.tau)
        got, sw = run.grid(wl.vis, wl.wt, wl.tau)
        assert_close(got, want, "cfg1 full grid")
        model = want.astype(np.complex64)              # the oracle's grid in the ABI's precision, not the GPU's
        want_v = rp.degrid(wl.uvw, wl.freq, wl.cf_index, model.astype(np.complex128), wl.tau, vis_in=wl.vis)
        assert_close(run.degrid(model, wl.tau, vis_in=wl.vis), want_v, "cfg1 full degrid")
    finally:
        run.close()


def test_degrid_variants_agree(B, ref):
    """Variant 1 (warp per point, the 'before' kernel and the fallback for oversized regions) against the oracle."""
    wl = W.make_workload(W.small_config(4))
    rng = np.random.default_rng(77)
    c = wl.cfg
    g = (rng.standard_normal((c.nterms, c.ncorr, c.ny, c.nx)) + 1j * rng.standard_normal((c.nterms, c.ncorr, c.ny, c.nx))).astype(np.complex64)
    want = ref_for(ref, wl).degrid(wl.uvw, wl.freq, wl.cf_index, g.astype(np.complex128), wl.tau, vis_in=wl.vis)
    run = run_for(B, wl)
    try:
        for variant in (0, 1):
            B.lra_set_variant(run.plan, 0, variant)
            assert_close(run.degrid(g, wl.tau, vis_in=wl.vis), want, f"degrid variant {variant}")
    finally:
        run.close()


# ---------------------------------------------------------------------------------------------------
# ABI corners: tile-only sort order, re-binning one plan, accumulate-into sumwt, a non-default stream, in-place degrid
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [3, 4])
def test_grid_and_degrid_under_sort_tile(B, ref, n):
    """LRA_SORT_TILE (mode 0): points of a tile stay in caller order, so a CF slab serves short runs; same results."""
    wl = W.make_workload(W.small_config(n))
    rp = ref_for(ref, wl, sort_mode=0)
    run = run_for(B, wl, sort_mode=0)
    try:
        assert_bin_equal(run.export(), rp.bin(wl.uvw, wl.freq, wl.cf_index))
        want, want_sw = rp.grid(wl.uvw, wl.freq, wl.cf_index, wl.vis, wl.wt, wl.tau)
        got, sw = run.grid(wl.vis, wl.wt, wl.tau)
        assert_close(got, want, "sort_mode 0 grid")
        assert np.abs(sw - want_sw).max() <= 1e-6 * np.abs(want_sw).max()
        model = want.astype(np.complex64)
        want_v = rp.degrid(wl.uvw, wl.freq, wl.cf_index, model.astype(np.complex128), wl.tau, vis_in=wl.vis)
        assert_close(run.degrid(model, wl.tau, vis_in=wl.vis), want_v, "sort_mode 0 degrid")
    finally:
        run.close()


def test_rebin_small_large_small(B, ref):
    """One plan binned with a short, a long and again a short row set: the plan's arrays grow and are reused."""
    wl = W.make_workload(W.small_config(3))
    rp = ref_for(ref, wl)
    run = run_for(B, wl)
    try:
        nrow = len(wl.uvw)
        for rows in (slice(0, nrow // 7), slice(0, nrow), slice(nrow // 3, nrow // 2)):
            uvw, cfi, vis, wt = wl.uvw[rows], wl.cf_index[rows], wl.vis[rows], wl.wt[rows]
            run.nrow = len(uvw)
            run.uvw, run.cfi = dev(uvw), dev(cfi)
            B.lra_bin(run.plan, run.uvw, wl.freq, run.cfi)
            assert_bin_equal(run.export(), rp.bin(uvw, wl.freq, cfi))
            want, want_sw = rp.grid(uvw, wl.freq, cfi, vis, wt, wl.tau)
            got, sw = run.grid(vis, wt, wl.tau)
            assert_close(got, want, f"re-bin rows {rows}")
            assert np.abs(sw - want_sw).max() <= 1e-6 * np.abs(want_sw).max()
            model = want.astype(np.complex64)
            want_v = rp.degrid(uvw, wl.freq, cfi, model.astype(np.complex128), wl.tau, vis_in=vis)
            assert_close(run.degrid(model, wl.tau, vis_in=vis), want_v, f"re-bin degrid rows {rows}")
    finally:
        run.close()


def test_sumwt_accumulates_and_degrid_in_place(B, ref):
    wl = W.make_workload(W.small_config(5))
    c = wl.cfg
    rp = ref_for(ref, wl, nterms=2)
    run = run_for(B, wl, nterms=2)
    try:
        sw0 = np.array([[3.0, -1.5], [0.25, 1e6]])[: 2, : c.ncorr]
        want, want_sw = rp.grid(wl.uvw, wl.freq, wl.cf_index, wl.vis, wl.wt, wl.tau, sumwt=sw0.copy())
        g = torch.zeros((2, c.ncorr, c.ny, c.nx), dtype=torch.complex64, device="cuda")
        sw = dev(sw0.copy())
        B.lra_grid(run.plan, dev(wl.vis), dev(wl.wt), dev(wl.tau), g, sw)
        torch.cuda.synchronize()
        assert_close(g.cpu().numpy(), want, "grid with sumwt accumulate-into")
        assert np.abs(sw.cpu().numpy() - want_sw).max() <= 1e-6 * np.abs(want_sw).max()
        # in-place residual: vis_out aliases vis_in
        model = want.astype(np.complex64)
        want_v = rp.degrid(wl.uvw, wl.freq, wl.cf_index, model.astype(np.complex128), wl.tau, vis_in=wl.vis)
        v = dev(wl.vis.copy())
        B.lra_degrid(run.plan, dev(model), dev(wl.tau), v, v)
        torch.cuda.synchronize()
        assert_close(v.cpu().numpy(), want_v, "in-place degrid")
    finally:
        run.close()


def test_non_default_stream(B, ref):
    """A plan bound to a stream of its own: every call is enqueued there and ordered with the caller's work by
    stream semantics only."""
    wl = W.make_workload(W.small_config(3))
    c = wl.cfg
    rp = ref_for(ref, wl)
    st = torch.cuda.Stream()
    plan = B.lra_plan_create(c.nx, c.ny, c.ncorr, c.nterms, c.oversampling, wl.scale_u, wl.scale_v, wl.cf.support,
                             wl.cf.offset, wl.cf.data, tile=TILE[1], tile_x=TILE[0], sort_mode=1, stream=st.cuda_stream)
    try:
        uvw, cfi, vis, wt = dev(wl.uvw), dev(wl.cf_index), dev(wl.vis), dev(wl.wt)
        torch.cuda.synchronize()
        with torch.cuda.stream(st):
            g = torch.zeros((c.nterms, c.ncorr, c.ny, c.nx), dtype=torch.complex64, device="cuda")
            sw = torch.zeros((c.nterms, c.ncorr), dtype=torch.float64, device="cuda")
            B.lra_bin(plan, uvw, wl.freq, cfi)
            B.lra_grid(plan, vis, wt, None, g, sw)
        st.synchronize()
        want, want_sw = rp.grid(wl.uvw, wl.freq, wl.cf_index, wl.vis, wl.wt, wl.tau)
        assert_close(g.cpu().numpy(), want, "grid on a non-default stream")
        model = want.astype(np.complex64)
        with torch.cuda.stream(st):
            res = torch.empty_like(vis)
            B.lra_degrid(plan, dev(model), None, vis, res)
        st.synchronize()
        want_v = rp.degrid(wl.uvw, wl.freq, wl.cf_index, model.astype(np.complex128), None, vis_in=wl.vis)
        assert_close(res.cpu().numpy(), want_v, "degrid on a non-default stream")
    finally:
        B.lra_plan_destroy(plan)


def test_repeated_calls_keep_parity(B, ref):
    """compute-sanitizer is closed on the GPU pool, so the mbarrier / TMA ring is exercised instead by repetition: 25
    grid + degrid calls on one plan (every ring slot recycled hundreds of times, producer and consumers in every
    relative timing the scheduler produces), each compared with the oracle."""
    wl = W.make_workload(W.small_config(3))
    rp = ref_for(ref, wl)
    want, _ = rp.grid(wl.uvw, wl.freq, wl.cf_index, wl.vis, wl.wt, wl.tau)
    model = want.astype(np.complex64)
    want_v = rp.degrid(wl.uvw, wl.freq, wl.cf_index, model.astype(np.complex128), wl.tau, vis_in=wl.vis)
    run = run_for(B, wl)
    try:
        for it in range(25):
            got, _ = run.grid(wl.vis, wl.wt, wl.tau)
            assert_close(got, want, f"grid, repetition {it}")
            assert_close(run.degrid(model, wl.tau, vis_in=wl.vis), want_v, f"degrid, repetition {it}")
    finally:
        run.close()


# ---------------------------------------------------------------------------------------------------
# NEXT-1: grid -> image (F^dagger, taper correction, sum-of-weights normalisation) and image -> grid (F)
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ny,nx,ncorr,nterms", [(64, 64, 1, 1), (96, 128, 2, 2), (254, 130, 2, 1)])
def test_image_and_model_grid(B, ref, ny, nx, ncorr, nterms):
    """Both transforms against the oracle's centred DFT (relative L2 <= 1e-5, max abs <= 1e-4 max|.|): sizes with
    nx/2 + ny/2 even and odd (the sign of the centring), non-square, several grids, with and without the factors."""
    rng = np.random.default_rng(nx + ny)
    sup, off, data = np.array([3], np.int32), np.array([0], np.int64), np.ones(9, np.complex64)
    plan = B.lra_plan_create(nx, ny, ncorr, nterms, 1, 1.0, 1.0, sup, off, data)
    try:
        g = (rng.standard_normal((nterms, ncorr, ny, nx)) + 1j * rng.standard_normal((nterms, ncorr, ny, nx))).astype(np.complex64)
        sw = rng.uniform(0.5, 3.0, (nterms, ncorr))
        cx, cy = rng.uniform(0.5, 2.0, nx).astype(np.float32), rng.uniform(0.5, 2.0, ny).astype(np.float32)
        img = torch.empty((nterms, ncorr, ny, nx), dtype=torch.float32, device="cuda")
        for use in (True, False):
            B.lra_image(plan, dev(g), dev(sw) if use else None, dev(cx) if use else None, dev(cy) if use else None, img)
            torch.cuda.synchronize()
            want = ref.image(g, sw if use else None, cx if use else None, cy if use else None)
            got = img.cpu().numpy().astype(np.float64)
            assert np.linalg.norm(got - want) <= 1e-5 * np.linalg.norm(want)
            assert np.abs(got - want).max() <= 1e-4 * np.abs(want).max()
        im = rng.standard_normal((nterms, ncorr, ny, nx)).astype(np.float32)
        out = torch.empty((nterms, ncorr, ny, nx), dtype=torch.complex64, device="cuda")
        B.lra_model_grid(plan, dev(im), dev(cx), dev(cy), out)
        torch.cuda.synchronize()
        assert_close(out.cpu().numpy(), ref.model_grid(im, cx, cy), "model grid")
    finally:
        B.lra_plan_destroy(plan)


def test_major_cycle_on_device(B, ref):
    """The whole UpdateDir of Eq. 23 on the device for cfg5-small: model image -> F -> degrid with fused residual ->
    grid (two Taylor terms) -> F^dagger with normalisation, against the same chain through the oracle."""
    wl = W.make_workload(W.small_config(5))
    c = wl.cfg
    rng = np.random.default_rng(55)
    model_img = np.zeros((1, c.ncorr, c.ny, c.nx), np.float32)
    for _ in range(20):
        y, x = rng.integers(c.ny // 10, c.ny - c.ny // 10), rng.integers(c.nx // 10, c.nx - c.nx // 10)
        model_img[0, :, y, x] = rng.uniform(0.1, 1.0)
    rp1, rp2 = ref_for(ref, wl, nterms=1), ref_for(ref, wl, nterms=2)
    mg = ref.model_grid(model_img).astype(np.complex64)                      # oracle chain
    res_want = rp1.degrid(wl.uvw, wl.freq, wl.cf_index, mg.astype(np.complex128), None, vis_in=wl.vis)
    g_want, sw_want = rp2.grid(wl.uvw, wl.freq, wl.cf_index, res_want.astype(np.complex64), wl.wt, wl.tau)
    img_want = ref.image(g_want.astype(np.complex64), sw_want)
    run1, run2 = run_for(B, wl, nterms=1), run_for(B, wl, nterms=2)
    try:
        d_mg = torch.empty((1, c.ncorr, c.ny, c.nx), dtype=torch.complex64, device="cuda")
        B.lra_model_grid(run1.plan, dev(model_img), None, None, d_mg)
        assert_close(d_mg.cpu().numpy(), mg, "model grid of the cycle")
        res = torch.empty((c.nrow, c.nchan, c.ncorr), dtype=torch.complex64, device="cuda")
        B.lra_degrid(run1.plan, d_mg, None, dev(wl.vis), res)
        g = torch.zeros((2, c.ncorr, c.ny, c.nx), dtype=torch.complex64, device="cuda")
        sw = torch.zeros((2, c.ncorr), dtype=torch.float64, device="cuda")
        B.lra_grid(run2.plan, res, dev(wl.wt), dev(wl.tau), g, sw)
        img = torch.empty((2, c.ncorr, c.ny, c.nx), dtype=torch.float32, device="cuda")
        B.lra_image(run2.plan, g, sw, None, None, img)
        torch.cuda.synchronize()
        got = img.cpu().numpy().astype(np.float64)
        assert np.linalg.norm(got - img_want) <= 1e-5 * np.linalg.norm(img_want) * 3      # three chained fp32 stages
        assert np.abs(got - img_want).max() <= 1e-4 * np.abs(img_want).max()
    finally:
        run1.close()
        run2.close()


# ---------------------------------------------------------------------------------------------------
# NEXT-4: the G-Jones solver (Eq. 19-21) fed by lra_degrid's model visibilities
# ---------------------------------------------------------------------------------------------------
def test_gain_solver_fed_by_degrid(B, ref):
    """Model visibilities of cfg5-small (degridded model grid), observed = g_i conj(g_j) * model + noise: Eq. 19 sums and the
    Eq. 20 / 21 iteration against the oracle (double on both sides: 1e-9 relative on the sums over the same complex64
    inputs, 1e-9 on the gains, identical iteration counts), with and without an explicit baseline index."""
    wl = W.make_workload(W.small_config(5))
    c = wl.cfg
    # the model visibilities: the oracle's prediction in the ABI's precision feeds BOTH solvers; lra_degrid's own
    # prediction (what a caller would feed) is checked against it first
    model = ref_for(ref, wl, nterms=1).degrid(wl.uvw, wl.freq, wl.cf_index, wl.model_grid.astype(np.complex128), None).astype(np.complex64)
    run = run_for(B, wl, nterms=1)
    try:
        assert_close(run.degrid(wl.model_grid, None), model, "model visibilities from lra_degrid")
    finally:
        run.close()
    d_model = dev(model)
    rng = np.random.default_rng(21)
    nant, nbl = W.N_ANT, W.N_BL
    a1, a2 = (x.astype(np.int32) for x in np.triu_indices(nant, 1))
    g = (1 + 0.2 * rng.standard_normal((nant, c.ncorr))) * np.exp(1j * rng.uniform(-1, 1, (nant, c.ncorr)))
    bl = (np.arange(c.nrow) % nbl).astype(np.int32)
    vis = (g[a1[bl]][:, None, :] * np.conj(g[a2[bl]])[:, None, :] * model
           + 0.05 * (rng.standard_normal(model.shape) + 1j * rng.standard_normal(model.shape))).astype(np.complex64)
    wt = wl.wt.copy()
    wt[rng.random(wt.shape) < 0.03] = 0.0
    want_x, want_w = ref.gain_accumulate(vis, model, wt, nbl)
    for bli in (None, bl[::-1].copy()):
        xs = torch.zeros((nbl, c.ncorr), dtype=torch.complex128, device="cuda")
        ws = torch.zeros((nbl, c.ncorr), dtype=torch.float64, device="cuda")
        if bli is None:
            B.lra_gain_accumulate(dev(vis), d_model, dev(wt), nbl, xs, ws)
            wx, ww = want_x, want_w
        else:
            B.lra_gain_accumulate(dev(vis), d_model, dev(wt), nbl, xs, ws, bl_index=dev(bli))
            wx, ww = ref.gain_accumulate(vis, model, wt, nbl, bl_index=bli)
        torch.cuda.synchronize()
        assert np.abs(xs.cpu().numpy() - wx).max() <= 1e-9 * np.abs(wx).max()
        assert np.abs(ws.cpu().numpy() - ww).max() <= 1e-9 * np.abs(ww).max()
    xs = torch.zeros((nbl, c.ncorr), dtype=torch.complex128, device="cuda")
    ws = torch.zeros((nbl, c.ncorr), dtype=torch.float64, device="cuda")
    B.lra_gain_accumulate(dev(vis), d_model, dev(wt), nbl, xs, ws)
    for alpha, delta, max_iter in ((0.5, 1e-8, 500), (1.0, 0.0, 7), (0.3, 1e-3, 1000)):
        want_g, want_it = ref.gain_solve(nant, a1, a2, want_x, want_w, alpha, delta, max_iter, np.ones((nant, c.ncorr)))
        gains = torch.ones((nant, c.ncorr), dtype=torch.complex128, device="cuda")
        it = torch.zeros(1, dtype=torch.int32, device="cuda")
        B.lra_gain_solve(dev(a1), dev(a2), xs, ws, alpha, delta, max_iter, gains, it)
        torch.cuda.synchronize()
        assert int(it.item()) == want_it
        assert np.abs(gains.cpu().numpy() - want_g).max() <= 1e-9
    sol = gains.cpu().numpy()
    assert np.abs(sol[a1] * np.conj(sol[a2]) - g[a1] * np.conj(g[a2])).max() < 0.05     # the gains are recovered

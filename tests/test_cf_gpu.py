"""GPU parity of lra_cf_generate (on-device CF construction) against oracle/lra_ref_cf.c,
sample by sample.  The CUDA path computes in fp64 and rounds once to complex64, so the bar is one float32 ulp of each
sample's magnitude plus 1e-7 of the kernel's peak (the two fp64 evaluations differ by ~1e-13 relative,
which can only move a sample across a float32 rounding boundary).  No oracle input comes from the CUDA path."""
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


def _offsets(sup, os_, gap=0):
    sizes = (np.asarray(sup, dtype=np.int64) * os_) ** 2 + gap
    return np.concatenate([[0], np.cumsum(sizes)[:-1]]).astype(np.int64), int(sizes.sum())


def _assert_cf_close(got, want64, what):
    want = want64.astype(np.complex64)
    peak = np.abs(want64).max()
    err = np.abs(got.astype(np.complex128) - want.astype(np.complex128))
    bound = 2.0 ** -22 * np.abs(want64) + 1e-7 * peak
    bad = err > bound
    assert not bad.any(), f"{what}: {bad.sum()} samples off, worst {err.max():.3e} (peak {peak:.3e})"


def _inputs(n, n_aterm, seed):
    rng = np.random.default_rng(seed)
    x = (np.arange(n) - n // 2) / (n / 2.0)
    taper = np.cos(0.5 * np.pi * x) ** 2 + 0.05 * rng.uniform(size=n)
    aterm = ((1.0 + 0.2 * rng.normal(size=(n_aterm, n, n))) * np.exp(0.3j * rng.normal(size=(n_aterm, n, n)))).astype(np.complex64)
    return taper, aterm


@pytest.mark.parametrize("n,os_", [(48, 4), (33, 3), (64, 8)])
def test_cf_generate_table1_rows_mixed_supports(B, ref, n, os_):
    """Every row of Table 1 (A, PS, W each ON or OFF), several supports in one call (the batch shares one phase table),
    a ragged last block (supports that are no multiple of the block sizes), gaps between kernels left untouched."""
    taper, aterm = _inputs(n, 3, 100 + n)
    fov = 0.05
    rows = [(True, True, True), (True, False, True), (True, True, False), (True, False, False), (False, True, True),
            (False, True, False)]
    for a_on, ps_on, w_on in rows:
        sup = np.array([5, 13, 1, 9, 31, 7], dtype=np.int32)
        w = np.array([0.0, 300.0, -120.5, 2500.0, 40.0, 7.0]) if w_on else None
        ia = np.array([0, 2, 1, 1, 0, 2], dtype=np.int32) if a_on else None
        off, total = _offsets(sup, os_, gap=3)
        out = torch.full((total,), 9.0 - 9.0j, dtype=torch.complex64, device="cuda")
        B.lra_cf_generate(out, n, os_, fov, sup, off, taper=dev(taper) if ps_on else None, aterm=dev(aterm) if a_on else None,
                          cf_w=w, cf_aterm=ia)
        got = out.cpu().numpy()
        for c, S in enumerate(sup):
            so = int(S) * os_
            want = ref.cf(n, os_, fov, int(S), taper=taper if ps_on else None, w_lambda=float(w[c]) if w_on else 0.0,
                          aterm=aterm[ia[c]].astype(np.complex128) if a_on else None)
            _assert_cf_close(got[off[c]: off[c] + so * so].reshape(so, so), want, f"rows {a_on, ps_on, w_on} kernel {c}")
            assert np.all(got[off[c] + so * so: off[c] + so * so + 3] == np.complex64(9.0 - 9.0j))


def test_cf_generate_unnormalised_and_default_aterm(B, ref):
    n, os_, S = 40, 4, 11
    taper, aterm = _inputs(n, 1, 7)
    off, total = _offsets([S, S], os_)
    out = torch.zeros(total, dtype=torch.complex64, device="cuda")
    B.lra_cf_generate(out, n, os_, 0.2, [S, S], off, taper=dev(taper), aterm=dev(aterm), cf_w=[15.0, -15.0], normalise=False)
    got = out.cpu().numpy().reshape(2, S * os_, S * os_)
    for c, w in enumerate((15.0, -15.0)):
        want = ref.cf(n, os_, 0.2, S, taper=taper, w_lambda=w, aterm=aterm[0].astype(np.complex128), normalise=False)
        _assert_cf_close(got[c], want, f"unnormalised {c}")


def test_cf_generate_w_projection_table_of_cfg3(B, ref):
    """The W-projection recipe of the benchmark workload (prolate taper x W, one kernel per w
    plane, support growing with w) built on the device, every kernel against the oracle; more kernels than one batch of
    work buffers holds at this size is exercised by test_cf_generate_many_batches."""
    cfg = W.full_config(3)
    n, os_ = (128 if cfg.s_max > 33 else 64), cfg.oversampling
    fov, w_max = 0.02, 4000.0
    taper1 = W.Prolate(cfg.s_min)
    x = (np.arange(n) - n // 2) / (n / 2.0)
    taper = taper1(x) / taper1.norm0
    planes = list(range(0, cfg.n_w, max(1, cfg.n_w // 12)))[:12] + [cfg.n_w - 1]
    sup = np.array([W.w_plane_support(cfg, p) for p in planes], dtype=np.int32)
    w = np.array([(p + 0.5) * w_max / cfg.n_w for p in planes])
    off, total = _offsets(sup, os_)
    out = torch.zeros(total, dtype=torch.complex64, device="cuda")
    B.lra_cf_generate(out, n, os_, fov, sup, off, taper=dev(taper), cf_w=w)
    got = out.cpu().numpy()
    for c, S in enumerate(sup):
        so = int(S) * os_
        _assert_cf_close(got[off[c]: off[c] + so * so].reshape(so, so), ref.cf(n, os_, fov, int(S), taper=taper, w_lambda=float(w[c])),
                         f"plane {planes[c]} S={S}")


def test_cf_generate_many_batches(B, ref):
    """Large supports shrink the batch (work buffers are bounded): 40 kernels of S = 129 at os = 8 do not fit one batch."""
    n, os_, S, n_cf = 160, 8, 129, 40
    taper, _ = _inputs(n, 1, 3)
    w = np.linspace(-2000.0, 2000.0, n_cf)
    off, total = _offsets([S] * n_cf, os_)
    out = torch.zeros(total, dtype=torch.complex64, device="cuda")
    B.lra_cf_generate(out, n, os_, 0.03, [S] * n_cf, off, taper=dev(taper), cf_w=w)
    so = S * os_
    for c in (0, 13, 26, 39):
        got = out[off[c]: off[c] + so * so].cpu().numpy().reshape(so, so)
        _assert_cf_close(got, ref.cf(n, os_, 0.03, S, taper=taper, w_lambda=float(w[c])), f"kernel {c}")


def test_generated_table_feeds_the_plan_from_device_memory(B, ref):
    """PreCompute -> lra_plan_create (cf_data in device memory) -> lra_bin -> lra_grid, against the oracle gridder run on the
    oracle's own CF table."""
    wl = W.make_workload(W.small_config(3))
    c = wl.cfg
    n, os_, fov = 64, c.oversampling, 0.02
    taper1 = W.Prolate(c.s_min)
    x = (np.arange(n) - n // 2) / (n / 2.0)
    taper = taper1(x) / taper1.norm0
    sup = np.asarray(wl.cf.support, dtype=np.int32)
    w = (np.arange(len(sup)) + 0.5) * 900.0 / len(sup)
    off, total = _offsets(sup, os_)
    table = torch.zeros(total, dtype=torch.complex64, device="cuda")
    B.lra_cf_generate(table, n, os_, fov, sup, off, taper=dev(taper), cf_w=w)
    want_table = np.concatenate([ref.cf(n, os_, fov, int(S), taper=taper, w_lambda=float(w[k])).astype(np.complex64).ravel()
                                 for k, S in enumerate(sup)])
    plan = B.lra_plan_create(c.nx, c.ny, c.ncorr, 1, os_, wl.scale_u, wl.scale_v, sup, off, table)
    try:
        B.lra_bin(plan, dev(wl.uvw), wl.freq, dev(wl.cf_index))
        g = torch.zeros((1, c.ncorr, c.ny, c.nx), dtype=torch.complex64, device="cuda")
        sw = torch.zeros((1, c.ncorr), dtype=torch.float64, device="cuda")
        B.lra_grid(plan, dev(wl.vis), dev(wl.wt), None, g, sw)
        torch.cuda.synchronize()
    finally:
        B.lra_plan_destroy(plan)
    rp = ref.RefPlan(c.nx, c.ny, c.ncorr, 1, os_, wl.scale_u, wl.scale_v, sup, off, want_table, tile=8, sort_mode=1, tile_x=8)
    want, want_sw = rp.grid(wl.uvw, wl.freq, wl.cf_index, wl.vis, wl.wt)
    got = g.cpu().numpy().astype(np.complex128)
    scale = np.abs(want).max()
    assert np.linalg.norm((got - want).ravel()) / np.linalg.norm(want.ravel()) <= 1e-5
    assert np.abs(got - want).max() <= 1e-4 * scale
    np.testing.assert_allclose(sw.cpu().numpy(), want_sw, rtol=1e-6)


def test_cf_generate_extreme_shapes(B, ref):
    """No oversampling, the smallest and the largest support, an odd raster, a raster smaller than the support."""
    for n, os_, sup in ((33, 1, [1, 3, 129]), (140, 2, [129]), (8, 4, [31])):
        taper, aterm = _inputs(n, 1, n + os_)
        w = np.linspace(-50.0, 900.0, len(sup))
        off, total = _offsets(sup, os_)
        out = torch.zeros(total, dtype=torch.complex64, device="cuda")
        B.lra_cf_generate(out, n, os_, 0.04, sup, off, taper=dev(taper), aterm=dev(aterm), cf_w=w)
        got = out.cpu().numpy()
        for c, S in enumerate(sup):
            so = S * os_
            want = ref.cf(n, os_, 0.04, S, taper=taper, w_lambda=float(w[c]), aterm=aterm[0].astype(np.complex128))
            _assert_cf_close(got[off[c]: off[c] + so * so].reshape(so, so), want, f"n={n} os={os_} S={S}")


def test_cf_generate_errors(B):
    out = torch.zeros(4096, dtype=torch.complex64, device="cuda")
    t = torch.ones(16, dtype=torch.float64, device="cuda")
    with pytest.raises(B.LraError):
        B.lra_cf_generate(out, 16, 2, 0.1, [4], [0], taper=t)                 # even support
    with pytest.raises(B.LraError):
        B.lra_cf_generate(out, 16, 2, -0.1, [5], [0], taper=t)                # fov <= 0
    with pytest.raises(B.LraError):
        B.lra_cf_generate(out, 16, 2, 0.1, [5], [4090], taper=t)              # table too small
    with pytest.raises(B.LraError):
        B.lra_cf_generate(out, 16, 2, 0.1, [5], [0], taper=t, cf_aterm=[0])   # A-term index without patterns
    with pytest.raises(B.LraError):
        B.lra_cf_generate(out, 16, 2, 0.1, [5], [0], taper=torch.ones(15, dtype=torch.float64, device="cuda"))
    z = torch.zeros((1, 16, 16), dtype=torch.complex64, device="cuda")
    with pytest.raises(B.LraError):
        B.lra_cf_generate(out, 16, 2, 0.1, [5], [0], aterm=z)                 # samples sum to zero: cannot normalise
    B.lra_cf_generate(out, 16, 2, 0.1, [5], [0], aterm=z, normalise=False)    # fine without normalisation
    assert float(out[:100].abs().max()) == 0.0

"""lra_phase_gradient_static (include/lra.h): the phase gradient of Eq. 27 with its phasor table in a file-scope device
array instead of plan-owned scratch, for callers that must not call cudaMalloc.  Checked against the existing path,
lra_phase_gradient on a plan (itself checked against the oracle in tests/test_awp_gpu.py), with that test's tolerance, on
calls in a row that share the static array.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

SU, SV = 0.013, -0.011    # pixels per wavelength


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2508_17187_b200 import binding
    binding.lib()
    return binding


def _plan(B, nx, ny, ncorr, nterms):
    """A plan of that geometry with a one-tap CF table: lra_phase_gradient only uses its sizes, scales and scratch."""
    return B.lra_plan_create(nx, ny, ncorr, nterms, 1, SU, SV, np.array([1], np.int32), np.array([0], np.int64),
                             np.ones(1, np.complex64))


def _rand(shape, seed):
    rng = np.random.default_rng(seed)
    return torch.from_numpy((rng.normal(size=shape) + 1j * rng.normal(size=shape)).astype(np.complex64)).cuda()


def _close(got, want, src):
    got, want = got.cpu().numpy(), want.cpu().numpy()
    assert np.abs(got - want).max() <= 4e-7 * np.abs(want).max() + 4e-7 * float(src.abs().max())


# (nterms, ncorr, ny, nx), (f, dl, dm), conjugate, accumulate: a large table first, then smaller ones that leave its tail
# in the static array, odd and non-square sizes, every mode
CALLS = [((2, 2, 200, 312), (0.9, 2.3e-3, -1.7e-3), False, False),
         ((1, 3, 65, 47), (1.2, -4.1e-3, 0.6e-3), True, False),
         ((1, 2, 96, 128), (0.5, 0.9e-3, 3.3e-3), False, True),
         ((2, 2, 200, 312), (0.7, -1.1e-3, 2.9e-3), True, False)]


def test_static_phase_gradient_matches_the_plan_path_on_calls_in_a_row(B):
    cases = []
    for k, (shape, fac, conj, acc) in enumerate(CALLS):
        src, dst0 = _rand(shape, 10 + k), _rand(shape, 20 + k)
        plan = _plan(B, shape[3], shape[2], shape[1], shape[0])
        try:
            want = dst0.clone()
            B.lra_phase_gradient(plan, src, *fac, want, conjugate=conj, accumulate=acc)
            torch.cuda.synchronize()
        finally:
            B.lra_plan_destroy(plan)
        cases.append((src, dst0, want, fac, conj, acc))
    # the calls in a row, nothing between them but stream order; outputs allocated beforehand
    outs = [dst0.clone() for _, dst0, _, _, _, _ in cases]
    for (src, _, _, fac, conj, acc), out in zip(cases, outs):     # warm-up: loads the kernels, resolves the symbol
        B.lra_phase_gradient_static(src, SU, SV, *fac, out.clone(), conjugate=conj, accumulate=acc)
    for rep in range(2):
        if rep:
            for (_, dst0, _, _, _, _), out in zip(cases, outs):
                out.copy_(dst0)
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        for (src, _, _, fac, conj, acc), out in zip(cases, outs):
            B.lra_phase_gradient_static(src, SU, SV, *fac, out, conjugate=conj, accumulate=acc)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free_before        # no device allocation by the calls
        for (src, _, want, _, _, _), out in zip(cases, outs):
            _close(out, want, src)
    assert B.lra_static_last_error() == ""


def test_static_phase_gradient_in_place_and_on_a_side_stream(B):
    shape, fac = (1, 2, 80, 72), (1.1, 1.9e-3, -0.4e-3)
    src = _rand(shape, 31)
    plan = _plan(B, shape[3], shape[2], shape[1], shape[0])
    try:
        want = torch.empty_like(src)
        B.lra_phase_gradient(plan, src, *fac, want)
        torch.cuda.synchronize()
    finally:
        B.lra_plan_destroy(plan)
    s = torch.cuda.Stream()
    buf = src.clone()
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        B.lra_phase_gradient_static(buf, SU, SV, *fac, buf)         # src == dst
    s.synchronize()
    _close(buf, want, src)


def test_static_phase_gradient_rejects_what_the_static_table_cannot_hold(B):
    lim = B.LRA_STATIC_MAX_AXES
    ok = torch.zeros((1, 1, lim - 1), dtype=torch.complex64, device="cuda")        # nx + ny == the maximum: accepted
    B.lra_phase_gradient_static(ok, SU, SV, 1.0, 0.0, 0.0, ok)
    torch.cuda.synchronize()
    big = torch.zeros((1, 1, lim), dtype=torch.complex64, device="cuda")           # one more
    with pytest.raises(B.LraError, match="LRA_STATIC_MAX_AXES"):
        B.lra_phase_gradient_static(big, SU, SV, 1.0, 0.0, 0.0, big)
    assert "exceeds" in B.lra_static_last_error()
    small = torch.zeros((1, 4, 4), dtype=torch.complex64, device="cuda")
    with pytest.raises(B.LraError):
        B.lra_phase_gradient_static(small, 0.0, SV, 1.0, 0.0, 0.0, small)          # zero scale
    with pytest.raises(B.LraError):
        B.lra_phase_gradient_static(small, SU, SV, float("nan"), 0.0, 0.0, small)
    with pytest.raises(B.LraError):
        B.lra_phase_gradient_static(small, SU, SV, 1.0, 0.0, 0.0, small[:, :2])    # shapes differ
    lib = B.lib()
    assert lib.lra_phase_gradient_static(4, 4, 1, SU, SV, None, 1.0, 0.0, 0.0, 0, 0, None, None) == B.LRA_EINVAL
    B.lra_phase_gradient_static(small, SU, SV, 1.0, 0.0, 0.0, small)               # still usable after the failures
    torch.cuda.synchronize()
    assert B.lra_static_last_error() == ""

"""Pins of the CF-construction oracle (oracle/lra_ref_cf.c) against what the paper and the mathematics fix.

Table 1 defines a CF as the uv-plane convolution of the terms that are ON; SURVEY.md Sec. 8(f)
NEXT-2 computes it as the Fourier transform of their image-plane product.  None of these tests calls the CUDA path.
"""
import cmath
import math
import os

import numpy as np
import pytest

from oracle import lra_ref

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "table1_cf_terms.txt")


def _c0(S, os_):
    return (S - 1) // 2 * os_ + (os_ - 1 - os_ // 2)


def test_transform_is_the_cropped_fft_of_the_zero_padded_image():
    """'FFT, crop': sample j is bin (j - c0) of the DFT of the image zero-padded to n_img*os (numpy's FFT)."""
    rng = np.random.default_rng(11)
    n, os_, S = 12, 4, 7
    img = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    K = lra_ref.cf(n, os_, 0.3, S, aterm=img, normalise=False)
    M = n * os_
    P = np.zeros((M, M), dtype=np.complex128)
    P[M // 2 - n // 2: M // 2 - n // 2 + n, M // 2 - n // 2: M // 2 - n // 2 + n] = img
    F = np.fft.fftshift(np.fft.fft2(np.fft.ifftshift(P)))       # centred bins: index k + M/2
    j = np.arange(S * os_) - _c0(S, os_) + M // 2
    np.testing.assert_allclose(K, F[np.ix_(j, j)], rtol=0, atol=1e-11)


def test_point_like_image_gives_a_phase_ramp():
    """A single image pixel (m0, l0) of value z transforms to z e^{-2 pi i (off_j (m0-n/2) + off_i (l0-n/2))/n}:
    pins the orientation (v slow, u fast), the sign of the exponent and the sample offsets."""
    n, os_, S = 10, 3, 5
    a = np.zeros((n, n), dtype=np.complex128)
    m0, l0, z = 7, 2, 0.5 - 1.25j
    a[m0, l0] = z
    K = lra_ref.cf(n, os_, 0.2, S, aterm=a, normalise=False)
    c0 = _c0(S, os_)
    for j in (0, 4, c0, S * os_ - 1):
        for i in (0, 1, c0, S * os_ - 2):
            want = z * cmath.exp(-2j * math.pi * (((j - c0) / os_) * (m0 - n // 2) + ((i - c0) / os_) * (l0 - n // 2)) / n)
            assert abs(K[j, i] - want) < 1e-13
    assert abs(K[c0, c0] - z) < 1e-15      # the centre sample (offset 0) is the sum of the image


def test_dirichlet_closed_form():
    """All terms OFF: the image is all ones and the CF is the product of two Dirichlet kernels
    D(x) = sum_{a=-n/2}^{n/2-1} e^{-2 pi i x a / n} = e^{i pi x / n} sin(pi x) / sin(pi x / n)."""
    n, os_, S = 16, 4, 9
    K = lra_ref.cf(n, os_, 0.1, S, normalise=False)
    off = (np.arange(S * os_) - _c0(S, os_)) / os_
    with np.errstate(divide="ignore", invalid="ignore"):
        D = np.exp(1j * np.pi * off / n) * np.sin(np.pi * off) / np.sin(np.pi * off / n)
    D[off == 0] = n
    np.testing.assert_allclose(K, np.outer(D, D), rtol=0, atol=1e-10)


def test_w_term_values_at_chosen_pixels():
    """W = e^{2 pi i w (sqrt(1 - l^2 - m^2) - 1)}: with fov/n = 0.2 the pixel 3 right of centre has l = 0.6, so
    sqrt(1 - l^2) - 1 = -0.2 and w = 2.5 gives W = e^{-i pi} = -1, w = 1.25 gives -i; the centre pixel has W = 1 for
    every w; a pixel outside the unit circle takes sqrt(.) = 0, i.e. W = e^{-2 pi i w}."""
    n, fov = 16, 3.2
    def one_pixel(m, l, w):
        a = np.zeros((n, n), dtype=np.complex128)
        a[m, l] = 1.0
        return lra_ref.cf(n, 1, fov, 1, aterm=a, w_lambda=w, normalise=False)[0, 0]
    assert abs(one_pixel(8, 11, 2.5) - (-1)) < 1e-14
    assert abs(one_pixel(8, 11, 1.25) - (-1j)) < 1e-14
    assert abs(one_pixel(11, 8, 1.25) - (-1j)) < 1e-14        # the same along m
    assert abs(one_pixel(8, 8, 123.456) - 1) < 1e-15
    assert abs(one_pixel(13, 13, 0.25) - (-1j)) < 1e-14       # l = m = 1.0: outside the unit circle, W = e^{-i pi/2}
    # l = 0.6, m = 0.8 lies on the unit circle: sqrt(0) - 1 = -1
    assert abs(one_pixel(12, 11, 0.5) - (-1)) < 1e-7


def test_taper_is_separable_and_multiplies_the_pixel():
    n = 8
    t = np.linspace(0.3, 1.7, n)
    a = np.zeros((n, n), dtype=np.complex128)
    a[6, 1] = 2.0
    got = lra_ref.cf(n, 1, 0.1, 1, taper=t, aterm=a, normalise=False)[0, 0]
    assert abs(got - 2.0 * t[1] * t[6]) < 1e-14


def test_table1_rows_off_terms_are_identities():
    """Every row of Table 1 (tests/golden/table1_cf_terms.txt): a term that is OFF is the identity of the product."""
    rows = [l.split() for l in open(GOLDEN) if l.strip() and not l.startswith("#")]
    assert len(rows) == 6
    rng = np.random.default_rng(5)
    n, os_, S, fov, w = 12, 2, 5, 0.4, 37.0
    t = np.hanning(n + 2)[1:-1] + 0.1
    A = (1 + 0.1 * rng.normal(size=(n, n))) * np.exp(0.2j * rng.normal(size=(n, n)))
    for name, aterm, psterm, wterm, label in rows:
        on = dict(taper=t if psterm == "ON" else None, aterm=A if aterm == "ON" else None,
                  w_lambda=w if wterm == "ON" else 0.0)
        ident = dict(taper=t if psterm == "ON" else np.ones(n), aterm=A if aterm == "ON" else np.ones((n, n)),
                     w_lambda=on["w_lambda"])
        np.testing.assert_allclose(lra_ref.cf(n, os_, fov, S, **on), lra_ref.cf(n, os_, fov, S, **ident), rtol=0, atol=1e-13)
        assert set(label.replace("*", " ").split()) == {x for x, f in (("A", aterm), ("PS", psterm), ("W", wterm)) if f == "ON"}


def test_product_in_the_image_plane_is_convolution_in_the_uv_plane():
    """Convolution theorem on the full set of bins (S os = n os): the CF of PS x W is the circular convolution of the
    CF of PS with the CF of W, divided by M^2 (Table 1: 'PS * W')."""
    n, os_ = 5, 2
    S, M = n, n * os_
    t = np.array([0.2, 0.7, 1.0, 0.6, 0.3])
    fov, w = 1.2, 3.3
    Kps = lra_ref.cf(n, os_, fov, S, taper=t, normalise=False)
    Kw = lra_ref.cf(n, os_, fov, S, w_lambda=w, normalise=False)
    Kpw = lra_ref.cf(n, os_, fov, S, taper=t, w_lambda=w, normalise=False)
    conv = np.zeros((M, M), dtype=np.complex128)
    for j in range(M):
        for i in range(M):
            for q in range(M):
                for p in range(M):
                    conv[j, i] += Kps[q, p] * Kw[(j - q + _c0(S, os_)) % M, (i - p + _c0(S, os_)) % M]
    np.testing.assert_allclose(Kpw, conv / (M * M), rtol=0, atol=1e-11)


def test_w_reflection_symmetry():
    """With a real, symmetric taper the image of -w is the conjugate of the image of +w, so (odd os: the sample
    offsets are symmetric about 0)  K_{-w}[j][i] = conj(K_{+w}[so-1-j][so-1-i])."""
    n, os_, S = 14, 3, 7
    t = np.hanning(n + 1)[:-1]           # t[0] = 0 and t[a] = t[n - a]: symmetric on the raster [-n/2, n/2)
    assert t[0] == 0 and np.allclose(t[1:], t[1:][::-1])
    Kp = lra_ref.cf(n, os_, 0.5, S, taper=t, w_lambda=41.0)
    Km = lra_ref.cf(n, os_, 0.5, S, taper=t, w_lambda=-41.0)
    np.testing.assert_allclose(Km, np.conj(Kp[::-1, ::-1]), rtol=0, atol=1e-12)
    K0 = lra_ref.cf(n, os_, 0.5, S, taper=t)
    assert np.abs(K0.imag).max() < 1e-12                   # w = 0: real and symmetric image, real kernel


def test_normalisation():
    """R12: the samples of a CF sum to os^2, for a complex kernel too."""
    rng = np.random.default_rng(3)
    n, os_, S = 10, 4, 5
    A = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n)) + 3
    K = lra_ref.cf(n, os_, 0.3, S, taper=np.hanning(n + 2)[1:-1], w_lambda=12.0, aterm=A)
    assert abs(K.sum() - os_ * os_) < 1e-12
    Ku = lra_ref.cf(n, os_, 0.3, S, taper=np.hanning(n + 2)[1:-1], w_lambda=12.0, aterm=A, normalise=False)
    np.testing.assert_allclose(K, Ku * (os_ * os_ / Ku.sum()), rtol=0, atol=1e-13)


def test_brute_force_double_loop():
    """The definition written out for a tiny case, all three terms ON."""
    n, os_, S, fov, w = 6, 2, 3, 0.9, 2.2
    rng = np.random.default_rng(8)
    t = rng.uniform(0.5, 1.0, n)
    A = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    K = lra_ref.cf(n, os_, fov, S, taper=t, w_lambda=w, aterm=A, normalise=False)
    c0 = _c0(S, os_)
    for j in range(S * os_):
        for i in range(S * os_):
            acc = 0j
            for m in range(n):
                for l in range(n):
                    ll, mm = (l - n // 2) * fov / n, (m - n // 2) * fov / n
                    wt = cmath.exp(2j * math.pi * w * (math.sqrt(max(0.0, 1 - ll * ll - mm * mm)) - 1))
                    ph = -2 * math.pi * ((j - c0) / os_ * (m - n // 2) + (i - c0) / os_ * (l - n // 2)) / n
                    acc += t[l] * t[m] * A[m, l] * wt * cmath.exp(1j * ph)
            assert abs(K[j, i] - acc) < 1e-12


def test_matches_the_workload_generator_tables():
    """The seeded generator (paper_2508_17187_b200/workloads.py, numpy matrix products) builds its PS x W kernels from the
    same definition; its float32 tables agree with the oracle to float32 rounding."""
    from paper_2508_17187_b200 import workloads as W
    S, os_, s_taper, w, fov, n = 9, 4, 7, 850.0, 0.02, 64
    k = W.w_kernel(S, os_, s_taper, w, fov, n_img=n)
    taper1 = W.Prolate(s_taper)
    x = (np.arange(n) - n // 2) / (n / 2.0)
    t = taper1(x) / taper1.norm0
    K = lra_ref.cf(n, os_, fov, S, taper=t, w_lambda=w)
    assert np.abs(K - k).max() < 2e-7 * np.abs(K).max()


def test_bad_arguments():
    with pytest.raises(RuntimeError):
        lra_ref.cf(8, 2, 0.1, 4)     # even support

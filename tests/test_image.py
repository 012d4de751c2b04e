"""Pins of the image-plane oracle (oracle/lra_ref_image.c; Eq. 23) against
things other than itself: the O(N^4) double sum written out, numpy's FFT with explicit shifts (a library routine the
centred DFT reduces to), the closed form of one grid pixel, Parseval / the round trip F F^dagger = nx ny, and the
point-source chain grid -> image with the analytic taper of pin P7.  No GPU."""
import numpy as np
import pytest


def test_image_equals_the_double_sum_written_out(ref):
    rng = np.random.default_rng(5)
    ny, nx = 6, 8
    g = rng.standard_normal((2, ny, nx)) + 1j * rng.standard_normal((2, ny, nx))
    sw, cx, cy = np.array([3.0, 0.5]), rng.uniform(0.5, 2, nx), rng.uniform(0.5, 2, ny)
    want = np.zeros((2, ny, nx))
    for t in range(2):
        for m in range(ny):
            for l in range(nx):
                acc = 0.0 + 0.0j
                for y in range(ny):
                    for x in range(nx):
                        acc += g[t, y, x] * np.exp(2j * np.pi * ((x - nx // 2) * (l - nx // 2) / nx + (y - ny // 2) * (m - ny // 2) / ny))
                want[t, m, l] = acc.real * cx[l] * cy[m] / sw[t]
    got = ref.image(g, sw, cx, cy)
    assert np.abs(got - want).max() <= 1e-12 * np.abs(want).max()
    # dropping a factor must fail: the three factors are distinguishable
    assert np.abs(ref.image(g, None, cx, cy) - want).max() > 1e-3 * np.abs(want).max()
    assert np.abs(ref.image(g, sw, None, cy) - want).max() > 1e-3 * np.abs(want).max()


@pytest.mark.parametrize("ny,nx", [(16, 16), (12, 20)])
def test_image_equals_numpy_fft_with_shifts(ref, ny, nx):
    rng = np.random.default_rng(6)
    g = rng.standard_normal((ny, nx)) + 1j * rng.standard_normal((ny, nx))
    want = (np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(g))) * nx * ny).real
    got = ref.image(g)
    assert np.abs(got - want).max() <= 1e-11 * np.abs(want).max()
    img = rng.standard_normal((ny, nx))
    want_g = np.fft.fftshift(np.fft.fft2(np.fft.ifftshift(img)))
    got_g = ref.model_grid(img)
    assert np.abs(got_g - want_g).max() <= 1e-11 * np.abs(want_g).max()


def test_single_pixel_closed_form_and_sign(ref):
    """One unit grid pixel at spatial frequency (a, b) images to cos(2 pi (a l / nx + b m / ny)); an imaginary unit
    pixel to -sin(...): fixes the sign of the exponent and which axis is which."""
    ny, nx, a, b = 10, 14, 3, -2
    g = np.zeros((ny, nx), complex)
    g[ny // 2 + b, nx // 2 + a] = 1.0
    l, m = np.meshgrid(np.arange(nx) - nx // 2, np.arange(ny) - ny // 2)
    arg = 2 * np.pi * (a * l / nx + b * m / ny)
    assert np.abs(ref.image(g) - np.cos(arg)).max() <= 1e-12
    assert np.abs(ref.image(1j * g) + np.sin(arg)).max() <= 1e-12
    # the forward transform of a unit image pixel at (l0, m0): e^{-2 pi i (x l0 / nx + y m0 / ny)}
    img = np.zeros((ny, nx))
    img[ny // 2 + 1, nx // 2 - 4] = 1.0
    x, y = np.meshgrid(np.arange(nx) - nx // 2, np.arange(ny) - ny // 2)
    assert np.abs(ref.model_grid(img) - np.exp(-2j * np.pi * (x * (-4) / nx + y * 1 / ny))).max() <= 1e-12


def test_round_trip_and_adjointness(ref):
    rng = np.random.default_rng(8)
    ny, nx = 12, 16
    img = rng.standard_normal((3, ny, nx))
    back = ref.image(ref.model_grid(img))
    assert np.abs(back - nx * ny * img).max() <= 1e-10 * nx * ny            # F^dagger F = nx ny on real images
    g = rng.standard_normal((ny, nx)) + 1j * rng.standard_normal((ny, nx))
    # <F^dagger g, i> = Re <g, F i> for real images i
    lhs = np.sum(ref.image(g) * img[0])
    rhs = np.sum(np.conj(g) * ref.model_grid(img[0])).real
    assert abs(lhs - rhs) <= 1e-10 * abs(lhs)


def test_point_source_through_grid_and_image(ref):
    """Pin P7 carried through the new step: visibilities of a unit point source, gridded by the oracle, imaged,
    taper-corrected and normalised give ~1 at the source pixel and ~0 elsewhere (amplitude within the oversampling
    quantisation of the positions)."""
    from paper_2508_17187_b200 import workloads as W
    n, S, os_ = 32, 7, 16
    K = W.ps_kernel(S, os_)
    rng = np.random.default_rng(9)
    nvis = 4000
    u = rng.uniform(-n * 0.35, n * 0.35, (nvis, 2))
    l0, m0 = 3, -5
    vis = np.exp(-2j * np.pi * (u[:, 0] * l0 / n + u[:, 1] * m0 / n)).astype(np.complex64).reshape(nvis, 1, 1)
    uvw = np.concatenate([u, np.zeros((nvis, 1))], 1)
    rp = ref.RefPlan(n, n, 1, 1, os_, 1.0, 1.0, np.array([S], np.int32), np.array([0], np.int64), K.ravel(), tile=8, sort_mode=1)
    g, sw = rp.grid(uvw, np.array([299792458.0]), None, vis, np.ones((nvis, 1, 1), np.float32))
    # image of the gridding kernel (the taper): DTFT of the fx = fy = 0 taps, separable for the prolate kernel
    h, c0 = (S - 1) // 2, (S - 1) // 2 * os_ + os_ // 2 - 1
    taps = K[c0, c0 - h * os_:c0 + h * os_ + 1:os_].real / np.sqrt(K[c0, c0].real)     # 1-D factor of the outer product
    lm = np.arange(n) - n // 2
    taper = np.array([np.sum(taps * np.cos(2 * np.pi * np.arange(-h, h + 1) * q / n)) for q in lm])
    img = ref.image(g, sw, 1.0 / taper, 1.0 / taper)[0, 0]
    peak = np.unravel_index(np.argmax(img), img.shape)
    assert peak == (n // 2 + m0, n // 2 + l0)
    assert abs(img[peak] - 1.0) < 0.05
    rest = img.copy()
    rest[peak[0] - 2:peak[0] + 3, peak[1] - 2:peak[1] + 3] = 0       # the main lobe of the box-sampled uv plane
    assert np.abs(rest[4:-4, 4:-4]).max() < 0.3                       # sinc sidelobes of a uniformly filled square

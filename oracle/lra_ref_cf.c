/* lra_ref_cf.c -- CPU ORACLE for the construction of one convolution function (CF).  TEST INFRASTRUCTURE ONLY
 * (same rules as lra_ref.c: only tests/, __graft_entry__.smoke() and bench.py's oracle legs may use it; it shares
 * nothing with the CUDA path).
 *
 * What it is: the plain definition, in double precision, of the CF of Table 1: the convolution in
 * the uv plane of the terms that are ON -- the anti-aliasing taper PS, the A-term and the W-term -- which is the Fourier
 * transform of their PRODUCT in the image plane (convolution theorem; "PS x W x A in the
 * image plane, batched FFT, crop"), "constructed from ideal kernels" once, in PreCompute
 * (PAPER.md:335-343, 380).
 *
 * Readings (R24-R26):
 *   - image raster: n_img x n_img pixels spanning the field of view, pixel a at direction cosine
 *     l_a = (a - n_img/2) * fov / n_img (the same for m along the slow axis);
 *   - PS term: separable, taper[l] * taper[m], samples supplied by the caller; OFF = all ones;
 *   - A-term: complex image-plane pattern aterm[m][l] supplied by the caller; OFF = 1;
 *   - W-term: e^{2 pi i w (sqrt(1 - l^2 - m^2) - 1)} with w in wavelengths (the sign with which the generator of
 *     SURVEY.md Sec. 8(d) builds its tables); outside the unit circle the square root is taken as 0; OFF = w = 0;
 *   - transform: K[j][i] = sum_m sum_l img[m][l] e^{-2 pi i (off_j (m - n/2) + off_i (l - n/2)) / n}, where sample j of
 *     an oversampled kernel of support S sits off_j = (j - c0)/os pixels from the centre, c0 = ((S-1)/2) os +
 *     (os - 1 - os/2) (the storage convention of lra.h, R3).  Because off_j n / n_img = (j - c0) n / (n_img os), this is
 *     bin (j - c0) of the DFT of the image zero-padded to n_img*os pixels: "FFT, crop";
 *   - normalisation (R12): K is scaled so that the sum of all its samples is os^2 (complex division by the sum).
 *
 * The double sum is evaluated as the iterated sum (first over l, then over m) with the phases of the axis tabulated
 * once.  tests/test_cf.py pins it against numpy's FFT of the zero-padded image, the closed form of the Dirichlet
 * kernel, the w -> -w reflection symmetry, Table 1's ON/OFF rows, and the O(n^2 (S os)^2) double loop written out.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

static const double TWO_PI = 6.283185307179586476925286766559;

/* taper [n_img] or NULL; aterm [n_img][n_img] complex pairs or NULL; K [(S os)][(S os)] complex pairs (v slow). */
int lra_ref_cf(int32_t n_img, int32_t os, double fov_rad, const double* taper, double w_lambda, const double* aterm,
               int32_t S, int32_t normalise, double* K) {
  if (n_img < 1 || os < 1 || S < 1 || (S & 1) == 0 || !K) return 1;
  const int32_t n = n_img, so = S * os, h = (S - 1) / 2, c0 = h * os + (os - 1 - os / 2);
  double* img = (double*)malloc((size_t)n * n * 2 * sizeof(double));
  double* pc = (double*)malloc((size_t)so * n * sizeof(double)); /* cos, sin of 2 pi off_j (a - n/2) / n */
  double* ps = (double*)malloc((size_t)so * n * sizeof(double));
  double* row = (double*)malloc((size_t)n * so * 2 * sizeof(double)); /* after the sum over l: [m][i] */
  if (!img || !pc || !ps || !row) return 2;
  for (int32_t m = 0; m < n; ++m)
    for (int32_t l = 0; l < n; ++l) {
      const double ll = (double)(l - n / 2) * fov_rad / n, mm = (double)(m - n / 2) * fov_rad / n;
      const double r2 = ll * ll + mm * mm;
      const double nterm = sqrt(r2 < 1.0 ? 1.0 - r2 : 0.0) - 1.0;
      const double ph = TWO_PI * w_lambda * nterm;
      double re = cos(ph), im = sin(ph);
      if (taper) { re *= taper[l] * taper[m]; im *= taper[l] * taper[m]; }
      if (aterm) {
        const double ar = aterm[((size_t)m * n + l) * 2], ai = aterm[((size_t)m * n + l) * 2 + 1];
        const double t = re * ar - im * ai;
        im = re * ai + im * ar;
        re = t;
      }
      img[((size_t)m * n + l) * 2] = re;
      img[((size_t)m * n + l) * 2 + 1] = im;
    }
  for (int32_t j = 0; j < so; ++j)
    for (int32_t a = 0; a < n; ++a) {
      const double ph = TWO_PI * ((double)(j - c0) / os) * (double)(a - n / 2) / n;
      pc[(size_t)j * n + a] = cos(ph);
      ps[(size_t)j * n + a] = sin(ph);
    }
  for (int32_t m = 0; m < n; ++m)
    for (int32_t i = 0; i < so; ++i) {
      double sr = 0.0, si = 0.0;
      for (int32_t l = 0; l < n; ++l) { /* e^{-i phase}: (cos, -sin) */
        const double a = img[((size_t)m * n + l) * 2], b = img[((size_t)m * n + l) * 2 + 1];
        const double c = pc[(size_t)i * n + l], s = -ps[(size_t)i * n + l];
        sr += a * c - b * s;
        si += a * s + b * c;
      }
      row[((size_t)m * so + i) * 2] = sr;
      row[((size_t)m * so + i) * 2 + 1] = si;
    }
  double tr = 0.0, ti = 0.0;
  for (int32_t j = 0; j < so; ++j)
    for (int32_t i = 0; i < so; ++i) {
      double sr = 0.0, si = 0.0;
      for (int32_t m = 0; m < n; ++m) {
        const double a = row[((size_t)m * so + i) * 2], b = row[((size_t)m * so + i) * 2 + 1];
        const double c = pc[(size_t)j * n + m], s = -ps[(size_t)j * n + m];
        sr += a * c - b * s;
        si += a * s + b * c;
      }
      K[((size_t)j * so + i) * 2] = sr;
      K[((size_t)j * so + i) * 2 + 1] = si;
      tr += sr;
      ti += si;
    }
  if (normalise) { /* K *= os^2 / (tr + i ti) */
    const double d = tr * tr + ti * ti;
    if (d == 0.0) { free(img); free(pc); free(ps); free(row); return 3; }
    const double fr = (double)os * os * tr / d, fi = -(double)os * os * ti / d;
    for (size_t e = 0; e < (size_t)so * so; ++e) {
      const double a = K[e * 2], b = K[e * 2 + 1];
      K[e * 2] = a * fr - b * fi;
      K[e * 2 + 1] = a * fi + b * fr;
    }
  }
  free(img); free(pc); free(ps); free(row);
  return 0;
}

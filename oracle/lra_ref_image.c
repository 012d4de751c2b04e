/* lra_ref_image.c -- CPU ORACLE for the transforms either side of the gridding path.  TEST INFRASTRUCTURE ONLY
 * (same rules as lra_ref.c: only tests/, __graft_entry__.smoke() and bench.py's oracle legs may use it; it shares
 * nothing with the CUDA path).
 *
 * What it is: the plain definition, in double precision, of
 *   - the residual / dirty image of Eq. 23: I^R = F^dagger [gridded data], with the image-plane
 *     correction for the gridding taper and the sum-of-weights normalisation that SURVEY.md Sec. 8(f) NEXT-1 names;
 *   - the forward transform F of a model image onto the uv grid (Eq. 6 / Eq. 23: "D F I^M").
 * Readings (R17-R19): the transform is the CENTRED discrete Fourier transform that pins P6 / P7 of
 * lra_ref.c already use -- uv pixel (x, y) is spatial frequency (x - nx/2, y - ny/2), image pixel (l, m) is
 * direction (l - nx/2, m - ny/2) / n -- with e^{+2 pi i ...} from grid to image and e^{-2 pi i ...} back, no 1/N
 * factor in either direction; the taper correction is a separable per-pixel factor corr_x[l] * corr_y[m] supplied by
 * the caller (the reciprocal of the image of the gridding kernel); the normalisation divides by sumwt[t][p].
 *
 * The double sum is evaluated as the iterated sum (first over x, then over y), which is the same sum in a fixed
 * order, with the phases of an axis tabulated once; the outer loops may run on several OpenMP threads (every output
 * element is summed by one thread in the same order, so the result does not depend on the thread count).
 * tests/test_image.py pins it against the O(N^4) double loop written out, against numpy's FFT with explicit shifts,
 * against the closed form of a single grid pixel, and by the round trip F F^dagger = nx * ny.
 *
 * Layouts: grid[ngrid][ny][nx] complex double as pairs; image[ngrid][ny][nx] double; corr_x[nx], corr_y[ny] double or
 * NULL (=> 1); sumwt[ngrid] double or NULL (=> 1).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

static const double TWO_PI = 6.283185307179586476925286766559;

/* cos and sin of 2 pi (a - n/2)(b - n/2) / n for all a, b in [0, n): the phases of one axis, tabulated once so that the
 * sums below are plain multiply-adds (the table is the definition's exponent, evaluated once per (a, b) pair). */
static int phase_table(int32_t n, double** c, double** s) {
  *c = (double*)malloc((size_t)n * n * sizeof(double));
  *s = (double*)malloc((size_t)n * n * sizeof(double));
  if (!*c || !*s) return 2;
  for (int32_t a = 0; a < n; ++a)
    for (int32_t b = 0; b < n; ++b) {
      const double ph = TWO_PI * (double)(a - n / 2) * (double)(b - n / 2) / (double)n;
      (*c)[(size_t)a * n + b] = cos(ph);
      (*s)[(size_t)a * n + b] = sin(ph);
    }
  return 0;
}

/* image[g][m][l] = Re( sum_y sum_x grid[g][y][x] e^{+2 pi i ((x - nx/2)(l - nx/2)/nx + (y - ny/2)(m - ny/2)/ny)} )
 *                  * corr_x[l] * corr_y[m] / sumwt[g] */
int lra_ref_image(int32_t ngrid, int32_t ny, int32_t nx, const double* grid, const double* sumwt, const double* corr_x,
                  const double* corr_y, double* image) {
  if (ngrid < 1 || nx < 1 || ny < 1 || !grid || !image) return 1;
  double* row = (double*)malloc((size_t)ny * nx * 2 * sizeof(double)); /* after the sum over x: [y][l] */
  double *cx, *sx, *cy, *sy;
  if (!row || phase_table(nx, &cx, &sx) || phase_table(ny, &cy, &sy)) return 2;
  for (int32_t g = 0; g < ngrid; ++g) {
    const double* G = grid + (size_t)g * ny * nx * 2;
#pragma omp parallel for schedule(static)
    for (int32_t y = 0; y < ny; ++y)
      for (int32_t l = 0; l < nx; ++l) {
        double sr = 0.0, si = 0.0;
        for (int32_t x = 0; x < nx; ++x) {
          const double c = cx[(size_t)x * nx + l], s = sx[(size_t)x * nx + l];
          const double a = G[((size_t)y * nx + x) * 2], b = G[((size_t)y * nx + x) * 2 + 1];
          sr += a * c - b * s;
          si += a * s + b * c;
        }
        row[((size_t)y * nx + l) * 2] = sr;
        row[((size_t)y * nx + l) * 2 + 1] = si;
      }
#pragma omp parallel for schedule(static)
    for (int32_t m = 0; m < ny; ++m)
      for (int32_t l = 0; l < nx; ++l) {
        double sr = 0.0;
        for (int32_t y = 0; y < ny; ++y)
          sr += row[((size_t)y * nx + l) * 2] * cy[(size_t)y * ny + m] - row[((size_t)y * nx + l) * 2 + 1] * sy[(size_t)y * ny + m];
        double f = 1.0;
        if (corr_x) f *= corr_x[l];
        if (corr_y) f *= corr_y[m];
        if (sumwt) f /= sumwt[g];
        image[((size_t)g * ny + m) * nx + l] = sr * f;
      }
  }
  free(row); free(cx); free(sx); free(cy); free(sy);
  return 0;
}

/* grid[g][y][x] = sum_m sum_l image[g][m][l] * corr_x[l] * corr_y[m]
 *                 * e^{-2 pi i ((x - nx/2)(l - nx/2)/nx + (y - ny/2)(m - ny/2)/ny)} */
int lra_ref_model_grid(int32_t ngrid, int32_t ny, int32_t nx, const double* image, const double* corr_x,
                       const double* corr_y, double* grid) {
  if (ngrid < 1 || nx < 1 || ny < 1 || !grid || !image) return 1;
  double* row = (double*)malloc((size_t)ny * nx * 2 * sizeof(double)); /* after the sum over l: [m][x] */
  double *cx, *sx, *cy, *sy;
  if (!row || phase_table(nx, &cx, &sx) || phase_table(ny, &cy, &sy)) return 2;
  for (int32_t g = 0; g < ngrid; ++g) {
    const double* I = image + (size_t)g * ny * nx;
#pragma omp parallel for schedule(static)
    for (int32_t m = 0; m < ny; ++m)
      for (int32_t x = 0; x < nx; ++x) {
        double sr = 0.0, si = 0.0;
        for (int32_t l = 0; l < nx; ++l) {   /* e^{-i phase}: cos, -sin */
          double v = I[(size_t)m * nx + l];
          if (corr_x) v *= corr_x[l];
          if (corr_y) v *= corr_y[m];
          sr += v * cx[(size_t)x * nx + l];
          si -= v * sx[(size_t)x * nx + l];
        }
        row[((size_t)m * nx + x) * 2] = sr;
        row[((size_t)m * nx + x) * 2 + 1] = si;
      }
#pragma omp parallel for schedule(static)
    for (int32_t y = 0; y < ny; ++y)
      for (int32_t x = 0; x < nx; ++x) {
        double sr = 0.0, si = 0.0;
        for (int32_t m = 0; m < ny; ++m) {
          const double c = cy[(size_t)y * ny + m], s = -sy[(size_t)y * ny + m];
          const double a = row[((size_t)m * nx + x) * 2], b = row[((size_t)m * nx + x) * 2 + 1];
          sr += a * c - b * s;
          si += a * s + b * c;
        }
        grid[(((size_t)g * ny + y) * nx + x) * 2] = sr;
        grid[(((size_t)g * ny + y) * nx + x) * 2 + 1] = si;
      }
  }
  free(row); free(cx); free(sx); free(cy); free(sy);
  return 0;
}

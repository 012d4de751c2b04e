/* lra_ref_gain.c -- CPU ORACLE for the G-Jones solver fed by degridded model visibilities.  TEST INFRASTRUCTURE ONLY
 * (same rules as lra_ref.c; shares nothing with the CUDA path).
 *
 * What it is: Sec. 5.1 of arxiv 2508.17187 in double precision, step by step in the paper's order:
 *   Eq. 19: X_ij = sum over the solution interval of V^c_ij(t, nu) [V^Mod_ij(t, nu)]^{-1}
 *   Eq. 20: grad g_i = sum_{j != i} g_j X_ij w_ij / sum_{j != i} |g_j|^2 w_ij
 *   Eq. 21: g_i^{k+1} = (1 - alpha) g_i^k + alpha grad g_i
 *   exit: |g^{k+1} - g^k| < delta
 * Readings (R21-R23): Eq. 19 is taken as the WEIGHTED AVERAGE the text calls it ("averaging the data"):
 * X_ij = sum wt V^c / V^Mod / sum wt, and w_ij = sum wt (samples with wt = 0 or V^Mod = 0 are skipped; a baseline
 * without samples has w_ij = 0 and drops out of Eq. 20); the sum over j != i runs over both orderings of a baseline --
 * a baseline stored as (i, j) gives antenna i the term g_j X_ij w_ij and antenna j the term g_i conj(X_ij) w_ij, because
 * X_ji = conj(X_ij) for R_ij = X_ij - g_i conj(g_j); all antennas are updated from the gains of iteration k (Jacobi);
 * the exit test is on max_i |g_i^{k+1} - g_i^k|; one polarisation product (correlation) at a time, independently.
 *
 * Layouts: vis, model [nrow][nchan][ncorr] complex64 as float pairs; wt [nrow][nchan][ncorr] float; bl_index[nrow] int32
 * or NULL (=> row r belongs to baseline r % nbl); xsum [nbl][ncorr] complex double as pairs (ACCUMULATED INTO: the
 * running sum of wt V^c / V^Mod, not yet divided); wsum [nbl][ncorr] double; ant1, ant2 [nbl] int32;
 * gains [nant][ncorr] complex double as pairs, in: g^0, out: the solution.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

/* Eq. 19, numerator and denominator of the weighted average */
int lra_ref_gain_accumulate(int64_t nrow, int32_t nchan, int32_t ncorr, int32_t nbl, const int32_t* bl_index,
                            const float* vis, const float* model, const float* wt, double* xsum, double* wsum) {
  for (int64_t r = 0; r < nrow; ++r) {
    const int64_t b = bl_index ? bl_index[r] : r % nbl;
    if (b < 0 || b >= nbl) continue;
    for (int32_t c = 0; c < nchan; ++c)
      for (int32_t p = 0; p < ncorr; ++p) {
        const int64_t i = (r * nchan + c) * ncorr + p;
        const double w = wt[i], mr = model[2 * i], mi = model[2 * i + 1], vr = vis[2 * i], vi = vis[2 * i + 1];
        const double den = mr * mr + mi * mi;
        if (!(w > 0.0) || !(den > 0.0)) continue;
        /* V / M = V conj(M) / |M|^2 */
        xsum[(b * ncorr + p) * 2] += w * ((vr * mr + vi * mi) / den);
        xsum[(b * ncorr + p) * 2 + 1] += w * ((vi * mr - vr * mi) / den);
        wsum[b * ncorr + p] += w;
      }
  }
  return 0;
}

/* Eq. 20, 21 and the exit test; returns the number of iterations done in *iters */
int lra_ref_gain_solve(int32_t nant, int32_t nbl, int32_t ncorr, const int32_t* ant1, const int32_t* ant2,
                       const double* xsum, const double* wsum, double alpha, double delta, int32_t max_iter,
                       double* gains, int32_t* iters) {
  double* num = (double*)malloc((size_t)nant * 2 * sizeof(double));
  double* den = (double*)malloc((size_t)nant * sizeof(double));
  if (!num || !den) return 2;
  int32_t worst = 0;
  for (int32_t p = 0; p < ncorr; ++p) {
    int32_t k = 0;
    for (; k < max_iter; ++k) {
      for (int32_t a = 0; a < nant; ++a) num[2 * a] = num[2 * a + 1] = den[a] = 0.0;
      for (int32_t b = 0; b < nbl; ++b) {
        const double w = wsum[b * ncorr + p];
        if (!(w > 0.0)) continue;
        const int32_t i = ant1[b], j = ant2[b];
        const double xr = xsum[(b * ncorr + p) * 2] / w, xi = xsum[(b * ncorr + p) * 2 + 1] / w;   /* X_ij */
        const double gir = gains[(i * ncorr + p) * 2], gii = gains[(i * ncorr + p) * 2 + 1];
        const double gjr = gains[(j * ncorr + p) * 2], gji = gains[(j * ncorr + p) * 2 + 1];
        /* antenna i: g_j X_ij w */
        num[2 * i] += (gjr * xr - gji * xi) * w;
        num[2 * i + 1] += (gjr * xi + gji * xr) * w;
        den[i] += (gjr * gjr + gji * gji) * w;
        /* antenna j: g_i conj(X_ij) w */
        num[2 * j] += (gir * xr + gii * xi) * w;
        num[2 * j + 1] += (gii * xr - gir * xi) * w;
        den[j] += (gir * gir + gii * gii) * w;
      }
      double change = 0.0;
      for (int32_t a = 0; a < nant; ++a) {
        if (!(den[a] > 0.0)) continue;                /* an antenna without data keeps its gain */
        double* g = gains + (a * ncorr + p) * 2;
        const double nr = (1.0 - alpha) * g[0] + alpha * (num[2 * a] / den[a]);
        const double ni = (1.0 - alpha) * g[1] + alpha * (num[2 * a + 1] / den[a]);
        const double d = hypot(nr - g[0], ni - g[1]);
        if (d > change) change = d;
        g[0] = nr; g[1] = ni;
      }
      if (change < delta) { ++k; break; }
    }
    if (k > worst) worst = k;
  }
  if (iters) *iters = worst;
  free(num); free(den);
  return 0;
}

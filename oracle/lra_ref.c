/* lra_ref.c -- CPU ORACLE for the gridding / degridding path.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build,
 * load or call this file.  It shares no code, header, table or helper with the CUDA path under
 * paper_2508_17187_b200/csrc/, and the product never falls back to it.
 *
 * What it is: the plain definition of the operators of arxiv 2508.17187 written as the obvious nested
 * loops in double precision (build: gcc -O2 -ffp-contract=off -fopenmp, so every * and + rounds once):
 *   - gridding  G(c_ij): "accumulation on a grid at the pixel corresponding to u_ij" of c_ij * w_ij * V
 *     (Eq. 7; weights outside G as in Eq. 23);
 *   - degridding D(c_ij): the reverse operator with the same kernel (Eq. 6), read as
 *     the exact adjoint of G with unit weights (reading R7);
 *   - "re-ordering for runtime performance" read as a stable uv-tile bucket sort
 *     of the visibility-point indices (reading R5).
 * The paper does not give the resampling arithmetic; every such choice is a numbered reading in
 * DESIGN.md (R1..R15) and is restated next to the line that implements it.
 *
 * Pins (tests/test_oracle_pins.py, all run without a GPU): P1 adjoint identity, P2 1x1-CF histogram,
 * P3 sum(grid), P4 single-visibility patch / phase sign, P5 Hermitian symmetry, P6 tiny-grid closed
 * form through an independent DFT formula, P7 point source, P8 partition invariance, P9 bin checks
 * with exact rational arithmetic.  No function here is "parity unpinned".
 *
 * Layouts (all host pointers, caller-owned, row-major, last index fastest):
 *   uvw[nrow][3] double metres; freq[nchan] double Hz; cf_index[nrow][nchan] int32 or NULL (=> 0);
 *   vis[nrow][nchan][ncorr] complex64 as float pairs; wt[nrow][nchan][ncorr] float;
 *   tau[nchan][nterms] float or NULL (=> 1); grid[nterms][ncorr][ny][nx] complex double as pairs;
 *   sumwt[nterms][ncorr] double; CF kernel c: (S_c*os)^2 complex64 at cf_data + 2*cf_offset[c].
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
  int32_t nx, ny, ncorr, nterms, oversampling, tile, sort_mode;
  double scale_u, scale_v;
  int32_t n_cf;
  const int32_t* cf_support;
  const int64_t* cf_offset;
  const float* cf_data;
  int32_t tile_x; /* R5: uv tiles are tile_x wide (u) and tile tall (v); 0 => square, tile_x = tile */
} lra_ref_desc;

enum { LRA_REF_SORT_TILE = 0, LRA_REF_SORT_TILE_CF = 1 };

typedef struct {
  int32_t ix, iy, fx, fy, cf, valid;
} ref_point;

static int64_t floordiv64(int64_t a, int64_t b) {
  int64_t q = a / b, r = a % b;
  return (r != 0 && ((r < 0) != (b < 0))) ? q - 1 : q;
}

/* One axis of steps 1-2 of the definition.
 *   R1: origin pixel n/2, scale in pixels per wavelength, uvw in metres scaled per channel by nu/c.
 *   R2: position rounded ONCE on the oversampled coordinate, round-half-up via floor(x + 0.5), in
 *       fp64 with every operation rounded separately; pixel and phase are then split exactly in
 *       integers, so they can never disagree.  Returns 0 if the coordinate is not finite / far off. */
static int axis_index(double coord_m, double s, int32_t n, int32_t os, int64_t* pix, int64_t* ph) {
  double p = coord_m * s;
  p = p + (double)(n / 2);
  double t = p * (double)os;
  t = t + 0.5;
  t = floor(t);
  /* finite and within a few pixels of the grid; anything else cannot be valid (R4) and must not
   * reach the integer conversion */
  if (!(t >= -4.0 * (double)os && t <= ((double)n + 4.0) * (double)os)) return 0;
  int64_t P = (int64_t)t;
  int64_t i = floordiv64(P + os / 2, os);
  *pix = i;
  *ph = P - i * os; /* in [-(os/2), os - 1 - os/2]: [-os/2, os/2 - 1] for even os; 0 for os = 1 */
  return 1;
}

/* Steps 1-3: pixel, sub-pixel phase, CF and validity of visibility point (r, c). */
static ref_point locate(const lra_ref_desc* d, const double* uvw, const double* freq, const int32_t* cf_index,
                        int32_t nchan, int64_t r, int32_t c) {
  ref_point q;
  memset(&q, 0, sizeof q);
  q.ix = q.iy = -1;
  /* su[c] = (freq[c] / c_light) * scale_u : one division, one multiplication (R2) */
  double lam_inv = freq[c] / 299792458.0;
  double su = lam_inv * d->scale_u;
  double sv = lam_inv * d->scale_v;
  int64_t ix, iy, fx, fy;
  int ok = axis_index(uvw[3 * r + 0], su, d->nx, d->oversampling, &ix, &fx);
  ok &= axis_index(uvw[3 * r + 1], sv, d->ny, d->oversampling, &iy, &fy);
  int32_t cf = cf_index ? cf_index[r * (int64_t)nchan + c] : 0;
  if (!ok || cf < 0 || cf >= d->n_cf) return q;
  int32_t S = d->cf_support[cf], h = (S - 1) / 2;
  /* R4: a footprint that leaves the grid invalidates the whole visibility point */
  if (ix - h < 0 || ix + h > d->nx - 1 || iy - h < 0 || iy + h > d->ny - 1) return q;
  q.ix = (int32_t)ix; q.iy = (int32_t)iy; q.fx = (int32_t)fx; q.fy = (int32_t)fy; q.cf = cf; q.valid = 1;
  return q;
}

/* R3: tap (j, i) of kernel K_cf for phase (fy, fx): K[(j*os - fy) + c0][(i*os - fx) + c0]; kernel is
 * (S*os)^2, row-major, v slow.  c0 = h*os + f_max with f_max = os - 1 - os/2 the largest phase, so
 * that tap -h of phase f_max is sample 0: c0 = h*os + os/2 - 1 for even os, c0 = h for os = 1. */
static inline const float* tap_ptr(const lra_ref_desc* d, const ref_point* q, int32_t j, int32_t i) {
  int32_t os = d->oversampling, S = d->cf_support[q->cf], h = (S - 1) / 2;
  int64_t n = (int64_t)S * os, c0 = (int64_t)h * os + (os - 1 - os / 2);
  int64_t row = (int64_t)j * os - q->fy + c0, col = (int64_t)i * os - q->fx + c0;
  return d->cf_data + 2 * (d->cf_offset[q->cf] + row * n + col);
}

/* Step 7: sort key (R5). */
static uint64_t sort_key(const lra_ref_desc* d, const ref_point* q) {
  if (!q->valid) return UINT64_MAX;
  int32_t Ty = d->tile, Tx = d->tile_x > 0 ? d->tile_x : d->tile, os = d->oversampling;
  uint64_t ntx = (uint64_t)((d->nx + Tx - 1) / Tx);
  uint64_t tile_id = (uint64_t)(q->iy / Ty) * ntx + (uint64_t)(q->ix / Tx);
  if (d->sort_mode == LRA_REF_SORT_TILE) return tile_id;
  return ((tile_id * (uint64_t)d->n_cf + (uint64_t)q->cf) * (uint64_t)os + (uint64_t)(q->fy + os / 2)) * (uint64_t)os +
         (uint64_t)(q->fx + os / 2);
}

/* ---------------------------------------------------------------------------------------------- */
/* lra_ref_bin: index + stable sort.  Outputs: ix, iy (int32), fx, fy (int8), key (u64) per point
 * [nrow*nchan] (invalid: ix = iy = -1, fx = fy = 0, key = 2^64-1); perm[n_valid] u32 = stable sort of
 * point indices k = r*nchan + c by key, invalid dropped; tile_start[ntiles+1] u32 = first position in
 * perm whose tile id >= q; *n_valid.  Any output pointer may be NULL. */
typedef struct { uint64_t key; uint32_t k; } ref_kv;

static void merge_sort_kv(ref_kv* a, ref_kv* tmp, int64_t n) {
  /* bottom-up merge sort: stable by construction, no library comparator involved */
  for (int64_t w = 1; w < n; w *= 2) {
    for (int64_t lo = 0; lo < n; lo += 2 * w) {
      int64_t mid = lo + w < n ? lo + w : n, hi = lo + 2 * w < n ? lo + 2 * w : n;
      int64_t i = lo, j = mid, o = lo;
      while (i < mid && j < hi) tmp[o++] = (a[j].key < a[i].key) ? a[j++] : a[i++];
      while (i < mid) tmp[o++] = a[i++];
      while (j < hi) tmp[o++] = a[j++];
    }
    memcpy(a, tmp, (size_t)n * sizeof(ref_kv));
  }
}

int lra_ref_bin(const lra_ref_desc* d, int64_t nrow, int32_t nchan, const double* uvw, const double* freq,
                const int32_t* cf_index, int32_t* ix, int32_t* iy, int8_t* fx, int8_t* fy, uint64_t* key,
                uint32_t* perm, uint32_t* tile_start, int64_t* n_valid) {
  int64_t np = nrow * nchan;
  ref_kv* kv = (ref_kv*)malloc((size_t)(np > 0 ? np : 1) * sizeof(ref_kv));
  ref_kv* tmp = (ref_kv*)malloc((size_t)(np > 0 ? np : 1) * sizeof(ref_kv));
  if (!kv || !tmp) { free(kv); free(tmp); return 2; }
  int64_t nv = 0;
  for (int64_t r = 0; r < nrow; ++r)
    for (int32_t c = 0; c < nchan; ++c) {
      int64_t k = r * nchan + c;
      ref_point q = locate(d, uvw, freq, cf_index, nchan, r, c);
      uint64_t ky = sort_key(d, &q);
      if (ix) ix[k] = q.ix;
      if (iy) iy[k] = q.iy;
      if (fx) fx[k] = (int8_t)q.fx;
      if (fy) fy[k] = (int8_t)q.fy;
      if (key) key[k] = ky;
      if (q.valid) { kv[nv].key = ky; kv[nv].k = (uint32_t)k; ++nv; }
    }
  merge_sort_kv(kv, tmp, nv);
  if (perm) for (int64_t i = 0; i < nv; ++i) perm[i] = kv[i].k;
  if (n_valid) *n_valid = nv;
  if (tile_start) {
    int32_t Ty = d->tile, Tx = d->tile_x > 0 ? d->tile_x : d->tile;
    int64_t ntiles = (int64_t)((d->nx + Tx - 1) / Tx) * ((d->ny + Ty - 1) / Ty);
    uint64_t per_tile = 1;
    if (d->sort_mode == LRA_REF_SORT_TILE_CF) per_tile = (uint64_t)d->n_cf * d->oversampling * d->oversampling;
    int64_t pos = 0;
    for (int64_t q = 0; q <= ntiles; ++q) {
      while (pos < nv && kv[pos].key / per_tile < (uint64_t)q) ++pos;
      tile_start[q] = (uint32_t)pos;
    }
    tile_start[ntiles] = (uint32_t)nv;
  }
  free(kv); free(tmp);
  return 0;
}

/* ---------------------------------------------------------------------------------------------- */
/* lra_ref_grid: steps 1-5.  grid and sumwt are accumulated into.
 * nthreads > 1: each thread owns a band of grid rows, walks ALL points in index order and applies only
 * the taps whose row is in its band, so every pixel sees the single-thread summation order (bit-identical
 * result, no atomics, no extra grids).  sumwt is summed by one serial pass in index order. */
int lra_ref_grid(const lra_ref_desc* d, int64_t nrow, int32_t nchan, const double* uvw, const double* freq,
                 const int32_t* cf_index, const float* vis, const float* wt, const float* tau, double* grid,
                 double* sumwt, int32_t nthreads) {
  const int32_t nc = d->ncorr, nt = d->nterms, nx = d->nx, ny = d->ny;
  int64_t np = nrow * nchan;
  ref_point* pts = (ref_point*)malloc((size_t)(np > 0 ? np : 1) * sizeof(ref_point));
  if (!pts) return 2;
  for (int64_t r = 0; r < nrow; ++r)
    for (int32_t c = 0; c < nchan; ++c) pts[r * nchan + c] = locate(d, uvw, freq, cf_index, nchan, r, c);
  /* R6: sumwt = sum over valid points of wt*tau, no CF factor */
  if (sumwt)
    for (int64_t k = 0; k < np; ++k) {
      if (!pts[k].valid) continue;
      int32_t c = (int32_t)(k % nchan);
      for (int32_t t = 0; t < nt; ++t)
        for (int32_t p = 0; p < nc; ++p) {
          double tw = tau ? (double)tau[c * nt + t] : 1.0;
          sumwt[t * nc + p] += (double)wt[k * nc + p] * tw;
        }
    }
  if (nthreads < 1) nthreads = 1;
  int32_t nbands = nthreads == 1 ? 1 : nthreads * 8;
  if (nbands > ny) nbands = ny;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
#endif
  for (int32_t b = 0; b < nbands; ++b) {
    int32_t y0 = (int32_t)((int64_t)ny * b / nbands), y1 = (int32_t)((int64_t)ny * (b + 1) / nbands);
    for (int64_t k = 0; k < np; ++k) {
      const ref_point* q = &pts[k];
      if (!q->valid) continue;
      int32_t S = d->cf_support[q->cf], h = (S - 1) / 2;
      if (q->iy + h < y0 || q->iy - h >= y1) continue;
      int32_t c = (int32_t)(k % nchan);
      for (int32_t t = 0; t < nt; ++t) {
        double tw = tau ? (double)tau[c * nt + t] : 1.0;
        for (int32_t p = 0; p < nc; ++p) {
          /* step 5: val = wt * tau * vis */
          double w = (double)wt[k * nc + p] * tw;
          double vr = w * (double)vis[2 * (k * nc + p)], vi = w * (double)vis[2 * (k * nc + p) + 1];
          double* g = grid + 2 * ((int64_t)(t * nc + p) * ny * nx);
          for (int32_t j = -h; j <= h; ++j) {
            int32_t y = q->iy + j;
            if (y < y0 || y >= y1) continue;
            for (int32_t i = -h; i <= h; ++i) {
              const float* cfp = tap_ptr(d, q, j, i);
              double cr = (double)cfp[0], ci = (double)cfp[1];
              double* px = g + 2 * ((int64_t)y * nx + (q->ix + i));
              px[0] += cr * vr - ci * vi;
              px[1] += cr * vi + ci * vr;
            }
          }
        }
      }
    }
  }
  free(pts);
  return 0;
}

/* ---------------------------------------------------------------------------------------------- */
/* lra_ref_degrid: step 6.  V[r][c][p] = sum_t tau[c][t] * sum_{j,i} conj(C(j,i)) * grid[t][p][iy+j][ix+i];
 * no weights, no normalisation (R7); invalid points => 0 (R4); with vis_in: out = vis_in - V.
 * vis_out[nrow][nchan][ncorr] complex double. */
int lra_ref_degrid(const lra_ref_desc* d, int64_t nrow, int32_t nchan, const double* uvw, const double* freq,
                   const int32_t* cf_index, const double* grid, const float* tau, const float* vis_in,
                   double* vis_out, int32_t nthreads) {
  const int32_t nc = d->ncorr, nt = d->nterms, nx = d->nx, ny = d->ny;
  int64_t np = nrow * nchan;
  if (nthreads < 1) nthreads = 1;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 256) num_threads(nthreads)
#endif
  for (int64_t k = 0; k < np; ++k) {
    int64_t r = k / nchan;
    int32_t c = (int32_t)(k % nchan);
    ref_point q = locate(d, uvw, freq, cf_index, nchan, r, c);
    for (int32_t p = 0; p < nc; ++p) {
      double ar = 0.0, ai = 0.0;
      if (q.valid) {
        int32_t S = d->cf_support[q.cf], h = (S - 1) / 2;
        for (int32_t t = 0; t < nt; ++t) {
          double tw = tau ? (double)tau[c * nt + t] : 1.0;
          const double* g = grid + 2 * ((int64_t)(t * nc + p) * ny * nx);
          double sr = 0.0, si = 0.0;
          for (int32_t j = -h; j <= h; ++j)
            for (int32_t i = -h; i <= h; ++i) {
              const float* cfp = tap_ptr(d, &q, j, i);
              double cr = (double)cfp[0], ci = -(double)cfp[1]; /* conj */
              const double* px = g + 2 * ((int64_t)(q.iy + j) * nx + (q.ix + i));
              sr += cr * px[0] - ci * px[1];
              si += cr * px[1] + ci * px[0];
            }
          ar += tw * sr;
          ai += tw * si;
        }
      }
      if (vis_in) {
        ar = (double)vis_in[2 * (k * nc + p)] - ar;
        ai = (double)vis_in[2 * (k * nc + p) + 1] - ai;
      }
      vis_out[2 * (k * nc + p)] = ar;
      vis_out[2 * (k * nc + p) + 1] = ai;
    }
  }
  return 0;
}

/* ---------------------------------------------------------------------------------------------- */
/* Sampled outputs for full-size parity: the value of n_pix chosen grid pixels, each computed one by
 * one from the definition (walk all points, keep the taps that land on the pixel).
 * pix[n_pix][4] int32 = (t, p, y, x); out[n_pix] complex double. */
int lra_ref_grid_pixels(const lra_ref_desc* d, int64_t nrow, int32_t nchan, const double* uvw, const double* freq,
                        const int32_t* cf_index, const float* vis, const float* wt, const float* tau,
                        int32_t n_pix, const int32_t* pix, double* out, int32_t nthreads) {
  const int32_t nc = d->ncorr, nt = d->nterms;
  int64_t np = nrow * nchan;
  ref_point* pts = (ref_point*)malloc((size_t)(np > 0 ? np : 1) * sizeof(ref_point));
  if (!pts) return 2;
  if (nthreads < 1) nthreads = 1;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads)
#endif
  for (int64_t k = 0; k < np; ++k) pts[k] = locate(d, uvw, freq, cf_index, nchan, k / nchan, (int32_t)(k % nchan));
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
#endif
  for (int32_t s = 0; s < n_pix; ++s) {
    int32_t t = pix[4 * s], p = pix[4 * s + 1], y = pix[4 * s + 2], x = pix[4 * s + 3];
    double ar = 0.0, ai = 0.0;
    for (int64_t k = 0; k < np; ++k) {
      const ref_point* q = &pts[k];
      if (!q->valid) continue;
      int32_t S = d->cf_support[q->cf], h = (S - 1) / 2;
      int32_t j = y - q->iy, i = x - q->ix;
      if (j < -h || j > h || i < -h || i > h) continue;
      int32_t c = (int32_t)(k % nchan);
      double tw = tau ? (double)tau[c * nt + t] : 1.0;
      double w = (double)wt[k * nc + p] * tw;
      double vr = w * (double)vis[2 * (k * nc + p)], vi = w * (double)vis[2 * (k * nc + p) + 1];
      const float* cfp = tap_ptr(d, q, j, i);
      double cr = (double)cfp[0], ci = (double)cfp[1];
      ar += cr * vr - ci * vi;
      ai += cr * vi + ci * vr;
    }
    out[2 * s] = ar;
    out[2 * s + 1] = ai;
  }
  free(pts);
  return 0;
}

/* Degridded value of n_sel chosen points k (all correlations), each from the definition, reading a
 * complex64 grid (as the GPU holds it) converted exactly to double.  out[n_sel][ncorr] complex double. */
int lra_ref_degrid_points(const lra_ref_desc* d, int64_t nrow, int32_t nchan, const double* uvw, const double* freq,
                          const int32_t* cf_index, const float* grid_c64, const float* tau, const float* vis_in,
                          int32_t n_sel, const int64_t* sel, double* out) {
  const int32_t nc = d->ncorr, nt = d->nterms, nx = d->nx, ny = d->ny;
  (void)nrow;
  for (int32_t s = 0; s < n_sel; ++s) {
    int64_t k = sel[s];
    int32_t c = (int32_t)(k % nchan);
    ref_point q = locate(d, uvw, freq, cf_index, nchan, k / nchan, c);
    for (int32_t p = 0; p < nc; ++p) {
      double ar = 0.0, ai = 0.0;
      if (q.valid) {
        int32_t S = d->cf_support[q.cf], h = (S - 1) / 2;
        for (int32_t t = 0; t < nt; ++t) {
          double tw = tau ? (double)tau[c * nt + t] : 1.0;
          const float* g = grid_c64 + 2 * ((int64_t)(t * nc + p) * ny * nx);
          double sr = 0.0, si = 0.0;
          for (int32_t j = -h; j <= h; ++j)
            for (int32_t i = -h; i <= h; ++i) {
              const float* cfp = tap_ptr(d, &q, j, i);
              double cr = (double)cfp[0], ci = -(double)cfp[1];
              const float* px = g + 2 * ((int64_t)(q.iy + j) * nx + (q.ix + i));
              sr += cr * (double)px[0] - ci * (double)px[1];
              si += cr * (double)px[1] + ci * (double)px[0];
            }
          ar += tw * sr;
          ai += tw * si;
        }
      }
      if (vis_in) {
        ar = (double)vis_in[2 * (k * nc + p)] - ar;
        ai = (double)vis_in[2 * (k * nc + p) + 1] - ai;
      }
      out[2 * (s * nc + p)] = ar;
      out[2 * (s * nc + p) + 1] = ai;
    }
  }
  return 0;
}

/* ---------------------------------------------------------------------------------------------- */
/* The general kernel of Eq. 27 and the sparse Mueller matrix of CFs:
 *     c_ij = CF_ij(nu, w, t)  f(ds_i - ds_j)  e^{2 pi i [s_o - (s(P) + ds_i + ds_j)] . u}
 * Readings R27-R29: the exponent lost its ". u" in print (G1); u is the uv coordinate of the GRID PIXEL the
 * tap lands on, u_X = (X - nx/2) / scale_u wavelengths (v likewise), so the factor is a phase gradient across the kernel;
 * the caller supplies, per row, an index into a table of (f, dl, dm) with (dl, dm) = s_o - (s(P) + ds_i + ds_j) in
 * direction cosines (Table 2's four modes are four ways of filling that table).  A Mueller element e = (grid plane p_e,
 * visibility correlation q_e) has its own kernel index per visibility point: gridding adds CF_e (x) [wt v]_{q_e} to plane
 * p_e, degridding adds conj(c_e) . G_{p_e} to correlation q_e.  sumwt counts wt * tau on the DIAGONAL elements only (a
 * leakage term adds no weight); validity (R4) is per element, since the support is.
 *   elem_grid, elem_corr [n_elem]; cf_index[e] -> int32 [nrow][nchan] (NULL: kernel 0); vis, wt [nrow][nchan][ncorr_vis];
 *   po_table [n_po][3] double (NULL: f = 1, no gradient), po_index [nrow] (NULL: entry 0); grid [nterms][d->ncorr][ny][nx]. */
static void po_factor(const lra_ref_desc* d, const double* po_table, const int32_t* po_index, int64_t r, int32_t X,
                      int32_t Y, double sign, double* fr, double* fi) {
  if (!po_table) { *fr = 1.0; *fi = 0.0; return; }
  const double* e = po_table + 3 * (po_index ? po_index[r] : 0);
  double ux = (double)(X - d->nx / 2) / d->scale_u, vy = (double)(Y - d->ny / 2) / d->scale_v;
  double ph = sign * 6.283185307179586476925286766559 * (e[1] * ux + e[2] * vy);
  *fr = e[0] * cos(ph);
  *fi = e[0] * sin(ph);
}

int lra_ref_grid_awp(const lra_ref_desc* d, int64_t nrow, int32_t nchan, const double* uvw, const double* freq,
                     int32_t n_elem, const int32_t* elem_grid, const int32_t* elem_corr, const int32_t* const* cf_index,
                     int32_t ncorr_vis, const float* vis, const float* wt, const float* tau, const double* po_table,
                     const int32_t* po_index, double* grid, double* sumwt) {
  const int32_t ng = d->ncorr, nt = d->nterms, nx = d->nx, ny = d->ny;
  for (int64_t r = 0; r < nrow; ++r)
    for (int32_t c = 0; c < nchan; ++c) {
      int64_t k = r * nchan + c;
      for (int32_t e = 0; e < n_elem; ++e) {
        int32_t p = elem_grid[e], qc = elem_corr[e];
        if (p < 0 || p >= ng || qc < 0 || qc >= ncorr_vis) return 1;
        ref_point q = locate(d, uvw, freq, cf_index ? cf_index[e] : 0, nchan, r, c);
        if (!q.valid) continue;
        int32_t S = d->cf_support[q.cf], h = (S - 1) / 2;
        for (int32_t t = 0; t < nt; ++t) {
          double tw = tau ? (double)tau[c * nt + t] : 1.0;
          double w = (double)wt[k * ncorr_vis + qc] * tw;
          double vr = w * (double)vis[2 * (k * ncorr_vis + qc)], vi = w * (double)vis[2 * (k * ncorr_vis + qc) + 1];
          if (sumwt && p == qc) sumwt[t * ng + p] += w;
          double* g = grid + 2 * ((int64_t)(t * ng + p) * ny * nx);
          for (int32_t j = -h; j <= h; ++j)
            for (int32_t i = -h; i <= h; ++i) {
              const float* cfp = tap_ptr(d, &q, j, i);
              double fr, fi;
              po_factor(d, po_table, po_index, r, q.ix + i, q.iy + j, 1.0, &fr, &fi);
              double cr = (double)cfp[0] * fr - (double)cfp[1] * fi, ci = (double)cfp[0] * fi + (double)cfp[1] * fr;
              double* px = g + 2 * ((int64_t)(q.iy + j) * nx + (q.ix + i));
              px[0] += cr * vr - ci * vi;
              px[1] += cr * vi + ci * vr;
            }
        }
      }
    }
  return 0;
}

/* vis_out[nrow][nchan][ncorr_vis] complex double = (vis_in or 0) - sum_e [q_e = q] sum_t tau sum_taps conj(c_e) G[t][p_e] */
int lra_ref_degrid_awp(const lra_ref_desc* d, int64_t nrow, int32_t nchan, const double* uvw, const double* freq,
                       int32_t n_elem, const int32_t* elem_grid, const int32_t* elem_corr, const int32_t* const* cf_index,
                       int32_t ncorr_vis, const double* grid, const float* tau, const double* po_table,
                       const int32_t* po_index, const float* vis_in, double* vis_out) {
  const int32_t ng = d->ncorr, nt = d->nterms, nx = d->nx, ny = d->ny;
  for (int64_t r = 0; r < nrow; ++r)
    for (int32_t c = 0; c < nchan; ++c) {
      int64_t k = r * nchan + c;
      for (int32_t qc = 0; qc < ncorr_vis; ++qc) vis_out[2 * (k * ncorr_vis + qc)] = vis_out[2 * (k * ncorr_vis + qc) + 1] = 0.0;
      for (int32_t e = 0; e < n_elem; ++e) {
        int32_t p = elem_grid[e], qc = elem_corr[e];
        if (p < 0 || p >= ng || qc < 0 || qc >= ncorr_vis) return 1;
        ref_point q = locate(d, uvw, freq, cf_index ? cf_index[e] : 0, nchan, r, c);
        if (!q.valid) continue;
        int32_t S = d->cf_support[q.cf], h = (S - 1) / 2;
        for (int32_t t = 0; t < nt; ++t) {
          double tw = tau ? (double)tau[c * nt + t] : 1.0;
          const double* g = grid + 2 * ((int64_t)(t * ng + p) * ny * nx);
          double sr = 0.0, si = 0.0;
          for (int32_t j = -h; j <= h; ++j)
            for (int32_t i = -h; i <= h; ++i) {
              const float* cfp = tap_ptr(d, &q, j, i);
              double fr, fi;
              po_factor(d, po_table, po_index, r, q.ix + i, q.iy + j, 1.0, &fr, &fi);
              /* conj(c f e^{i ph}) */
              double cr = (double)cfp[0] * fr - (double)cfp[1] * fi, ci = -((double)cfp[0] * fi + (double)cfp[1] * fr);
              const double* px = g + 2 * ((int64_t)(q.iy + j) * nx + (q.ix + i));
              sr += cr * px[0] - ci * px[1];
              si += cr * px[1] + ci * px[0];
            }
          vis_out[2 * (k * ncorr_vis + qc)] += tw * sr;
          vis_out[2 * (k * ncorr_vis + qc) + 1] += tw * si;
        }
      }
      for (int32_t qc = 0; qc < ncorr_vis; ++qc) {
        double ar = vis_out[2 * (k * ncorr_vis + qc)], ai = vis_out[2 * (k * ncorr_vis + qc) + 1];
        if (vis_in) {
          ar = (double)vis_in[2 * (k * ncorr_vis + qc)] - ar;
          ai = (double)vis_in[2 * (k * ncorr_vis + qc) + 1] - ai;
        }
        vis_out[2 * (k * ncorr_vis + qc)] = ar;
        vis_out[2 * (k * ncorr_vis + qc) + 1] = ai;
      }
    }
  return 0;
}

/* dst (+)= f e^{sign 2 pi i (dl u_X + dm v_Y)} src, all planes: the same factor applied to a whole grid (a group of
 * visibilities that share one pointing term; Table 2 "mosaic imaging, no PO correction"). */
int lra_ref_phase_gradient(const lra_ref_desc* d, int32_t nplanes, const double* src, double f, double dl, double dm,
                           int32_t conjugate, int32_t accumulate, double* dst) {
  double e[3] = {f, dl, dm};
  for (int32_t g = 0; g < nplanes; ++g)
    for (int32_t Y = 0; Y < d->ny; ++Y)
      for (int32_t X = 0; X < d->nx; ++X) {
        double fr, fi;
        po_factor(d, e, 0, 0, X, Y, conjugate ? -1.0 : 1.0, &fr, &fi);
        int64_t o = 2 * (((int64_t)g * d->ny + Y) * d->nx + X);
        double a = src[o], b = src[o + 1];
        double rr = a * fr - b * fi, ri = a * fi + b * fr;
        if (accumulate) { dst[o] += rr; dst[o + 1] += ri; } else { dst[o] = rr; dst[o + 1] = ri; }
      }
  return 0;
}

int lra_ref_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

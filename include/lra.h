/* lra.h -- C ABI of liblra: gridding (G) and degridding (D) of radio-interferometric visibilities on
 * one NVIDIA B200 (sm_100a).
 *
 * Operations (arxiv 2508.17187; line numbers are /root/reference/PAPER.md):
 *   G(c_ij): resample irregularly sampled weighted visibilities onto the regular uv grid, "accumulation
 *            on a grid at the pixel corresponding to u_ij"            -- Eq. 7
 *   D(c_ij): the reverse operator, resampling the gridded model at the visibility coordinates
 *            (model prediction V^Mod)                                 -- Eq. 6
 *   W_ij [V - V^Mod]: weights outside G, residual between D and G     -- Eq. 23 / 26
 *   c_ij = CF_ij(nu, w, t): "in practice a kernel applies to a set of data points"; the caller picks the
 *            kernel of every visibility point through cf_index        -- Eq. 27
 *   re-ordering of the data for runtime performance (PreSolvePrep / InLoopPrep)  -- PAPER.md:345, 429
 *   one-time caching of the kernels (PreCompute)                      -- PAPER.md:207, 335-343, 380
 * The resampling arithmetic the paper leaves open is fixed by readings R1..R15 in DESIGN.md.
 *
 * Call chain:  lra_plan_create -> lra_bin -> lra_grid / lra_degrid (any number, any order) -> lra_plan_destroy
 *
 * Conventions
 *   - "device" pointers are CUDA device memory on the plan's device, owned by the caller (e.g. allocated by
 *     PyTorch); the library never frees them and does not keep them past the stream work of the call that
 *     received them -- EXCEPT the geometry arrays given to lra_bin (uvw_m is not kept; see lra_bin).
 *   - "host" pointers are ordinary host memory, read during the call only.
 *   - Every call returns an lra_status.  No exceptions cross the ABI.  Calls enqueue work on the plan's
 *     stream and return without synchronising unless stated otherwise.
 *   - A visibility point k = r*nchan + c is one (row, channel); its ncorr samples share position and kernel.
 *   - complex64 = two consecutive floats (re, im).
 */
#ifndef LRA_H_
#define LRA_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  LRA_OK = 0,
  LRA_EINVAL = 1, /* bad argument (null pointer, size out of range, even support, ...) */
  LRA_ENOMEM = 2, /* host or device allocation failed                                   */
  LRA_ECUDA = 3,  /* a CUDA runtime call failed; see lra_last_cuda_error                */
  LRA_ESTATE = 4  /* call out of order (lra_grid before lra_bin, ...)                   */
} lra_status;

enum { LRA_SORT_TILE = 0, LRA_SORT_TILE_CF = 1 };

typedef struct lra_plan lra_plan; /* opaque */

typedef struct {
  int32_t nx, ny;         /* grid size in pixels; u along x (fastest), v along y; origin pixel (nx/2, ny/2) [R1] */
  int32_t ncorr, nterms;  /* grids per call = nterms*ncorr; 1 <= ncorr <= 4, 1 <= nterms <= 4                  */
  int32_t oversampling;   /* os >= 1: sub-pixel phases per pixel of the CF table [R3]                        */
  int32_t tile;           /* uv-tile height (v) in pixels used by the bucket sort, power of two in [4, 1024];
                             0 = the library default, 8 x 8 tiles [R5]                                               */
  int32_t sort_mode;      /* LRA_SORT_TILE | LRA_SORT_TILE_CF [R5]                                             */
  double scale_u, scale_v; /* pixels per wavelength along u and v; sign allowed [R1]                            */
  int32_t n_cf;           /* number of kernels in the CF table                                                 */
  const int32_t* cf_support; /* host [n_cf]: support S_c in pixels, odd, 1 <= S_c <= 129                        */
  const int64_t* cf_offset;  /* host [n_cf]: element (complex64) offset of kernel c inside cf_data              */
  const void* cf_data;    /* host OR device (e.g. lra_cf_generate's output; the unified address space tells which),
                             complex64: kernel c is (S_c*os)^2 samples, row-major, v slow; sample m of a
                             row sits (m - c0)/os pixels from the kernel centre, c0 = h*os + (os-1-os/2) [R3]   */
  int32_t device;         /* CUDA device ordinal                                                               */
  void* stream;           /* cudaStream_t all work of this plan is enqueued on (NULL = legacy default stream)  */
  int32_t tile_x;         /* uv-tile width (u) in pixels, power of two in [4, 1024]; 0 = square tiles (= tile)  */
} lra_plan_desc;

/* PreCompute: validates the descriptor, copies the CF table to the device and re-lays
 * every oversampled kernel into phase-major slabs [cf][fy][fx][S][tile_x + S - 1] (zero padded rows) so that
 * the S*S taps one visibility point needs are one contiguous piece.  Synchronises the plan's stream before returning (the host table may be freed).
 * Errors: LRA_EINVAL, LRA_ENOMEM, LRA_ECUDA.  *out is NULL on failure. */
int lra_plan_create(lra_plan** out, const lra_plan_desc* desc);

/* Frees everything the plan owns (CF slabs, bin arrays, scratch).  Synchronises the plan's stream. */
int lra_plan_destroy(lra_plan* p);

/* Re-ordering: for every visibility point computes grid pixel (ix, iy), sub-pixel phase
 * (fx, fy), validity [R2, R4] and the sort key [R5], then stable-sorts the valid point indices by key (the
 * per-tile start offsets follow from the sorted keys and are produced when lra_bin_export asks for them).  The result
 * stays in the plan and is consumed by lra_grid / lra_degrid.
 *   nrow, nchan : npoints = nrow*nchan must be < 2^31
 *   uvw_m       : device double [nrow][3], baseline coordinates in metres
 *   freq_hz     : HOST double [nchan]  (small; the per-channel scale (freq/c)*scale is formed on the host)
 *   cf_index    : device int32 [nrow][nchan] kernel of every point, or NULL (=> kernel 0)
 * The input arrays are not referenced after the call's stream work completes.
 * Synchronises the plan's stream ONCE, between its two passes over the sorted points (the host sizes the work lists of
 * lra_grid / lra_degrid from the per-class counts), and again whenever the plan's arrays have to grow.  The few hundred
 * bytes that cross the bus inside the call (the per-channel scales, the list sizes) go through kernels on pinned, mapped
 * memory, not through cudaMemcpy, so the call does not queue behind bulk transfers the caller has in flight on other
 * streams.
 * Errors: LRA_EINVAL, LRA_ENOMEM (growing the plan's bin arrays), LRA_ECUDA. */
int lra_bin(lra_plan* p, int64_t nrow, int32_t nchan, const double* uvw_m, const double* freq_hz,
            const int32_t* cf_index);

/* Copies the bin result out for checking (all device pointers, each may be NULL to skip it):
 *   ix, iy int32 [npoints], fx, fy int8 [npoints], key uint64 [npoints]  (invalid point: ix = iy = -1,
 *   fx = fy = 0, key = 2^64-1); perm uint32 [npoints] (first n_valid entries meaningful);
 *   tile_start uint32 [ntiles+1], ntiles = ceil(nx/tile_x)*ceil(ny/tile); n_valid: HOST int64.
 * Synchronises the plan's stream.  Errors: LRA_ESTATE before lra_bin. */
int lra_bin_export(lra_plan* p, int32_t* ix, int32_t* iy, int8_t* fx, int8_t* fy, uint64_t* key, uint32_t* perm,
                   uint32_t* tile_start, int64_t* n_valid);

/* Gridding (Eq. 7 with the weights of Eq. 23):
 *   grid[t][p][iy+j][ix+i] += CF[cf][fy][fx][j][i] * (wt[k][p] * tau[c][t] * vis[k][p])   for all taps (j, i)
 *   sumwt[t][p]            += wt[k][p] * tau[c][t]                                         [R6]
 * over the valid points of the last lra_bin.  fp32 multiply-add, fp32 accumulation.
 *   vis_c64  : device complex64 [nrow][nchan][ncorr]
 *   wt       : device float [nrow][nchan][ncorr]   (flags are expressed as weight 0 [R4])
 *   tau      : device float [nchan][nterms] Taylor weights, or NULL (=> 1) [R11]
 *   grid_c64 : device complex64 [nterms][ncorr][ny][nx], ACCUMULATED INTO (caller zeroes it)
 *   sumwt    : device double [nterms][ncorr], accumulated into; may be NULL
 * Errors: LRA_ESTATE before lra_bin, LRA_EINVAL, LRA_ECUDA. */
int lra_grid(lra_plan* p, const void* vis_c64, const float* wt, const float* tau, void* grid_c64, double* sumwt);

/* Degridding (Eq. 6; exact adjoint of lra_grid with unit weights [R7]):
 *   V[k][p] = sum_t tau[c][t] * sum_{j,i} conj(CF[cf][fy][fx][j][i]) * grid[t][p][iy+j][ix+i]
 *   vis_out[k][p] = vis_in ? vis_in[k][p] - V[k][p] : V[k][p]        (fused residual of Eq. 23)
 * Invalid points get V = 0.  vis_out is overwritten for ALL nrow*nchan*ncorr samples.
 *   grid_c64   : device complex64 [nterms][ncorr][ny][nx], read only
 *   vis_in_c64 : device complex64 [nrow][nchan][ncorr] or NULL;  vis_out_c64: device, same shape
 *                (vis_out may alias vis_in)
 * Errors: LRA_ESTATE before lra_bin, LRA_EINVAL, LRA_ECUDA. */
int lra_degrid(lra_plan* p, const void* grid_c64, const float* tau, const void* vis_in_c64, void* vis_out_c64);

/* The transforms either side of the path (Eq. 23: I^R = F^dagger G W [...];
 * PAPER.md:346 "UpdateDir"), readings R17-R19 of DESIGN.md.  nx and ny must be even.
 *
 * lra_image: the residual / dirty image of the gridded data,
 *   image[t][p][m][l] = Re( sum_{y,x} grid[t][p][y][x] e^{+2 pi i ((x-nx/2)(l-nx/2)/nx + (y-ny/2)(m-ny/2)/ny)} )
 *                       * corr_x[l] * corr_y[m] / sumwt[t][p]
 * (centred inverse DFT without 1/N, the image-plane correction for the gridding taper as a separable factor, and the
 * sum-of-weights normalisation).  cuFFT C2C does the transform; the sign / correction / normalisation kernels are the
 * library's own.
 *   grid_c64 : device complex64 [nterms][ncorr][ny][nx], read only
 *   sumwt    : device double [nterms][ncorr] or NULL (=> 1);  corr_x: device float [nx] or NULL (=> 1);  corr_y: [ny]
 *   image    : device float [nterms][ncorr][ny][nx], overwritten
 * lra_model_grid: the forward transform of a model image onto the uv grid (the "F I^M" that lra_degrid reads),
 *   grid[t][p][y][x] = sum_{m,l} image[t][p][m][l] corr_x[l] corr_y[m] e^{-2 pi i (...)}      (grid overwritten).
 * The plan keeps a complex scratch grid and the cuFFT plan (allocated on first use).
 * Errors: LRA_EINVAL (odd nx / ny, NULL grid / image), LRA_ENOMEM, LRA_ECUDA (also any cuFFT failure). */
int lra_image(lra_plan* p, const void* grid_c64, const double* sumwt, const float* corr_x, const float* corr_y,
              float* image);
int lra_model_grid(lra_plan* p, const float* image, const float* corr_x, const float* corr_y, void* grid_c64);

/* The G-Jones solver fed by degridded model visibilities (Sec. 5.1),
 * readings R21-R23 of DESIGN.md.  Plan-free: device ordinal and cudaStream_t are arguments; both calls only enqueue.
 *
 * lra_gain_accumulate, Eq. 19 over one solution interval:
 *   xsum[b][p] += sum wt * V[k][p] / M[k][p],  wsum[b][p] += sum wt     over the samples k of baseline b with wt > 0, M != 0
 * (so that X_ij = xsum / wsum, the weighted average, and w_ij = wsum).  Ratio and sums in double.
 *   bl_index : device int32 [nrow], baseline of every row, or NULL (=> row r belongs to baseline r % nbl)
 *   vis_c64, model_c64 : device complex64 [nrow][nchan][ncorr] (model = lra_degrid's output without vis_in)
 *   wt : device float [nrow][nchan][ncorr];  xsum: device complex double [nbl][ncorr];  wsum: device double [nbl][ncorr];
 *   both ACCUMULATED INTO (caller zeroes them; partitions of the interval may be added call by call).
 * lra_gain_solve, Eq. 20 / 21 for every correlation independently, from the gains given:
 *   grad g_i = sum_b [i = ant1: g_j X_b w_b | i = ant2: g_j conj(X_b) w_b] / sum_b |g_j|^2 w_b   (j = the other antenna)
 *   g_i <- (1 - alpha) g_i + alpha grad g_i    (all antennas from the gains of iteration k)
 * until max_i |g_i^{k+1} - g_i^k| < delta or max_iter iterations.
 *   ant1, ant2 : device int32 [nbl];  gains: device complex double [nant][ncorr], in: g^0, out: the solution;
 *   iters : device int32, the iterations done (largest over the correlations), or NULL.   nant <= 1024.
 * Errors: LRA_EINVAL, LRA_ECUDA. */
int lra_gain_accumulate(int32_t device, void* stream, int64_t nrow, int32_t nchan, int32_t ncorr, int32_t nbl,
                        const int32_t* bl_index, const void* vis_c64, const void* model_c64, const float* wt,
                        double* xsum, double* wsum);
int lra_gain_solve(int32_t device, void* stream, int32_t nant, int32_t nbl, int32_t ncorr, const int32_t* ant1,
                   const int32_t* ant2, const double* xsum, const double* wsum, double alpha, double delta,
                   int32_t max_iter, double* gains, int32_t* iters);

/* ---- PreCompute: construction of the CF table on the device ----------------------
 * Table 1 configures a CF as the uv-plane convolution of the terms that are ON -- the anti-aliasing
 * prolate-spheroidal taper PS, the A-term, the W-term -- "constructed from ideal kernels", computed once in
 * PreCompute or on demand by the CFCache.  The convolution is evaluated as the Fourier
 * transform of the product of the terms in the image plane (readings R24-R26 in DESIGN.md):
 *   img[m][l] = taper[l] taper[m] * aterm[a_c][m][l] * e^{2 pi i w_c (sqrt(1 - l^2 - m^2) - 1)},
 *               l = (l_index - n_img/2) fov_rad / n_img, likewise m; sqrt of a negative number taken as 0;
 *   K_c[j][i] = sum_m sum_l img[m][l] e^{-2 pi i (off_j (m - n_img/2) + off_i (l - n_img/2)) / n_img},
 *               off_j = (j - c0)/os, c0 as in lra_plan_desc.cf_data (= the n_img*os-point DFT of the zero-padded image,
 *               cropped to the (S_c os)^2 samples about the centre);
 *   normalise != 0: K_c is scaled (complex) so that its samples sum to os^2.
 * A term is OFF when its pointer is NULL: taper NULL = PSTerm OFF, aterm NULL (n_aterm 0) = ATerm OFF, cf_w NULL = WTerm
 * OFF; the six rows of Table 1 are the six combinations with at least one term ON.  Arithmetic is fp64, the result is
 * rounded once to complex64.  A caller grows a table "with usage" by calling again with the new kernels
 * and offsets past the old ones. */
typedef struct {
  int32_t n_img;             /* image raster is n_img x n_img over the field of view, 2 <= n_img <= 512                */
  int32_t oversampling;      /* os, as in lra_plan_desc                                                               */
  double fov_rad;            /* field of view spanned by the raster, in direction-cosine units (radians), > 0         */
  const double* taper;       /* DEVICE double [n_img] or NULL: separable image-plane taper                            */
  int32_t n_aterm;           /* number of A-term patterns (0 = ATerm OFF)                                             */
  const void* aterm;         /* DEVICE complex64 [n_aterm][n_img][n_img] (m slow, l fast) or NULL                     */
  int32_t n_cf;              /* kernels to build                                                                      */
  const int32_t* cf_support; /* host [n_cf]: support S_c, odd, 1 <= S_c <= 129                                        */
  const int64_t* cf_offset;  /* host [n_cf]: element offset of kernel c in cf_data (regions must not overlap)         */
  const double* cf_w;        /* host [n_cf]: w of kernel c in wavelengths, or NULL (WTerm OFF)                        */
  const int32_t* cf_aterm;   /* host [n_cf]: A-term pattern of kernel c, or NULL (pattern 0 for all)                  */
  int32_t normalise;         /* != 0: scale every kernel to sum os^2 [R12]                                            */
  int32_t device;            /* CUDA device ordinal                                                                   */
  void* stream;              /* cudaStream_t the work is enqueued on                                                  */
} lra_cf_desc;

/* Writes the n_cf kernels into cf_data (DEVICE complex64, caller-owned, large enough for every offset + (S_c os)^2).
 * Allocates and frees its own work buffers (<= ~256 MB) and synchronises the stream before returning.
 * Errors: LRA_EINVAL (bad argument; also a kernel whose samples sum to 0 or NaN when normalise != 0 -- the other kernels
 * are still written), LRA_ENOMEM, LRA_ECUDA (lra_cf_last_cuda_error() returns the cudaError_t of this thread's last
 * failure). */
int lra_cf_generate(const lra_cf_desc* desc, void* cf_data_c64);
int lra_cf_last_cuda_error(void);

/* ---- the data-dependent terms of Eq. 27 and per-element Mueller CFs ----------------
 *   c_ij(P, nu, w) = CF_ij(nu, w, t)  f(ds_i - ds_j)  e^{2 pi i [s_o - (s(P) + ds_i + ds_j)] . u}      (Eq. 27)
 * "the rest of the terms ... represents the data-dependent perturbations applied on-the-fly"; s_o, s(P) and
 * the antenna pointing offsets ds_i are input meta-data (Table 2).  Readings R27-R29: u is the
 * uv coordinate of the grid pixel a tap lands on, u_X = (X - nx/2)/scale_u, v_Y = (Y - ny/2)/scale_v (wavelengths); the
 * caller reduces the meta-data to a table po_table[n_po][3] = (f, dl, dm), (dl, dm) = s_o - (s(P) + ds_i + ds_j) in
 * direction cosines, and a per-row index po_index[nrow] into it.  Gridding uses c f e^{+2 pi i (dl u_X + dm v_Y)},
 * degridding its conjugate; sumwt carries no f [R6].  Table 2's modes: single pointing without PO = the plain calls;
 * mosaic without PO = one call per pointing with po_index NULL (every row uses entry 0: the tiled kernels run unchanged
 * and the factor is applied to the grid once); with PO correction = per-row entries (direct kernels).
 *   po_table : HOST double [n_po][3], 1 <= n_po <= 2^20, finite;  po_index : DEVICE int32 [nrow] or NULL; rows whose index
 *   is outside [0, n_po) are skipped (they add nothing to the grid; their model visibility is 0).  Other arguments as
 *   lra_grid / lra_degrid.  The first call with po_index NULL allocates one scratch grid in the plan.
 * lra_phase_gradient: dst (+)= f e^{+-2 pi i (dl u_X + dm v_Y)} src on all nterms*ncorr planes of a grid (- with
 *   conjugate != 0; += with accumulate != 0; src == dst allowed without accumulate).
 * Errors: LRA_EINVAL, LRA_ESTATE (before lra_bin), LRA_ENOMEM, LRA_ECUDA. */
int lra_phase_gradient(lra_plan* p, const void* src_c64, double f, double dl, double dm, int32_t conjugate,
                       int32_t accumulate, void* dst_c64);
int lra_grid_po(lra_plan* p, const void* vis_c64, const float* wt, const float* tau, int32_t n_po, const double* po_table,
                const int32_t* po_index, void* grid_c64, double* sumwt);
int lra_degrid_po(lra_plan* p, const void* grid_c64, const float* tau, int32_t n_po, const double* po_table,
                  const int32_t* po_index, const void* vis_in_c64, void* vis_out_c64);

/* lra_phase_gradient for callers that must not allocate (CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc).  The operation is lra_phase_gradient's (the pointing factor of Eq. 27, reading R27):
 *   dst[g][Y][X] (+)= f e^{+-2 pi i (dl (X - nx/2)/scale_u + dm (Y - ny/2)/scale_v)} src[g][Y][X],  g < nplanes,
 * "-" with conjugate != 0, "+=" with accumulate != 0; src == dst allowed without accumulate.  It takes no plan: the
 * geometry is passed in, the CURRENT device is used and the two kernels are enqueued on `stream` (a cudaStream_t; NULL =
 * the default stream); the call returns without synchronising.
 *   src, dst : DEVICE complex64 [nplanes][ny][nx], caller-owned;  scale_u, scale_v : pixels per wavelength, non-zero.
 * Scratch: the nx + ny phasors the kernels share live in a file-scope device array of LRA_STATIC_MAX_AXES complex64
 * (512 KiB, held by every GPU that loads the library until the process exits).  The call issues no cudaMalloc, cudaFree or
 * allocating library call; the first call on a device resolves the array's address (cudaGetSymbolAddress) and reads the
 * SM count, so make one call per device before capturing a graph.  Every call on a device uses the SAME array and
 * rewrites the entries it reads (nothing needs clearing): calls whose kernels overlap on the GPU (different streams
 * without a dependency between them, or concurrent host threads on different streams) race -- order them on one stream or
 * with events.
 * Errors: LRA_EINVAL (NULL src / dst, nx, ny or nplanes < 1, nx + ny > LRA_STATIC_MAX_AXES, NaN factor, zero scale),
 * LRA_ECUDA; lra_static_last_error() returns a description of this thread's last failure ("" after a success). */
#define LRA_STATIC_MAX_AXES 65536
int lra_phase_gradient_static(int32_t nx, int32_t ny, int32_t nplanes, double scale_u, double scale_v, const void* src_c64,
                              double f, double dl, double dm, int32_t conjugate, int32_t accumulate, void* dst_c64,
                              void* stream);
const char* lra_static_last_error(void);

/* Sparse Mueller matrix of CFs: element e = (grid plane elem_grid[e], visibility correlation elem_corr[e])
 * has its own kernel index per visibility point, cf_index[e] (HOST array of n_elem DEVICE pointers to int32 [nrow][nchan],
 * NULL entry = kernel 0).  Gridding adds CF_e (x) [wt V]_{elem_corr[e]} to plane elem_grid[e]; degridding subtracts (adds,
 * without vis_in) conj(c_e) . G_{elem_grid[e]} from correlation elem_corr[e].  Only the elements listed are computed (the
 * matrix "can be configured to include only terms that are significant").  sumwt [ngrid] receives wt * tau of the DIAGONAL
 * elements (elem_grid == elem_corr) only [R29].  The plan must have ncorr = nterms = 1 (one plane of geometry); every
 * element re-bins it (lra_bin with the element's indices), so the plan is left binned for the last element.
 *   vis, wt : DEVICE [nrow][nchan][ncorr_vis]; grid : DEVICE complex64 [ngrid][ny][nx]; tau : DEVICE [nchan] or NULL;
 *   n_po = 0 disables the pointing term (po_table, po_index as above otherwise); n_elem <= 16, ncorr_vis, ngrid <= 4.
 * Both synchronise the stream before returning (they free their gather buffers). */
int lra_grid_mueller(lra_plan* p, int64_t nrow, int32_t nchan, const double* uvw_m, const double* freq_hz, int32_t n_elem,
                     const int32_t* elem_grid, const int32_t* elem_corr, const int32_t* const* cf_index, int32_t ncorr_vis,
                     const void* vis_c64, const float* wt, const float* tau, int32_t n_po, const double* po_table,
                     const int32_t* po_index, int32_t ngrid, void* grid_c64, double* sumwt);
int lra_degrid_mueller(lra_plan* p, int64_t nrow, int32_t nchan, const double* uvw_m, const double* freq_hz, int32_t n_elem,
                       const int32_t* elem_grid, const int32_t* elem_corr, const int32_t* const* cf_index, int32_t ncorr_vis,
                       int32_t ngrid, const void* grid_c64, const float* tau, int32_t n_po, const double* po_table,
                       const int32_t* po_index, const void* vis_in_c64, void* vis_out_c64);

/* Number of kernel launches the plan has enqueued since creation (for bench.py's gpu_launches). */
int64_t lra_launch_count(const lra_plan* p);

/* Sum over the valid points of the last lra_bin of S^2 (taps per correlation and term); synchronises. */
int lra_tap_count(lra_plan* p, int64_t* n_valid, int64_t* sum_s2);

/* Selects the gridding / degridding kernel variant: 0 = default (fastest verified), other values are
 * listed in DESIGN.md (1 = plain global-atomic gridder kept as the "before" profile). */
int lra_set_variant(lra_plan* p, int32_t grid_variant, int32_t degrid_variant);

/* Measurement aids (not on the hot path; synchronous).  lra_diag_fma_tflops: FP32 FMA throughput of `device`
 * in TFLOP/s from an FMA-only kernel -- the compute term of the gridding roofline.
 * lra_diag_l2_gbs: read bandwidth in GB/s of an `mbytes`-MiB buffer kept in L2 -- the bound on CF-slab traffic. */
int lra_diag_fma_tflops(int device, double* tflops);
int lra_diag_l2_gbs(int device, int mbytes, double* gbs);

const char* lra_strerror(int code);
/* cudaGetErrorString of the last failing CUDA call of this plan ("" if none). */
const char* lra_last_cuda_error(const lra_plan* p);

#ifdef __cplusplus
}
#endif
#endif /* LRA_H_ */

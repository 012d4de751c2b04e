// lra_internal.cuh -- plan object and helpers shared by the translation units of liblra.so.
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "lra.h"

// One sorted visibility point as the gridder / degridder consume it (16 bytes, one LDG.128).
//   x: ix | iy << 16        (grid pixel of the footprint CENTRE; nx, ny <= 32768)
//   y: slab offset in 16-byte units (float offset >> 2; every slab is 16-byte aligned)
//   z: k = r*nchan + c      (index of the point in the caller's arrays)
//   w: S | cf << 8          (support in pixels, kernel number)
typedef uint4 lra_rec;

#define LRA_NCLASS 65  // support classes: class (S - 1) / 2 for S = 1, 3, .., 129
#define LRA_NAUX 4     // internal streams the per-class launches of one call are spread over
#define LRA_MAX_DEVICES 64

struct lra_plan {
  // ---- descriptor (host copies) ----
  int32_t nx, ny, ncorr, nterms, os, tile, tile_x, sort_mode, n_cf;   // tiles are tile_x wide (u) by tile tall (v)
  double scale_u, scale_v;
  int device;
  cudaStream_t stream;
  std::vector<int32_t> cf_support;
  std::vector<int64_t> slab_off;   // float offset of slab (cf, 0, 0) in `slabs`
  std::vector<int32_t> slab_stride;  // floats per slab of kernel cf: 2 * lra_slab_complex(S, tile_x)
  int32_t max_support;
  int32_t ntx, nty, ntiles;
  // ---- device: CF store ----
  float* slabs;             // [cf][fy][fx] phase-major slabs of interleaved complex taps, see lra_slab_complex()
  int64_t slab_elems;       // total floats
  int32_t* d_cf_support;    // [n_cf]
  int64_t* d_slab_off;      // [n_cf]
  // ---- device: bin state ----
  int64_t npoints, capacity;
  int64_t nrow;
  int32_t nchan;
  bool binned;
  int32_t *ix, *iy;
  int8_t *fx, *fy;
  uint64_t* key;            // exported key per point
  uint64_t *skey[2];        // radix-sort key double buffer
  uint32_t *sval[2];        // radix-sort value double buffer; sorted result ends in sval[sorted_buf]
  int sorted_buf;
  uint32_t* hist;           // radix histograms
  int64_t hist_capacity;
  uint32_t* tile_start;     // [ntiles + 1]; filled on demand by lra_bin_export (nothing else reads it)
  bool tile_start_done;
  unsigned long long per_tile;   // keys per tile of the last lra_bin
  lra_rec* urec;            // [npoints] the records in caller order (written by the index kernel)
  lra_rec* rec;             // [npoints] sorted records (first n_valid meaningful)
  unsigned long long* counters;  // see lra_pipe.cuh
  double *d_su, *d_sv;      // per-channel scale tables
  int32_t su_capacity;
  // ---- work lists of the region kernels (lra_work.cu; geometry only, rebuilt by every lra_bin) ----
  uint4* work;              // items of all classes, grouped by class
  int64_t work_capacity;
  uint32_t* batch;          // batch records (16 words each), grouped by class; an item's are consecutive
  int64_t batch_capacity;   // batches
  uint4* pw;                // [npoints] per sorted position: {word, k | fallback << 31, step masks / chunk range} (lra_pipe.cuh)
  int64_t pw_capacity;      // points
  float* prep;              // gridder: wt*tau*V of every sorted point, FFMA2 operand form; degridder: sorted results
  int64_t prep_capacity;    // floats
  int64_t n_items[LRA_NCLASS], item_off[LRA_NCLASS];     // items per support class, first item of the class in `work`
  int64_t n_batches[LRA_NCLASS], batch_off[LRA_NCLASS];  // batches per class, first batch of the class in `batch`
  cudaStream_t aux[LRA_NAUX];          // per-class launches run concurrently on these, forked from / joined to `stream`
  cudaEvent_t ev_fork, ev_join[LRA_NAUX];
  // ---- image-plane transforms (lra_image.cu) ----
  float2* fft_work;         // complex scratch [nterms*ncorr][ny][nx]
  int fft_plan;             // cufftHandle (0 = none yet)
  bool fft_ready;
  // ---- Eq. 27 terms (lra_awp.cu) ----
  void* awp_buf;            // gradient phasor table (nx + ny complex) and the uploaded (f, dl, dm) table
  size_t awp_bytes;
  float2* po_scratch;       // one grid [nterms*ncorr][ny][nx], allocated by the first call that needs it
  // ---- pinned, mapped host memory for the few words that cross the bus inside lra_bin: written / read by tiny kernels,
  //      so that they never queue behind a caller's bulk transfers on the copy engines ----
  unsigned long long* h_counts;   // [256] list sizes, device -> host
  double* h_scale;                // [2 * h_scale_capacity] per-channel scales, host -> device
  int32_t h_scale_capacity;
  // ---- misc ----
  int32_t grid_variant, degrid_variant;
  int64_t launches;
  cudaError_t last_err;
  int sm_count;
};

// Slab layout (one slab = the S*S taps of one kernel at one sub-pixel phase, what one visibility point needs).
// A region kernel works on a REGION of RX = S + tile_x - 1 columns (tile + halo) whose pixels are numbered
// e = y*RX + x, and it reads the tap that a point with footprint origin (ox, oy) puts on pixel e at the linear
// slab index e - (oy*RX + ox).  So a slab is stored with the region's pitch, as interleaved COMPLEX values (one
// 8-byte shared-memory load gives a lane its tap): tap (j, i), 0 <= j, i < S, at complex index j*RX + i, and the
// RX - S pad values that end each row ZERO.  A lane that looks at a pixel beside the footprint therefore reads a
// zero instead of branching (the zeros before and after the slab live in shared memory, lra_pipe.cuh).
// The slab is rounded up to an even number of complex values (16 bytes) so that one TMA bulk copy moves it.
__host__ __device__ inline int lra_slab_complex(int S, int tile_x) { return (S * (S + tile_x - 1) + 1) & ~1; }
__host__ __device__ inline int lra_tap_index(int S, int tile_x, int j, int i) { return j * (S + tile_x - 1) + i; }

#define LRA_CUDA(p, call)                         \
  do {                                            \
    cudaError_t e__ = (call);                     \
    if (e__ != cudaSuccess) {                     \
      if (p) (p)->last_err = e__;                 \
      return e__ == cudaErrorMemoryAllocation ? LRA_ENOMEM : LRA_ECUDA; \
    }                                             \
  } while (0)

#define LRA_LAUNCH_CHECK(p)                       \
  do {                                            \
    (p)->launches++;                              \
    LRA_CUDA(p, cudaGetLastError());              \
  } while (0)

// implemented in lra_grid.cu / lra_degrid.cu / lra_bin.cu / lra_work.cu
int lra_grid_impl(lra_plan* p, const float2* vis, const float* wt, const float* tau, float2* grid, double* sumwt);
int lra_degrid_impl(lra_plan* p, const float2* grid, const float* tau, const float2* vis_in, float2* vis_out);
int lra_build_work(lra_plan* p);
int lra_bin_impl(lra_plan* p, int64_t nrow, int32_t nchan, const double* uvw, const double* freq_host,
                 const int32_t* cf_index);

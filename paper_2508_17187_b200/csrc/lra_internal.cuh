// lra_internal.cuh -- plan object and helpers shared by the translation units of liblra.so.
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "lra.h"

// One sorted visibility point as the gridder / degridder consume it (16 bytes, one LDG.128).
//   x: ix | iy << 16        (grid pixel of the footprint CENTRE; nx, ny <= 32768)
//   y: slab element offset >> 1 (slabs are padded to an even number of complex64 => 16-byte aligned)
//   z: k = r*nchan + c      (index of the point in the caller's arrays)
//   w: S | cf << 8          (support in pixels, kernel number)
typedef uint4 lra_rec;

struct lra_plan {
  // ---- descriptor (host copies) ----
  int32_t nx, ny, ncorr, nterms, os, tile, sort_mode, n_cf;
  double scale_u, scale_v;
  int device;
  cudaStream_t stream;
  std::vector<int32_t> cf_support;
  std::vector<int64_t> slab_off;   // element offset of slab (cf, 0, 0) in `slabs`
  std::vector<int32_t> slab_stride;  // elements per slab of kernel cf: S*S rounded up to even
  int32_t max_support;
  int32_t ntx, nty, ntiles;
  // ---- device: CF store ----
  float2* slabs;            // [cf][fy][fx][S][S] phase-major, each slab 16-byte aligned
  int64_t slab_elems;
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
  uint32_t* tile_start;     // [ntiles + 1]
  lra_rec* rec;             // [npoints] sorted records (first n_valid meaningful)
  unsigned long long* counters;  // [0] n_valid, [1] sum S^2, [2..] scratch
  double *d_su, *d_sv;      // per-channel scale tables
  int32_t su_capacity;
  // ---- gridder work list ----
  void* work;               // uint4 work items for the tiled gridder
  uint32_t* item_off;       // [ntiles + 1] first work item of every tile
  int64_t work_capacity;
  // ---- misc ----
  int32_t grid_variant, degrid_variant;
  int64_t launches;
  cudaError_t last_err;
  int sm_count;
};

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

// implemented in lra_grid.cu / lra_degrid.cu / lra_bin.cu
int lra_grid_impl(lra_plan* p, const float2* vis, const float* wt, const float* tau, float2* grid, double* sumwt);
int lra_degrid_impl(lra_plan* p, const float2* grid, const float* tau, const float2* vis_in, float2* vis_out);
int lra_build_work(lra_plan* p);
void lra_scan_kernel_launch(lra_plan* p, uint32_t* a, long long m);
int lra_bin_impl(lra_plan* p, int64_t nrow, int32_t nchan, const double* uvw, const double* freq_host,
                 const int32_t* cf_index);

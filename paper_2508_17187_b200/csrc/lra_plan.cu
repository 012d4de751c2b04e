// lra_plan.cu -- plan life cycle, CF ingest (PreCompute) and the thin C-ABI entry
// points that validate arguments and forward to the kernels' host drivers.
#include <new>
#include <string.h>

#include <nvtx3/nvToolsExt.h>

#include "lra_pipe.cuh"

// NVTX range over one ABI call (one range per call; header-only NVTX 3, a no-op without a profiler).
struct lra_nvtx_range {
  explicit lra_nvtx_range(const char* name) { nvtxRangePushA(name); }
  ~lra_nvtx_range() { nvtxRangePop(); }
};

// Re-lay one oversampled kernel into phase-major slabs of interleaved complex taps (reading
// R3; layout in lra_internal.cuh):  tap (j + h, i + h) of slab (fyi, fxi) = K[(j*os - fy) + c0][(i*os - fx) + c0],
//   fy = fyi - os/2, c0 = h*os + (os-1-os/2).
// One thread per output complex value; the padding values are zero-filled.
__global__ void lra_relayout_kernel(const float2* __restrict__ K, float2* __restrict__ slab, int S, int os,
                                    int slab_complex, int tile_x) {
  const int h = (S - 1) / 2;
  const int rx = S + tile_x - 1;
  const int c0 = h * os + (os - 1 - os / 2);
  const int64_t n = (int64_t)os * os * slab_complex;
  const int64_t ld = (int64_t)S * os;
  for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
    const int phase = (int)(e / slab_complex), t = (int)(e % slab_complex);
    float2 v = make_float2(0.f, 0.f);
    const int jj = t / rx, ii = t - jj * rx;
    if (jj < S && ii < S) {
      const int fyi = phase / os, fxi = phase % os;
      const int j = jj - h, i = ii - h;
      const int row = j * os - (fyi - os / 2) + c0, col = i * os - (fxi - os / 2) + c0;
      v = K[row * ld + col];
    }
    slab[e] = v;
  }
}

static int is_pow2(int x) { return x > 0 && (x & (x - 1)) == 0; }

extern "C" int lra_plan_create(lra_plan** out, const lra_plan_desc* d) {
  lra_nvtx_range nvtx_("lra_plan_create");
  if (!out) return LRA_EINVAL;
  *out = nullptr;
  if (!d || d->nx < 1 || d->ny < 1 || d->nx > 32768 || d->ny > 32768) return LRA_EINVAL;
  if (d->ncorr < 1 || d->ncorr > 4 || d->nterms < 1 || d->nterms > 4) return LRA_EINVAL;
  if (d->oversampling < 1 || d->oversampling > 64) return LRA_EINVAL;
  // tile = 0: the library's default, 8 x 8; tile_x = 0 with tile != 0: square tiles
  int tile = d->tile == 0 ? 8 : d->tile;
  int tile_x = d->tile_x == 0 ? (d->tile == 0 ? 8 : tile) : d->tile_x;
  if (!is_pow2(tile) || tile < 4 || tile > 1024 || !is_pow2(tile_x) || tile_x < 4 || tile_x > 1024) return LRA_EINVAL;
  if (d->sort_mode != LRA_SORT_TILE && d->sort_mode != LRA_SORT_TILE_CF) return LRA_EINVAL;
  if (d->n_cf < 1 || d->n_cf > (1 << 24) || !d->cf_support || !d->cf_offset || !d->cf_data) return LRA_EINVAL;
  if (!(d->scale_u == d->scale_u) || !(d->scale_v == d->scale_v)) return LRA_EINVAL;
  for (int c = 0; c < d->n_cf; ++c) {
    int S = d->cf_support[c];
    if (S < 1 || S > 129 || (S & 1) == 0 || d->cf_offset[c] < 0) return LRA_EINVAL;
  }
  lra_plan* p = new (std::nothrow) lra_plan();
  if (!p) return LRA_ENOMEM;
  p->nx = d->nx; p->ny = d->ny; p->ncorr = d->ncorr; p->nterms = d->nterms; p->os = d->oversampling;
  p->tile = tile; p->tile_x = tile_x; p->sort_mode = d->sort_mode; p->n_cf = d->n_cf;
  p->scale_u = d->scale_u; p->scale_v = d->scale_v;
  p->device = d->device; p->stream = (cudaStream_t)d->stream;
  p->ntx = (p->nx + tile_x - 1) / tile_x; p->nty = (p->ny + tile - 1) / tile; p->ntiles = p->ntx * p->nty;
  p->last_err = cudaSuccess;
  p->cf_support.assign(d->cf_support, d->cf_support + d->n_cf);
  p->slab_off.resize(d->n_cf);
  p->slab_stride.resize(d->n_cf);
  int64_t total = 0, max_in = 0;
  p->max_support = 1;
  for (int c = 0; c < d->n_cf; ++c) {
    int S = p->cf_support[c];
    p->slab_stride[c] = 2 * lra_slab_complex(S, tile_x);
    p->slab_off[c] = total;
    total += (int64_t)p->os * p->os * p->slab_stride[c];
    int64_t n_in = (int64_t)S * p->os * S * p->os;
    if (n_in > max_in) max_in = n_in;
    if (S > p->max_support) p->max_support = S;
  }
  if ((total >> 2) >= (int64_t)1 << 32) { delete p; return LRA_EINVAL; }
  p->slab_elems = total;

  float2* staging = nullptr;
  auto fail = [&](int code) { if (staging) cudaFree(staging); lra_plan_destroy(p); return code; };
#define CK(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { p->last_err = e__; \
    return fail(e__ == cudaErrorMemoryAllocation ? LRA_ENOMEM : LRA_ECUDA); } } while (0)
  CK(cudaSetDevice(p->device));
  CK(cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, p->device));
  CK(cudaMalloc(&p->slabs, (size_t)total * sizeof(float)));
  CK(cudaMalloc(&p->d_cf_support, (size_t)d->n_cf * sizeof(int32_t)));
  CK(cudaMalloc(&p->d_slab_off, (size_t)d->n_cf * sizeof(int64_t)));
  CK(cudaMalloc(&p->counters, LRA_NCOUNTER * sizeof(unsigned long long)));
  CK(cudaMemsetAsync(p->counters, 0, LRA_NCOUNTER * sizeof(unsigned long long), p->stream));
  for (int s = 0; s < LRA_NAUX; ++s) {
    CK(cudaStreamCreateWithFlags(&p->aux[s], cudaStreamNonBlocking));
    CK(cudaEventCreateWithFlags(&p->ev_join[s], cudaEventDisableTiming));
  }
  CK(cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming));
  CK(cudaMalloc(&p->tile_start, (size_t)(p->ntiles + 1) * sizeof(uint32_t)));
  CK(cudaHostAlloc(&p->h_counts, 256 * sizeof(unsigned long long), cudaHostAllocMapped));
  CK(cudaMemcpyAsync(p->d_cf_support, p->cf_support.data(), (size_t)d->n_cf * sizeof(int32_t), cudaMemcpyHostToDevice, p->stream));
  CK(cudaMemcpyAsync(p->d_slab_off, p->slab_off.data(), (size_t)d->n_cf * sizeof(int64_t), cudaMemcpyHostToDevice, p->stream));
  // Kernels are staged one at a time through a buffer sized for the largest, so the device never holds two
  // copies of a large table (cfg4: 616 MB).
  CK(cudaMalloc(&staging, (size_t)max_in * sizeof(float2)));
  for (int c = 0; c < d->n_cf; ++c) {
    int S = p->cf_support[c];
    int64_t n_in = (int64_t)S * p->os * S * p->os;
    const float2* src = (const float2*)d->cf_data + d->cf_offset[c];
    CK(cudaMemcpyAsync(staging, src, (size_t)n_in * sizeof(float2), cudaMemcpyDefault, p->stream));   // host or device table
    int64_t n_out = (int64_t)p->os * p->os * (p->slab_stride[c] / 2);
    int blocks = (int)((n_out + 255) / 256);
    if (blocks > 4096) blocks = 4096;
    lra_relayout_kernel<<<blocks, 256, 0, p->stream>>>(staging, reinterpret_cast<float2*>(p->slabs + p->slab_off[c]), S, p->os,
                                                       p->slab_stride[c] / 2, tile_x);
    p->launches++;
    CK(cudaGetLastError());
  }
  CK(cudaStreamSynchronize(p->stream));
  cudaFree(staging);
  staging = nullptr;
#undef CK
  *out = p;
  return LRA_OK;
}

void lra_fft_release(lra_plan* p);   // lra_image.cu

extern "C" int lra_plan_destroy(lra_plan* p) {
  if (!p) return LRA_EINVAL;
  cudaSetDevice(p->device);
  cudaStreamSynchronize(p->stream);
  lra_fft_release(p);
  void* ptrs[] = {p->slabs, p->d_cf_support, p->d_slab_off, p->ix, p->iy, p->fx, p->fy, p->key, p->skey[0], p->skey[1],
                  p->sval[0], p->sval[1], p->hist, p->tile_start, p->rec, p->urec, p->counters, p->d_su, p->d_sv, p->work, p->batch, p->pw, p->prep, p->awp_buf, p->po_scratch};
  for (void* q : ptrs)
    if (q) cudaFree(q);
  for (int s = 0; s < LRA_NAUX; ++s) {
    if (p->aux[s]) { cudaStreamSynchronize(p->aux[s]); cudaStreamDestroy(p->aux[s]); }
    if (p->ev_join[s]) cudaEventDestroy(p->ev_join[s]);
  }
  if (p->ev_fork) cudaEventDestroy(p->ev_fork);
  if (p->h_counts) cudaFreeHost(p->h_counts);
  if (p->h_scale) cudaFreeHost(p->h_scale);
  delete p;
  return LRA_OK;
}

extern "C" int lra_bin(lra_plan* p, int64_t nrow, int32_t nchan, const double* uvw_m, const double* freq_hz,
                       const int32_t* cf_index) {
  lra_nvtx_range nvtx_("lra_bin");
  if (!p || nrow < 0 || nchan < 1 || (nrow > 0 && !uvw_m) || !freq_hz) return LRA_EINVAL;
  if (nrow * (int64_t)nchan >= ((int64_t)1 << 31)) return LRA_EINVAL;
  LRA_CUDA(p, cudaSetDevice(p->device));
  return lra_bin_impl(p, nrow, nchan, uvw_m, freq_hz, cf_index);
}

extern "C" int lra_grid(lra_plan* p, const void* vis, const float* wt, const float* tau, void* grid, double* sumwt) {
  lra_nvtx_range nvtx_("lra_grid");
  if (!p) return LRA_EINVAL;
  if (!p->binned) return LRA_ESTATE;
  if (!grid || (p->npoints > 0 && (!vis || !wt))) return LRA_EINVAL;
  LRA_CUDA(p, cudaSetDevice(p->device));
  return lra_grid_impl(p, (const float2*)vis, wt, tau, (float2*)grid, sumwt);
}

extern "C" int lra_degrid(lra_plan* p, const void* grid, const float* tau, const void* vis_in, void* vis_out) {
  lra_nvtx_range nvtx_("lra_degrid");
  if (!p) return LRA_EINVAL;
  if (!p->binned) return LRA_ESTATE;
  if (!grid || (p->npoints > 0 && !vis_out)) return LRA_EINVAL;
  LRA_CUDA(p, cudaSetDevice(p->device));
  return lra_degrid_impl(p, (const float2*)grid, tau, (const float2*)vis_in, (float2*)vis_out);
}

extern "C" int64_t lra_launch_count(const lra_plan* p) { return p ? p->launches : 0; }

extern "C" int lra_tap_count(lra_plan* p, int64_t* n_valid, int64_t* sum_s2) {
  if (!p) return LRA_EINVAL;
  if (!p->binned) return LRA_ESTATE;
  unsigned long long h[2];
  LRA_CUDA(p, cudaMemcpyAsync(h, p->counters, sizeof h, cudaMemcpyDeviceToHost, p->stream));
  LRA_CUDA(p, cudaStreamSynchronize(p->stream));
  if (n_valid) *n_valid = (int64_t)h[0];
  if (sum_s2) *sum_s2 = (int64_t)h[1];
  return LRA_OK;
}

extern "C" int lra_set_variant(lra_plan* p, int32_t grid_variant, int32_t degrid_variant) {
  if (!p || grid_variant < 0 || grid_variant > 1 || degrid_variant < 0 || degrid_variant > 1) return LRA_EINVAL;
  p->grid_variant = grid_variant;
  p->degrid_variant = degrid_variant;
  return LRA_OK;
}

extern "C" const char* lra_strerror(int code) {
  switch (code) {
    case LRA_OK: return "ok";
    case LRA_EINVAL: return "invalid argument";
    case LRA_ENOMEM: return "out of memory";
    case LRA_ECUDA: return "CUDA error";
    case LRA_ESTATE: return "call out of order (lra_bin first)";
    default: return "unknown error";
  }
}

extern "C" const char* lra_last_cuda_error(const lra_plan* p) {
  if (!p || p->last_err == cudaSuccess) return "";
  return cudaGetErrorString(p->last_err);
}

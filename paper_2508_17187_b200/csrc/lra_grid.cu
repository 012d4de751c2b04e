// lra_grid.cu -- gridding G(c_ij) (Eq. 7) with the weights of Eq. 23:
//   grid[t][p][iy+j][ix+i] += CF[cf][fy][fx][j][i] * (wt * tau_t * V),   sumwt[t][p] += wt * tau_t   [R6]
// fp32 multiply-add, fp32 accumulation.  Kernels:
//   lra_sumwt_kernel        : sum of weights for variant 1 (variant 0 sums them in lra_prepare_kernel)
//   lra_grid_atomic_kernel  : variant 1, one CTA per visibility point, every tap a global float atomic (the
//                             "before" design kept for profiling and as a second implementation in the tests)
//   lra_grid_region_kernel  : variant 0 (default), lra_grid_region.cu
#include "lra_pipe.cuh"

#define LRA_MAXG 16  // nterms * ncorr <= 4 * 4

__device__ __forceinline__ void lra_red_add(float* addr, float v) {
  asm volatile("red.global.add.f32 [%0], %1;" ::"l"(addr), "f"(v) : "memory");
}

// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
lra_sumwt_kernel(const lra_rec* __restrict__ rec, const unsigned long long* __restrict__ counters,
                 const float* __restrict__ wt, const float* __restrict__ tau, int nchan, int ncorr, int nterms,
                 double* __restrict__ sumwt) {
  const long long n = (long long)counters[0];
  double acc[LRA_MAXG];
#pragma unroll
  for (int g = 0; g < LRA_MAXG; ++g) acc[g] = 0.0;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    uint32_t k = rec[i].z;
    int c = (int)(k % (uint32_t)nchan);
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      if (t >= nterms) break;
      float tw = tau ? tau[c * nterms + t] : 1.0f;
#pragma unroll
      for (int p = 0; p < 4; ++p) {
        if (p >= ncorr) break;
        acc[t * 4 + p] += (double)(wt[(size_t)k * ncorr + p] * tw);
      }
    }
  }
  __shared__ double sh[8][LRA_MAXG];
  const int l = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
  for (int g = 0; g < LRA_MAXG; ++g) {
    double v = acc[g];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if (l == 0) sh[w][g] = v;
  }
  __syncthreads();
  if (threadIdx.x < LRA_MAXG) {
    int t = threadIdx.x >> 2, pp = threadIdx.x & 3;
    if (t < nterms && pp < ncorr) {
      double v = 0.0;
      for (int ww = 0; ww < 8; ++ww) v += sh[ww][threadIdx.x];
      atomicAdd(&sumwt[t * ncorr + pp], v);
    }
  }
}

// ---------------------------------------------------------------------------------------------------
// variant 1: one CTA walks visibility points; its 256 threads split the S*S taps; every tap update is two
// red.global.add.f32.  No staging, no reuse: this is the design the tiled kernel is measured against.
__global__ void __launch_bounds__(256)
lra_grid_atomic_kernel(const lra_rec* __restrict__ rec, const unsigned long long* __restrict__ counters,
                       const float* __restrict__ slabs, const float2* __restrict__ vis, const float* __restrict__ wt,
                       const float* __restrict__ tau, int nchan, int ncorr, int nterms, int nx, int ny,
                       int tile_x, lra_fallback_mask fb, int only_fallback, float2* __restrict__ grid) {
  const long long n = (long long)counters[0];
  const size_t plane = (size_t)nx * ny;
  for (long long i = blockIdx.x; i < n; i += gridDim.x) {
    const lra_rec r = rec[i];
    const int ix = r.x & 0xffff, iy = r.x >> 16, S = r.w & 0xff, h = (S - 1) >> 1;
    if (only_fallback && !lra_is_fallback(fb, S)) continue;   // the region kernels do those
    const float2* slab = reinterpret_cast<const float2*>(slabs + ((size_t)r.y << 2));
    const uint32_t k = r.z;
    const int c = (int)(k % (uint32_t)nchan);
    float2 val[LRA_MAXG];
#pragma unroll
    for (int t = 0; t < 4; ++t)
#pragma unroll
      for (int p = 0; p < 4; ++p) {
        float2 v = make_float2(0.f, 0.f);
        if (t < nterms && p < ncorr) {
          float w = wt[(size_t)k * ncorr + p] * (tau ? tau[c * nterms + t] : 1.0f);
          float2 x = vis[(size_t)k * ncorr + p];
          v = make_float2(w * x.x, w * x.y);
        }
        val[t * 4 + p] = v;
      }
    for (int e = threadIdx.x; e < S * S; e += 256) {
      const int j = e / S, ii = e - j * S;
      const float2 cf = slab[lra_tap_index(S, tile_x, j, ii)];
      const size_t pix = (size_t)(iy - h + j) * nx + (ix - h + ii);
#pragma unroll
      for (int t = 0; t < 4; ++t)
#pragma unroll
        for (int p = 0; p < 4; ++p)
          if (t < nterms && p < ncorr) {
            const float2 v = val[t * 4 + p];
            float* g = (float*)(grid + (size_t)(t * ncorr + p) * plane + pix);
            lra_red_add(g, cf.x * v.x - cf.y * v.y);
            lra_red_add(g + 1, cf.x * v.y + cf.y * v.x);
          }
    }
  }
}

int lra_sumwt_launch(lra_plan* p, const float* wt, const float* tau, double* sumwt) {
  lra_sumwt_kernel<<<p->sm_count * 4, 256, 0, p->stream>>>(p->rec, p->counters, wt, tau, p->nchan, p->ncorr, p->nterms, sumwt);
  LRA_LAUNCH_CHECK(p);
  return LRA_OK;
}

// defined in lra_grid_region.cu
int lra_grid_region_launch(lra_plan* p, const float2* vis, const float* wt, const float* tau, float2* grid, double* sumwt);

int lra_grid_impl(lra_plan* p, const float2* vis, const float* wt, const float* tau, float2* grid, double* sumwt) {
  if (p->npoints == 0) return LRA_OK;
  const bool all_atomic = p->grid_variant == 1;
  if (sumwt && all_atomic) {   // variant 0 sums the weights in lra_prepare_kernel
    lra_sumwt_kernel<<<p->sm_count * 4, 256, 0, p->stream>>>(p->rec, p->counters, wt, tau, p->nchan, p->ncorr,
                                                            p->nterms, sumwt);
    LRA_LAUNCH_CHECK(p);
  }
  bool fallback = false;
  for (int c = 0; c < LRA_NCLASS; ++c)
    if (p->n_items[c] > 0 && lra_make_geom(2 * c + 1, p->tile_x, p->tile, p->ncorr * p->nterms).nw == 0) fallback = true;
  if (all_atomic || fallback) {  // regions that fit no group of the region kernel (or the "before" variant)
    lra_grid_atomic_kernel<<<p->sm_count * 16, 256, 0, p->stream>>>(p->rec, p->counters, p->slabs, vis, wt, tau,
                                                                     p->nchan, p->ncorr, p->nterms, p->nx, p->ny,
                                                                     p->tile_x, lra_make_fallback_mask(p->tile_x, p->tile, p->ncorr * p->nterms), all_atomic ? 0 : 1, grid);
    LRA_LAUNCH_CHECK(p);
    if (all_atomic) return LRA_OK;
  }
  return lra_grid_region_launch(p, vis, wt, tau, grid, sumwt);
}

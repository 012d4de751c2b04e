// lra_degrid.cu -- degridding D(c_ij) (Eq. 6), the exact adjoint of G with unit weights [R7]:
//   V[k][p] = sum_t tau[c][t] * sum_{j,i} conj(CF[cf][fy][fx][j][i]) * grid[t][p][iy+j][ix+i]
//   vis_out = vis_in ? vis_in - V : V   (fused residual of Eq. 23); invalid points: V = 0 [R4]
// fp32 multiply-add; per-lane partial sums over taps, then a warp-shuffle tree.
//
// Kernels:
//   lra_degrid_init_kernel   : vis_out = vis_in (or 0) for every sample, so that points dropped by lra_bin get V = 0
//   lra_degrid_region_kernel : variant 0 (default), lra_degrid_region.cu
//   lra_degrid_warp_kernel   : variant 1 and the fallback for regions too large for the region kernel: one warp per
//                            sorted visibility point.  Points are visited in tile order, so the
//                            warps resident on an SM read overlapping grid patches (L1 / L2 hits) and, with
//                            LRA_SORT_TILE_CF, the same CF slabs.
#include "lra_pipe.cuh"

__global__ void __launch_bounds__(256)
lra_degrid_init_kernel(const float2* __restrict__ vis_in, float2* __restrict__ vis_out, long long nsamples) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < nsamples; i += (long long)gridDim.x * blockDim.x)
    vis_out[i] = vis_in ? vis_in[i] : make_float2(0.f, 0.f);
}

template <int NC>
__global__ void __launch_bounds__(256)
lra_degrid_warp_kernel(const lra_rec* __restrict__ rec, const unsigned long long* __restrict__ counters,
                       const float* __restrict__ slabs, const float2* __restrict__ grid, const float* __restrict__ tau,
                       const float2* vis_in, float2* vis_out, int nchan, int nterms, int nx, int ny, int tile_x,
                       lra_fallback_mask fb, int only_fallback) {
  const long long n = (long long)counters[0];
  const size_t plane = (size_t)nx * ny;
  const int lane = threadIdx.x & 31;
  const long long warp0 = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5;
  const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
  for (long long i = warp0; i < n; i += nwarps) {
    const lra_rec r = rec[i];
    const int ix = r.x & 0xffff, iy = r.x >> 16, S = r.w & 0xff, h = (S - 1) >> 1;
    if (only_fallback && !lra_is_fallback(fb, S)) continue;   // the region kernels do those
    const float2* slab = reinterpret_cast<const float2*>(slabs + ((size_t)r.y << 2));
    const unsigned k = r.z;
    const int c = (int)(k % (unsigned)nchan);
    float tw[4];
#pragma unroll
    for (int t = 0; t < 4; ++t) tw[t] = (t < nterms) ? (tau ? tau[c * nterms + t] : 1.0f) : 0.f;
    float2 acc[NC];
#pragma unroll
    for (int p = 0; p < NC; ++p) acc[p] = make_float2(0.f, 0.f);
    const float2* g0 = grid + (size_t)(iy - h) * nx + (ix - h);
    for (int j = 0; j < S; ++j) {
      for (int ii = lane; ii < S; ii += 32) {
        const float2 cf = slab[lra_tap_index(S, tile_x, j, ii)];
        const float2* gp = g0 + (size_t)j * nx + ii;
#pragma unroll
        for (int p = 0; p < NC; ++p) {
          float2 gs = make_float2(0.f, 0.f);
          for (int t = 0; t < nterms; ++t) {
            const float2 g = gp[(size_t)(t * NC + p) * plane];
            gs.x = fmaf(tw[t], g.x, gs.x);
            gs.y = fmaf(tw[t], g.y, gs.y);
          }
          // conj(cf) * gs
          acc[p].x = fmaf(cf.x, gs.x, acc[p].x);
          acc[p].x = fmaf(cf.y, gs.y, acc[p].x);
          acc[p].y = fmaf(cf.x, gs.y, acc[p].y);
          acc[p].y = fmaf(-cf.y, gs.x, acc[p].y);
        }
      }
    }
#pragma unroll
    for (int p = 0; p < NC; ++p) {
      for (int o = 16; o > 0; o >>= 1) {
        acc[p].x += __shfl_xor_sync(0xffffffffu, acc[p].x, o);
        acc[p].y += __shfl_xor_sync(0xffffffffu, acc[p].y, o);
      }
    }
    if (lane == 0) {
#pragma unroll
      for (int p = 0; p < NC; ++p) {
        float2 o = acc[p];
        if (vis_in) {
          const float2 vi = vis_in[(size_t)k * NC + p];
          o = make_float2(vi.x - acc[p].x, vi.y - acc[p].y);
        }
        vis_out[(size_t)k * NC + p] = o;
      }
    }
  }
}

// defined in lra_degrid_region.cu
int lra_degrid_region_launch(lra_plan* p, const float2* grid, const float* tau, const float2* vis_in, float2* vis_out);

int lra_degrid_impl(lra_plan* p, const float2* grid, const float* tau, const float2* vis_in, float2* vis_out) {
  if (p->npoints == 0) return LRA_OK;
  const long long nsamples = p->npoints * (long long)p->ncorr;
  if (vis_in != vis_out) {
    lra_degrid_init_kernel<<<p->sm_count * 8, 256, 0, p->stream>>>(vis_in, vis_out, nsamples);
    LRA_LAUNCH_CHECK(p);
  }
  const bool all_warp = p->degrid_variant == 1;
  bool fallback = false;
  for (int c = 0; c < LRA_NCLASS; ++c)
    if (p->n_items[c] > 0 && lra_make_geom(2 * c + 1, p->tile_x, p->tile, p->ncorr * p->nterms).nw == 0) fallback = true;
  if (all_warp || fallback) {   // regions that fit no group of the region kernel (or the "before" variant)
    const int blocks = p->sm_count * 8;
#define LRA_DG(NC)                                                                                                  \
  lra_degrid_warp_kernel<NC><<<blocks, 256, 0, p->stream>>>(p->rec, p->counters, p->slabs, grid, tau, vis_in, vis_out, \
                                                            p->nchan, p->nterms, p->nx, p->ny, p->tile_x,             \
                                                            lra_make_fallback_mask(p->tile_x, p->tile, p->ncorr * p->nterms), all_warp ? 0 : 1)
    switch (p->ncorr) {
      case 1: LRA_DG(1); break;
      case 2: LRA_DG(2); break;
      case 3: LRA_DG(3); break;
      default: LRA_DG(4); break;
    }
#undef LRA_DG
    LRA_LAUNCH_CHECK(p);
    if (all_warp) return LRA_OK;
  }
  return lra_degrid_region_launch(p, grid, tau, vis_in, vis_out);
}

// lra_degrid_region.cu -- host driver of the default degridder (variant 0) and its finish kernel.  The tap-loop
// kernels are in lra_degrid_region.cuh (design notes there), instantiated in lra_degrid_region_ng*.cu.
//
// Operation: Eq. 6 of arxiv 2508.17187, SURVEY Sec. 8(a) row a5.
#include "lra_region.cuh"

template <int NG>
int lra_degrid_launch_ng(lra_plan* p, const lra_region_args& a, const lra_geom& q, int c, cudaStream_t st);

// V[k][p] = sum_t tau[c][t] * res[(t, p)][i];  vis_out[k][p] = vis_in ? vis_in[k][p] - V : V   for sorted position i
// whose support class the region kernels handle (the others were written by the fallback kernel).  Grid g = t*ncorr + p
// is grid g % LRA_NGMAX of pass g / LRA_NGMAX; res = [pass][sorted position][grids of the pass] complex.  One thread
// per point.
__global__ void __launch_bounds__(256)
lra_degrid_finish_kernel(const uint4* __restrict__ pw, const unsigned long long* __restrict__ counters,
                         const float2* __restrict__ res, const float* __restrict__ tau, bool residual,
                         float2* vis_out, int nchan, int ncorr, int nterms, long long npoints) {
  const long long n = (long long)counters[0];
  const int ng = ncorr * nterms;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const uint4 w4 = __ldcs(pw + i);
    if (w4.y & 0x80000000u) continue;   // a fallback class: written by the fallback kernel
    const unsigned k = w4.y;
    const int c = (int)(k % (unsigned)nchan);
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      if (p >= ncorr) break;
      float vx = 0.f, vy = 0.f;
      for (int t = 0; t < nterms; ++t) {
        const int g = t * ncorr + p, pass = g / LRA_NGMAX, gl = g - pass * LRA_NGMAX;
        const int ngp = ng - pass * LRA_NGMAX >= LRA_NGMAX ? LRA_NGMAX : ng - pass * LRA_NGMAX;
        const float2 v = __ldcs(res + (size_t)npoints * LRA_NGMAX * pass + (size_t)i * ngp + gl);
        const float tw = tau ? tau[c * nterms + t] : 1.0f;
        vx = fmaf(tw, v.x, vx);
        vy = fmaf(tw, v.y, vy);
      }
      float2 o = make_float2(vx, vy);
      if (residual) {   // lra_degrid_init_kernel has copied vis_in to vis_out: reading it back here touches the sector that
                        // is written next, where a read of vis_in[k] would fetch a second one
        const float2 vi = vis_out[(size_t)k * ncorr + p];
        o = make_float2(vi.x - vx, vi.y - vy);
      }
      vis_out[(size_t)k * ncorr + p] = o;
    }
  }
}

int lra_degrid_region_launch(lra_plan* p, const float2* grid, const float* tau, const float2* vis_in, float2* vis_out) {
  const int ng = p->ncorr * p->nterms;
  const int64_t n = p->npoints;
  int rc = LRA_OK;
  // results of all passes, [pass][sorted position][grid of the pass] complex: shares the gridder's scratch buffer
  const int64_t need = n * ng * 2 + 64;
  if (need > p->prep_capacity) {
    LRA_CUDA(p, cudaStreamSynchronize(p->stream));
    if (p->prep) { cudaFree(p->prep); p->prep = nullptr; p->prep_capacity = 0; }
    LRA_CUDA(p, cudaMalloc(&p->prep, (size_t)need * sizeof(float)));
    p->prep_capacity = need;
  }
  LRA_CUDA(p, cudaMemsetAsync(p->counters + LRA_TICKET0, 0, LRA_NTICKET * sizeof(unsigned long long), p->stream));
  lra_region_args a;
  a.slabs = p->slabs;
  a.prep = p->pw;   // 16 bytes per point: slab offset word and chunk range
  a.plane = (long long)p->nx * p->ny;
  a.nx = p->nx; a.ny = p->ny; a.tile_x = p->tile_x; a.tile_y = p->tile; a.ntx = p->ntx;
  LRA_CUDA(p, cudaEventRecord(p->ev_fork, p->stream));
  for (int s = 0; s < LRA_NAUX; ++s) LRA_CUDA(p, cudaStreamWaitEvent(p->aux[s], p->ev_fork, 0));
  int ticket = 0, turn = 0;
  const int npass = (ng + LRA_NGMAX - 1) / LRA_NGMAX;
  for (int pass = 0; pass < npass && rc == LRA_OK; ++pass) {
    const int ngp = ng - pass * LRA_NGMAX >= LRA_NGMAX ? LRA_NGMAX : ng - pass * LRA_NGMAX;
    a.res = reinterpret_cast<float2*>(p->prep) + (size_t)n * LRA_NGMAX * pass;
    a.grid = const_cast<float2*>(grid) + (size_t)(pass * LRA_NGMAX) * a.plane;
    for (int c = LRA_NCLASS - 1; c >= 0 && rc == LRA_OK; --c) {
      if (p->n_items[c] == 0) continue;
      const lra_geom q = lra_make_geom(2 * c + 1, p->tile_x, p->tile, ng);
      if (q.nw == 0) continue;
      if (ticket >= LRA_NTICKET) { rc = LRA_EINVAL; break; }
      a.ticket = p->counters + LRA_TICKET0 + ticket++;
      cudaStream_t st = p->aux[turn++ % LRA_NAUX];
      switch (ngp) {
        case 1: rc = lra_degrid_launch_ng<1>(p, a, q, c, st); break;
        case 2: rc = lra_degrid_launch_ng<2>(p, a, q, c, st); break;
        case 3: rc = lra_degrid_launch_ng<3>(p, a, q, c, st); break;
        default: rc = lra_degrid_launch_ng<4>(p, a, q, c, st); break;
      }
    }
  }
  for (int s = 0; s < LRA_NAUX; ++s) {
    LRA_CUDA(p, cudaEventRecord(p->ev_join[s], p->aux[s]));
    LRA_CUDA(p, cudaStreamWaitEvent(p->stream, p->ev_join[s], 0));
  }
  if (rc) return rc;
  // four blocks per SM: the scatter to caller order runs fastest at half occupancy (measured on cfg3, whole lra_degrid call:
  // 8 blocks of 256 per SM 28.10 ms, 4: 27.75, 2: 27.95, 1: 28.74; 1 x 1024: 27.78)
  lra_degrid_finish_kernel<<<p->sm_count * 4, 256, 0, p->stream>>>(p->pw, p->counters, reinterpret_cast<const float2*>(p->prep),
                                                                  tau, vis_in != nullptr, vis_out, p->nchan, p->ncorr, p->nterms,
                                                                  (long long)n);
  LRA_LAUNCH_CHECK(p);
  return LRA_OK;
}

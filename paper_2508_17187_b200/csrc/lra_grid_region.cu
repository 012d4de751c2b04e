// lra_grid_region.cu -- host driver of the default gridder (variant 0) and its prepare kernel.  The tap-loop kernels
// are in lra_grid_region.cuh (design notes there), instantiated in lra_grid_region_ng*.cu.
//
// Operation: Eq. 7 / Eq. 23 of arxiv 2508.17187, SURVEY Sec. 8(a) rows a3, a4.
#include "lra_region.cuh"

template <int NG>
int lra_grid_launch_ng(lra_plan* p, const lra_region_args& a, const lra_geom& q, int c, cudaStream_t st);

// wt * tau * V of every sorted point in the form the tap loop consumes (reading R6: (wt*tau)*V in fp32).  Grid
// g = t*ncorr + p belongs to pass g / LRA_NGMAX; the record of sorted position i in a pass of n grids is
//   n x float4 (vx, vy, -vy, vx), then uint4 (word, z, w, 0)                            [lra_point_bytes(n) bytes]
// with word and the step masks / chunk range (z, w) from lra_work.cu (lra_pipe.cuh).  Every pass but the last holds LRA_NGMAX grids, so
// pass j starts npoints * j * lra_point_bytes(LRA_NGMAX) bytes into `prep`.  One thread per point; the same pass over
// the weights also gives sumwt[t][p] += wt*tau (fp64 partials per thread, block tree, one atomic per block and grid).
// NCORR, NTERMS > 0: sizes known at compile time (the common shapes: the fp64 sumwt partials then take NCORR * NTERMS
// register pairs instead of 16: 48 instead of 140 registers); NCORR = 0: any shape up to 4 x 4.
// Launched with ONE block of 256 threads per SM: the pass is a random gather (16 + 8 useful bytes per point out of two
// 64-byte DRAM bursts) and runs fastest with 256-512 gathers in flight per SM -- measured on cfg3, whole lra_grid call:
// 1 x 256 threads per SM 20.22 ms, 2 x 256 20.53, 4 x 256 20.63, 8 x 256 (full occupancy) 20.85, 1 x 128 20.78,
// 1 x 512 20.42, 1 x 1024 20.57; two or four points per thread in flight: 20.24 / 20.41.
#define LRA_PREP_THREADS 256
template <int NCORR, int NTERMS>
__global__ void __launch_bounds__(LRA_PREP_THREADS)
lra_prepare_kernel(const unsigned long long* __restrict__ counters, const uint4* __restrict__ pw,
                   const float2* __restrict__ vis, const float* __restrict__ wt, const float* __restrict__ tau,
                   int nchan, int ncorr_rt, int nterms_rt, long long npoints, unsigned char* __restrict__ prep,
                   double* __restrict__ sumwt, int fast2) {
  const long long n = (long long)counters[0];
  const int ncorr = NCORR ? NCORR : ncorr_rt, nterms = NCORR ? NTERMS : nterms_rt;
  constexpr int MC = NCORR ? NCORR : 4, MT = NCORR ? NTERMS : 4;
  const int ng = ncorr * nterms;
  double acc[MT * MC];
#pragma unroll
  for (int g = 0; g < MT * MC; ++g) acc[g] = 0.0;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const uint4 w4 = pw[i];
    const unsigned k = w4.y & 0x7fffffffu;
    const int c = (int)(k % (unsigned)nchan);
    float2 v[MC];
    float w[MC];
    if (MC == 2 && fast2) {   // two correlations, 16-byte aligned vis: one load each
      const float4 vv = *reinterpret_cast<const float4*>(vis + (size_t)k * 2);
      const float2 ww = *reinterpret_cast<const float2*>(wt + (size_t)k * 2);
      v[0] = make_float2(vv.x, vv.y); v[1] = make_float2(vv.z, vv.w); w[0] = ww.x; w[1] = ww.y;
    } else {
#pragma unroll
      for (int p = 0; p < MC; ++p)
        if (p < ncorr) { v[p] = vis[(size_t)k * ncorr + p]; w[p] = wt[(size_t)k * ncorr + p]; }
    }
#pragma unroll
    for (int t = 0; t < MT; ++t) {
      if (t >= nterms) break;
      const float tw = tau ? tau[c * nterms + t] : 1.0f;
#pragma unroll
      for (int p = 0; p < MC; ++p) {
        if (p >= ncorr) break;
        const float wgt = w[p] * tw;
        acc[t * MC + p] += (double)wgt;
        const float vx = wgt * v[p].x, vy = wgt * v[p].y;
        const int g = t * ncorr + p, pass = g / LRA_NGMAX, gl = g - pass * LRA_NGMAX;
        const int ngp = ng - pass * LRA_NGMAX >= LRA_NGMAX ? LRA_NGMAX : ng - pass * LRA_NGMAX;
        unsigned char* rec = prep + (size_t)npoints * pass * lra_point_bytes(LRA_NGMAX) + (size_t)i * lra_point_bytes(ngp);
        reinterpret_cast<float4*>(rec)[gl] = make_float4(vx, vy, -vy, vx);
        if (gl == 0) reinterpret_cast<uint4*>(rec)[ngp] = make_uint4(w4.x, w4.z, w4.w, 0u);
      }
    }
  }
  if (!sumwt) return;
  __shared__ double sh[LRA_PREP_THREADS / 32][MT * MC];
  const int l = threadIdx.x & 31, wp = threadIdx.x >> 5;
#pragma unroll
  for (int g = 0; g < MT * MC; ++g) {
    double x = acc[g];
    for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
    if (l == 0) sh[wp][g] = x;
  }
  __syncthreads();
  if (threadIdx.x < MT * MC) {
    const int t = threadIdx.x / MC, pp = threadIdx.x % MC;
    if (t < nterms && pp < ncorr) {
      double x = 0.0;
      for (int ww = 0; ww < (int)(blockDim.x >> 5); ++ww) x += sh[ww][threadIdx.x];
      atomicAdd(&sumwt[t * ncorr + pp], x);
    }
  }
}

int lra_grid_region_launch(lra_plan* p, const float2* vis, const float* wt, const float* tau, float2* grid, double* sumwt) {
  const int ng = p->ncorr * p->nterms;
  const int64_t n = p->npoints;
  int rc = LRA_OK;
  // records of all passes (bytes; prep_capacity counts floats)
  const int npass = (ng + LRA_NGMAX - 1) / LRA_NGMAX;
  const int64_t need = (n * ((npass - 1) * lra_point_bytes(LRA_NGMAX) + lra_point_bytes(ng - (npass - 1) * LRA_NGMAX)) + 3) / 4 + 64;
  if (need > p->prep_capacity) {
    LRA_CUDA(p, cudaStreamSynchronize(p->stream));
    if (p->prep) { cudaFree(p->prep); p->prep = nullptr; p->prep_capacity = 0; }
    LRA_CUDA(p, cudaMalloc(&p->prep, (size_t)need * sizeof(float)));
    p->prep_capacity = need;
  }
  {
    const int fast2 = p->ncorr == 2 && ((uintptr_t)vis & 15) == 0 && ((uintptr_t)wt & 7) == 0;
    unsigned char* prep = reinterpret_cast<unsigned char*>(p->prep);
#define LRA_PREPARE(NC, NT) lra_prepare_kernel<NC, NT><<<p->sm_count, LRA_PREP_THREADS, 0, p->stream>>>(p->counters, p->pw, vis, wt, tau, \
                                p->nchan, p->ncorr, p->nterms, (long long)n, prep, sumwt, fast2)
    if (p->ncorr == 2 && p->nterms == 1) LRA_PREPARE(2, 1);
    else if (p->ncorr == 2 && p->nterms == 2) LRA_PREPARE(2, 2);
    else if (p->ncorr == 4 && p->nterms == 1) LRA_PREPARE(4, 1);
    else if (p->ncorr == 1 && p->nterms == 1) LRA_PREPARE(1, 1);
    else LRA_PREPARE(0, 0);
#undef LRA_PREPARE
  }
  LRA_LAUNCH_CHECK(p);
  LRA_CUDA(p, cudaMemsetAsync(p->counters + LRA_TICKET0, 0, LRA_NTICKET * sizeof(unsigned long long), p->stream));
  lra_region_args a;
  a.slabs = p->slabs;
  a.plane = (long long)p->nx * p->ny;
  a.nx = p->nx; a.ny = p->ny; a.tile_x = p->tile_x; a.tile_y = p->tile; a.ntx = p->ntx;
  a.res = nullptr; a.out_off = 0;
  // the per-class launches are independent: spread them over the plan's internal streams
  LRA_CUDA(p, cudaEventRecord(p->ev_fork, p->stream));
  for (int s = 0; s < LRA_NAUX; ++s) LRA_CUDA(p, cudaStreamWaitEvent(p->aux[s], p->ev_fork, 0));
  int ticket = 0, turn = 0;
  for (int pass = 0; pass < npass && rc == LRA_OK; ++pass) {
    const int ngp = ng - pass * LRA_NGMAX >= LRA_NGMAX ? LRA_NGMAX : ng - pass * LRA_NGMAX;
    a.prep = reinterpret_cast<const unsigned char*>(p->prep) + (size_t)n * pass * lra_point_bytes(LRA_NGMAX);
    a.grid = grid + (size_t)(pass * LRA_NGMAX) * a.plane;
    for (int c = LRA_NCLASS - 1; c >= 0 && rc == LRA_OK; --c) {   // large supports first: their items are the longest
      if (p->n_items[c] == 0) continue;
      const lra_geom q = lra_make_geom(2 * c + 1, p->tile_x, p->tile, ng);
      if (q.nw == 0) continue;                                    // done by the fallback kernel
      if (ticket >= LRA_NTICKET) { rc = LRA_EINVAL; break; }
      a.ticket = p->counters + LRA_TICKET0 + ticket++;
      cudaStream_t st = p->aux[turn++ % LRA_NAUX];
      switch (ngp) {
        case 1: rc = lra_grid_launch_ng<1>(p, a, q, c, st); break;
        case 2: rc = lra_grid_launch_ng<2>(p, a, q, c, st); break;
        case 3: rc = lra_grid_launch_ng<3>(p, a, q, c, st); break;
        default: rc = lra_grid_launch_ng<4>(p, a, q, c, st); break;
      }
    }
  }
  for (int s = 0; s < LRA_NAUX; ++s) {
    LRA_CUDA(p, cudaEventRecord(p->ev_join[s], p->aux[s]));
    LRA_CUDA(p, cudaStreamWaitEvent(p->stream, p->ev_join[s], 0));
  }
  return rc;
}

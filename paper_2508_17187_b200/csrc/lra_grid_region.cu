// lra_grid_region.cu -- the default gridder (variant 0): region-owning CTAs that accumulate in REGISTERS with packed
// fp32x2 FMAs and read the convolution function from a TMA-fed shared-memory ring.
//
// Operation: Eq. 7 / Eq. 23 of arxiv 2508.17187, tap loop of SURVEY Sec. 8(a) rows a3, a4.
//
// Design (B200-first; the paper's Kokkos kernel is prior art only):
//   * lra_bin left the visibility points sorted by uv tile (8 x 8 pixels by default), then by CF slab.  A work item
//     (lra_work.cu) is a run of at most LRA_CHUNK points of one tile and one support S; persistent CTAs take items
//     through an atomic ticket, so the dense centre of a VLA-like uv plane is spread over many CTAs.
//   * A CTA owns the item's region = tile + halo, RX x RY = (tile_x + S - 1) x (tile + S - 1) pixels, numbered
//     linearly e = y*RX + x.  Consumer warp w owns, at step s, the 64 consecutive pixels from 64*(NW*s + w); a lane
//     owns two of them, 32 apart.  The accumulators of those pixels stay in registers for the whole item and are
//     added to the HBM grid once per item with red.global.add.v2.f32 (row a4).
//   * The tile is small so that most of the region lies inside every footprint (S*S of (S+7)*(S+7) pixels): EVERY
//     lane updates its pixels for EVERY point, with no test and no divergence.  The CF slab is stored with the
//     region's pitch RX and zeros around the S x S taps (lra_internal.cuh), so the tap of pixel e for a point whose
//     footprint starts at linear pixel `off` is simply slab[e - off]: a warp reads 32 CONSECUTIVE floats per load (no
//     bank conflicts whatever RX is) and the lanes outside the footprint read zeros.
//   * The tap update is done two pixels at a time with FFMA2 (fma.rn.f32x2): the pair (cre(e), cre(e+32))
//     multiplies the point's duplicated value (vx, vx), so a complex multiply-add of two pixels on two grids is
//     8 FFMA2 fed by 4 shared-memory loads -- the FP32 pipe and the shared-memory port saturate together.
//   * lra_prepare_kernel first gathers vis / weight in SORTED order and writes wt*tau*V (in the duplicated form the
//     FFMA2s want, with the point's slab offset beside it) as a contiguous stream.
//   * The producer warp walks the batch stream of lra_work.cu and issues, per batch (= up to 12 slab runs of an
//     item), TMA bulk copies (cp.async.bulk + mbarrier complete_tx): the prepared values of its points and its CF
//     slabs, from L2 into a ring of shared-memory slots; item boundaries ride in the batch headers, so the consumers
//     never touch the work list and synchronise once per batch, not once per slab.
// Regions that fit no group (very large supports or tiles) take the global-atomic kernel of lra_grid.cu.
#include "lra_region.cuh"

// wt * tau * V of every sorted point in the form the FFMA2s consume (reading R6: (wt*tau)*V in fp32):
//   grid g = t*ncorr + p belongs to pass g/2; a pass holds [position][gl][8] = (vx, vx, vy, vy, -vy, -vy, pw, 0)
// with pw (lra_pipe.cuh) in the record of the pass's first grid.  One thread per point; the same pass over the
// weights also gives sumwt[t][p] += wt*tau (fp64 partials per thread, block tree, one atomic per block and grid).
__global__ void __launch_bounds__(256)
lra_prepare_kernel(const unsigned long long* __restrict__ counters, const uint4* __restrict__ pw,
                   const float2* __restrict__ vis, const float* __restrict__ wt, const float* __restrict__ tau,
                   int nchan, int ncorr, int nterms, long long npoints, float4* __restrict__ prep,
                   double* __restrict__ sumwt, int fast2) {
  const long long n = (long long)counters[0];
  const int ng = ncorr * nterms;
  double acc[16];
#pragma unroll
  for (int g = 0; g < 16; ++g) acc[g] = 0.0;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const uint4 w4 = pw[i];
    const unsigned k = w4.y;
    const float word = __uint_as_float(w4.x);
    const int c = (int)(k % (unsigned)nchan);
    float2 v[4];
    float w[4];
    if (fast2) {   // two correlations, 16-byte aligned vis: one load each
      const float4 vv = *reinterpret_cast<const float4*>(vis + (size_t)k * 2);
      const float2 ww = *reinterpret_cast<const float2*>(wt + (size_t)k * 2);
      v[0] = make_float2(vv.x, vv.y); v[1] = make_float2(vv.z, vv.w); w[0] = ww.x; w[1] = ww.y;
    } else {
#pragma unroll
      for (int p = 0; p < 4; ++p)
        if (p < ncorr) { v[p] = vis[(size_t)k * ncorr + p]; w[p] = wt[(size_t)k * ncorr + p]; }
    }
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      if (t >= nterms) break;
      const float tw = tau ? tau[c * nterms + t] : 1.0f;
#pragma unroll
      for (int p = 0; p < 4; ++p) {
        if (p >= ncorr) break;
        const float wgt = w[p] * tw;
        acc[t * 4 + p] += (double)wgt;
        const float vx = wgt * v[p].x, vy = wgt * v[p].y;
        const int g = t * ncorr + p, pass = g >> 1, gl = g & 1, ngp = ng - 2 * pass >= 2 ? 2 : 1;
        float4* dst = prep + ((size_t)npoints * 2 * pass + (size_t)i * ngp + gl) * 2;
        dst[0] = make_float4(vx, vx, vy, vy);
        dst[1] = make_float4(-vy, -vy, word, 0.f);
      }
    }
  }
  if (!sumwt) return;
  __shared__ double sh[8][16];
  const int l = threadIdx.x & 31, wp = threadIdx.x >> 5;
#pragma unroll
  for (int g = 0; g < 16; ++g) {
    double x = acc[g];
    for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
    if (l == 0) sh[wp][g] = x;
  }
  __syncthreads();
  if (threadIdx.x < 16) {
    const int t = threadIdx.x >> 2, pp = threadIdx.x & 3;
    if (t < nterms && pp < ncorr) {
      double x = 0.0;
      for (int ww = 0; ww < 8; ++ww) x += sh[ww][threadIdx.x];
      atomicAdd(&sumwt[t * ncorr + pp], x);
    }
  }
}

// One step of one point: the two pixels (e, e + 32) this lane owns at step s, on NG grids.
template <int NW, int NG>
__device__ __forceinline__ void lra_grid_step(const float* __restrict__ re, const float* __restrict__ im, int s,
                                              const lra_u64 (&vxx)[NG], const lra_u64 (&vyy)[NG],
                                              const lra_u64 (&nvy)[NG], lra_u64 (&acc)[NG][2]) {
  const lra_u64 cre = lra_pack2(re[s * 64 * NW], re[s * 64 * NW + 32]);
  const lra_u64 cim = lra_pack2(im[s * 64 * NW], im[s * 64 * NW + 32]);
#pragma unroll
  for (int g = 0; g < NG; ++g) {
    acc[g][0] = lra_fma2(cre, vxx[g], acc[g][0]);
    acc[g][0] = lra_fma2(cim, nvy[g], acc[g][0]);
    acc[g][1] = lra_fma2(cre, vyy[g], acc[g][1]);
    acc[g][1] = lra_fma2(cim, vxx[g], acc[g][1]);
  }
}

template <int NW, int KS, int NG>
__global__ void __launch_bounds__((NW + 1) * 32, lra_ctas_per_sm(NW, KS)) lra_grid_region_kernel(const lra_region_args a) {
  extern __shared__ __align__(128) unsigned char smem[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t sbase = lra_smem_u32(smem);
  const uint32_t full0 = sbase, empty0 = sbase + 128, slots0 = sbase + LRA_RING_HDR;
  lra_region_ring_init<NW>(a, smem, full0, empty0);
  if (warp == NW) {
    lra_region_producer<NW, 0>(a, a.prep, NG * 32, smem + LRA_RING_HDR, full0, empty0, slots0);
    return;
  }
  // -------------------------------------------------------------------- consumer warps
  lra_u64 acc[KS][NG][2];
#pragma unroll
  for (int s = 0; s < KS; ++s)
#pragma unroll
    for (int g = 0; g < NG; ++g) acc[s][g][0] = acc[s][g][1] = 0ull;
  uint32_t slot = 0, par = 0;
  const int lane_off = a.slab0 + 4 * (64 * warp + lane);
  const int im_off = a.stride_bytes;
  for (;;) {
    lra_mbar_wait(full0 + 8 * slot, par);
    const unsigned char* sp = smem + LRA_RING_HDR + (size_t)slot * a.slot_bytes;
    const uint4 h = *reinterpret_cast<const uint4*>(sp);
    const unsigned count = h.y & 0xff;
    const unsigned char* base = sp + lane_off;
    const ulonglong2* vp = reinterpret_cast<const ulonglong2*>(sp + LRA_SLOT_VAL);
    for (unsigned q = 0; q < count; ++q, vp += 2 * NG) {
      lra_u64 vxx[NG], vyy[NG], nvy[NG];
      const ulonglong2 v0 = vp[0], v1 = vp[1];
      vxx[0] = v0.x; vyy[0] = v0.y; nvy[0] = v1.x;
      if (NG == 2) {
        const ulonglong2 v2 = vp[2];
        vxx[NG - 1] = v2.x; vyy[NG - 1] = v2.y;
        nvy[NG - 1] = reinterpret_cast<const lra_u64*>(vp)[6];
      }
      const float* re = reinterpret_cast<const float*>(base + (uint32_t)v1.y);
      const float* im = reinterpret_cast<const float*>(base + (uint32_t)v1.y + im_off);
#pragma unroll
      for (int s = 0; s < KS; ++s) lra_grid_step<NW, NG>(re, im, s, vxx, vyy, nvy, acc[s]);
    }
    __syncwarp();
    if (lane == 0) lra_mbar_arrive(empty0 + 8 * slot);
    if (h.y & LRA_BATCH_LAST) {
      // ---- row a4: add the item's region to the grid, once ----
      const int hh = (a.S - 1) >> 1;
      const int ty = (int)(h.w / (unsigned)a.ntx), tx = (int)(h.w - (unsigned)ty * a.ntx);
      const int x0 = tx * a.tile_x - hh, y0 = ty * a.tile_y - hh;
      const unsigned magic = 0xffffffffu / (unsigned)a.rx + 1u;
#pragma unroll
      for (int s = 0; s < KS; ++s) {
        {
#pragma unroll
          for (int half = 0; half < 2; ++half) {
            const unsigned e = 64u * (NW * s + warp) + 32u * half + lane;
            const int y = (int)__umulhi(e, magic), x = (int)e - y * a.rx;
            const int gx = x0 + x, gy = y0 + y;
            const bool ok = y < a.ry && gx >= 0 && gx < a.nx && gy >= 0 && gy < a.ny;
#pragma unroll
            for (int g = 0; g < NG; ++g) {
              float r0, r1, i0, i1;
              lra_unpack2(acc[s][g][0], r0, r1);
              lra_unpack2(acc[s][g][1], i0, i1);
              const float vr = half ? r1 : r0, vi = half ? i1 : i0;
              if (ok && (vr != 0.f || vi != 0.f)) lra_red_add_v2(a.grid + (size_t)g * a.plane + (size_t)gy * a.nx + gx, vr, vi);
            }
          }
#pragma unroll
          for (int g = 0; g < NG; ++g) acc[s][g][0] = acc[s][g][1] = 0ull;
        }
      }
    }
    if (h.y & LRA_BATCH_END) break;
    if (++slot == (uint32_t)a.nslot) { slot = 0; par ^= 1; }
  }
}

// ---------------------------------------------------------------------------------------------------
template <int NW, int KS, int NG>
static int lra_launch_class(lra_plan* p, lra_region_args a, const lra_geom& q, int c, cudaStream_t st) {
  int smem = 0;
  if (!lra_region_ring(q, NG * 32, &a, &smem)) return LRA_EINVAL;
  auto kern = lra_grid_region_kernel<NW, KS, NG>;
  static int attr_smem[LRA_MAX_DEVICES];   // per instantiation and device: the opt-in is made once, not per launch
  if (p->device < 0 || p->device >= LRA_MAX_DEVICES || attr_smem[p->device] < smem) {
    LRA_CUDA(p, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    if (p->device >= 0 && p->device < LRA_MAX_DEVICES) attr_smem[p->device] = smem;
  }
  a.work = p->work + p->item_off[c];
  a.n_items = (unsigned)p->n_items[c];
  a.batch = reinterpret_cast<const uint4*>(p->batch) + (size_t)p->batch_off[c] * 4;
  int ctas = p->sm_count * lra_ctas_per_sm(NW, KS);
  if ((int64_t)ctas > p->n_items[c]) ctas = (int)p->n_items[c];
  kern<<<ctas, (NW + 1) * 32, smem, st>>>(a);
  LRA_LAUNCH_CHECK(p);
  return LRA_OK;
}

template <int NW, int NG>
static int lra_launch_class_ks(lra_plan* p, const lra_region_args& a, const lra_geom& q, int c, cudaStream_t st) {
  switch (q.ks) {
    case 1: return lra_launch_class<NW, 1, NG>(p, a, q, c, st);
    case 2: return lra_launch_class<NW, 2, NG>(p, a, q, c, st);
    case 3: return lra_launch_class<NW, 3, NG>(p, a, q, c, st);
    case 4: return lra_launch_class<NW, 4, NG>(p, a, q, c, st);
    case 5: return lra_launch_class<NW, 5, NG>(p, a, q, c, st);
    case 6: return lra_launch_class<NW, 6, NG>(p, a, q, c, st);
    default: break;
  }
  if constexpr (lra_ks_max(NW) > 6) {
    switch (q.ks) {
      case 7: return lra_launch_class<NW, 7, NG>(p, a, q, c, st);
      case 8: return lra_launch_class<NW, 8, NG>(p, a, q, c, st);
      case 9: return lra_launch_class<NW, 9, NG>(p, a, q, c, st);
      default: break;
    }
  }
  return LRA_EINVAL;
}

template <int NG>
static int lra_launch_class_nw(lra_plan* p, const lra_region_args& a, const lra_geom& q, int c, cudaStream_t st) {
  switch (q.nw) {
    case 2: return lra_launch_class_ks<2, NG>(p, a, q, c, st);
    case 4: return lra_launch_class_ks<4, NG>(p, a, q, c, st);
    case 8: return lra_launch_class_ks<8, NG>(p, a, q, c, st);
    case 16: return lra_launch_class_ks<16, NG>(p, a, q, c, st);
    default: return LRA_EINVAL;
  }
}

int lra_grid_region_launch(lra_plan* p, const float2* vis, const float* wt, const float* tau, float2* grid, double* sumwt) {
  const int ng = p->ncorr * p->nterms;
  const int64_t n = p->npoints;
  int rc = LRA_OK;
  // prepared values of all passes
  const int64_t need = n * ng * 8;
  if (need > p->prep_capacity) {
    LRA_CUDA(p, cudaStreamSynchronize(p->stream));
    if (p->prep) { cudaFree(p->prep); p->prep = nullptr; p->prep_capacity = 0; }
    LRA_CUDA(p, cudaMalloc(&p->prep, (size_t)need * sizeof(float)));
    p->prep_capacity = need;
  }
  lra_prepare_kernel<<<p->sm_count * 8, 256, 0, p->stream>>>(p->counters, p->pw, vis, wt, tau, p->nchan, p->ncorr, p->nterms,
                                                            (long long)n, (float4*)p->prep, sumwt,
                                                            p->ncorr == 2 && ((uintptr_t)vis & 15) == 0 && ((uintptr_t)wt & 7) == 0);
  LRA_LAUNCH_CHECK(p);
  LRA_CUDA(p, cudaMemsetAsync(p->counters + LRA_TICKET0, 0, LRA_NTICKET * sizeof(unsigned long long), p->stream));
  lra_region_args a;
  a.slabs = p->slabs;
  a.plane = (long long)p->nx * p->ny;
  a.nx = p->nx; a.ny = p->ny; a.tile_x = p->tile_x; a.tile_y = p->tile; a.ntx = p->ntx;
  // the per-class launches are independent: spread them over the plan's internal streams
  LRA_CUDA(p, cudaEventRecord(p->ev_fork, p->stream));
  for (int s = 0; s < LRA_NAUX; ++s) LRA_CUDA(p, cudaStreamWaitEvent(p->aux[s], p->ev_fork, 0));
  int ticket = 0, turn = 0;
  for (int pass = 0; 2 * pass < ng && rc == LRA_OK; ++pass) {
    const int ngp = ng - 2 * pass >= 2 ? 2 : 1;
    a.prep = p->prep + (size_t)n * 2 * pass * 8;
    a.grid = grid + (size_t)(2 * pass) * a.plane;
    for (int c = LRA_NCLASS - 1; c >= 0 && rc == LRA_OK; --c) {   // large supports first: their items are the longest
      if (p->n_items[c] == 0) continue;
      const lra_geom q = lra_make_geom(2 * c + 1, p->tile_x, p->tile);
      if (q.group == LRA_NGROUP - 1) continue;                    // done by the fallback kernel
      a.ticket = p->counters + LRA_TICKET0 + ticket++;
      cudaStream_t st = p->aux[turn++ % LRA_NAUX];
      rc = ngp == 2 ? lra_launch_class_nw<2>(p, a, q, c, st) : lra_launch_class_nw<1>(p, a, q, c, st);
    }
  }
  for (int s = 0; s < LRA_NAUX; ++s) {
    LRA_CUDA(p, cudaEventRecord(p->ev_join[s], p->aux[s]));
    LRA_CUDA(p, cudaStreamWaitEvent(p->stream, p->ev_join[s], 0));
  }
  return rc;
}

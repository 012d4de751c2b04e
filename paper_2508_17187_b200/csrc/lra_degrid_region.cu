// lra_degrid_region.cu -- the default degridder (variant 0): the adjoint of lra_grid_region.cu with the data flow
// turned round.
//
// Operation: Eq. 6 of arxiv 2508.17187, D(c_ij) read as the exact adjoint of G (reading R7), row a5
// of SURVEY Sec. 8(a):  V[k][p] = sum_t tau[c][t] * sum_{j,i} conj(CF[j][i]) * grid[t][p][iy+j][ix+i].
//
// Design: same items, batches, CF slab ring and producer warp as the gridder (lra_region.cuh, lra_work.cu).  A CTA
// loads the item's region of the MODEL grid into registers once (the grid tile is read once per item), pixel e of
// the region in the lane that owns it.  For every point every lane multiplies its pixels with the conjugated taps
// (same FFMA2 pairing, same zero-padded slab addressing as the gridder, no test), which leaves 32 partial sums per
// value in a warp.  Four points at a time, the 4 x NG complex partials are reduced across the lanes with a
// transposing shuffle butterfly (one shuffle per value instead of five), added across the consumer warps with
// shared-memory atomics into the slot, and written out by the producer warp, in sorted order, when the slot is
// recycled.  lra_degrid_finish_kernel then applies the Taylor weights, the fused residual of Eq. 23 and the sorted
// -> caller order scatter.
#include "lra_region.cuh"

// GP (1, 2 or 4) points of a batch against the region in registers: per-lane partial sums, then a transposing
// butterfly after which lane l holds the warp total of value l % V (V = GP x NG x (re, im)), then one shared-memory
// atomic per value into the slot.  `left` (< GP only for GP = 4: 3 points) is the number of points that exist.
template <int NW, int KS, int NG, int GP>
__device__ __forceinline__ void lra_degrid_points(const lra_u64 (&gre)[KS][NG], const lra_u64 (&gim)[KS][NG],
                                                  const unsigned char* base, int im_off, const uint4* pv, unsigned left,
                                                  float* out, int lane) {
  constexpr int V = 2 * NG * GP;
  float v[V];
#pragma unroll
  for (int u = 0; u < GP; ++u) {
    lra_u64 are[NG], aia[NG], aib[NG];
#pragma unroll
    for (int g = 0; g < NG; ++g) are[g] = aia[g] = aib[g] = 0ull;
    const uint32_t word = pv[GP == 4 && u == 3 && left < 4 ? 2 : u].x;   // a missing 4th point repeats the 3rd ...
    const float* re = reinterpret_cast<const float*>(base + word);
    const float* im = reinterpret_cast<const float*>(base + word + im_off);
#pragma unroll
    for (int s = 0; s < KS; ++s) {
      const lra_u64 cre = lra_pack2(re[s * 64 * NW], re[s * 64 * NW + 32]);
      const lra_u64 cim = lra_pack2(im[s * 64 * NW], im[s * 64 * NW + 32]);
#pragma unroll
      for (int g = 0; g < NG; ++g) {   // conj(c) * G = (cre*Gre + cim*Gim) + i (cre*Gim - cim*Gre)
        are[g] = lra_fma2(cre, gre[s][g], are[g]);
        are[g] = lra_fma2(cim, gim[s][g], are[g]);
        aia[g] = lra_fma2(cre, gim[s][g], aia[g]);
        aib[g] = lra_fma2(cim, gre[s][g], aib[g]);
      }
    }
#pragma unroll
    for (int g = 0; g < NG; ++g) {
      float r0, r1, a0, a1, b0, b1;
      lra_unpack2(are[g], r0, r1);
      lra_unpack2(aia[g], a0, a1);
      lra_unpack2(aib[g], b0, b1);
      v[(u * NG + g) * 2 + 0] = r0 + r1;
      v[(u * NG + g) * 2 + 1] = (a0 + a1) - (b0 + b1);
    }
  }
#pragma unroll
  for (int w = 1, n = V; n > 1; w <<= 1, n >>= 1) {
    const bool up = (lane & w) != 0;
#pragma unroll
    for (int i = 0; i < n / 2; ++i) {
      const float keep = up ? v[2 * i + 1] : v[2 * i], send = up ? v[2 * i] : v[2 * i + 1];
      v[i] = keep + __shfl_xor_sync(0xffffffffu, send, w);
    }
  }
#pragma unroll
  for (int w = V; w < 32; w <<= 1) v[0] += __shfl_xor_sync(0xffffffffu, v[0], w);
  if (lane < V && (unsigned)(lane / (2 * NG)) < left) atomicAdd(out + lane, v[0]);   // ... and is dropped here
}

template <int NW, int KS, int NG>
__global__ void __launch_bounds__((NW + 1) * 32, lra_ctas_per_sm(NW, KS)) lra_degrid_region_kernel(const lra_region_args a) {
  extern __shared__ __align__(128) unsigned char smem[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t sbase = lra_smem_u32(smem);
  const uint32_t full0 = sbase, empty0 = sbase + 128, slots0 = sbase + LRA_RING_HDR;
  lra_region_ring_init<NW>(a, smem, full0, empty0);
  if (warp == NW) {
    lra_region_producer<NW, NG>(a, a.prep, 16, smem + LRA_RING_HDR, full0, empty0, slots0);
    return;
  }
  // -------------------------------------------------------------------- consumer warps
  lra_u64 gre[KS][NG], gim[KS][NG];   // the region of the model grid: (re(e), re(e + 32)), (im(e), im(e + 32))
  bool fresh = true;
  uint32_t slot = 0, par = 0;
  const int lane_off = a.slab0 + 4 * (64 * warp + lane);
  const int im_off = a.stride_bytes;
  for (;;) {
    lra_mbar_wait(full0 + 8 * slot, par);
    unsigned char* sp = smem + LRA_RING_HDR + (size_t)slot * a.slot_bytes;
    const uint4 h = *reinterpret_cast<const uint4*>(sp);
    const unsigned count = h.y & 0xff;
    if (fresh && count) {
      // ---- the item's region of the model grid, once ----
      const int hh = (a.S - 1) >> 1;
      const int ty = (int)(h.w / (unsigned)a.ntx), tx = (int)(h.w - (unsigned)ty * a.ntx);
      const int x0 = tx * a.tile_x - hh, y0 = ty * a.tile_y - hh;
      const unsigned magic = 0xffffffffu / (unsigned)a.rx + 1u;
#pragma unroll
      for (int s = 0; s < KS; ++s) {
        float2 v[2][NG];
#pragma unroll
        for (int half = 0; half < 2; ++half) {
          const unsigned e = 64u * (NW * s + warp) + 32u * half + lane;
          const int y = (int)__umulhi(e, magic), x = (int)e - y * a.rx;
          const int gx = x0 + x, gy = y0 + y;
          const bool ok = y < a.ry && gx >= 0 && gx < a.nx && gy >= 0 && gy < a.ny;
#pragma unroll
          for (int g = 0; g < NG; ++g)
            v[half][g] = ok ? a.grid[(size_t)g * a.plane + (size_t)gy * a.nx + gx] : make_float2(0.f, 0.f);
        }
#pragma unroll
        for (int g = 0; g < NG; ++g) {
          gre[s][g] = lra_pack2_keep(v[0][g].x, v[1][g].x);
          gim[s][g] = lra_pack2_keep(v[0][g].y, v[1][g].y);
        }
      }
      fresh = false;
    }
    const unsigned char* base = sp + lane_off;
    const uint4* pv = reinterpret_cast<const uint4*>(sp + LRA_SLOT_VAL);
    float* out = reinterpret_cast<float*>(sp + a.out_off);
    for (unsigned q0 = 0; q0 < count; q0 += 4) {
      const unsigned left = count - q0;
      if (left >= 3) lra_degrid_points<NW, KS, NG, 4>(gre, gim, base, im_off, pv + q0, left, out + q0 * (2 * NG), lane);
      else if (left == 2) lra_degrid_points<NW, KS, NG, 2>(gre, gim, base, im_off, pv + q0, left, out + q0 * (2 * NG), lane);
      else lra_degrid_points<NW, KS, NG, 1>(gre, gim, base, im_off, pv + q0, left, out + q0 * (2 * NG), lane);
    }
    __syncwarp();
    if (lane == 0) lra_mbar_arrive(empty0 + 8 * slot);
    if (h.y & LRA_BATCH_LAST) fresh = true;
    if (h.y & LRA_BATCH_END) break;
    if (++slot == (uint32_t)a.nslot) { slot = 0; par ^= 1; }
  }
}

// V[k][p] = sum_t tau[c][t] * res[(t, p)][i];  vis_out[k][p] = vis_in ? vis_in[k][p] - V : V   for sorted position i
// whose support class the region kernels handle (the others were written by the fallback kernel).  One thread per point.
__global__ void __launch_bounds__(256)
lra_degrid_finish_kernel(const uint4* __restrict__ pw, const unsigned long long* __restrict__ counters,
                         const float2* __restrict__ res, const float* __restrict__ tau, const float2* vis_in,
                         float2* vis_out, int nchan, int ncorr, int nterms, long long npoints, int tile_x, int tile_y) {
  const long long n = (long long)counters[0];
  const int ng = ncorr * nterms;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const uint4 w4 = pw[i];
    if (lra_make_geom((int)w4.z, tile_x, tile_y).group == LRA_NGROUP - 1) continue;
    const unsigned k = w4.y;
    const int c = (int)(k % (unsigned)nchan);
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      if (p >= ncorr) break;
      float vx = 0.f, vy = 0.f;
      for (int t = 0; t < nterms; ++t) {
        const int g = t * ncorr + p, pass = g >> 1, gl = g & 1, ngp = ng - 2 * pass >= 2 ? 2 : 1;
        const float2 v = res[(size_t)npoints * 2 * pass + (size_t)i * ngp + gl];
        const float tw = tau ? tau[c * nterms + t] : 1.0f;
        vx = fmaf(tw, v.x, vx);
        vy = fmaf(tw, v.y, vy);
      }
      float2 o = make_float2(vx, vy);
      if (vis_in) {
        const float2 vi = vis_in[(size_t)k * ncorr + p];
        o = make_float2(vi.x - vx, vi.y - vy);
      }
      vis_out[(size_t)k * ncorr + p] = o;
    }
  }
}

// ---------------------------------------------------------------------------------------------------
template <int NW, int KS, int NG>
static int lra_degrid_launch_class(lra_plan* p, lra_region_args a, const lra_geom& q, int c, cudaStream_t st) {
  int smem = 0;
  if (!lra_region_ring(q, 16 + 8 * NG, &a, &smem)) return LRA_EINVAL;
  auto kern = lra_degrid_region_kernel<NW, KS, NG>;
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
static int lra_degrid_launch_ks(lra_plan* p, const lra_region_args& a, const lra_geom& q, int c, cudaStream_t st) {
  switch (q.ks) {
    case 1: return lra_degrid_launch_class<NW, 1, NG>(p, a, q, c, st);
    case 2: return lra_degrid_launch_class<NW, 2, NG>(p, a, q, c, st);
    case 3: return lra_degrid_launch_class<NW, 3, NG>(p, a, q, c, st);
    case 4: return lra_degrid_launch_class<NW, 4, NG>(p, a, q, c, st);
    case 5: return lra_degrid_launch_class<NW, 5, NG>(p, a, q, c, st);
    case 6: return lra_degrid_launch_class<NW, 6, NG>(p, a, q, c, st);
    default: break;
  }
  if constexpr (lra_ks_max(NW) > 6) {
    switch (q.ks) {
      case 7: return lra_degrid_launch_class<NW, 7, NG>(p, a, q, c, st);
      case 8: return lra_degrid_launch_class<NW, 8, NG>(p, a, q, c, st);
      case 9: return lra_degrid_launch_class<NW, 9, NG>(p, a, q, c, st);
      default: break;
    }
  }
  return LRA_EINVAL;
}

template <int NG>
static int lra_degrid_launch_nw(lra_plan* p, const lra_region_args& a, const lra_geom& q, int c, cudaStream_t st) {
  switch (q.nw) {
    case 2: return lra_degrid_launch_ks<2, NG>(p, a, q, c, st);
    case 4: return lra_degrid_launch_ks<4, NG>(p, a, q, c, st);
    case 8: return lra_degrid_launch_ks<8, NG>(p, a, q, c, st);
    case 16: return lra_degrid_launch_ks<16, NG>(p, a, q, c, st);
    default: return LRA_EINVAL;
  }
}

int lra_degrid_region_launch(lra_plan* p, const float2* grid, const float* tau, const float2* vis_in, float2* vis_out) {
  const int ng = p->ncorr * p->nterms;
  const int64_t n = p->npoints;
  int rc = LRA_OK;
  // results of all passes, [pass][sorted position][grid of the pass] complex: shares the gridder's scratch buffer
  const int64_t need = n * ng * 8;
  if (need > p->prep_capacity) {
    LRA_CUDA(p, cudaStreamSynchronize(p->stream));
    if (p->prep) { cudaFree(p->prep); p->prep = nullptr; p->prep_capacity = 0; }
    LRA_CUDA(p, cudaMalloc(&p->prep, (size_t)need * sizeof(float)));
    p->prep_capacity = need;
  }
  LRA_CUDA(p, cudaMemsetAsync(p->counters + LRA_TICKET0, 0, LRA_NTICKET * sizeof(unsigned long long), p->stream));
  lra_region_args a;
  a.slabs = p->slabs;
  a.prep = reinterpret_cast<const float*>(p->pw);   // 16 bytes per point: the slab offset word
  a.plane = (long long)p->nx * p->ny;
  a.nx = p->nx; a.ny = p->ny; a.tile_x = p->tile_x; a.tile_y = p->tile; a.ntx = p->ntx;
  LRA_CUDA(p, cudaEventRecord(p->ev_fork, p->stream));
  for (int s = 0; s < LRA_NAUX; ++s) LRA_CUDA(p, cudaStreamWaitEvent(p->aux[s], p->ev_fork, 0));
  int ticket = 0, turn = 0;
  for (int pass = 0; 2 * pass < ng && rc == LRA_OK; ++pass) {
    const int ngp = ng - 2 * pass >= 2 ? 2 : 1;
    a.res = reinterpret_cast<float2*>(p->prep) + (size_t)n * 2 * pass;
    a.grid = const_cast<float2*>(grid) + (size_t)(2 * pass) * a.plane;
    for (int c = LRA_NCLASS - 1; c >= 0 && rc == LRA_OK; --c) {
      if (p->n_items[c] == 0) continue;
      const lra_geom q = lra_make_geom(2 * c + 1, p->tile_x, p->tile);
      if (q.group == LRA_NGROUP - 1) continue;
      a.ticket = p->counters + LRA_TICKET0 + ticket++;
      cudaStream_t st = p->aux[turn++ % LRA_NAUX];
      rc = ngp == 2 ? lra_degrid_launch_nw<2>(p, a, q, c, st) : lra_degrid_launch_nw<1>(p, a, q, c, st);
    }
  }
  for (int s = 0; s < LRA_NAUX; ++s) {
    LRA_CUDA(p, cudaEventRecord(p->ev_join[s], p->aux[s]));
    LRA_CUDA(p, cudaStreamWaitEvent(p->stream, p->ev_join[s], 0));
  }
  if (rc) return rc;
  lra_degrid_finish_kernel<<<p->sm_count * 8, 256, 0, p->stream>>>(p->pw, p->counters, reinterpret_cast<const float2*>(p->prep),
                                                                  tau, vis_in, vis_out, p->nchan, p->ncorr, p->nterms,
                                                                  (long long)n, p->tile_x, p->tile);
  LRA_LAUNCH_CHECK(p);
  return LRA_OK;
}

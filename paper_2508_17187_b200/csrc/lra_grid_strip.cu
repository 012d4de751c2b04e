// lra_grid_strip.cu -- the default gridder (variant 0): strip-owning CTAs that accumulate in REGISTERS with packed
// fp32x2 FMAs and read the convolution function from a TMA-fed shared-memory ring.
//
// Operation: Eq. 7 / Eq. 23 of arxiv 2508.17187, tap loop of SURVEY Sec. 8(a) rows a3, a4.
//
// Design (B200-first; the paper's Kokkos kernel is prior art only):
//   * lra_bin left the visibility points sorted by uv tile -- by default a narrow STRIP, 8 pixels wide (u) and 64
//     tall (v) -- then by CF slab.  A work item (lra_work.cu) is a run of at most LRA_CHUNK points of one strip and
//     one support S; persistent CTAs take items through an atomic ticket, so the dense centre of a VLA-like uv
//     plane is spread over many CTAs.
//   * A CTA owns the item's region = strip + halo, RX x RY = (tile_x + S - 1) x (tile + S - 1) pixels, numbered
//     linearly e = y*RX + x.  Consumer warp w owns, at step s, the 64 consecutive pixels from 64*(NW*s + w); a lane
//     owns two of them, 32 apart.  The accumulators of those pixels stay in registers for the whole item and are
//     added to the HBM grid once per item with red.global.add.v2.f32 (row a4).
//   * The region is narrow so that most of its columns lie inside every footprint: the CF slab is stored with the
//     region's pitch RX and zeros around the S x S taps (lra_internal.cuh), and the tap of pixel e for a point
//     whose footprint starts at linear pixel `off` is simply slab[e - off].  A warp therefore reads 32 CONSECUTIVE
//     floats per load (no bank conflicts whatever RX is), lanes outside the footprint read zeros, and there is no
//     per-pixel test.  Which of its steps meet the footprint at all is a bit mask that lra_bin precomputed per
//     (point, warp); the warp skips the other steps with uniform branches.
//   * The tap update is done two pixels at a time with FFMA2 (fma.rn.f32x2): the pair (cre(e), cre(e+32))
//     multiplies the point's duplicated value (vx, vx), so a complex multiply-add of two pixels on two grids is
//     8 FFMA2 fed by 4 shared-memory loads -- the FP32 pipe and the shared-memory port saturate together.
//   * lra_prepare_kernel first gathers vis / weight in SORTED order and writes wt*tau*V (in the duplicated form the
//     FFMA2s want) as a contiguous stream, so the random accesses are spread over the whole GPU.
//   * The producer warp walks the stage stream of lra_work.cu and issues, per stage (= the points of an item that
//     share one slab), four TMA bulk copies (cp.async.bulk + mbarrier complete_tx): per-point words, prepared
//     values and the two planes of the CF slab, from L2 into a ring of shared-memory slots; item boundaries ride
//     in the stage headers, so the consumers never touch the work list.
// Regions that fit no group (very large supports or tiles) take the global-atomic kernel of lra_grid.cu.
#include <stdlib.h>

#include "lra_pipe.cuh"

struct lra_strip_args {
  const uint4* work;            // items of this launch's group
  unsigned n_items;
  unsigned long long* ticket;
  const uint4* stage_hdr;       // stage headers of this group
  const uint32_t* pw;           // [sorted position][LRA_PW_STRIDE]
  const float* slabs;
  const float* prep;            // this pass: [sorted position][NG][8] duplicated wt * tau * V
  float2* grid;                 // first grid of this pass
  long long plane;              // pixels per grid
  int nx, ny, tile_x, tile_y, ntx;
  int nslot, slot_bytes, plane_bytes;   // ring geometry: slots, bytes per slot, bytes per slab plane incl. margin
  int debug;                    // measurement aid (LRA_DEBUG env): 1 = consumers skip the taps
};

// slot layout (bytes): header | per-point words | prepared values | re plane | im plane; every plane starts with a
// margin of 64 zero floats that is written once at kernel start and never again.
#define LRA_SLOT_PW 128
#define LRA_SLOT_VAL (LRA_SLOT_PW + LRA_RUNMAX * LRA_PW_STRIDE * 4)
#define LRA_MARGIN_BYTES 256
__host__ __device__ inline int lra_slot_plane0(int ng) { return LRA_SLOT_VAL + LRA_RUNMAX * ng * 32; }
#define LRA_RING_HDR 256   // full / empty barriers of up to 16 slots

// wt * tau * V of every sorted point in the form the FFMA2s consume (reading R6: (wt*tau)*V in fp32):
//   grid g = t*ncorr + p belongs to pass g/2; a pass holds [position][gl][8] = (vx, vx, vy, vy, -vy, -vy, 0, 0)
__global__ void __launch_bounds__(256)
lra_prepare_kernel(const lra_rec* __restrict__ rec, const unsigned long long* __restrict__ counters,
                   const float2* __restrict__ vis, const float* __restrict__ wt, const float* __restrict__ tau,
                   int nchan, int ncorr, int nterms, long long npoints, float4* __restrict__ prep) {
  const long long n = (long long)counters[0] * ncorr;
  const int ng = ncorr * nterms;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
    const long long i = e / ncorr;
    const int p = (int)(e - i * ncorr);
    const unsigned k = rec[i].z;
    const float2 v = vis[(size_t)k * ncorr + p];
    const float w = wt[(size_t)k * ncorr + p];
    const int c = (int)(k % (unsigned)nchan);
    for (int t = 0; t < nterms; ++t) {
      const float wgt = w * (tau ? tau[c * nterms + t] : 1.0f);
      const float vx = wgt * v.x, vy = wgt * v.y;
      const int g = t * ncorr + p, pass = g >> 1, gl = g & 1, ngp = ng - 2 * pass >= 2 ? 2 : 1;
      float4* dst = prep + ((size_t)npoints * 2 * pass + (size_t)i * ngp + gl) * 2;
      dst[0] = make_float4(vx, vx, vy, vy);
      dst[1] = make_float4(-vy, -vy, 0.f, 0.f);
    }
  }
}

template <int NW, int KS, int NG, int MINB>
__global__ void __launch_bounds__((NW + 1) * 32, MINB) lra_grid_strip_kernel(const lra_strip_args a) {
  extern __shared__ __align__(128) unsigned char smem[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t sbase = lra_smem_u32(smem);
  const uint32_t full0 = sbase, empty0 = sbase + 128, slots0 = sbase + LRA_RING_HDR;
  const int plane0 = lra_slot_plane0(NG);
  if (threadIdx.x == 0) {
    for (int s = 0; s < a.nslot; ++s) { lra_mbar_init(full0 + 8 * s, 1); lra_mbar_init(empty0 + 8 * s, NW); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  for (int i = threadIdx.x; i < a.nslot * 128; i += (NW + 1) * 32) {
    const int s = i >> 7, pl = (i >> 6) & 1, j = i & 63;
    *reinterpret_cast<float*>(smem + LRA_RING_HDR + (size_t)s * a.slot_bytes + plane0 + pl * a.plane_bytes + 4 * j) = 0.f;
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  __syncthreads();

  if (warp == NW) {
    // ------------------------------------------------------------------ producer warp
    uint32_t slot = 0, par = 0;
    auto issue = [&](const uint4 h) {       // lane 0 only
      const uint32_t sa = slots0 + slot * a.slot_bytes, fb = full0 + 8 * slot;
      lra_mbar_wait(empty0 + 8 * slot, par ^ 1);
      asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(sa), "r"(h.x), "r"(h.y), "r"(h.z), "r"(h.w) : "memory");
      if (h.y & LRA_STAGE_END) { lra_mbar_arrive(fb); return; }
      const uint32_t count = h.y & 0xff, S = (h.y >> 8) & 0xff;
      const uint32_t pf = (uint32_t)lra_plane_floats((int)S, a.tile_x);
      lra_mbar_arrive_expect_tx(fb, count * (LRA_PW_STRIDE * 4 + NG * 32) + 8 * pf);
      lra_tma_load_1d(sa + LRA_SLOT_PW, a.pw + (size_t)h.x * LRA_PW_STRIDE, count * LRA_PW_STRIDE * 4, fb);
      lra_tma_load_1d(sa + LRA_SLOT_VAL, a.prep + (size_t)h.x * NG * 8, count * NG * 32, fb);
      const float* slab = a.slabs + ((size_t)h.z << 2);
      lra_tma_load_1d(sa + plane0 + LRA_MARGIN_BYTES, slab, 4 * pf, fb);
      lra_tma_load_1d(sa + plane0 + a.plane_bytes + LRA_MARGIN_BYTES, slab + pf, 4 * pf, fb);
    };
    for (;;) {
      unsigned long long t = 0;
      if (lane == 0) t = atomicAdd(a.ticket, 1ull);
      t = __shfl_sync(0xffffffffu, t, 0);
      if (t >= a.n_items) break;
      const uint4 item = a.work[t];
      for (unsigned b = 0; b < item.z; b += 32) {
        uint4 hd = make_uint4(0, 0, 0, 0);
        if (b + lane < item.z) hd = a.stage_hdr[(size_t)item.y + b + lane];
        const unsigned m = item.z - b < 32u ? item.z - b : 32u;
        for (unsigned j = 0; j < m; ++j) {
          uint4 h;
          h.x = __shfl_sync(0xffffffffu, hd.x, j); h.y = __shfl_sync(0xffffffffu, hd.y, j);
          h.z = __shfl_sync(0xffffffffu, hd.z, j); h.w = __shfl_sync(0xffffffffu, hd.w, j);
          if (lane == 0) issue(h);
          if (++slot == (uint32_t)a.nslot) { slot = 0; par ^= 1; }
        }
      }
    }
    if (lane == 0) issue(make_uint4(0, LRA_STAGE_END, 0, 0));
    return;
  }

  // -------------------------------------------------------------------- consumer warps
  lra_u64 acc[KS][NG][2];
#pragma unroll
  for (int s = 0; s < KS; ++s)
#pragma unroll
    for (int g = 0; g < NG; ++g) acc[s][g][0] = acc[s][g][1] = 0ull;
  uint32_t slot = 0, par = 0;
  const int lane_off = plane0 + LRA_MARGIN_BYTES + 4 * (64 * warp + lane);
  for (;;) {
    lra_mbar_wait(full0 + 8 * slot, par);
    const unsigned char* sp = smem + LRA_RING_HDR + (size_t)slot * a.slot_bytes;
    const uint4 h = *reinterpret_cast<const uint4*>(sp);
    const unsigned count = a.debug == 1 ? 0u : (h.y & 0xff);
    const unsigned char* re0 = sp + lane_off;
    const unsigned* words = reinterpret_cast<const unsigned*>(sp + LRA_SLOT_PW) + warp;
    for (unsigned q = 0; q < count; ++q) {
      const unsigned word = words[q * LRA_PW_STRIDE];
      if ((word >> 16) == 0) continue;
      const float* re = reinterpret_cast<const float*>(re0 - (word & 0xffffu));
      const float* im = reinterpret_cast<const float*>(re0 - (word & 0xffffu) + a.plane_bytes);
      const ulonglong2* vp = reinterpret_cast<const ulonglong2*>(sp + LRA_SLOT_VAL + q * (NG * 32));
      lra_u64 vxx[NG], vyy[NG], nvy[NG];
#pragma unroll
      for (int g = 0; g < NG; ++g) {
        const ulonglong2 v0 = vp[2 * g];
        vxx[g] = v0.x; vyy[g] = v0.y;
        nvy[g] = reinterpret_cast<const lra_u64*>(vp)[4 * g + 2];
      }
#pragma unroll
      for (int s = 0; s < KS; ++s) {
        if (word & (0x10000u << s)) {
          const lra_u64 cre = lra_pack2(re[s * 64 * NW], re[s * 64 * NW + 32]);
          const lra_u64 cim = lra_pack2(im[s * 64 * NW], im[s * 64 * NW + 32]);
#pragma unroll
          for (int g = 0; g < NG; ++g) {
            acc[s][g][0] = lra_fma2(cre, vxx[g], acc[s][g][0]);
            acc[s][g][0] = lra_fma2(cim, nvy[g], acc[s][g][0]);
            acc[s][g][1] = lra_fma2(cre, vyy[g], acc[s][g][1]);
            acc[s][g][1] = lra_fma2(cim, vxx[g], acc[s][g][1]);
          }
        }
      }
    }
    __syncwarp();
    if (lane == 0) lra_mbar_arrive(empty0 + 8 * slot);
    if (h.y & LRA_STAGE_LAST) {
      // ---- row a4: add the item's region to the grid, once ----
      const int S = (h.y >> 8) & 0xff, hh = (S - 1) >> 1;
      const int rx = S + a.tile_x - 1, ry = S + a.tile_y - 1;
      const int ty = (int)(h.w / (unsigned)a.ntx), tx = (int)(h.w - (unsigned)ty * a.ntx);
      const int x0 = tx * a.tile_x - hh, y0 = ty * a.tile_y - hh;
      const unsigned magic = 0xffffffffu / (unsigned)rx + 1u;
#pragma unroll
      for (int s = 0; s < KS; ++s) {
#pragma unroll
        for (int half = 0; half < 2; ++half) {
          const unsigned e = 64u * (NW * s + warp) + 32u * half + lane;
          const int y = (int)__umulhi(e, magic), x = (int)e - y * rx;
          const int gx = x0 + x, gy = y0 + y;
          const bool ok = y < ry && gx >= 0 && gx < a.nx && gy >= 0 && gy < a.ny;
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
    if (h.y & LRA_STAGE_END) break;
    if (++slot == (uint32_t)a.nslot) { slot = 0; par ^= 1; }
  }
}

// ---------------------------------------------------------------------------------------------------
template <int NW, int KS, int NG, int MINB>
static int lra_launch_group(lra_plan* p, lra_strip_args a, int g, int pf_max, int ticket) {
  const int plane_bytes = (LRA_MARGIN_BYTES + 4 * pf_max + 127) & ~127;
  const int slot_bytes = lra_slot_plane0(NG) + 2 * plane_bytes;
  const int budget = (MINB >= 4 ? 54 : MINB == 3 ? 72 : MINB == 2 ? 110 : 222) * 1024;
  int nslot = (budget - LRA_RING_HDR) / slot_bytes;
  if (nslot > 16) nslot = 16;
  if (nslot < 2) return LRA_EINVAL;
  const char* env = getenv("LRA_NSLOT");
  if (env && atoi(env) >= 2 && atoi(env) < nslot) nslot = atoi(env);
  const int smem = LRA_RING_HDR + nslot * slot_bytes;
  auto kern = lra_grid_strip_kernel<NW, KS, NG, MINB>;
  LRA_CUDA(p, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  a.work = p->work + p->item_off[g];
  a.n_items = (unsigned)p->n_items[g];
  a.stage_hdr = p->stage_hdr + p->stage_off[g];
  a.ticket = p->counters + LRA_TICKET0 + ticket;
  a.nslot = nslot; a.slot_bytes = slot_bytes; a.plane_bytes = plane_bytes;
  int ctas = p->sm_count * MINB;
  if ((int64_t)ctas > p->n_items[g]) ctas = (int)p->n_items[g];
  kern<<<ctas, (NW + 1) * 32, smem, p->stream>>>(a);
  LRA_LAUNCH_CHECK(p);
  return LRA_OK;
}

int lra_grid_strip_launch(lra_plan* p, const float2* vis, const float* wt, const float* tau, float2* grid) {
  const int ng = p->ncorr * p->nterms;
  const int64_t n = p->npoints;
  int rc;
  // prepared values of all passes
  const int64_t need = n * ng * 8;
  if (need > p->prep_capacity) {
    LRA_CUDA(p, cudaStreamSynchronize(p->stream));
    if (p->prep) { cudaFree(p->prep); p->prep = nullptr; p->prep_capacity = 0; }
    LRA_CUDA(p, cudaMalloc(&p->prep, (size_t)need * sizeof(float)));
    p->prep_capacity = need;
  }
  lra_prepare_kernel<<<p->sm_count * 8, 256, 0, p->stream>>>(p->rec, p->counters, vis, wt, tau, p->nchan, p->ncorr,
                                                            p->nterms, (long long)n, (float4*)p->prep);
  LRA_LAUNCH_CHECK(p);
  LRA_CUDA(p, cudaMemsetAsync(p->counters + LRA_TICKET0, 0, LRA_NTICKET * sizeof(unsigned long long), p->stream));
  int pf_max[LRA_NGROUP] = {0, 0, 0, 0, 0};
  for (int c = 0; c < p->n_cf; ++c) {
    const int S = p->cf_support[c], g = lra_group_of(S, p->tile_x, p->tile);
    const int pf = lra_plane_floats(S, p->tile_x);
    if (pf > pf_max[g]) pf_max[g] = pf;
  }
  lra_strip_args a;
  a.pw = p->pw; a.slabs = p->slabs;
  a.plane = (long long)p->nx * p->ny;
  a.nx = p->nx; a.ny = p->ny; a.tile_x = p->tile_x; a.tile_y = p->tile; a.ntx = p->ntx;
  const char* dbg = getenv("LRA_DEBUG");
  a.debug = dbg ? atoi(dbg) : 0;
  int ticket = 0;
  for (int pass = 0; 2 * pass < ng; ++pass) {
    const int ngp = ng - 2 * pass >= 2 ? 2 : 1;
    a.prep = p->prep + (size_t)n * 2 * pass * 8;
    a.grid = grid + (size_t)(2 * pass) * a.plane;
    for (int g = LRA_NGROUP - 2; g >= 0; --g) {   // large supports first: their items are the longest
      if (p->n_items[g] == 0) continue;
      const int t = ticket++;
      if (ngp == 2) {
        if (g == 0) rc = lra_launch_group<4, 8, 2, 3>(p, a, g, pf_max[g], t);
        else if (g == 1) rc = lra_launch_group<8, 8, 2, 2>(p, a, g, pf_max[g], t);
        else if (g == 2) rc = lra_launch_group<16, 7, 2, 1>(p, a, g, pf_max[g], t);
        else rc = lra_launch_group<16, 9, 2, 1>(p, a, g, pf_max[g], t);
      } else {
        if (g == 0) rc = lra_launch_group<4, 8, 1, 3>(p, a, g, pf_max[g], t);
        else if (g == 1) rc = lra_launch_group<8, 8, 1, 2>(p, a, g, pf_max[g], t);
        else if (g == 2) rc = lra_launch_group<16, 7, 1, 1>(p, a, g, pf_max[g], t);
        else rc = lra_launch_group<16, 9, 1, 1>(p, a, g, pf_max[g], t);
      }
      if (rc) return rc;
    }
  }
  return LRA_OK;
}

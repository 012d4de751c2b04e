// lra_grid_tiled.cu -- the default gridder (variant 0): tile-owning CTAs that accumulate in REGISTERS.
//
// Operation: Eq. 7 / Eq. 23 of arxiv 2508.17187, tap loop of SURVEY Sec. 8(a) rows a3, a4.
//
// Design (B200-first; the paper's Kokkos kernel is prior art only):
//   * lra_bin left the visibility points sorted by uv tile (T = 32).  A work item is one tile plus a chunk
//     of at most LRA_CHUNK of its points; items are handed out to persistent CTAs through an atomic ticket,
//     so the dense centre of a VLA-like uv plane (100x the mean density) is spread over many CTAs.
//   * A CTA owns the item's region = tile + halo, R x R pixels (R = 64 for supports <= 33, R = 96 for
//     supports <= 65).  Every consumer thread owns a fixed set of region pixels (lane <-> x, warp <-> y) and
//     keeps their accumulators in registers for the whole item: the tap update is 4 FFMA per correlation
//     with no atomic, no shared-memory read-modify-write, and the region is flushed to HBM exactly once per
//     item with red.global.add.v2.f32 (row a4).
//   * One producer warp runs ahead of the consumer warps: it reads the sorted records, gathers vis / weight,
//     forms wt*tau*V, writes the per-point parameters into a shared-memory ring and pulls the point's CF slab
//     (S*S complex64, contiguous thanks to the phase-major re-layout) from L2 into shared memory with one
//     TMA bulk copy (cp.async.bulk + mbarrier complete_tx).  Consecutive points with the same slab share one
//     copy.  Consumers wait on the stage's "full" mbarrier, do their taps from shared memory (LDS.64, lanes on
//     consecutive taps: conflict free) and release the stage through its "empty" mbarrier.
//   * Rows are warp-uniform (a warp skips rows outside the footprint with a uniform branch); columns are
//     predicated per lane.
// Supports > 65 (none in the five configurations) take the global-atomic path of lra_grid.cu.
#include "lra_internal.cuh"

#define LRA_CHUNK 512      // points per work item
#define LRA_RUNMAX 32      // points per pipeline stage (one producer-warp batch)

// ---------------------------------------------------------------------------------------------------
// PTX wrappers: mbarrier + 1-D TMA bulk copy
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t lra_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void lra_mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(lra_smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void lra_mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(lra_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void lra_mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(lra_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void lra_mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(lra_smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void lra_tma_load_1d(void* smem_dst, const void* gmem_src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   lra_smem_u32(smem_dst)), "l"(gmem_src), "r"(bytes), "r"(lra_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void lra_red_add_v2(float2* addr, float2 v) {
  asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(addr), "f"(v.x), "f"(v.y) : "memory");
}

// ---------------------------------------------------------------------------------------------------
// work list: item = {tile, first sorted position, count, class}; class 0: S <= 33, 1: S <= 65, 2: larger
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
lra_work_count_kernel(const uint32_t* __restrict__ tile_start, int ntiles, uint32_t* __restrict__ item_off) {
  int q = blockIdx.x * blockDim.x + threadIdx.x;
  if (q > ntiles) return;
  uint32_t cnt = q < ntiles ? tile_start[q + 1] - tile_start[q] : 0u;
  item_off[q] = (cnt + LRA_CHUNK - 1) / LRA_CHUNK;
}

__global__ void __launch_bounds__(256)
lra_work_fill_kernel(const uint32_t* __restrict__ tile_start, int ntiles, const uint32_t* __restrict__ item_off,
                     uint4* __restrict__ work, unsigned long long* __restrict__ counters) {
  int q = blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= ntiles) return;
  uint32_t lo = tile_start[q], hi = tile_start[q + 1], o = item_off[q];
  for (uint32_t s = lo; s < hi; s += LRA_CHUNK, ++o) work[o] = make_uint4((uint32_t)q, s, min(hi - s, (uint32_t)LRA_CHUNK), 0u);
  if (q == ntiles - 1) counters[2] = item_off[ntiles];
}

__global__ void __launch_bounds__(256)
lra_work_class_kernel(const lra_rec* __restrict__ rec, uint4* __restrict__ work, unsigned long long* __restrict__ counters) {
  const unsigned n_items = (unsigned)counters[2];
  const int lane = threadIdx.x & 31;
  for (unsigned it = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; it < n_items; it += (gridDim.x * blockDim.x) >> 5) {
    uint4 w = work[it];
    unsigned smax = 0;
    for (unsigned i = lane; i < w.z; i += 32) smax = max(smax, rec[w.y + i].w & 0xffu);
    for (int o = 16; o > 0; o >>= 1) smax = max(smax, __shfl_xor_sync(0xffffffffu, smax, o));
    if (lane == 0) {
      unsigned cls = smax <= 33 ? 0u : (smax <= 65 ? 1u : 2u);
      work[it].w = cls;
      atomicAdd(&counters[8 + cls], 1ull);
    }
  }
}

// ---------------------------------------------------------------------------------------------------
// shared-memory stage of the producer/consumer ring
// ---------------------------------------------------------------------------------------------------
template <int NG>
struct lra_point_params {
  int ox, oy, S, pad;     // footprint origin in region coordinates, support
  float2 val[NG];         // wt * tau * V for the NG grids of this pass
};

struct lra_stage_hdr {
  int count;              // points in this run; 0 = end of item
  int x0, y0;             // region origin in grid pixels (valid in the end-of-item marker)
  int last;               // end-of-item marker only: 1 = no more items
};

struct lra_tiled_args {
  const lra_rec* rec;
  const uint4* work;
  unsigned long long* counters;
  int ticket;            // index into counters of this launch's work ticket
  const float2* slabs;
  const float2* vis;
  const float* wt;
  const float* tau;
  float2* grid;
  int nchan, ncorr, nterms, nx, ny, tile, ntx;
  int g0, ng_total;      // this pass handles grids g0 .. g0+NG-1 of ng_total = nterms*ncorr (g = t*ncorr + p)
};

template <int NB, int NG, int NSTAGE>
struct lra_tiled_smem {
  static constexpr int SMAX = 32 * NB - 31;
  static constexpr int SLAB_BYTES = ((SMAX * SMAX + 1) / 2) * 16;
  alignas(128) unsigned char slab[NSTAGE][SLAB_BYTES];
  lra_point_params<NG> params[NSTAGE][LRA_RUNMAX];
  lra_stage_hdr hdr[NSTAGE];
  uint64_t full[NSTAGE], empty[NSTAGE];
};

// NB x-blocks of 32 columns, RPW rows per consumer warp, NW consumer warps (+1 producer warp), NG grids per pass.
template <int NB, int RPW, int NW, int NG, int CLS, int NSTAGE, int MINB>
__global__ void __launch_bounds__((NW + 1) * 32, MINB) lra_grid_tiled_kernel(const lra_tiled_args a) {
  constexpr int RX = 32 * NB;
  constexpr int SMAX = RX - 31, HMAX = (SMAX - 1) / 2;
  static_assert(RPW * NW == RX, "square region");
  using Smem = lra_tiled_smem<NB, NG, NSTAGE>;
  extern __shared__ __align__(128) unsigned char lra_smem_raw[];
  Smem& sm = *reinterpret_cast<Smem*>(lra_smem_raw);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

  if (threadIdx.x == 0) {
    for (int s = 0; s < NSTAGE; ++s) { lra_mbar_init(&sm.full[s], 1); lra_mbar_init(&sm.empty[s], NW); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  int stage = 0;
  uint32_t phase = 0;

  if (warp == NW) {
    // ------------------------------- producer warp -------------------------------
    const unsigned n_items = (unsigned)a.counters[2];
    for (;;) {
      unsigned it = 0xffffffffu;
      if (lane == 0) {
        for (;;) {
          unsigned t = (unsigned)atomicAdd(&a.counters[a.ticket], 1ull);
          if (t >= n_items) break;
          if (a.work[t].w == (unsigned)CLS) { it = t; break; }
        }
      }
      it = __shfl_sync(0xffffffffu, it, 0);
      if (it == 0xffffffffu) {
        lra_mbar_wait(&sm.empty[stage], phase ^ 1u);
        if (lane == 0) {
          sm.hdr[stage].count = 0; sm.hdr[stage].x0 = 0; sm.hdr[stage].y0 = 0; sm.hdr[stage].last = 1;
          lra_mbar_arrive(&sm.full[stage]);
        }
        break;
      }
      const uint4 w = a.work[it];
      const int tx = (int)(w.x % (unsigned)a.ntx), ty = (int)(w.x / (unsigned)a.ntx);
      const int x0 = tx * a.tile - HMAX, y0 = ty * a.tile - HMAX;
      for (unsigned base = 0; base < w.z; base += 32) {
        const int n = min(32u, w.z - base);
        lra_rec r = make_uint4(0, 0xffffffffu, 0, 1);
        lra_point_params<NG> pp;
        pp.ox = pp.oy = 0; pp.S = 1; pp.pad = 0;
#pragma unroll
        for (int g = 0; g < NG; ++g) pp.val[g] = make_float2(0.f, 0.f);
        if (lane < n) {
          r = a.rec[w.y + base + lane];
          const int S = r.w & 0xff, h = (S - 1) >> 1;
          pp.S = S;
          pp.ox = (int)(r.x & 0xffff) - h - x0;
          pp.oy = (int)(r.x >> 16) - h - y0;
          const unsigned k = r.z;
          const int c = (int)(k % (unsigned)a.nchan);
#pragma unroll
          for (int g = 0; g < NG; ++g) {
            const int gi = a.g0 + g;
            if (gi < a.ng_total) {
              const int t = gi / a.ncorr, p = gi - t * a.ncorr;
              const float wgt = a.wt[(size_t)k * a.ncorr + p] * (a.tau ? a.tau[c * a.nterms + t] : 1.0f);
              const float2 v = a.vis[(size_t)k * a.ncorr + p];
              pp.val[g] = make_float2(wgt * v.x, wgt * v.y);
            }
          }
        }
        const unsigned prev = __shfl_up_sync(0xffffffffu, r.y, 1);
        const bool head = lane < n && (lane == 0 || r.y != prev);
        unsigned mask = __ballot_sync(0xffffffffu, head);
        while (mask) {
          const int s = __ffs(mask) - 1;
          mask &= mask - 1;
          const int e = mask ? __ffs(mask) - 1 : n;
          lra_mbar_wait(&sm.empty[stage], phase ^ 1u);
          if (lane >= s && lane < e) sm.params[stage][lane - s] = pp;
          if (lane == s) { sm.hdr[stage].count = e - s; sm.hdr[stage].x0 = x0; sm.hdr[stage].y0 = y0; sm.hdr[stage].last = 0; }
          __syncwarp();
          if (lane == s) {
            const uint32_t bytes = (uint32_t)(((pp.S * pp.S + 1) >> 1) * 16);
            lra_mbar_arrive_expect_tx(&sm.full[stage], bytes);
            lra_tma_load_1d(sm.slab[stage], a.slabs + ((size_t)r.y << 1), bytes, &sm.full[stage]);
          }
          if (++stage == NSTAGE) { stage = 0; phase ^= 1u; }
        }
      }
      // end-of-item marker: consumers flush their registers to the grid
      lra_mbar_wait(&sm.empty[stage], phase ^ 1u);
      if (lane == 0) {
        sm.hdr[stage].count = 0; sm.hdr[stage].x0 = x0; sm.hdr[stage].y0 = y0; sm.hdr[stage].last = 0;
        lra_mbar_arrive(&sm.full[stage]);
      }
      if (++stage == NSTAGE) { stage = 0; phase ^= 1u; }
    }
  } else {
    // ------------------------------- consumer warps -------------------------------
    float2 acc[RPW][NB][NG];
#pragma unroll
    for (int m = 0; m < RPW; ++m)
#pragma unroll
      for (int b = 0; b < NB; ++b)
#pragma unroll
        for (int g = 0; g < NG; ++g) acc[m][b][g] = make_float2(0.f, 0.f);
    const size_t plane = (size_t)a.nx * a.ny;
    for (;;) {
      lra_mbar_wait(&sm.full[stage], phase);
      const lra_stage_hdr hdr = sm.hdr[stage];
      if (hdr.count == 0) {
#pragma unroll
        for (int m = 0; m < RPW; ++m)
#pragma unroll
          for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int g = 0; g < NG; ++g) {
              const float2 v = acc[m][b][g];
              if (a.g0 + g < a.ng_total && (v.x != 0.f || v.y != 0.f)) {
                const int y = hdr.y0 + warp + NW * m, x = hdr.x0 + lane + 32 * b;
                lra_red_add_v2(a.grid + (size_t)(a.g0 + g) * plane + (size_t)y * a.nx + x, v);
              }
              acc[m][b][g] = make_float2(0.f, 0.f);
            }
      } else {
        const float2* sl = reinterpret_cast<const float2*>(sm.slab[stage]);
        for (int q = 0; q < hdr.count; ++q) {
          const lra_point_params<NG>& P = sm.params[stage][q];
          const int S = P.S;
          const int ci = lane - P.ox, rj = warp - P.oy;
          float2 val[NG];
#pragma unroll
          for (int g = 0; g < NG; ++g) val[g] = P.val[g];
#pragma unroll
          for (int m = 0; m < RPW; ++m) {
            const int j = rj + NW * m;
            if ((unsigned)j < (unsigned)S) {
              const float2* row = sl + j * S + ci;
#pragma unroll
              for (int b = 0; b < NB; ++b) {
                if ((unsigned)(ci + 32 * b) < (unsigned)S) {
                  const float2 cf = row[32 * b];
#pragma unroll
                  for (int g = 0; g < NG; ++g) {
                    acc[m][b][g].x = fmaf(cf.x, val[g].x, acc[m][b][g].x);
                    acc[m][b][g].x = fmaf(-cf.y, val[g].y, acc[m][b][g].x);
                    acc[m][b][g].y = fmaf(cf.x, val[g].y, acc[m][b][g].y);
                    acc[m][b][g].y = fmaf(cf.y, val[g].x, acc[m][b][g].y);
                  }
                }
              }
            }
          }
        }
      }
      __syncwarp();
      if (lane == 0) lra_mbar_arrive(&sm.empty[stage]);
      if (++stage == NSTAGE) { stage = 0; phase ^= 1u; }
      if (hdr.count == 0 && hdr.last) break;
    }
  }
}

// Class-2 items (supports > 65): every tap a global atomic, one CTA per item.
__global__ void __launch_bounds__(256)
lra_grid_items_atomic_kernel(const lra_tiled_args a, int cls) {
  const unsigned n_items = (unsigned)a.counters[2];
  const size_t plane = (size_t)a.nx * a.ny;
  for (unsigned it = blockIdx.x; it < n_items; it += gridDim.x) {
    const uint4 w = a.work[it];
    if ((int)w.w != cls) continue;
    for (unsigned q = 0; q < w.z; ++q) {
      const lra_rec r = a.rec[w.y + q];
      const int ix = r.x & 0xffff, iy = r.x >> 16, S = r.w & 0xff, h = (S - 1) >> 1;
      const float2* slab = a.slabs + ((size_t)r.y << 1);
      const unsigned k = r.z;
      const int c = (int)(k % (unsigned)a.nchan);
      for (int gi = 0; gi < a.ng_total; ++gi) {
        const int t = gi / a.ncorr, p = gi - t * a.ncorr;
        const float wgt = a.wt[(size_t)k * a.ncorr + p] * (a.tau ? a.tau[c * a.nterms + t] : 1.0f);
        const float2 x = a.vis[(size_t)k * a.ncorr + p];
        const float2 v = make_float2(wgt * x.x, wgt * x.y);
        for (int e = threadIdx.x; e < S * S; e += 256) {
          const int j = e / S, i = e - j * S;
          const float2 cf = slab[e];
          float2 u;
          u.x = fmaf(-cf.y, v.y, cf.x * v.x);
          u.y = fmaf(cf.y, v.x, cf.x * v.y);
          lra_red_add_v2(a.grid + (size_t)gi * plane + (size_t)(iy - h + j) * a.nx + (ix - h + i), u);
        }
      }
    }
  }
}

// Called at the end of lra_bin: the work list depends on the geometry only.
int lra_build_work(lra_plan* p) {
  const int64_t n = p->npoints;
  int64_t cap = (n < p->ntiles ? n : p->ntiles) + n / LRA_CHUNK + 2;
  if (cap > p->work_capacity) {
    LRA_CUDA(p, cudaStreamSynchronize(p->stream));
    if (p->work) { cudaFree(p->work); p->work = nullptr; }
    LRA_CUDA(p, cudaMalloc(&p->work, (size_t)cap * sizeof(uint4)));
    p->work_capacity = cap;
  }
  if (!p->item_off) LRA_CUDA(p, cudaMalloc(&p->item_off, (size_t)(p->ntiles + 1) * sizeof(uint32_t)));
  const int tb = (p->ntiles + 1 + 255) / 256;
  lra_work_count_kernel<<<tb, 256, 0, p->stream>>>(p->tile_start, p->ntiles, p->item_off);
  LRA_LAUNCH_CHECK(p);
  lra_scan_kernel_launch(p, p->item_off, p->ntiles + 1);
  LRA_LAUNCH_CHECK(p);
  lra_work_fill_kernel<<<tb, 256, 0, p->stream>>>(p->tile_start, p->ntiles, p->item_off, (uint4*)p->work, p->counters);
  LRA_LAUNCH_CHECK(p);
  lra_work_class_kernel<<<p->sm_count * 4, 256, 0, p->stream>>>(p->rec, (uint4*)p->work, p->counters);
  LRA_LAUNCH_CHECK(p);
  return LRA_OK;
}

template <int NB, int RPW, int NW, int NG, int CLS, int NSTAGE, int MINB>
static int lra_launch_tiled(lra_plan* p, const lra_tiled_args& a) {
  using Smem = lra_tiled_smem<NB, NG, NSTAGE>;
  auto kern = lra_grid_tiled_kernel<NB, RPW, NW, NG, CLS, NSTAGE, MINB>;
  LRA_CUDA(p, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem)));
  kern<<<p->sm_count * MINB, (NW + 1) * 32, sizeof(Smem), p->stream>>>(a);
  LRA_LAUNCH_CHECK(p);
  return LRA_OK;
}

int lra_grid_tiled_launch(lra_plan* p, const float2* vis, const float* wt, const float* tau, float2* grid) {
  lra_tiled_args a;
  a.rec = p->rec; a.work = (const uint4*)p->work; a.counters = p->counters; a.slabs = p->slabs;
  a.vis = vis; a.wt = wt; a.tau = tau; a.grid = grid;
  a.nchan = p->nchan; a.ncorr = p->ncorr; a.nterms = p->nterms; a.nx = p->nx; a.ny = p->ny; a.tile = p->tile; a.ntx = p->ntx;
  a.ng_total = p->nterms * p->ncorr;
  LRA_CUDA(p, cudaMemsetAsync(p->counters + 16, 0, 48 * sizeof(unsigned long long), p->stream));
  int ticket = 16, rc;
  const int NGP = a.ng_total == 1 ? 1 : 2;
  for (int g0 = 0; g0 < a.ng_total; g0 += NGP) {
    a.g0 = g0;
    a.ticket = ticket++;
    if (NGP == 1) rc = lra_launch_tiled<2, 8, 8, 1, 0, 4, 2>(p, a); else rc = lra_launch_tiled<2, 8, 8, 2, 0, 4, 2>(p, a);
    if (rc) return rc;
    a.ticket = ticket++;
    if (NGP == 1) rc = lra_launch_tiled<3, 6, 16, 1, 1, 3, 1>(p, a); else rc = lra_launch_tiled<3, 6, 16, 2, 1, 3, 1>(p, a);
    if (rc) return rc;
  }
  a.g0 = 0;
  lra_grid_items_atomic_kernel<<<p->sm_count * 8, 256, 0, p->stream>>>(a, 2);
  LRA_LAUNCH_CHECK(p);
  return LRA_OK;
}

// lra_region.cuh -- what the region gridder (lra_grid_region.cu) and the region degridder (lra_degrid_region.cu) share:
// kernel arguments, the layout of a ring slot, the producer warp and the ring set-up.
// Product code: shares nothing with oracle/.
#pragma once
#include "lra_pipe.cuh"

struct lra_region_args {
  const uint4* work;            // items of this launch's support class
  unsigned n_items;
  unsigned long long* ticket;
  const uint4* batch;           // batch records of this class (4 x uint4 each)
  const float* slabs;
  const void* prep;             // this pass: per sorted position lra_point_bytes (gridder) or the 16-byte pw record
  float2* grid;                 // first grid of this pass
  long long plane;              // pixels per grid
  int nx, ny, tile_x, tile_y, ntx;
  int S, rx, ry, ks;            // the class's geometry (lra_make_geom)
  int core_bytes, stride_bytes, gap_bytes;   // slab as copied; slab + zeros; zeros before the first slab
  int nslot, slot_bytes, slab0; // ring geometry: slots, bytes per slot, offset of the slab area inside a slot
  int out_off;                  // degridder: offset of the per-point results inside a slot
  float2* res;                  // degridder: this pass's results, [sorted position][grids of the pass]
};

// slot layout (bytes): batch record (64) | pad | per-point values | slab area.  The slab area is gap, slab of run 0,
// gap, slab of run 1, ...: the kernel zeroes it once and the copies only ever write the slabs, so the gaps stay
// zero for the whole launch (one launch = one support class = one geometry).
#define LRA_SLOT_VAL 128
#define LRA_RING_HDR 256   // full barriers at +0, empty barriers at +128, the degridder's second empty set at +192 (<= 4 slots)
#define LRA_EMPTY_OUT 64   // offset of that second set from the first: "the results of the slot may be written out"

// Producer warp, shared by the gridder and the degridder: walks the items (atomic ticket) and their batches and
// fills the ring: batch record, `val_bytes` per point from `vals` (if any) and the slab planes.  OUTW > 0 (degridder):
// before a slot is refilled, the OUTW complex results per point its consumers left in it are written to a.res and
// zeroed again.
template <int NW, int OUTW>
__device__ __forceinline__ void lra_region_producer(const lra_region_args& a, const void* vals, uint32_t val_bytes,
                                                    unsigned char* slots, uint32_t full0, uint32_t empty0, uint32_t slots0) {
  const int lane = threadIdx.x & 31;
  const uint32_t slab0 = (uint32_t)a.slab0;
  uint32_t slot = 0, par = 0, issued = 0;
  auto write_out_h = [&](uint32_t s, const uint4 h) {   // all lanes; every consumer warp has released slot s; h: its header
    unsigned char* sp = slots + (size_t)s * a.slot_bytes;
    const unsigned cnt = (h.y & 0xff) * OUTW;
    float2* out = reinterpret_cast<float2*>(sp + a.out_off);
    for (unsigned i = lane; i < cnt; i += 32) {
      a.res[(size_t)h.x * OUTW + i] = out[i];
      out[i] = make_float2(0.f, 0.f);
    }
  };
  auto write_out = [&](uint32_t s) { write_out_h(s, *reinterpret_cast<const uint4*>(slots + (size_t)s * a.slot_bytes)); };
  // tickets and item records are fetched one item ahead, batch records eight batches ahead: lane l of a group of
  // eight batches holds quarter l % 4 of the record of batch l / 4
  unsigned long long t_nxt = 0;
  if (lane == 0) t_nxt = atomicAdd(a.ticket, 1ull);
  t_nxt = __shfl_sync(0xffffffffu, t_nxt, 0);
  uint4 item_nxt = make_uint4(0, 0, 0, 0);
  if (t_nxt < a.n_items) item_nxt = a.work[t_nxt];
  for (;;) {
    if (t_nxt >= a.n_items) break;
    const uint4 item = item_nxt;
    if (lane == 0) t_nxt = atomicAdd(a.ticket, 1ull);
    t_nxt = __shfl_sync(0xffffffffu, t_nxt, 0);
    if (t_nxt < a.n_items) item_nxt = a.work[t_nxt];
    const uint4* rec4 = a.batch + (size_t)item.y * 4;
    const unsigned nb = item.z;
    uint4 nxt = make_uint4(0, 0, 0, 0);
    if ((unsigned)(lane >> 2) < nb) nxt = rec4[lane];
    for (unsigned b0 = 0; b0 < nb; b0 += 8) {
      const uint4 cur = nxt;
      if (b0 + 8 + (lane >> 2) < nb) nxt = rec4[(size_t)(b0 + 8) * 4 + lane];
      const unsigned m = nb - b0 < 8u ? nb - b0 : 8u;
      for (unsigned j = 0; j < m; ++j) {
        // lane 4j owns the batch: slot hand-over, record, prepared values
        const uint32_t sa = slots0 + slot * a.slot_bytes, fb = full0 + 8 * slot;
        const uint32_t nr = __shfl_sync(0xffffffffu, cur.z, 4 * j) & 0xff;
        // degridder: the results the slot's previous batch left are written out AFTER the copies of the new batch have
        // been issued (they touch other parts of the slot), so the write-out hides behind the copies' latency instead
        // of delaying them; the barrier's arrival, which the consumers wait for besides the bytes, comes last
        uint4 h_old = make_uint4(0u, 0u, 0u, 0u);
        const bool had = OUTW > 0 && issued >= (uint32_t)a.nslot;
        if (OUTW > 0) {
          if (lane == 0) lra_mbar_wait(empty0 + 8 * slot, par ^ 1);
          __syncwarp();
          if (had) h_old = *reinterpret_cast<const uint4*>(slots + (size_t)slot * a.slot_bytes);
          __syncwarp();
        }
        ++issued;
        if (lane == (int)(4 * j)) {
          const uint32_t count = cur.y & 0xff;
          const bool pv = vals != nullptr;
          lra_mbar_wait(empty0 + 8 * slot, par ^ 1);
          asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(sa), "r"(cur.x), "r"(cur.y), "r"(cur.z), "r"(cur.w) : "memory");
          const uint32_t bytes = (pv ? count * val_bytes : 0u) + nr * (uint32_t)a.core_bytes;
          if (OUTW > 0) lra_mbar_expect_tx(fb, bytes);
          else lra_mbar_arrive_expect_tx(fb, bytes);
          if (pv) lra_tma_load_1d(sa + LRA_SLOT_VAL, reinterpret_cast<const unsigned char*>(vals) + (size_t)cur.x * val_bytes, count * val_bytes, fb);
        }
        __syncwarp();   // the slot is free from here on
        // one lane issues every slab copy (copies issued from several lanes were measured 20 % slower); slab r of the
        // batch: quarter r / 4 + 1 of its record holds the offset in component r % 4
        for (uint32_t r = 0; r < nr; ++r) {
          const uint32_t c = r & 3;
          const uint32_t pick = c == 0 ? cur.x : c == 1 ? cur.y : c == 2 ? cur.z : cur.w;
          const uint32_t off16 = __shfl_sync(0xffffffffu, pick, 4 * j + 1 + (r >> 2));
          if (lane == 0) {
            const unsigned char* src_b = reinterpret_cast<const unsigned char*>(a.slabs) + ((size_t)off16 << 4);
            lra_tma_load_1d(sa + slab0 + a.gap_bytes + r * a.stride_bytes, src_b, a.core_bytes, fb);
          }
        }
        if (OUTW > 0) {
          if (had) {   // the consumers release the slot's results later than its taps (lra_degrid_region.cuh)
            if (lane == 0) lra_mbar_wait(empty0 + LRA_EMPTY_OUT + 8 * slot, par ^ 1);
            __syncwarp();
            write_out_h(slot, h_old);
          }
          __syncwarp();
          if (lane == (int)(4 * j)) lra_mbar_arrive(fb);
        }
        if (++slot == (uint32_t)a.nslot) { slot = 0; par ^= 1; }
      }
    }
  }
  if (OUTW > 0) {   // drain: results of the batches still in the ring
    for (uint32_t u = 0; u < (uint32_t)a.nslot; ++u) {
      uint32_t s = slot + u, p = par ^ 1;
      if (s >= (uint32_t)a.nslot) { s -= a.nslot; p = par; }
      if (s >= issued) continue;
      if (lane == 0) lra_mbar_wait(empty0 + LRA_EMPTY_OUT + 8 * s, p);
      __syncwarp();
      write_out(s);
      __syncwarp();
    }
  }
  if (lane == 0) {   // end marker
    lra_mbar_wait(empty0 + 8 * slot, par ^ 1);
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(slots0 + slot * a.slot_bytes), "r"(0), "r"(LRA_BATCH_END), "r"(0), "r"(0) : "memory");
    lra_mbar_arrive(full0 + 8 * slot);
  }
}

// The taps of the two pixels this lane owns at one step: {re(e), im(e), re(e + 32), im(e + 32)}.
struct lra_taps { uint32_t v[4]; };

// Loads of one step (predicated off when the step lies outside the point's chunk range).
template <int IMM>
__device__ __forceinline__ void lra_step_load(lra_taps& t, uint32_t addr, uint32_t on) {
  asm volatile("{\n.reg .pred p;\nsetp.ne.u32 p, %6, 0;\n"
               "@p ld.shared.v2.b32 {%0, %1}, [%4+%5];\n"
               "@p ld.shared.v2.b32 {%2, %3}, [%4+%5+256];\n}"
               : "+r"(t.v[0]), "+r"(t.v[1]), "+r"(t.v[2]), "+r"(t.v[3]) : "r"(addr), "n"(IMM), "r"(on));
}

// Step mask of a point for consumer warp `warp` of NW: bit s is set iff chunk NW*s + warp lies in the point's chunk
// range [c_lo, c_hi] (range = c_lo | c_hi << 16, from lra_work.cu).  Warp-uniform.
template <int NW>
__device__ __forceinline__ uint32_t lra_step_mask(uint32_t range, int warp) {
  constexpr int LG = NW == 1 ? 0 : NW == 2 ? 1 : NW == 4 ? 2 : NW == 8 ? 3 : 4;
  const int c_lo = (int)(range & 0xffffu), c_hi = (int)(range >> 16);
  const int s_lo = (c_lo - warp + NW - 1) >> LG, s_hi = (c_hi - warp) >> LG;   // s_hi >= s_lo - 1 >= -1
  return (1u << (s_hi + 1)) - (1u << s_lo);
}
// A value behind an opaque move: it lives in an ordinary (not a uniform) register, so that the predicates of the tap
// loads come from one R2P / per-step LOP3 instead of a uniform extract plus a uniform-to-predicate move each.
__device__ __forceinline__ uint32_t lra_opaque(uint32_t x) {
  uint32_t y;
  asm volatile("mov.b32 %0, %1;" : "=r"(y) : "r"(x));
  return y;
}

// Step mask of a point for consumer warp `warp` from the (z, w) words of its pw record (lra_pipe.cuh): a byte picked
// from the words for NW <= 8 (two uniform instructions), computed from the chunk range for NW = 16.
template <int NW>
__device__ __forceinline__ uint32_t lra_point_mask(uint32_t z, uint32_t w, int warp) {
  if constexpr (NW <= 4) return (z >> (8 * warp)) & 0xffu;
  else if constexpr (NW == 8) return ((warp < 4 ? z : w) >> (8 * (warp & 3))) & 0xffu;
  else return lra_step_mask<NW>(z, warp);
}

// The tap loads of a point, steps [B, KS): predicated on the bits of `mask`.
template <int NW, int KS, int B>
__device__ __forceinline__ void lra_load_steps(lra_taps (&T)[KS], uint32_t addr, uint32_t mask) {
  if constexpr (B < KS) {
    lra_step_load<B * 512 * NW>(T[B], addr, mask & (1u << B));
    lra_load_steps<NW, KS, B + 1>(T, addr, mask);
  }
}

// Ring set-up shared by the gridder and the degridder: barriers, zeroed slab areas.
template <int NW>
__device__ __forceinline__ void lra_region_ring_init(const lra_region_args& a, unsigned char* smem,
                                                     uint32_t full0, uint32_t empty0) {
  if (threadIdx.x == 0) {
    for (int s = 0; s < a.nslot; ++s) {
      lra_mbar_init(full0 + 8 * s, 1);
      lra_mbar_init(empty0 + 8 * s, lra_cw(NW) * 32);
      lra_mbar_init(empty0 + LRA_EMPTY_OUT + 8 * s, lra_cw(NW) * 32);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  const int area16 = (a.slot_bytes - LRA_SLOT_VAL) >> 4;   // everything behind the batch record
  for (int s = 0; s < a.nslot; ++s) {
    uint4* z = reinterpret_cast<uint4*>(smem + LRA_RING_HDR + (size_t)s * a.slot_bytes + LRA_SLOT_VAL);
    for (int i = threadIdx.x; i < area16; i += (lra_cw(NW) + 1) * 32) z[i] = make_uint4(0, 0, 0, 0);
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  __syncthreads();
}

// Ring geometry of a class for a kernel that keeps `val_bytes` per point in the slot.  Returns false if not even
// one slot fits (the class then takes the fallback kernels).
static inline bool lra_region_ring(const lra_geom& q, int ngp, bool degrid, int val_bytes, lra_region_args* a, int* smem_bytes) {
  const int slab0 = (LRA_SLOT_VAL + q.per_batch * LRA_RUNMAX * val_bytes + 127) & ~127;
  const int slot_bytes = (slab0 + 8 * (LRA_GAP + q.per_batch * q.stride) + 127) & ~127;
  int nslot = (lra_cta_smem(q.nw, q.ks, ngp, degrid) - LRA_RING_HDR) / slot_bytes;
  if (nslot < 1) return false;
  if (nslot > 4) nslot = 4;
  a->S = q.S; a->rx = q.rx; a->ry = q.ry; a->ks = q.ks;
  a->core_bytes = 8 * q.core; a->stride_bytes = 8 * q.stride; a->gap_bytes = 8 * LRA_GAP;
  a->nslot = nslot; a->slot_bytes = slot_bytes; a->slab0 = slab0;
  a->out_off = LRA_SLOT_VAL + q.per_batch * LRA_RUNMAX * 16;   // degridder: 16 bytes per point come first
  *smem_bytes = LRA_RING_HDR + nslot * slot_bytes;
  return true;
}

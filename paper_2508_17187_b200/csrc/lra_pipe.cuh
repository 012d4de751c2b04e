// lra_pipe.cuh -- pieces shared by lra_work.cu, the region gridder and the region degridder: the geometry of a support
// class (consumer warps, steps, shared-memory layout of a slab), the format of the batch stream that lra_work.cu
// builds and the kernels consume, and PTX wrappers (mbarrier, 1-D TMA bulk copy, packed fp32x2 FMA, vector reductions
// to global memory).
// Product code: shares nothing with oracle/.
#pragma once
#include "lra_internal.cuh"

#define LRA_CHUNK 1024     // sorted positions per work-list chunk = upper bound on the points of one work item
#define LRA_RUNMAX 16      // points of one slab run inside a batch (longer runs are cut and load their slab again)
#define LRA_BATCH_SLABS 12 // slab runs per batch at most
#define LRA_BATCH_POINTS (LRA_RUNMAX * LRA_BATCH_SLABS)
#ifndef LRA_SLOTS_TARGET
#define LRA_SLOTS_TARGET 2   // ring slots per CTA the batch size is chosen for
#endif
#ifndef LRA_CTA_CAP
#define LRA_CTA_CAP 10      // CTAs per SM at most
#endif
#ifndef LRA_REGS_PER_STEP
#define LRA_REGS_PER_STEP 12   // 8 accumulators + 4 taps in flight per step; 10 (one more CTA per SM) measured no faster
#endif
#define LRA_KSMAX 9        // steps per consumer warp at most: 9 * 2 pixels * 2 grids * (re, im) = 72 accumulators

typedef unsigned long long lra_u64;

// ---------------------------------------------------------------------------------------------------
// Geometry of a support class.  A region kernel keeps a region of RX*RY pixels (tile + halo, RX = tile_x + S - 1,
// RY = tile + S - 1) in the registers of NW consumer warps: pixel e = y*RX + x belongs to warp (e / 64) % NW, step
// e / (64*NW), lane e % 32, half (e / 32) % 2, i.e. at step s a warp owns the 64 consecutive pixels that start at
// 64*(NW*s + warp) and a lane owns two of them, 32 apart (the two halves of one FFMA2).  NW = 2, 4, 8 or 16 is the
// smallest for which ks = ceil(RX*RY / (64*NW)) <= lra_ks_max(NW) (the register budget that still leaves two CTAs of
// NW = 8 on an SM); a region too large for NW = 16 goes to the fallback kernels (global atomics).  Every lane reads a
// tap for every point, at linear slab index e - off with
// off = oy*RX + ox <= pre, so a slab plane sits in shared memory between zeros: `gap` floats before (>= pre) and
// after (>= the pixels past the last tap) -- consecutive planes share a gap, which no copy ever writes.
// ---------------------------------------------------------------------------------------------------
struct lra_geom {
  int S, rx, ry, group, nw, ks;   // group = log2(nw) - 1, or LRA_NGROUP - 1 for the fallback
  int core;                       // floats per slab plane as stored and copied (lra_plane_floats)
  int gap, stride;                // floats of zeros between planes; stride = core + gap
  int per_batch;                  // slab runs per batch
};
#ifndef LRA_KSLIM
#define LRA_KSLIM 9
#endif
__host__ __device__ constexpr int lra_ks_max(int nw) { return nw == 16 ? LRA_KSMAX : nw == 8 ? (LRA_KSLIM < 7 ? LRA_KSLIM : 7) : LRA_KSLIM; }
// CTAs per SM the (NW, KS) kernel is built for: ~12 registers per step (8 accumulators, 4 taps in flight) + 36.
__host__ __device__ constexpr int lra_ctas_per_sm(int nw, int ks) {
  if (nw == 8 && ks == 7) return 2;   // 112 registers: measured without spills
  const int regs = (LRA_REGS_PER_STEP * ks + 36 + 7) / 8 * 8, r = 65536 / ((nw + 1) * 32 * regs);
  return r < 1 ? 1 : r > LRA_CTA_CAP ? LRA_CTA_CAP : r;
}
// Shared memory of a CTA and of one ring slot (3 slots per CTA at least, whenever a slab fits).
__host__ __device__ constexpr int lra_cta_smem(int nw, int ks) { return (227 * 1024) / lra_ctas_per_sm(nw, ks) - 1024; }
__host__ __device__ inline lra_geom lra_make_geom(int S, int tile_x, int tile_y) {
  lra_geom q;
  q.S = S; q.rx = S + tile_x - 1; q.ry = S + tile_y - 1;
  const int slots = q.rx * q.ry;
  q.group = LRA_NGROUP - 1; q.nw = 0; q.ks = 0;
  for (int g = 0; g < LRA_NGROUP - 1; ++g)
    if (slots <= 64 * (2 << g) * lra_ks_max(2 << g)) { q.group = g; q.nw = 2 << g; q.ks = (slots + 64 * q.nw - 1) / (64 * q.nw); break; }
  q.core = lra_plane_floats(S, tile_x);
  const int pre = (tile_y - 1) * q.rx + tile_x - 1, post = 64 * q.nw * q.ks - S * q.rx;
  q.gap = ((pre > post ? pre : post) + 3) & ~3;
  q.stride = q.core + q.gap;
  q.per_batch = 1;
  if (q.group < LRA_NGROUP - 1) {   // a third of the CTA's shared memory per slot: 384 bytes of values + a slab per run
    const int r = ((lra_cta_smem(q.nw, q.ks) - 512) / LRA_SLOTS_TARGET - 256 - 4 * q.gap) / (LRA_RUNMAX * 64 + 8 * q.stride);
    q.per_batch = r < 1 ? 1 : r > LRA_BATCH_SLABS ? LRA_BATCH_SLABS : r;
    // even one slab per slot must fit the CTA's shared memory (values + record + ring header: 1 KB), else fall back
    if (4 * (q.gap + 2 * q.stride) + 1024 > lra_cta_smem(q.nw, q.ks)) { q.group = LRA_NGROUP - 1; q.per_batch = 1; }
  }
  return q;
}
__host__ __device__ inline int lra_class_of(int S) { return (S - 1) >> 1; }

// ---------------------------------------------------------------------------------------------------
// Batch stream (built once per lra_bin by lra_work.cu; geometry only, reused by every lra_grid / lra_degrid).
//   item  = maximal run of sorted positions with the same uv tile and the same support, cut at multiples of
//           LRA_CHUNK: uint4 {tile id, first batch (class-relative), number of batches, S}.  One CTA accumulates an
//           item's region in registers and adds it to the grid once.  Items are grouped by support class.
//   run   = at most LRA_RUNMAX consecutive points of an item that share one CF slab.
//   batch = per_batch consecutive runs of one item: what occupies one slot of a CTA's shared-memory ring.
//           64 bytes: uint4 {first sorted position, count | flags, runs, tile id}, then the slab offsets of its
//           runs in 16-byte units (uint32 x 12).  LRA_BATCH_LAST marks the last batch of its item.
//   pw    = for every sorted position 16 bytes (one TMA granule) {word, k, S, 0}; word = the byte offset, inside the
//           slot's slab area, of the float the lane that owns pixel 0 of the region reads for this point:
//           4 * (gap + run * 2 * stride - (oy*RX + ox)).
// ---------------------------------------------------------------------------------------------------
#define LRA_BATCH_LAST 0x40000000u
#define LRA_BATCH_END 0x80000000u

// counters (unsigned long long): [0] n_valid, [1] sum S^2; per support class c: [128 + c] items, [256 + c] batches,
// [384 + c] item cursor, [512 + c] batch cursor, [640 + c] first item, [768 + c] first batch; [1024..2047] work
// tickets of the launches of one call.
#define LRA_NCOUNTER 2048
#define LRA_CNT_ITEMS 128
#define LRA_CNT_BATCHES 256
#define LRA_CNT_ITEM_CUR 384
#define LRA_CNT_BATCH_CUR 512
#define LRA_CNT_ITEM_OFF 640
#define LRA_CNT_BATCH_OFF 768
#define LRA_TICKET0 1024
#define LRA_NTICKET 1024

// ---------------------------------------------------------------------------------------------------
// PTX wrappers
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t lra_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void lra_mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void lra_mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void lra_mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void lra_mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar), "r"(parity), "r"(0x989680u) : "memory");   // suspend-time hint: park, do not spin
}
// One contiguous piece, global (L2) -> shared, completion counted in bytes on `bar`.
__device__ __forceinline__ void lra_tma_load_1d(uint32_t smem_dst, const void* gmem_src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_dst),
               "l"(gmem_src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void lra_red_add_v2(float2* addr, float re, float im) {
  asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(addr), "f"(re), "f"(im) : "memory");
}
// Packed fp32x2: d = a * b + c on both halves, one issue slot for two FMAs (FFMA2 on sm_100a).
__device__ __forceinline__ lra_u64 lra_fma2(lra_u64 a, lra_u64 b, lra_u64 c) {
  lra_u64 d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}
__device__ __forceinline__ lra_u64 lra_pack2(float lo, float hi) {
  lra_u64 d;
  asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi));
  return d;
}
// A pair that lives across a whole item as an FFMA2 *input*: produced by an FFMA2 (x * 1 + 0), which makes the register
// allocator keep it in an aligned register pair instead of re-assembling it from two single registers before every use.
__device__ __forceinline__ lra_u64 lra_pack2_keep(float lo, float hi) {
  lra_u64 d, x, one;
  asm("mov.b64 %0, {%1, %2};" : "=l"(x) : "f"(lo), "f"(hi));
  asm("mov.b64 %0, {%1, %1};" : "=l"(one) : "f"(1.0f));
  asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(x), "l"(one), "l"(0ull));
  return d;
}
__device__ __forceinline__ void lra_unpack2(lra_u64 v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}

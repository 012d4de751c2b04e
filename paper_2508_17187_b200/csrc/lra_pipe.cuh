// lra_pipe.cuh -- pieces shared by the strip gridder and the strip degridder: PTX wrappers (mbarrier, 1-D TMA bulk
// copy, packed fp32x2 FMA, vector reductions to global memory), the kernel configurations ("groups") and the
// format of the stage stream that lra_work.cu builds and the kernels consume.
// Product code: shares nothing with oracle/.
#pragma once
#include "lra_internal.cuh"

#define LRA_CHUNK 1024     // sorted positions per work-list chunk = upper bound on the points of one work item
#define LRA_RUNMAX 16      // points per pipeline stage
#define LRA_PW_STRIDE 16   // per-point words: one per consumer warp, 16 = the largest warp count of a group

typedef unsigned long long lra_u64;

// ---------------------------------------------------------------------------------------------------
// Groups.  A strip kernel keeps a region of RX*RY pixels (tile + halo, RX = tile_x + S - 1, RY = tile + S - 1) in
// the registers of NW consumer warps: pixel e = y*RX + x belongs to warp (e / 64) % NW, lane e % 32, step
// e / (64*NW), half (e / 32) % 2, i.e. at step s a warp owns the 64 consecutive pixels that start at
// 64*(NW*s + warp) and a lane owns two of them, 32 apart (the two halves of one FFMA2).  A group is one
// compile-time choice of (NW, KS = steps); an item goes to the smallest group whose 64*NW*KS pixels hold its
// region, and to the fallback group (global atomics, no limit) if none does.
// ---------------------------------------------------------------------------------------------------
__host__ __device__ inline int lra_group_nw(int g) { return g == 0 ? 4 : g == 1 ? 8 : 16; }
__host__ __device__ inline int lra_group_ks(int g) { return g == 0 ? 8 : g == 1 ? 8 : g == 2 ? 7 : 9; }
__host__ __device__ inline int lra_group_slots(int g) { return 64 * lra_group_nw(g) * lra_group_ks(g); }
__host__ __device__ inline int lra_group_of(int S, int tile_x, int tile_y) {
  const int slots = (S + tile_x - 1) * (S + tile_y - 1);
  for (int g = 0; g < LRA_NGROUP - 1; ++g)
    if (slots <= lra_group_slots(g)) return g;
  return LRA_NGROUP - 1;
}

// ---------------------------------------------------------------------------------------------------
// Stage stream (built once per lra_bin by lra_work.cu; geometry only, reused by every lra_grid / lra_degrid).
//   item  = maximal run of sorted positions with the same uv tile and the same support, cut at multiples of
//           LRA_CHUNK: uint4 {tile id, first stage (group-relative), number of stages, S}.  One CTA accumulates an
//           item's region in registers and adds it to the grid once.
//   stage = run of at most LRA_RUNMAX points of one item that share one CF slab, i.e. what occupies one slot of a
//           CTA's shared-memory ring: uint4 {first sorted position, count | S << 8 | flags, slab offset in
//           16-byte units, tile id}.  LRA_STAGE_LAST marks the last stage of its item.
//   pw    = for every sorted position, LRA_PW_STRIDE words, one per consumer warp w of the point's group:
//           4*(oy*RX + ox) in the low half (byte offset of the point's footprint origin in the region) and, in
//           the high half, bit s set <=> the 64 pixels warp w owns at step s meet the point's footprint.
// ---------------------------------------------------------------------------------------------------
#define LRA_STAGE_LAST 0x40000000u
#define LRA_STAGE_END 0x80000000u

// counters[0] n_valid, [1] sum S^2, [8..15] items per group, [16..23] stages per group, [24..31] item cursors,
// [32..39] stage cursors, [40..47] item offsets, [48..55] stage offsets, [64..127] work tickets of the launches.
#define LRA_TICKET0 64
#define LRA_NTICKET 64

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
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar), "r"(parity) : "memory");
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
__device__ __forceinline__ void lra_unpack2(lra_u64 v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ float lra_lds(uint32_t addr) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ uint32_t lra_lds_u32(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ uint4 lra_lds_v4(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
  return v;
}
__device__ __forceinline__ void lra_lds_2x64(uint32_t addr, lra_u64& a, lra_u64& b) {
  asm volatile("ld.shared.v2.u64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "r"(addr));
}
__device__ __forceinline__ lra_u64 lra_lds_u64(uint32_t addr) {
  lra_u64 v;
  asm volatile("ld.shared.u64 %0, [%1];" : "=l"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ void lra_sts_v4(uint32_t addr, uint4 v) {
  asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

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
#define LRA_CTA_CAP 12      // CTAs per SM at most
#endif
#define LRA_KSCAP 8         // steps per consumer warp at most (the step mask of a point is 8 bits wide)
#define LRA_NGMAX 4         // grids per pass at most (more grids: several passes over the same batch stream)
#define LRA_GAP 64          // complex zeros before, between and after the slabs of a ring slot

typedef unsigned long long lra_u64;

// ---------------------------------------------------------------------------------------------------
// Geometry of a support class.  A region kernel keeps a region of RX*RY pixels (tile + halo, RX = tile_x + S - 1,
// RY = tile + S - 1) in the registers of NW consumer warps: pixel e = y*RX + x belongs to chunk e / 64; chunk c
// belongs to warp c % NW, step c / NW, i.e. at step s a warp owns the 64 consecutive pixels that start at
// 64*(NW*s + warp) and a lane owns two of them, 32 apart, each as one complex accumulator (an aligned register
// pair) per grid.  NW = 1, 2, 4, 8 or 16 is the smallest for which KS = ceil(chunks / NW) <= lra_ks_max(grids per
// pass); KS is rounded up to an even number where that still fits (fewer kernel instantiations; the surplus steps are
// never active).  A region too large for NW = 16 goes to the fallback kernels (global atomics).
// A point with footprint origin (ox, oy) inside the region puts tap (j, i) on pixel off + j*RX + i, off = oy*RX + ox,
// so its taps lie in the pixel range [off, off + L), L = (S-1)*RX + S: a lane reads the tap of pixel e at linear slab
// index e - off, and only the chunks c_lo = off/64 .. c_hi = (off + L - 1)/64 of the region are visited (the rest of
// the region lies above or below the footprint).  Inside the visited range a lane beside the footprint reads one
// of the zeros that end every slab row, or one of the LRA_GAP zeros around the slab in shared memory.
// ---------------------------------------------------------------------------------------------------
struct lra_geom {
  int S, rx, ry, nw, ks;          // nw = 0: the fallback kernels
  int span;                       // L: pixels from the first to the last tap of a footprint
  int core;                       // complex values per slab as stored and copied (lra_slab_complex)
  int stride;                     // core + LRA_GAP
  int per_batch;                  // slab runs per batch
};
__host__ __device__ constexpr int lra_ks_max(int ngp) { return ngp == 1 ? 8 : ngp == 2 ? 6 : 4; }
__host__ __device__ constexpr int lra_grids_per_pass(int ng) { return ng < LRA_NGMAX ? ng : LRA_NGMAX; }
// Registers per thread the (NW, KS, NG) kernels are built for.  lra_regs_need: the fewest registers (a multiple of 8)
// with which ptxas builds the kernel without spilling (per step 4 accumulators per grid and 4 tap values in flight,
// plus addressing and the point's values; the degridder also holds the partial sums of four points), found by
// compiling every (KS, NG) under a range of register limits.  CTAs per SM follow from it, and the kernel is then given
// all the registers that this number of CTAs leaves (lra_regs).
__host__ __device__ constexpr int lra_regs_need(int ks, int ngp, bool degrid) {
  // rows: grids per pass 1..4; columns: KS 1..8
  constexpr int G[4][8] = {{48, 48, 56, 64, 80, 80, 104, 104}, {48, 56, 64, 80, 96, 96, 96, 96}, {64, 72, 88, 112, 112, 112, 112, 112}, {80, 96, 120, 136, 136, 136, 136, 136}};
  constexpr int D[4][8] = {{48, 56, 56, 64, 80, 80, 96, 96}, {56, 64, 64, 80, 96, 96, 96, 96}, {64, 80, 96, 112, 112, 112, 112, 112}, {72, 104, 120, 136, 136, 136, 136, 136}};
  return degrid ? D[ngp - 1][ks - 1] : G[ngp - 1][ks - 1];
}
// The register file is 16384 registers per SM sub-partition and the warps of the resident CTAs are dealt round to the
// four sub-partitions: C CTAs of NW + 1 warps put ceil((NW + 1) * C / 4) warps on the fullest one.
#ifndef LRA_PS_WARPS
#define LRA_PS_WARPS 3   // consumer warps of a CTA whose whole region fits ONE warp's registers (nw = 1); with the producer
                         // a CTA is four warps, one per SM sub-partition (measured on cfg3: 3 -> 55.95, 4 -> 56.05, 7 -> 56.35 ms per step)
#endif
// Consumer warps per CTA.  nw >= 2: the warps split the PIXELS of the region (chunk c belongs to warp c % nw) and every
// warp visits every point.  nw = 1: a warp holds the whole region, and LRA_PS_WARPS such warps split the POINTS of a
// batch instead (point q belongs to warp q % LRA_PS_WARPS): a point is visited once, its bookkeeping is paid once (the
// degridder also reduces it across lanes once), and the warps' regions are added up by the flush.  Measured on cfg3
// against two pixel-splitting warps: S = 9: gridder -1 %, degridder -34 %; S = 11: gridder -8 %, degridder -23 %.
__host__ __device__ constexpr int lra_cw(int nw) { return nw == 1 ? LRA_PS_WARPS : nw; }
__host__ __device__ constexpr int lra_warps_per_smsp(int nw, int ctas) { return ((lra_cw(nw) + 1) * ctas + 3) / 4; }
__host__ __device__ constexpr int lra_ctas_per_sm(int nw, int ks, int ngp, bool degrid) {
  int r = 1;
  while (r < LRA_CTA_CAP && (lra_cw(nw) + 1) * (r + 1) <= 64 && lra_warps_per_smsp(nw, r + 1) * 32 * lra_regs_need(ks, ngp, degrid) <= 16384) ++r;
  return r;
}
__host__ __device__ constexpr int lra_regs(int nw, int ks, int ngp, bool degrid) {
  const int r = 16384 / (32 * lra_warps_per_smsp(nw, lra_ctas_per_sm(nw, ks, ngp, degrid))) / 8 * 8;
  return r > 168 ? 168 : r;
}
#ifdef LRA_FORCE_NREG   // build aid: find the registers a kernel needs
#define LRA_MAXNREG(nw, ks, ng, degrid) (LRA_FORCE_NREG + 0 * (ks))
#else
#define LRA_MAXNREG(nw, ks, ng, degrid) lra_regs(nw, ks, ng, degrid)
#endif
// Shared memory of a CTA.  The batch stream (lra_work.cu) is cut for the gridder's CTAs, the smaller ones.
__host__ __device__ constexpr int lra_cta_smem(int nw, int ks, int ngp, bool degrid) { return (227 * 1024) / lra_ctas_per_sm(nw, ks, ngp, degrid) - 1024; }
// Bytes per point in a ring slot: gridder 16 per grid (vx, vy, -vy, vx) + 16 (word, chunk range); degridder 16 (the
// pw record) + 8 per grid (results).
__host__ __device__ constexpr int lra_point_bytes(int ngp) { return 16 * ngp + 16; }
__host__ __device__ inline lra_geom lra_make_geom(int S, int tile_x, int tile_y, int ng) {
  lra_geom q;
  const int ngp = lra_grids_per_pass(ng);
  q.S = S; q.rx = S + tile_x - 1; q.ry = S + tile_y - 1;
  q.span = (S - 1) * q.rx + S;
  const int chunks = (q.rx * q.ry + 63) / 64;
  q.nw = 0; q.ks = 0;
#ifndef LRA_KS_PREF
#define LRA_KS_PREF 8   // preferred steps per warp (measured on cfg3: 3, i.e. more and lighter warps, is 8 % slower: the per-point overhead of a warp dominates)
#endif
  for (int pass = 0; pass < 2 && q.nw == 0; ++pass) {
    const int lim = pass == 0 && LRA_KS_PREF < lra_ks_max(ngp) ? LRA_KS_PREF : lra_ks_max(ngp);
#ifndef LRA_NW_MIN
#define LRA_NW_MIN 2   // consumer warps per CTA at least: with one, half of the resident warps are producers (measured on cfg3: 1 -> 2: -0.6 ms gridder, -0.4 ms degridder; 4: worse)
#endif
    for (int nw = 1; nw <= 16; nw <<= 1) {
      if (nw == 1 ? LRA_PS_WARPS < 2 && LRA_NW_MIN > 1 : nw < LRA_NW_MIN) continue;
      int ks = (chunks + nw - 1) / nw;
      if (ks == 7 || (ks == 5 && ngp > 2)) ++ks;   // the kernels are instantiated for KS = 1, 2, 3, 4, 5 (one or two grids), 6, 8
      if (ks > lim) continue;
      q.nw = nw; q.ks = ks;
      break;
    }
  }
  q.core = lra_slab_complex(S, tile_x);
  q.stride = q.core + LRA_GAP;
  q.per_batch = 1;
  if (q.nw) {
    const int r = ((lra_cta_smem(q.nw, q.ks, ngp, false) - 512) / LRA_SLOTS_TARGET - 256 - 8 * LRA_GAP) / (LRA_RUNMAX * lra_point_bytes(ngp) + 8 * q.stride);
    q.per_batch = r < 1 ? 1 : r > LRA_BATCH_SLABS ? LRA_BATCH_SLABS : r;
    // even one slab per slot must fit the CTA's shared memory (values + record + ring header: 1.5 KB), else fall back
    if (8 * (LRA_GAP + q.stride) + LRA_RUNMAX * lra_point_bytes(ngp) + 1536 > lra_cta_smem(q.nw, q.ks, ngp, false)) { q.nw = 0; q.ks = 0; q.per_batch = 1; }
  }
  return q;
}
__host__ __device__ inline int lra_class_of(int S) { return (S - 1) >> 1; }
// Which support classes take the fallback kernels (bit c of lo for c < 64, bit c - 64 of hi): computed once on the
// host, so that per-point kernels need not evaluate the geometry.
struct lra_fallback_mask { unsigned long long lo; unsigned hi; };
inline lra_fallback_mask lra_make_fallback_mask(int tile_x, int tile_y, int ng) {
  lra_fallback_mask m = {0ull, 0u};
  for (int c = 0; c < LRA_NCLASS; ++c)
    if (lra_make_geom(2 * c + 1, tile_x, tile_y, ng).nw == 0) { if (c < 64) m.lo |= 1ull << c; else m.hi |= 1u << (c - 64); }
  return m;
}
__device__ __forceinline__ bool lra_is_fallback(const lra_fallback_mask& m, int S) {
  const int c = lra_class_of(S);
  return c < 64 ? (m.lo >> c) & 1ull : (m.hi >> (c - 64)) & 1u;
}

// ---------------------------------------------------------------------------------------------------
// Batch stream (built once per lra_bin by lra_work.cu; geometry only, reused by every lra_grid / lra_degrid).
//   item  = maximal run of sorted positions with the same uv tile and the same support, cut at multiples of
//           LRA_CHUNK: uint4 {tile id, first batch (class-relative), number of batches, S}.  One CTA accumulates an
//           item's region in registers and adds it to the grid once.  Items are grouped by support class.
//   run   = at most LRA_RUNMAX consecutive points of an item that share one CF slab.
//   batch = per_batch consecutive runs of one item: what occupies one slot of a CTA's shared-memory ring.
//           64 bytes: uint4 {first sorted position, count | flags, runs, tile id}, then the slab offsets of its
//           runs in 16-byte units (uint32 x 12).  LRA_BATCH_LAST marks the last batch of its item.
//   pw    = for every sorted position 16 bytes (one TMA granule) {word, k | fallback << 31, z, w}; word = the byte
//           offset (signed), inside the slot's slab area, of the complex value the lane that owns pixel 0 of the
//           region would read for this point: 8 * (LRA_GAP + run * stride - off), off = oy*RX + ox; k = the point's
//           index in the caller's arrays, bit 31 set if its class takes the fallback kernels; for NW <= 8, byte w of
//           (z, w) = the step mask of consumer warp w (bit s: chunk NW*s + w lies in [c_lo, c_hi], the first and last
//           chunk of the region that the footprint touches); for NW = 16, z = c_lo | c_hi << 16.
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
// The arrival under a (warp-uniform) condition, as a branch around it: the address arithmetic of the barrier is skipped too
__device__ __forceinline__ void lra_mbar_arrive_if(uint32_t bar, uint32_t cond) {
  asm volatile("{\n.reg .pred p;\nsetp.eq.u32 p, %1, 0;\n@p bra.uni NOARR_%=;\nmbarrier.arrive.shared::cta.b64 _, [%0];\nNOARR_%=:\n}" ::"r"(bar), "r"(cond) : "memory");
}
// Adds to the transaction count only: the phase still needs the arrival (lra_mbar_arrive), which may come later.
__device__ __forceinline__ void lra_mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
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
// The same under a predicate formed inside the statement (no divergent branch around the reduction): pixel e belongs to the
// region (e < npix) and the value is not +-0.
__device__ __forceinline__ void lra_red_add_v2_nz(float2* addr, lra_u64 v, uint32_t e, uint32_t npix) {
  asm volatile(
      "{\n.reg .pred p, q;\n.reg .b32 lo, hi, t;\nmov.b64 {lo, hi}, %1;\nor.b32 t, lo, hi;\nshl.b32 t, t, 1;\n"
      "setp.lt.u32 q, %2, %3;\nsetp.ne.and.u32 p, t, 0, q;\n@p red.global.add.v2.f32 [%0], {lo, hi};\n}"
      ::"l"(addr), "l"(v), "r"(e), "r"(npix) : "memory");
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

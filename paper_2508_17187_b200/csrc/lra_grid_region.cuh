// lra_grid_region.cuh -- the default gridder (variant 0): region-owning CTAs that accumulate in REGISTERS with packed
// fp32x2 FMAs and read the convolution function from a TMA-fed shared-memory ring.  Kernel template and its launch
// dispatch; instantiated per number of grids in lra_grid_region_ng*.cu, driven by lra_grid_region.cu.
//
// Operation: Eq. 7 / Eq. 23 of arxiv 2508.17187, tap loop of SURVEY Sec. 8(a) rows a3, a4.
//
// Design (B200-first; the paper's Kokkos kernel is prior art only):
//   * lra_bin left the visibility points sorted by uv tile (8 x 8 pixels by default), then by CF slab.  A work item
//     (lra_work.cu) is a run of at most LRA_CHUNK points of one tile and one support S; persistent CTAs take items
//     through an atomic ticket, so the dense centre of a VLA-like uv plane is spread over many CTAs.
//   * A CTA owns the item's region = tile + halo, RX x RY = (tile_x + S - 1) x (tile + S - 1) pixels, numbered
//     linearly e = y*RX + x.  Consumer warp w owns, at step s, the 64 consecutive pixels from 64*(NW*s + w); a lane
//     owns two of them, 32 apart.  The complex accumulator of a pixel is one aligned register pair per grid, kept for
//     the whole item and added to the HBM grid once per item with red.global.add.v2.f32 (row a4).
//   * The CF slab is stored with the region's pitch RX as interleaved complex taps with zeros ending each row
//     (lra_internal.cuh), so the tap of pixel e for a point whose footprint starts at linear pixel `off` is simply
//     slab[e - off]: one 8-byte shared-memory load per lane and pixel, 32 consecutive values per warp (no bank
//     conflicts whatever RX is); lanes beside the footprint read zeros.
//   * A point's taps lie in the pixel range [off, off + L): a warp runs only its steps inside that range.  The step
//     mask of a point is warp-uniform and lives in uniform registers, so a skipped step costs one uniform branch and
//     two predicated-off loads, no FMA-pipe time: the rows of the region above and below the footprint are free.
//     (Measured alternative, rejected: one indirect jump per point to straight-line code of its step range; fewer
//     instructions, but the jump's latency made it 10 % slower.)
//   * The tap update of one pixel on one grid is two FFMA2 (fma.rn.f32x2) with the tap as the scalar operand:
//       acc(re, im) += cre * (vx, vy);   acc(re, im) += cim * (-vy, vx)
//     (ptxas folds the duplicated tap into the FFMA2's scalar-broadcast operand form), so two 8-byte loads feed
//     4 * NG FFMA2: the FP32 pipe and the shared-memory port saturate together at NG = 2 and the pipe alone binds at
//     NG = 4.
//   * The loads are software-pipelined by hand (the branches around the steps keep the compiler from doing it): a
//     step multiplies the taps of point q and then reloads the same registers with the taps of point q + 1, so a
//     tap is in flight for a whole point.
//   * lra_prepare_kernel first gathers vis / weight in SORTED order and writes, per point, the NG operand pairs
//     (vx, vy, -vy, vx) = wt*tau*V and the point's slab offset and chunk range as one contiguous record.
//   * The producer warp walks the batch stream of lra_work.cu and issues, per batch (= up to 12 slab runs of an
//     item), TMA bulk copies (cp.async.bulk + mbarrier complete_tx): the records of its points and its CF slabs,
//     from L2 into a ring of shared-memory slots; item boundaries ride in the batch headers, so the consumers
//     never touch the work list and synchronise once per batch, not once per slab.
// Regions that fit no (NW, KS) take the global-atomic kernel of lra_grid.cu.
#pragma once
#include <type_traits>
// Whether an instantiation gets the second, cheaper code path of the flush for regions inside the grid (below).  Measured:
// cfg3 gridder 19.78 -> 19.23 ms, cfg5 13.91 -> 13.48 ms; with four grids and three steps ptxas then builds the TAP LOOP of
// the 4- and 8-warp kernels with 15 % more register moves (cfg4: those classes +5 %, the call 33.25 -> 33.90 ms), so these
// keep the single path (cfg4 33.15 ms, cfg5 13.52 ms).
__host__ __device__ constexpr bool lra_fast_flush(int nw, int ks, int ng) { return !(ng == 4 && ks == 3 && nw < 16); }

#include "lra_region.cuh"

// One step of the software pipeline: the FMAs of the CURRENT point on the two pixels this lane owns at the step
// (acc[pixel][grid] = (re, im), taps t = {re(e), im(e), re(e + 32), im(e + 32)}), under a uniform branch on `on`, then
// the loads of the NEXT point's taps for the same step into the same registers (predicated on `on_next`): the taps
// of a step are in flight for one whole point.
template <int NG, int IMM>
__device__ __forceinline__ void lra_step(lra_u64 (&acc)[2][NG], const lra_u64 (&V)[NG], const lra_u64 (&W)[NG], lra_taps& t,
                                         uint32_t on, uint32_t addr, uint32_t on_next) {
  if constexpr (NG == 1) {
    asm volatile(
        "{\n.reg .pred p, q;\n.reg .b64 ar, ai, br, bi;\nsetp.eq.u32 p, %8, 0;\n@p bra.uni SKIP_%=;\n"
        "mov.b64 ar, {%2, %2};\nmov.b64 ai, {%3, %3};\nmov.b64 br, {%4, %4};\nmov.b64 bi, {%5, %5};\n"
        "fma.rn.f32x2 %0, ar, %6, %0;\nfma.rn.f32x2 %1, br, %6, %1;\n"
        "fma.rn.f32x2 %0, ai, %7, %0;\nfma.rn.f32x2 %1, bi, %7, %1;\n"
        "SKIP_%=:\nsetp.ne.u32 q, %11, 0;\n"
        "@q ld.shared.v2.b32 {%2, %3}, [%9+%10];\n@q ld.shared.v2.b32 {%4, %5}, [%9+%10+256];\n}"
        : "+l"(acc[0][0]), "+l"(acc[1][0]), "+r"(t.v[0]), "+r"(t.v[1]), "+r"(t.v[2]), "+r"(t.v[3])
        : "l"(V[0]), "l"(W[0]), "r"(on), "r"(addr), "n"(IMM), "r"(on_next));
  }
  if constexpr (NG == 2) {
    asm volatile(
        "{\n.reg .pred p, q;\n.reg .b64 ar, ai, br, bi;\nsetp.eq.u32 p, %12, 0;\n@p bra.uni SKIP_%=;\n"
        "mov.b64 ar, {%4, %4};\nmov.b64 ai, {%5, %5};\nmov.b64 br, {%6, %6};\nmov.b64 bi, {%7, %7};\n"
        "fma.rn.f32x2 %0, ar, %8, %0;\nfma.rn.f32x2 %1, ar, %10, %1;\n"
        "fma.rn.f32x2 %2, br, %8, %2;\nfma.rn.f32x2 %3, br, %10, %3;\n"
        "fma.rn.f32x2 %0, ai, %9, %0;\nfma.rn.f32x2 %1, ai, %11, %1;\n"
        "fma.rn.f32x2 %2, bi, %9, %2;\nfma.rn.f32x2 %3, bi, %11, %3;\n"
        "SKIP_%=:\nsetp.ne.u32 q, %15, 0;\n"
        "@q ld.shared.v2.b32 {%4, %5}, [%13+%14];\n@q ld.shared.v2.b32 {%6, %7}, [%13+%14+256];\n}"
        : "+l"(acc[0][0]), "+l"(acc[0][1]), "+l"(acc[1][0]), "+l"(acc[1][1]), "+r"(t.v[0]), "+r"(t.v[1]), "+r"(t.v[2]), "+r"(t.v[3])
        : "l"(V[0]), "l"(W[0]), "l"(V[1]), "l"(W[1]), "r"(on), "r"(addr), "n"(IMM), "r"(on_next));
  }
  if constexpr (NG == 3) {
    asm volatile(
        "{\n.reg .pred p, q;\n.reg .b64 ar, ai, br, bi;\nsetp.eq.u32 p, %16, 0;\n@p bra.uni SKIP_%=;\n"
        "mov.b64 ar, {%6, %6};\nmov.b64 ai, {%7, %7};\nmov.b64 br, {%8, %8};\nmov.b64 bi, {%9, %9};\n"
        "fma.rn.f32x2 %0, ar, %10, %0;\nfma.rn.f32x2 %1, ar, %12, %1;\n"
        "fma.rn.f32x2 %2, ar, %14, %2;\nfma.rn.f32x2 %3, br, %10, %3;\n"
        "fma.rn.f32x2 %4, br, %12, %4;\nfma.rn.f32x2 %5, br, %14, %5;\n"
        "fma.rn.f32x2 %0, ai, %11, %0;\nfma.rn.f32x2 %1, ai, %13, %1;\n"
        "fma.rn.f32x2 %2, ai, %15, %2;\nfma.rn.f32x2 %3, bi, %11, %3;\n"
        "fma.rn.f32x2 %4, bi, %13, %4;\nfma.rn.f32x2 %5, bi, %15, %5;\n"
        "SKIP_%=:\nsetp.ne.u32 q, %19, 0;\n"
        "@q ld.shared.v2.b32 {%6, %7}, [%17+%18];\n@q ld.shared.v2.b32 {%8, %9}, [%17+%18+256];\n}"
        : "+l"(acc[0][0]), "+l"(acc[0][1]), "+l"(acc[0][2]), "+l"(acc[1][0]), "+l"(acc[1][1]), "+l"(acc[1][2]), "+r"(t.v[0]), "+r"(t.v[1]), "+r"(t.v[2]), "+r"(t.v[3])
        : "l"(V[0]), "l"(W[0]), "l"(V[1]), "l"(W[1]), "l"(V[2]), "l"(W[2]), "r"(on), "r"(addr), "n"(IMM), "r"(on_next));
  }
  if constexpr (NG == 4) {
    asm volatile(
        "{\n.reg .pred p, q;\n.reg .b64 ar, ai, br, bi;\nsetp.eq.u32 p, %20, 0;\n@p bra.uni SKIP_%=;\n"
        "mov.b64 ar, {%8, %8};\nmov.b64 ai, {%9, %9};\nmov.b64 br, {%10, %10};\nmov.b64 bi, {%11, %11};\n"
        "fma.rn.f32x2 %0, ar, %12, %0;\nfma.rn.f32x2 %1, ar, %14, %1;\n"
        "fma.rn.f32x2 %2, ar, %16, %2;\nfma.rn.f32x2 %3, ar, %18, %3;\n"
        "fma.rn.f32x2 %4, br, %12, %4;\nfma.rn.f32x2 %5, br, %14, %5;\n"
        "fma.rn.f32x2 %6, br, %16, %6;\nfma.rn.f32x2 %7, br, %18, %7;\n"
        "fma.rn.f32x2 %0, ai, %13, %0;\nfma.rn.f32x2 %1, ai, %15, %1;\n"
        "fma.rn.f32x2 %2, ai, %17, %2;\nfma.rn.f32x2 %3, ai, %19, %3;\n"
        "fma.rn.f32x2 %4, bi, %13, %4;\nfma.rn.f32x2 %5, bi, %15, %5;\n"
        "fma.rn.f32x2 %6, bi, %17, %6;\nfma.rn.f32x2 %7, bi, %19, %7;\n"
        "SKIP_%=:\nsetp.ne.u32 q, %23, 0;\n"
        "@q ld.shared.v2.b32 {%8, %9}, [%21+%22];\n@q ld.shared.v2.b32 {%10, %11}, [%21+%22+256];\n}"
        : "+l"(acc[0][0]), "+l"(acc[0][1]), "+l"(acc[0][2]), "+l"(acc[0][3]), "+l"(acc[1][0]), "+l"(acc[1][1]), "+l"(acc[1][2]), "+l"(acc[1][3]), "+r"(t.v[0]), "+r"(t.v[1]), "+r"(t.v[2]), "+r"(t.v[3])
        : "l"(V[0]), "l"(W[0]), "l"(V[1]), "l"(W[1]), "l"(V[2]), "l"(W[2]), "l"(V[3]), "l"(W[3]), "r"(on), "r"(addr), "n"(IMM), "r"(on_next));
  }
}

// Steps [B, KS) of a point, unrolled.
template <int NW, int NG, int KS, int B>
__device__ __forceinline__ void lra_run_steps(lra_u64 (&acc)[KS][2][NG], const lra_u64 (&V)[NG], const lra_u64 (&W)[NG],
                                              lra_taps (&T)[KS], uint32_t mask, uint32_t addr_next, uint32_t mask_next) {
  if constexpr (B < KS) {
    lra_step<NG, B * 512 * NW>(acc[B], V, W, T[B], mask & (1u << B), addr_next, mask_next & (1u << B));
    lra_run_steps<NW, NG, KS, B + 1>(acc, V, W, T, mask, addr_next, mask_next);
  }
}

template <int NW, int KS, int NG>
__global__ void __launch_bounds__((lra_cw(NW) + 1) * 32) __maxnreg__(LRA_MAXNREG(NW, KS, NG, false)) lra_grid_region_kernel(const lra_region_args a) {
  extern __shared__ __align__(128) unsigned char smem[];
  const int lane = threadIdx.x & 31;
  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);   // provably warp-uniform: uniform registers
  const uint32_t sbase = lra_smem_u32(smem);
  const uint32_t full0 = sbase, empty0 = sbase + 128, slots0 = sbase + LRA_RING_HDR;
  lra_region_ring_init<NW>(a, smem, full0, empty0);
  constexpr int PB = lra_point_bytes(NG);
  constexpr int PS = NW == 1 ? LRA_PS_WARPS : 1;   // point-split warps (lra_cw in lra_pipe.cuh)
  const int pwarp = PS > 1 ? 0 : warp;             // which chunks of the region this warp owns
  const unsigned first = PS > 1 ? (unsigned)warp : 0u;   // its first point of a batch
  if (warp == lra_cw(NW)) {
    lra_region_producer<NW, 0>(a, a.prep, PB, smem + LRA_RING_HDR, full0, empty0, slots0);
    return;
  }
  // -------------------------------------------------------------------- consumer warps
  lra_u64 acc[KS][2][NG];
#pragma unroll
  for (int s = 0; s < KS; ++s)
#pragma unroll
    for (int g = 0; g < NG; ++g) acc[s][0][g] = acc[s][1][g] = 0ull;
  lra_taps T[KS];
#pragma unroll
  for (int s = 0; s < KS; ++s) T[s].v[0] = T[s].v[1] = T[s].v[2] = T[s].v[3] = 0u;
  uint32_t slot = 0, par = 0;
  const uint32_t lane_off = (uint32_t)a.slab0 + 8u * (64u * pwarp + lane);
  for (;;) {
    lra_mbar_wait(full0 + 8 * slot, par);
    const unsigned char* sp = smem + LRA_RING_HDR + (size_t)slot * a.slot_bytes;
    const uint4 h = *reinterpret_cast<const uint4*>(sp);
    const unsigned count = h.y & 0xff;
    const uint32_t lane_base = slots0 + slot * a.slot_bytes + lane_off;
    const unsigned char* rec = sp + LRA_SLOT_VAL + first * PB;
    // software pipeline over the points of the batch: while a step multiplies the taps of point q it reloads its tap
    // registers for point q + 1; the record of point q + 1 is read while point q runs
    // (the record's tail is {word, z, w, 0}: 8 bytes are enough up to four consumer warps)
    using tail_t = typename std::conditional<(NW <= 4), uint2, uint4>::type;
    auto tail_w = [](const tail_t& t) { if constexpr (NW <= 4) return 0u; else return t.z; };
    tail_t wc = *reinterpret_cast<const tail_t*>(rec + 16 * NG);
    uint32_t mask = first < count ? lra_point_mask<NW>(wc.y, tail_w(wc), pwarp) : 0u;
    lra_load_steps<NW, KS, 0>(T, lane_base + wc.x, mask);
    for (unsigned q = first; q < count; q += PS) {
      lra_u64 V[NG], W[NG];
#pragma unroll
      for (int g = 0; g < NG; ++g) {
        const ulonglong2 v = *reinterpret_cast<const ulonglong2*>(rec + 16 * g);
        V[g] = v.x; W[g] = v.y;
      }
      rec += PS * PB;
      wc = *reinterpret_cast<const tail_t*>(rec + 16 * NG);
      const uint32_t addr_next = lane_base + wc.x, mask_next = q + PS < count ? lra_point_mask<NW>(wc.y, tail_w(wc), pwarp) : 0u;
      lra_run_steps<NW, NG, KS, 0>(acc, V, W, T, mask, addr_next, lra_opaque(mask_next));
      mask = mask_next;
    }
    lra_mbar_arrive(empty0 + 8 * slot);   // every lane, after its own reads of the slot: no divergent branch in the loop
    if (h.y & LRA_BATCH_LAST) {
      // ---- row a4: add the item's region to the grid, once ----
      const int hh = (a.S - 1) >> 1;
      const int ty = (int)(h.w / (unsigned)a.ntx), tx = (int)(h.w - (unsigned)ty * a.ntx);
      const int x0 = tx * a.tile_x - hh, y0 = ty * a.tile_y - hh;
      const unsigned magic = 0xffffffffu / (unsigned)a.rx + 1u;
      if (lra_fast_flush(NW, KS, NG) && x0 >= 0 && y0 >= 0 && x0 + a.rx <= a.nx && y0 + a.ry <= a.ny) {
        // the region lies inside the grid (all tiles but those along its edges): no per-pixel bounds tests, one address per
        // pixel, the reductions predicated instead of branched around
        float2* const g00 = a.grid + ((ptrdiff_t)y0 * a.nx + x0);
        const unsigned npix = (unsigned)(a.rx * a.ry);
#pragma unroll
        for (int s = 0; s < KS; ++s) {
#pragma unroll
          for (int half = 0; half < 2; ++half) {
            const unsigned e = 64u * (NW * s + pwarp) + 32u * half + lane;
            const int y = (int)__umulhi(e, magic), x = (int)e - y * a.rx;
            float2* const px = g00 + (y * a.nx + x);
#pragma unroll
            for (int g = 0; g < NG; ++g) {
              lra_red_add_v2_nz(px + (size_t)g * a.plane, acc[s][half][g], e, npix);
              acc[s][half][g] = 0ull;
            }
          }
        }
      } else
#pragma unroll
      for (int s = 0; s < KS; ++s) {
#pragma unroll
        for (int half = 0; half < 2; ++half) {
          const unsigned e = 64u * (NW * s + pwarp) + 32u * half + lane;
          const int y = (int)__umulhi(e, magic), x = (int)e - y * a.rx;
          const int gx = x0 + x, gy = y0 + y;
          const bool ok = y < a.ry && gx >= 0 && gx < a.nx && gy >= 0 && gy < a.ny;
#pragma unroll
          for (int g = 0; g < NG; ++g) {
            float vr, vi;
            lra_unpack2(acc[s][half][g], vr, vi);
            if (ok && (vr != 0.f || vi != 0.f)) lra_red_add_v2(a.grid + (size_t)g * a.plane + (size_t)gy * a.nx + gx, vr, vi);
            acc[s][half][g] = 0ull;
          }
        }
      }
    }
    if (h.y & LRA_BATCH_END) break;
    if (++slot == (uint32_t)a.nslot) { slot = 0; par ^= 1; }
  }
}

// ---------------------------------------------------------------------------------------------------
template <int NW, int KS, int NG>
static int lra_grid_launch_class(lra_plan* p, lra_region_args a, const lra_geom& q, int c, cudaStream_t st) {
  int smem = 0;
  if (!lra_region_ring(q, lra_grids_per_pass(p->ncorr * p->nterms), false, lra_point_bytes(NG), &a, &smem)) return LRA_EINVAL;
  auto kern = lra_grid_region_kernel<NW, KS, NG>;
  static int attr_smem[LRA_MAX_DEVICES];   // per instantiation and device: the opt-in is made once, not per launch
  if (p->device < 0 || p->device >= LRA_MAX_DEVICES || attr_smem[p->device] < smem) {
    LRA_CUDA(p, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    if (p->device >= 0 && p->device < LRA_MAX_DEVICES) attr_smem[p->device] = smem;
  }
  a.work = p->work + p->item_off[c];
  a.n_items = (unsigned)p->n_items[c];
  a.batch = reinterpret_cast<const uint4*>(p->batch) + (size_t)p->batch_off[c] * 4;
  int ctas = p->sm_count * lra_ctas_per_sm(NW, KS, lra_grids_per_pass(p->ncorr * p->nterms), false);   // what the ring was sized for
  if ((int64_t)ctas > p->n_items[c]) ctas = (int)p->n_items[c];
  kern<<<ctas, (lra_cw(NW) + 1) * 32, smem, st>>>(a);
  LRA_LAUNCH_CHECK(p);
  return LRA_OK;
}

template <int NW, int NG>
static int lra_grid_launch_ks(lra_plan* p, const lra_region_args& a, const lra_geom& q, int c, cudaStream_t st) {
  // the (NW, KS) of a class come from the plan's grids per pass; a remainder pass of fewer grids runs the same steps
  switch (q.ks) {
    case 1: return lra_grid_launch_class<NW, 1, NG>(p, a, q, c, st);
    case 2: return lra_grid_launch_class<NW, 2, NG>(p, a, q, c, st);
    case 3: return lra_grid_launch_class<NW, 3, NG>(p, a, q, c, st);
    case 4: return lra_grid_launch_class<NW, 4, NG>(p, a, q, c, st);
    default: break;
  }
  if constexpr (NG <= 2) {
    if (q.ks == 5) return lra_grid_launch_class<NW, 5, NG>(p, a, q, c, st);
    if (q.ks == 6) return lra_grid_launch_class<NW, 6, NG>(p, a, q, c, st);
  }
  if constexpr (NG == 1) {
    if (q.ks == 8) return lra_grid_launch_class<NW, 8, NG>(p, a, q, c, st);
  }
  return LRA_EINVAL;
}

// One launch: the items of support class c, NG grids starting at a.grid.
template <int NG>
int lra_grid_launch_ng(lra_plan* p, const lra_region_args& a, const lra_geom& q, int c, cudaStream_t st) {
  switch (q.nw) {
    case 1: return lra_grid_launch_ks<1, NG>(p, a, q, c, st);
    case 2: return lra_grid_launch_ks<2, NG>(p, a, q, c, st);
    case 4: return lra_grid_launch_ks<4, NG>(p, a, q, c, st);
    case 8: return lra_grid_launch_ks<8, NG>(p, a, q, c, st);
    case 16: return lra_grid_launch_ks<16, NG>(p, a, q, c, st);
    default: return LRA_EINVAL;
  }
}

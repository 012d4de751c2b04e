// lra_degrid_region.cuh -- the default degridder (variant 0): the adjoint of lra_grid_region.cuh with the data flow
// turned round.  Kernel template and its launch dispatch; instantiated per number of grids in
// lra_degrid_region_ng*.cu, driven by lra_degrid_region.cu.
//
// Operation: Eq. 6 of arxiv 2508.17187, D(c_ij) read as the exact adjoint of G (reading R7), row a5
// of SURVEY Sec. 8(a):  V[k][p] = sum_t tau[c][t] * sum_{j,i} conj(CF[j][i]) * grid[t][p][iy+j][ix+i].
//
// Design: same items, batches, CF slab ring, producer warp, chunk ownership and step masks as the gridder
// (lra_region.cuh, lra_work.cu).  A CTA loads the item's region of the MODEL grid into registers once (the grid tile
// is read once per item), pixel e of the region as one (re, im) register pair per grid in the lane that owns it.  For
// every point a lane forms, over its pixels inside the point's chunk range,
//     P1 += cre * (Gre, Gim),   P2 += cim * (Gre, Gim)          (two FFMA2 per pixel and grid, the tap as the scalar)
// and conj(c) * G summed over the pixels is (P1.re + P2.im, P1.im - P2.re).  That leaves 32 partial sums per value in
// a warp.  Four points at a time, the 4 x NG complex partials are reduced across the lanes with a transposing shuffle
// butterfly (one shuffle per value instead of five), added across the consumer warps with shared-memory atomics into
// the slot, and written out by the producer warp, in sorted order, when the slot is recycled.
// lra_degrid_finish_kernel then applies the Taylor weights, the fused residual of Eq. 23 and the sorted -> caller
// order scatter.
#pragma once
#include "lra_region.cuh"

// One step of the software pipeline: the FMAs of the CURRENT point on the two pixels this lane owns at the step (taps
// t = {re(e), im(e), re(e + 32), im(e + 32)}), under a uniform branch on `on`, then the loads of the NEXT point's taps
// for the same step into the same registers.
template <int NG, int IMM>
__device__ __forceinline__ void lra_dstep(lra_u64 (&P1)[NG], lra_u64 (&P2)[NG], const lra_u64 (&G)[2][NG], lra_taps& t,
                                          uint32_t on, uint32_t addr, uint32_t on_next) {
  if constexpr (NG == 1) {
    asm volatile(
        "{\n.reg .pred p, q;\n.reg .b64 ar, ai, br, bi;\nsetp.eq.u32 p, %8, 0;\n@p bra.uni SKIP_%=;\n"
        "mov.b64 ar, {%2, %2};\nmov.b64 ai, {%3, %3};\nmov.b64 br, {%4, %4};\nmov.b64 bi, {%5, %5};\n"
        "fma.rn.f32x2 %0, ar, %6, %0;\nfma.rn.f32x2 %1, ai, %6, %1;\n"
        "fma.rn.f32x2 %0, br, %7, %0;\nfma.rn.f32x2 %1, bi, %7, %1;\n"
        "SKIP_%=:\nsetp.ne.u32 q, %11, 0;\n"
        "@q ld.shared.v2.b32 {%2, %3}, [%9+%10];\n@q ld.shared.v2.b32 {%4, %5}, [%9+%10+256];\n}"
        : "+l"(P1[0]), "+l"(P2[0]), "+r"(t.v[0]), "+r"(t.v[1]), "+r"(t.v[2]), "+r"(t.v[3])
        : "l"(G[0][0]), "l"(G[1][0]), "r"(on), "r"(addr), "n"(IMM), "r"(on_next));
  }
  if constexpr (NG == 2) {
    asm volatile(
        "{\n.reg .pred p, q;\n.reg .b64 ar, ai, br, bi;\nsetp.eq.u32 p, %12, 0;\n@p bra.uni SKIP_%=;\n"
        "mov.b64 ar, {%4, %4};\nmov.b64 ai, {%5, %5};\nmov.b64 br, {%6, %6};\nmov.b64 bi, {%7, %7};\n"
        "fma.rn.f32x2 %0, ar, %8, %0;\nfma.rn.f32x2 %2, ai, %8, %2;\n"
        "fma.rn.f32x2 %1, ar, %9, %1;\nfma.rn.f32x2 %3, ai, %9, %3;\n"
        "fma.rn.f32x2 %0, br, %10, %0;\nfma.rn.f32x2 %2, bi, %10, %2;\n"
        "fma.rn.f32x2 %1, br, %11, %1;\nfma.rn.f32x2 %3, bi, %11, %3;\n"
        "SKIP_%=:\nsetp.ne.u32 q, %15, 0;\n"
        "@q ld.shared.v2.b32 {%4, %5}, [%13+%14];\n@q ld.shared.v2.b32 {%6, %7}, [%13+%14+256];\n}"
        : "+l"(P1[0]), "+l"(P1[1]), "+l"(P2[0]), "+l"(P2[1]), "+r"(t.v[0]), "+r"(t.v[1]), "+r"(t.v[2]), "+r"(t.v[3])
        : "l"(G[0][0]), "l"(G[0][1]), "l"(G[1][0]), "l"(G[1][1]), "r"(on), "r"(addr), "n"(IMM), "r"(on_next));
  }
  if constexpr (NG == 3) {
    asm volatile(
        "{\n.reg .pred p, q;\n.reg .b64 ar, ai, br, bi;\nsetp.eq.u32 p, %16, 0;\n@p bra.uni SKIP_%=;\n"
        "mov.b64 ar, {%6, %6};\nmov.b64 ai, {%7, %7};\nmov.b64 br, {%8, %8};\nmov.b64 bi, {%9, %9};\n"
        "fma.rn.f32x2 %0, ar, %10, %0;\nfma.rn.f32x2 %3, ai, %10, %3;\n"
        "fma.rn.f32x2 %1, ar, %11, %1;\nfma.rn.f32x2 %4, ai, %11, %4;\n"
        "fma.rn.f32x2 %2, ar, %12, %2;\nfma.rn.f32x2 %5, ai, %12, %5;\n"
        "fma.rn.f32x2 %0, br, %13, %0;\nfma.rn.f32x2 %3, bi, %13, %3;\n"
        "fma.rn.f32x2 %1, br, %14, %1;\nfma.rn.f32x2 %4, bi, %14, %4;\n"
        "fma.rn.f32x2 %2, br, %15, %2;\nfma.rn.f32x2 %5, bi, %15, %5;\n"
        "SKIP_%=:\nsetp.ne.u32 q, %19, 0;\n"
        "@q ld.shared.v2.b32 {%6, %7}, [%17+%18];\n@q ld.shared.v2.b32 {%8, %9}, [%17+%18+256];\n}"
        : "+l"(P1[0]), "+l"(P1[1]), "+l"(P1[2]), "+l"(P2[0]), "+l"(P2[1]), "+l"(P2[2]), "+r"(t.v[0]), "+r"(t.v[1]), "+r"(t.v[2]), "+r"(t.v[3])
        : "l"(G[0][0]), "l"(G[0][1]), "l"(G[0][2]), "l"(G[1][0]), "l"(G[1][1]), "l"(G[1][2]), "r"(on), "r"(addr), "n"(IMM), "r"(on_next));
  }
  if constexpr (NG == 4) {
    asm volatile(
        "{\n.reg .pred p, q;\n.reg .b64 ar, ai, br, bi;\nsetp.eq.u32 p, %20, 0;\n@p bra.uni SKIP_%=;\n"
        "mov.b64 ar, {%8, %8};\nmov.b64 ai, {%9, %9};\nmov.b64 br, {%10, %10};\nmov.b64 bi, {%11, %11};\n"
        "fma.rn.f32x2 %0, ar, %12, %0;\nfma.rn.f32x2 %4, ai, %12, %4;\n"
        "fma.rn.f32x2 %1, ar, %13, %1;\nfma.rn.f32x2 %5, ai, %13, %5;\n"
        "fma.rn.f32x2 %2, ar, %14, %2;\nfma.rn.f32x2 %6, ai, %14, %6;\n"
        "fma.rn.f32x2 %3, ar, %15, %3;\nfma.rn.f32x2 %7, ai, %15, %7;\n"
        "fma.rn.f32x2 %0, br, %16, %0;\nfma.rn.f32x2 %4, bi, %16, %4;\n"
        "fma.rn.f32x2 %1, br, %17, %1;\nfma.rn.f32x2 %5, bi, %17, %5;\n"
        "fma.rn.f32x2 %2, br, %18, %2;\nfma.rn.f32x2 %6, bi, %18, %6;\n"
        "fma.rn.f32x2 %3, br, %19, %3;\nfma.rn.f32x2 %7, bi, %19, %7;\n"
        "SKIP_%=:\nsetp.ne.u32 q, %23, 0;\n"
        "@q ld.shared.v2.b32 {%8, %9}, [%21+%22];\n@q ld.shared.v2.b32 {%10, %11}, [%21+%22+256];\n}"
        : "+l"(P1[0]), "+l"(P1[1]), "+l"(P1[2]), "+l"(P1[3]), "+l"(P2[0]), "+l"(P2[1]), "+l"(P2[2]), "+l"(P2[3]), "+r"(t.v[0]), "+r"(t.v[1]), "+r"(t.v[2]), "+r"(t.v[3])
        : "l"(G[0][0]), "l"(G[0][1]), "l"(G[0][2]), "l"(G[0][3]), "l"(G[1][0]), "l"(G[1][1]), "l"(G[1][2]), "l"(G[1][3]), "r"(on), "r"(addr), "n"(IMM), "r"(on_next));
  }
}

template <int NW, int NG, int KS, int B>
__device__ __forceinline__ void lra_drun_steps(lra_u64 (&P1)[NG], lra_u64 (&P2)[NG], const lra_u64 (&G)[KS][2][NG],
                                               lra_taps (&T)[KS], uint32_t mask, uint32_t addr_next, uint32_t mask_next) {
  if constexpr (B < KS) {
    lra_dstep<NG, B * 512 * NW>(P1, P2, G[B], T[B], mask & (1u << B), addr_next, mask_next & (1u << B));
    lra_drun_steps<NW, NG, KS, B + 1>(P1, P2, G, T, mask, addr_next, mask_next);
  }
}

template <int NW, int KS, int NG>
__global__ void __launch_bounds__((lra_cw(NW) + 1) * 32) __maxnreg__(LRA_MAXNREG(NW, KS, NG, true)) lra_degrid_region_kernel(const lra_region_args a) {
  extern __shared__ __align__(128) unsigned char smem[];
  const int lane = threadIdx.x & 31;
  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);   // provably warp-uniform: uniform registers
  const uint32_t sbase = lra_smem_u32(smem);
  const uint32_t full0 = sbase, empty0 = sbase + 128, slots0 = sbase + LRA_RING_HDR;
  lra_region_ring_init<NW>(a, smem, full0, empty0);
  constexpr int PS = NW == 1 ? LRA_PS_WARPS : 1;   // point-split warps (lra_cw in lra_pipe.cuh)
  const int pwarp = PS > 1 ? 0 : warp;             // which chunks of the region this warp owns
  const unsigned first = PS > 1 ? (unsigned)warp : 0u;   // its first point of a batch
  if (warp == lra_cw(NW)) {
    lra_region_producer<NW, NG>(a, a.prep, 16, smem + LRA_RING_HDR, full0, empty0, slots0);
    return;
  }
  // -------------------------------------------------------------------- consumer warps
  constexpr int V = NG == 1 ? 8 : NG == 2 ? 16 : 32;   // values of four points (2 * NG each), padded to a power of two
  lra_u64 G[KS][2][NG];   // the region of the model grid: (re, im) of the lane's two pixels at every step
  lra_taps T[KS];
#pragma unroll
  for (int s = 0; s < KS; ++s) T[s].v[0] = T[s].v[1] = T[s].v[2] = T[s].v[3] = 0u;
  bool fresh = true;
  uint32_t slot = 0, par = 0;
  const uint32_t lane_off = (uint32_t)a.slab0 + 8u * (64u * pwarp + lane);
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
      if (NG <= 2 && x0 >= 0 && y0 >= 0 && x0 + a.rx <= a.nx && y0 + a.ry <= a.ny) {
        // the region lies inside the grid (all tiles but those along its edges): no per-pixel bounds tests, one address per pixel
        // (one or two grids; with four the second code path costs more than it saves: cfg4 43.95 -> 44.33 ms)
        const float2* const g00 = a.grid + ((ptrdiff_t)y0 * a.nx + x0);
        const unsigned npix = (unsigned)(a.rx * a.ry);
#pragma unroll
        for (int s = 0; s < KS; ++s) {
#pragma unroll
          for (int half = 0; half < 2; ++half) {
            const unsigned e = 64u * (NW * s + pwarp) + 32u * half + lane;
            const int y = (int)__umulhi(e, magic), x = (int)e - y * a.rx;
            const float2* const px = g00 + (y * a.nx + x);
#pragma unroll
            for (int g = 0; g < NG; ++g) {
              const float2 v = e < npix ? px[(size_t)g * a.plane] : make_float2(0.f, 0.f);
              G[s][half][g] = lra_pack2(v.x, v.y);
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
            const float2 v = ok ? a.grid[(size_t)g * a.plane + (size_t)gy * a.nx + gx] : make_float2(0.f, 0.f);
            G[s][half][g] = lra_pack2(v.x, v.y);
          }
        }
      }
      fresh = false;
    }
    const uint32_t lane_base = slots0 + slot * a.slot_bytes + lane_off;
    const unsigned char* rec = sp + LRA_SLOT_VAL + 16 * first;   // 16 bytes per point: the pw record {word, k, z, w} (lra_pipe.cuh)
    float* out = reinterpret_cast<float*>(sp + a.out_off);
    // software pipeline over the points of the batch (as in the gridder), four points per reduction
    uint4 pc = *reinterpret_cast<const uint4*>(rec);
    uint32_t mask = first < count ? lra_point_mask<NW>(pc.z, pc.w, pwarp) : 0u;
    lra_load_steps<NW, KS, 0>(T, lane_base + pc.x, mask);
    // Two releases per slot: its taps and records once this warp has loaded the last of them (the producer may then start
    // the copies of the slot's next batch), its results at the end of the batch.
    if (first >= count) lra_mbar_arrive(empty0 + 8 * slot);
    const uint32_t bar_taps = empty0 + 8 * slot;
    for (unsigned q0 = first; q0 < count; q0 += 4 * PS) {   // this warp's points q0, q0 + PS, q0 + 2 PS, q0 + 3 PS
      float v[V];
#pragma unroll
      for (int i = 0; i < V; ++i) v[i] = 0.f;
      // index in this group of the warp's last point of the batch (>= 4: a later group).  One comparison per point against it
      // is the cheaper form of the two tail conditions for one or two grids (cfg3 degridder 26.88 -> 26.67 ms); with three or
      // four grids the plain conditions are (cfg4 44.88 -> 43.98 ms)
      const unsigned last_u = (count - 1u - q0) / PS;
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        rec += 16 * PS;
        pc = *reinterpret_cast<const uint4*>(rec);
        const uint32_t addr_next = lane_base + pc.x, mask_next = (NG <= 2 ? (unsigned)u < last_u : q0 + (u + 1) * PS < count) ? lra_point_mask<NW>(pc.z, pc.w, pwarp) : 0u;
        // the warp's last point of the batch: its taps were loaded during the point before (the arrival is ordered
        // after those loads), nothing of the slot but the result area is touched from here on
        lra_mbar_arrive_if(bar_taps, NG <= 2 ? last_u == (unsigned)u : (q0 + u * PS < count && q0 + (u + 1) * PS >= count));
        lra_u64 P1[NG], P2[NG];
#pragma unroll
        for (int g = 0; g < NG; ++g) P1[g] = P2[g] = 0ull;
        lra_drun_steps<NW, NG, KS, 0>(P1, P2, G, T, mask, addr_next, lra_opaque(mask_next));
#pragma unroll
        for (int g = 0; g < NG; ++g) {   // conj(c) * G = (cre*Gre + cim*Gim) + i (cre*Gim - cim*Gre)
          float p1r, p1i, p2r, p2i;
          lra_unpack2(P1[g], p1r, p1i);
          lra_unpack2(P2[g], p2r, p2i);
          v[(u * NG + g) * 2 + 0] = p1r + p2i;
          v[(u * NG + g) * 2 + 1] = p1i - p2r;
        }
        mask = mask_next;
      }
      // transposing butterfly: afterwards lane l holds the warp total of value l % V
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
      const unsigned pt = q0 + (unsigned)(lane / (2 * NG)) * PS;   // the point whose value this lane holds
      if (lane < 8 * NG && pt < count) atomicAdd(out + pt * (2 * NG) + lane % (2 * NG), v[0]);
    }
    lra_mbar_arrive(empty0 + LRA_EMPTY_OUT + 8 * slot);   // every lane (no divergent branch in the loop): the results are complete
    if (h.y & LRA_BATCH_LAST) fresh = true;
    if (h.y & LRA_BATCH_END) break;
    if (++slot == (uint32_t)a.nslot) { slot = 0; par ^= 1; }
  }
}

// ---------------------------------------------------------------------------------------------------
template <int NW, int KS, int NG>
static int lra_degrid_launch_class(lra_plan* p, lra_region_args a, const lra_geom& q, int c, cudaStream_t st) {
  int smem = 0;
  if (!lra_region_ring(q, lra_grids_per_pass(p->ncorr * p->nterms), true, 16 + 8 * NG, &a, &smem)) return LRA_EINVAL;
  auto kern = lra_degrid_region_kernel<NW, KS, NG>;
  static int attr_smem[LRA_MAX_DEVICES];   // per instantiation and device: the opt-in is made once, not per launch
  if (p->device < 0 || p->device >= LRA_MAX_DEVICES || attr_smem[p->device] < smem) {
    LRA_CUDA(p, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    if (p->device >= 0 && p->device < LRA_MAX_DEVICES) attr_smem[p->device] = smem;
  }
  a.work = p->work + p->item_off[c];
  a.n_items = (unsigned)p->n_items[c];
  a.batch = reinterpret_cast<const uint4*>(p->batch) + (size_t)p->batch_off[c] * 4;
  int ctas = p->sm_count * lra_ctas_per_sm(NW, KS, lra_grids_per_pass(p->ncorr * p->nterms), true);   // what the ring was sized for
  if ((int64_t)ctas > p->n_items[c]) ctas = (int)p->n_items[c];
  kern<<<ctas, (lra_cw(NW) + 1) * 32, smem, st>>>(a);
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
    default: break;
  }
  if constexpr (NG <= 2) {
    if (q.ks == 5) return lra_degrid_launch_class<NW, 5, NG>(p, a, q, c, st);
    if (q.ks == 6) return lra_degrid_launch_class<NW, 6, NG>(p, a, q, c, st);
  }
  if constexpr (NG == 1) {
    if (q.ks == 8) return lra_degrid_launch_class<NW, 8, NG>(p, a, q, c, st);
  }
  return LRA_EINVAL;
}

// One launch: the items of support class c, NG grids starting at a.grid.
template <int NG>
int lra_degrid_launch_ng(lra_plan* p, const lra_region_args& a, const lra_geom& q, int c, cudaStream_t st) {
  switch (q.nw) {
    case 1: return lra_degrid_launch_ks<1, NG>(p, a, q, c, st);
    case 2: return lra_degrid_launch_ks<2, NG>(p, a, q, c, st);
    case 4: return lra_degrid_launch_ks<4, NG>(p, a, q, c, st);
    case 8: return lra_degrid_launch_ks<8, NG>(p, a, q, c, st);
    case 16: return lra_degrid_launch_ks<16, NG>(p, a, q, c, st);
    default: return LRA_EINVAL;
  }
}

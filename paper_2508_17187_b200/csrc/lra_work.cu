// lra_work.cu -- item list, stage stream and per-point words for the strip gridder / degridder, built at the end of
// lra_bin (they depend on the geometry only and are reused by every lra_grid / lra_degrid call until the next
// lra_bin).  Part of "re-ordering for runtime performance": the sorted order itself is the
// bit-exact contract of lra_bin; this file only says how that order is cut into pieces for the CTAs.
// Formats: lra_pipe.cuh.
#include "lra_pipe.cuh"

struct lra_work_args {
  const lra_rec* rec;
  unsigned long long* counters;
  int shift_x, shift_y, ntx, tile_x, tile_y;
  uint4* work;
  uint4* stage_hdr;
};

// exclusive prefix sum over the block (256 threads); returns the block total through `total`
__device__ __forceinline__ unsigned lra_block_excl_sum(unsigned v, unsigned* warp_buf, unsigned& total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  unsigned incl = v;
  for (int o = 1; o < 32; o <<= 1) {
    const unsigned y = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += y;
  }
  __syncthreads();
  if (lane == 31) warp_buf[warp] = incl;
  __syncthreads();
  unsigned base = 0;
  total = 0;
  for (int w = 0; w < 8; ++w) { if (w < warp) base += warp_buf[w]; total += warp_buf[w]; }
  return base + incl - v;
}
// running maximum over the block of a per-thread value (int, -1 = none), exclusive of the own thread
__device__ __forceinline__ int lra_block_excl_max(int v, int* warp_buf) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int incl = v;
  for (int o = 1; o < 32; o <<= 1) {
    const int y = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl = max(incl, y);
  }
  __syncthreads();
  if (lane == 31) warp_buf[warp] = incl;
  __syncthreads();
  int base = -1;
  for (int w = 0; w < warp; ++w) base = max(base, warp_buf[w]);
  int excl = __shfl_up_sync(0xffffffffu, incl, 1);
  if (lane == 0) excl = -1;
  return max(base, excl);
}

// One block per chunk of LRA_CHUNK sorted positions, 4 positions per thread.  FILL = false counts the items and
// stages of every group; FILL = true writes them (group offsets are in counters[40..55] by then).
template <bool FILL>
__global__ void __launch_bounds__(256) lra_work_kernel(const lra_work_args a) {
  const long long n = (long long)a.counters[0];
  const long long lo = (long long)blockIdx.x * LRA_CHUNK;
  if (lo >= n) return;
  const long long hi = lo + LRA_CHUNK < n ? lo + LRA_CHUNK : n;
  __shared__ unsigned warp_buf[8];
  __shared__ int warp_buf_i[8];
  __shared__ unsigned grp_cnt[2][8];
  __shared__ unsigned item_pos[LRA_CHUNK], item_first_stage[LRA_CHUNK + 1], item_base[LRA_CHUNK], stage_pos[LRA_CHUNK + 1];
  __shared__ unsigned short stage_item[LRA_CHUNK];
  __shared__ unsigned char item_grp[LRA_CHUNK];
  if (threadIdx.x < 16) grp_cnt[threadIdx.x >> 3][threadIdx.x & 7] = 0;
  // ---- flags of the thread's 4 consecutive positions ----
  const long long i0 = lo + threadIdx.x * 4;
  unsigned item_f = 0, slab_f = 0, tl[4], gr[4];
  long long prev_t = -1;
  int prev_s = -1;
  unsigned prev_slab = 0xffffffffu;
  if (i0 > lo && i0 - 1 < hi) {
    const lra_rec r = a.rec[i0 - 1];
    prev_t = (long long)((r.x >> 16) >> a.shift_y) * a.ntx + ((r.x & 0xffff) >> a.shift_x);
    prev_s = (int)(r.w & 0xff);
    prev_slab = r.y;
  }
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    const long long i = i0 + e;
    tl[e] = 0; gr[e] = 0;
    if (i < hi) {
      const lra_rec r = a.rec[i];
      const long long t = (long long)((r.x >> 16) >> a.shift_y) * a.ntx + ((r.x & 0xffff) >> a.shift_x);
      const int s = (int)(r.w & 0xff);
      if (i == lo || t != prev_t || s != prev_s) item_f |= 1u << e;
      if ((item_f >> e & 1u) || r.y != prev_slab) slab_f |= 1u << e;
      tl[e] = (unsigned)t; gr[e] = (unsigned)lra_group_of(s, a.tile_x, a.tile_y);
      prev_t = t; prev_s = s; prev_slab = r.y;
    }
  }
  // ---- stage heads: slab heads plus a cut every LRA_RUNMAX points of a run ----
  int last_head = -1;   // chunk-relative position of the last slab head at or before the thread's positions
#pragma unroll
  for (int e = 0; e < 4; ++e)
    if (slab_f >> e & 1u) last_head = threadIdx.x * 4 + e;
  int run_head = lra_block_excl_max(last_head, warp_buf_i);
  unsigned stage_f = 0;
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    if (i0 + e >= hi) break;
    if (slab_f >> e & 1u) run_head = threadIdx.x * 4 + e;
    if (((threadIdx.x * 4 + e - run_head) & (LRA_RUNMAX - 1)) == 0) stage_f |= 1u << e;
  }
  unsigned n_items_blk, n_stages_blk;
  unsigned ir = lra_block_excl_sum(__popc(item_f), warp_buf, n_items_blk);
  unsigned sr = lra_block_excl_sum(__popc(stage_f), warp_buf, n_stages_blk);
  if (!FILL) {
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      if (item_f >> e & 1u) atomicAdd(&grp_cnt[0][gr[e]], 1u);
      if (stage_f >> e & 1u) atomicAdd(&grp_cnt[1][gr[e]], 1u);
    }
    __syncthreads();
    if (threadIdx.x < 16 && grp_cnt[threadIdx.x >> 3][threadIdx.x & 7])
      atomicAdd(&a.counters[8 + threadIdx.x], (unsigned long long)grp_cnt[threadIdx.x >> 3][threadIdx.x & 7]);
    return;
  }
  // ---- block-local lists ----
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    if (item_f >> e & 1u) {
      item_pos[ir] = tl[e];      // the item's tile id
      item_first_stage[ir] = sr;
      item_grp[ir] = (unsigned char)gr[e];
      ++ir;
    }
    if (stage_f >> e & 1u) {
      stage_pos[sr] = (unsigned)(i0 + e);
      stage_item[sr] = (unsigned short)(ir - 1);
      ++sr;
    }
  }
  if (threadIdx.x == 0) { item_first_stage[n_items_blk] = n_stages_blk; stage_pos[n_stages_blk] = (unsigned)hi; }
  __syncthreads();
  for (unsigned j = threadIdx.x; j < n_items_blk; j += 256) {
    const unsigned g = item_grp[j], first = item_first_stage[j], nst = item_first_stage[j + 1] - first;
    const unsigned base = (unsigned)atomicAdd(&a.counters[32 + g], (unsigned long long)nst);
    const unsigned long long idx = a.counters[40 + g] + atomicAdd(&a.counters[24 + g], 1ull);
    const unsigned S = a.rec[stage_pos[first]].w & 0xff;
    a.work[idx] = make_uint4(item_pos[j], base, nst, S);
    item_base[j] = base;
  }
  __syncthreads();
  for (unsigned j = threadIdx.x; j < n_stages_blk; j += 256) {
    const unsigned it = stage_item[j], g = item_grp[it];
    const unsigned pos = stage_pos[j], cnt = stage_pos[j + 1] - pos;
    const unsigned long long gidx = a.counters[48 + g] + item_base[it] + (j - item_first_stage[it]);
    const lra_rec r = a.rec[pos];
    const unsigned last = (j + 1 == item_first_stage[it + 1]) ? LRA_STAGE_LAST : 0u;
    a.stage_hdr[gidx] = make_uint4(pos, cnt | ((r.w & 0xff) << 8) | last, r.y, item_pos[it]);
  }
}

// pw words of every sorted position (format: lra_pipe.cuh).
__global__ void __launch_bounds__(256)
lra_point_words_kernel(const lra_rec* __restrict__ rec, const unsigned long long* __restrict__ counters, int shift_x,
                       int shift_y, int tile_x, int tile_y, uint4* __restrict__ pw) {
  const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i >= (long long)counters[0]) return;
  const lra_rec r = rec[i];
  const int S = r.w & 0xff, h = (S - 1) >> 1, ix = r.x & 0xffff, iy = r.x >> 16;
  const int rx = S + tile_x - 1;
  const int ox = ix - ((ix >> shift_x) << shift_x), oy = iy - ((iy >> shift_y) << shift_y);   // origin - (tile origin - h)
  (void)h;
  const int off = oy * rx + ox, len = (S - 1) * rx + S;     // footprint = linear pixels [off, off + len)
  const int g = lra_group_of(S, tile_x, tile_y);
  unsigned w16[LRA_PW_STRIDE];
#pragma unroll
  for (int w = 0; w < LRA_PW_STRIDE; ++w) w16[w] = 0;
  if (g < LRA_NGROUP - 1) {
    const int nw = lra_group_nw(g), ks = lra_group_ks(g);
#pragma unroll
    for (int w = 0; w < LRA_PW_STRIDE; ++w) {
      if (w >= nw) break;
      unsigned m = 0;
      for (int s = 0; s < ks; ++s) {
        const int a0 = 64 * (nw * s + w);
        if (a0 + 63 >= off && a0 < off + len) m |= 1u << s;
      }
      w16[w] = (unsigned)(4 * off) | (m << 16);
    }
  }
  uint4* dst = pw + (size_t)i * (LRA_PW_STRIDE / 4);
#pragma unroll
  for (int q = 0; q < LRA_PW_STRIDE / 4; ++q) dst[q] = make_uint4(w16[4 * q], w16[4 * q + 1], w16[4 * q + 2], w16[4 * q + 3]);
}

template <typename T>
static int lra_grow(lra_plan* p, T** ptr, int64_t* cap, int64_t need) {
  if (need <= *cap) return LRA_OK;
  if (*ptr) { cudaFree(*ptr); *ptr = nullptr; *cap = 0; }
  const int64_t want = need + need / 8 + 64;
  LRA_CUDA(p, cudaMalloc(ptr, (size_t)want * sizeof(T)));
  *cap = want;
  return LRA_OK;
}

int lra_build_work(lra_plan* p) {
  for (int g = 0; g < 8; ++g) { p->n_items[g] = 0; p->item_off[g] = 0; p->n_stages[g] = 0; p->stage_off[g] = 0; }
  const int64_t n = p->npoints;
  if (n == 0) return LRA_OK;
  lra_work_args a;
  a.rec = p->rec; a.counters = p->counters; a.ntx = p->ntx; a.tile_x = p->tile_x; a.tile_y = p->tile;
  a.work = nullptr; a.stage_hdr = nullptr;
  a.shift_x = a.shift_y = 0;
  while ((1 << a.shift_x) < p->tile_x) ++a.shift_x;
  while ((1 << a.shift_y) < p->tile) ++a.shift_y;
  const int blocks = (int)((n + LRA_CHUNK - 1) / LRA_CHUNK);
  int rc;
  // counters[8..63] were zeroed at the start of lra_bin
  lra_work_kernel<false><<<blocks, 256, 0, p->stream>>>(a);
  LRA_LAUNCH_CHECK(p);
  unsigned long long h[16], off[16];
  LRA_CUDA(p, cudaMemcpyAsync(h, p->counters + 8, sizeof h, cudaMemcpyDeviceToHost, p->stream));
  LRA_CUDA(p, cudaStreamSynchronize(p->stream));
  int64_t items = 0, stages = 0;
  for (int g = 0; g < 8; ++g) {
    p->n_items[g] = (int64_t)h[g];
    p->n_stages[g] = (int64_t)h[8 + g];
    p->item_off[g] = items;
    p->stage_off[g] = stages;
    off[g] = (unsigned long long)items;
    off[8 + g] = (unsigned long long)stages;
    items += p->n_items[g];
    stages += p->n_stages[g];
  }
  if ((rc = lra_grow(p, &p->work, &p->work_capacity, items))) return rc;
  if ((rc = lra_grow(p, &p->stage_hdr, &p->stage_capacity, stages))) return rc;
  int64_t pw_words = p->pw_capacity * LRA_PW_STRIDE;
  if ((rc = lra_grow(p, &p->pw, &pw_words, n * LRA_PW_STRIDE))) return rc;
  p->pw_capacity = pw_words / LRA_PW_STRIDE;
  LRA_CUDA(p, cudaMemcpyAsync(p->counters + 40, off, sizeof off, cudaMemcpyHostToDevice, p->stream));
  a.work = p->work; a.stage_hdr = p->stage_hdr;
  lra_work_kernel<true><<<blocks, 256, 0, p->stream>>>(a);
  LRA_LAUNCH_CHECK(p);
  lra_point_words_kernel<<<(int)((n + 255) / 256), 256, 0, p->stream>>>(p->rec, p->counters, a.shift_x, a.shift_y, p->tile_x,
                                                                       p->tile, (uint4*)p->pw);
  LRA_LAUNCH_CHECK(p);
  LRA_CUDA(p, cudaStreamSynchronize(p->stream));  // `off` is stack-owned
  return LRA_OK;
}

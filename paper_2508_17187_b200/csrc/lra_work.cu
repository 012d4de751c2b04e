// lra_work.cu -- item list, batch stream and per-point words for the region gridder / degridder, built at the end of
// lra_bin (they depend on the geometry only and are reused by every lra_grid / lra_degrid call until the next
// lra_bin).  Part of "re-ordering for runtime performance": the sorted order itself is the
// bit-exact contract of lra_bin; this file only says how that order is cut into pieces for the CTAs.
// Formats: lra_pipe.cuh.
#include "lra_pipe.cuh"

struct lra_work_args {
  const lra_rec* rec;
  unsigned long long* counters;
  int shift_x, shift_y, ntx, tile_x, tile_y, ng;
  uint4* work;
  uint32_t* batch;     // 16 words per batch
  uint4* pw;           // one 16-byte record per sorted position: {word, k | fallback << 31, masks / chunk range}
  unsigned item_off[LRA_NCLASS], batch_off[LRA_NCLASS];   // FILL pass: first item / batch of every class (from the host)
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
// batches of every support class; FILL = true writes them (class offsets are in the counters by then).
template <bool FILL>
__global__ void __launch_bounds__(256) lra_work_kernel(const lra_work_args a) {
  const long long n = (long long)a.counters[0];
  const long long lo = (long long)blockIdx.x * LRA_CHUNK;
  if (lo >= n) return;
  const long long hi = lo + LRA_CHUNK < n ? lo + LRA_CHUNK : n;
  __shared__ unsigned warp_buf[8];
  __shared__ int warp_buf_i[8];
  __shared__ unsigned cls_cnt[2][LRA_NCLASS];
  __shared__ unsigned item_tile[LRA_CHUNK], item_first_run[LRA_CHUNK + 1], item_base[LRA_CHUNK], run_pos[LRA_CHUNK + 1];
  __shared__ unsigned short run_item[LRA_CHUNK];
  __shared__ unsigned char item_sup[LRA_CHUNK];
  __shared__ lra_geom geom[LRA_NCLASS];   // per support class, once per block (lra_make_geom is not cheap)
  if (threadIdx.x < LRA_NCLASS) geom[threadIdx.x] = lra_make_geom(2 * threadIdx.x + 1, a.tile_x, a.tile_y, a.ng);
  if (threadIdx.x < 2 * LRA_NCLASS) (&cls_cnt[0][0])[threadIdx.x] = 0;
  // ---- flags of the thread's 4 consecutive positions ----
  const long long i0 = lo + threadIdx.x * 4;
  unsigned item_f = 0, slab_f = 0, tl[4], sp[4];
  long long prev_t = -1;
  int prev_s = -1;
  unsigned prev_slab = 0xffffffffu;
  if (i0 > lo && i0 - 1 < hi) {
    const lra_rec r = a.rec[i0 - 1];
    prev_t = (long long)((r.x >> 16) >> a.shift_y) * a.ntx + ((r.x & 0xffff) >> a.shift_x);
    prev_s = (int)(r.w & 0xff);
    prev_slab = r.y;
  }
  lra_rec rc[4];
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    const long long i = i0 + e;
    tl[e] = 0; sp[e] = 1;
    if (i < hi) {
      const lra_rec r = a.rec[i];
      rc[e] = r;
      const long long t = (long long)((r.x >> 16) >> a.shift_y) * a.ntx + ((r.x & 0xffff) >> a.shift_x);
      const int s = (int)(r.w & 0xff);
      if (i == lo || t != prev_t || s != prev_s) item_f |= 1u << e;
      if ((item_f >> e & 1u) || r.y != prev_slab) slab_f |= 1u << e;
      tl[e] = (unsigned)t; sp[e] = (unsigned)s;
      prev_t = t; prev_s = s; prev_slab = r.y;
    }
  }
  // ---- run heads: slab heads plus a cut every LRA_RUNMAX points of a slab run ----
  int last_head = -1;   // chunk-relative position of the last slab head at or before the thread's positions
#pragma unroll
  for (int e = 0; e < 4; ++e)
    if (slab_f >> e & 1u) last_head = threadIdx.x * 4 + e;
  int run_head = lra_block_excl_max(last_head, warp_buf_i);
  unsigned run_f = 0;
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    if (i0 + e < hi) {
      if (slab_f >> e & 1u) run_head = threadIdx.x * 4 + e;
      if (((threadIdx.x * 4 + e - run_head) & (LRA_RUNMAX - 1)) == 0) run_f |= 1u << e;
    }
  }
  unsigned n_items_blk, n_runs_blk;
  unsigned ir = lra_block_excl_sum(__popc(item_f), warp_buf, n_items_blk);
  unsigned rr = lra_block_excl_sum(__popc(run_f), warp_buf, n_runs_blk);
  // ---- block-local lists ----
  unsigned my_run[4];
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    if (item_f >> e & 1u) {
      item_tile[ir] = tl[e];
      item_first_run[ir] = rr;
      item_sup[ir] = (unsigned char)sp[e];
      ++ir;
    }
    if (run_f >> e & 1u) {
      run_pos[rr] = (unsigned)(i0 + e);
      run_item[rr] = (unsigned short)(ir - 1);
      ++rr;
    }
    my_run[e] = rr - 1;
  }
  if (threadIdx.x == 0) { item_first_run[n_items_blk] = n_runs_blk; run_pos[n_runs_blk] = (unsigned)hi; }
  __syncthreads();
  // ---- items: batches per item, global slots ----
  for (unsigned j = threadIdx.x; j < n_items_blk; j += 256) {
    const unsigned S = item_sup[j], c = (unsigned)lra_class_of((int)S);
    const unsigned nruns = item_first_run[j + 1] - item_first_run[j];
    const unsigned per = (unsigned)geom[c].per_batch;
    const unsigned nb = (nruns + per - 1) / per;
    if (!FILL) {
      atomicAdd(&cls_cnt[0][c], 1u);
      atomicAdd(&cls_cnt[1][c], nb);
    } else {
      const unsigned base = (unsigned)atomicAdd(&a.counters[LRA_CNT_BATCH_CUR + c], (unsigned long long)nb);
      const unsigned long long idx = a.item_off[c] + atomicAdd(&a.counters[LRA_CNT_ITEM_CUR + c], 1ull);
      a.work[idx] = make_uint4(item_tile[j], base, nb, S);
      item_base[j] = base;
    }
  }
  __syncthreads();
  if (!FILL) {
    if (threadIdx.x < LRA_NCLASS) {
      if (cls_cnt[0][threadIdx.x]) atomicAdd(&a.counters[LRA_CNT_ITEMS + threadIdx.x], (unsigned long long)cls_cnt[0][threadIdx.x]);
      if (cls_cnt[1][threadIdx.x]) atomicAdd(&a.counters[LRA_CNT_BATCHES + threadIdx.x], (unsigned long long)cls_cnt[1][threadIdx.x]);
    }
    return;
  }
  // ---- batches: header and slab table, one thread per run ----
  for (unsigned j = threadIdx.x; j < n_runs_blk; j += 256) {
    const unsigned it = run_item[j], S = item_sup[it], c = (unsigned)lra_class_of((int)S);
    const unsigned first_run = item_first_run[it], nruns = item_first_run[it + 1] - first_run;
    const unsigned per = (unsigned)geom[c].per_batch;
    const unsigned q = j - first_run, b = q / per, r = q - b * per;
    uint32_t* rec16 = a.batch + ((unsigned long long)a.batch_off[c] + item_base[it] + b) * 16ull;
    rec16[4 + r] = a.rec[run_pos[j]].y;
    if (r == 0) {
      const unsigned nr = nruns - b * per < per ? nruns - b * per : per;
      const unsigned first = run_pos[j], count = run_pos[j + nr] - first;
      const unsigned last = (b * per + nr == nruns) ? LRA_BATCH_LAST : 0u;
      rec16[0] = first; rec16[1] = count | last; rec16[2] = nr; rec16[3] = item_tile[it];
    }
  }
  // ---- per-point words ----
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    const long long i = i0 + e;
    if (i < hi) {
      const unsigned j = my_run[e], it = run_item[j];
      const lra_geom& q = geom[lra_class_of((int)sp[e])];
      const unsigned r = (j - item_first_run[it]) % (unsigned)q.per_batch;
      const int ix = rc[e].x & 0xffff, iy = rc[e].x >> 16;
      const int ox = ix - ((ix >> a.shift_x) << a.shift_x), oy = iy - ((iy >> a.shift_y) << a.shift_y);
      const int off = oy * q.rx + ox;
      const int c_lo = off >> 6, c_hi = (off + q.span - 1) >> 6;
      unsigned mz = (unsigned)c_lo | (unsigned)c_hi << 16, mw = 0u;
      if (q.nw >= 1 && q.nw <= 8) {   // the step masks of the consumer warps, one byte each (lra_region.cuh)
        unsigned long long m = 0ull;
        const int lg = __ffs(q.nw) - 1;   // NW is a power of two
        for (int w = 0; w < q.nw; ++w) {
          const int s_lo = (c_lo - w + q.nw - 1) >> lg, s_hi = (c_hi - w) >> lg;   // arithmetic shift: -1 if c_hi < w
          if (s_hi >= s_lo) m |= (unsigned long long)(((2u << s_hi) - (1u << s_lo)) & 0xffu) << (8 * w);
        }
        mz = (unsigned)m; mw = (unsigned)(m >> 32);
      }
      a.pw[i] = make_uint4((unsigned)(8 * (LRA_GAP + (int)r * q.stride - off)), rc[e].z | (q.nw == 0 ? 0x80000000u : 0u), mz, mw);
    }
  }
}

__global__ void __launch_bounds__(256) lra_counts_to_host_kernel(const unsigned long long* __restrict__ src, unsigned long long* dst) {
  dst[threadIdx.x] = src[threadIdx.x];
  __threadfence_system();
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
  for (int c = 0; c < LRA_NCLASS; ++c) { p->n_items[c] = 0; p->item_off[c] = 0; p->n_batches[c] = 0; p->batch_off[c] = 0; }
  const int64_t n = p->npoints;
  if (n == 0) return LRA_OK;
  lra_work_args a;
  a.rec = p->rec; a.counters = p->counters; a.ntx = p->ntx; a.tile_x = p->tile_x; a.tile_y = p->tile; a.ng = p->ncorr * p->nterms;
  a.work = nullptr; a.batch = nullptr; a.pw = nullptr;
  for (int c = 0; c < LRA_NCLASS; ++c) a.item_off[c] = a.batch_off[c] = 0;
  a.shift_x = a.shift_y = 0;
  while ((1 << a.shift_x) < p->tile_x) ++a.shift_x;
  while ((1 << a.shift_y) < p->tile) ++a.shift_y;
  const int blocks = (int)((n + LRA_CHUNK - 1) / LRA_CHUNK);
  int rc;
  // the class counters were zeroed at the start of lra_bin
  lra_work_kernel<false><<<blocks, 256, 0, p->stream>>>(a);
  LRA_LAUNCH_CHECK(p);
  static_assert(LRA_CNT_BATCHES == LRA_CNT_ITEMS + 128 && LRA_CNT_BATCH_OFF == LRA_CNT_ITEM_OFF + 128, "counter layout");
  // the list sizes go to the host through a kernel that writes pinned, mapped memory: a cudaMemcpy would queue on the
  // copy engine behind whatever bulk transfer the caller has in flight on another stream (measured: 29 ms per step in
  // bench.py's pipelined end-to-end loop)
  unsigned long long* hd = nullptr;
  LRA_CUDA(p, cudaHostGetDevicePointer(&hd, p->h_counts, 0));
  lra_counts_to_host_kernel<<<1, 256, 0, p->stream>>>(p->counters + LRA_CNT_ITEMS, hd);
  LRA_LAUNCH_CHECK(p);
  LRA_CUDA(p, cudaStreamSynchronize(p->stream));   // the one host synchronisation of lra_bin: the list sizes
  const unsigned long long* h = p->h_counts;
  int64_t items = 0, batches = 0;
  for (int c = 0; c < LRA_NCLASS; ++c) {
    p->n_items[c] = (int64_t)h[c];
    p->n_batches[c] = (int64_t)h[128 + c];
    p->item_off[c] = items;
    p->batch_off[c] = batches;
    a.item_off[c] = (unsigned)items;
    a.batch_off[c] = (unsigned)batches;
    items += p->n_items[c];
    batches += p->n_batches[c];
  }
  if ((rc = lra_grow(p, &p->work, &p->work_capacity, items))) return rc;
  int64_t bwords = p->batch_capacity * 16;
  if ((rc = lra_grow(p, &p->batch, &bwords, batches * 16))) return rc;
  p->batch_capacity = bwords / 16;
  if ((rc = lra_grow(p, &p->pw, &p->pw_capacity, n))) return rc;
  a.work = p->work; a.batch = p->batch; a.pw = p->pw;
  lra_work_kernel<true><<<blocks, 256, 0, p->stream>>>(a);
  LRA_LAUNCH_CHECK(p);
  return LRA_OK;
}

// lra_bin.cu -- coordinate/index kernel and the hand-written stable LSD radix sort behind lra_bin
// ("re-ordering for runtime performance"; readings R2, R4, R5 in DESIGN.md).
// Integer / fp64 work only; every output must be bit-exact against the oracle.
#include "lra_pipe.cuh"

// ---------------------------------------------------------------------------------------------------
// a1: coordinate / index.  One thread per visibility point k = r*nchan + c.
// fp64 with every operation rounded separately (__dmul_rn / __dadd_rn: no FMA contraction) [R2]:
//   px = u*su[c] + nx/2;  t = floor(px*os + 0.5);  P = (int64)t;  ix = floordiv(P + os/2, os);  fx = P - ix*os
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ bool lra_axis_index(double coord_m, double s, int n, int os, int& pix, int& ph) {
  double px = __dadd_rn(__dmul_rn(coord_m, s), (double)(n / 2));
  double t = floor(__dadd_rn(__dmul_rn(px, (double)os), 0.5));
  if (!(t >= -4.0 * (double)os && t <= ((double)n + 4.0) * (double)os)) return false;  // also rejects NaN / inf
  long long P = (long long)t;
  long long a = P + os / 2;
  long long q = a / os, r = a % os;
  if (r < 0) { q -= 1; }
  pix = (int)q;
  ph = (int)(P - q * os);
  return true;
}

struct lra_index_args {
  int nx, ny, os, tile_x, tile_y, ntx, ntiles, sort_mode, n_cf, nchan;
  long long npoints;
  unsigned long long invalid_sort_key;  // ntiles * per_tile: sorts after every valid key
};

__global__ void __launch_bounds__(256)
lra_index_kernel(lra_index_args a, const double* __restrict__ uvw, const double* __restrict__ su,
                 const double* __restrict__ sv, const int32_t* __restrict__ cf_index,
                 const int32_t* __restrict__ cf_support, int32_t* __restrict__ ix_o, int32_t* __restrict__ iy_o,
                 int8_t* __restrict__ fx_o, int8_t* __restrict__ fy_o, uint64_t* __restrict__ key_o,
                 uint64_t* __restrict__ skey_o, uint32_t* __restrict__ sval_o, unsigned long long* __restrict__ counters,
                 const int64_t* __restrict__ slab_off, lra_rec* __restrict__ urec) {
  long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  unsigned long long nvalid = 0, s2 = 0;
  if (k < a.npoints) {
    long long r = k / a.nchan;
    int c = (int)(k - r * a.nchan);
    int ix = -1, iy = -1, fx = 0, fy = 0;
    bool ok = lra_axis_index(uvw[3 * r + 0], su[c], a.nx, a.os, ix, fx);
    ok &= lra_axis_index(uvw[3 * r + 1], sv[c], a.ny, a.os, iy, fy);
    int cf = cf_index ? cf_index[k] : 0;
    ok = ok && cf >= 0 && cf < a.n_cf;
    int S = 1;
    if (ok) {
      S = cf_support[cf];
      int h = (S - 1) / 2;
      ok = ix - h >= 0 && ix + h <= a.nx - 1 && iy - h >= 0 && iy + h <= a.ny - 1;  // R4
    }
    unsigned long long key = ~0ull, skey = a.invalid_sort_key;
    if (ok) {
      unsigned long long tile_id = (unsigned long long)(iy / a.tile_y) * a.ntx + (unsigned long long)(ix / a.tile_x);
      key = tile_id;
      if (a.sort_mode == LRA_SORT_TILE_CF)
        key = ((tile_id * a.n_cf + cf) * a.os + (fy + a.os / 2)) * a.os + (fx + a.os / 2);
      skey = key;
      nvalid = 1;
      s2 = (unsigned long long)S * S;
    } else {
      ix = iy = -1; fx = fy = 0;
    }
    ix_o[k] = ix; iy_o[k] = iy; fx_o[k] = (int8_t)fx; fy_o[k] = (int8_t)fy; key_o[k] = key;
    skey_o[k] = skey; sval_o[k] = (uint32_t)k;
    if (ok) {   // the record the gridder / degridder consume (lra_internal.cuh), gathered into sorted order later
      const int phase = (fy + a.os / 2) * a.os + (fx + a.os / 2);
      const long long off = slab_off[cf] + (long long)phase * (2 * lra_slab_complex(S, a.tile_x));
      urec[k] = make_uint4((uint32_t)ix | ((uint32_t)iy << 16), (uint32_t)(off >> 2), (uint32_t)k, (uint32_t)S | ((uint32_t)cf << 8));
    }
  }
  // block totals -> two atomics per block
  __shared__ unsigned long long sh[2][8];
  for (int o = 16; o > 0; o >>= 1) {
    nvalid += __shfl_down_sync(0xffffffffu, nvalid, o);
    s2 += __shfl_down_sync(0xffffffffu, s2, o);
  }
  int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  if (l == 0) { sh[0][w] = nvalid; sh[1][w] = s2; }
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long n = 0, s = 0;
    for (int i = 0; i < 8; ++i) { n += sh[0][i]; s += sh[1][i]; }
    if (n) { atomicAdd(&counters[0], n); atomicAdd(&counters[1], s); }
  }
}

// ---------------------------------------------------------------------------------------------------
// a2: stable LSD radix sort, 8 bits per pass, (uint64 key, uint32 value) pairs.
// Each block owns a contiguous span of `span` elements (a multiple of 256) and walks it in rounds of 256
// consecutive elements, one per thread, so input order is preserved inside every digit bucket.
//   pass = histogram kernel -> one-block exclusive scan over [digit][block] -> scatter kernel.
// ---------------------------------------------------------------------------------------------------
#define LRA_RADIX 256

__global__ void __launch_bounds__(256)
lra_radix_hist_kernel(const uint64_t* __restrict__ keys, long long n, int span, int shift, uint32_t* __restrict__ hist) {
  __shared__ uint32_t h[LRA_RADIX];
  h[threadIdx.x] = 0;
  __syncthreads();
  long long lo = (long long)blockIdx.x * span, hi = lo + span < n ? lo + span : n;
  for (long long i = lo + threadIdx.x; i < hi; i += 256) atomicAdd(&h[(unsigned)(keys[i] >> shift) & 255u], 1u);
  __syncthreads();
  hist[(size_t)threadIdx.x * gridDim.x + blockIdx.x] = h[threadIdx.x];
}

// Exclusive scan of the histogram hist[digit][block] in digit-major order, in two small steps instead of one block
// walking all 256 * blocks entries: block d scans row d in place (exclusive) and leaves the row total in tot[d];
// lra_scan_tot_kernel then turns tot[] into the exclusive scan over the digits, which the scatter adds.
__global__ void __launch_bounds__(1024) lra_scan_rows_kernel(uint32_t* __restrict__ hist, int blocks, uint32_t* __restrict__ tot) {
  __shared__ uint32_t warp_tot[32];
  __shared__ uint32_t carry;
  uint32_t* a = hist + (size_t)blockIdx.x * blocks;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  const int l = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (int base = 0; base < blocks; base += 1024) {
    const int i = base + threadIdx.x;
    uint32_t v = i < blocks ? a[i] : 0u, x = v;
    for (int o = 1; o < 32; o <<= 1) {
      uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
      if (l >= o) x += y;
    }
    if (l == 31) warp_tot[w] = x;
    __syncthreads();
    if (w == 0) {
      uint32_t t = warp_tot[l], s = t;
      for (int o = 1; o < 32; o <<= 1) {
        uint32_t y = __shfl_up_sync(0xffffffffu, s, o);
        if (l >= o) s += y;
      }
      warp_tot[l] = s - t;  // exclusive
    }
    __syncthreads();
    const uint32_t c = carry;
    if (i < blocks) a[i] = c + warp_tot[w] + (x - v);
    __syncthreads();
    if (threadIdx.x == 1023) carry = c + warp_tot[31] + x;
    __syncthreads();
  }
  if (threadIdx.x == 0) tot[blockIdx.x] = carry;
}
__global__ void __launch_bounds__(LRA_RADIX) lra_scan_tot_kernel(uint32_t* __restrict__ tot) {
  __shared__ uint32_t warp_tot[8];
  const int l = threadIdx.x & 31, w = threadIdx.x >> 5;
  const uint32_t v = tot[threadIdx.x];
  uint32_t x = v;
  for (int o = 1; o < 32; o <<= 1) {
    uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
    if (l >= o) x += y;
  }
  if (l == 31) warp_tot[w] = x;
  __syncthreads();
  uint32_t base = 0;
  for (int ww = 0; ww < w; ++ww) base += warp_tot[ww];
  tot[threadIdx.x] = base + x - v;
}

// One pass of the least-significant-digit radix sort: block b moves the keys of its span [b*span, (b+1)*span) to their
// places, 4,096 keys at a time.  The keys of a round are ranked (stably: by warp, sub-round, lane), staged in shared memory
// in digit order, and only then written out: every digit's keys of a round form one run of consecutive addresses (16 keys
// = 128 bytes on average) instead of 4,096 isolated 8-byte writes.
#define LRA_SORT_TILE_KEYS 4096
#define LRA_SORT_ITEMS 16   // keys per thread and round: warp w owns keys [w*512, (w+1)*512) of the round
struct lra_scatter_smem {
  uint64_t keys[LRA_SORT_TILE_KEYS];
  uint32_t vals[LRA_SORT_TILE_KEYS];
  uint32_t warp_cnt[8][LRA_RADIX];   // running count of (warp, digit); after the prefix step: keys of lower warps
  uint32_t digit_off[LRA_RADIX];     // running global offset of every digit for this block
  uint32_t lstart[LRA_RADIX];        // first staged position of the digit in this round
  uint32_t gdelta[LRA_RADIX];        // global position minus staged position
  uint32_t wsum[8];
};

__global__ void __launch_bounds__(256)
lra_radix_scatter_kernel(const uint64_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in,
                         uint64_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out, long long n, int span,
                         int shift, const uint32_t* __restrict__ hist_scanned, const uint32_t* __restrict__ digit_base) {
  extern __shared__ __align__(16) unsigned char lra_scatter_raw[];
  lra_scatter_smem& sm = *reinterpret_cast<lra_scatter_smem*>(lra_scatter_raw);
  const int t = threadIdx.x, l = t & 31, w = t >> 5;
  sm.digit_off[t] = hist_scanned[(size_t)t * gridDim.x + blockIdx.x] + digit_base[t];
  for (int i = 0; i < 8; ++i) sm.warp_cnt[i][t] = 0;
  __syncthreads();
  const long long lo = (long long)blockIdx.x * span, hi = lo + span < n ? lo + span : n;
  for (long long base = lo; base < hi; base += LRA_SORT_TILE_KEYS) {
    const int cnt = (int)(hi - base < LRA_SORT_TILE_KEYS ? hi - base : LRA_SORT_TILE_KEYS);
    uint64_t key[LRA_SORT_ITEMS];
    uint32_t val[LRA_SORT_ITEMS];
    uint32_t rank[LRA_SORT_ITEMS];   // rank among the warp's keys of the same digit, digit in the top byte
#pragma unroll
    for (int r = 0; r < LRA_SORT_ITEMS; ++r) {
      const int i = w * (32 * LRA_SORT_ITEMS) + r * 32 + l;
      const bool act = i < cnt;
      key[r] = act ? keys_in[base + i] : 0;
      val[r] = act ? vals_in[base + i] : 0;
    }
#pragma unroll
    for (int r = 0; r < LRA_SORT_ITEMS; ++r) {
      const int i = w * (32 * LRA_SORT_ITEMS) + r * 32 + l;
      const bool act = i < cnt;
      const unsigned d = (unsigned)(key[r] >> shift) & 255u;
      // lanes of this warp with the same digit (inactive lanes get a digit of their own: 256 + lane)
      const unsigned peers = __match_any_sync(0xffffffffu, act ? d : 256u + l);
      const unsigned below = __popc(peers & ((1u << l) - 1u));
      uint32_t old = 0;
      if (act && below == 0) { old = sm.warp_cnt[w][d]; sm.warp_cnt[w][d] = old + __popc(peers); }
      old = __shfl_sync(0xffffffffu, old, __ffs(peers) - 1);
      rank[r] = (old + below) | (d << 24) | (act ? 0u : 0x800000u);
      __syncwarp();
    }
    __syncthreads();
    {   // thread t = digit t: keys of lower warps, then the exclusive scan of the digit totals over the block
      uint32_t run = 0;
#pragma unroll
      for (int ww = 0; ww < 8; ++ww) { const uint32_t c = sm.warp_cnt[ww][t]; sm.warp_cnt[ww][t] = run; run += c; }
      uint32_t x = run;
      for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, x, o); if (l >= o) x += y; }
      if (l == 31) sm.wsum[w] = x;
      __syncthreads();
      uint32_t before = 0;
      for (int ww = 0; ww < w; ++ww) before += sm.wsum[ww];
      const uint32_t start = before + x - run;
      sm.lstart[t] = start;
      sm.gdelta[t] = sm.digit_off[t] - start;
      sm.digit_off[t] += run;
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < LRA_SORT_ITEMS; ++r) {
      if (rank[r] & 0x800000u) continue;
      const unsigned d = rank[r] >> 24;
      const uint32_t pos = sm.lstart[d] + sm.warp_cnt[w][d] + (rank[r] & 0x7fffffu);
      sm.keys[pos] = key[r];
      sm.vals[pos] = val[r];
    }
    __syncthreads();
    for (int i = t; i < cnt; i += 256) {
      const uint64_t k = sm.keys[i];
      const uint32_t pos = sm.gdelta[(unsigned)(k >> shift) & 255u] + (uint32_t)i;
      keys_out[pos] = k;
      vals_out[pos] = sm.vals[i];
    }
    for (int i = 0; i < 8; ++i) sm.warp_cnt[i][t] = 0;
    __syncthreads();
  }
}

// ---------------------------------------------------------------------------------------------------
// tile_start[q] = first position in the sorted order whose tile id >= q; thread i compares position i with
// i-1 (position -1 has tile -1, position npoints has tile ntiles; invalid points carry tile ntiles).
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
lra_tile_start_kernel(const uint64_t* __restrict__ sorted_keys, long long n, unsigned long long per_tile, int ntiles,
                      uint32_t* __restrict__ tile_start) {
  long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i > n) return;
  long long t_here = i < n ? (long long)(sorted_keys[i] / per_tile) : (long long)ntiles;
  long long t_prev = i > 0 ? (long long)(sorted_keys[i - 1] / per_tile) : -1;
  if (t_here > ntiles) t_here = ntiles;
  for (long long q = t_prev + 1; q <= t_here; ++q) tile_start[q] = (uint32_t)i;
}

// Sorted records for the gridder / degridder: one 16-byte gather per sorted position (see lra_internal.cuh).
__global__ void __launch_bounds__(256)
lra_record_kernel(const uint32_t* __restrict__ perm, const unsigned long long* __restrict__ counters,
                  const lra_rec* __restrict__ urec, lra_rec* __restrict__ rec) {
  long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i >= (long long)counters[0]) return;
  rec[i] = urec[perm[i]];
}

__global__ void __launch_bounds__(256)
lra_scale_from_host_kernel(const double* __restrict__ h, double* __restrict__ su, double* __restrict__ sv, int nchan) {
  const int i = blockIdx.x * 256 + threadIdx.x;
  if (i < nchan) su[i] = h[i];
  else if (i < 2 * nchan) sv[i - nchan] = h[i];
}

template <typename T>
static int lra_regrow(lra_plan* p, T** ptr, size_t count) {
  if (*ptr) { cudaFree(*ptr); *ptr = nullptr; }
  LRA_CUDA(p, cudaMalloc(ptr, (count ? count : 1) * sizeof(T)));
  return LRA_OK;
}

int lra_bin_impl(lra_plan* p, int64_t nrow, int32_t nchan, const double* uvw, const double* freq_host,
                 const int32_t* cf_index) {
  const int64_t n = nrow * nchan;
  p->binned = false;
  int rc;
  if (n > p->capacity) {
    LRA_CUDA(p, cudaStreamSynchronize(p->stream));
    p->capacity = 0;   // a failure part-way leaves freed (null) arrays behind: the next call must grow again
    if ((rc = lra_regrow(p, &p->ix, n))) return rc;
    if ((rc = lra_regrow(p, &p->iy, n))) return rc;
    if ((rc = lra_regrow(p, &p->fx, n))) return rc;
    if ((rc = lra_regrow(p, &p->fy, n))) return rc;
    if ((rc = lra_regrow(p, &p->key, n))) return rc;
    for (int b = 0; b < 2; ++b) {
      if ((rc = lra_regrow(p, &p->skey[b], n))) return rc;
      if ((rc = lra_regrow(p, &p->sval[b], n))) return rc;
    }
    if ((rc = lra_regrow(p, &p->rec, n))) return rc;
    if ((rc = lra_regrow(p, &p->urec, n))) return rc;
    p->capacity = n;
  }
  if (nchan > p->su_capacity) {
    LRA_CUDA(p, cudaStreamSynchronize(p->stream));
    p->su_capacity = 0;
    if ((rc = lra_regrow(p, &p->d_su, nchan))) return rc;
    if ((rc = lra_regrow(p, &p->d_sv, nchan))) return rc;
    p->su_capacity = nchan;
  }
  if (nchan > p->h_scale_capacity) {
    LRA_CUDA(p, cudaStreamSynchronize(p->stream));
    if (p->h_scale) { cudaFreeHost(p->h_scale); p->h_scale = nullptr; p->h_scale_capacity = 0; }
    LRA_CUDA(p, cudaHostAlloc(&p->h_scale, (size_t)2 * nchan * sizeof(double), cudaHostAllocMapped));
    p->h_scale_capacity = nchan;
  }
  // per-channel scale, formed on the host in IEEE double: su[c] = (freq[c] / c) * scale_u  [R2]
  // (lra_bin ends with a host synchronisation, so the previous call's kernel has read h_scale long ago; the table goes to
  // the device through a kernel reading pinned, mapped memory rather than a cudaMemcpy: see lra_work.cu)
  double* su = p->h_scale;
  double* sv = p->h_scale + nchan;
  for (int c = 0; c < nchan; ++c) {
    volatile double lam_inv = freq_host[c] / 299792458.0;
    volatile double a = lam_inv * p->scale_u, b = lam_inv * p->scale_v;
    su[c] = a; sv[c] = b;
  }
  if (nrow * (int64_t)nchan > 0) {   // (an empty call enqueues nothing that reads h_scale, and ends without a synchronisation)
    double* hd = nullptr;
    LRA_CUDA(p, cudaHostGetDevicePointer(&hd, p->h_scale, 0));
    lra_scale_from_host_kernel<<<(2 * nchan + 255) / 256, 256, 0, p->stream>>>(hd, p->d_su, p->d_sv, nchan);
    LRA_LAUNCH_CHECK(p);
  }
  LRA_CUDA(p, cudaMemsetAsync(p->counters, 0, LRA_TICKET0 * sizeof(unsigned long long), p->stream));

  unsigned long long per_tile = 1;
  if (p->sort_mode == LRA_SORT_TILE_CF) per_tile = (unsigned long long)p->n_cf * p->os * p->os;
  const unsigned long long invalid_key = (unsigned long long)p->ntiles * per_tile;
  p->nrow = nrow; p->nchan = nchan; p->npoints = n;
  p->per_tile = per_tile; p->tile_start_done = false;   // per-tile offsets are computed by lra_bin_export on demand
  p->sorted_buf = 0;
  if (n > 0) {
    lra_index_args a;
    a.nx = p->nx; a.ny = p->ny; a.os = p->os; a.tile_x = p->tile_x; a.tile_y = p->tile; a.ntx = p->ntx; a.ntiles = p->ntiles;
    a.sort_mode = p->sort_mode; a.n_cf = p->n_cf; a.nchan = nchan; a.npoints = n; a.invalid_sort_key = invalid_key;
    int blocks = (int)((n + 255) / 256);
    lra_index_kernel<<<blocks, 256, 0, p->stream>>>(a, uvw, p->d_su, p->d_sv, cf_index, p->d_cf_support, p->ix, p->iy,
                                                    p->fx, p->fy, p->key, p->skey[0], p->sval[0], p->counters, p->d_slab_off,
                                                    p->urec);
    LRA_LAUNCH_CHECK(p);
    // radix passes over the bits of invalid_key (the largest sort key)
    int nbits = 0;
    while (nbits < 64 && (invalid_key >> nbits) != 0) ++nbits;
    int passes = (nbits + 7) / 8;
    if (passes < 1) passes = 1;
    // span per block: a multiple of 256, about 4 blocks per SM
    int64_t want_blocks = (int64_t)p->sm_count * 4;
    int64_t span = ((n + want_blocks - 1) / want_blocks + 255) / 256 * 256;
    if (span < 2048) span = 2048;
    int sblocks = (int)((n + span - 1) / span);
    int64_t hist_n = (int64_t)LRA_RADIX * sblocks;
    if (hist_n > p->hist_capacity) {
      LRA_CUDA(p, cudaStreamSynchronize(p->stream));
      p->hist_capacity = 0;
      if ((rc = lra_regrow(p, &p->hist, hist_n + LRA_RADIX))) return rc;   // + the per-digit totals
      p->hist_capacity = hist_n;
    }
    LRA_CUDA(p, cudaFuncSetAttribute(lra_radix_scatter_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(lra_scatter_smem)));
    int cur = 0;
    for (int ps = 0; ps < passes; ++ps) {
      int shift = 8 * ps;
      lra_radix_hist_kernel<<<sblocks, 256, 0, p->stream>>>(p->skey[cur], n, (int)span, shift, p->hist);
      LRA_LAUNCH_CHECK(p);
      lra_scan_rows_kernel<<<LRA_RADIX, 1024, 0, p->stream>>>(p->hist, sblocks, p->hist + hist_n);
      LRA_LAUNCH_CHECK(p);
      lra_scan_tot_kernel<<<1, LRA_RADIX, 0, p->stream>>>(p->hist + hist_n);
      LRA_LAUNCH_CHECK(p);
      lra_radix_scatter_kernel<<<sblocks, 256, sizeof(lra_scatter_smem), p->stream>>>(p->skey[cur], p->sval[cur], p->skey[cur ^ 1],
                                                               p->sval[cur ^ 1], n, (int)span, shift, p->hist, p->hist + hist_n);
      LRA_LAUNCH_CHECK(p);
      cur ^= 1;
    }
    p->sorted_buf = cur;
    lra_record_kernel<<<blocks, 256, 0, p->stream>>>(p->sval[cur], p->counters, p->urec, p->rec);
    LRA_LAUNCH_CHECK(p);
    if ((rc = lra_build_work(p))) return rc;
  } else {
    LRA_CUDA(p, cudaMemsetAsync(p->tile_start, 0, (size_t)(p->ntiles + 1) * sizeof(uint32_t), p->stream));
  }
  p->binned = true;
  return LRA_OK;
}

extern "C" int lra_bin_export(lra_plan* p, int32_t* ix, int32_t* iy, int8_t* fx, int8_t* fy, uint64_t* key,
                              uint32_t* perm, uint32_t* tile_start, int64_t* n_valid) {
  if (!p) return LRA_EINVAL;
  if (!p->binned) return LRA_ESTATE;
  LRA_CUDA(p, cudaSetDevice(p->device));
  const size_t n = (size_t)p->npoints;
  const cudaMemcpyKind k = cudaMemcpyDeviceToDevice;
  if (n) {
    if (ix) LRA_CUDA(p, cudaMemcpyAsync(ix, p->ix, n * 4, k, p->stream));
    if (iy) LRA_CUDA(p, cudaMemcpyAsync(iy, p->iy, n * 4, k, p->stream));
    if (fx) LRA_CUDA(p, cudaMemcpyAsync(fx, p->fx, n, k, p->stream));
    if (fy) LRA_CUDA(p, cudaMemcpyAsync(fy, p->fy, n, k, p->stream));
    if (key) LRA_CUDA(p, cudaMemcpyAsync(key, p->key, n * 8, k, p->stream));
    if (perm) LRA_CUDA(p, cudaMemcpyAsync(perm, p->sval[p->sorted_buf], n * 4, k, p->stream));
  }
  if (tile_start) {
    if (!p->tile_start_done) {
      if (n) {
        lra_tile_start_kernel<<<(int)((n + 1 + 255) / 256), 256, 0, p->stream>>>(p->skey[p->sorted_buf], (long long)n, p->per_tile,
                                                                                 p->ntiles, p->tile_start);
        LRA_LAUNCH_CHECK(p);
      } else {
        LRA_CUDA(p, cudaMemsetAsync(p->tile_start, 0, (size_t)(p->ntiles + 1) * sizeof(uint32_t), p->stream));
      }
      p->tile_start_done = true;
    }
    LRA_CUDA(p, cudaMemcpyAsync(tile_start, p->tile_start, (size_t)(p->ntiles + 1) * 4, k, p->stream));
  }
  unsigned long long nv = 0;
  LRA_CUDA(p, cudaMemcpyAsync(&nv, p->counters, sizeof nv, cudaMemcpyDeviceToHost, p->stream));
  LRA_CUDA(p, cudaStreamSynchronize(p->stream));
  if (n_valid) *n_valid = (int64_t)nv;
  return LRA_OK;
}

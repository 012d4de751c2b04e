// lra_gain.cu -- the G-Jones solver fed by degridded model visibilities (Sec. 5.1 of
// arxiv 2508.17187):
//   lra_gain_accumulate : Eq. 19, the sums of wt * V^c / V^Mod and of wt per baseline and correlation
//   lra_gain_solve      : Eq. 20 / 21 iterated to |g^{k+1} - g^k| < delta
// Readings R21-R23.  V^Mod is what lra_degrid writes without vis_in ("PreCompute ... the D and the F
// operators").
//
// lra_gain_accumulate is HBM-bound (20 bytes read per sample): a grid-stride pass over the samples, ratio and sums in
// double, per-block partial sums per (baseline, correlation) in shared memory (shared double atomics), one global
// double atomic per block and entry.  lra_gain_solve is tiny (nant <= 1024 gains): one CTA, one thread per antenna,
// every thread walks the baseline list (Jacobi update from the gains of iteration k in shared memory).
// Product code: shares nothing with oracle/.
#include "lra_internal.cuh"

#define LRA_GAIN_SMEM_ENTRIES 2048   // (baseline, correlation) entries a block keeps in shared memory (48 KB)

__global__ void __launch_bounds__(256)
lra_gain_accumulate_kernel(long long nsamples, int nchan, int ncorr, int nbl, const int32_t* __restrict__ bl_index,
                           const float2* __restrict__ vis, const float2* __restrict__ model, const float* __restrict__ wt,
                           double* __restrict__ xsum, double* __restrict__ wsum, int use_smem) {
  __shared__ double sh[LRA_GAIN_SMEM_ENTRIES * 3];
  const int nent = nbl * ncorr;
  if (use_smem) {
    for (int i = threadIdx.x; i < nent * 3; i += blockDim.x) sh[i] = 0.0;
    __syncthreads();
  }
  const long long per_row = (long long)nchan * ncorr;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < nsamples; i += (long long)gridDim.x * blockDim.x) {
    const float w = wt[i];
    const float2 m = model[i], v = vis[i];
    const double den = (double)m.x * m.x + (double)m.y * m.y;
    if (!(w > 0.f) || !(den > 0.0)) continue;
    const long long r = i / per_row;
    const int p = (int)(i % ncorr);
    const long long b = bl_index ? (long long)bl_index[r] : r % nbl;
    if (b < 0 || b >= nbl) continue;
    const double xr = (double)w * (((double)v.x * m.x + (double)v.y * m.y) / den);   // V / M = V conj(M) / |M|^2
    const double xi = (double)w * (((double)v.y * m.x - (double)v.x * m.y) / den);
    const int e = (int)b * ncorr + p;
    if (use_smem) {
      atomicAdd(&sh[e * 3], xr); atomicAdd(&sh[e * 3 + 1], xi); atomicAdd(&sh[e * 3 + 2], (double)w);
    } else {
      atomicAdd(&xsum[e * 2], xr); atomicAdd(&xsum[e * 2 + 1], xi); atomicAdd(&wsum[e], (double)w);
    }
  }
  if (use_smem) {
    __syncthreads();
    for (int e = threadIdx.x; e < nent; e += blockDim.x) {
      if (sh[e * 3 + 2] != 0.0) {
        atomicAdd(&xsum[e * 2], sh[e * 3]); atomicAdd(&xsum[e * 2 + 1], sh[e * 3 + 1]); atomicAdd(&wsum[e], sh[e * 3 + 2]);
      }
    }
  }
}

// One CTA; thread a < nant owns antenna a.  Shared: the gains of iteration k (complex double) and the largest change.
__global__ void __launch_bounds__(1024)
lra_gain_solve_kernel(int nant, int nbl, int ncorr, const int32_t* __restrict__ ant1, const int32_t* __restrict__ ant2,
                      const double* __restrict__ xsum, const double* __restrict__ wsum, double alpha, double delta, int max_iter,
                      double* __restrict__ gains, int32_t* __restrict__ iters) {
  extern __shared__ double g[];          // [nant][2]
  __shared__ double change_sh[32];
  __shared__ int stop;
  const int a = threadIdx.x;
  int worst = 0;
  for (int p = 0; p < ncorr; ++p) {
    if (a < nant) { g[2 * a] = gains[(a * ncorr + p) * 2]; g[2 * a + 1] = gains[(a * ncorr + p) * 2 + 1]; }
    if (a == 0) stop = 0;
    __syncthreads();
    int k = 0;
    for (; k < max_iter; ++k) {
      double nr = 0.0, ni = 0.0, den = 0.0;
      if (a < nant) {
        for (int b = 0; b < nbl; ++b) {           // baselines in list order: the summation order of the definition
          const int i = ant1[b], j = ant2[b];
          if (i != a && j != a) continue;
          const double w = wsum[b * ncorr + p];
          if (!(w > 0.0)) continue;
          const double xr = xsum[(b * ncorr + p) * 2] / w, xi = xsum[(b * ncorr + p) * 2 + 1] / w;
          if (i == a) {                            // g_j X_ij w
            const double gr = g[2 * j], gi = g[2 * j + 1];
            nr += (gr * xr - gi * xi) * w; ni += (gr * xi + gi * xr) * w; den += (gr * gr + gi * gi) * w;
          }
          if (j == a) {                            // g_i conj(X_ij) w
            const double gr = g[2 * i], gi = g[2 * i + 1];
            nr += (gr * xr + gi * xi) * w; ni += (gi * xr - gr * xi) * w; den += (gr * gr + gi * gi) * w;
          }
        }
      }
      __syncthreads();                             // every thread has read the gains of iteration k
      double d = 0.0;
      if (a < nant && den > 0.0) {
        const double r1 = (1.0 - alpha) * g[2 * a] + alpha * (nr / den), i1 = (1.0 - alpha) * g[2 * a + 1] + alpha * (ni / den);
        d = hypot(r1 - g[2 * a], i1 - g[2 * a + 1]);
        g[2 * a] = r1; g[2 * a + 1] = i1;
      }
      for (int o = 16; o > 0; o >>= 1) d = fmax(d, __shfl_xor_sync(0xffffffffu, d, o));
      if ((threadIdx.x & 31) == 0) change_sh[threadIdx.x >> 5] = d;
      __syncthreads();
      if (a == 0) {
        double m = 0.0;
        for (int w = 0; w < (int)((blockDim.x + 31) >> 5); ++w) m = fmax(m, change_sh[w]);
        stop = m < delta;
      }
      __syncthreads();
      if (stop) { ++k; break; }
    }
    if (k > worst) worst = k;
    if (a < nant) { gains[(a * ncorr + p) * 2] = g[2 * a]; gains[(a * ncorr + p) * 2 + 1] = g[2 * a + 1]; }
    __syncthreads();
  }
  if (a == 0 && iters) *iters = worst;
}

static int lra_gain_cuda(cudaError_t e) { return e == cudaSuccess ? LRA_OK : e == cudaErrorMemoryAllocation ? LRA_ENOMEM : LRA_ECUDA; }

extern "C" int lra_gain_accumulate(int32_t device, void* stream, int64_t nrow, int32_t nchan, int32_t ncorr, int32_t nbl,
                                   const int32_t* bl_index, const void* vis_c64, const void* model_c64, const float* wt,
                                   double* xsum, double* wsum) {
  if (nrow < 0 || nchan < 1 || ncorr < 1 || ncorr > 4 || nbl < 1 || !xsum || !wsum) return LRA_EINVAL;
  if (nrow > 0 && (!vis_c64 || !model_c64 || !wt)) return LRA_EINVAL;
  int rc = lra_gain_cuda(cudaSetDevice(device));
  if (rc || nrow == 0) return rc;
  int sms = 0;
  if ((rc = lra_gain_cuda(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device)))) return rc;
  const long long n = (long long)nrow * nchan * ncorr;
  long long blocks = (n + 255) / 256;
  if (blocks > sms * 8LL) blocks = sms * 8LL;
  lra_gain_accumulate_kernel<<<(int)blocks, 256, 0, (cudaStream_t)stream>>>(n, nchan, ncorr, nbl, bl_index, (const float2*)vis_c64,
                                                                           (const float2*)model_c64, wt, xsum, wsum,
                                                                           nbl * ncorr <= LRA_GAIN_SMEM_ENTRIES);
  return lra_gain_cuda(cudaGetLastError());
}

extern "C" int lra_gain_solve(int32_t device, void* stream, int32_t nant, int32_t nbl, int32_t ncorr, const int32_t* ant1,
                              const int32_t* ant2, const double* xsum, const double* wsum, double alpha, double delta,
                              int32_t max_iter, double* gains, int32_t* iters) {
  if (nant < 1 || nant > 1024 || nbl < 1 || ncorr < 1 || ncorr > 4 || !ant1 || !ant2 || !xsum || !wsum || !gains || max_iter < 0)
    return LRA_EINVAL;
  int rc = lra_gain_cuda(cudaSetDevice(device));
  if (rc) return rc;
  const int threads = (nant + 31) / 32 * 32;
  lra_gain_solve_kernel<<<1, threads, (size_t)nant * 2 * sizeof(double), (cudaStream_t)stream>>>(nant, nbl, ncorr, ant1, ant2, xsum, wsum,
                                                                                               alpha, delta, max_iter, gains, iters);
  return lra_gain_cuda(cudaGetLastError());
}

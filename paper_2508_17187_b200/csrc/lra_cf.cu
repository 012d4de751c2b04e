// lra_cf.cu -- on-device construction of the CF table (the paper's PreCompute /
// ConvFunc / CFCache role; Table 1):
//   lra_cf_generate : for every requested kernel, the product of the terms that are ON in the image plane
//                     (PS taper x A-term x W-term), its Fourier transform at the (S os)^2 oversampled uv samples of the
//                     storage convention of lra.h ("FFT, crop"), normalised to sum os^2, written as complex64 into the
//                     caller's device table -- the table lra_plan_create takes.
// Readings R24-R26.
//
// Only the (S os)^2 samples that are kept are computed: sample j of an axis is bin (j - c0) of the n_img*os-point DFT of
// the zero-padded image, so the transform is two small dense contractions per kernel,
//     T[m][i] = sum_l img[m][l] E[i][l],     K[j][i] = sum_m T[m][i] E[j][m],     E[j][a] = e^{-2 pi i off_j (a - n/2)/n},
// instead of a padded FFT of (n_img os)^2 points of which (S/n_img)^2 would survive the crop.  Arithmetic is fp64
// throughout (phases by sincospi of an exactly reduced argument): the table is built once, and its float32 samples are then
// exact roundings of the definition rather than carrying the error of a float32 transform.  One phase table serves every
// support: off depends on (j - h os) only, so the table is indexed by q = j + (h_max - h) os.
// Product code: shares nothing with oracle/.
#include <algorithm>
#include <vector>

#include <nvtx3/nvToolsExt.h>

#include "lra_internal.cuh"

namespace {

constexpr int LRA_CF_TI = 128;   // threads per block, along the fast uv sample index i
constexpr int LRA_CF_TR = 4;     // rows (m or j) per thread: one table load feeds four accumulators

struct lra_cf_item {   // one kernel of the batch
  double w;            // wavelengths
  long long out;       // element offset into cf_data
  int support, aterm;  // aterm < 0: OFF
};

// Et[a][q] = e^{-2 pi i ((q - c0max)/os) (a - n/2) / n}, a-major so that neighbouring samples are neighbouring words
__global__ void __launch_bounds__(256) lra_cf_phase_kernel(double2* __restrict__ Et, int n, int os, int nq, int c0max) {
  const int total = n * nq;
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < total; e += gridDim.x * blockDim.x) {
    const int a = e / nq, q = e - a * nq;
    // turns = (q - c0max)(a - n/2) / (os n): reduce the integer numerator mod (os n) exactly before dividing
    const long long den = (long long)os * n;
    long long num = ((long long)(q - c0max) * (a - n / 2)) % den;
    double s, c;
    sincospi(-2.0 * (double)num / (double)den, &s, &c);
    Et[e] = make_double2(c, s);
  }
}

// img[b][m][l] = taper[l] taper[m] A[m][l] e^{2 pi i w (sqrt(1 - l^2 - m^2) - 1)}
__global__ void __launch_bounds__(256)
lra_cf_image_kernel(const lra_cf_item* __restrict__ items, const double* __restrict__ taper, const float2* __restrict__ aterm,
                    double2* __restrict__ img, int n, double fov) {
  const lra_cf_item it = items[blockIdx.y];
  double2* out = img + (size_t)blockIdx.y * n * n;
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n * n; e += gridDim.x * blockDim.x) {
    const int m = e / n, l = e - m * n;
    const double ll = (double)(l - n / 2) * fov / n, mm = (double)(m - n / 2) * fov / n;
    const double r2 = ll * ll + mm * mm;
    const double nterm = sqrt(r2 < 1.0 ? 1.0 - r2 : 0.0) - 1.0;
    double s, c;
    sincospi(2.0 * it.w * nterm, &s, &c);
    if (taper) { const double t = taper[l] * taper[m]; c *= t; s *= t; }
    if (it.aterm >= 0) {
      const float2 a = aterm[(size_t)it.aterm * n * n + e];
      const double t = c * (double)a.x - s * (double)a.y;
      s = c * (double)a.y + s * (double)a.x;
      c = t;
    }
    out[e] = make_double2(c, s);
  }
}

__device__ __forceinline__ void lra_cmac(double2& acc, const double2 a, const double2 b) {
  acc.x += a.x * b.x - a.y * b.y;
  acc.y += a.x * b.y + a.y * b.x;
}

// T[b][m][i] = sum_l img[b][m][l] Et[l][q0 + i];  block: LRA_CF_TI samples i x LRA_CF_TR rows m; img rows staged in smem
__global__ void __launch_bounds__(LRA_CF_TI)
lra_cf_rows_kernel(const lra_cf_item* __restrict__ items, const double2* __restrict__ img, const double2* __restrict__ Et,
                   double2* __restrict__ T, int n, int os, int nq, int hmax, int so_max) {
  extern __shared__ double2 lra_cf_smem[];
  const lra_cf_item it = items[blockIdx.z];
  const int so = it.support * os, q0 = (hmax - (it.support - 1) / 2) * os;
  const int i = blockIdx.x * LRA_CF_TI + threadIdx.x, m0 = blockIdx.y * LRA_CF_TR;
  if (blockIdx.x * LRA_CF_TI >= so) return;
  const double2* src = img + ((size_t)blockIdx.z * n + m0) * n;
  const int rows = min(LRA_CF_TR, n - m0);
  for (int e = threadIdx.x; e < rows * n; e += LRA_CF_TI) lra_cf_smem[e] = src[e];
  __syncthreads();
  if (i >= so) return;
  double2 acc[LRA_CF_TR];
#pragma unroll
  for (int r = 0; r < LRA_CF_TR; ++r) acc[r] = make_double2(0.0, 0.0);
  for (int l = 0; l < n; ++l) {
    const double2 e = Et[(size_t)l * nq + q0 + i];
#pragma unroll
    for (int r = 0; r < LRA_CF_TR; ++r)
      if (r < rows) lra_cmac(acc[r], lra_cf_smem[r * n + l], e);
  }
#pragma unroll
  for (int r = 0; r < LRA_CF_TR; ++r)
    if (r < rows) T[((size_t)blockIdx.z * n + m0 + r) * so_max + i] = acc[r];
}

// Kd[b][j][i] = sum_m T[b][m][i] Et[m][q0 + j];  block: LRA_CF_TI samples i x LRA_CF_TR rows j; the rows' phases in smem.
// Also writes the block's partial sum of its samples (summed in a fixed order) for the normalisation.
__global__ void __launch_bounds__(LRA_CF_TI)
lra_cf_cols_kernel(const lra_cf_item* __restrict__ items, const double2* __restrict__ T, const double2* __restrict__ Et,
                   double2* __restrict__ Kd, double2* __restrict__ partial, int n, int os, int nq, int hmax, int so_max) {
  extern __shared__ double2 lra_cf_smem[];
  __shared__ double2 red[LRA_CF_TI];
  const lra_cf_item it = items[blockIdx.z];
  const int so = it.support * os, q0 = (hmax - (it.support - 1) / 2) * os;
  const int i = blockIdx.x * LRA_CF_TI + threadIdx.x, j0 = blockIdx.y * LRA_CF_TR;
  const int slot = (blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
  if (blockIdx.x * LRA_CF_TI >= so || j0 >= so) {
    if (threadIdx.x == 0) partial[slot] = make_double2(0.0, 0.0);
    return;
  }
  const int rows = min(LRA_CF_TR, so - j0);
  for (int e = threadIdx.x; e < rows * n; e += LRA_CF_TI) {
    const int r = e / n, m = e - r * n;
    lra_cf_smem[e] = Et[(size_t)m * nq + q0 + j0 + r];
  }
  __syncthreads();
  double2 acc[LRA_CF_TR];
#pragma unroll
  for (int r = 0; r < LRA_CF_TR; ++r) acc[r] = make_double2(0.0, 0.0);
  if (i < so) {
    const double2* t = T + (size_t)blockIdx.z * n * so_max + i;
    for (int m = 0; m < n; ++m) {
      const double2 v = t[(size_t)m * so_max];
#pragma unroll
      for (int r = 0; r < LRA_CF_TR; ++r)
        if (r < rows) lra_cmac(acc[r], v, lra_cf_smem[r * n + m]);
    }
#pragma unroll
    for (int r = 0; r < LRA_CF_TR; ++r)
      if (r < rows) Kd[((size_t)blockIdx.z * so_max + j0 + r) * so_max + i] = acc[r];
  }
  double2 s = make_double2(0.0, 0.0);
#pragma unroll
  for (int r = 0; r < LRA_CF_TR; ++r) { s.x += acc[r].x; s.y += acc[r].y; }   // rows past the end hold 0
  red[threadIdx.x] = s;
  __syncthreads();
  for (int w = LRA_CF_TI / 2; w > 0; w >>= 1) {
    if (threadIdx.x < w) { red[threadIdx.x].x += red[threadIdx.x + w].x; red[threadIdx.x].y += red[threadIdx.x + w].y; }
    __syncthreads();
  }
  if (threadIdx.x == 0) partial[slot] = red[0];
}

// cf_data[out + j so + i] = (float2)(Kd[b][j][i] * os^2 / sum(Kd[b]))
__global__ void __launch_bounds__(256)
lra_cf_finish_kernel(const lra_cf_item* __restrict__ items, const double2* __restrict__ Kd, const double2* __restrict__ partial,
                     int nparts, float2* __restrict__ cf_data, int os, int so_max, int normalise, int* __restrict__ bad) {
  __shared__ double2 red[256];
  const lra_cf_item it = items[blockIdx.y];
  const int so = it.support * os;
  double2 f = make_double2(1.0, 0.0);
  if (normalise) {
    double2 s = make_double2(0.0, 0.0);
    for (int e = threadIdx.x; e < nparts; e += 256) {   // same partition and order in every block: one value per kernel
      const double2 v = partial[(size_t)blockIdx.y * nparts + e];
      s.x += v.x; s.y += v.y;
    }
    red[threadIdx.x] = s;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
      if (threadIdx.x < w) { red[threadIdx.x].x += red[threadIdx.x + w].x; red[threadIdx.x].y += red[threadIdx.x + w].y; }
      __syncthreads();
    }
    const double2 t = red[0];
    const double d = t.x * t.x + t.y * t.y;
    if (d == 0.0 || !(d == d)) {
      if (threadIdx.x == 0 && blockIdx.x == 0) atomicExch(bad, 1);
      return;
    }
    f = make_double2((double)os * os * t.x / d, -(double)os * os * t.y / d);
  }
  const double2* src = Kd + (size_t)blockIdx.y * so_max * so_max;
  float2* dst = cf_data + it.out;
  for (int e = blockIdx.x * 256 + threadIdx.x; e < so * so; e += gridDim.x * 256) {
    const int j = e / so, i = e - j * so;
    const double2 v = src[(size_t)j * so_max + i];
    dst[e] = make_float2((float)(v.x * f.x - v.y * f.y), (float)(v.x * f.y + v.y * f.x));
  }
}

struct lra_cf_buffers {
  void* ptr[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  ~lra_cf_buffers() { for (void* q : ptr) if (q) cudaFree(q); }
};

}  // namespace

static thread_local cudaError_t lra_cf_last_err = cudaSuccess;

extern "C" int lra_cf_last_cuda_error(void) { return (int)lra_cf_last_err; }

extern "C" int lra_cf_generate(const lra_cf_desc* d, void* cf_data) {
  nvtxRangePushA("lra_cf_generate");
  struct pop { ~pop() { nvtxRangePop(); } } nvtx_;
  if (!d || !cf_data) return LRA_EINVAL;
  if (d->n_img < 2 || d->n_img > 512 || d->oversampling < 1 || d->oversampling > 64) return LRA_EINVAL;
  if (!(d->fov_rad > 0.0) || d->n_cf < 1 || d->n_cf > (1 << 24) || !d->cf_support || !d->cf_offset) return LRA_EINVAL;
  if (d->n_aterm < 0 || (d->n_aterm > 0 && !d->aterm) || (d->cf_aterm && d->n_aterm < 1)) return LRA_EINVAL;
  const int n = d->n_img, os = d->oversampling;
  int smax = 1;
  for (int c = 0; c < d->n_cf; ++c) {
    const int S = d->cf_support[c];
    if (S < 1 || S > 129 || (S & 1) == 0 || d->cf_offset[c] < 0) return LRA_EINVAL;
    if (d->cf_aterm && (d->cf_aterm[c] < 0 || d->cf_aterm[c] >= d->n_aterm)) return LRA_EINVAL;
    if (d->cf_w && !(d->cf_w[c] == d->cf_w[c])) return LRA_EINVAL;
    smax = std::max(smax, S);
  }
  const int hmax = (smax - 1) / 2, nq = smax * os, c0max = hmax * os + (os - 1 - os / 2), so_max = nq;
  cudaStream_t st = (cudaStream_t)d->stream;
#define CK(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { lra_cf_last_err = e__; \
    return e__ == cudaErrorMemoryAllocation ? LRA_ENOMEM : LRA_ECUDA; } } while (0)
  CK(cudaSetDevice(d->device));
  // batch size: bound the fp64 work buffers (image, T, K) to about 256 MB
  const size_t per_cf = ((size_t)n * n + (size_t)n * so_max + (size_t)so_max * so_max) * sizeof(double2);
  int batch = (int)std::max<size_t>(1, std::min<size_t>((size_t)d->n_cf, ((size_t)256 << 20) / per_cf));
  batch = std::min(batch, 65535);
  const int gx = (so_max + LRA_CF_TI - 1) / LRA_CF_TI, gy_rows = (n + LRA_CF_TR - 1) / LRA_CF_TR,
            gy_cols = (so_max + LRA_CF_TR - 1) / LRA_CF_TR, nparts = gx * gy_cols;
  lra_cf_buffers buf;
  double2 *Et, *img, *T, *Kd, *partial;
  lra_cf_item* items;
  int* bad;
  CK(cudaMalloc(&buf.ptr[0], (size_t)n * nq * sizeof(double2)));
  CK(cudaMalloc(&buf.ptr[1], (size_t)batch * n * n * sizeof(double2)));
  CK(cudaMalloc(&buf.ptr[2], (size_t)batch * n * so_max * sizeof(double2)));
  CK(cudaMalloc(&buf.ptr[3], (size_t)batch * so_max * so_max * sizeof(double2)));
  CK(cudaMalloc(&buf.ptr[4], (size_t)batch * nparts * sizeof(double2)));
  CK(cudaMalloc(&buf.ptr[5], (size_t)d->n_cf * sizeof(lra_cf_item) + sizeof(int)));
  Et = (double2*)buf.ptr[0]; img = (double2*)buf.ptr[1]; T = (double2*)buf.ptr[2]; Kd = (double2*)buf.ptr[3];
  partial = (double2*)buf.ptr[4]; items = (lra_cf_item*)buf.ptr[5];
  bad = (int*)(items + d->n_cf);
  std::vector<lra_cf_item> h(d->n_cf);
  for (int c = 0; c < d->n_cf; ++c) {
    h[c].w = d->cf_w ? d->cf_w[c] : 0.0;
    h[c].out = d->cf_offset[c];
    h[c].support = d->cf_support[c];
    h[c].aterm = d->n_aterm > 0 ? (d->cf_aterm ? d->cf_aterm[c] : 0) : -1;
  }
  CK(cudaMemcpyAsync(items, h.data(), (size_t)d->n_cf * sizeof(lra_cf_item), cudaMemcpyHostToDevice, st));
  CK(cudaMemsetAsync(bad, 0, sizeof(int), st));
  lra_cf_phase_kernel<<<std::min((n * nq + 255) / 256, 1184), 256, 0, st>>>(Et, n, os, nq, c0max);
  CK(cudaGetLastError());
  const size_t smem = (size_t)LRA_CF_TR * n * sizeof(double2);
  for (int c0 = 0; c0 < d->n_cf; c0 += batch) {
    const int nb = std::min(batch, d->n_cf - c0);
    lra_cf_image_kernel<<<dim3(std::min((n * n + 255) / 256, 64), nb), 256, 0, st>>>(items + c0, (const double*)d->taper,
                                                                                     (const float2*)d->aterm, img, n, d->fov_rad);
    lra_cf_rows_kernel<<<dim3(gx, gy_rows, nb), LRA_CF_TI, smem, st>>>(items + c0, img, Et, T, n, os, nq, hmax, so_max);
    lra_cf_cols_kernel<<<dim3(gx, gy_cols, nb), LRA_CF_TI, smem, st>>>(items + c0, T, Et, Kd, partial, n, os, nq, hmax, so_max);
    lra_cf_finish_kernel<<<dim3(std::min((so_max * so_max + 255) / 256, 32), nb), 256, 0, st>>>(
        items + c0, Kd, partial, nparts, (float2*)cf_data, os, so_max, d->normalise, bad);
    CK(cudaGetLastError());
  }
  int hbad = 0;
  CK(cudaMemcpyAsync(&hbad, bad, sizeof(int), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));   // the work buffers are freed on return
#undef CK
  return hbad ? LRA_EINVAL : LRA_OK;
}

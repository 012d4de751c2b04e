// lra_image.cu -- the transforms either side of the gridding path:
//   lra_image      : I^R = F^dagger of the gridded data (Eq. 23; "UpdateDir") with the
//                    image-plane taper correction and the sum-of-weights normalisation
//   lra_model_grid : F of a model image onto the uv grid (the input of lra_degrid; Eq. 6 / Eq. 23)
// Readings R17-R19: centred DFT, e^{+} towards the image, no 1/N, separable correction factor.
//
// The transform itself is cuFFT C2C (a plain library FFT, as SURVEY Sec. 8(f) specifies).  The centring costs no
// data movement: for even n,  e^{+-2 pi i (x - n/2)(l - n/2)/n} = (-1)^(n/2) (-1)^x (-1)^l e^{+-2 pi i x l / n},  so the
// library's own kernels multiply by (-1)^(x+y) on the way in and by (-1)^(l+m) (-1)^(nx/2 + ny/2) on the way out, fused
// with the real part / correction / normalisation (lra_image) or with the correction (lra_model_grid).  HBM-bound:
// 8 + 8 bytes per pixel in, 8 + 4 out around the FFT.
// Product code: shares nothing with oracle/.
#include <cufft.h>

#include "lra_internal.cuh"

// work[g][y][x] = (-1)^(x+y) * grid[g][y][x]
__global__ void __launch_bounds__(256)
lra_image_pre_kernel(const float2* __restrict__ grid, float2* __restrict__ work, int nx, long long n) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const long long r = i / nx;                    // g*ny + y; ny is even, so its parity is y's
    const float s = (((i - r * nx) + r) & 1) ? -1.f : 1.f;
    const float2 v = grid[i];
    work[i] = make_float2(s * v.x, s * v.y);
  }
}

// image[g][m][l] = sign * (-1)^(l+m) * Re(work[g][m][l]) * corr_x[l] * corr_y[m] / sumwt[g]
__global__ void __launch_bounds__(256)
lra_image_post_kernel(const float2* __restrict__ work, const double* __restrict__ sumwt, const float* __restrict__ corr_x,
                      const float* __restrict__ corr_y, float* __restrict__ image, int nx, int ny, long long n, float sign) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const long long r = i / nx;
    const int l = (int)(i - r * nx), m = (int)(r % ny), g = (int)(r / ny);
    float f = ((l + m) & 1) ? -sign : sign;
    if (corr_x) f *= corr_x[l];
    if (corr_y) f *= corr_y[m];
    float v = work[i].x * f;
    if (sumwt) v = (float)((double)v / sumwt[g]);
    image[i] = v;
  }
}

// work[g][m][l] = (-1)^(l+m) * image[g][m][l] * corr_x[l] * corr_y[m]
__global__ void __launch_bounds__(256)
lra_model_pre_kernel(const float* __restrict__ image, const float* __restrict__ corr_x, const float* __restrict__ corr_y,
                     float2* __restrict__ work, int nx, int ny, long long n) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const long long r = i / nx;
    const int l = (int)(i - r * nx), m = (int)(r % ny);
    float f = ((l + m) & 1) ? -1.f : 1.f;
    if (corr_x) f *= corr_x[l];
    if (corr_y) f *= corr_y[m];
    work[i] = make_float2(image[i] * f, 0.f);
  }
}

// grid[g][y][x] = sign * (-1)^(x+y) * work[g][y][x]
__global__ void __launch_bounds__(256)
lra_model_post_kernel(const float2* __restrict__ work, float2* __restrict__ grid, int nx, long long n, float sign) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const long long r = i / nx;
    const float s = (((i - r * nx) + r) & 1) ? -sign : sign;
    const float2 v = work[i];
    grid[i] = make_float2(s * v.x, s * v.y);
  }
}

static int lra_fft_setup(lra_plan* p) {
  if (p->fft_ready) return LRA_OK;
  if ((p->nx & 1) || (p->ny & 1)) return LRA_EINVAL;
  const int ng = p->ncorr * p->nterms;
  const size_t n = (size_t)ng * p->nx * p->ny;
  if (!p->fft_work) LRA_CUDA(p, cudaMalloc(&p->fft_work, n * sizeof(float2)));
  cufftHandle h;
  int dims[2] = {p->ny, p->nx};
  if (cufftPlanMany(&h, 2, dims, nullptr, 1, p->nx * p->ny, nullptr, 1, p->nx * p->ny, CUFFT_C2C, ng) != CUFFT_SUCCESS) {
    p->last_err = cudaErrorUnknown;
    return LRA_ECUDA;
  }
  if (cufftSetStream(h, p->stream) != CUFFT_SUCCESS) { cufftDestroy(h); p->last_err = cudaErrorUnknown; return LRA_ECUDA; }
  p->fft_plan = (int)h;
  p->fft_ready = true;
  return LRA_OK;
}

void lra_fft_release(lra_plan* p) {
  if (p->fft_ready) cufftDestroy((cufftHandle)p->fft_plan);
  p->fft_ready = false;
  if (p->fft_work) cudaFree(p->fft_work);
  p->fft_work = nullptr;
}

extern "C" int lra_image(lra_plan* p, const void* grid_c64, const double* sumwt, const float* corr_x, const float* corr_y,
                         float* image) {
  if (!p || !grid_c64 || !image) return LRA_EINVAL;
  LRA_CUDA(p, cudaSetDevice(p->device));
  int rc = lra_fft_setup(p);
  if (rc) return rc;
  const long long n = (long long)p->ncorr * p->nterms * p->nx * p->ny;
  const int blocks = p->sm_count * 8;
  lra_image_pre_kernel<<<blocks, 256, 0, p->stream>>>((const float2*)grid_c64, p->fft_work, p->nx, n);
  LRA_LAUNCH_CHECK(p);
  if (cufftExecC2C((cufftHandle)p->fft_plan, (cufftComplex*)p->fft_work, (cufftComplex*)p->fft_work, CUFFT_INVERSE) != CUFFT_SUCCESS) {
    p->last_err = cudaErrorUnknown;
    return LRA_ECUDA;
  }
  const float sign = (((p->nx / 2) + (p->ny / 2)) & 1) ? -1.f : 1.f;
  lra_image_post_kernel<<<blocks, 256, 0, p->stream>>>(p->fft_work, sumwt, corr_x, corr_y, image, p->nx, p->ny, n, sign);
  LRA_LAUNCH_CHECK(p);
  return LRA_OK;
}

extern "C" int lra_model_grid(lra_plan* p, const float* image, const float* corr_x, const float* corr_y, void* grid_c64) {
  if (!p || !grid_c64 || !image) return LRA_EINVAL;
  LRA_CUDA(p, cudaSetDevice(p->device));
  int rc = lra_fft_setup(p);
  if (rc) return rc;
  const long long n = (long long)p->ncorr * p->nterms * p->nx * p->ny;
  const int blocks = p->sm_count * 8;
  lra_model_pre_kernel<<<blocks, 256, 0, p->stream>>>(image, corr_x, corr_y, p->fft_work, p->nx, p->ny, n);
  LRA_LAUNCH_CHECK(p);
  if (cufftExecC2C((cufftHandle)p->fft_plan, (cufftComplex*)p->fft_work, (cufftComplex*)p->fft_work, CUFFT_FORWARD) != CUFFT_SUCCESS) {
    p->last_err = cudaErrorUnknown;
    return LRA_ECUDA;
  }
  const float sign = (((p->nx / 2) + (p->ny / 2)) & 1) ? -1.f : 1.f;
  lra_model_post_kernel<<<blocks, 256, 0, p->stream>>>(p->fft_work, (float2*)grid_c64, p->nx, n, sign);
  LRA_LAUNCH_CHECK(p);
  return LRA_OK;
}

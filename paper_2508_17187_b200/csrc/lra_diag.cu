// lra_diag.cu -- roofline denominators measured on the device the plan runs on (the FP32 FMA
// peak is measured with an FMA-only microbenchmark because MEASURED_PEAKS.json has no FP32 entry) and the
// L2 -> SM read bandwidth that bounds CF-slab traffic.  Measurement aids only; not on the hot path.
#include "lra_internal.cuh"

__global__ void __launch_bounds__(1024, 2) lra_diag_fma_kernel(float* out, int iters, float a, float b) {
  float x[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) x[i] = (float)(threadIdx.x + i);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
      for (int i = 0; i < 16; ++i) x[i] = fmaf(x[i], a, b);
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += x[i];
  if (s == 12345.678f) out[0] = s;
}

__global__ void __launch_bounds__(1024, 2) lra_diag_l2_kernel(const float4* __restrict__ buf, size_t n_vec, int reps, float* out) {
  float s = 0.f;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (int r = 0; r < reps; ++r)
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n_vec; i += stride) {
      float4 v = __ldg(buf + i);
      s += v.x + v.y + v.z + v.w;
    }
  if (s == 12345.678f) out[0] = s;
}

// FP32 FMA throughput in TFLOP/s (2 flop per FMA), best of `trials`.
extern "C" int lra_diag_fma_tflops(int device, double* tflops) {
  if (!tflops) return LRA_EINVAL;
  if (cudaSetDevice(device) != cudaSuccess) return LRA_ECUDA;
  int sms = 0;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
  float* out = nullptr;
  if (cudaMalloc(&out, 4) != cudaSuccess) return LRA_ENOMEM;
  cudaEvent_t a, b;
  cudaEventCreate(&a); cudaEventCreate(&b);
  const int iters = 4096;
  double best = 0.0;
  for (int t = 0; t < 5; ++t) {
    cudaEventRecord(a);
    lra_diag_fma_kernel<<<sms * 2, 1024>>>(out, iters, 1.0000001f, 1e-9f);
    cudaEventRecord(b);
    if (cudaEventSynchronize(b) != cudaSuccess) { cudaFree(out); return LRA_ECUDA; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    double fl = 2.0 * (double)sms * 2 * 1024 * (double)iters * 8 * 16;
    double tf = fl / (ms * 1e-3) / 1e12;
    if (tf > best) best = tf;
  }
  cudaEventDestroy(a); cudaEventDestroy(b);
  cudaFree(out);
  *tflops = best;
  return LRA_OK;
}

// Read bandwidth of an L2-resident buffer (`mbytes` MiB, read `reps` times by all SMs) in GB/s.
extern "C" int lra_diag_l2_gbs(int device, int mbytes, double* gbs) {
  if (!gbs || mbytes < 1) return LRA_EINVAL;
  if (cudaSetDevice(device) != cudaSuccess) return LRA_ECUDA;
  int sms = 0;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
  size_t bytes = (size_t)mbytes << 20;
  float4* buf = nullptr;
  float* out = nullptr;
  if (cudaMalloc(&buf, bytes) != cudaSuccess || cudaMalloc(&out, 4) != cudaSuccess) { cudaFree(buf); return LRA_ENOMEM; }
  cudaMemset(buf, 0, bytes);
  cudaEvent_t a, b;
  cudaEventCreate(&a); cudaEventCreate(&b);
  const int reps = 20;
  double best = 0.0;
  for (int t = 0; t < 4; ++t) {
    cudaEventRecord(a);
    lra_diag_l2_kernel<<<sms * 2, 1024>>>(buf, bytes / 16, reps, out);
    cudaEventRecord(b);
    if (cudaEventSynchronize(b) != cudaSuccess) { cudaFree(buf); cudaFree(out); return LRA_ECUDA; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    double g = (double)bytes * reps / (ms * 1e-3) / 1e9;
    if (t > 0 && g > best) best = g;
  }
  cudaEventDestroy(a); cudaEventDestroy(b);
  cudaFree(buf); cudaFree(out);
  *gbs = best;
  return LRA_OK;
}

// peaks.cu — the two issue-rate peaks the blend kernels' roofline is quoted against, MEASURED on the device the
// bench runs on ("both must be confirmed by a 20-line FMA-chain / ex2 micro-benchmark on the box"):
//   FP32 lane-instructions per second (independent FFMA chains, all four sub-partitions of every SM busy), and
//   MUFU operations per second (independent ex2.approx chains).
// Not part of the hot path: satsplat_measure_peaks synchronises the device and is called once by bench.py.
#include "internal.cuh"

namespace satsplat {

constexpr int kPeakChains = 8;      // independent dependency chains per thread (FFMA latency 4 cycles, 2 warps/scheduler suffice)
constexpr int kPeakThreads = 256;
constexpr int kPeakCtasPerSm = 8;   // 2048 threads per SM

__global__ void __launch_bounds__(kPeakThreads) peak_fma_kernel(float* out, int iters, float a, float b) {
  float x[kPeakChains];
#pragma unroll
  for (int k = 0; k < kPeakChains; ++k) x[k] = (float)(threadIdx.x + k) * 1e-3f;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u)
#pragma unroll
      for (int k = 0; k < kPeakChains; ++k) x[k] = __fmaf_rn(x[k], a, b);
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < kPeakChains; ++k) s += x[k];
  if (s == 12345.678f) out[0] = s;   // never true: keeps the chains alive
}

__global__ void __launch_bounds__(kPeakThreads) peak_ex2_kernel(float* out, int iters) {
  float x[kPeakChains];
#pragma unroll
  for (int k = 0; k < kPeakChains; ++k) x[k] = (float)(threadIdx.x + k) * 1e-3f;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u)
#pragma unroll
      for (int k = 0; k < kPeakChains; ++k) x[k] = fast_exp2(-x[k]);   // x in [0, 1] -> 2^-x in [0.5, 1]: bounded
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < kPeakChains; ++k) s += x[k];
  if (s == 12345.678f) out[0] = s;
}

}  // namespace satsplat

using namespace satsplat;

extern "C" int satsplat_measure_peaks(int device, double* fp32_lane_inst_per_s, double* mufu_per_s, int* sm_count) {
  if (!fp32_lane_inst_per_s || !mufu_per_s) return SATSPLAT_E_INVALID;
  if (cudaSetDevice(device) != cudaSuccess) return SATSPLAT_E_CUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return SATSPLAT_E_CUDA;
  if (sm_count) *sm_count = prop.multiProcessorCount;
  float* d = nullptr;
  cudaEvent_t e0, e1;
  if (cudaMalloc(&d, 256) != cudaSuccess) return SATSPLAT_E_CUDA;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  const int grid = prop.multiProcessorCount * kPeakCtasPerSm;
  double best[2] = {0.0, 0.0};
  for (int which = 0; which < 2; ++which) {
    const int iters = which == 0 ? 4096 : 1024;
    for (int rep = 0; rep < 5; ++rep) {   // first repetition warms up the clocks; best of the rest
      cudaEventRecord(e0, 0);
      if (which == 0)
        peak_fma_kernel<<<grid, kPeakThreads>>>(d, iters, 0.999f, 1e-3f);
      else
        peak_ex2_kernel<<<grid, kPeakThreads>>>(d, iters);
      cudaEventRecord(e1, 0);
      if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(d); return SATSPLAT_E_CUDA; }
      float ms = 0.f;
      cudaEventElapsedTime(&ms, e0, e1);
      const double ops = (double)grid * kPeakThreads * (double)iters * 8.0 * kPeakChains;
      if (rep > 0 && ms > 0.f) best[which] = fmax(best[which], ops / (ms * 1e-3));
    }
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d);
  *fp32_lane_inst_per_s = best[0];
  *mufu_per_s = best[1];
  return cudaGetLastError() == cudaSuccess ? SATSPLAT_OK : SATSPLAT_E_CUDA;
}

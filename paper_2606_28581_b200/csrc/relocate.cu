// relocate.cu — (f3, second half) relocation of dead surfels onto live ones (PAPER.md:200 cites the 3DGS-MCMC strategy [22]).
//   dead = opacity <= o_min; every dead surfel draws a live source with probability proportional to opacity (inverse
//   transform on the double-precision cumulative sum of the live opacities, the caller's uniform numbers); a source drawn by
//   n - 1 dead surfels is split into n copies of opacity o' = 1 - (1 - alpha)^(1/n) whose scales are multiplied by alpha / D,
//   D = sum_{i=1..n} sum_{k<i} C(i-1,k) (-1)^k o'^(k+1) / sqrt(k+1): n copies composited at the centre give alpha back and the
//   composited profile through the centre keeps its integral.  The Adam state of every touched surfel is cleared.
// Runs every few hundred iterations; HBM/latency-bound, five small kernels + the cumulative sum.
#include "internal.cuh"

namespace satsplat {

__global__ void __launch_bounds__(256) reloc_weights_kernel(long long N, const float* __restrict__ logits, float logit_min,
                                                            double* __restrict__ w, uint32_t* __restrict__ count,
                                                            int32_t* __restrict__ src) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const float l = logits[i];
  const bool dead = l <= logit_min;                      // alpha <= o_min, decided on the logit (monotone, no exp)
  w[i] = dead ? 0.0 : 1.0 / (1.0 + exp(-(double)l));
  count[i] = 0u;
  src[i] = dead ? -2 : -1;                               // -2: dead, source not drawn yet; -1: live
}

__global__ void __launch_bounds__(256) reloc_draw_kernel(long long N, const float* __restrict__ u, const double* __restrict__ cdf,
                                                         const double* __restrict__ total, uint32_t* __restrict__ count,
                                                         int32_t* __restrict__ src) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N || src[i] != -2) return;
  const double tot = *total;
  if (!(tot > 0.0)) { src[i] = -1; return; }             // nothing alive: nothing moves
  const double target = (double)u[i] * tot;
  long long lo = 0, hi = N - 1;
  while (lo < hi) {
    const long long mid = (lo + hi) >> 1;
    if (cdf[mid] > target) hi = mid; else lo = mid + 1;
  }
  src[i] = (int32_t)lo;
  atomicAdd(count + lo, 1u);
}

__global__ void __launch_bounds__(128) reloc_factors_kernel(long long N, const uint32_t* __restrict__ count, const float* __restrict__ logits,
                                                            const float* __restrict__ scales, float o_min, int n_max,
                                                            float2* __restrict__ new_scale, float* __restrict__ new_logit) {
  const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= N || count[j] == 0u) return;
  const int n = min((int)count[j] + 1, n_max);
  const double alpha = 1.0 / (1.0 + exp(-(double)logits[j]));
  const double o_new = 1.0 - pow(1.0 - alpha, 1.0 / (double)n);
  double denom = 0.0;
  for (int i = 1; i <= n; ++i) {
    double binom = 1.0, opow = o_new, sign = 1.0;        // C(i-1, 0), o'^(0+1)
    for (int k = 0; k < i; ++k) {
      denom += sign * binom * opow * rsqrt((double)(k + 1));
      binom = binom * (double)(i - 1 - k) / (double)(k + 1);
      opow *= o_new;
      sign = -sign;
    }
  }
  const double f = alpha / denom;
  const float2 sc = reinterpret_cast<const float2*>(scales)[j];
  new_scale[j] = make_float2((float)(sc.x * f), (float)(sc.y * f));
  const double oc = fmin(fmax(o_new, (double)o_min), 1.0 - 1e-7);
  new_logit[j] = (float)log(oc / (1.0 - oc));
}

__global__ void __launch_bounds__(256) reloc_apply_kernel(long long N, const int32_t* __restrict__ src, const uint32_t* __restrict__ count,
                                                          const float2* __restrict__ new_scale, const float* __restrict__ new_logit,
                                                          float* __restrict__ means, float* __restrict__ quats, float* __restrict__ scales,
                                                          float* __restrict__ logits, float* __restrict__ rgb, float* __restrict__ adam_m,
                                                          float* __restrict__ adam_v, int32_t* __restrict__ src_out) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int32_t j = src[i];
  if (src_out) src_out[i] = j;
  const bool moved = j >= 0, split = count[i] > 0u;      // a dead surfel is never a source and a source is never dead
  if (!moved && !split) return;
  const long long t = moved ? j : i;
  if (moved) {
#pragma unroll
    for (int c = 0; c < 3; ++c) { means[3 * i + c] = means[3 * t + c]; rgb[3 * i + c] = rgb[3 * t + c]; }
    reinterpret_cast<float4*>(quats)[i] = reinterpret_cast<const float4*>(quats)[t];
  }
  reinterpret_cast<float2*>(scales)[i] = new_scale[t];
  logits[i] = new_logit[t];
  if (adam_m && adam_v) {
    // state layout of satsplat_adam_step: groups of width 3, 4, 2, 1, 3 at 16-byte aligned offsets
    const int width[5] = {3, 4, 2, 1, 3};
    long long off = 0;
#pragma unroll
    for (int g = 0; g < 5; ++g) {
      for (int c = 0; c < width[g]; ++c) { adam_m[off + (long long)width[g] * i + c] = 0.f; adam_v[off + (long long)width[g] * i + c] = 0.f; }
      off += ((long long)N * width[g] + 3) & ~3LL;
    }
  }
}

int64_t relocate_scratch_bytes(int64_t N) { return N * 8 + cdf_scan_partials(N) * 8 + N * (4 + 4 + 8 + 4) + 256; }

cudaError_t launch_relocate(int64_t N, float* means, float* quats, float* scales, float* logits, float* rgb, float* adam_m,
                            float* adam_v, const float* u, float o_min, int n_max, void* scratch, int32_t* src_out, cudaStream_t s) {
  if (N == 0) return cudaSuccess;
  char* p = reinterpret_cast<char*>(scratch);
  double* cdf = reinterpret_cast<double*>(p);              p += N * 8;
  double* partial = reinterpret_cast<double*>(p);          p += cdf_scan_partials(N) * 8;
  float2* new_scale = reinterpret_cast<float2*>(p);        p += N * 8;
  uint32_t* count = reinterpret_cast<uint32_t*>(p);        p += N * 4;
  int32_t* src = reinterpret_cast<int32_t*>(p);            p += N * 4;
  float* new_logit = reinterpret_cast<float*>(p);
  const float logit_min = (float)log((double)o_min / (1.0 - (double)o_min));
  const int nb = (int)((N + 255) / 256);
  g_kernel_launches += 4;
  reloc_weights_kernel<<<nb, 256, 0, s>>>(N, logits, logit_min, cdf, count, src);
  double* total;
  cudaError_t e = launch_cdf_scan(cdf, N, partial, &total, s);
  if (e != cudaSuccess) return e;
  reloc_draw_kernel<<<nb, 256, 0, s>>>(N, u, cdf, total, count, src);
  reloc_factors_kernel<<<(int)((N + 127) / 128), 128, 0, s>>>(N, count, logits, scales, o_min, n_max, new_scale, new_logit);
  reloc_apply_kernel<<<nb, 256, 0, s>>>(N, src, count, new_scale, new_logit, means, quats, scales, logits, rgb, adam_m, adam_v, src_out);
  return cudaGetLastError();
}

}  // namespace satsplat

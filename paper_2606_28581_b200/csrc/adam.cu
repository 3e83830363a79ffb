// adam.cu — (f3) fused Adam step over the five surfel parameter groups (Adam with per-group learning
// rates), one launch for all 13 N values.  Element-wise and HBM-bound: per value 4 B parameter + 4 B gradient + 8 B
// state read, 4 B parameter + 8 B state written = 28 B.  Every group is a contiguous fp32 array, walked as float4
// (the group sizes 3N, 4N, 2N, N, 3N are handled with a scalar tail); the scale group is stepped in log space
// (theta = log s, dL/dtheta = s dL/ds, s <- s exp(-step)) so that the library's linear scales stay positive.
#include "internal.cuh"

namespace satsplat {

struct AdamGroup {
  float* p;
  const float* g;
  float* m;
  float* v;
  long long n;      // values in the group
  float lr;
  int log_space;
};

struct AdamParams {
  AdamGroup grp[5];
  long long vec_end[5];   // cumulative number of float4 work items up to and including group k
  float beta1, beta2, eps, inv_c1, inv_sqrt_c2;   // bias corrections 1/(1 - b1^t), 1/sqrt(1 - b2^t)
};

__device__ __forceinline__ void adam_one(float& p, float g, float& m, float& v, float lr, bool log_space, const AdamParams& A) {
  if (log_space) g *= p;
  m = A.beta1 * m + (1.0f - A.beta1) * g;
  v = A.beta2 * v + (1.0f - A.beta2) * g * g;
  const float step = lr * (m * A.inv_c1) / (sqrtf(v) * A.inv_sqrt_c2 + A.eps);
  p = log_space ? p * expf(-step) : p - step;
}

__global__ void __launch_bounds__(256) adam_kernel(const __grid_constant__ AdamParams A) {
  const long long total = A.vec_end[4];
  for (long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x; w < total; w += (long long)gridDim.x * blockDim.x) {
    int k = 0;
#pragma unroll
    for (int q = 0; q < 4; ++q) k += (w >= A.vec_end[q]);
    const AdamGroup& G = A.grp[k];
    const long long i4 = w - (k ? A.vec_end[k - 1] : 0);   // float4 index inside the group
    const long long base = 4 * i4;
    if (base + 4 <= G.n) {
      float4 p = reinterpret_cast<float4*>(G.p)[i4];
      const float4 g = reinterpret_cast<const float4*>(G.g)[i4];
      float4 m = reinterpret_cast<float4*>(G.m)[i4], v = reinterpret_cast<float4*>(G.v)[i4];
      adam_one(p.x, g.x, m.x, v.x, G.lr, G.log_space, A);
      adam_one(p.y, g.y, m.y, v.y, G.lr, G.log_space, A);
      adam_one(p.z, g.z, m.z, v.z, G.lr, G.log_space, A);
      adam_one(p.w, g.w, m.w, v.w, G.lr, G.log_space, A);
      reinterpret_cast<float4*>(G.p)[i4] = p;
      reinterpret_cast<float4*>(G.m)[i4] = m;
      reinterpret_cast<float4*>(G.v)[i4] = v;
    } else {
      for (long long e = base; e < G.n; ++e) {   // ragged tail of the group (n not a multiple of 4)
        float p = G.p[e], m = G.m[e], v = G.v[e];
        adam_one(p, G.g[e], m, v, G.lr, G.log_space, A);
        G.p[e] = p; G.m[e] = m; G.v[e] = v;
      }
    }
  }
}

cudaError_t launch_adam(int64_t N, float* const params[5], const float* const grads[5], float* m, float* v, const float lrs[5],
                        float beta1, float beta2, float eps, int step, cudaStream_t s) {
  if (N == 0) return cudaSuccess;
  static const int width[5] = {3, 4, 2, 1, 3};
  AdamParams A;
  long long off = 0, vec = 0;
  for (int k = 0; k < 5; ++k) {
    A.grp[k].p = params[k];
    A.grp[k].g = grads[k];
    A.grp[k].m = m + off;
    A.grp[k].v = v + off;
    A.grp[k].n = (long long)N * width[k];
    A.grp[k].lr = lrs[k];
    A.grp[k].log_space = (k == 2);
    off += (A.grp[k].n + 3) & ~3LL;   // every group's state starts 16-byte aligned
    vec += (A.grp[k].n + 3) / 4;
    A.vec_end[k] = vec;
  }
  A.beta1 = beta1; A.beta2 = beta2; A.eps = eps;
  A.inv_c1 = (float)(1.0 / (1.0 - pow((double)beta1, (double)step)));
  A.inv_sqrt_c2 = (float)(1.0 / sqrt(1.0 - pow((double)beta2, (double)step)));
  const long long blocks = (vec + 255) / 256;
  ++g_kernel_launches;
  const int64_t cap = (int64_t)current_sm_count() * 16;
  adam_kernel<<<(int)(blocks < cap ? blocks : cap), 256, 0, s>>>(A);
  return cudaGetLastError();
}

}  // namespace satsplat

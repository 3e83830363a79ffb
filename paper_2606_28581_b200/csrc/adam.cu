// adam.cu — (f3) fused Adam step over the five surfel parameter groups (Adam with per-group learning
// rates), one launch for all 13 N values.  Element-wise and HBM-bound: per value 4 B parameter + 4 B gradient + 8 B
// state read, 4 B parameter + 8 B state written = 28 B.  Every group is a contiguous fp32 array, walked as float4
// (the group sizes 3N, 4N, 2N, N, 3N are handled with a scalar tail); the scale group is stepped in log space
// (theta = log s, dL/dtheta = s dL/ds, s <- s exp(-step)) so that the library's linear scales stay positive.
#include <stddef.h>

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

// Per-camera groups (1e-4 camera delta matrices, 1e-3 camera gain and bias; Eq. 15, Eq. 1): the 23 values of the
// view selected by the device index (dF row 8, [C | c] 12, ambient 3) take one Adam step with that view's own state and step
// counter.  One warp; the view index, the counters and the parameters all live on the device, so the launch is identical for
// every view and every iteration of a captured graph.
struct CameraAdamParams {
  const int32_t* view_index;
  float* views;             // the DEVICE satsplat_view_params table as floats
  int stride, off_cc, off_ambient;   // floats per view, float offsets of cc[12] and ambient[3] inside one
  float* dF;                // [V,8] or NULL
  float* v_dF_all;          // [V,8] (read; the view's row is cleared afterwards if clear_v_dF)
  const float* v_cc;        // [12] or NULL
  const float* v_ambient;   // [3] or NULL
  float *m, *v;             // [V,23] each
  int32_t* steps;           // [V]
  float lr[3], beta1, beta2, eps;
  int n_views, clear_v_dF;
};

__global__ void __launch_bounds__(32) camera_adam_kernel(const __grid_constant__ CameraAdamParams A) {
  const int e = threadIdx.x;
  int vi = A.view_index ? *A.view_index : 0;
  vi = min(max(vi, 0), A.n_views - 1);
  const int t = A.steps[vi] + 1;
  __syncwarp();
  if (e == 0) A.steps[vi] = t;
  if (e >= 23) return;
  const int grp = e < 8 ? 0 : (e < 20 ? 1 : 2);
  float* p;
  const float* g;
  if (grp == 0) { p = A.dF ? A.dF + 8 * vi + e : nullptr; g = A.v_dF_all ? A.v_dF_all + 8 * vi + e : nullptr; }
  else if (grp == 1) { p = A.views + (size_t)vi * A.stride + A.off_cc + (e - 8); g = A.v_cc ? A.v_cc + (e - 8) : nullptr; }
  else { p = A.views + (size_t)vi * A.stride + A.off_ambient + (e - 20); g = A.v_ambient ? A.v_ambient + (e - 20) : nullptr; }
  if (!p || !g) return;     // group not stepped: its parameters and state stay as they are
  const float grad = *g;
  float m = A.m[23 * vi + e], v = A.v[23 * vi + e];
  m = A.beta1 * m + (1.0f - A.beta1) * grad;
  v = A.beta2 * v + (1.0f - A.beta2) * grad * grad;
  // bias corrections from the view's own counter (double: 23 threads, not a hot loop)
  const float inv_c1 = (float)(1.0 / (1.0 - pow((double)A.beta1, (double)t)));
  const float inv_sqrt_c2 = (float)(1.0 / sqrt(1.0 - pow((double)A.beta2, (double)t)));
  *p = *p - A.lr[grp] * (m * inv_c1) / (sqrtf(v) * inv_sqrt_c2 + A.eps);
  A.m[23 * vi + e] = m;
  A.v[23 * vi + e] = v;
  if (grp == 0 && A.clear_v_dF) A.v_dF_all[8 * vi + e] = 0.f;
}

cudaError_t launch_camera_adam(int n_views, const int32_t* view_index, satsplat_view_params* views, float* dF, float* v_dF_all,
                               const float* v_cc, const float* v_ambient, float* m, float* v, int32_t* steps, const float lr[3],
                               float beta1, float beta2, float eps, int clear_v_dF, cudaStream_t s) {
  CameraAdamParams A;
  A.view_index = view_index;
  A.views = reinterpret_cast<float*>(views);
  A.stride = (int)(sizeof(satsplat_view_params) / sizeof(float));
  A.off_cc = (int)(offsetof(satsplat_view_params, cc) / sizeof(float));
  A.off_ambient = (int)(offsetof(satsplat_view_params, ambient) / sizeof(float));
  A.dF = dF; A.v_dF_all = v_dF_all; A.v_cc = v_cc; A.v_ambient = v_ambient;
  A.m = m; A.v = v; A.steps = steps;
  for (int k = 0; k < 3; ++k) A.lr[k] = lr[k];
  A.beta1 = beta1; A.beta2 = beta2; A.eps = eps;
  A.n_views = n_views; A.clear_v_dF = clear_v_dF;
  ++g_kernel_launches;
  camera_adam_kernel<<<1, 32, 0, s>>>(A);
  return cudaGetLastError();
}

}  // namespace satsplat

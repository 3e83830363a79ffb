// losses.cu — (f1) the loss stage that turns one rendered view into the upstream gradients of the rasteriser's
// backward: image L1 + SSIM (11x11 Gaussian window, sigma 1.5, zero padding, as used by 3DGS), mean depth distortion, and
// the normal-consistency term between the rendered normal and the normal of the depth map (Eq. 13;
// weights :349).  Two tile kernels, both stencil + point-wise and HBM/L2-bound:
//   ssim_stats_kernel   16x16 output tile + 5-pixel halo of I and I* in shared memory, separable blur of the five
//                       moments (I, I*, I^2, I*^2, I I*) per channel, SSIM map and its three partial derivative
//                       maps (w.r.t. mu_1, E[I^2], E[I I*]) written out (36 B / pixel), SSIM sum reduced per CTA;
//   loss_upstream_kernel  separable blur of the three derivative maps (the window is symmetric: adjoint = blur) ->
//                       dSSIM/dI; L1 sign; Eq. 13: the world point map is affine in the depth, so the un-normalised
//                       normal is c = c0 + dx c1 + dy c2 with dx, dy the central depth differences and three constant
//                       vectors per camera; its gradient is gathered from the four neighbours; writes v_rgba, v_geom,
//                       v_aux and reduces the loss terms.
#include "internal.cuh"

namespace satsplat {

constexpr int kLT = 16;            // output tile
constexpr int kLR = 5;             // window radius
constexpr int kLW = kLT + 2 * kLR; // tile + halo = 26

struct LossParams {
  int W, H;
  float g[11];                     // Gaussian window (sums to 1)
  float w_l1, w_ssim, w_dist, w_normal;
  float inv_npx;                   // 1 / (H W)
  float c0[3], c1[3], c2[3], sgn;  // Eq. 13 constants: c = c0 + dx c1 + dy c2, N_d = sgn c / |c|
  float z_bg;
  const float4* rgba;
  const float4* geom;
  const float4* aux;
  const float4* target;
  float4* part;                    // [3][H*W] derivative maps (mu, s11, s12), xyz = channels
  float4* v_rgba;
  float4* v_geom;
  float4* v_aux;
  float* sums;                     // [0] sum |I - I*|, [1] sum SSIM map, [2] sum distortion, [3] sum (1 - A N_r.N_d)
};

constexpr float kC1 = 0.01f * 0.01f, kC2 = 0.03f * 0.03f;

__device__ __forceinline__ float block_sum_256(float v, float* s_red) {
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
  if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = v;
  __syncthreads();
  float r = 0.f;
  if (threadIdx.x < 8) r = s_red[threadIdx.x];
  if (threadIdx.x < 32) {
#pragma unroll
    for (int d = 4; d > 0; d >>= 1) r += __shfl_xor_sync(0xffffffffu, r, d);
  }
  __syncthreads();
  return r;   // valid in thread 0
}

__global__ void __launch_bounds__(256) ssim_stats_kernel(const __grid_constant__ LossParams P) {
  __shared__ float s_ij[6][kLW][kLW + 1];  // I (0..2) and I* (3..5) with halo, zero outside the image
  float (*const s_i)[kLW][kLW + 1] = s_ij, (*const s_j)[kLW][kLW + 1] = s_ij + 3;
  __shared__ float s_h[15][kLT][kLW + 1];   // horizontally blurred moments, TRANSPOSED [map][column][row]: bank-conflict free
  __shared__ float s_red[8];
  const int x0 = blockIdx.x * kLT, y0 = blockIdx.y * kLT;
  for (int e = threadIdx.x; e < kLW * kLW; e += 256) {
    const int ly = e / kLW, lx = e % kLW;
    const int x = x0 + lx - kLR, y = y0 + ly - kLR;
    float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a;
    if (x >= 0 && x < P.W && y >= 0 && y < P.H) {
      a = P.rgba[(size_t)y * P.W + x];
      b = P.target[(size_t)y * P.W + x];
    }
    s_i[0][ly][lx] = a.x; s_i[1][ly][lx] = a.y; s_i[2][ly][lx] = a.z;
    s_j[0][ly][lx] = b.x; s_j[1][ly][lx] = b.y; s_j[2][ly][lx] = b.z;
  }
  __syncthreads();
  // horizontal pass, register-blocked: a task = 8 consecutive outputs of one row of one channel; its 18 inputs of I and
  // I* are read once and slide through the 11 taps in registers (3744 -> 936 shared loads per 26 x 16 x 3 block)
  for (int e = threadIdx.x; e < kLW * 2 * 3; e += 256) {
    const int half = e / (kLW * 3), c = (e / kLW) % 3, r = e % kLW;     // lanes of a warp: consecutive rows
    float a[18], b[18];
#pragma unroll
    for (int k = 0; k < 18; ++k) { a[k] = s_i[c][r][half * 8 + k]; b[k] = s_j[c][r][half * 8 + k]; }
#pragma unroll
    for (int o = 0; o < 8; ++o) {
      float m1 = 0.f, m2 = 0.f, e11 = 0.f, e22 = 0.f, e12 = 0.f;
#pragma unroll
      for (int k = 0; k < 11; ++k) {
        const float w = P.g[k], wa = w * a[o + k], wb = w * b[o + k];
        m1 += wa; m2 += wb; e11 += wa * a[o + k]; e22 += wb * b[o + k]; e12 += wa * b[o + k];
      }
      const int col = half * 8 + o;
      s_h[c * 5 + 0][col][r] = m1; s_h[c * 5 + 1][col][r] = m2; s_h[c * 5 + 2][col][r] = e11;
      s_h[c * 5 + 3][col][r] = e22; s_h[c * 5 + 4][col][r] = e12;
    }
  }
  __syncthreads();
  // vertical pass, register-blocked: a task = 8 consecutive outputs of one column of one of the 15 maps; results go to
  // s_v (aliasing the input tiles, which are no longer needed) for the per-pixel SSIM arithmetic
  static_assert(15 * kLT * (kLT + 1) <= 6 * kLW * (kLW + 1), "s_v must fit in s_ij");
  float (*s_v)[kLT][kLT + 1] = reinterpret_cast<float (*)[kLT][kLT + 1]>(&s_ij[0][0][0]);
  for (int e = threadIdx.x; e < 15 * kLT * 2; e += 256) {
    const int half = e / (15 * kLT), q = (e / kLT) % 15, col = e % kLT;   // lanes of a warp: 16 columns x 2 maps
    float a[18];
#pragma unroll
    for (int k = 0; k < 18; ++k) a[k] = s_h[q][col][half * 8 + k];
#pragma unroll
    for (int o = 0; o < 8; ++o) {
      float acc = 0.f;
#pragma unroll
      for (int k = 0; k < 11; ++k) acc += P.g[k] * a[o + k];
      s_v[q][half * 8 + o][col] = acc;
    }
  }
  __syncthreads();
  const int lx = threadIdx.x & 15, ly = threadIdx.x >> 4;
  const int x = x0 + lx, y = y0 + ly;
  const bool inside = x < P.W && y < P.H;
  float dmu[3], ds11[3], ds12[3], ssim_sum = 0.f;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const float mu1 = s_v[c * 5 + 0][ly][lx], mu2 = s_v[c * 5 + 1][ly][lx], e11 = s_v[c * 5 + 2][ly][lx];
    const float e22 = s_v[c * 5 + 3][ly][lx], e12 = s_v[c * 5 + 4][ly][lx];
    const float s11 = e11 - mu1 * mu1, s22 = e22 - mu2 * mu2, s12 = e12 - mu1 * mu2;
    const float a = 2.f * mu1 * mu2 + kC1, b = 2.f * s12 + kC2;
    const float cc = mu1 * mu1 + mu2 * mu2 + kC1, d = s11 + s22 + kC2;
    const float icd = 1.0f / (cc * d);
    const float m = a * b * icd;
    const float d_mu1 = 2.f * mu2 * b * icd - m * 2.f * mu1 / cc;
    ds11[c] = -m / d;
    ds12[c] = 2.f * a * icd;
    dmu[c] = d_mu1 - 2.f * mu1 * ds11[c] - mu2 * ds12[c];
    if (inside) ssim_sum += m;
  }
  if (inside) {
    const size_t o = (size_t)y * P.W + x, n = (size_t)P.W * P.H;
    P.part[o] = make_float4(dmu[0], dmu[1], dmu[2], 0.f);
    P.part[n + o] = make_float4(ds11[0], ds11[1], ds11[2], 0.f);
    P.part[2 * n + o] = make_float4(ds12[0], ds12[1], ds12[2], 0.f);
  }
  const float tot = block_sum_256(ssim_sum, s_red);
  if (threadIdx.x == 0) atomicAdd(P.sums + 1, tot);
}

__global__ void __launch_bounds__(256) loss_upstream_kernel(const __grid_constant__ LossParams P) {
  __shared__ float s_p[9][kLW][kLW + 1];     // derivative maps with halo, zero outside the image
  __shared__ float s_h[9][kLT][kLW + 1];     // transposed [map][column][row]
  __shared__ float s_zv[kLT + 4][kLT + 4];   // depth z_v = D + (1 - A) z_bg, halo 2
  __shared__ float s_vd[2][kLT + 2][kLT + 2]; // v_dx, v_dy of the normal term, halo 1
  __shared__ float s_red[8];
  const int x0 = blockIdx.x * kLT, y0 = blockIdx.y * kLT;
  const size_t n = (size_t)P.W * P.H;
  for (int e = threadIdx.x; e < kLW * kLW; e += 256) {
    const int ly = e / kLW, lx = e % kLW;
    const int x = x0 + lx - kLR, y = y0 + ly - kLR;
    float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a, c = a;
    if (x >= 0 && x < P.W && y >= 0 && y < P.H) {
      const size_t o = (size_t)y * P.W + x;
      a = P.part[o]; b = P.part[n + o]; c = P.part[2 * n + o];
    }
    s_p[0][ly][lx] = a.x; s_p[1][ly][lx] = a.y; s_p[2][ly][lx] = a.z;
    s_p[3][ly][lx] = b.x; s_p[4][ly][lx] = b.y; s_p[5][ly][lx] = b.z;
    s_p[6][ly][lx] = c.x; s_p[7][ly][lx] = c.y; s_p[8][ly][lx] = c.z;
  }
  for (int e = threadIdx.x; e < (kLT + 4) * (kLT + 4); e += 256) {
    const int ly = e / (kLT + 4), lx = e % (kLT + 4);
    const int x = x0 + lx - 2, y = y0 + ly - 2;
    float zv = 0.f;
    if (x >= 0 && x < P.W && y >= 0 && y < P.H) {
      const size_t o = (size_t)y * P.W + x;
      zv = P.geom[o].w + (1.0f - P.rgba[o].w) * P.z_bg;
    }
    s_zv[ly][lx] = zv;
  }
  __syncthreads();
  // horizontal blur of the nine derivative maps, register-blocked (8 outputs per task, 18 inputs read once)
  for (int e = threadIdx.x; e < kLW * 2 * 9; e += 256) {
    const int half = e / (kLW * 9), c = (e / kLW) % 9, r = e % kLW;
    float a[18];
#pragma unroll
    for (int k = 0; k < 18; ++k) a[k] = s_p[c][r][half * 8 + k];
#pragma unroll
    for (int o = 0; o < 8; ++o) {
      float acc = 0.f;
#pragma unroll
      for (int k = 0; k < 11; ++k) acc += P.g[k] * a[o + k];
      s_h[c][half * 8 + o][r] = acc;
    }
  }
  // normal term on the tile + halo 1: v_dx, v_dy (what each pixel's own term sends to its depth differences)
  float my_nd[3] = {0.f, 0.f, 0.f}, my_nloss = 0.f;
  for (int e = threadIdx.x; e < (kLT + 2) * (kLT + 2); e += 256) {
    const int ly = e / (kLT + 2), lx = e % (kLT + 2);
    const int x = x0 + lx - 1, y = y0 + ly - 1;
    float vdx = 0.f, vdy = 0.f;
    if (x >= 1 && x < P.W - 1 && y >= 1 && y < P.H - 1) {      // interior pixel of the image
      const size_t o = (size_t)y * P.W + x;
      const float dx = s_zv[ly + 1][lx + 2] - s_zv[ly + 1][lx], dy = s_zv[ly + 2][lx + 1] - s_zv[ly][lx + 1];
      const float cx = P.c0[0] + dx * P.c1[0] + dy * P.c2[0], cy = P.c0[1] + dx * P.c1[1] + dy * P.c2[1];
      const float cz = P.c0[2] + dx * P.c1[2] + dy * P.c2[2];
      const float icn = rsqrtf(cx * cx + cy * cy + cz * cz);
      const float nx = cx * icn, ny = cy * icn, nz = cz * icn;   // c / |c|
      const float4 gm = P.geom[o];
      const float A = P.rgba[o].w;
      // v_Nd = -w_normal A N_r / npx ; v_c = sgn (v_Nd - n (n . v_Nd)) / |c|
      const float k = -P.w_normal * A * P.inv_npx;
      const float v0 = k * gm.x, v1 = k * gm.y, v2 = k * gm.z;
      const float dt = nx * v0 + ny * v1 + nz * v2;
      const float s = P.sgn * icn;
      const float vcx = s * (v0 - nx * dt), vcy = s * (v1 - ny * dt), vcz = s * (v2 - nz * dt);
      vdx = vcx * P.c1[0] + vcy * P.c1[1] + vcz * P.c1[2];
      vdy = vcx * P.c2[0] + vcy * P.c2[1] + vcz * P.c2[2];
    }
    s_vd[0][ly][lx] = vdx;
    s_vd[1][ly][lx] = vdy;
  }
  __syncthreads();
  // vertical blur, register-blocked; results in s_v (aliasing s_p, which the horizontal pass has consumed)
  static_assert(9 * kLT * (kLT + 1) <= 9 * kLW * (kLW + 1), "s_v must fit in s_p");
  float (*s_v)[kLT][kLT + 1] = reinterpret_cast<float (*)[kLT][kLT + 1]>(&s_p[0][0][0]);
  for (int e = threadIdx.x; e < 9 * kLT * 2; e += 256) {
    const int half = e / (9 * kLT), q = (e / kLT) % 9, col = e % kLT;
    float a[18];
#pragma unroll
    for (int k = 0; k < 18; ++k) a[k] = s_h[q][col][half * 8 + k];
#pragma unroll
    for (int o = 0; o < 8; ++o) {
      float acc = 0.f;
#pragma unroll
      for (int k = 0; k < 11; ++k) acc += P.g[k] * a[o + k];
      s_v[q][half * 8 + o][col] = acc;
    }
  }
  __syncthreads();
  const int lx = threadIdx.x & 15, ly = threadIdx.x >> 4;
  const int x = x0 + lx, y = y0 + ly;
  const bool inside = x < P.W && y < P.H;
  float l1 = 0.f, dist = 0.f;
  if (inside) {
    const size_t o = (size_t)y * P.W + x;
    const float4 I = P.rgba[o], J = P.target[o], gm = P.geom[o], ax = P.aux[o];
    float bl[9];
#pragma unroll
    for (int c = 0; c < 9; ++c) bl[c] = s_v[c][ly][lx];
    const float Iv[3] = {I.x, I.y, I.z}, Jv[3] = {J.x, J.y, J.z};
    float vI[3];
    const float k1 = P.w_l1 * P.inv_npx * (1.0f / 3.0f), ks = -P.w_ssim * P.inv_npx * (1.0f / 3.0f);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const float d = Iv[c] - Jv[c];
      l1 += fabsf(d);
      const float sg = d > 0.f ? 1.f : (d < 0.f ? -1.f : 0.f);
      vI[c] = k1 * sg + ks * (bl[c] + 2.f * Iv[c] * bl[3 + c] + Jv[c] * bl[6 + c]);
    }
    dist = ax.y;
    // normal term of this pixel (for the loss value and v_N_r) and the gathered depth gradient
    const bool interior = x >= 1 && x < P.W - 1 && y >= 1 && y < P.H - 1;
    if (interior) {
      const float dx = s_zv[ly + 2][lx + 3] - s_zv[ly + 2][lx + 1], dy = s_zv[ly + 3][lx + 2] - s_zv[ly + 1][lx + 2];
      const float cx = P.c0[0] + dx * P.c1[0] + dy * P.c2[0], cy = P.c0[1] + dx * P.c1[1] + dy * P.c2[1];
      const float cz = P.c0[2] + dx * P.c1[2] + dy * P.c2[2];
      const float icn = P.sgn * rsqrtf(cx * cx + cy * cy + cz * cz);
      my_nd[0] = cx * icn; my_nd[1] = cy * icn; my_nd[2] = cz * icn;
    }
    my_nloss = 1.0f - I.w * (gm.x * my_nd[0] + gm.y * my_nd[1] + gm.z * my_nd[2]);
    // v_zv(x, y) = v_dx(x-1, y) - v_dx(x+1, y) + v_dy(x, y-1) - v_dy(x, y+1)
    const float v_zv = s_vd[0][ly + 1][lx] - s_vd[0][ly + 1][lx + 2] + s_vd[1][ly][lx + 1] - s_vd[1][ly + 2][lx + 1];
    const float kn = -P.w_normal * I.w * P.inv_npx;
    P.v_rgba[o] = make_float4(vI[0], vI[1], vI[2], -P.z_bg * v_zv);
    P.v_geom[o] = make_float4(kn * my_nd[0], kn * my_nd[1], kn * my_nd[2], v_zv);
    P.v_aux[o] = make_float4(0.f, P.w_dist * P.inv_npx, 0.f, 0.f);
  }
  const float t0 = block_sum_256(l1, s_red);
  const float t2 = block_sum_256(dist, s_red);
  const float t3 = block_sum_256(inside ? my_nloss : 0.f, s_red);
  if (threadIdx.x == 0) {
    atomicAdd(P.sums + 0, t0);
    atomicAdd(P.sums + 2, t2);
    atomicAdd(P.sums + 3, t3);
  }
}

cudaError_t launch_losses(const LossHost& L, cudaStream_t s) {
  LossParams P;
  P.W = L.W; P.H = L.H;
  double g[11], gs = 0.0;
  for (int k = 0; k < 11; ++k) { const double x = k - 5; g[k] = exp(-(x * x) / (2.0 * 1.5 * 1.5)); gs += g[k]; }
  for (int k = 0; k < 11; ++k) P.g[k] = (float)(g[k] / gs);
  P.w_l1 = L.w_l1; P.w_ssim = L.w_ssim; P.w_dist = L.w_dist; P.w_normal = L.w_normal;
  P.inv_npx = (float)(1.0 / ((double)L.W * L.H));
  for (int k = 0; k < 3; ++k) { P.c0[k] = L.c0[k]; P.c1[k] = L.c1[k]; P.c2[k] = L.c2[k]; }
  P.sgn = L.sgn; P.z_bg = L.z_bg;
  P.rgba = reinterpret_cast<const float4*>(L.rgba); P.geom = reinterpret_cast<const float4*>(L.geom);
  P.aux = reinterpret_cast<const float4*>(L.aux); P.target = reinterpret_cast<const float4*>(L.target);
  P.part = reinterpret_cast<float4*>(L.scratch);
  P.v_rgba = reinterpret_cast<float4*>(L.v_rgba); P.v_geom = reinterpret_cast<float4*>(L.v_geom);
  P.v_aux = reinterpret_cast<float4*>(L.v_aux);
  P.sums = L.sums;
  cudaError_t e = cudaMemsetAsync(L.sums, 0, 8 * sizeof(float), s);
  if (e != cudaSuccess) return e;
  const dim3 grid((L.W + kLT - 1) / kLT, (L.H + kLT - 1) / kLT);
  g_kernel_launches += 2;
  ssim_stats_kernel<<<grid, 256, 0, s>>>(P);
  loss_upstream_kernel<<<grid, 256, 0, s>>>(P);
  return cudaGetLastError();
}

}  // namespace satsplat

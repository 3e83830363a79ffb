// blend_backward.cu — (a4) backward of the per-tile compositing and of the Eq. 1 epilogue.
//
// Per pixel: epilogue backward first (gradients of the 3x4 colour correction, the ambient light, the
// reprojection constants; scatter into the sun-depth gradient), then the tile list is walked in REVERSE order:
// T_i is recovered as T_{i+1}/(1 - a_i), the suffix sum S_i = sum_{k>i} w_k phi_k is carried, and each
// contributing (pixel, surfel) pair produces 16 gradient values (c, M = Q^-1, alpha, z_c, r, rgb, n) in the record slots.
// Those are reduced across the warp with a transposed shuffle butterfly (16 shuffles instead of 80), across
// the CTA's warps with shared-memory atomics, and only then flushed once per (tile, surfel) with coalesced
// global atomics into the per-surfel gradient records.  FP32-issue + atomics bound.
#include "internal.cuh"

namespace satsplat {

struct BwdParams {
  DevCamera cam;
  DevShading sh;
  const uint32_t* ranges;
  const uint32_t* vals;
  const float4* rec;
  const float4* v_rgba;
  const float4* v_geom;
  const float4* v_aux;
  const float* v_sun_in;   // depth-only mode: upstream of the sun map
  const float4* px_a;
  const float4* px_b;
  const int2* px_i;
  float* vrec;
  float* v_sun_depth;      // scatter target (may be NULL)
  float* red;              // [23] = cc(12) ambient(3) reproj(8), accumulated with atomics (may be NULL)
};

constexpr int kBatchB = 256;

// Sum 16 per-lane values over the warp.  On return lane l (l even) holds the total of slot
// ((l>>4)&1)*8 + ((l>>3)&1)*4 + ((l>>2)&1)*2 + ((l>>1)&1) in v[0].
__device__ __forceinline__ float warp_reduce16_transposed(float (&v)[16], int lane) {
  {
    const bool hi = lane & 16;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const float send = hi ? v[k] : v[k + 8];
      const float keep = hi ? v[k + 8] : v[k];
      v[k] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
  }
  {
    const bool hi = lane & 8;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const float send = hi ? v[k] : v[k + 4];
      const float keep = hi ? v[k + 4] : v[k];
      v[k] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
    }
  }
  {
    const bool hi = lane & 4;
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      const float send = hi ? v[k] : v[k + 2];
      const float keep = hi ? v[k + 2] : v[k];
      v[k] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
    }
  }
  {
    const bool hi = lane & 2;
    const float send = hi ? v[0] : v[1];
    const float keep = hi ? v[1] : v[0];
    v[0] = keep + __shfl_xor_sync(0xffffffffu, send, 2);
  }
  v[0] += __shfl_xor_sync(0xffffffffu, v[0], 1);
  return v[0];
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
  return v;
}

template <bool DEPTH_ONLY>
__global__ void __launch_bounds__(256, 3) blend_backward_kernel(const __grid_constant__ BwdParams P) {
  __shared__ float4 s_r0[kBatchB], s_r1[kBatchB], s_r2[kBatchB], s_r3[kBatchB];
  __shared__ float4 s_bb[kBatchB];
  __shared__ uint32_t s_id[kBatchB];
  __shared__ float s_grad[kBatchB * 16];
  __shared__ float s_red[8][24];
  __shared__ int s_max[8];

  const int tile = blockIdx.y * P.cam.TX + blockIdx.x;
  const uint32_t start = P.ranges[2 * tile];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int ix = blockIdx.x * kTile + (warp & 1) * 8 + (lane & 7);
  const int iy = blockIdx.y * kTile + (warp >> 1) * 4 + (lane >> 3);
  const bool inside = ix < P.cam.W && iy < P.cam.H;
  const float px = (float)ix + 0.5f, py = (float)iy + 0.5f;
  const size_t o = (size_t)iy * P.cam.W + ix;
  const float wx0 = (float)(blockIdx.x * kTile + (warp & 1) * 8) + 0.5f, wx1 = wx0 + 7.0f;
  const float wy0 = (float)(blockIdx.y * kTile + (warp >> 1) * 4) + 0.5f, wy1 = wy0 + 3.0f;

  // ---- per-pixel state and epilogue backward ----
  float T = 1.f, Tf = 1.f, zref = 0.f, M1 = 0.f, M2 = 0.f, A = 0.f;
  float va0 = 0.f, va1 = 0.f, va2 = 0.f, vN0 = 0.f, vN1 = 0.f, vN2 = 0.f, vD = 0.f, vL = 0.f, vmed = 0.f, vT = 0.f;
  int last = 0, mi = -1;
  float red[23];
#pragma unroll
  for (int k = 0; k < 23; ++k) red[k] = 0.f;
  if (inside) {
    const float4 a = P.px_a[o];
    const int2 li = P.px_i[o];
    Tf = a.x; T = Tf; A = 1.0f - Tf; last = li.x; mi = li.y;
    if (DEPTH_ONLY) {
      // sun_depth = sum w (z - z_bg) + z_bg  (since sum w + T_f = 1): phi = v (z - z_bg), no T_f term
      vD = P.v_sun_in[o];
      zref = P.cam.z_bg;
    } else {
      zref = a.y; M1 = a.z; M2 = a.w;
      const float4 b = P.px_b[o];
      float vI0 = 0.f, vI1 = 0.f, vI2 = 0.f, vA = 0.f;
      if (P.v_rgba) { const float4 t = P.v_rgba[o]; vI0 = t.x; vI1 = t.y; vI2 = t.z; vA = t.w; }
      if (P.v_geom) { const float4 t = P.v_geom[o]; vN0 = t.x; vN1 = t.y; vN2 = t.z; vD = t.w; }
      if (P.v_aux) { const float4 t = P.v_aux[o]; vmed = t.x; vL = t.y; }
      const float* cc = P.sh.cc;
      const float V = b.w;
      const float ac0 = cc[0] * b.x + cc[1] * b.y + cc[2] * b.z + cc[3];
      const float ac1 = cc[4] * b.x + cc[5] * b.y + cc[6] * b.z + cc[7];
      const float ac2 = cc[8] * b.x + cc[9] * b.y + cc[10] * b.z + cc[11];
      const float s0 = V + (1.f - V) * P.sh.ambient[0], s1 = V + (1.f - V) * P.sh.ambient[1], s2 = V + (1.f - V) * P.sh.ambient[2];
      const float vs0 = vI0 * ac0, vs1 = vI1 * ac1, vs2 = vI2 * ac2;     // d/d shade
      const float vc0 = vI0 * s0, vc1 = vI1 * s1, vc2 = vI2 * s2;        // d/d corrected albedo
      const float vV = vs0 * (1.f - P.sh.ambient[0]) + vs1 * (1.f - P.sh.ambient[1]) + vs2 * (1.f - P.sh.ambient[2]);
      red[0] = vc0 * b.x; red[1] = vc0 * b.y; red[2] = vc0 * b.z; red[3] = vc0;
      red[4] = vc1 * b.x; red[5] = vc1 * b.y; red[6] = vc1 * b.z; red[7] = vc1;
      red[8] = vc2 * b.x; red[9] = vc2 * b.y; red[10] = vc2 * b.z; red[11] = vc2;
      red[12] = vs0 * (1.f - V); red[13] = vs1 * (1.f - V); red[14] = vs2 * (1.f - V);
      va0 = cc[0] * vc0 + cc[4] * vc1 + cc[8] * vc2;
      va1 = cc[1] * vc0 + cc[5] * vc1 + cc[9] * vc2;
      va2 = cc[2] * vc0 + cc[6] * vc1 + cc[10] * vc2;
      if (P.sh.shadows_on) {
        const float D = __fmaf_rn(zref, A, M1);
        const ShadowTap t = shadow_tap(P.sh, P.cam, px, py, D, Tf);
        if (t.in_map) {
          const int x0 = t.x0, y0 = t.y0, x1 = t.x1, y1 = t.y1;
          const float fx = t.fx, fy = t.fy, h = t.h;
          const float* Dm = P.sh.sun_depth;
          const int SW = P.sh.sun_w;
          const float d00 = __ldg(Dm + y0 * SW + x0), d01 = __ldg(Dm + y0 * SW + x1);
          const float d10 = __ldg(Dm + y1 * SW + x0), d11 = __ldg(Dm + y1 * SW + x1);
          const float v_gap = -P.sh.slope * V * (1.f - V) * vV;
          float v_zv = v_gap;
          const float v_ds = -v_gap;
          if (P.v_sun_depth) {
            atomicAdd(P.v_sun_depth + y0 * SW + x0, v_ds * (1.f - fy) * (1.f - fx));
            atomicAdd(P.v_sun_depth + y0 * SW + x1, v_ds * (1.f - fy) * fx);
            atomicAdd(P.v_sun_depth + y1 * SW + x0, v_ds * fy * (1.f - fx));
            atomicAdd(P.v_sun_depth + y1 * SW + x1, v_ds * fy * fx);
          }
          const float dds_dx = (1.f - fy) * (d01 - d00) + fy * (d11 - d10);
          const float dds_dy = (1.f - fx) * (d10 - d00) + fx * (d11 - d01);
          const float v_xs = v_ds * dds_dx, v_ys = v_ds * dds_dy;
          v_zv -= P.sh.reproj[2] * v_xs + P.sh.reproj[6] * v_ys;   // h = b_z - z_v
          red[15] = v_xs * px; red[16] = v_xs * py; red[17] = v_xs * h; red[18] = v_xs;
          red[19] = v_ys * px; red[20] = v_ys * py; red[21] = v_ys * h; red[22] = v_ys;
          vD += v_zv;                 // z_v = D + T_f z_bg
          vT += P.cam.z_bg * v_zv;
        }
      }
      vT += -vA + va0 * P.cam.bg[0] + va1 * P.cam.bg[1] + va2 * P.cam.bg[2];   // A = 1 - T_f ; albedo = C + T_f bg
      vT -= vD * zref;                                                          // D = M1' + z_ref (1 - T_f)
    }
  }
  // ---- reduce the 23 epilogue gradients over the CTA, one atomic each ----
  if (!DEPTH_ONLY && P.red) {
#pragma unroll
    for (int k = 0; k < 23; ++k) {
      const float r = warp_sum(red[k]);
      if (lane == 0) s_red[warp][k] = r;
    }
    __syncthreads();
    if (threadIdx.x < 23) {
      float r = 0.f;
#pragma unroll
      for (int w = 0; w < 8; ++w) r += s_red[w][threadIdx.x];
      if (r != 0.f) atomicAdd(P.red + threadIdx.x, r);
    }
  }
  // ---- CTA-wide maximum of `last` ----
  {
    const int m = __reduce_max_sync(0xffffffffu, last);
    if (lane == 0) s_max[warp] = m;
  }
  for (int k = threadIdx.x; k < kBatchB * 16; k += 256) s_grad[k] = 0.f;
  __syncthreads();
  int max_last = 0;
#pragma unroll
  for (int w = 0; w < 8; ++w) max_last = max(max_last, s_max[w]);

  const float TfvT = Tf * vT;
  float Ssum = 0.f;
  const int slot = ((lane >> 4) & 1) * 8 + ((lane >> 3) & 1) * 4 + ((lane >> 2) & 1) * 2 + ((lane >> 1) & 1);

  const int nb = (max_last + kBatchB - 1) / kBatchB;
  for (int b = nb - 1; b >= 0; --b) {
    const int rel0 = b * kBatchB;
    const int n = min(kBatchB, max_last - rel0);
    if ((int)threadIdx.x < n) {
      const uint32_t id = P.vals[start + rel0 + threadIdx.x];
      const float4* r = P.rec + 4 * (size_t)id;
      s_id[threadIdx.x] = id;
      const float4 q0 = r[0], q1 = r[1];
      s_r0[threadIdx.x] = q0;
      s_r1[threadIdx.x] = q1;
      s_bb[threadIdx.x] = splat_bbox(q0, q1);
      s_r2[threadIdx.x] = r[2];
      if (!DEPTH_ONLY) s_r3[threadIdx.x] = r[3];
    }
    __syncthreads();
    const int wlast = __reduce_max_sync(0xffffffffu, last);   // nothing beyond this index matters to this warp
    for (int g0 = ((n - 1) >> 5) << 5; g0 >= 0; g0 -= 32) {
      bool hit = false;
      if (g0 + lane < n && rel0 + g0 + lane < wlast) {
        const float4 bb = s_bb[g0 + lane];
        hit = bb.x <= wx1 && bb.y >= wx0 && bb.z <= wy1 && bb.w >= wy0;
      }
      unsigned mask = __ballot_sync(0xffffffffu, hit);
      while (mask) {
      const int bit = 31 - __clz(mask);
      mask &= ~(1u << bit);
      const int j = g0 + bit;
      const float4 r0 = s_r0[j], r1 = s_r1[j];
      const float dx = px - r0.x, dy = py - r0.y;
      const float u = r0.z * dx + r0.w * dy, v = r1.x * dx + r1.y * dy;
      const float rho3 = u * u + v * v, rho2 = 2.0f * (dx * dx + dy * dy);
      const float rho = fminf(rho3, rho2);
      const float G = __expf(-0.5f * rho);
      const float aG = r1.z * G;
      const float a = fminf(kAlphaMax, aG);
      const bool active = (rel0 + j < last) && (rho <= kRhoCut) && (a >= kAlphaMin);
      if (!__any_sync(0xffffffffu, active)) continue;
      float g[16];
#pragma unroll
      for (int k = 0; k < 16; ++k) g[k] = 0.f;
      if (active) {
        const float4 r2 = s_r2[j];
        const bool lowpass = !(rho3 <= rho2);
        const float z = lowpass ? r1.w : r1.w + (r2.x * dx + r2.y * dy);
        const float zs = z - zref;
        const float om = 1.0f - a;
        const float Ti = T / om;
        const float w = a * Ti;
        float phi, v_z;
        if (DEPTH_ONLY) {
          phi = vD * zs;
          v_z = w * vD;
        } else {
          const float4 r3 = s_r3[j];
          const float psi = zs * zs * A - 2.0f * zs * M1 + M2;
          phi = va0 * r2.z + va1 * r2.w + va2 * r3.x + vN0 * r3.y + vN1 * r3.z + vN2 * r3.w + vD * zs + vL * psi;
          v_z = w * (vD + 2.0f * vL * (zs * A - M1)) + ((rel0 + j == mi) ? vmed : 0.f);
          g[10] = w * va0; g[11] = w * va1; g[12] = w * va2;
          g[13] = w * vN0; g[14] = w * vN1; g[15] = w * vN2;
        }
        const float v_a = Ti * phi - (Ssum + TfvT) / om;
        Ssum += w * phi;
        T = Ti;
        float v_rho = 0.f;
        if (aG < kAlphaMax) {
          g[6] = G * v_a;
          v_rho = -0.5f * G * r1.z * v_a;
        }
        g[7] = v_z;
        float vd0, vd1;
        if (!lowpass) {
          // z = z_c + g.d = z_c - r.(u,v): accumulate the gradients of M = Q^-1 and r directly,
          //   v_d = Q^T (v_uv - v_z r) = v_z g + Q^T v_uv,   v_M = -v_d (u,v)^T,   v_r = -v_z (u,v)
          // (no multiplication by Q^2 afterwards: well conditioned for nearly edge-on surfels)
          const float vu = 2.0f * u * v_rho, vv = 2.0f * v * v_rho;
          vd0 = v_z * r2.x + r0.z * vu + r1.x * vv;
          vd1 = v_z * r2.y + r0.w * vu + r1.y * vv;
          g[2] = -vd0 * u; g[3] = -vd0 * v; g[4] = -vd1 * u; g[5] = -vd1 * v;
          g[8] = -v_z * u; g[9] = -v_z * v;
        } else {
          vd0 = 4.0f * dx * v_rho;
          vd1 = 4.0f * dy * v_rho;
        }
        g[0] = -vd0;
        g[1] = -vd1;
      }
      const float tot = warp_reduce16_transposed(g, lane);
      if (!(lane & 1) && tot != 0.f) atomicAdd(&s_grad[j * 16 + slot], tot);
      }
    }
    __syncthreads();
    // flush this batch: one coalesced atomic per non-zero gradient component of each (tile, surfel) pair
#pragma unroll 4
    for (int k = threadIdx.x; k < n * 16; k += 256) {
      const float gval = s_grad[k];
      if (gval != 0.f) {
        atomicAdd(P.vrec + 16 * (size_t)s_id[k >> 4] + (k & 15), gval);
        s_grad[k] = 0.f;
      }
    }
    __syncthreads();
  }
}

cudaError_t launch_blend_backward(satsplat_ctx* c, const DevShading& sh, const float* v_rgba, const float* v_geom,
                                  const float* v_aux, const float* v_sun_depth_in, bool depth_only, float* v_cc,
                                  float* v_ambient, float* v_sun_depth, float* v_reproj, cudaStream_t s) {
  BwdParams P;
  P.cam = c->cam;
  P.sh = sh;
  P.ranges = c->ranges;
  P.vals = c->vals[c->sorted];
  P.rec = c->rec;
  P.v_rgba = reinterpret_cast<const float4*>(v_rgba);
  P.v_geom = reinterpret_cast<const float4*>(v_geom);
  P.v_aux = reinterpret_cast<const float4*>(v_aux);
  P.v_sun_in = v_sun_depth_in;
  P.px_a = c->px_a;
  P.px_b = c->px_b;
  P.px_i = c->px_i;
  P.vrec = c->vrec;
  P.v_sun_depth = v_sun_depth;
  const bool want_red = !depth_only && (v_cc || v_ambient || v_reproj);
  P.red = want_red ? c->red_buf : nullptr;
  if (want_red) cudaMemsetAsync(c->red_buf, 0, 32 * sizeof(float), s);
  const dim3 grid(c->cam.TX, c->cam.TY);
  ++g_kernel_launches;
  if (depth_only)
    blend_backward_kernel<true><<<grid, 256, 0, s>>>(P);
  else
    blend_backward_kernel<false><<<grid, 256, 0, s>>>(P);
  return cudaGetLastError();
}

}  // namespace satsplat

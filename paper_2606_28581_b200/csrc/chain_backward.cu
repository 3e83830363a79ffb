// chain_backward.cu — per-surfel chain rule from the gradient moment records of the blend backward (layout in
// blend_backward.cu) to the record gradients (c, M = Q^-1, alpha, z_c, r, rgb, n) and on to the surfel parameters
// (means, quats, scales, opacity logits, rgb) and the 2x4 camera delta dF (Eq. 15), through
// Eq. 8-11.  One thread per surfel; the 8 dF partials are reduced over the CTA (shuffles + shared memory) before
// one atomic each.  The moment records are cleared as they are consumed, so the context never needs a separate
// memset pass.  HBM-bound: 80 B moments read + cleared, 45 B inputs read, 52 B read-modify-write.
#include "internal.cuh"

namespace satsplat {

__device__ __forceinline__ float warp_sum_f(float v) {
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
  return v;
}

template <bool DEV>
__global__ void __launch_bounds__(256) chain_backward_kernel(DevCamera camv, const float* __restrict__ cam_dev, int N, const float* __restrict__ means,
                                                             const float* __restrict__ quats, const float* __restrict__ scales,
                                                             const float* __restrict__ logits, const uint32_t* __restrict__ count,
                                                             const uint8_t* __restrict__ flags, float4* __restrict__ vrec,
                                                             float* __restrict__ v_means, float* __restrict__ v_quats,
                                                             float* __restrict__ v_scales, float* __restrict__ v_logits,
                                                             float* __restrict__ v_rgb, float* __restrict__ v_dF,
                                                             const float* __restrict__ epi, float* __restrict__ v_cc,
                                                             float* __restrict__ v_ambient, float* __restrict__ v_reproj) {
  __shared__ float s_red[8][8];
  // the 23 epilogue gradients of the blend backward (kRedCopies partial copies in `epi`) are summed into the caller's
  // v_cc / v_ambient / v_reproj by the first CTA: no launch of their own
  if (epi && blockIdx.x == 0 && threadIdx.x < 23) {
    const int k = threadIdx.x;
    float* dst = k < 12 ? (v_cc ? v_cc + k : nullptr) : (k < 15 ? (v_ambient ? v_ambient + (k - 12) : nullptr) : (v_reproj ? v_reproj + (k - 15) : nullptr));
    if (dst) {
      float a = 0.f;
      for (int c = 0; c < kRedCopies; ++c) a += epi[c * 32 + k];
      *dst += a;
    }
  }
  // The CTA's 256 surfels are contiguous in every array: the 80-B moment records and the 12-B rows (means, v_means,
  // v_rgb) are moved between HBM and shared memory as coalesced float4 streams, and every load of the kernel is
  // issued before the first use (one DRAM round trip).
  __shared__ float4 s_v[256 * (kVrec / 4)];
  __shared__ __align__(16) float s_p[256 * 3], s_vm[256 * 3], s_vc[256 * 3];
  const int base = blockIdx.x * 256, t = threadIdx.x;
  const int i = base + t;
  const int nb = min(256, N - base);                      // surfels of this CTA
  {
    const float4* gv = vrec + (kVrec / 4) * (size_t)base;
#pragma unroll
    for (int k = 0; k < kVrec / 4; ++k) {
      const int e = t + 256 * k;
      if (e < nb * (kVrec / 4)) s_v[e] = gv[e];
    }
    if (nb == 256) {
      if (t < 192) {
        reinterpret_cast<float4*>(s_p)[t] = reinterpret_cast<const float4*>(means + 3 * (size_t)base)[t];
        if (v_means) reinterpret_cast<float4*>(s_vm)[t] = reinterpret_cast<const float4*>(v_means + 3 * (size_t)base)[t];
        if (v_rgb) reinterpret_cast<float4*>(s_vc)[t] = reinterpret_cast<const float4*>(v_rgb + 3 * (size_t)base)[t];
      }
    } else {
      for (int e = t; e < nb * 3; e += 256) {
        s_p[e] = means[3 * (size_t)base + e];
        if (v_means) s_vm[e] = v_means[3 * (size_t)base + e];
        if (v_rgb) s_vc[e] = v_rgb[3 * (size_t)base + e];
      }
    }
  }
  // per-thread rows, fetched before the barrier so that they overlap the staging
  const bool have = i < N;
  const uint32_t cnt = have ? count[i] : 0u;
  const uint8_t fl = have ? flags[i] : (uint8_t)0;
  const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
  float4 q = make_float4(1.f, 0.f, 0.f, 0.f), cur = zero4;
  float2 sc = make_float2(1.f, 1.f), vsc = make_float2(0.f, 0.f);
  float lg = 0.f, vlg = 0.f;
  if (have) {
    q = reinterpret_cast<const float4*>(quats)[i];
    sc = reinterpret_cast<const float2*>(scales)[i];
    lg = logits[i];
    if (v_quats) cur = reinterpret_cast<const float4*>(v_quats)[i];
    if (v_scales) vsc = reinterpret_cast<const float2*>(v_scales)[i];
    if (v_logits) vlg = v_logits[i];
  }
  __syncthreads();
  {
    // clear the consumed moment records; only now that their loads have landed: a store to a line whose fill is
    // still in flight serialises behind it (measured: 0.12 ms with the clear next to the load, 0.05 ms here)
    float4* gv = vrec + (kVrec / 4) * (size_t)base;
#pragma unroll
    for (int k = 0; k < kVrec / 4; ++k) {
      const int e = t + 256 * k;
      if (e < nb * (kVrec / 4)) gv[e] = zero4;
    }
  }
  float dF[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) dF[k] = 0.f;
  if (cnt > 0) {
    const float4 m0 = s_v[5 * t], m1 = s_v[5 * t + 1], m2 = s_v[5 * t + 2], m3 = s_v[5 * t + 3], m4 = s_v[5 * t + 4];
    const float p0 = s_p[3 * t], p1 = s_p[3 * t + 1], p2 = s_p[3 * t + 2];
    const CamRef<DEV> camr{camv, cam_dev};
    const float B00 = camr.Fp(0), B01 = camr.Fp(1), B02 = camr.Fp(2);
    const float B10 = camr.Fp(4), B11 = camr.Fp(5), B12 = camr.Fp(6);
    const float qn = sqrtf(q.x * q.x + q.y * q.y + q.z * q.z + q.w * q.w);
    const float inv = 1.0f / qn;
    const float w = q.x * inv, x = q.y * inv, y = q.z * inv, z = q.w * inv;
    const float tu0 = 1.f - 2.f * (y * y + z * z), tu1 = 2.f * (x * y + w * z), tu2 = 2.f * (x * z - w * y);
    const float tv0 = 2.f * (x * y - w * z), tv1 = 1.f - 2.f * (x * x + z * z), tv2 = 2.f * (y * z + w * x);
    const float au0 = B00 * tu0 + B01 * tu1 + B02 * tu2, au1 = B10 * tu0 + B11 * tu1 + B12 * tu2;
    const float av0 = B00 * tv0 + B01 * tv1 + B02 * tv2, av1 = B10 * tv0 + B11 * tv1 + B12 * tv2;
    const float M00 = sc.x * au0, M01 = sc.y * av0, M10 = sc.x * au1, M11 = sc.y * av1;   // M = B' R S' (Eq. 8)
    const float alpha = 1.0f / (1.0f + expf(-lg));
    // moments -> record gradients, slots g0 = (c_x, c_y, M00, M01)  g1 = (M10, M11, alpha, z_c)  g2 = (r_0, r_1, red, green)
    // g3 = (blue, n_x, n_y, n_z).  Per pair: v_uv = 2 s (u,v); v_d = t g + Q^T v_uv (4 s d for low-pass pairs);
    // v_c = -v_d; v_M = -v_d (u,v)^T; v_r = -t (u,v); v_alpha = G v_a = -2 s / alpha; v_zc = t.
    float4 g0, g1, g2, g3;
    {
      // Q = M^-1 and the depth slope g = -r Q are recomputed from the inputs (Eq. 8-10) instead of re-read from the record
      const float idet = 1.0f / (M00 * M11 - M01 * M10);
      const float Q00 = M11 * idet, Q01 = -M01 * idet, Q10 = -M10 * idet, Q11 = M00 * idet;
      const float rr0 = sc.x * tu2, rr1 = sc.y * tv2;
      const float ga = -(rr0 * Q00 + rr1 * Q10), gb = -(rr0 * Q01 + rr1 * Q11);
      const float suu = m0.x, suv = m0.y, svv = m0.z, Su = m0.w, Sv = m1.x, Tu = m1.y, Tv = m1.z, T0np = m1.w;
      g0.x = -(4.0f * m2.x); g0.y = -(4.0f * m2.y);
      g0.z = 0.f; g0.w = 0.f; g1.x = 0.f; g1.y = 0.f; g2.x = 0.f; g2.y = 0.f;
      if (!(fl & F_DEGENERATE)) {
        g0.x -= T0np * ga + 2.0f * (Q00 * Su + Q10 * Sv);
        g0.y -= T0np * gb + 2.0f * (Q01 * Su + Q11 * Sv);
        g0.z = -(ga * Tu + 2.0f * (Q00 * suu + Q10 * suv));
        g0.w = -(ga * Tv + 2.0f * (Q00 * suv + Q10 * svv));
        g1.x = -(gb * Tu + 2.0f * (Q01 * suu + Q11 * suv));
        g1.y = -(gb * Tv + 2.0f * (Q01 * suv + Q11 * svv));
        g2.x = -Tu; g2.y = -Tv;
      }
      g1.z = -2.0f * m2.w / alpha;
      g1.w = m2.z;
      g2.z = m3.x; g2.w = m3.y; g3.x = m3.z; g3.y = m3.w; g3.z = m4.x; g3.w = m4.y;
    }
    // gradient record slots: g0 = (c_x, c_y, M00, M01)  g1 = (M10, M11, alpha, z_c)  g2 = (r_0, r_1, red, green)  g3 = (blue, n_x, n_y, n_z)
    // v_logit = v_alpha alpha (1 - alpha) = -2 (sum s) (1 - alpha), with 1 - alpha = sigmoid(-logit) evaluated directly: for a
    // nearly opaque surfel (logit 10) the difference 1 - alpha of the rounded alpha carries 1e-3 of relative error
    if (v_logits) v_logits[i] = vlg - 2.0f * m2.w * (1.0f / (1.0f + expf(lg)));
    if (v_rgb) { s_vc[3 * t] += g2.z; s_vc[3 * t + 1] += g2.w; s_vc[3 * t + 2] += g3.x; }
    const float sg = (fl & F_FLIPPED) ? -1.f : 1.f;
    float vtu0 = 0.f, vtu1 = 0.f, vtu2 = 0.f, vtv0 = 0.f, vtv1 = 0.f, vtv2 = 0.f;
    const float vn0 = sg * g3.y, vn1 = sg * g3.z, vn2 = sg * g3.w;
    const float vc0 = g0.x, vc1 = g0.y;
    float vs0 = 0.f, vs1 = 0.f;
    if (!(fl & F_DEGENERATE)) {
      // gradient record slots 2..5 hold v_M (M = B' R S' = Q^-1), slots 8..9 hold v_r (r = (s_u t_u.z, s_v t_v.z))
      const float vM00 = g0.z, vM01 = g0.w, vM10 = g1.x, vM11 = g1.y;
      const float vr0 = g2.x, vr1 = g2.y;
      vs0 = vM00 * au0 + vM10 * au1 + vr0 * tu2;
      vs1 = vM01 * av0 + vM11 * av1 + vr1 * tv2;
      const float vau0 = sc.x * vM00, vau1 = sc.x * vM10, vav0 = sc.y * vM01, vav1 = sc.y * vM11;
      vtu0 = B00 * vau0 + B10 * vau1; vtu1 = B01 * vau0 + B11 * vau1; vtu2 = B02 * vau0 + B12 * vau1 + sc.x * vr0;
      vtv0 = B00 * vav0 + B10 * vav1; vtv1 = B01 * vav0 + B11 * vav1; vtv2 = B02 * vav0 + B12 * vav1 + sc.y * vr1;
      dF[0] = vau0 * tu0 + vav0 * tv0; dF[1] = vau0 * tu1 + vav0 * tv1; dF[2] = vau0 * tu2 + vav0 * tv2;
      dF[4] = vau1 * tu0 + vav1 * tv0; dF[5] = vau1 * tu1 + vav1 * tv1; dF[6] = vau1 * tu2 + vav1 * tv2;
    }
    if (v_scales) reinterpret_cast<float2*>(v_scales)[i] = make_float2(vsc.x + vs0, vsc.y + vs1);
    // c = B p + b ; z_c = b_z - p_z
    if (v_means) {
      s_vm[3 * t] += B00 * vc0 + B10 * vc1;
      s_vm[3 * t + 1] += B01 * vc0 + B11 * vc1;
      s_vm[3 * t + 2] += B02 * vc0 + B12 * vc1 - g1.w;
    }
    dF[0] += vc0 * p0; dF[1] += vc0 * p1; dF[2] += vc0 * p2; dF[3] = vc0;
    dF[4] += vc1 * p0; dF[5] += vc1 * p1; dF[6] += vc1 * p2; dF[7] = vc1;
    // R = [t_u | t_v | n] -> unit quaternion -> raw quaternion.  G[r][c] = dL/dR[r][c]
    if (v_quats) {
      const float G00 = vtu0, G01 = vtv0, G02 = vn0, G10 = vtu1, G11 = vtv1, G12 = vn1, G20 = vtu2, G21 = vtv2, G22 = vn2;
      const float vw = 2.f * (x * (G21 - G12) + y * (G02 - G20) + z * (G10 - G01));
      const float vx = 2.f * (-2.f * x * (G11 + G22) + y * (G01 + G10) + z * (G02 + G20) + w * (G21 - G12));
      const float vy = 2.f * (x * (G01 + G10) - 2.f * y * (G00 + G22) + z * (G12 + G21) + w * (G02 - G20));
      const float vz = 2.f * (x * (G02 + G20) + y * (G12 + G21) - 2.f * z * (G00 + G11) + w * (G10 - G01));
      const float dotq = w * vw + x * vx + y * vy + z * vz;
      float4* vq = reinterpret_cast<float4*>(v_quats) + i;
      cur.x += (vw - w * dotq) * inv; cur.y += (vx - x * dotq) * inv; cur.z += (vy - y * dotq) * inv; cur.w += (vz - z * dotq) * inv;
      *vq = cur;
    }
  }
  __syncthreads();
  if (nb == 256) {
    if (t < 192) {
      if (v_means) reinterpret_cast<float4*>(v_means + 3 * (size_t)base)[t] = reinterpret_cast<const float4*>(s_vm)[t];
      if (v_rgb) reinterpret_cast<float4*>(v_rgb + 3 * (size_t)base)[t] = reinterpret_cast<const float4*>(s_vc)[t];
    }
  } else {
    for (int e = t; e < nb * 3; e += 256) {
      if (v_means) v_means[3 * (size_t)base + e] = s_vm[e];
      if (v_rgb) v_rgb[3 * (size_t)base + e] = s_vc[e];
    }
  }
  if (v_dF) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const float r = warp_sum_f(dF[k]);
      if (lane == 0) s_red[warp][k] = r;
    }
    __syncthreads();
    if (threadIdx.x < 8) {
      float r = 0.f;
#pragma unroll
      for (int wv = 0; wv < 8; ++wv) r += s_red[wv][threadIdx.x];
      if (r != 0.f) atomicAdd(v_dF + threadIdx.x, r);
    }
  }
}

cudaError_t launch_chain_backward(satsplat_ctx* c, const float* means, const float* quats, const float* scales,
                                  const float* logits, float* v_means, float* v_quats, float* v_scales, float* v_logits,
                                  float* v_rgb, float* v_dF, const float* epi, float* v_cc, float* v_ambient, float* v_reproj,
                                  cudaStream_t s) {
  if (c->N == 0) {   // no surfel: only the epilogue sums are left to deliver (background pixels still feed the colour correction)
    if (epi && v_cc) launch_add_small(v_cc, epi, 12, s);
    if (epi && v_ambient) launch_add_small(v_ambient, epi + 12, 3, s);
    if (epi && v_reproj) launch_add_small(v_reproj, epi + 15, 8, s);
    return cudaGetLastError();
  }
  ++g_kernel_launches;
  const int grid = (int)((c->N + 255) / 256);
  if (c->cam_dev)
    chain_backward_kernel<true><<<grid, 256, 0, s>>>(c->cam, c->cam_dev, (int)c->N, means, quats, scales, logits, c->count, c->flags,
                                                     reinterpret_cast<float4*>(c->vrec), v_means, v_quats, v_scales, v_logits, v_rgb, v_dF, epi, v_cc, v_ambient,
                                                     v_reproj);
  else
    chain_backward_kernel<false><<<grid, 256, 0, s>>>(c->cam, nullptr, (int)c->N, means, quats, scales, logits, c->count, c->flags,
                                                      reinterpret_cast<float4*>(c->vrec), v_means, v_quats, v_scales, v_logits, v_rgb, v_dF, epi, v_cc, v_ambient,
                                                     v_reproj);
  return cudaGetLastError();
}

// adjoint of the Eq. 16 sun camera with respect to F' (include/satsplat.h: satsplat_sun_camera_backward)
__global__ void sun_camera_backward_kernel(float sc0, float sc1, float s0, float s1, const float* __restrict__ v_F_sun,
                                           const float* __restrict__ v_reproj, float* __restrict__ v_dF) {
  const int r = threadIdx.x >> 2, c = threadIdx.x & 3;   // 8 threads: one per entry of the 2x4 matrix
  if (r >= 2) return;
  const float sc = r ? sc1 : sc0;
  const float vs = v_F_sun ? v_F_sun[4 * r + c] : 0.f;
  const float vs2 = (v_F_sun ? v_F_sun[4 * r + 2] : 0.f) + (v_reproj ? v_reproj[4 * r + 2] : 0.f);
  const float sdir = c == 0 ? s0 : (c == 1 ? s1 : (c == 2 ? 1.0f : 0.0f));
  v_dF[4 * r + c] += sc * (vs - sdir * vs2);
}
cudaError_t launch_sun_camera_backward(float sc0, float sc1, float s0, float s1, const float* v_F_sun, const float* v_reproj,
                                       float* v_dF, cudaStream_t s) {
  ++g_kernel_launches;
  sun_camera_backward_kernel<<<1, 32, 0, s>>>(sc0, sc1, s0, s1, v_F_sun, v_reproj, v_dF);
  return cudaGetLastError();
}

// dst[k] += sum over the kRedCopies copies of src[copy * 32 + k]
__global__ void add_small_kernel(float* dst, const float* src, int n) {
  if ((int)threadIdx.x < n) {
    float a = 0.f;
    for (int c = 0; c < kRedCopies; ++c) a += src[c * 32 + threadIdx.x];
    dst[threadIdx.x] += a;
  }
}
cudaError_t launch_add_small(float* dst, const float* src, int n, cudaStream_t s) {
  ++g_kernel_launches;
  add_small_kernel<<<1, 32, 0, s>>>(dst, src, n);
  return cudaGetLastError();
}

}  // namespace satsplat

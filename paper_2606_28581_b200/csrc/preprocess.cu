// preprocess.cu — (a1) per-surfel preprocess (PAPER.md:97-131, Eq. 6-12; :140) and record export.
//
// One thread per surfel.  Everything that feeds an integer decision (tile rect, count, depth key, degenerate /
// flip flags) is computed with explicitly rounded single operations (__f*_rn intrinsics are never contracted by
// nvcc), in the op sequence DESIGN.md "Binning contract" writes down, so that the result is bit-reproducible.
// HBM-bound: reads 56 B, writes 64 B record + 8 B rect + 4 B count + 4 B key + 1 B flag per surfel.
#include "internal.cuh"

namespace satsplat {

__device__ __forceinline__ float sum2(float a, float b, float c, float d) { return __fmaf_rn(a, b, __fmul_rn(c, d)); }
__device__ __forceinline__ float diff2(float a, float b, float c, float d) { return __fmaf_rn(a, b, -__fmul_rn(c, d)); }
__device__ __forceinline__ float one_minus_twice(float s) { return __fsub_rn(1.0f, __fmul_rn(2.0f, s)); }
__device__ __forceinline__ float twice(float s) { return __fmul_rn(2.0f, s); }
__device__ __forceinline__ int tile_of(float v, int T) {
  float t = floorf(__fmul_rn(v, 0.0625f));
  t = fminf(fmaxf(t, -1.0f), (float)T);
  return (int)t;
}

template <bool DEV>
__global__ void __launch_bounds__(256) preprocess_kernel(DevCamera camv, const float* __restrict__ cam_dev, int N, const float* __restrict__ means,
                                                         const float* __restrict__ quats, const float* __restrict__ scales,
                                                         const float* __restrict__ logits, const float* __restrict__ rgb,
                                                         float4* __restrict__ rec, float4* __restrict__ bbox, ushort4* __restrict__ rect,
                                                         uint32_t* __restrict__ count, uint32_t* __restrict__ depth_key,
                                                         uint8_t* __restrict__ flags, uint32_t* __restrict__ tile_count) {
  // records leave through shared memory so that the CTA's 256 x 64 B go out as one contiguous float4 stream
  __shared__ float4 s_rec[256 * 4];
  const CamRef<DEV> camr{camv, cam_dev};
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  int cnt = 0, tx0 = 0, tx1 = 0, ty0 = 0, ty1 = 0;
  if (i < N) {
  const float px = means[3 * i], py = means[3 * i + 1], pz = means[3 * i + 2];
  const float cr = rgb[3 * i], cg = rgb[3 * i + 1], cb = rgb[3 * i + 2];
  const float4 q = reinterpret_cast<const float4*>(quats)[i];
  const float2 sc = reinterpret_cast<const float2*>(scales)[i];
  const float logit = logits[i];
  const float B00 = camr.Fp(0), B01 = camr.Fp(1), B02 = camr.Fp(2), b0 = camr.Fp(3);
  const float B10 = camr.Fp(4), B11 = camr.Fp(5), B12 = camr.Fp(6), b1 = camr.Fp(7);
  uint8_t fl = 0;
  // 1. normalise the quaternion (w,x,y,z)
  const float n2 = __fmaf_rn(q.w, q.w, __fmaf_rn(q.z, q.z, __fmaf_rn(q.y, q.y, __fmul_rn(q.x, q.x))));
  const float inv = __fdiv_rn(1.0f, __fsqrt_rn(n2));
  const float w = __fmul_rn(q.x, inv), x = __fmul_rn(q.y, inv), y = __fmul_rn(q.z, inv), z = __fmul_rn(q.w, inv);
  // 2. rotation columns (Eq. 3-4): t_u, t_v, n
  const float tu0 = one_minus_twice(sum2(y, y, z, z)), tu1 = twice(sum2(x, y, w, z)), tu2 = twice(diff2(x, z, w, y));
  const float tv0 = twice(diff2(x, y, w, z)), tv1 = one_minus_twice(sum2(x, x, z, z)), tv2 = twice(sum2(y, z, w, x));
  float n0 = twice(sum2(x, z, w, y)), n1 = twice(diff2(y, z, w, x)), nz = one_minus_twice(sum2(x, x, y, y));
  // 3. M = B' R S' (Eq. 8)
  const float aux = __fmaf_rn(B02, tu2, __fmaf_rn(B01, tu1, __fmul_rn(B00, tu0)));
  const float auy = __fmaf_rn(B12, tu2, __fmaf_rn(B11, tu1, __fmul_rn(B10, tu0)));
  const float avx = __fmaf_rn(B02, tv2, __fmaf_rn(B01, tv1, __fmul_rn(B00, tv0)));
  const float avy = __fmaf_rn(B12, tv2, __fmaf_rn(B11, tv1, __fmul_rn(B10, tv0)));
  const float M00 = __fmul_rn(sc.x, aux), M10 = __fmul_rn(sc.x, auy), M01 = __fmul_rn(sc.y, avx), M11 = __fmul_rn(sc.y, avy);
  // 4. projected centre
  const float cx = __fmaf_rn(B02, pz, __fmaf_rn(B01, py, __fmaf_rn(B00, px, b0)));
  const float cy = __fmaf_rn(B12, pz, __fmaf_rn(B11, py, __fmaf_rn(B10, px, b1)));
  // 5. height depth (Eq. 11) and order-preserving key
  const float zc = __fsub_rn(camr.b_z(), pz);
  uint32_t k = __float_as_uint(zc);
  k = (k & 0x80000000u) ? ~k : (k | 0x80000000u);
  // 6. extent
  const float ex = __fmaf_rn(M01, M01, __fmul_rn(M00, M00)), ey = __fmaf_rn(M11, M11, __fmul_rn(M10, M10));
  const float extx = fmaxf(__fmul_rn(3.0f, __fsqrt_rn(ex)), kMinExtent);
  const float exty = fmaxf(__fmul_rn(3.0f, __fsqrt_rn(ey)), kMinExtent);
  // 8. cull
  const bool cull = logit < kLogitCull || !(n2 > 0.0f) || !(sc.x > 0.0f) || !(sc.y > 0.0f) || !isfinite(n2) ||
                    !isfinite(cx) || !isfinite(cy) || !isfinite(extx) || !isfinite(exty) || !isfinite(zc);
  if (!cull) {
    // 7. tile rect
    tx0 = min(max(tile_of(__fsub_rn(cx, extx), camv.TX), 0), camv.TX);
    tx1 = min(max(tile_of(__fadd_rn(cx, extx), camv.TX) + 1, 0), camv.TX);
    ty0 = min(max(tile_of(__fsub_rn(cy, exty), camv.TY), 0), camv.TY);
    ty1 = min(max(tile_of(__fadd_rn(cy, exty), camv.TY) + 1, 0), camv.TY);
  } else {
    fl |= F_CULLED;
  }
  cnt = cull ? 0 : max(tx1 - tx0, 0) * max(ty1 - ty0, 0);
  rect[i] = make_ushort4((unsigned short)tx0, (unsigned short)ty0, (unsigned short)tx1, (unsigned short)ty1);
  count[i] = (uint32_t)cnt;
  depth_key[i] = k;
  // 10. record
  const float det = __fmaf_rn(M00, M11, -__fmul_rn(M01, M10));
  float Q00 = kDegenerateQ, Q01 = 0.f, Q10 = 0.f, Q11 = kDegenerateQ, g0 = 0.f, g1 = 0.f;
  if (!(fabsf(det) > kDetEps)) {
    fl |= F_DEGENERATE;
  } else {
    const float id = __fdiv_rn(1.0f, det);
    Q00 = __fmul_rn(M11, id); Q01 = __fmul_rn(-M01, id); Q10 = __fmul_rn(-M10, id); Q11 = __fmul_rn(M00, id);
    const float r0 = __fmul_rn(sc.x, tu2), r1 = __fmul_rn(sc.y, tv2);
    g0 = -__fmaf_rn(r1, Q10, __fmul_rn(r0, Q00));
    g1 = -__fmaf_rn(r1, Q11, __fmul_rn(r0, Q01));
  }
  const float dotv = __fmaf_rn(nz, camr.vd(2), __fmaf_rn(n1, camr.vd(1), __fmul_rn(n0, camr.vd(0))));
  if (dotv > 0.0f) { n0 = -n0; n1 = -n1; nz = -nz; fl |= F_FLIPPED; }
  const float alpha = 1.0f / (1.0f + expf(-logit));
  flags[i] = fl;
  float4* r = s_rec + 4 * threadIdx.x;      // culled surfels: the slot is written too, and never read
  r[0] = make_float4(cx, cy, Q00, Q01);
  r[1] = make_float4(Q10, Q11, alpha, zc);
  r[2] = make_float4(g0, g1, cr, cg);
  r[3] = make_float4(cb, n0, n1, nz);
  bbox[i] = splat_bbox(r[0], r[1]);
  }
  __syncthreads();
  {
    const int nb = min(256, N - (int)(blockIdx.x * blockDim.x));
    float4* out = rec + 4 * (size_t)blockIdx.x * blockDim.x;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int e = threadIdx.x + 256 * k;
      if (e < 4 * nb) out[e] = s_rec[e];
    }
  }
  // tile-sort binning: count the (tile, surfel) pairs per tile with fire-and-forget RED atomics; surfels covering
  // many tiles (oversized splats) are expanded by the whole warp
  if (tile_count == nullptr) return;
  if (cnt > 0 && cnt <= 16) {
    for (int ty = ty0; ty < ty1; ++ty)
      for (int tx = tx0; tx < tx1; ++tx) atomicAdd(tile_count + (size_t)(ty * camv.TX + tx) * kCtrStride, 1u);
  }
  unsigned big = __ballot_sync(0xffffffffu, cnt > 16);
  const int lane = threadIdx.x & 31;
  while (big) {
    const int src = __ffs(big) - 1;
    big &= big - 1;
    const int c2 = __shfl_sync(0xffffffffu, cnt, src);
    const int x0 = __shfl_sync(0xffffffffu, tx0, src), y0 = __shfl_sync(0xffffffffu, ty0, src);
    const int w = __shfl_sync(0xffffffffu, tx1, src) - x0;
    for (int q = lane; q < c2; q += 32) atomicAdd(tile_count + (size_t)((y0 + q / w) * camv.TX + x0 + q % w) * kCtrStride, 1u);
  }
}

cudaError_t launch_preprocess(satsplat_ctx* c, int64_t N, const float* means, const float* quats, const float* scales,
                              const float* logits, const float* rgb, cudaStream_t s) {
  if (N == 0) return cudaSuccess;
  const int threads = 256;
  const int blocks = (int)((N + threads - 1) / threads);
  ++g_kernel_launches;
  uint32_t* tc = c->binning_mode == SATSPLAT_BINNING_TILESORT ? c->tile_count : nullptr;
  if (c->cam_dev)
    preprocess_kernel<true><<<blocks, threads, 0, s>>>(c->cam, c->cam_dev, (int)N, means, quats, scales, logits, rgb, c->rec, c->bbox,
                                                       reinterpret_cast<ushort4*>(c->rect), c->count, c->depth_key, c->flags, tc);
  else
    preprocess_kernel<false><<<blocks, threads, 0, s>>>(c->cam, nullptr, (int)N, means, quats, scales, logits, rgb, c->rec, c->bbox,
                                                        reinterpret_cast<ushort4*>(c->rect), c->count, c->depth_key, c->flags, tc);
  return cudaGetLastError();
}

// test access: canonical record order (c_x, c_y, Q00, Q01, Q10, Q11, z_c, g0, g1, alpha, r, g, b, n_x, n_y, n_z)
__global__ void export_records_kernel(int N, const float4* __restrict__ rec, const uint32_t* __restrict__ count,
                                      const uint8_t* __restrict__ flags, float* __restrict__ out,
                                      uint8_t* __restrict__ flags_out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  float v[16];
  if (count[i] > 0) {
    const float4 a = rec[4 * (size_t)i], b = rec[4 * (size_t)i + 1], c = rec[4 * (size_t)i + 2], d = rec[4 * (size_t)i + 3];
    const bool deg = flags[i] & F_DEGENERATE;
    v[0] = a.x; v[1] = a.y; v[2] = deg ? 0.f : a.z; v[3] = deg ? 0.f : a.w; v[4] = deg ? 0.f : b.x; v[5] = deg ? 0.f : b.y;
    v[6] = b.w; v[7] = c.x; v[8] = c.y; v[9] = b.z; v[10] = c.z; v[11] = c.w; v[12] = d.x; v[13] = d.y; v[14] = d.z; v[15] = d.w;
  } else {
    for (int k = 0; k < 16; ++k) v[k] = 0.f;
  }
  for (int k = 0; k < 16; ++k) out[16 * (size_t)i + k] = v[k];
  if (flags_out) flags_out[i] = flags[i];
}

cudaError_t launch_export_records(satsplat_ctx* c, float* records_out, uint8_t* flags_out, cudaStream_t s) {
  if (c->N == 0) return cudaSuccess;
  ++g_kernel_launches;
  export_records_kernel<<<(int)((c->N + 255) / 256), 256, 0, s>>>((int)c->N, c->rec, c->count, c->flags, records_out, flags_out);
  return cudaGetLastError();
}

}  // namespace satsplat

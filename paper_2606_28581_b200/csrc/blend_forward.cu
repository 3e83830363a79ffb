// blend_forward.cu — (a3) per-16x16-tile front-to-back compositing (Eq. 14) of colour,
// alpha, expected depth, normal, median depth and the depth-distortion term, with the Eq. 12 lower-bounded
// Gaussian evaluated through the exact per-splat affine map u = Q (x - c) (Eq. 9), and (a5) the Eq. 1 epilogue
// (colour correction + soft shadow test against the sun-view depth map) fused after the loop.
//
// One thread per pixel; a warp owns an 8x4 pixel block and walks the tile's list on its own (no CTA barrier).  Per
// group of 32 list entries, lane l turns entry l's precomputed bounding box into the bit mask of the block's pixels
// it covers; entries with a non-empty mask have their records gathered into the warp's shared-memory slots; a 32x32
// bit transpose across the warp (5 shuffles) hands every pixel the mask of entries whose box covers it, and each
// pixel then walks only its own candidates, in list order (the walk diverges across lanes; the per-pair test and
// the blend are exactly those of Eq. 9/12/14).  FP32-issue bound.
#include "internal.cuh"

namespace satsplat {

struct FwdParams {
  DevCamera cam;
  DevShading sh;
  const float* cam_dev;   // device-resident camera / shading records (DEV instantiations only)
  const float* sh_dev;
  const uint32_t* ranges;
  const uint32_t* vals;
  const float4* rec;
  const float4* bbox;
  float4* out_rgba;
  float4* out_geom;
  float4* out_aux;
  float* sun_depth_out;
  float4* px_a;
  float4* px_b;
  int2* px_i;
  int32_t* px_visited;
  int32_t* px_contrib;
};

#ifndef SATSPLAT_FWD_WARPS
#define SATSPLAT_FWD_WARPS 4
#endif
#ifndef SATSPLAT_FWD_MINB
#define SATSPLAT_FWD_MINB 8
#endif
#ifndef SATSPLAT_FWD_BULK
#define SATSPLAT_FWD_BULK 0   // 1: gather the records with one 64-byte cp.async.bulk each, completion on an mbarrier (measured trial)
#endif
constexpr int kWarpsF = SATSPLAT_FWD_WARPS;   // warps per CTA; a 16x16 tile is 8 warps (8x4 px each)
constexpr int kThreadsF = 32 * kWarpsF;

// 32x32 bit-matrix transpose across the warp: lane l passes row l, and receives column l (bit b = bit l of lane b's row).
__device__ __forceinline__ uint32_t warp_transpose_bits(uint32_t x, int lane) {
  uint32_t m = 0x0000FFFFu;
#pragma unroll
  for (int j = 16; j >= 1; j >>= 1) {
    const uint32_t y = __shfl_xor_sync(0xffffffffu, x, j);
    x = (lane & j) ? ((x & ~m) | ((y >> j) & m)) : ((x & m) | ((y << j) & ~m));
    m ^= m << (j >> 1);
  }
  return x;
}

#if SATSPLAT_FWD_BULK
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* b, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity) {
  asm volatile(
      "{\n .reg .pred p;\n WAIT_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n @!p bra WAIT_%=;\n}\n" ::"r"(smem_u32(b)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* b) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src),
               "r"(bytes), "r"(smem_u32(b))
               : "memory");
}
#endif

// Bit p (p = 8 * row + column) set iff pixel p of the 8x4 block whose first pixel centre is (wx0, wy0) lies inside the
// bounding box bb = (x_min, x_max, y_min, y_max).
__device__ __forceinline__ uint32_t block_cover_mask(const float4 bb, float wx0, float wy0) {
  const int c0 = (int)fmaxf(ceilf(bb.x - wx0), 0.0f), c1 = (int)fminf(floorf(bb.y - wx0), 7.0f);
  const int r0 = (int)fmaxf(ceilf(bb.z - wy0), 0.0f), r1 = (int)fminf(floorf(bb.w - wy0), 3.0f);
  if (c0 > c1 || r0 > r1) return 0u;
  const uint32_t cols = (2u << c1) - (1u << c0);
  const uint32_t rows = (2u << r1) - (1u << r0);
  return cols * ((rows * 0x00204081u) & 0x01010101u);
}

template <bool DEPTH_ONLY, bool DEV>
__global__ void __launch_bounds__(kThreadsF, SATSPLAT_FWD_MINB) blend_forward_kernel(const __grid_constant__ FwdParams P) {
  const CamRef<DEV> cam{P.cam, P.cam_dev};
  const ShRef<DEV> sh{P.sh, P.sh_dev};
  // per warp, double buffered: the records of a group's survivors as four float4 planes (lanes of a warp read
  // different entries at the same time)
#if SATSPLAT_FWD_BULK
  constexpr int kRecF = DEPTH_ONLY ? 3 : 4;
  __shared__ __align__(64) float4 s_rec[2][kWarpsF][32][kRecF];   // records as they sit in HBM (one bulk copy each)
  __shared__ __align__(8) uint64_t s_bar[2][kWarpsF];             // one mbarrier per warp and buffer
#else
  __shared__ float4 s_r0[2][kWarpsF][32], s_r1[2][kWarpsF][32], s_r2[2][kWarpsF][32], s_r3[2][DEPTH_ONLY ? 1 : kWarpsF][32];
#endif

  // CTA blockIdx.y holds warps [blockIdx.y * kWarpsF, +kWarpsF) of tile column blockIdx.x
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int gw = blockIdx.y * kWarpsF + warp, ty = gw >> 3, wi = gw & 7;
  const int tile = ty * P.cam.TX + blockIdx.x;
  const uint32_t start = P.ranges[2 * tile], end = P.ranges[2 * tile + 1];
  const int bx0 = blockIdx.x * kTile + (wi & 1) * 8, by0 = ty * kTile + (wi >> 1) * 4;
  const int ix = bx0 + (lane & 7), iy = by0 + (lane >> 3);
  const bool inside = ix < P.cam.W && iy < P.cam.H;
  const float px = (float)ix + 0.5f, py = (float)iy + 0.5f;
  const float wx0 = (float)bx0 + 0.5f, wy0 = (float)by0 + 0.5f;   // first pixel centre of this warp's 8x4 block

  float T = 1.f, C0 = 0.f, C1 = 0.f, C2 = 0.f, N0 = 0.f, N1 = 0.f, N2 = 0.f;
  float M1 = 0.f, M2 = 0.f, L = 0.f, zref = 0.f, med = cam.z_bg();
  int mi = -1, last = 0, visited = 0, ncontrib = 0;
  bool done = !inside;

  // Every warp walks the tile's list on its own (no CTA barrier), in groups of 32 entries, software-pipelined:
  // surfel ids are fetched three groups ahead, boxes two groups ahead, and the survivors' records are gathered one
  // group ahead with asynchronous copies into the other half of the double buffer.
  const int len = (int)(end - start);
  const int ngroups = (len + 31) >> 5;
  constexpr uint32_t kNoId = 0xffffffffu;
  auto fetch_id = [&](int cc) -> uint32_t {
    const int idx = cc * 32 + lane;
    return idx < len ? P.vals[start + idx] : kNoId;
  };
  const float4 bb_none = make_float4(1e30f, -1e30f, 1e30f, -1e30f);
  auto fetch_bb = [&](uint32_t id) -> float4 { return id != kNoId ? P.bbox[id] : bb_none; };
  // lane l turns entry l's bounding box into the mask of block pixels it covers; survivors (non-empty masks) have
  // their records gathered into the warp's slots (slot = lane) of buffer `buf`
#if SATSPLAT_FWD_BULK
  if (lane == 0) { mbar_init(&s_bar[0][warp], 1); mbar_init(&s_bar[1][warp], 1); }
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  __syncwarp();
  uint32_t bar_phase = 0u;   // bit b: parity the next wait on buffer b expects
  auto gather = [&](uint32_t id, uint32_t cover, int buf) {
    // the buffer was last read with ordinary loads: order them before the asynchronous-proxy writes
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    const unsigned surv = __ballot_sync(0xffffffffu, cover != 0u);
    if (lane == 0) mbar_expect_tx(&s_bar[buf][warp], (uint32_t)__popc(surv) * 16u * kRecF);
    __syncwarp();
    if (cover != 0u) bulk_g2s(&s_rec[buf][warp][lane][0], P.rec + 4 * (size_t)id, 16u * kRecF, &s_bar[buf][warp]);
  };
#else
  auto gather = [&](uint32_t id, uint32_t cover, int buf) {
    if (cover != 0u) {
      const float4* r = P.rec + 4 * (size_t)id;
      cp_async16(&s_r0[buf][warp][lane], r);
      cp_async16(&s_r1[buf][warp][lane], r + 1);
      cp_async16(&s_r2[buf][warp][lane], r + 2);
      if (!DEPTH_ONLY) cp_async16(&s_r3[buf][warp][lane], r + 3);
    }
    cp_async_commit();
  };
#endif
  uint32_t id_a = fetch_id(0), id_b = fetch_id(1), id_c = fetch_id(2);   // groups c, c+1, c+2
  float4 bb_a = fetch_bb(id_a);
  float4 bb_b = fetch_bb(id_b);
  uint32_t cover = block_cover_mask(bb_a, wx0, wy0);
  gather(id_a, cover, 0);
  int c = 0;
  for (; c < ngroups; ++c) {
    if (__all_sync(0xffffffffu, done)) break;   // this warp's 8x4 pixels are all finished
    // next group: boxes -> cover masks -> record gather in flight while this group is walked
    const uint32_t cover_n = block_cover_mask(bb_b, wx0, wy0);
    gather(id_b, cover_n, (c + 1) & 1);
    const float4 bb_c = fetch_bb(id_c);
    const uint32_t id_d = fetch_id(c + 3);
    // the 32x32 bit transpose hands every pixel the mask of entries whose box covers it
    uint32_t m = warp_transpose_bits(cover, lane);
    if (done) m = 0u;
    const int buf = c & 1;
#if SATSPLAT_FWD_BULK
    mbar_wait(&s_bar[buf][warp], (bar_phase >> buf) & 1u);   // this group's records have landed
    bar_phase ^= 1u << buf;
#else
    cp_async_wait<1>();   // this group's records have landed
#endif
    __syncwarp();
    const int rel0 = c * 32;
    // every pixel walks its own candidates, in list order
    while (m) {
      const int j = __ffs(m) - 1;
      m &= m - 1;
#if SATSPLAT_FWD_BULK
      const float4 r0 = s_rec[buf][warp][j][0], r1 = s_rec[buf][warp][j][1];
#else
      const float4 r0 = s_r0[buf][warp][j], r1 = s_r1[buf][warp][j];
#endif
      const PairEval E = pair_eval(r0, r1, px, py);                           // Eq. 9, Eq. 12
      if (!(E.rho <= kRhoCut)) continue;
      const float a = E.a;
      if (a < kAlphaMin) continue;
      const float Tn = T * (1.0f - a);
      if (Tn < kTMin) { done = true; visited = rel0 + j + 1; break; }
      const float w = a * T;
#if SATSPLAT_FWD_BULK
      const float4 r2 = s_rec[buf][warp][j][2];
#else
      const float4 r2 = s_r2[buf][warp][j];
#endif
      const float z = pair_depth(E, r1.w, r2.x, r2.y);                        // Eq. 6 depth at the intersection
      if (DEPTH_ONLY) {
        M1 += w * z;
      } else {
#if SATSPLAT_FWD_BULK
        const float4 r3 = s_rec[buf][warp][j][kRecF - 1];
#else
        const float4 r3 = s_r3[buf][warp][j];
#endif
        if (ncontrib == 0) zref = z;
        const float zs = z - zref;   // distortion accumulated in a per-pixel shifted depth frame (fp32 cancellation)
        if (T > 0.5f) { med = z; mi = rel0 + j; }
        L += w * (zs * zs * (1.0f - T) + M2 - 2.0f * zs * M1);
        C0 += w * r2.z; C1 += w * r2.w; C2 += w * r3.x;
        N0 += w * r3.y; N1 += w * r3.z; N2 += w * r3.w;
        M1 += w * zs;
        M2 += w * zs * zs;
      }
      T = Tn;
      last = rel0 + j + 1;
      ++ncontrib;
    }
    __syncwarp();
    cover = cover_n;
    id_b = id_c; bb_b = bb_c; id_c = id_d;
  }
#if SATSPLAT_FWD_BULK
  // exactly one armed phase is left unconsumed (group c, whether the loop broke off or ran out): its copies may still
  // be in flight and must land before the CTA can exit
  mbar_wait(&s_bar[c & 1][warp], (bar_phase >> (c & 1)) & 1u);
#else
  cp_async_wait<0>();
#endif
  if (!inside) return;
  if (visited == 0) visited = (int)(end - start);
  const size_t o = (size_t)iy * P.cam.W + ix;
  const float A = 1.0f - T;
  if (DEPTH_ONLY) {
    P.sun_depth_out[o] = M1 + T * cam.z_bg();
    P.px_a[o] = make_float4(T, 0.f, 0.f, 0.f);
    P.px_i[o] = make_int2(last, -1);
  } else {
    const float D = __fmaf_rn(zref, A, M1);
    const float al0 = C0 + T * cam.bg(0), al1 = C1 + T * cam.bg(1), al2 = C2 + T * cam.bg(2);
    float V = 1.0f;
    if (P.sh.shadows_on) {
      const ShadowTap t = shadow_tap(sh, cam, P.sh.sun_w, P.sh.sun_h, px, py, D, T);
      if (t.in_map) {
        const float* Dm = P.sh.sun_depth;
        const int SW = P.sh.sun_w;
        const float d00 = __ldg(Dm + t.y0 * SW + t.x0), d01 = __ldg(Dm + t.y0 * SW + t.x1);
        const float d10 = __ldg(Dm + t.y1 * SW + t.x0), d11 = __ldg(Dm + t.y1 * SW + t.x1);
        const float ds = (1.f - t.fy) * ((1.f - t.fx) * d00 + t.fx * d01) + t.fy * ((1.f - t.fx) * d10 + t.fx * d11);
        const float gap = t.zv - ds;
        V = 1.0f / (1.0f + __expf(sh.slope() * (gap - sh.bias())));
      }
    }
    const float ac0 = sh.cc(0) * al0 + sh.cc(1) * al1 + sh.cc(2) * al2 + sh.cc(3);
    const float ac1 = sh.cc(4) * al0 + sh.cc(5) * al1 + sh.cc(6) * al2 + sh.cc(7);
    const float ac2 = sh.cc(8) * al0 + sh.cc(9) * al1 + sh.cc(10) * al2 + sh.cc(11);
    const float s0 = V + (1.f - V) * sh.ambient(0), s1 = V + (1.f - V) * sh.ambient(1), s2 = V + (1.f - V) * sh.ambient(2);
    if (P.out_rgba) P.out_rgba[o] = make_float4(ac0 * s0, ac1 * s1, ac2 * s2, A);   // Eq. 1
    if (P.out_geom) P.out_geom[o] = make_float4(N0, N1, N2, D);
    if (P.out_aux) P.out_aux[o] = make_float4(med, L, V, T);
    P.px_a[o] = make_float4(T, zref, M1, M2);
    P.px_b[o] = make_float4(al0, al1, al2, V);
    P.px_i[o] = make_int2(last, mi);
  }
  if (P.px_visited) {   // SATSPLAT_OPT_DEBUG_PLANES: instrumentation, not part of the method
    P.px_visited[o] = visited;
    P.px_contrib[o] = ncontrib;
  }
}

cudaError_t launch_blend_forward(satsplat_ctx* c, const DevShading& sh, const float* sh_dev, float* out_rgba, float* out_geom,
                                 float* out_aux, float* sun_depth_out, bool depth_only, cudaStream_t s) {
  FwdParams P;
  P.cam = c->cam;
  P.sh = sh;
  P.cam_dev = c->cam_dev;
  P.sh_dev = sh_dev;
  P.ranges = c->ranges;
  P.vals = c->vals[c->sorted];
  P.rec = c->rec;
  P.bbox = c->bbox;
  P.out_rgba = reinterpret_cast<float4*>(out_rgba);
  P.out_geom = reinterpret_cast<float4*>(out_geom);
  P.out_aux = reinterpret_cast<float4*>(out_aux);
  P.sun_depth_out = sun_depth_out;
  P.px_a = c->px_a;
  P.px_b = c->px_b;
  P.px_i = c->px_i;
  P.px_visited = c->debug_planes ? c->px_visited : nullptr;
  P.px_contrib = c->debug_planes ? c->px_contrib : nullptr;
  c->planes_valid = c->debug_planes;
  const dim3 grid(c->cam.TX, c->cam.TY * (8 / kWarpsF));
  ++g_kernel_launches;
  const bool dev = c->cam_dev != nullptr;   // the view's shading record travels with a device camera (sh_dev is NULL for depth-only passes)
  if (depth_only) {
    if (dev) blend_forward_kernel<true, true><<<grid, kThreadsF, 0, s>>>(P);
    else blend_forward_kernel<true, false><<<grid, kThreadsF, 0, s>>>(P);
  } else {
    if (dev) blend_forward_kernel<false, true><<<grid, kThreadsF, 0, s>>>(P);
    else blend_forward_kernel<false, false><<<grid, kThreadsF, 0, s>>>(P);
  }
  return cudaGetLastError();
}

}  // namespace satsplat

// blend_backward.cu — (a4) backward of the per-tile compositing and of the Eq. 1 epilogue.
//
// Per pixel: epilogue backward first (gradients of the 3x4 colour correction, the ambient light, the
// reprojection constants; scatter into the sun-depth gradient), then the tile list is walked in REVERSE order:
// T_i is recovered as T_{i+1}/(1 - a_i) and the suffix sum S_i = sum_{k>i} w_k phi_k is carried.
//
// A warp owns an 8x4 pixel block and walks the tile's list on its own (no CTA barrier in the walk): per group of
// 32 list entries it culls by bounding box (one entry per lane, ballot) and gathers only the survivors' records
// into its shared-memory slots.  The walk only produces, per contributing (pixel, surfel) pair, the three scalars
// the gradients are linear in (dL/d rho, dL/d z, w) and the pair's local coordinates; the lanes that hit the same
// surfel append them, ballot-compacted, to a per-warp segment buffer.  Every eight segments the warp turns into
// eight teams of 4 lanes: a team walks one segment with all lanes busy, accumulates the 18 gradient moments of
// that surfel, reduces them over its 4 lanes (transposed butterfly) and adds them to the surfel's moment record
// with 16-byte vector REDs.  FP32-issue bound.
#include "internal.cuh"

namespace satsplat {

struct BwdParams {
  DevCamera cam;
  DevShading sh;
  const float* cam_dev;   // device-resident camera / shading records (DEV instantiations only)
  const float* sh_dev;
  const uint32_t* ranges;
  const uint32_t* vals;
  const float4* rec;
  const float4* bbox;
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

#ifndef SATSPLAT_BWD_WARPS
#define SATSPLAT_BWD_WARPS 4
#endif
#ifndef SATSPLAT_BWD_MINB
#define SATSPLAT_BWD_MINB 6
#endif
constexpr int kWarpsB = SATSPLAT_BWD_WARPS;   // warps per CTA: 8 = one 16x16 tile, 4 = its upper or lower half
constexpr int kThreadsB = 32 * kWarpsB;
#ifndef SATSPLAT_BWD_TEAM
#define SATSPLAT_BWD_TEAM 4
#endif
constexpr int kTeam = SATSPLAT_BWD_TEAM;   // lanes per team (4 or 8)
constexpr int kSegs = 32 / kTeam;         // (warp, surfel) segments per accumulation round: one per team

// ---- per-surfel gradient record (internal; consumed and cleared by chain_backward_kernel) -----------------------
// The blend backward does not form the 16 parameter gradients per (pixel, surfel) pair.  Every per-pair gradient
// is a per-pair scalar times a polynomial in the surfel-local coordinates (u, v) = Q (x - c), so it accumulates
// 18 moments per surfel and the chain kernel (once per surfel) turns them into gradients:
//   s = dL/d rho (0 where alpha' is clamped), t = dL/d z, w = blend weight;   np = Eq. 9 term active, lp = low-pass
//    0 sum_np s u u    1 sum_np s u v    2 sum_np s v v    3 sum_np s u
//    4 sum_np s v      5 sum_np t u      6 sum_np t v      7 sum_np t
//    8 sum_lp s dx     9 sum_lp s dy    10 sum t          11 sum s
//   12..14 sum w v_albedo              15..17 sum w v_normal            18, 19 unused
// All products are formed from the same fp32 (u, v) the per-pair form would use, so this is the per-pair sum with
// the common factors (Q, g, alpha) pulled out: same conditioning for nearly edge-on surfels.

__device__ __forceinline__ void red_add_v4(float* p, float a, float b, float c, float d) {
  asm volatile("red.global.add.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}
__device__ __forceinline__ void red_add_v2(float* p, float a, float b) {
  asm volatile("red.global.add.v2.f32 [%0], {%1,%2};" ::"l"(p), "f"(a), "f"(b) : "memory");
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
  return v;
}

// Sum 16 per-lane values over a team of kTeam consecutive lanes.  On return every lane holds, in v[0..3], the team
// totals of slots base..base+3: kTeam = 8: base = ((lane>>2)&1)*8 + ((lane>>1)&1)*4 (lanes 2k, 2k+1 hold the same
// four); kTeam = 4: base = ((lane>>1)&1)*8 + (lane&1)*4 (every lane holds a different four).
__device__ __forceinline__ void team_reduce16(float (&v)[16], int lane) {
  {
    const bool hi = lane & (kTeam / 2);
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const float send = hi ? v[k] : v[k + 8];
      const float keep = hi ? v[k + 8] : v[k];
      v[k] = keep + __shfl_xor_sync(0xffffffffu, send, kTeam / 2);
    }
  }
  {
    const bool hi = lane & (kTeam / 4);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const float send = hi ? v[k] : v[k + 4];
      const float keep = hi ? v[k + 4] : v[k];
      v[k] = keep + __shfl_xor_sync(0xffffffffu, send, kTeam / 4);
    }
  }
  if (kTeam == 8) {
#pragma unroll
    for (int k = 0; k < 4; ++k) v[k] += __shfl_xor_sync(0xffffffffu, v[k], 1);
  }
}

// Sum 32 per-lane values over the warp: on return lane l holds the total of slot l.
__device__ __forceinline__ float warp_reduce32_transposed(float (&v)[32], int lane) {
#pragma unroll
  for (int h = 16; h >= 1; h >>= 1) {
    const bool hi = lane & h;
#pragma unroll
    for (int k = 0; k < h; ++k) {
      const float send = hi ? v[k] : v[k + h];
      const float keep = hi ? v[k + h] : v[k];
      v[k] = keep + __shfl_xor_sync(0xffffffffu, send, h);
    }
  }
  return v[0];
}

template <bool DEPTH_ONLY, bool DEV>
__global__ void __launch_bounds__(kThreadsB, SATSPLAT_BWD_MINB) blend_backward_kernel(const __grid_constant__ BwdParams P) {
  const CamRef<DEV> cam{P.cam, P.cam_dev};
  const ShRef<DEV> sh{P.sh, P.sh_dev};
  constexpr int kRecV = DEPTH_ONLY ? 3 : 4;
  __shared__ float4 s_wrec[kWarpsB][32][kRecV];   // per warp: records of the current group's survivors
  __shared__ int2 s_widx[kWarpsB][32];            //           and their (list index, surfel id)
  // per warp: pending pairs (s, t, w, source lane | low-pass flag) and their local coordinates: (u, v), or (dx, dy)
  // for low-pass pairs; kSegs segments of up to 32 pairs each (dynamic shared memory: kPairBytes per CTA)
  extern __shared__ float4 s_dyn[];

  // CTA blockIdx.y holds warps [blockIdx.y * kWarpsB, +kWarpsB) of tile column blockIdx.x; a tile has 8 warps (8x4 px each)
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int gw = blockIdx.y * kWarpsB + warp, ty = gw >> 3, wi = gw & 7;
  const int tile = ty * P.cam.TX + blockIdx.x;
  const uint32_t start = P.ranges[2 * tile];
  const int bx0 = blockIdx.x * kTile + (wi & 1) * 8, by0 = ty * kTile + (wi >> 1) * 4;
  const int ix = bx0 + (lane & 7), iy = by0 + (lane >> 3);
  const bool inside = ix < P.cam.W && iy < P.cam.H;
  const float px = (float)ix + 0.5f, py = (float)iy + 0.5f;
  const size_t o = (size_t)iy * P.cam.W + ix;
  const float wx0 = (float)bx0 + 0.5f, wx1 = wx0 + 7.0f;
  const float wy0 = (float)by0 + 0.5f, wy1 = wy0 + 3.0f;

  // ---- per-pixel state and epilogue backward ----
  float T = 1.f, Tf = 1.f, zref = 0.f, M1 = 0.f, M2 = 0.f, A = 0.f;
  float va0 = 0.f, va1 = 0.f, va2 = 0.f, vN0 = 0.f, vN1 = 0.f, vN2 = 0.f, vD = 0.f, vL = 0.f, vmed = 0.f, vT = 0.f;
  int last = 0, mi = -1;
  if (inside) {
    const float4 a = P.px_a[o];
    const int2 li = P.px_i[o];
    Tf = a.x; T = Tf; A = 1.0f - Tf; last = li.x; mi = li.y;
    if (DEPTH_ONLY) {
      // sun_depth = sum w (z - z_bg) + z_bg  (since sum w + T_f = 1): phi = v (z - z_bg), no T_f term
      vD = P.v_sun_in[o];
      zref = cam.z_bg();
      // A texel no view pixel looked up has no upstream gradient (40-60 % of a sun map at C3): every gradient term of its
      // pairs is exactly zero, so it takes no part in the walk (a block of such texels skips the walk altogether).
      if (vD == 0.f) last = 0;
    }
  }
  if (!DEPTH_ONLY) {
    float red[32];
#pragma unroll
    for (int k = 0; k < 32; ++k) red[k] = 0.f;
    if (inside) {
      const float4 a = P.px_a[o];
      zref = a.y; M1 = a.z; M2 = a.w;
      const float4 b = P.px_b[o];
      float vI0 = 0.f, vI1 = 0.f, vI2 = 0.f, vA = 0.f;
      if (P.v_rgba) { const float4 t = P.v_rgba[o]; vI0 = t.x; vI1 = t.y; vI2 = t.z; vA = t.w; }
      if (P.v_geom) { const float4 t = P.v_geom[o]; vN0 = t.x; vN1 = t.y; vN2 = t.z; vD = t.w; }
      if (P.v_aux) { const float4 t = P.v_aux[o]; vmed = t.x; vL = t.y; }
      float cc[12];
#pragma unroll
      for (int k = 0; k < 12; ++k) cc[k] = sh.cc(k);
      const float am0 = sh.ambient(0), am1 = sh.ambient(1), am2 = sh.ambient(2);
      const float V = b.w;
      const float ac0 = cc[0] * b.x + cc[1] * b.y + cc[2] * b.z + cc[3];
      const float ac1 = cc[4] * b.x + cc[5] * b.y + cc[6] * b.z + cc[7];
      const float ac2 = cc[8] * b.x + cc[9] * b.y + cc[10] * b.z + cc[11];
      const float s0 = V + (1.f - V) * am0, s1 = V + (1.f - V) * am1, s2 = V + (1.f - V) * am2;
      const float vs0 = vI0 * ac0, vs1 = vI1 * ac1, vs2 = vI2 * ac2;     // d/d shade
      const float vc0 = vI0 * s0, vc1 = vI1 * s1, vc2 = vI2 * s2;        // d/d corrected albedo
      const float vV = vs0 * (1.f - am0) + vs1 * (1.f - am1) + vs2 * (1.f - am2);
      red[0] = vc0 * b.x; red[1] = vc0 * b.y; red[2] = vc0 * b.z; red[3] = vc0;
      red[4] = vc1 * b.x; red[5] = vc1 * b.y; red[6] = vc1 * b.z; red[7] = vc1;
      red[8] = vc2 * b.x; red[9] = vc2 * b.y; red[10] = vc2 * b.z; red[11] = vc2;
      red[12] = vs0 * (1.f - V); red[13] = vs1 * (1.f - V); red[14] = vs2 * (1.f - V);
      va0 = cc[0] * vc0 + cc[4] * vc1 + cc[8] * vc2;
      va1 = cc[1] * vc0 + cc[5] * vc1 + cc[9] * vc2;
      va2 = cc[2] * vc0 + cc[6] * vc1 + cc[10] * vc2;
      if (P.sh.shadows_on) {
        const float D = __fmaf_rn(zref, A, M1);
        const ShadowTap t = shadow_tap(sh, cam, P.sh.sun_w, P.sh.sun_h, px, py, D, Tf);
        if (t.in_map) {
          const int x0 = t.x0, y0 = t.y0, x1 = t.x1, y1 = t.y1;
          const float fx = t.fx, fy = t.fy, h = t.h;
          const float* Dm = P.sh.sun_depth;
          const int SW = P.sh.sun_w;
          const float d00 = __ldg(Dm + y0 * SW + x0), d01 = __ldg(Dm + y0 * SW + x1);
          const float d10 = __ldg(Dm + y1 * SW + x0), d11 = __ldg(Dm + y1 * SW + x1);
          const float v_gap = -sh.slope() * V * (1.f - V) * vV;
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
          v_zv -= sh.reproj(2) * v_xs + sh.reproj(6) * v_ys;   // h = b_z - z_v
          red[15] = v_xs * px; red[16] = v_xs * py; red[17] = v_xs * h; red[18] = v_xs;
          red[19] = v_ys * px; red[20] = v_ys * py; red[21] = v_ys * h; red[22] = v_ys;
          vD += v_zv;                 // z_v = D + T_f z_bg
          vT += cam.z_bg() * v_zv;
        }
      }
      vT += -vA + va0 * cam.bg(0) + va1 * cam.bg(1) + va2 * cam.bg(2);   // A = 1 - T_f ; albedo = C + T_f bg
      vT -= vD * zref;                                                          // D = M1' + z_ref (1 - T_f)
      // a pixel without any upstream gradient (masked out of the loss) contributes exact zeros: it skips the walk
      if (vI0 == 0.f && vI1 == 0.f && vI2 == 0.f && vA == 0.f && vN0 == 0.f && vN1 == 0.f && vN2 == 0.f && vD == 0.f && vmed == 0.f &&
          vL == 0.f)
        last = 0;
    }
    // ---- reduce the 23 epilogue gradients over the warp (transposed butterfly); one RED per value into one of kRedCopies
    // copies of the 23-vector (spread by warp: no hot address, and no CTA barrier); add_small sums the copies ----
    if (P.red) {
      const float r = warp_reduce32_transposed(red, lane);
      if (lane < 23 && r != 0.f) atomicAdd(P.red + (gw & (kRedCopies - 1)) * 32 + lane, r);
    }
  }
  const float TfvT = Tf * vT;
  const float zmean = A > 0.f ? M1 / A : 0.f;          // weighted mean depth of the pixel (shifted frame)
  const float zvar = A > 0.f ? fmaxf(M2 - M1 * zmean, 0.f) : 0.f;
  float Ssum = 0.f;
  const unsigned lt_mask = (1u << lane) - 1u;
  const int team = lane / kTeam, tl = lane % kTeam;
  float4* const p4 = s_dyn + warp * (kSegs * 32);
  float2* const p2 = reinterpret_cast<float2*>(s_dyn + kWarpsB * (kSegs * 32)) + warp * (kSegs * 32);
  // pending (warp, surfel) segments: team q keeps surfel id and pair count of segment q in its lanes' registers
  int nseg = 0, wmax = 0, my_cnt = 0;
  uint32_t my_id = 0;

  // Accumulate the pending segments: team q walks the pairs of segment q (8 at a time), sums the 18 moments,
  // reduces them over its 8 lanes and adds them to the surfel's gradient record with vector REDs.
  auto flush = [&]() {
    __syncwarp();
    float acc[16], e0 = 0.f, e1 = 0.f;
#pragma unroll
    for (int k = 0; k < 16; ++k) acc[k] = 0.f;
    for (int i0 = 0; i0 < wmax; i0 += kTeam) {   // warp-uniform trip count: the loop body shuffles
      const int i = i0 + tl;
      float4 q = make_float4(0.f, 0.f, 0.f, 0.f);
      float2 ab = make_float2(0.f, 0.f);
      if (i < my_cnt) { q = p4[team * 32 + i]; ab = p2[team * 32 + i]; }
      const int info = __float_as_int(q.w);
      const bool lp = info & 32;
      const float s_np = lp ? 0.f : q.x, s_lp = lp ? q.x : 0.f, t_np = lp ? 0.f : q.y;
      const float su = s_np * ab.x, sv = s_np * ab.y;
      acc[0] += su * ab.x; acc[1] += su * ab.y; acc[2] += sv * ab.y; acc[3] += su;
      acc[4] += sv; acc[5] += t_np * ab.x; acc[6] += t_np * ab.y; acc[7] += t_np;
      acc[8] += s_lp * ab.x; acc[9] += s_lp * ab.y; acc[10] += q.y; acc[11] += q.x;
      if (!DEPTH_ONLY) {
        const int src = info & 31;
        acc[12] += q.z * __shfl_sync(0xffffffffu, va0, src);
        acc[13] += q.z * __shfl_sync(0xffffffffu, va1, src);
        acc[14] += q.z * __shfl_sync(0xffffffffu, va2, src);
        acc[15] += q.z * __shfl_sync(0xffffffffu, vN0, src);
        e0 += q.z * __shfl_sync(0xffffffffu, vN1, src);
        e1 += q.z * __shfl_sync(0xffffffffu, vN2, src);
      }
    }
    team_reduce16(acc, lane);
    if (!DEPTH_ONLY) {
#pragma unroll
      for (int d = kTeam / 2; d > 0; d >>= 1) {
        e0 += __shfl_xor_sync(0xffffffffu, e0, d);
        e1 += __shfl_xor_sync(0xffffffffu, e1, d);
      }
    }
    if (my_cnt > 0) {
      float* dst = P.vrec + (size_t)my_id * kVrec;
      if (kTeam == 8) {
        const int base = ((tl >> 2) & 1) * 8 + ((tl >> 1) & 1) * 4;
        if (!(tl & 1)) {
          if (!DEPTH_ONLY || base < 12) red_add_v4(dst + base, acc[0], acc[1], acc[2], acc[3]);
        } else if (!DEPTH_ONLY && tl == 1) {
          red_add_v2(dst + 16, e0, e1);
        }
      } else {
        const int base = ((tl >> 1) & 1) * 8 + (tl & 1) * 4;
        if (!DEPTH_ONLY || base < 12) red_add_v4(dst + base, acc[0], acc[1], acc[2], acc[3]);
        if (!DEPTH_ONLY && tl == 3) red_add_v2(dst + 16, e0, e1);
      }
    }
    nseg = 0; wmax = 0; my_cnt = 0;
    __syncwarp();
  };

  // ---- the walk: every warp is on its own (no CTA barrier below this line) ----
  // The tile list is consumed in groups of 32 entries, last group first.  Per group: lane l takes entry l, tests its
  // bounding box against the warp's 8x4 block (ballot), and the survivors' records are gathered into the warp's
  // shared-memory slots in walk order.  Surfel ids are fetched two groups ahead and boxes one group ahead, so only
  // the record gather waits on memory.
  const int wlast = __reduce_max_sync(0xffffffffu, last);   // nothing beyond this index matters to this warp
  float4 (*const wrec)[kRecV] = s_wrec[warp];
  int2* const widx = s_widx[warp];
  const unsigned gt_mask = ~((2u << lane) - 1u);
  constexpr uint32_t kNoId = 0xffffffffu;
  auto fetch_id = [&](int cc) -> uint32_t {
    const int idx = cc * 32 + lane;
    return (cc >= 0 && idx < wlast) ? P.vals[start + idx] : kNoId;
  };
  const float4 bb_none = make_float4(1e30f, -1e30f, 1e30f, -1e30f);
  int c = (wlast + 31) / 32 - 1;
  uint32_t id_cur = fetch_id(c);
  float4 bb_cur = id_cur != kNoId ? P.bbox[id_cur] : bb_none;
  uint32_t id_nxt = fetch_id(c - 1);
  for (; c >= 0; --c) {
    const float4 bb_nxt = id_nxt != kNoId ? P.bbox[id_nxt] : bb_none;
    const uint32_t id_nn = fetch_id(c - 2);
    const bool hit = bb_cur.x <= wx1 && bb_cur.y >= wx0 && bb_cur.z <= wy1 && bb_cur.w >= wy0;
    const unsigned mask = __ballot_sync(0xffffffffu, hit);
    const int nsurv = __popc(mask);
    if (hit) {
      const int slot = __popc(mask & gt_mask);   // highest list index first
      const float4* r = P.rec + 4 * (size_t)id_cur;
      const float4 q0 = r[0], q1 = r[1], q2 = r[2];
      wrec[slot][0] = q0; wrec[slot][1] = q1; wrec[slot][2] = q2;
      if (!DEPTH_ONLY) wrec[slot][3] = r[3];
      widx[slot] = make_int2(c * 32 + lane, (int)id_cur);
    }
    __syncwarp();
    // the depth-only pass evaluates two survivors per trip (independent instruction streams for the scheduler) and
    // composites them in order; the view pass has no registers to spare for that and takes them one by one
    struct Eval { const float4* e; int2 ji; PairEval p; float zc; bool active; };
    auto evaluate = [&](int sv) -> Eval {
      Eval E;
      E.e = wrec[sv];
      E.ji = widx[sv];
      const float4 r0 = E.e[0], r1 = E.e[1];
      E.p = pair_eval(r0, r1, px, py);       // the forward's arithmetic, bit for bit: same decisions
      E.zc = r1.w;
      E.active = (E.ji.x < last) && (E.p.rho <= kRhoCut) && (E.p.a >= kAlphaMin);
      return E;
    };
    auto composite = [&](const Eval& E) {
      const unsigned hm = __ballot_sync(0xffffffffu, E.active);
      if (hm == 0) return;
      if (E.active) {
        const float4 r2 = E.e[2];
        const bool lowpass = !(E.p.rho3 <= E.p.rho2);
        const float z = pair_depth(E.p, E.zc, r2.x, r2.y);
        const float zs = z - zref;
        const float rc = fast_rcp(1.0f - E.p.a);
        const float Ti = T * rc;
        const float w = E.p.a * Ti;
        float phi, v_z;
        if (DEPTH_ONLY) {
          phi = vD * zs;
          v_z = w * vD;
        } else {
          const float4 r3 = E.e[3];
          // psi = z^2 A - 2 z M1 + M2 = A (z - m)^2 + (M2 - M1^2 / A) with m = M1 / A: no cancellation per pair
          const float dz = zs - zmean;
          const float psi = A * dz * dz + zvar;
          phi = va0 * r2.z + va1 * r2.w + va2 * r3.x + vN0 * r3.y + vN1 * r3.z + vN2 * r3.w + vD * zs + vL * psi;
          v_z = w * (vD + 2.0f * vL * A * dz) + ((E.ji.x == mi) ? vmed : 0.f);
        }
        const float v_a = Ti * phi - (Ssum + TfvT) * rc;
        Ssum += w * phi;
        T = Ti;
        const float v_rho = (E.p.aG < kAlphaMax) ? -0.5f * E.p.aG * v_a : 0.f;   // alpha' = alpha G unless clamped
        const int pos = nseg * 32 + __popc(hm & lt_mask);
        p4[pos] = make_float4(v_rho, v_z, w, __int_as_float(lane | (lowpass ? 32 : 0)));
        p2[pos] = lowpass ? make_float2(E.p.dx, E.p.dy) : make_float2(E.p.u, E.p.v);
      }
      const int cnt = __popc(hm);
      if (team == nseg) { my_cnt = cnt; my_id = (uint32_t)E.ji.y; }
      wmax = max(wmax, cnt);
      if (++nseg == kSegs) flush();
    };
    int sv = 0;
    if (DEPTH_ONLY) {
      for (; sv + 1 < nsurv; sv += 2) {
        const Eval E0 = evaluate(sv), E1 = evaluate(sv + 1);
        composite(E0);
        composite(E1);
      }
    }
    for (; sv < nsurv; ++sv) composite(evaluate(sv));
    __syncwarp();
    id_cur = id_nxt; bb_cur = bb_nxt; id_nxt = id_nn;
  }
  if (nseg) flush();
}

constexpr int kPairBytesB = kWarpsB * kSegs * 32 * (int)(sizeof(float4) + sizeof(float2));

// the dynamic shared-memory limit is a per-device function attribute: set for the current device by satsplat_create
cudaError_t init_blend_backward_attrs() {
  cudaError_t e = cudaFuncSetAttribute(blend_backward_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kPairBytesB);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(blend_backward_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kPairBytesB);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(blend_backward_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kPairBytesB);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(blend_backward_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kPairBytesB);
  return e;
}

cudaError_t launch_blend_backward(satsplat_ctx* c, const DevShading& sh, const float* sh_dev, const float* v_rgba, const float* v_geom,
                                  const float* v_aux, const float* v_sun_depth_in, bool depth_only, bool want_epilogue_sums,
                                  float* v_sun_depth, cudaStream_t s) {
  BwdParams P;
  P.cam = c->cam;
  P.sh = sh;
  P.cam_dev = c->cam_dev;
  P.sh_dev = sh_dev;
  P.ranges = c->ranges;
  P.vals = c->vals[c->sorted];
  P.rec = c->rec;
  P.bbox = c->bbox;
  P.v_rgba = reinterpret_cast<const float4*>(v_rgba);
  P.v_geom = reinterpret_cast<const float4*>(v_geom);
  P.v_aux = reinterpret_cast<const float4*>(v_aux);
  P.v_sun_in = v_sun_depth_in;
  P.px_a = c->px_a;
  P.px_b = c->px_b;
  P.px_i = c->px_i;
  P.vrec = c->vrec;
  P.v_sun_depth = v_sun_depth;
  const bool want_red = !depth_only && want_epilogue_sums;
  P.red = want_red ? c->red_buf : nullptr;
  if (want_red) {
    const cudaError_t e = cudaMemsetAsync(c->red_buf, 0, kRedCopies * 32 * sizeof(float), s);
    if (e != cudaSuccess) return e;
  }
  const dim3 grid(c->cam.TX, c->cam.TY * (8 / kWarpsB));
  constexpr int kPairBytes = kPairBytesB;
  ++g_kernel_launches;
  const bool dev = c->cam_dev != nullptr;
  if (depth_only) {
    if (dev) blend_backward_kernel<true, true><<<grid, kThreadsB, kPairBytes, s>>>(P);
    else blend_backward_kernel<true, false><<<grid, kThreadsB, kPairBytes, s>>>(P);
  } else {
    if (dev) blend_backward_kernel<false, true><<<grid, kThreadsB, kPairBytes, s>>>(P);
    else blend_backward_kernel<false, false><<<grid, kThreadsB, kPairBytes, s>>>(P);
  }
  return cudaGetLastError();
}

}  // namespace satsplat

// losses.cu — (f1) the loss stage that turns one rendered view into the upstream gradients of the rasteriser's
// backward: image L1 + SSIM (11x11 Gaussian window, sigma 1.5, zero padding, as used by 3DGS), mean depth distortion, and
// the normal-consistency term between the rendered normal and the normal of the depth map (Eq. 13;
// weights :349).  Three kernels:
//   ssim_stats_kernel    ROLLING column strips: a CTA owns 64 image columns and a run of rows and marches down the rows;
//                        thread = (column, colour channel).  Per row: the 74 pixels of I and I* (strip + 5-pixel halo)
//                        are copied into an 8-row ring in shared memory by cp.async (issued four rows ahead; the 4-byte
//                        copies transpose the float4 pixels into per-channel (I, I*) pairs; the CTA barrier per row is an
//                        mbarrier whose arrive and wait are one row apart), the thread blurs the moments
//                        (I, I*, I^2 + I*^2, I I*) of its channel horizontally (11 taps) and scatters the result
//                        into the 11 pending output rows it keeps in REGISTERS (vertical pass: no shared-memory round
//                        trip, no vertical halo recomputation); the row that completes gives the SSIM value and its
//                        three partial derivatives (w.r.t. mu_1, E[I^2], E[I I*]), written as one float4 per channel
//                        (48 B / pixel).  The moments are carried as (m1, m2) / (e11, e22) pairs in packed f32x2
//                        arithmetic (fma.rn.f32x2: two FMAs per issue slot; the kernel is bound by instruction issue).
//   normal_term_kernel   32x16 tiles: Eq. 13.  The world point map is affine in the depth, so the un-normalised normal
//                        is c = c0 + dx c1 + dy c2 with dx, dy the central depth differences and three constant vectors
//                        per camera; its gradient is gathered from the four neighbours; writes v_geom, v_aux and the
//                        depth gradient v_zv (4 B / pixel scratch), reduces the distortion and normal terms.  Runs on a
//                        side stream BESIDE ssim_stats_kernel (it depends on the rendered images only).
//   ssim_adjoint_kernel  rolling strips, vertical pass first: blur of the three derivative maps per channel (the window is
//                        symmetric: adjoint = blur) -> dSSIM/dI; L1 sign; writes v_rgba (alpha channel from v_zv),
//                        reduces the L1 term.  Three phases per row on three different rows, one barrier per row.
#include "internal.cuh"

#include <cstdlib>
#include <map>
#include <mutex>

namespace satsplat {

constexpr int kSW = 64;                 // columns of a strip
constexpr int kSR = 5;                  // window radius
constexpr int kSIn = kSW + 2 * kSR;     // staged columns: strip + halo = 74
constexpr int kSThreads = 3 * kSW;      // thread = (column, channel)
constexpr int kNX = 32, kNY = 16;       // tile of the normal-term kernel (256 threads, two rows each)

struct LossParams {
  int W, H;
  int rows;                        // rows per strip segment (rolling kernels)
  float g[11];                     // Gaussian window (sums to 1)
  float w_l1, w_ssim, w_dist, w_normal;
  float inv_npx;                   // 1 / (H W)
  float c0[3], c1[3], c2[3], sgn;  // Eq. 13 constants: c = c0 + dx c1 + dy c2, N_d = sgn c / |c|
  float z_bg;
  const float4* rgba;
  const float4* geom;
  const float4* aux;
  const float4* target;
  float4* part;                    // [3][H*W] per channel: (d/d mu_1, d/d E[I^2], d/d E[I I*], 0) of the SSIM map
  float* vzv;                      // [H*W] dL/dz_v of the normal term
  float4* v_rgba;
  float4* v_geom;
  float4* v_aux;
  float* sums;                     // [0] sum |I - I*|, [1] sum SSIM map, [2] sum distortion, [3] sum (1 - A N_r.N_d)
};

constexpr float kC1 = 0.01f * 0.01f, kC2 = 0.03f * 0.03f;

// packed pairs of fp32 (sm_100: one issue slot for two FMAs)
using f32x2 = unsigned long long;
__device__ __forceinline__ f32x2 pk(float lo, float hi) {
  f32x2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r;
}
__device__ __forceinline__ void upk(f32x2 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
  f32x2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
  f32x2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r;
}

// cp.async of BYTES (4, 8, 16) from global to shared memory, zero-filled when !valid (the source is then not read)
// (sa: shared-window address, taken once per thread with smem_addr(): the conversion reads a special register)
__device__ __forceinline__ unsigned smem_addr(const void* smem) { return (unsigned)__cvta_generic_to_shared(smem); }
template <int BYTES>
__device__ __forceinline__ void cp_async_zfill(unsigned sa, const void* gmem, bool valid) {
  const int src = valid ? BYTES : 0;
  if constexpr (BYTES == 16)
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(sa), "l"(gmem), "r"(src) : "memory");
  else
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2, %3;" ::"r"(sa), "l"(gmem), "n"(BYTES), "r"(src) : "memory");
}

constexpr int kStages = 4;              // rows in flight in the rolling kernels' shared-memory ring

// mbarrier as a CTA barrier whose two halves are an iteration apart (arrive now, wait at the top of the next row):
// the warps of a CTA may drift by one row instead of meeting at every row
__device__ __forceinline__ void mbar_init(unsigned sa, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(sa), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned sa) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(sa) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned sa, unsigned parity) {
  asm volatile("{\n .reg .pred p;\n WAIT_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n @!p bra WAIT_%=;\n}\n" ::"r"(sa),
               "r"(parity)
               : "memory");
}

template <int NT>
__device__ __forceinline__ float block_sum(float v, float* s_red) {   // NT threads (a multiple of 32, <= 1024); valid in thread 0
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
  if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = v;
  __syncthreads();
  float r = 0.f;
  if (threadIdx.x == 0) {
#pragma unroll
    for (int k = 0; k < NT / 32; ++k) r += s_red[k];
  }
  __syncthreads();
  return r;
}

// Slot of output row y in the rotating register file of pending rows: with the rows of a segment processed in blocks of
// 11 (j = position in the block), input row r = r0 + j feeds output row r + 5 - k with weight g[k]; that row lives in slot
// (j + 5 - k) mod 11, a compile-time constant once j and k are unrolled.  The row completed by input row r is r - 5
// (k = 10): slot (j + 6) mod 11, which the next input row re-opens with its k = 0 term.
__host__ __device__ constexpr int slot_of(int j, int k) { return (j + 5 - k + 11) % 11; }

#ifndef SATSPLAT_STATS_MINB
#define SATSPLAT_STATS_MINB 3
#endif
__global__ void __launch_bounds__(kSThreads, SATSPLAT_STATS_MINB) ssim_stats_kernel(const __grid_constant__ LossParams P) {
  constexpr int kRing = 8, kAhead = 4;        // ring of staged rows; a row is copied kAhead rows before it is read
  __shared__ f32x2 s_ab[kRing][3][kSIn];      // (I, I*) per channel, zero outside the image
  __shared__ __align__(8) unsigned long long s_bar;
  __shared__ float s_red[kSThreads / 32];
  const int tid = threadIdx.x, col = tid & (kSW - 1), c = tid >> 6;
  const int x0 = blockIdx.x * kSW, x = x0 + col;
  const int ys = blockIdx.y * P.rows, ye = min(P.H, ys + P.rows);
  const size_t n = (size_t)P.W * P.H;
  // staging role: threads 0..73 copy I, 74..147 copy I* of one pixel of the row (three 4-byte cp.async: the copy
  // transposes the float4 pixels into per-channel (I, I*) pairs)
  const int which = tid >= kSIn ? 1 : 0, lx = tid - which * kSIn;
  const int gx = x0 - kSR + lx;
  const bool stager = tid < 2 * kSIn;
  const bool st_in = stager && gx >= 0 && gx < P.W;
  const float* const src = reinterpret_cast<const float*>(which ? P.target : P.rgba);
  long long soff = ((long long)(ys - kSR) * P.W + gx) * 4;   // float offset of (row, gx), advanced by one row per stage_row()
  int srow = ys - kSR, sstage = 0;
  const unsigned sa_stage = smem_addr(reinterpret_cast<float*>(&s_ab[0][0][stager ? lx : 0]) + which);
  auto stage_row = [&]() {   // called for consecutive rows; always commits a group
    if (stager) {
      const bool ok = st_in && (unsigned)srow < (unsigned)P.H;
      const float* g = ok ? src + soff : src;
      const unsigned d = sa_stage + sstage * (unsigned)sizeof(s_ab[0]);
      cp_async_zfill<4>(d, g, ok);
      cp_async_zfill<4>(d + 8 * kSIn, g + 1, ok);
      cp_async_zfill<4>(d + 16 * kSIn, g + 2, ok);
    }
    cp_async_commit();
    soff += 4ll * P.W; ++srow; sstage = (sstage + 1) & (kRing - 1);
  };
  f32x2 w2[6];
#pragma unroll
  for (int k = 0; k < 6; ++k) w2[k] = pk(P.g[k], P.g[k]);
  // pending output rows: (mu_1, mu_2) and (E[I^2] + E[I*^2], E[I I*]) -- SSIM and its derivatives need the two second
  // moments only through their sum, so four blurred maps per channel are carried, not five
  f32x2 accM[11], accS[11];
#pragma unroll
  for (int k = 0; k < 11; ++k) { accM[k] = 0ull; accS[k] = 0ull; }
  float ssim_sum = 0.f;
  const int r_first = ys - kSR, r_last = ye - 1 + kSR;
  // Row pipeline.  Phase k of the mbarrier completes when every thread's copies of row r_first + k have landed; a thread
  // arrives for phase k + 1 at the top of step k (before its arithmetic) and waits for phase k at the top of step k: a
  // warp runs at most one row ahead of the slowest.  The stage overwritten at step k (row k + 4) was read at step k - 4.
  const unsigned bar = smem_addr(&s_bar);
  if (tid == 0) mbar_init(bar, kSThreads);
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  __syncthreads();
#pragma unroll
  for (int k = 0; k < kAhead; ++k) stage_row();
  cp_async_wait<kAhead - 1>();
  mbar_arrive(bar);
  for (int r0 = r_first; r0 <= r_last; r0 += 11) {
#pragma unroll
    for (int j = 0; j < 11; ++j) {
      const int r = r0 + j;
      if (r > r_last) break;
      const int it = r - r_first, buf = it & (kRing - 1);
      mbar_wait(bar, it & 1);         // everybody's copies of row r have landed; everybody is done with row r - 2
      stage_row();                    // row r + 4 into the stage of row r - 4
      cp_async_wait<kAhead - 1>();    // this thread's copies of row r + 1 have landed
      mbar_arrive(bar);
      // horizontal pass of this thread's channel
      const f32x2* const row = &s_ab[buf][c][col];
      f32x2 hM = 0ull, hE = 0ull;
      float hX = 0.f;
#pragma unroll
      for (int k = 0; k < 11; ++k) {
        const f32x2 ab = row[k];
        const f32x2 wab = mul2(w2[k < 6 ? k : 10 - k], ab);
        float a, b, wa, wb;
        upk(ab, a, b);
        upk(wab, wa, wb);
        hM = fma2(w2[k < 6 ? k : 10 - k], ab, hM);
        hE = fma2(wab, ab, hE);
        hX = fmaf(wa, b, hX);
      }
      float h11, h22;
      upk(hE, h11, h22);
      const f32x2 hS = pk(h11 + h22, hX);
      // vertical pass: scatter into the pending rows (k = 0 opens a row)
#pragma unroll
      for (int k = 0; k < 11; ++k) {
        const int s = slot_of(j, k), kk = k < 6 ? k : 10 - k;
        if (k == 0) {
          accM[s] = mul2(w2[kk], hM); accS[s] = mul2(w2[kk], hS);
        } else {
          accM[s] = fma2(w2[kk], hM, accM[s]); accS[s] = fma2(w2[kk], hS, accS[s]);
        }
      }
      const int y = r - kSR;
      if (y >= ys && x < P.W) {   // the completed row
        const int s = slot_of(j, 10);
        float mu1, mu2, ess, e12;
        upk(accM[s], mu1, mu2);
        upk(accS[s], ess, e12);
        const float mm = mu1 * mu1 + mu2 * mu2, s12 = e12 - mu1 * mu2;
        const float a = 2.f * mu1 * mu2 + kC1, b = 2.f * s12 + kC2;
        const float cc = mm + kC1, d = (ess - mm) + kC2;          // sigma_1^2 + sigma_2^2 = E[I^2] + E[I*^2] - mu_1^2 - mu_2^2
        const float icc = __fdividef(1.0f, cc), id = __fdividef(1.0f, d), icd = icc * id;
        const float m = a * b * icd;
        const float d_mu1 = 2.f * mu2 * b * icd - m * 2.f * mu1 * icc;
        const float ds11 = -m * id;
        const float ds12 = 2.f * a * icd;
        const float dmu = d_mu1 - 2.f * mu1 * ds11 - mu2 * ds12;
        P.part[(size_t)c * n + (size_t)y * P.W + x] = make_float4(dmu, ds11, ds12, 0.f);
        ssim_sum += m;
      }
    }
  }
  cp_async_wait<0>();
  const float tot = block_sum<kSThreads>(ssim_sum, s_red);
  if (tid == 0) atomicAdd(P.sums + 1, tot);
}

// Eq. 13 at one pixel from its four depth neighbours: the unit normal N_d = sgn c / |c| and 1 / |c|
__device__ __forceinline__ void depth_normal(const LossParams& P, float dx, float dy, float nd[3], float& icn) {
  const float cx = P.c0[0] + dx * P.c1[0] + dy * P.c2[0], cy = P.c0[1] + dx * P.c1[1] + dy * P.c2[1];
  const float cz = P.c0[2] + dx * P.c1[2] + dy * P.c2[2];
  icn = rsqrtf(cx * cx + cy * cy + cz * cz);
  nd[0] = cx * icn; nd[1] = cy * icn; nd[2] = cz * icn;   // c / |c| (orientation applied by the caller)
}

__global__ void __launch_bounds__(256) normal_term_kernel(const __grid_constant__ LossParams P) {
  // one round of global loads: rendered normal + depth (geom) and alpha of the tile with a 2-pixel halo, everything
  // after that reads shared memory
  __shared__ float4 s_g[kNY + 4][kNX + 4];       // geom: (N_r, D), zero outside the image
  __shared__ float s_a[kNY + 4][kNX + 4];        // alpha
  __shared__ float s_zv[kNY + 4][kNX + 4];       // depth z_v = D + (1 - A) z_bg, zero outside the image
  __shared__ float s_vd[2][kNY + 2][kNX + 2];    // v_dx, v_dy: what each pixel's own term sends to its depth differences, halo 1
  __shared__ float s_red[8];
  const int x0 = blockIdx.x * kNX, y0 = blockIdx.y * kNY;
  const int lx = threadIdx.x & (kNX - 1), wy = threadIdx.x >> 5;
  const int x = x0 + lx;
  // own pixels' distortion (global loads issued with the rest)
  float dist = 0.f;
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    const int y = y0 + wy + h * (kNY / 2);
    if (x < P.W && y < P.H) dist += __ldg(&P.aux[(size_t)y * P.W + x].y);
  }
  for (int e = threadIdx.x; e < (kNY + 4) * (kNX + 4); e += 256) {
    const int ey = e / (kNX + 4), ex = e % (kNX + 4);
    const int gx = x0 + ex - 2, gy = y0 + ey - 2;
    float4 gm = make_float4(0.f, 0.f, 0.f, 0.f);
    float A = 0.f, zv = 0.f;
    if (gx >= 0 && gx < P.W && gy >= 0 && gy < P.H) {
      const size_t o = (size_t)gy * P.W + gx;
      gm = __ldg(P.geom + o);
      A = __ldg(&P.rgba[o].w);
      zv = gm.w + (1.0f - A) * P.z_bg;
    }
    s_g[ey][ex] = gm; s_a[ey][ex] = A; s_zv[ey][ex] = zv;
  }
  __syncthreads();
  for (int e = threadIdx.x; e < (kNY + 2) * (kNX + 2); e += 256) {
    const int ey = e / (kNX + 2), ex = e % (kNX + 2);
    const int gx = x0 + ex - 1, gy = y0 + ey - 1;
    float vdx = 0.f, vdy = 0.f;
    if (gx >= 1 && gx < P.W - 1 && gy >= 1 && gy < P.H - 1) {      // interior pixel of the image
      const float dx = s_zv[ey + 1][ex + 2] - s_zv[ey + 1][ex], dy = s_zv[ey + 2][ex + 1] - s_zv[ey][ex + 1];
      float nd[3], icn;
      depth_normal(P, dx, dy, nd, icn);
      const float4 gm = s_g[ey + 1][ex + 1];
      // v_Nd = -w_normal A N_r / npx ; v_c = sgn (v_Nd - n (n . v_Nd)) / |c|
      const float k = -P.w_normal * s_a[ey + 1][ex + 1] * P.inv_npx;
      const float v0 = k * gm.x, v1 = k * gm.y, v2 = k * gm.z;
      const float dt = nd[0] * v0 + nd[1] * v1 + nd[2] * v2;
      const float s = P.sgn * icn;
      const float vcx = s * (v0 - nd[0] * dt), vcy = s * (v1 - nd[1] * dt), vcz = s * (v2 - nd[2] * dt);
      vdx = vcx * P.c1[0] + vcy * P.c1[1] + vcz * P.c1[2];
      vdy = vcx * P.c2[0] + vcy * P.c2[1] + vcz * P.c2[2];
    }
    s_vd[0][ey][ex] = vdx;
    s_vd[1][ey][ex] = vdy;
  }
  __syncthreads();
  float nloss = 0.f;
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    const int ly = wy + h * (kNY / 2);
    const int y = y0 + ly;
    if (x < P.W && y < P.H) {
      const size_t o = (size_t)y * P.W + x;
      const float4 gm = s_g[ly + 2][lx + 2];
      const float A = s_a[ly + 2][lx + 2];
      float nd[3] = {0.f, 0.f, 0.f};
      if (x >= 1 && x < P.W - 1 && y >= 1 && y < P.H - 1) {
        const float dx = s_zv[ly + 2][lx + 3] - s_zv[ly + 2][lx + 1], dy = s_zv[ly + 3][lx + 2] - s_zv[ly + 1][lx + 2];
        float icn;
        depth_normal(P, dx, dy, nd, icn);
        nd[0] *= P.sgn; nd[1] *= P.sgn; nd[2] *= P.sgn;
      }
      nloss += 1.0f - A * (gm.x * nd[0] + gm.y * nd[1] + gm.z * nd[2]);
      // v_zv(x, y) = v_dx(x-1, y) - v_dx(x+1, y) + v_dy(x, y-1) - v_dy(x, y+1)
      const float v_zv = s_vd[0][ly + 1][lx] - s_vd[0][ly + 1][lx + 2] + s_vd[1][ly][lx + 1] - s_vd[1][ly + 2][lx + 1];
      const float kn = -P.w_normal * A * P.inv_npx;
      P.v_geom[o] = make_float4(kn * nd[0], kn * nd[1], kn * nd[2], v_zv);
      P.v_aux[o] = make_float4(0.f, P.w_dist * P.inv_npx, 0.f, 0.f);
      P.vzv[o] = v_zv;
    }
  }
  const float t2 = block_sum<256>(dist, s_red);
  const float t3 = block_sum<256>(nloss, s_red);
  if (threadIdx.x == 0) {
    atomicAdd(P.sums + 2, t2);
    atomicAdd(P.sums + 3, t3);
  }
}

// ssim_adjoint_kernel: vertical pass first.  A CTA owns 64 image columns and a run of rows; every step takes one new row
// of the derivative maps and runs three phases on three different rows (one barrier per step, double-buffered hand-over):
//   A  thread = (staged column of 74, channel): its float4 of the row (prefetched three rows ahead by a cp.async into a
//      slot of shared memory only this thread reads: a prefetch that holds no registers and needs no barrier) goes into
//      the 11 pending rows it keeps in registers (vertical blur); the completed row is handed over in shared memory
//      (9 maps x 74 columns);
//   B  thread = (map, 4 consecutive columns): horizontal blur of the row completed by the previous step: 16 values read
//      once (4 LDS.128) slide through the 11 taps in registers;
//   C  thread = pixel: dL/dI from the nine blurred maps of the row before that, L1 sign, float4 store of v_rgba (I, I*
//      and v_zv of the pixel prefetched the same way).
constexpr int kAThreads = 224;               // 7 warps: A on 222 threads, B on threads 0..143, C on threads 160..223
constexpr int kVP = 80;                      // staged row, padded to a multiple of 4 floats

#ifndef SATSPLAT_ADJ_MINB
#define SATSPLAT_ADJ_MINB 4
#endif
__global__ void __launch_bounds__(kAThreads, SATSPLAT_ADJ_MINB) ssim_adjoint_kernel(const __grid_constant__ LossParams P) {
  __shared__ __align__(16) float s_v[2][9][kVP];   // vertically blurred row, [map = 3 channel + (mu, 11, 12)][staged column]
  __shared__ __align__(16) float s_b[2][9][kSW];   // fully blurred row
  __shared__ float4 s_pa[kStages][kAThreads];      // A's prefetch slots
  __shared__ float4 s_ci[kStages][2][kSW];         // C's prefetch slots: I, I*
  __shared__ float s_cz[kStages][kSW];             //                     v_zv
  __shared__ float s_red[kAThreads / 32];
  const int tid = threadIdx.x;
  const int x0 = blockIdx.x * kSW;
  const int ys = blockIdx.y * P.rows, ye = min(P.H, ys + P.rows);
  const size_t n = (size_t)P.W * P.H;
  for (int e = tid; e < 2 * 9 * kVP; e += kAThreads) (&s_v[0][0][0])[e] = 0.f;
  // ---- role A
  const bool role_a = tid < 3 * kSIn;
  const int ch_a = role_a ? tid / kSIn : 0, sc_a = tid % kSIn;
  const int gx_a = x0 - kSR + sc_a;
  const bool in_a = role_a && gx_a >= 0 && gx_a < P.W;
  f32x2 w2[6];
#pragma unroll
  for (int k = 0; k < 6; ++k) w2[k] = pk(P.g[k], P.g[k]);
  // pending output rows in 12 rotating slots (11 live + 1 spare: a rotation period that is a multiple of the 4 prefetch
  // stages and of the 2 hand-over buffers, so that every shared-memory address below is a compile-time offset)
  f32x2 accP[12];   // vertically blurred (d/d mu_1, d/d E[I^2])
  float accQ[12];   // d/d E[I I*]
#pragma unroll
  for (int k = 0; k < 12; ++k) { accP[k] = 0ull; accQ[k] = 0.f; }
  // ---- role B
  const bool role_b = tid < 9 * (kSW / 4);
  const int q_b = tid / (kSW / 4), g_b = tid % (kSW / 4);
  // ---- role C
  const bool role_c = tid >= kAThreads - kSW;
  const int col_c = tid - (kAThreads - kSW), x_c = x0 + col_c;
  const bool in_c = role_c && x_c < P.W;
  // prefetch of step f (A: map row ys - 5 + f; C: image row ys + f - 12), one commit group per step, consecutive steps
  int fstep = 0;
  long long aoff = (long long)ch_a * n + (long long)(ys - kSR) * P.W + gx_a;
  long long coff = (long long)(ys - 12) * P.W + x_c;
  const int T = (ye - ys) + 2 * kSR;
  const unsigned sa_pa = smem_addr(&s_pa[0][tid]), sa_ci = smem_addr(&s_ci[0][0][role_c ? col_c : 0]),
                 sa_cz = smem_addr(&s_cz[0][role_c ? col_c : 0]);
  auto prefetch = [&](int st) {
    const bool ok_a = in_a && (unsigned)(ys - kSR + fstep) < (unsigned)P.H;
    cp_async_zfill<16>(sa_pa + st * (unsigned)sizeof(s_pa[0]), ok_a ? P.part + aoff : P.part, ok_a);
    if (role_c) {
      const bool ok_c = in_c && fstep >= 12 && fstep - 12 < ye - ys;
      cp_async_zfill<16>(sa_ci + st * (unsigned)sizeof(s_ci[0]), ok_c ? P.rgba + coff : P.rgba, ok_c);
      cp_async_zfill<16>(sa_ci + st * (unsigned)sizeof(s_ci[0]) + (unsigned)sizeof(s_ci[0][0]), ok_c ? P.target + coff : P.target, ok_c);
      cp_async_zfill<4>(sa_cz + st * (unsigned)sizeof(s_cz[0]), ok_c ? P.vzv + coff : P.vzv, ok_c);
    }
    cp_async_commit();
    aoff += P.W; coff += P.W; ++fstep;
  };
#pragma unroll
  for (int k = 0; k < kStages - 1; ++k) prefetch(k);
  const float k1 = P.w_l1 * P.inv_npx * (1.0f / 3.0f), ks = -P.w_ssim * P.inv_npx * (1.0f / 3.0f);
  float l1 = 0.f;
  // step t: A takes map row ys - 5 + t and completes output row y = ys - 10 + t, B works on row y - 1, C on row y - 2
  __syncthreads();
  for (int t0 = 0; t0 < T + 2; t0 += 12) {
#pragma unroll
    for (int j = 0; j < 12; ++j) {
      const int t = t0 + j;
      if (t >= T + 2) break;
      const int y = ys - 2 * kSR + t;
      constexpr int kMask = kStages - 1;
      const int st = j & kMask, bt = j & 1;     // = t & 3, t & 1
      cp_async_wait<kStages - 2>();   // this thread's prefetch of step t has landed
      if (t < T) {   // ---- A
        const float4 p = s_pa[st][tid];
        const f32x2 hP = pk(p.x, p.y);
        const float hQ = p.z;
#pragma unroll
        for (int k = 0; k < 11; ++k) {
          const int s = (j + 5 - k + 12) % 12, kk = k < 6 ? k : 10 - k;
          float wl, wh;
          upk(w2[kk], wl, wh);
          if (k == 0) {
            accP[s] = mul2(w2[kk], hP); accQ[s] = wl * hQ;
          } else {
            accP[s] = fma2(w2[kk], hP, accP[s]); accQ[s] = fmaf(wl, hQ, accQ[s]);
          }
        }
        if (y >= ys && role_a) {
          const int s = (j + 7) % 12;
          float bmu, b11;
          upk(accP[s], bmu, b11);
          float* d = &s_v[bt][ch_a * 3][sc_a];
          d[0] = bmu; d[kVP] = b11; d[2 * kVP] = accQ[s];
        }
      }
      if (role_b && y - 1 >= ys && y - 1 < ye) {   // ---- B
        const float4* src = reinterpret_cast<const float4*>(&s_v[bt ^ 1][q_b][4 * g_b]);
        const float4 a0 = src[0], a1 = src[1], a2 = src[2], a3 = src[3];
        const float v[16] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w, a2.x, a2.y, a2.z, a2.w, a3.x, a3.y, a3.z, a3.w};
        float o[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int k = 0; k < 11; ++k) {
          float wl, wh;
          upk(w2[k < 6 ? k : 10 - k], wl, wh);
#pragma unroll
          for (int i = 0; i < 4; ++i) o[i] = fmaf(wl, v[i + k], o[i]);
        }
        *reinterpret_cast<float4*>(&s_b[bt ^ 1][q_b][4 * g_b]) = make_float4(o[0], o[1], o[2], o[3]);
      }
      if (role_c && y - 2 >= ys && y - 2 < ye) {   // ---- C
        const float4 I = s_ci[st][0][col_c], J = s_ci[st][1][col_c];
        const float vz = s_cz[st][col_c];
        const float* b = &s_b[bt][0][col_c];
        const float Iv[3] = {I.x, I.y, I.z}, Jv[3] = {J.x, J.y, J.z};
        float vI[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const float d = Iv[c] - Jv[c];
          if (in_c) l1 += fabsf(d);
          const float sg = d > 0.f ? 1.f : (d < 0.f ? -1.f : 0.f);
          vI[c] = k1 * sg + ks * (b[(3 * c) * kSW] + 2.f * Iv[c] * b[(3 * c + 1) * kSW] + Jv[c] * b[(3 * c + 2) * kSW]);
        }
        if (in_c) P.v_rgba[(size_t)(y - 2) * P.W + x_c] = make_float4(vI[0], vI[1], vI[2], -P.z_bg * vz);
      }
      prefetch((j + kStages - 1) & kMask);   // step t + 3 into the slots of step t - 1
      __syncthreads();
    }
  }
  cp_async_wait<0>();
  const float t0s = block_sum<kAThreads>(l1, s_red);
  if (tid == 0) atomicAdd(P.sums + 0, t0s);
}

// Rows per strip segment: the strips x segments grid fills `waves` rounds of the CTAs the device holds at once (one round:
// every CTA marches in step, no tail), with at least 16 rows per segment (a segment recomputes 10 warm-up rows).
static int segment_rows(int W, int H, int ctas_per_sm) {
  static const double waves = [] { const char* e = getenv("SATSPLAT_LOSS_WAVES"); return e ? atof(e) : 1.0; }();   // tuning knob
  const int strips = (W + kSW - 1) / kSW;
  const long long target = (long long)(current_sm_count() * ctas_per_sm * waves);
  long long segs = target / strips;
  if (segs < 1) segs = 1;
  const long long most = (H + 15) / 16;
  if (segs > most) segs = most;
  return (int)((H + segs - 1) / segs);
}

// The normal-term kernel depends only on the rendered images: it runs on a side stream beside ssim_stats_kernel (which is
// bound by instruction issue at 18 warps per SM and leaves threads, registers and HBM bandwidth for it) and joins before
// ssim_adjoint_kernel.  Fork and join are events: no host synchronisation, capturable in a CUDA graph.
struct LossSide { cudaStream_t stream = nullptr; cudaEvent_t fork = nullptr, join = nullptr; };
static LossSide* loss_side() {
  static std::mutex mu;
  static std::map<int, LossSide> per_device;
  static const bool enabled = [] { const char* e = getenv("SATSPLAT_LOSS_OVERLAP"); return !e || atoi(e) != 0; }();   // 0: one stream (A/B)
  if (!enabled) return nullptr;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return nullptr;
  std::lock_guard<std::mutex> lock(mu);
  LossSide& S = per_device[dev];
  if (!S.stream) {
    if (cudaStreamCreateWithFlags(&S.stream, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&S.fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&S.join, cudaEventDisableTiming) != cudaSuccess) {
      S = LossSide();
      (void)cudaGetLastError();
      return nullptr;
    }
  }
  return &S;
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
  P.vzv = L.scratch + (size_t)12 * L.W * L.H;
  P.v_rgba = reinterpret_cast<float4*>(L.v_rgba); P.v_geom = reinterpret_cast<float4*>(L.v_geom);
  P.v_aux = reinterpret_cast<float4*>(L.v_aux);
  P.sums = L.sums;
  cudaError_t e = cudaMemsetAsync(L.sums, 0, 8 * sizeof(float), s);
  if (e != cudaSuccess) return e;
  static const int occ_stats = [] { int b = 0; cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, ssim_stats_kernel, kSThreads, 0); return b > 0 ? b : 1; }();
  static const int occ_adj = [] { int b = 0; cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, ssim_adjoint_kernel, kAThreads, 0); return b > 0 ? b : 1; }();
  const int strips = (L.W + kSW - 1) / kSW;
  g_kernel_launches += 3;
  LossSide* const side = loss_side();
  cudaStream_t sn = s;
  if (side) {
    if ((e = cudaEventRecord(side->fork, s)) != cudaSuccess) return e;
    if ((e = cudaStreamWaitEvent(side->stream, side->fork, 0)) != cudaSuccess) return e;
    sn = side->stream;
  }
  P.rows = segment_rows(L.W, L.H, occ_stats);
  ssim_stats_kernel<<<dim3(strips, (L.H + P.rows - 1) / P.rows), kSThreads, 0, s>>>(P);
  normal_term_kernel<<<dim3((L.W + kNX - 1) / kNX, (L.H + kNY - 1) / kNY), 256, 0, sn>>>(P);
  if (side) {
    if ((e = cudaEventRecord(side->join, sn)) != cudaSuccess) return e;
    if ((e = cudaStreamWaitEvent(s, side->join, 0)) != cudaSuccess) return e;
  }
  P.rows = segment_rows(L.W, L.H, occ_adj);
  ssim_adjoint_kernel<<<dim3(strips, (L.H + P.rows - 1) / P.rows), kAThreads, 0, s>>>(P);
  return cudaGetLastError();
}

}  // namespace satsplat

// internal.cuh — shared declarations of the CUDA path (NOT part of the C ABI; never seen by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

#include "../../include/satsplat.h"

namespace satsplat {

// ---- method constants ------------------------------------------------
constexpr int kTile = 16;
constexpr float kRhoCut = 9.0f;            // 3-sigma
constexpr float kAlphaMin = 1.0f / 255.0f;
constexpr float kAlphaMax = 0.99f;
constexpr float kTMin = 1e-4f;
constexpr float kDetEps = 1e-6f;           // |det(B'_xy R S')| <= eps -> degenerate
constexpr float kLogitCull = -5.5373342f;  // sigmoid(l) < 1/255
constexpr float kMinExtent = 2.1213204f;   // 3 sigma, sigma = 1/sqrt(2) px (Eq. 12)
constexpr float kDegenerateQ = 1e12f;      // Q = kDegenerateQ * I encodes "rho3 = +inf" for degenerate surfels

constexpr float kNegHalfLog2e = -0.72134752044448170368f;   // exp(-rho/2) = 2^(rho * kNegHalfLog2e)

enum : uint8_t { F_CULLED = 1, F_DEGENERATE = 2, F_FLIPPED = 4 };

// 2^x, one MUFU.EX2 (x is in [-6.5, 0] here: no range reduction, no denormals)
__device__ __forceinline__ float fast_exp2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// 1/x, one MUFU.RCP (x is in [0.01, 1] here)
__device__ __forceinline__ float fast_rcp(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// 16-byte asynchronous global -> shared copy (LDGSTS), and the wait for all but the n most recent commit groups
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  const uint32_t sa = (uint32_t)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// ---- device-side camera ------------------------------------------------------------------------------------
struct DevCamera {
  int W, H, TX, TY;
  float Fp[8];  // F + dF (fp32 add, Eq. 15)
  float vd[3];
  float b_z, z_bg;
  float bg[3];
};

struct DevShading {
  float cc[12];
  float ambient[3];
  int shadows_on;
  int sun_w, sun_h;
  const float* sun_depth;
  float reproj[8];
  float bias, slope;
};

// ---- device-resident camera block (row f2: satsplat_camera_chain writes it, the *_device calls read it) ---------------
// floats [0,16) view camera, [16,32) sun camera, [32,48) nearby camera, each (Fp[8], view_dir[3], b_z, z_bg, bg[3]);
// [48,76) shading of the view: cc[12], ambient[3], reproj[8], depth_bias, slope, 3 unused;  SATSPLAT_CAMERA_BLOCK_FLOATS = 80
constexpr int kCamFloats = 16;
constexpr int kBlockShading = 48;

// Camera / shading values of a kernel: kernel-argument copies (DEV = false: the host-struct calls) or loads from the
// device-resident block (DEV = true).  W, H, TX, TY, the sun map pointer and its size are host-known in both modes.
template <bool DEV>
struct CamRef {
  const DevCamera& c;
  const float* d;   // 16-float camera record of the block (DEV only)
  __device__ __forceinline__ float Fp(int k) const { return DEV ? __ldg(d + k) : c.Fp[k]; }
  __device__ __forceinline__ float vd(int k) const { return DEV ? __ldg(d + 8 + k) : c.vd[k]; }
  __device__ __forceinline__ float b_z() const { return DEV ? __ldg(d + 11) : c.b_z; }
  __device__ __forceinline__ float z_bg() const { return DEV ? __ldg(d + 12) : c.z_bg; }
  __device__ __forceinline__ float bg(int k) const { return DEV ? __ldg(d + 13 + k) : c.bg[k]; }
};
template <bool DEV>
struct ShRef {
  const DevShading& s;
  const float* d;   // 28-float shading record of the block (DEV only)
  __device__ __forceinline__ float cc(int k) const { return DEV ? __ldg(d + k) : s.cc[k]; }
  __device__ __forceinline__ float ambient(int k) const { return DEV ? __ldg(d + 12 + k) : s.ambient[k]; }
  __device__ __forceinline__ float reproj(int k) const { return DEV ? __ldg(d + 15 + k) : s.reproj[k]; }
  __device__ __forceinline__ float bias() const { return DEV ? __ldg(d + 23) : s.bias; }
  __device__ __forceinline__ float slope() const { return DEV ? __ldg(d + 24) : s.slope; }
};

// ---- record layout in HBM: 4 x float4 = 64 B per surfel, 64-B aligned --------------------------------------
//   r0 = (c_x, c_y, Q00, Q01)   r1 = (Q10, Q11, alpha, z_c)   r2 = (g0, g1, red, green)   r3 = (blue, n_x, n_y, n_z)
// The first two float4 are all the per-pair test needs; the last two are only read by contributing pairs.
// Gradient records (vrec) are kVrec floats of per-surfel moments: layout in blend_backward.cu.
constexpr int kVrec = 20;
constexpr int kRedCopies = 64;   // copies of the 23 epilogue-gradient sums (cc, ambient, reproj) the backward spreads its REDs over

// Per-tile pair counters / scatter cursors are spaced kCtrStride words apart: the 2 M returning atomics of a C3 pass land on
// 16 K counters; packed, 32 of them share a 128-byte line and serialise in one L2 atomic unit (measured)
#ifndef SATSPLAT_CTR_STRIDE
#define SATSPLAT_CTR_STRIDE 8
#endif
constexpr int kCtrStride = SATSPLAT_CTR_STRIDE;

// sort configuration
constexpr int kSortThreads = 256;
constexpr int kSortItems = 8;
constexpr int kSortTile = kSortThreads * kSortItems;  // 2048 keys
constexpr int kSortBlocks = 296;                      // fixed grid of the radix passes (K lives on the device; sizes the digit table)

struct Status {           // device-resident status words
  unsigned int K;         // duplicated keys of the last preprocess (may exceed capacity)
  unsigned int overflow;  // K > max_duplicates
  unsigned int pad[2];
};

// Conservative screen-space bounding box (x_min, x_max, y_min, y_max) of the pixel centres a splat can touch
// (rho <= 9 under Eq. 12): the 3-sigma ellipse of M = Q^-1, widened to the 3-sigma low-pass disc, slightly inflated
// so that fp32 rounding can never drop a contributor.  Used only to skip work; the per-pixel rho test decides.
__device__ __forceinline__ float4 splat_bbox(const float4 r0, const float4 r1) {
  const float det = r0.z * r1.y - r0.w * r1.x;
  const float id = 3.0f / fabsf(det);
  float ex = id * sqrtf(r1.y * r1.y + r0.w * r0.w);   // 3 |row 0 of M|
  float ey = id * sqrtf(r1.x * r1.x + r0.z * r0.z);   // 3 |row 1 of M|
  ex = fmaxf(ex, kMinExtent) * 1.0001f + 1e-3f;
  ey = fmaxf(ey, kMinExtent) * 1.0001f + 1e-3f;
  if (!(ex < 1e30f)) ex = 1e30f;                       // NaN / inf (det underflow) -> never culled
  if (!(ey < 1e30f)) ey = 1e30f;
  return make_float4(r0.x - ex, r0.x + ex, r0.y - ey, r0.y + ey);
}

// Shadow-test lookup shared by the forward epilogue and its backward so that both take the same in-map /
// texel decisions from the same bits.  The reprojection x_s = R_x x + k_h h + k_0 is evaluated
// in double precision: at 2048 px an fp32 x_s carries ~1e-4 px of rounding, which a building edge in the sun map
// (tens of metres per texel) turns into a visible error of the soft test and of every gradient through it.
struct ShadowTap {
  bool in_map;
  int x0, y0, x1, y1;
  float fx, fy, h, zv;
};
template <class SH, class CAM>
__device__ __forceinline__ ShadowTap shadow_tap(const SH& sh, const CAM& cam, int sun_w, int sun_h, float px, float py, float D, float T) {
  ShadowTap t;
  t.zv = __fmaf_rn(T, cam.z_bg(), D);        // z_v = D + T_f z_bg
  t.h = __fsub_rn(cam.b_z(), t.zv);          // world height seen at this pixel
  const double dpx = (double)px, dpy = (double)py, dh = (double)t.h;
  const double xs = fma((double)sh.reproj(2), dh, fma((double)sh.reproj(1), dpy, fma((double)sh.reproj(0), dpx, (double)sh.reproj(3))));
  const double ys = fma((double)sh.reproj(6), dh, fma((double)sh.reproj(5), dpy, fma((double)sh.reproj(4), dpx, (double)sh.reproj(7))));
  t.in_map = xs >= 0.5 && xs <= (double)sun_w - 0.5 && ys >= 0.5 && ys <= (double)sun_h - 0.5;
  const double tx = xs - 0.5, ty = ys - 0.5;
  // clamp in double before the conversion (far outside the map the product would overflow an int)
  t.x0 = (int)fmin(fmax(floor(tx), 0.0), (double)(sun_w - 1));
  t.y0 = (int)fmin(fmax(floor(ty), 0.0), (double)(sun_h - 1));
  t.fx = (float)(tx - (double)t.x0);
  t.fy = (float)(ty - (double)t.y0);
  t.x1 = min(t.x0 + 1, sun_w - 1);
  t.y1 = min(t.y0 + 1, sun_h - 1);
  return t;
}

// Per-(pixel, surfel) evaluation of Eq. 9 / Eq. 12, shared by the forward and the backward blend so that both take
// the same decisions (rho cut, alpha skip, depth branch, clamp) from the same bits: every operation is an explicitly
// rounded intrinsic, so the result does not depend on the contraction choices of the compiler in either kernel.
struct PairEval {
  float dx, dy, u, v, rho3, rho2, rho, aG, a;
};
__device__ __forceinline__ PairEval pair_eval(const float4 r0, const float4 r1, float px, float py) {
  PairEval E;
  E.dx = __fsub_rn(px, r0.x);
  E.dy = __fsub_rn(py, r0.y);
  E.u = __fmaf_rn(r0.z, E.dx, __fmul_rn(r0.w, E.dy));                       // Eq. 9: (u, v) = Q (x - c)
  E.v = __fmaf_rn(r1.x, E.dx, __fmul_rn(r1.y, E.dy));
  E.rho3 = __fmaf_rn(E.u, E.u, __fmul_rn(E.v, E.v));
  E.rho2 = __fmul_rn(2.0f, __fmaf_rn(E.dx, E.dx, __fmul_rn(E.dy, E.dy)));   // Eq. 12 low-pass term, sigma^2 = 1/2
  E.rho = fminf(E.rho3, E.rho2);
  E.aG = __fmul_rn(r1.z, fast_exp2(__fmul_rn(E.rho, kNegHalfLog2e)));      // alpha exp(-rho / 2)
  E.a = fminf(kAlphaMax, E.aG);
  return E;
}
// depth of the pair (Eq. 6 at the intersection; the centre depth where the low-pass term wins)
__device__ __forceinline__ float pair_depth(const PairEval& E, float zc, float g0, float g1) {
  return (E.rho3 <= E.rho2) ? __fadd_rn(zc, __fmaf_rn(g0, E.dx, __fmul_rn(g1, E.dy))) : zc;
}

}  // namespace satsplat

struct satsplat_ctx {
  int device;
  int sm_count;           // multiprocessors of `device` (grid sizing of the fixed-grid kernels)
  int64_t max_surfels, max_dup;
  int32_t max_w, max_h;
  int64_t scratch_bytes;
  // per-surfel
  float4* rec;            // [N*4]
  float4* bbox;           // [N] conservative screen-space box of each record (splat_bbox), for the blend kernels' culling
  uint16_t* rect;         // [N*4]
  uint32_t* count;        // [N]
  uint32_t* offset;       // [N+1] exclusive scan
  uint32_t* depth_key;    // [N]
  uint8_t* flags;         // [N]
  float* vrec;            // [N*kVrec] gradient moment records, kept zero between calls (the chain kernel clears them)
  uint32_t* block_sums;   // scan scratch
  // binning
  uint64_t* keys[2];
  uint32_t* vals[2];
  int sorted;             // which buffer holds the sorted result
  uint32_t* hist;         // [256 * kSortBlocks]
  uint32_t* ranges;       // [tiles*2]
  uint32_t* tile_count;   // [tiles] tile-sort binning: pair count per tile, then the scatter cursor
  uint32_t* tile_start;   // [tiles] exclusive scan of tile_count
  uint32_t* worklist;     // [3*tiles] tiles too long for the small-tile sort: 257-1024, 1025-4096, longer
  uint32_t* wl_count;     // [4] lengths of the three worklists
  int binning_mode;       // SATSPLAT_BINNING_TILESORT (default) or SATSPLAT_BINNING_RADIX
  int split_backward;     // SATSPLAT_OPT_SPLIT_BACKWARD: the backward calls stop after the blend; satsplat_backward_chain finishes
  int chain_pending;      // a blend backward has left moment records (and epilogue sums: chain_epi) for satsplat_backward_chain
  int chain_epi;
  cudaStream_t bin_stream;   // the long tile lists are sorted on this stream beside the short ones (forked from / joined to the caller's)
  cudaEvent_t bin_ev[2];
  satsplat::Status* status;
  // per-pixel state kept for the backward
  float4* px_a;           // (T_f, z_ref, M1', M2')
  float4* px_b;           // (albedo r,g,b, V)
  int2* px_i;             // (last, median list index)
  int32_t* px_last;       // planes for debug/statistics
  int32_t* px_visited;
  int32_t* px_contrib;
  int debug_planes;       // SATSPLAT_OPT_DEBUG_PLANES: the forward stores px_visited / px_contrib
  int planes_valid;       // ... and the last forward did
  float* red_buf;         // small reduction scratch (dF, cc, ambient, reproj)
  // host state
  satsplat::DevCamera cam;
  const float* cam_dev;   // device-resident camera record (16 floats of a camera block) of the last satsplat_preprocess_device, else NULL
  int64_t N;
  const float *in_means, *in_quats, *in_scales, *in_logits;  // caller buffers of the last preprocess (chain backward)
  int preprocessed, forwarded, depth_only;
  // e2e staging buffers (lazily sized inside create)
  // host-buffer iteration (satsplat_iteration_host*): two staging slots so that the copies of consecutive steps overlap
  float* e2e_in[2];       // means..rgb, sub-arrays at 16-byte aligned offsets
  float* e2e_up[2];       // upstream gradients (3 images)
  float* e2e_out[2];      // images
  float* e2e_grads[2];    // surfel gradient groups + dF cc ambient reproj dF_sun, loss sums (8) at + 48
  float* e2e_target[2];   // training step: target image
  float* e2e_loss[2];     // training step: scratch of the loss stage
  cudaStream_t e2e_stream[3];   // uploads / downloads / view-pass preprocess, beside the caller's stream
  cudaEvent_t e2e_ev[2][6];     // per slot: surfels up, upstream up, forward done, backward done, everything down, view preprocess done
  int e2e_busy[2];              // slot has a begin without its end
  cudaStream_t e2e_caller[2];   // the caller's stream of the step in flight on a slot (both slots must use the same one)
  int staging_ready;            // satsplat_reserve_host_staging allocated everything above (set last, after the last success)
  float* e2e_sun;               // sun-context role: sun map + its gradient
  // profiling
  int profiling;
  cudaEvent_t ev[2 * SATSPLAT_NUM_STAGES];
  int ev_used[SATSPLAT_NUM_STAGES];
  char err[512];
};

namespace satsplat {

extern std::atomic<long long> g_kernel_launches;  // cumulative kernel launches of this process (bench.py's gpu_launches)

// multiprocessors of the current device (for the kernels launched without a context)
inline int current_sm_count() {
  int dev = 0, n = 148;
  if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
  return n;
}

// launchers (each enqueues on `s`, returns the cudaError_t of the launch)
cudaError_t launch_preprocess(satsplat_ctx* c, int64_t N, const float* means, const float* quats, const float* scales,
                              const float* logits, const float* rgb, cudaStream_t s);
cudaError_t launch_scan(satsplat_ctx* c, int64_t N, cudaStream_t s);
cudaError_t launch_duplicate(satsplat_ctx* c, int64_t N, cudaStream_t s);
cudaError_t launch_sort(satsplat_ctx* c, cudaStream_t s);
cudaError_t launch_ranges(satsplat_ctx* c, cudaStream_t s);
cudaError_t launch_tile_scan(satsplat_ctx* c, cudaStream_t s);
cudaError_t launch_tile_scatter(satsplat_ctx* c, int64_t N, cudaStream_t s);
cudaError_t launch_tile_sort(satsplat_ctx* c, cudaStream_t s);
// sh_dev: 28-float shading record of a device camera block (NULL: the values of `sh`); the camera comes from c->cam_dev / c->cam
cudaError_t launch_blend_forward(satsplat_ctx* c, const DevShading& sh, const float* sh_dev, float* out_rgba, float* out_geom,
                                 float* out_aux, float* sun_depth_out, bool depth_only, cudaStream_t s);
cudaError_t launch_blend_backward(satsplat_ctx* c, const DevShading& sh, const float* sh_dev, const float* v_rgba, const float* v_geom,
                                  const float* v_aux, const float* v_sun_depth_in, bool depth_only, bool want_epilogue_sums,
                                  float* v_sun_depth, cudaStream_t s);
cudaError_t launch_chain_backward(satsplat_ctx* c, const float* means, const float* quats, const float* scales,
                                  const float* logits, float* v_means, float* v_quats, float* v_scales, float* v_logits,
                                  float* v_rgb, float* v_dF, const float* epi, float* v_cc, float* v_ambient, float* v_reproj,
                                  cudaStream_t s);
cudaError_t launch_add_small(float* dst, const float* src, int n, cudaStream_t s);
struct LossHost {   // arguments of the loss stage (losses.cu)
  int W, H;
  float w_l1, w_ssim, w_dist, w_normal;
  float c0[3], c1[3], c2[3], sgn, z_bg;
  const float *rgba, *geom, *aux, *target;
  float *scratch, *v_rgba, *v_geom, *v_aux, *sums;
};
cudaError_t launch_losses(const LossHost& L, cudaStream_t s);
int64_t init_scratch_bytes(int W, int H, int64_t N);
int64_t cdf_scan_partials(int64_t M);
cudaError_t launch_cdf_scan(double* w, long long M, double* partial, double** total_out, cudaStream_t s);
int64_t relocate_scratch_bytes(int64_t N);
cudaError_t launch_relocate(int64_t N, float* means, float* quats, float* scales, float* logits, float* rgb, float* adam_m,
                            float* adam_v, const float* u, float o_min, int n_max, void* scratch, int32_t* src_out, cudaStream_t s);
cudaError_t launch_init_from_dsm(const float* dsm, int W, int H, float cell, float ox, float oy, int64_t N, const float* u,
                                 const float* jx, const float* jy, void* scratch, float* means, float* quats, float* scales,
                                 int32_t* cells_out, cudaStream_t s);
cudaError_t launch_adam(int64_t N, float* const params[5], const float* const grads[5], float* m, float* v, const float lrs[5],
                        float beta1, float beta2, float eps, int step, cudaStream_t s);
cudaError_t launch_camera_adam(int n_views, const int32_t* view_index, satsplat_view_params* views, float* dF, float* v_dF_all,
                               const float* v_cc, const float* v_ambient, float* m, float* v, int32_t* steps, const float lr[3],
                               float beta1, float beta2, float eps, int clear_v_dF, cudaStream_t s);
cudaError_t launch_sun_camera_backward(float sc0, float sc1, float s0, float s1, const float* v_F_sun, const float* v_reproj,
                                       float* v_dF, cudaStream_t s);
cudaError_t launch_camera_chain(const satsplat_view_params* views, const float* dF_all, const int32_t* view_index, float* block,
                                cudaStream_t s);
cudaError_t launch_camera_chain_backward(const satsplat_view_params* views, const float* dF_all, const int32_t* view_index,
                                         const float* v_dF_view, const float* v_F_sun, const float* v_reproj, const float* v_F_nearby,
                                         float* v_dF_all, cudaStream_t s);
cudaError_t launch_advance_index(int32_t* view_index, int32_t stride, int32_t n_views, cudaStream_t s);
// per-device function attributes (dynamic shared-memory limits) of the kernels that need them; called by satsplat_create
cudaError_t init_blend_backward_attrs();
cudaError_t init_binning_attrs();
cudaError_t launch_export_records(satsplat_ctx* c, float* records_out, uint8_t* flags_out, cudaStream_t s);
void set_thread_error(const char* msg);   // api.cu: message of satsplat_last_error(NULL) on the calling thread

}  // namespace satsplat

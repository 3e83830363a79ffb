// api.cu — the C ABI of include/satsplat.h: context (scratch arena), argument checks, launch sequencing.
// No kernel lives here; every step of the path runs in the kernels of the other translation units.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "camera_math.cuh"
#include "internal.cuh"

using namespace satsplat;

namespace satsplat {
std::atomic<long long> g_kernel_launches{0};
}

namespace {

thread_local char g_err[512] = "";
}  // namespace

namespace satsplat {
// for entry points that live in other translation units: the message satsplat_last_error(NULL) returns on this thread
void set_thread_error(const char* msg) { snprintf(g_err, sizeof(g_err), "%s", msg); }
}  // namespace satsplat

namespace {

int fail(satsplat_ctx* c, int code, const char* fmt, const char* a = "") {
  char* dst = c ? c->err : g_err;
  snprintf(dst, 512, fmt, a);
  return code;
}

#define CU(call)                                                                       \
  do {                                                                                 \
    cudaError_t e_ = (call);                                                           \
    if (e_ != cudaSuccess) return fail(ctx, SATSPLAT_E_CUDA, #call ": %s", cudaGetErrorString(e_)); \
  } while (0)

template <typename T>
cudaError_t dalloc(satsplat_ctx* c, T** p, size_t n) {
  const size_t bytes = ((n * sizeof(T) + 255) / 256) * 256;
  cudaError_t e = cudaMalloc((void**)p, bytes ? bytes : 256);
  if (e == cudaSuccess) c->scratch_bytes += (int64_t)(bytes ? bytes : 256);
  return e;
}

void set_camera(satsplat_ctx* c, const satsplat_camera* cam) {
  DevCamera& d = c->cam;
  d.W = cam->width;
  d.H = cam->height;
  d.TX = (cam->width + kTile - 1) / kTile;
  d.TY = (cam->height + kTile - 1) / kTile;
  for (int i = 0; i < 8; ++i) d.Fp[i] = cam->F[i] + cam->dF[i];  // Eq. 15 (one fp32 rounding)
  for (int i = 0; i < 3; ++i) d.vd[i] = cam->view_dir[i];
  d.b_z = cam->b_z;
  d.z_bg = cam->z_bg;
  for (int i = 0; i < 3; ++i) d.bg[i] = cam->bg_rgb[i];
}

DevShading make_shading(const satsplat_shading* s) {
  DevShading d;
  memset(&d, 0, sizeof(d));
  if (!s) {
    d.cc[0] = d.cc[5] = d.cc[10] = 1.f;
    return d;
  }
  memcpy(d.cc, s->cc, sizeof(d.cc));
  memcpy(d.ambient, s->ambient, sizeof(d.ambient));
  d.shadows_on = s->shadows_on ? 1 : 0;
  d.sun_w = s->sun_width;
  d.sun_h = s->sun_height;
  d.sun_depth = s->sun_depth;
  memcpy(d.reproj, s->reproj, sizeof(d.reproj));
  d.bias = s->depth_bias;
  d.slope = s->slope;
  return d;
}

struct StageTimer {
  satsplat_ctx* c;
  cudaStream_t s;
  int stage;
  StageTimer(satsplat_ctx* c_, int stage_, cudaStream_t s_) : c(c_), s(s_), stage(stage_) {
    if (c->profiling) { cudaEventRecord(c->ev[2 * stage], s); }
  }
  ~StageTimer() {
    if (c->profiling) { cudaEventRecord(c->ev[2 * stage + 1], s); c->ev_used[stage] = 1; }
  }
};

void clear_stage_marks(satsplat_ctx* c, std::initializer_list<int> stages) {
  for (int s : stages) c->ev_used[s] = 0;
}

}  // namespace

extern "C" {

const char* satsplat_version(void) { return "satsplat-b200 0.1 (sm_100a)"; }

int64_t satsplat_kernel_launches(void) { return (int64_t)g_kernel_launches.load(); }

const char* satsplat_last_error(const satsplat_ctx* ctx) { return ctx ? ctx->err : g_err; }

int64_t satsplat_scratch_bytes(const satsplat_ctx* ctx) { return ctx ? ctx->scratch_bytes : 0; }

int satsplat_create(satsplat_ctx** out, int device, int64_t max_surfels, int32_t max_w, int32_t max_h,
                    int64_t max_dup) {
  if (!out) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_create: out is NULL");
  *out = nullptr;
  if (max_surfels < 0 || max_surfels >= (1ll << 31) || max_w <= 0 || max_h <= 0 || max_dup < 0 || max_dup >= (1ll << 32) - 1 ||
      max_w > 65535 * kTile || max_h > 65535 * kTile)
    return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_create: size out of range");
  satsplat_ctx* ctx = (satsplat_ctx*)calloc(1, sizeof(satsplat_ctx));
  if (!ctx) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_create: out of host memory");
  ctx->device = device;
  ctx->max_surfels = max_surfels;
  ctx->max_dup = max_dup;
  ctx->max_w = max_w;
  ctx->max_h = max_h;
  cudaError_t e = cudaSetDevice(device);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, device);
  if (e == cudaSuccess) e = init_blend_backward_attrs();
  if (e == cudaSuccess) e = init_binning_attrs();
  const size_t N = (size_t)max_surfels, K = (size_t)max_dup;
  const size_t tiles = (size_t)((max_w + kTile - 1) / kTile) * (size_t)((max_h + kTile - 1) / kTile);
  const size_t px = (size_t)max_w * (size_t)max_h;
#define A(call) if (e == cudaSuccess) e = (call)
  A(dalloc(ctx, &ctx->rec, N * 4));
  A(dalloc(ctx, &ctx->bbox, N));
  A(dalloc(ctx, &ctx->rect, N * 4));
  A(dalloc(ctx, &ctx->count, N));
  A(dalloc(ctx, &ctx->offset, N + 1));
  A(dalloc(ctx, &ctx->depth_key, N));
  A(dalloc(ctx, &ctx->flags, N));
  A(dalloc(ctx, &ctx->vrec, N * satsplat::kVrec));
  A(dalloc(ctx, &ctx->block_sums, (N / 4096 > tiles / 2048 ? N / 4096 : tiles / 2048) + 2));
  A(dalloc(ctx, &ctx->keys[0], K));
  A(dalloc(ctx, &ctx->keys[1], K));
  A(dalloc(ctx, &ctx->vals[0], K));
  A(dalloc(ctx, &ctx->vals[1], K));
  A(dalloc(ctx, &ctx->hist, (size_t)256 * kSortBlocks));
  A(dalloc(ctx, &ctx->ranges, tiles * 2));
  A(dalloc(ctx, &ctx->status, 1));
  A(dalloc(ctx, &ctx->tile_count, tiles * satsplat::kCtrStride));
  A(dalloc(ctx, &ctx->tile_start, tiles));
  A(dalloc(ctx, &ctx->worklist, tiles * 3));
  A(dalloc(ctx, &ctx->wl_count, 4));
  A(cudaMemset(ctx->tile_count, 0, tiles * satsplat::kCtrStride * sizeof(uint32_t)));
  A(dalloc(ctx, &ctx->px_a, px));
  A(dalloc(ctx, &ctx->px_b, px));
  A(dalloc(ctx, &ctx->px_i, px));
  A(dalloc(ctx, &ctx->px_visited, px));
  A(dalloc(ctx, &ctx->px_contrib, px));
  A(dalloc(ctx, &ctx->red_buf, satsplat::kRedCopies * 32));
  A(cudaMemset(ctx->vrec, 0, N ? N * satsplat::kVrec * sizeof(float) : 4));
  A(cudaMemset(ctx->status, 0, sizeof(Status)));
  for (int i = 0; i < 2 * SATSPLAT_NUM_STAGES; ++i) A(cudaEventCreate(&ctx->ev[i]));
  A(cudaStreamCreateWithFlags(&ctx->bin_stream, cudaStreamNonBlocking));
  for (int i = 0; i < 2; ++i) A(cudaEventCreateWithFlags(&ctx->bin_ev[i], cudaEventDisableTiming));
#undef A
  if (e != cudaSuccess) {
    fail(nullptr, SATSPLAT_E_CUDA, "satsplat_create: %s", cudaGetErrorString(e));
    satsplat_destroy(ctx);
    return SATSPLAT_E_CUDA;
  }
  strcpy(ctx->err, "ok");
  *out = ctx;
  return SATSPLAT_OK;
}

void satsplat_destroy(satsplat_ctx* ctx) {
  if (!ctx) return;
  cudaSetDevice(ctx->device);
  void* ptrs[] = {ctx->rec, ctx->bbox, ctx->rect, ctx->count, ctx->offset, ctx->depth_key, ctx->flags, ctx->vrec, ctx->block_sums,
                  ctx->keys[0], ctx->keys[1], ctx->vals[0], ctx->vals[1], ctx->hist, ctx->ranges, ctx->status, ctx->tile_count,
                  ctx->tile_start, ctx->worklist, ctx->wl_count, ctx->px_a,
                  ctx->px_b, ctx->px_i, ctx->px_visited, ctx->px_contrib, ctx->red_buf, ctx->e2e_in[0], ctx->e2e_in[1],
                  ctx->e2e_up[0], ctx->e2e_up[1], ctx->e2e_out[0], ctx->e2e_out[1], ctx->e2e_grads[0], ctx->e2e_grads[1],
                  ctx->e2e_target[0], ctx->e2e_target[1], ctx->e2e_loss[0], ctx->e2e_loss[1], ctx->e2e_sun};
  for (void* p : ptrs)
    if (p) cudaFree(p);
  for (int i = 0; i < 2 * SATSPLAT_NUM_STAGES; ++i)
    if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
  if (ctx->bin_stream) cudaStreamDestroy(ctx->bin_stream);
  for (int i = 0; i < 2; ++i)
    if (ctx->bin_ev[i]) cudaEventDestroy(ctx->bin_ev[i]);
  for (int i = 0; i < 3; ++i)
    if (ctx->e2e_stream[i]) cudaStreamDestroy(ctx->e2e_stream[i]);
  for (int i = 0; i < 12; ++i)
    if (ctx->e2e_ev[i / 6][i % 6]) cudaEventDestroy(ctx->e2e_ev[i / 6][i % 6]);
  free(ctx);
}

int satsplat_sun_camera(const satsplat_camera* view, float azimuth, float elevation, int32_t sun_w, int32_t sun_h,
                        const float viewport[4], satsplat_camera* sun_out, float reproj_out[8]) {
  if (!view || !viewport || !sun_out || !reproj_out || sun_w <= 0 || sun_h <= 0)
    return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_sun_camera: bad argument");
  const double te = tan((double)elevation);
  if (!(fabs(te) > 1e-12)) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_sun_camera: elevation must be non-zero");
  double Fp[8];
  for (int i = 0; i < 8; ++i) Fp[i] = (double)(float)(view->F[i] + view->dF[i]);  // the camera the rasteriser uses
  const double s0 = cos((double)azimuth) / te, s1 = sin((double)azimuth) / te;     // Eq. S2
  memset(sun_out, 0, sizeof(*sun_out));
  sun_out->width = sun_w;
  sun_out->height = sun_h;
  if (!sun_camera_math(Fp, s0, s1, viewport, sun_out->F, reproj_out))             // Eq. 16 + viewport; shared with the device chain
    return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_sun_camera: singular view camera");
  const double ce = cos((double)elevation);
  sun_out->view_dir[0] = (float)(-cos((double)azimuth) * ce);
  sun_out->view_dir[1] = (float)(-sin((double)azimuth) * ce);
  sun_out->view_dir[2] = (float)(-sin((double)elevation));
  sun_out->b_z = view->b_z;
  sun_out->z_bg = view->z_bg;
  return SATSPLAT_OK;
}

int satsplat_sun_camera_backward(const satsplat_camera* view, float azimuth, float elevation, const float viewport[4],
                                 const float* v_F_sun, const float* v_reproj, float* v_dF, satsplat_stream stream) {
  if (!view || !viewport || !v_dF) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_sun_camera_backward: NULL argument");
  const double te = tan((double)elevation);
  if (!(fabs(te) > 1e-12)) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_sun_camera_backward: elevation must be non-zero");
  const float s0 = (float)(cos((double)azimuth) / te), s1 = (float)(sin((double)azimuth) / te);   // Eq. S2
  cudaError_t e = launch_sun_camera_backward(viewport[0], viewport[1], s0, s1, v_F_sun, v_reproj, v_dF, (cudaStream_t)stream);
  if (e != cudaSuccess) return fail(nullptr, SATSPLAT_E_CUDA, "satsplat_sun_camera_backward: %s", cudaGetErrorString(e));
  return SATSPLAT_OK;
}

int64_t satsplat_loss_scratch_floats(int32_t width, int32_t height) { return (int64_t)13 * width * height; }

int satsplat_loss_upstream(const satsplat_camera* cam, const satsplat_loss_weights* w, const float* out_rgba,
                           const float* out_geom, const float* out_aux, const float* target_rgba, float* scratch,
                           float* v_rgba, float* v_geom, float* v_aux, float* loss_sums, satsplat_stream stream) {
  if (!cam || !w || !out_rgba || !out_geom || !out_aux || !target_rgba || !scratch || !v_rgba || !v_geom || !v_aux || !loss_sums)
    return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_loss_upstream: NULL argument");
  if (cam->width <= 0 || cam->height <= 0) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_loss_upstream: bad image size");
  // Eq. 13 constants: p_s = (B2^-1 (x - b - B3 h), h), h = b_z - z_v, is affine in z_v, so with the central differences
  // dx, dy of z_v:  grad_x p x grad_y p = c0 + dx c1 + dy c2
  double Fp[8];
  for (int i = 0; i < 8; ++i) Fp[i] = (double)(float)(cam->F[i] + cam->dF[i]);
  const double det = Fp[0] * Fp[5] - Fp[1] * Fp[4];
  if (!(fabs(det) > 0)) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_loss_upstream: singular camera");
  const double Bi[2][2] = {{Fp[5] / det, -Fp[1] / det}, {-Fp[4] / det, Fp[0] / det}};
  const double k[3] = {Bi[0][0] * Fp[2] + Bi[0][1] * Fp[6], Bi[1][0] * Fp[2] + Bi[1][1] * Fp[6], -1.0};
  const double ax[3] = {2.0 * Bi[0][0], 2.0 * Bi[1][0], 0.0}, ay[3] = {2.0 * Bi[0][1], 2.0 * Bi[1][1], 0.0};
  auto cross = [](const double* a, const double* b, double* c) {
    c[0] = a[1] * b[2] - a[2] * b[1]; c[1] = a[2] * b[0] - a[0] * b[2]; c[2] = a[0] * b[1] - a[1] * b[0];
  };
  double c0[3], c1[3], c2[3];
  cross(ax, ay, c0); cross(k, ay, c1); cross(ax, k, c2);
  LossHost L;
  L.W = cam->width; L.H = cam->height;
  L.w_l1 = w->w_l1; L.w_ssim = w->w_ssim; L.w_dist = w->w_dist; L.w_normal = w->w_normal;
  for (int i = 0; i < 3; ++i) { L.c0[i] = (float)c0[i]; L.c1[i] = (float)c1[i]; L.c2[i] = (float)c2[i]; }
  L.sgn = (c0[0] * cam->view_dir[0] + c0[1] * cam->view_dir[1] + c0[2] * cam->view_dir[2]) > 0 ? -1.f : 1.f;
  L.z_bg = cam->z_bg;
  L.rgba = out_rgba; L.geom = out_geom; L.aux = out_aux; L.target = target_rgba;
  L.scratch = scratch; L.v_rgba = v_rgba; L.v_geom = v_geom; L.v_aux = v_aux; L.sums = loss_sums;
  cudaError_t e = launch_losses(L, (cudaStream_t)stream);
  if (e != cudaSuccess) return fail(nullptr, SATSPLAT_E_CUDA, "satsplat_loss_upstream: %s", cudaGetErrorString(e));
  return SATSPLAT_OK;
}

int64_t satsplat_init_scratch_bytes(int32_t dsm_w, int32_t dsm_h, int64_t N) {
  if (dsm_w <= 0 || dsm_h <= 0 || N < 0) return 0;
  return init_scratch_bytes(dsm_w, dsm_h, N);
}

int satsplat_init_from_dsm(const float* dsm, int32_t dsm_w, int32_t dsm_h, float cell, float origin_x, float origin_y, int64_t N,
                           const float* u, const float* jx, const float* jy, void* scratch, float* means, float* quats,
                           float* scales, int32_t* cells_out, satsplat_stream stream) {
  if (!dsm || dsm_w <= 0 || dsm_h <= 0 || !(cell > 0.f) || N < 0) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_init_from_dsm: bad argument");
  if (N > 0 && (!u || !jx || !jy || !scratch || !means || !quats || !scales))
    return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_init_from_dsm: NULL pointer");
  cudaError_t e = launch_init_from_dsm(dsm, dsm_w, dsm_h, cell, origin_x, origin_y, N, u, jx, jy, scratch, means, quats, scales,
                                       cells_out, (cudaStream_t)stream);
  if (e != cudaSuccess) return fail(nullptr, SATSPLAT_E_CUDA, "satsplat_init_from_dsm: %s", cudaGetErrorString(e));
  return SATSPLAT_OK;
}

int64_t satsplat_relocate_scratch_bytes(int64_t N) { return N < 0 ? 0 : relocate_scratch_bytes(N); }

int satsplat_relocate(int64_t N, float* means, float* quats, float* scales, float* opacity_logits, float* rgb, float* adam_m,
                      float* adam_v, const float* u, float o_min, int32_t n_max, void* scratch, int32_t* src_out,
                      satsplat_stream stream) {
  if (N < 0 || !(o_min > 0.f && o_min < 1.f) || n_max < 1 || (adam_m == nullptr) != (adam_v == nullptr))
    return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_relocate: bad argument");
  if (N > 0 && (!means || !quats || !scales || !opacity_logits || !rgb || !u || !scratch))
    return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_relocate: NULL pointer");
  cudaError_t e = launch_relocate(N, means, quats, scales, opacity_logits, rgb, adam_m, adam_v, u, o_min, n_max, scratch, src_out,
                                  (cudaStream_t)stream);
  if (e != cudaSuccess) return fail(nullptr, SATSPLAT_E_CUDA, "satsplat_relocate: %s", cudaGetErrorString(e));
  return SATSPLAT_OK;
}

int64_t satsplat_adam_state_floats(int64_t N) {
  static const int width[5] = {3, 4, 2, 1, 3};
  int64_t t = 0;
  for (int k = 0; k < 5; ++k) t += (N * width[k] + 3) & ~(int64_t)3;
  return t;
}

int satsplat_adam_step(int64_t N, float* means, float* quats, float* scales, float* opacity_logits, float* rgb,
                       const float* v_means, const float* v_quats, const float* v_scales, const float* v_opacity_logits,
                       const float* v_rgb, float* adam_m, float* adam_v, const satsplat_adam* hp, satsplat_stream stream) {
  if (N < 0 || !hp) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_adam_step: bad argument");
  if (N > 0 && (!means || !quats || !scales || !opacity_logits || !rgb || !v_means || !v_quats || !v_scales ||
                !v_opacity_logits || !v_rgb || !adam_m || !adam_v))
    return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_adam_step: NULL pointer");
  if (hp->step < 1 || !(hp->beta1 >= 0.f && hp->beta1 < 1.f) || !(hp->beta2 >= 0.f && hp->beta2 < 1.f))
    return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_adam_step: step must be >= 1 and the betas in [0, 1)");
  float* const params[5] = {means, quats, scales, opacity_logits, rgb};
  const float* const grads[5] = {v_means, v_quats, v_scales, v_opacity_logits, v_rgb};
  cudaError_t e = launch_adam(N, params, grads, adam_m, adam_v, hp->lr, hp->beta1, hp->beta2, hp->eps, hp->step, (cudaStream_t)stream);
  if (e != cudaSuccess) return fail(nullptr, SATSPLAT_E_CUDA, "satsplat_adam_step: %s", cudaGetErrorString(e));
  return SATSPLAT_OK;
}

int satsplat_adam_step_cameras(int32_t n_views, const int32_t* view_index, satsplat_view_params* views, float* dF, float* v_dF_all,
                               const float* v_cc, const float* v_ambient, float* adam_m, float* adam_v, int32_t* steps,
                               const satsplat_camera_adam* hp, int32_t clear_v_dF, satsplat_stream stream) {
  if (n_views <= 0 || !views || !adam_m || !adam_v || !steps || !hp)
    return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_adam_step_cameras: bad argument");
  if ((dF == nullptr) != (v_dF_all == nullptr))
    return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_adam_step_cameras: dF and v_dF_all must both be given or both be NULL");
  if (!(hp->beta1 >= 0.f && hp->beta1 < 1.f) || !(hp->beta2 >= 0.f && hp->beta2 < 1.f))
    return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_adam_step_cameras: the betas must be in [0, 1)");
  cudaError_t e = launch_camera_adam(n_views, view_index, views, dF, v_dF_all, v_cc, v_ambient, adam_m, adam_v, steps, hp->lr, hp->beta1,
                                     hp->beta2, hp->eps, clear_v_dF ? 1 : 0, (cudaStream_t)stream);
  if (e != cudaSuccess) return fail(nullptr, SATSPLAT_E_CUDA, "satsplat_adam_step_cameras: %s", cudaGetErrorString(e));
  return SATSPLAT_OK;
}

namespace {
// The blend half of a split backward accumulates per-surfel moment records with REDs and only the chain clears them: a
// second blend backward, a new preprocess or an option change in between would leave stale moments for the next chain.
const char* const kChainPendingMsg = "%s: a split backward is pending on this context; call satsplat_backward_chain first";
// (a1) + (a2) on the context's current camera (host copy in ctx->cam, or the device record ctx->cam_dev)
int preprocess_common(satsplat_ctx* ctx, int64_t N, const float* means, const float* quats, const float* scales,
                      const float* opacity_logits, const float* rgb, cudaStream_t s) {
  if (ctx->chain_pending) return fail(ctx, SATSPLAT_E_STATE, kChainPendingMsg, "satsplat_preprocess");
  ctx->N = N;
  ctx->in_means = means; ctx->in_quats = quats; ctx->in_scales = scales; ctx->in_logits = opacity_logits;
  ctx->preprocessed = 0;
  ctx->forwarded = 0;
  clear_stage_marks(ctx, {0, 1, 2, 3, 4, 5, 6, 7});
  if (ctx->binning_mode == SATSPLAT_BINNING_TILESORT) {
    // tile_count is all zero here: create() clears it, tile_scan turns it into the scatter cursor and the tile
    // sort clears it again, all on this stream
    { StageTimer t(ctx, SATSPLAT_STAGE_PREPROCESS, s); CU(launch_preprocess(ctx, N, means, quats, scales, opacity_logits, rgb, s)); }
    { StageTimer t(ctx, SATSPLAT_STAGE_SCAN, s); CU(launch_tile_scan(ctx, s)); }
    { StageTimer t(ctx, SATSPLAT_STAGE_DUPLICATE, s); CU(launch_tile_scatter(ctx, N, s)); }
    { StageTimer t(ctx, SATSPLAT_STAGE_SORT, s); CU(launch_tile_sort(ctx, s)); }
  } else {
    { StageTimer t(ctx, SATSPLAT_STAGE_PREPROCESS, s); CU(launch_preprocess(ctx, N, means, quats, scales, opacity_logits, rgb, s)); }
    { StageTimer t(ctx, SATSPLAT_STAGE_SCAN, s); CU(launch_scan(ctx, N, s)); }
    { StageTimer t(ctx, SATSPLAT_STAGE_DUPLICATE, s); CU(launch_duplicate(ctx, N, s)); }
    { StageTimer t(ctx, SATSPLAT_STAGE_SORT, s); CU(launch_sort(ctx, s)); }
    { StageTimer t(ctx, SATSPLAT_STAGE_RANGES, s); CU(launch_ranges(ctx, s)); }
  }
  ctx->preprocessed = 1;
  return SATSPLAT_OK;
}
}  // namespace

int satsplat_preprocess(satsplat_ctx* ctx, const satsplat_camera* cam, int64_t N, const float* means,
                        const float* quats, const float* scales, const float* opacity_logits, const float* rgb,
                        satsplat_stream stream) {
  if (!ctx) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_preprocess: ctx is NULL");
  if (!cam || N < 0 || (N > 0 && (!means || !quats || !scales || !opacity_logits || !rgb)))
    return fail(ctx, SATSPLAT_E_INVALID, "satsplat_preprocess: NULL argument");
  if (N > ctx->max_surfels) return fail(ctx, SATSPLAT_E_INVALID, "satsplat_preprocess: N exceeds max_surfels");
  if (cam->width <= 0 || cam->height <= 0 || cam->width > ctx->max_w || cam->height > ctx->max_h)
    return fail(ctx, SATSPLAT_E_INVALID, "satsplat_preprocess: image size exceeds the context");
  CU(cudaSetDevice(ctx->device));
  set_camera(ctx, cam);
  ctx->cam_dev = nullptr;
  return preprocess_common(ctx, N, means, quats, scales, opacity_logits, rgb, (cudaStream_t)stream);
}

int satsplat_preprocess_device(satsplat_ctx* ctx, int32_t width, int32_t height, const float* block, int32_t which, int64_t N,
                               const float* means, const float* quats, const float* scales, const float* opacity_logits,
                               const float* rgb, satsplat_stream stream) {
  if (!ctx) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_preprocess_device: ctx is NULL");
  if (!block || which < 0 || which > 2 || N < 0 || (N > 0 && (!means || !quats || !scales || !opacity_logits || !rgb)))
    return fail(ctx, SATSPLAT_E_INVALID, "satsplat_preprocess_device: bad argument");
  if (N > ctx->max_surfels) return fail(ctx, SATSPLAT_E_INVALID, "satsplat_preprocess_device: N exceeds max_surfels");
  if (width <= 0 || height <= 0 || width > ctx->max_w || height > ctx->max_h)
    return fail(ctx, SATSPLAT_E_INVALID, "satsplat_preprocess_device: image size exceeds the context");
  CU(cudaSetDevice(ctx->device));
  memset(&ctx->cam, 0, sizeof(ctx->cam));           // the float fields live on the device; only the sizes are host values
  ctx->cam.W = width;
  ctx->cam.H = height;
  ctx->cam.TX = (width + kTile - 1) / kTile;
  ctx->cam.TY = (height + kTile - 1) / kTile;
  ctx->cam_dev = block + kCamFloats * which;
  return preprocess_common(ctx, N, means, quats, scales, opacity_logits, rgb, (cudaStream_t)stream);
}

namespace {
int forward_common(satsplat_ctx* ctx, const DevShading& sh, const float* sh_dev, float* out_rgba, float* out_geom, float* out_aux,
                   cudaStream_t s) {
  clear_stage_marks(ctx, {5, 6, 7});
  { StageTimer t(ctx, SATSPLAT_STAGE_BLEND_FWD, s); CU(launch_blend_forward(ctx, sh, sh_dev, out_rgba, out_geom, out_aux, nullptr, false, s)); }
  ctx->forwarded = 1;
  ctx->depth_only = 0;
  return SATSPLAT_OK;
}

int backward_common(satsplat_ctx* ctx, const DevShading& sh, const float* sh_dev, const float* v_rgba, const float* v_geom,
                    const float* v_aux, float* v_means, float* v_quats, float* v_scales, float* v_opacity_logits, float* v_rgb,
                    float* v_dF, float* v_cc, float* v_ambient, float* v_sun_depth, float* v_reproj, cudaStream_t s) {
  if (ctx->chain_pending) return fail(ctx, SATSPLAT_E_STATE, kChainPendingMsg, "satsplat_render_backward");
  clear_stage_marks(ctx, {6, 7});
  // the 23 epilogue sums (cc, ambient, reproj) are left in red_buf by the blend; the chain kernel's first CTA delivers them
  const bool epi = ctx->split_backward || v_cc || v_ambient || v_reproj;
  {
    StageTimer t(ctx, SATSPLAT_STAGE_BLEND_BWD, s);
    CU(launch_blend_backward(ctx, sh, sh_dev, v_rgba, v_geom, v_aux, nullptr, false, epi, v_sun_depth, s));
  }
  if (ctx->split_backward) {   // SATSPLAT_OPT_SPLIT_BACKWARD: satsplat_backward_chain finishes the call
    ctx->chain_pending = 1;
    ctx->chain_epi = 1;
    return SATSPLAT_OK;
  }
  {
    StageTimer t(ctx, SATSPLAT_STAGE_CHAIN_BWD, s);
    CU(launch_chain_backward(ctx, ctx->in_means, ctx->in_quats, ctx->in_scales, ctx->in_logits, v_means, v_quats, v_scales,
                             v_opacity_logits, v_rgb, v_dF, epi ? ctx->red_buf : nullptr, v_cc, v_ambient, v_reproj, s));
  }
  return SATSPLAT_OK;
}

// shading of the *_device calls: the float constants come from the block, the sun map and its size from the caller
DevShading device_shading(const float* sun_depth, int32_t sun_w, int32_t sun_h) {
  DevShading d;
  memset(&d, 0, sizeof(d));
  d.shadows_on = sun_depth ? 1 : 0;
  d.sun_depth = sun_depth;
  d.sun_w = sun_w;
  d.sun_h = sun_h;
  return d;
}
}  // namespace

int satsplat_render_forward(satsplat_ctx* ctx, const satsplat_shading* shading, float* out_rgba, float* out_geom,
                            float* out_aux, satsplat_stream stream) {
  if (!ctx) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_render_forward: ctx is NULL");
  if (!ctx->preprocessed) return fail(ctx, SATSPLAT_E_STATE, "satsplat_render_forward: call satsplat_preprocess first");
  if (ctx->cam_dev) return fail(ctx, SATSPLAT_E_STATE, "satsplat_render_forward: device camera in use, call satsplat_render_forward_device");
  if (shading && shading->shadows_on && (!shading->sun_depth || shading->sun_width <= 0 || shading->sun_height <= 0))
    return fail(ctx, SATSPLAT_E_INVALID, "satsplat_render_forward: shadows_on without a sun depth map");
  CU(cudaSetDevice(ctx->device));
  return forward_common(ctx, make_shading(shading), nullptr, out_rgba, out_geom, out_aux, (cudaStream_t)stream);
}

int satsplat_render_forward_device(satsplat_ctx* ctx, const float* block, const float* sun_depth, int32_t sun_width,
                                   int32_t sun_height, float* out_rgba, float* out_geom, float* out_aux, satsplat_stream stream) {
  if (!ctx) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_render_forward_device: ctx is NULL");
  if (!ctx->preprocessed || !ctx->cam_dev)
    return fail(ctx, SATSPLAT_E_STATE, "satsplat_render_forward_device: call satsplat_preprocess_device first");
  if (!block || (sun_depth && (sun_width <= 0 || sun_height <= 0)))
    return fail(ctx, SATSPLAT_E_INVALID, "satsplat_render_forward_device: bad argument");
  CU(cudaSetDevice(ctx->device));
  return forward_common(ctx, device_shading(sun_depth, sun_width, sun_height), block + kBlockShading, out_rgba, out_geom, out_aux,
                        (cudaStream_t)stream);
}

int satsplat_shadow_map(satsplat_ctx* ctx, float* sun_depth_out, satsplat_stream stream) {
  if (!ctx) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_shadow_map: ctx is NULL");
  if (!sun_depth_out) return fail(ctx, SATSPLAT_E_INVALID, "satsplat_shadow_map: output is NULL");
  if (!ctx->preprocessed) return fail(ctx, SATSPLAT_E_STATE, "satsplat_shadow_map: call satsplat_preprocess first");
  cudaStream_t s = (cudaStream_t)stream;
  CU(cudaSetDevice(ctx->device));
  const DevShading sh = make_shading(nullptr);
  clear_stage_marks(ctx, {5, 6, 7});
  { StageTimer t(ctx, SATSPLAT_STAGE_BLEND_FWD, s); CU(launch_blend_forward(ctx, sh, nullptr, nullptr, nullptr, nullptr, sun_depth_out, true, s)); }
  ctx->forwarded = 1;
  ctx->depth_only = 1;
  return SATSPLAT_OK;
}

int satsplat_render_backward(satsplat_ctx* ctx, const satsplat_shading* shading, const float* v_rgba,
                             const float* v_geom, const float* v_aux, float* v_means, float* v_quats,
                             float* v_scales, float* v_opacity_logits, float* v_rgb, float* v_dF, float* v_cc,
                             float* v_ambient, float* v_sun_depth, float* v_reproj, satsplat_stream stream) {
  if (!ctx) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_render_backward: ctx is NULL");
  if (!ctx->forwarded || ctx->depth_only)
    return fail(ctx, SATSPLAT_E_STATE, "satsplat_render_backward: call satsplat_render_forward first");
  if (ctx->cam_dev) return fail(ctx, SATSPLAT_E_STATE, "satsplat_render_backward: device camera in use, call satsplat_render_backward_device");
  if (shading && shading->shadows_on && (!shading->sun_depth || shading->sun_width <= 0 || shading->sun_height <= 0))
    return fail(ctx, SATSPLAT_E_INVALID, "satsplat_render_backward: shadows_on without a sun depth map");
  CU(cudaSetDevice(ctx->device));
  return backward_common(ctx, make_shading(shading), nullptr, v_rgba, v_geom, v_aux, v_means, v_quats, v_scales, v_opacity_logits,
                         v_rgb, v_dF, v_cc, v_ambient, v_sun_depth, v_reproj, (cudaStream_t)stream);
}

int satsplat_render_backward_device(satsplat_ctx* ctx, const float* block, const float* sun_depth, int32_t sun_width,
                                    int32_t sun_height, const float* v_rgba, const float* v_geom, const float* v_aux,
                                    float* v_means, float* v_quats, float* v_scales, float* v_opacity_logits, float* v_rgb,
                                    float* v_dF, float* v_cc, float* v_ambient, float* v_sun_depth, float* v_reproj,
                                    satsplat_stream stream) {
  if (!ctx) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_render_backward_device: ctx is NULL");
  if (!ctx->forwarded || ctx->depth_only || !ctx->cam_dev)
    return fail(ctx, SATSPLAT_E_STATE, "satsplat_render_backward_device: call satsplat_render_forward_device first");
  if (!block || (sun_depth && (sun_width <= 0 || sun_height <= 0)))
    return fail(ctx, SATSPLAT_E_INVALID, "satsplat_render_backward_device: bad argument");
  CU(cudaSetDevice(ctx->device));
  return backward_common(ctx, device_shading(sun_depth, sun_width, sun_height), block + kBlockShading, v_rgba, v_geom, v_aux, v_means,
                         v_quats, v_scales, v_opacity_logits, v_rgb, v_dF, v_cc, v_ambient, v_sun_depth, v_reproj, (cudaStream_t)stream);
}

int satsplat_shadow_map_backward(satsplat_ctx* ctx, const float* v_sun_depth, float* v_means, float* v_quats,
                                 float* v_scales, float* v_opacity_logits, float* v_dF_sun, satsplat_stream stream) {
  if (!ctx) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_shadow_map_backward: ctx is NULL");
  if (!v_sun_depth) return fail(ctx, SATSPLAT_E_INVALID, "satsplat_shadow_map_backward: v_sun_depth is NULL");
  if (!ctx->forwarded || !ctx->depth_only)
    return fail(ctx, SATSPLAT_E_STATE, "satsplat_shadow_map_backward: call satsplat_shadow_map first");
  if (ctx->chain_pending) return fail(ctx, SATSPLAT_E_STATE, kChainPendingMsg, "satsplat_shadow_map_backward");
  cudaStream_t s = (cudaStream_t)stream;
  CU(cudaSetDevice(ctx->device));
  const DevShading sh = make_shading(nullptr);
  clear_stage_marks(ctx, {6, 7});
  {
    StageTimer t(ctx, SATSPLAT_STAGE_BLEND_BWD, s);
    CU(launch_blend_backward(ctx, sh, nullptr, nullptr, nullptr, nullptr, v_sun_depth, true, false, nullptr, s));
  }
  if (ctx->split_backward) {
    ctx->chain_pending = 1;
    ctx->chain_epi = 0;
    return SATSPLAT_OK;
  }
  {
    StageTimer t(ctx, SATSPLAT_STAGE_CHAIN_BWD, s);
    CU(launch_chain_backward(ctx, ctx->in_means, ctx->in_quats, ctx->in_scales, ctx->in_logits, v_means, v_quats, v_scales,
                             v_opacity_logits, nullptr, v_dF_sun, nullptr, nullptr, nullptr, nullptr, s));
  }
  return SATSPLAT_OK;
}

int satsplat_backward_chain(satsplat_ctx* ctx, float* v_means, float* v_quats, float* v_scales, float* v_opacity_logits, float* v_rgb,
                            float* v_dF, float* v_cc, float* v_ambient, float* v_reproj, satsplat_stream stream) {
  if (!ctx) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_backward_chain: ctx is NULL");
  if (!ctx->chain_pending) return fail(ctx, SATSPLAT_E_STATE, "satsplat_backward_chain: no split backward call is pending on this context");
  cudaStream_t s = (cudaStream_t)stream;
  CU(cudaSetDevice(ctx->device));
  ctx->chain_pending = 0;
  {
    StageTimer t(ctx, SATSPLAT_STAGE_CHAIN_BWD, s);
    CU(launch_chain_backward(ctx, ctx->in_means, ctx->in_quats, ctx->in_scales, ctx->in_logits, v_means, v_quats, v_scales,
                             v_opacity_logits, ctx->depth_only ? nullptr : v_rgb, v_dF, ctx->chain_epi ? ctx->red_buf : nullptr, v_cc,
                             v_ambient, v_reproj, s));
  }
  return SATSPLAT_OK;
}

int satsplat_view_params_fill(const satsplat_camera* cam, const satsplat_shading* shading, const satsplat_sun* sun,
                              float nearby_d_azimuth, float nearby_d_elevation, satsplat_view_params* out) {
  if (!cam || !out) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_view_params_fill: NULL argument");
  memset(out, 0, sizeof(*out));
  memcpy(out->F, cam->F, sizeof(out->F));
  memcpy(out->view_dir, cam->view_dir, sizeof(out->view_dir));
  out->b_z = cam->b_z;
  out->z_bg = cam->z_bg;
  memcpy(out->bg_rgb, cam->bg_rgb, sizeof(out->bg_rgb));
  out->cc[0] = out->cc[5] = out->cc[10] = 1.f;
  out->depth_bias = 0.5f;
  out->slope = 4.f;
  if (shading) {
    memcpy(out->cc, shading->cc, sizeof(out->cc));
    memcpy(out->ambient, shading->ambient, sizeof(out->ambient));
    out->depth_bias = shading->depth_bias;
    out->slope = shading->slope;
  }
  out->nearby_d_azimuth = nearby_d_azimuth;
  out->nearby_d_elevation = nearby_d_elevation;
  out->sun_viewport[0] = out->sun_viewport[1] = 1.f;
  out->sun_s[0] = out->sun_s[1] = 0.0;
  out->sun_view_dir[2] = -1.f;
  if (sun) {
    const double te = tan((double)sun->elevation);
    if (!(fabs(te) > 1e-12)) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_view_params_fill: elevation must be non-zero");
    out->sun_s[0] = cos((double)sun->azimuth) / te;   // Eq. S2, exactly as satsplat_sun_camera
    out->sun_s[1] = sin((double)sun->azimuth) / te;
    memcpy(out->sun_viewport, sun->viewport, sizeof(out->sun_viewport));
    const double ce = cos((double)sun->elevation);
    out->sun_view_dir[0] = (float)(-cos((double)sun->azimuth) * ce);
    out->sun_view_dir[1] = (float)(-sin((double)sun->azimuth) * ce);
    out->sun_view_dir[2] = (float)(-sin((double)sun->elevation));
  }
  return SATSPLAT_OK;
}

int satsplat_camera_chain(const satsplat_view_params* views, const float* dF, const int32_t* view_index, float* block,
                          satsplat_stream stream) {
  if (!views || !block) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_camera_chain: NULL argument");
  const cudaError_t e = launch_camera_chain(views, dF, view_index, block, (cudaStream_t)stream);
  if (e != cudaSuccess) return fail(nullptr, SATSPLAT_E_CUDA, "satsplat_camera_chain: %s", cudaGetErrorString(e));
  return SATSPLAT_OK;
}

int satsplat_camera_chain_backward(const satsplat_view_params* views, const float* dF, const int32_t* view_index,
                                   const float* v_dF_view, const float* v_F_sun, const float* v_reproj, const float* v_F_nearby,
                                   float* v_dF_all, satsplat_stream stream) {
  if (!views || !v_dF_all) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_camera_chain_backward: NULL argument");
  const cudaError_t e = launch_camera_chain_backward(views, dF, view_index, v_dF_view, v_F_sun, v_reproj, v_F_nearby, v_dF_all,
                                                     (cudaStream_t)stream);
  if (e != cudaSuccess) return fail(nullptr, SATSPLAT_E_CUDA, "satsplat_camera_chain_backward: %s", cudaGetErrorString(e));
  return SATSPLAT_OK;
}

int satsplat_advance_view_index(int32_t* view_index, int32_t stride, int32_t n_views, satsplat_stream stream) {
  if (!view_index || n_views <= 0) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_advance_view_index: bad argument");
  const cudaError_t e = launch_advance_index(view_index, stride, n_views, (cudaStream_t)stream);
  if (e != cudaSuccess) return fail(nullptr, SATSPLAT_E_CUDA, "satsplat_advance_view_index: %s", cudaGetErrorString(e));
  return SATSPLAT_OK;
}

int satsplat_sync_status(satsplat_ctx* ctx, int64_t* K, satsplat_stream stream) {
  if (!ctx) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_sync_status: ctx is NULL");
  CU(cudaSetDevice(ctx->device));
  Status st;
  CU(cudaMemcpyAsync(&st, ctx->status, sizeof(Status), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
  CU(cudaStreamSynchronize((cudaStream_t)stream));
  if (K) *K = (int64_t)st.K;
  if (st.overflow) return fail(ctx, SATSPLAT_E_CAPACITY, "duplicated keys exceed max_duplicates");
  return SATSPLAT_OK;
}

int satsplat_debug_bins(satsplat_ctx* ctx, int64_t* K, const uint64_t** keys, const uint32_t** vals,
                        const uint32_t** tile_ranges, const uint16_t** rects, const uint32_t** counts,
                        satsplat_stream stream) {
  if (!ctx) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_debug_bins: ctx is NULL");
  if (!ctx->preprocessed) return fail(ctx, SATSPLAT_E_STATE, "satsplat_debug_bins: call satsplat_preprocess first");
  int64_t k = 0;
  const int rc = satsplat_sync_status(ctx, &k, stream);
  if (K) *K = k;
  if (keys) *keys = ctx->keys[ctx->sorted];
  if (vals) *vals = ctx->vals[ctx->sorted];
  if (tile_ranges) *tile_ranges = ctx->ranges;
  if (rects) *rects = ctx->rect;
  if (counts) *counts = ctx->count;
  return rc;
}

int satsplat_debug_records(satsplat_ctx* ctx, float* records_out, uint8_t* flags_out, satsplat_stream stream) {
  if (!ctx) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_debug_records: ctx is NULL");
  if (!records_out) return fail(ctx, SATSPLAT_E_INVALID, "satsplat_debug_records: records_out is NULL");
  if (!ctx->preprocessed) return fail(ctx, SATSPLAT_E_STATE, "satsplat_debug_records: call satsplat_preprocess first");
  CU(cudaSetDevice(ctx->device));
  CU(launch_export_records(ctx, records_out, flags_out, (cudaStream_t)stream));
  return SATSPLAT_OK;
}

int satsplat_debug_planes(satsplat_ctx* ctx, const int32_t** n_visited, const int32_t** n_contrib) {
  if (!ctx) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_debug_planes: ctx is NULL");
  if (!ctx->forwarded) return fail(ctx, SATSPLAT_E_STATE, "satsplat_debug_planes: no forward pass yet");
  if (!ctx->planes_valid)
    return fail(ctx, SATSPLAT_E_STATE, "satsplat_debug_planes: the last forward ran without SATSPLAT_OPT_DEBUG_PLANES = 1");
  if (n_visited) *n_visited = ctx->px_visited;
  if (n_contrib) *n_contrib = ctx->px_contrib;
  return SATSPLAT_OK;
}

int satsplat_set_option(satsplat_ctx* ctx, int32_t option, int32_t value) {
  if (!ctx) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_set_option: ctx is NULL");
  if (option == SATSPLAT_OPT_SPLIT_BACKWARD && (value == 0 || value == 1)) {
    if (ctx->chain_pending) return fail(ctx, SATSPLAT_E_STATE, kChainPendingMsg, "satsplat_set_option");
    ctx->split_backward = value;
    return SATSPLAT_OK;
  }
  if (option == SATSPLAT_OPT_DEBUG_PLANES && (value == 0 || value == 1)) {
    ctx->debug_planes = value;
    return SATSPLAT_OK;
  }
  if (option == SATSPLAT_OPT_BINNING && (value == SATSPLAT_BINNING_TILESORT || value == SATSPLAT_BINNING_RADIX)) {
    ctx->binning_mode = value;
    ctx->preprocessed = 0;
    ctx->forwarded = 0;
    return SATSPLAT_OK;
  }
  return fail(ctx, SATSPLAT_E_INVALID, "satsplat_set_option: unknown option or value");
}

int satsplat_set_profiling(satsplat_ctx* ctx, int32_t enabled) {
  if (!ctx) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_set_profiling: ctx is NULL");
  ctx->profiling = enabled ? 1 : 0;
  for (int i = 0; i < SATSPLAT_NUM_STAGES; ++i) ctx->ev_used[i] = 0;
  return SATSPLAT_OK;
}

int satsplat_stage_ms(satsplat_ctx* ctx, float* ms_out) {
  if (!ctx || !ms_out) return fail(ctx, SATSPLAT_E_INVALID, "satsplat_stage_ms: NULL argument");
  CU(cudaSetDevice(ctx->device));
  for (int i = 0; i < SATSPLAT_NUM_STAGES; ++i) {
    ms_out[i] = 0.f;
    if (ctx->profiling && ctx->ev_used[i]) {
      CU(cudaEventSynchronize(ctx->ev[2 * i + 1]));
      CU(cudaEventElapsedTime(&ms_out[i], ctx->ev[2 * i], ctx->ev[2 * i + 1]));
    }
  }
  return SATSPLAT_OK;
}

namespace {
// float offset of sub-array k of the packed surfel staging (means 3N, quats 4N, scales 2N, logits N, rgb 3N): every
// sub-array starts on a 16-byte boundary whatever N is (the kernels use float4 / float2 accesses on them)
inline size_t align4(size_t x) { return (x + 3) & ~(size_t)3; }
struct Pack { size_t off[6]; };
inline Pack pack_offsets(size_t n) {
  static const int w[5] = {3, 4, 2, 1, 3};
  Pack p;
  p.off[0] = 0;
  for (int k = 0; k < 5; ++k) p.off[k + 1] = p.off[k] + align4(n * (size_t)w[k]);
  return p;
}
}  // namespace

namespace {
// frees whatever a failed satsplat_reserve_host_staging left behind, so that a retry starts from nothing
void release_staging(satsplat_ctx* ctx) {
  float** bufs[] = {ctx->e2e_in, ctx->e2e_up, ctx->e2e_out, ctx->e2e_grads, ctx->e2e_target, ctx->e2e_loss};
  for (float** b : bufs)
    for (int k = 0; k < 2; ++k)
      if (b[k]) { cudaFree(b[k]); b[k] = nullptr; }
  for (int k = 0; k < 2; ++k)
    for (int i = 0; i < 6; ++i)
      if (ctx->e2e_ev[k][i]) { cudaEventDestroy(ctx->e2e_ev[k][i]); ctx->e2e_ev[k][i] = nullptr; }
  for (int i = 0; i < 3; ++i)
    if (ctx->e2e_stream[i]) { cudaStreamDestroy(ctx->e2e_stream[i]); ctx->e2e_stream[i] = nullptr; }
}

cudaError_t allocate_staging(satsplat_ctx* ctx) {
  const size_t mpx = (size_t)ctx->max_w * ctx->max_h;
  const Pack pk = pack_offsets((size_t)ctx->max_surfels);
  cudaError_t e;
#define TRY(call) if ((e = (call)) != cudaSuccess) return e
  for (int k = 0; k < 2; ++k) {
    TRY(dalloc(ctx, &ctx->e2e_in[k], pk.off[5] + 4));
    TRY(dalloc(ctx, &ctx->e2e_up[k], mpx * 12));
    TRY(dalloc(ctx, &ctx->e2e_out[k], mpx * 12));
    TRY(dalloc(ctx, &ctx->e2e_grads[k], pk.off[5] + 64));
    TRY(dalloc(ctx, &ctx->e2e_target[k], mpx * 4));
    TRY(dalloc(ctx, &ctx->e2e_loss[k], (size_t)satsplat_loss_scratch_floats(ctx->max_w, ctx->max_h)));
    for (int i = 0; i < 6; ++i) TRY(cudaEventCreateWithFlags(&ctx->e2e_ev[k][i], cudaEventDisableTiming));
  }
  for (int i = 0; i < 3; ++i) TRY(cudaStreamCreateWithFlags(&ctx->e2e_stream[i], cudaStreamNonBlocking));
#undef TRY
  return cudaSuccess;
}
}  // namespace

int satsplat_reserve_host_staging(satsplat_ctx* ctx, satsplat_ctx* sun_ctx) {
  if (!ctx) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_reserve_host_staging: ctx is NULL");
  CU(cudaSetDevice(ctx->device));
  if (!ctx->staging_ready) {
    const int64_t before = ctx->scratch_bytes;
    const cudaError_t e = allocate_staging(ctx);
    if (e != cudaSuccess) {      // nothing half-built survives: a later call tries again from scratch
      release_staging(ctx);
      ctx->scratch_bytes = before;
      return fail(ctx, SATSPLAT_E_CUDA, "satsplat_reserve_host_staging: %s", cudaGetErrorString(e));
    }
    ctx->staging_ready = 1;
  }
  if (sun_ctx && !sun_ctx->e2e_sun) {   // its own field: a context may serve as view context and as sun context
    const size_t mpx = (size_t)sun_ctx->max_w * sun_ctx->max_h;
    const cudaError_t e = dalloc(sun_ctx, &sun_ctx->e2e_sun, mpx * 2);   // sun map + its gradient
    if (e != cudaSuccess) return fail(ctx, SATSPLAT_E_CUDA, "satsplat_reserve_host_staging: %s", cudaGetErrorString(e));
  }
  return SATSPLAT_OK;
}

// One step with host buffers.  lw == NULL: the upstream gradients come from the host (h_v_*); lw != NULL (training step):
// they are written on the device by the loss stage from the rendered images and the uploaded target, and the loss sums
// come back with the gradients.
static int host_step_enqueue(satsplat_ctx* ctx, satsplat_ctx* sun_ctx, int32_t slot, const satsplat_camera* cam,
                           const satsplat_sun* sun, const satsplat_shading* shading, int64_t N,
                           const float* h_means, const float* h_quats, const float* h_scales,
                           const float* h_logits, const float* h_rgb, const float* h_v_rgba, const float* h_v_geom,
                           const float* h_v_aux, float* h_out_rgba, float* h_out_geom, float* h_out_aux,
                           float* h_grads, const satsplat_loss_weights* lw, const float* h_target, float* h_sums,
                           satsplat_stream stream) {
  if (!ctx) return fail(nullptr, SATSPLAT_E_INVALID, "satsplat_iteration_host: ctx is NULL");
  if (lw && (!h_target || !h_sums)) return fail(ctx, SATSPLAT_E_INVALID, "satsplat_training_step_host: bad argument");
  if (!cam || !shading || !h_means || !h_quats || !h_scales || !h_logits || !h_rgb || !h_grads || N <= 0 || slot < 0 || slot > 1)
    return fail(ctx, SATSPLAT_E_INVALID, "satsplat_iteration_host: bad argument");
  // every size is checked before the first copy is enqueued
  if (N > ctx->max_surfels) return fail(ctx, SATSPLAT_E_INVALID, "satsplat_iteration_host: N exceeds max_surfels");
  if (cam->width <= 0 || cam->height <= 0 || cam->width > ctx->max_w || cam->height > ctx->max_h)
    return fail(ctx, SATSPLAT_E_INVALID, "satsplat_iteration_host: image size exceeds the context");
  const bool shadows = shading->shadows_on != 0;
  if (shadows) {
    if (!sun_ctx || !sun) return fail(ctx, SATSPLAT_E_INVALID, "satsplat_iteration_host: shadows need sun_ctx and sun");
    if (N > sun_ctx->max_surfels || sun->width <= 0 || sun->height <= 0 || sun->width > sun_ctx->max_w || sun->height > sun_ctx->max_h)
      return fail(ctx, SATSPLAT_E_INVALID, "satsplat_iteration_host: sun map size or N exceeds the sun context");
  }
  if (!ctx->staging_ready || (shadows && !sun_ctx->e2e_sun))
    return fail(ctx, SATSPLAT_E_STATE, "satsplat_iteration_host: call satsplat_reserve_host_staging first");
  if (ctx->e2e_busy[slot]) return fail(ctx, SATSPLAT_E_STATE, "satsplat_iteration_host_begin: slot still in flight (call _end)");
  // the two slots share the contexts' scratch (records, lists, per-pixel state, moment records, the sun map): their kernels
  // are ordered only by running on ONE stream
  if (ctx->e2e_busy[slot ^ 1] && ctx->e2e_caller[slot ^ 1] != (cudaStream_t)stream)
    return fail(ctx, SATSPLAT_E_STATE, "satsplat_iteration_host_begin: the step in flight on the other slot was begun on a different stream");
  if (ctx->split_backward || (shadows && sun_ctx->split_backward))
    return fail(ctx, SATSPLAT_E_STATE, "satsplat_iteration_host: the contexts are in SATSPLAT_OPT_SPLIT_BACKWARD mode");
  cudaStream_t s = (cudaStream_t)stream;
  CU(cudaSetDevice(ctx->device));
  // the sun camera and the reprojection constants are derived from F' = F + dF (Eq. 16, cascade of Fig. 1)
  satsplat_camera sun_cam;
  satsplat_shading sh = *shading;
  if (shadows) {
    const int rc0 = satsplat_sun_camera(cam, sun->azimuth, sun->elevation, sun->width, sun->height, sun->viewport, &sun_cam, sh.reproj);
    if (rc0) return fail(ctx, rc0, "satsplat_iteration_host: %s", satsplat_last_error(nullptr));
  }
  const size_t n = (size_t)N, px = (size_t)cam->width * cam->height;
  const size_t spx = shadows ? (size_t)sun->width * sun->height : 0;
  // Three queues.  Every host->device copy of the step goes up on the upload stream as soon as it is enqueued: while the
  // caller's stream is still busy with the kernels of the previous step (other slot), this step's 257 MB are already
  // crossing PCIe.  The caller's stream carries the kernels; the images come down on the download stream while the
  // backward runs, the gradients after it (PCIe is full duplex).
  cudaStream_t s_up = ctx->e2e_stream[0], s_down = ctx->e2e_stream[1], s_view = ctx->e2e_stream[2];
  cudaEvent_t* ev = ctx->e2e_ev[slot];   // 0 surfels up, 1 upstream up, 2 forward done, 3 backward done, 4 everything down, 5 view preprocess done
  const Pack pk = pack_offsets(n);
  float* d_in[5];
  const float* h_in[5] = {h_means, h_quats, h_scales, h_logits, h_rgb};
  static const int width[5] = {3, 4, 2, 1, 3};
  for (int k = 0; k < 5; ++k) {
    d_in[k] = ctx->e2e_in[slot] + pk.off[k];
    CU(cudaMemcpyAsync(d_in[k], h_in[k], n * width[k] * sizeof(float), cudaMemcpyHostToDevice, s_up));
  }
  CU(cudaEventRecord(ev[0], s_up));
  float* d_up[3] = {nullptr, nullptr, nullptr};
  const float* h_up[3] = {h_v_rgba, h_v_geom, h_v_aux};
  for (int k = 0; k < 3; ++k)
    if (lw) {
      d_up[k] = ctx->e2e_up[slot] + (size_t)k * 4 * (size_t)ctx->max_w * ctx->max_h;
    } else if (h_up[k]) {
      d_up[k] = ctx->e2e_up[slot] + (size_t)k * 4 * (size_t)ctx->max_w * ctx->max_h;
      CU(cudaMemcpyAsync(d_up[k], h_up[k], px * 16, cudaMemcpyHostToDevice, s_up));
    }
  if (lw) CU(cudaMemcpyAsync(ctx->e2e_target[slot], h_target, px * 16, cudaMemcpyHostToDevice, s_up));
  CU(cudaEventRecord(ev[1], s_up));
  float* d_out[3];
  for (int k = 0; k < 3; ++k) d_out[k] = ctx->e2e_out[slot] + (size_t)k * 4 * (size_t)ctx->max_w * ctx->max_h;
  // device gradients: the five surfel groups at 16-byte aligned offsets, then dF(8) cc(12) ambient(3) reproj(8) dF_sun(8)
  float* g = ctx->e2e_grads[slot];
  CU(cudaMemsetAsync(g, 0, (pk.off[5] + 40) * sizeof(float), s));
  float* g_grp[5];
  for (int k = 0; k < 5; ++k) g_grp[k] = g + pk.off[k];
  float *g_dF = g + pk.off[5], *g_cc = g_dF + 8, *g_amb = g_cc + 12, *g_rep = g_dF + 24, *g_dFs = g_dF + 32;
  float* d_sun = nullptr;
  float* d_vsun = nullptr;
  int rc;
  CU(cudaStreamWaitEvent(s, ev[0], 0));
  if (shadows) {
    // the view pass's preprocess + binning needs the surfels only: it runs beside the sun pass.  It follows the caller's
    // stream up to here (the previous step's backward reads the view context's records) and joins before render_forward.
    CU(cudaEventRecord(ev[5], s));
    CU(cudaStreamWaitEvent(s_view, ev[5], 0));
    if ((rc = satsplat_preprocess(ctx, cam, N, d_in[0], d_in[1], d_in[2], d_in[3], d_in[4], (satsplat_stream)s_view))) return rc;
    CU(cudaEventRecord(ev[5], s_view));
    d_sun = sun_ctx->e2e_sun;
    d_vsun = d_sun + (size_t)sun_ctx->max_w * sun_ctx->max_h;
    if ((rc = satsplat_preprocess(sun_ctx, &sun_cam, N, d_in[0], d_in[1], d_in[2], d_in[3], d_in[4], stream))) return rc;
    if ((rc = satsplat_shadow_map(sun_ctx, d_sun, stream))) return rc;
    CU(cudaMemsetAsync(d_vsun, 0, spx * sizeof(float), s));
    sh.sun_depth = d_sun;
    sh.sun_width = sun->width;
    sh.sun_height = sun->height;
  }
  if (shadows) CU(cudaStreamWaitEvent(s, ev[5], 0));
  else if ((rc = satsplat_preprocess(ctx, cam, N, d_in[0], d_in[1], d_in[2], d_in[3], d_in[4], stream))) return rc;
  if ((rc = satsplat_render_forward(ctx, &sh, d_out[0], d_out[1], d_out[2], stream))) return rc;
  CU(cudaEventRecord(ev[2], s));
  float* h_out[3] = {h_out_rgba, h_out_geom, h_out_aux};
  CU(cudaStreamWaitEvent(s_down, ev[2], 0));
  for (int k = 0; k < 3; ++k)
    if (h_out[k]) CU(cudaMemcpyAsync(h_out[k], d_out[k], px * 16, cudaMemcpyDeviceToHost, s_down));
  CU(cudaStreamWaitEvent(s, ev[1], 0));
  float* const d_sums = g + pk.off[5] + 48;
  if (lw && (rc = satsplat_loss_upstream(cam, lw, d_out[0], d_out[1], d_out[2], ctx->e2e_target[slot], ctx->e2e_loss[slot], d_up[0],
                                         d_up[1], d_up[2], d_sums, stream)))
    return rc;
  if ((rc = satsplat_render_backward(ctx, &sh, d_up[0], d_up[1], d_up[2], g_grp[0], g_grp[1], g_grp[2], g_grp[3], g_grp[4], g_dF,
                                     g_cc, g_amb, d_vsun, shadows ? g_rep : nullptr, stream)))
    return rc;
  if (shadows) {
    if ((rc = satsplat_shadow_map_backward(sun_ctx, d_vsun, g_grp[0], g_grp[1], g_grp[2], g_grp[3], g_dFs, stream))) return rc;
    // cascade: the gradients of the sun camera and of the reprojection constants flow back into dF (Eq. 16 adjoint)
    if ((rc = satsplat_sun_camera_backward(cam, sun->azimuth, sun->elevation, sun->viewport, g_dFs, g_rep, g_dF, stream))) return rc;
  }
  CU(cudaEventRecord(ev[3], s));
  // h_grads stays packed (means 3N, quats 4N, scales 2N, logits N, rgb 3N, dF 8, cc 12, ambient 3)
  CU(cudaStreamWaitEvent(s_down, ev[3], 0));
  size_t ho = 0;
  for (int k = 0; k < 5; ++k) {
    CU(cudaMemcpyAsync(h_grads + ho, g_grp[k], n * width[k] * sizeof(float), cudaMemcpyDeviceToHost, s_down));
    ho += n * width[k];
  }
  CU(cudaMemcpyAsync(h_grads + ho, g_dF, 23 * sizeof(float), cudaMemcpyDeviceToHost, s_down));
  if (lw) CU(cudaMemcpyAsync(h_sums, d_sums, 8 * sizeof(float), cudaMemcpyDeviceToHost, s_down));
  CU(cudaEventRecord(ev[4], s_down));
  ctx->e2e_busy[slot] = 1;
  ctx->e2e_caller[slot] = s;
  return SATSPLAT_OK;
}

// A failure after the first copy was enqueued (a refused preprocess, a CUDA error) would leave asynchronous copies from and to
// the caller's buffers in flight on a slot that is not marked busy: drain the queues before reporting it, so that the caller
// may free or reuse its buffers as soon as _begin has returned an error.
static int host_step_begin(satsplat_ctx* ctx, satsplat_ctx* sun_ctx, int32_t slot, const satsplat_camera* cam,
                           const satsplat_sun* sun, const satsplat_shading* shading, int64_t N,
                           const float* h_means, const float* h_quats, const float* h_scales,
                           const float* h_logits, const float* h_rgb, const float* h_v_rgba, const float* h_v_geom,
                           const float* h_v_aux, float* h_out_rgba, float* h_out_geom, float* h_out_aux,
                           float* h_grads, const satsplat_loss_weights* lw, const float* h_target, float* h_sums,
                           satsplat_stream stream) {
  const int rc = host_step_enqueue(ctx, sun_ctx, slot, cam, sun, shading, N, h_means, h_quats, h_scales, h_logits, h_rgb, h_v_rgba,
                                   h_v_geom, h_v_aux, h_out_rgba, h_out_geom, h_out_aux, h_grads, lw, h_target, h_sums, stream);
  if (rc != SATSPLAT_OK && ctx && ctx->staging_ready) {
    for (int i = 0; i < 3; ++i) cudaStreamSynchronize(ctx->e2e_stream[i]);
    cudaStreamSynchronize((cudaStream_t)stream);
  }
  return rc;
}

int satsplat_iteration_host_begin(satsplat_ctx* ctx, satsplat_ctx* sun_ctx, int32_t slot, const satsplat_camera* cam,
                                  const satsplat_sun* sun, const satsplat_shading* shading, int64_t N,
                                  const float* h_means, const float* h_quats, const float* h_scales,
                                  const float* h_logits, const float* h_rgb, const float* h_v_rgba, const float* h_v_geom,
                                  const float* h_v_aux, float* h_out_rgba, float* h_out_geom, float* h_out_aux,
                                  float* h_grads, satsplat_stream stream) {
  return host_step_begin(ctx, sun_ctx, slot, cam, sun, shading, N, h_means, h_quats, h_scales, h_logits, h_rgb, h_v_rgba, h_v_geom,
                         h_v_aux, h_out_rgba, h_out_geom, h_out_aux, h_grads, nullptr, nullptr, nullptr, stream);
}

int satsplat_training_step_host_begin(satsplat_ctx* ctx, satsplat_ctx* sun_ctx, int32_t slot, const satsplat_camera* cam,
                                      const satsplat_sun* sun, const satsplat_shading* shading,
                                      const satsplat_loss_weights* weights, int64_t N, const float* h_means,
                                      const float* h_quats, const float* h_scales, const float* h_logits, const float* h_rgb,
                                      const float* h_target_rgba, float* h_out_rgba, float* h_grads, float* h_loss_sums,
                                      satsplat_stream stream) {
  if (!weights) return fail(ctx, SATSPLAT_E_INVALID, "satsplat_training_step_host: weights is NULL");
  return host_step_begin(ctx, sun_ctx, slot, cam, sun, shading, N, h_means, h_quats, h_scales, h_logits, h_rgb, nullptr, nullptr,
                         nullptr, h_out_rgba, nullptr, nullptr, h_grads, weights, h_target_rgba, h_loss_sums, stream);
}

int satsplat_iteration_host_end(satsplat_ctx* ctx, int32_t slot) {
  if (!ctx || slot < 0 || slot > 1) return fail(ctx, SATSPLAT_E_INVALID, "satsplat_iteration_host_end: bad argument");
  if (!ctx->e2e_busy[slot]) return fail(ctx, SATSPLAT_E_STATE, "satsplat_iteration_host_end: no begin on this slot");
  CU(cudaSetDevice(ctx->device));
  ctx->e2e_busy[slot] = 0;
  CU(cudaEventSynchronize(ctx->e2e_ev[slot][4]));   // images and gradients are in the host buffers
  CU(cudaEventSynchronize(ctx->e2e_ev[slot][3]));
  return SATSPLAT_OK;
}

int satsplat_iteration_host(satsplat_ctx* ctx, satsplat_ctx* sun_ctx, const satsplat_camera* cam,
                            const satsplat_sun* sun, const satsplat_shading* shading, int64_t N,
                            const float* h_means, const float* h_quats, const float* h_scales,
                            const float* h_logits, const float* h_rgb, const float* h_v_rgba, const float* h_v_geom,
                            const float* h_v_aux, float* h_out_rgba, float* h_out_geom, float* h_out_aux,
                            float* h_grads, satsplat_stream stream) {
  const int rc = satsplat_iteration_host_begin(ctx, sun_ctx, 0, cam, sun, shading, N, h_means, h_quats, h_scales, h_logits, h_rgb,
                                               h_v_rgba, h_v_geom, h_v_aux, h_out_rgba, h_out_geom, h_out_aux, h_grads, stream);
  if (rc) return rc;
  return satsplat_iteration_host_end(ctx, 0);
}

int satsplat_training_step_host_end(satsplat_ctx* ctx, int32_t slot) { return satsplat_iteration_host_end(ctx, slot); }

int satsplat_training_step_host(satsplat_ctx* ctx, satsplat_ctx* sun_ctx, const satsplat_camera* cam, const satsplat_sun* sun,
                                const satsplat_shading* shading, const satsplat_loss_weights* weights, int64_t N,
                                const float* h_means, const float* h_quats, const float* h_scales, const float* h_logits,
                                const float* h_rgb, const float* h_target_rgba, float* h_out_rgba, float* h_grads,
                                float* h_loss_sums, satsplat_stream stream) {
  const int rc = satsplat_training_step_host_begin(ctx, sun_ctx, 0, cam, sun, shading, weights, N, h_means, h_quats, h_scales,
                                                   h_logits, h_rgb, h_target_rgba, h_out_rgba, h_grads, h_loss_sums, stream);
  if (rc) return rc;
  return satsplat_iteration_host_end(ctx, 0);
}

}  // extern "C"

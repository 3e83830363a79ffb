/* satsplat.h — C ABI of the B200-native affine-2DGS rasteriser (SatSplat hot path, arxiv/paper_2606_28581).
 *
 * Boundary of the product: plain C, plain pointers and sizes, no C++ or torch types.  Every pointer
 * argument says whether it is a HOST or a DEVICE pointer.  Citations are PAPER.md line numbers
 * (/root/reference/PAPER.md at build time) plus the equation they fall in.
 *
 * Conventions
 *   - Every function returns an int: SATSPLAT_OK (0) or a negative SATSPLAT_E_* code.  No exception or C++
 *     type crosses the ABI.  satsplat_last_error(ctx) returns a message owned by the context.
 *   - Ownership: the caller owns every input and output buffer.  The opaque satsplat_ctx owns only scratch
 *     (per-surfel records, tile rects, counts/offsets, key/value double buffers, tile ranges, per-pixel
 *     state, per-surfel gradient records), sized ONCE at satsplat_create from
 *     (max_surfels, max_width, max_height, max_duplicates).  The hot calls (preprocess / shadow_map /
 *     render_forward / render_backward / shadow_map_backward) allocate nothing, never synchronise with the
 *     host, and enqueue all work on the caller's stream.  Exceeding max_duplicates sets a device flag that
 *     satsplat_sync_status surfaces as SATSPLAT_E_CAPACITY (outputs of that pass are then undefined but no
 *     out-of-bounds access happens).
 *   - One context per camera pass in flight: the view pass and the sun pass of one training iteration use
 *     two contexts so that both stay alive for the backward.
 *   - Layouts: fp32, row-major, contiguous, 16-byte aligned device buffers.
 *       surfels  means[N,3]  quats[N,4] (w,x,y,z; need not be unit)  scales[N,2] (linear, > 0, world units)
 *                opacity_logits[N]  rgb[N,3]                                        (PAPER.md:69-79 Eq. 3-4, :145)
 *       images   [H,W,4] float4 groups:
 *                out_rgba = (I_r, I_g, I_b, A)       Eq. 1 colour (:59) and alpha = 1 - T
 *                out_geom = (N_x, N_y, N_z, D)       blended world normal (:133) and expected depth sum w z (Eq. 14)
 *                out_aux  = (median depth, distortion, V, T)   V = sun visibility (:55), T = final transmittance
 *     Pixel (i,j) has its centre at (i+0.5, j+0.5), x to the right, y down.  F maps WORLD UNITS DIRECTLY TO
 *     THESE PIXEL COORDINATES (the caller folds the paper's NDC step, :63, into F).
 *   - Gradient outputs are ACCUMULATED INTO (+=) caller-zeroed buffers, because the view pass and the sun
 *     pass both contribute to the same surfel gradients.
 *   - Method constants: 16x16 tiles (:140); sigma = 1/sqrt(2) px (Eq. 12);
 *     rho cut-off 9; alpha skip 1/255; alpha clamp 0.99; transmittance stop 1e-4; |det| <= 1e-6 => degenerate.
 */
#ifndef SATSPLAT_H_
#define SATSPLAT_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SATSPLAT_OK 0
#define SATSPLAT_E_INVALID (-1)  /* null pointer, bad shape, N or image larger than the context was created for */
#define SATSPLAT_E_CAPACITY (-2) /* duplicated keys K exceeded max_duplicates (reported by satsplat_sync_status) */
#define SATSPLAT_E_CUDA (-3)     /* a CUDA runtime call failed; message in satsplat_last_error */
#define SATSPLAT_E_STATE (-4)    /* calls out of order (e.g. render_forward before preprocess) */

typedef struct satsplat_ctx satsplat_ctx;
typedef void* satsplat_stream; /* a cudaStream_t (0 = default stream) */

/* One affine camera (PAPER.md:63-65 Eq. 2, :97-105 Eq. 6-7, :155-163 Eq. 15).  HOST struct, passed by pointer. */
typedef struct {
  int32_t width, height; /* pixels; tiles are 16x16 (:140) */
  float F[8];            /* 2x4 row-major [B_xy | b_xy]: world -> pixel                      (Eq. 2, 7) */
  float dF[8];           /* 2x4 delta; the effective camera is F' = F + dF (fp32 add)        (Eq. 15)   */
  float view_dir[3];     /* unit viewing direction, sensor -> scene (prop. to B_x x B_y)     (:165)     */
  float b_z;             /* max_altitude: depth z = b_z - world_z                            (Eq. 11)   */
  float z_bg;            /* background depth composited behind the last surfel                          */
  float bg_rgb[3];       /* background albedo                                                           */
} satsplat_camera;

/* Image formation I = (C A + c) (.) (V + (1 - V) L_a)  (Eq. 1) and the soft shadow test
 * V = sigmoid(-slope (z_view - d_sun(x_s) - depth_bias)) with x_s = R_x x + k_h h + k_0 (:153, :165-167).
 * HOST struct; sun_depth is a DEVICE pointer. */
typedef struct {
  float cc[12];           /* 3x4 row-major [C | c]; identity + zero bias = no correction */
  float ambient[3];       /* L_a */
  int32_t shadows_on;     /* 0: V == 1 everywhere and the sun fields are ignored */
  int32_t sun_width, sun_height;
  const float* sun_depth; /* DEVICE [sun_height, sun_width]: background-composited sun-view depth (satsplat_shadow_map) */
  float reproj[8];        /* 2x4 [R_x | k_h | k_0] from satsplat_sun_camera */
  float depth_bias, slope;
} satsplat_shading;

/* ---- lifetime ------------------------------------------------------------------------------------------ */
/* Allocates all scratch on `device` (cudaMalloc; the only allocating call besides satsplat_reserve_host_staging).  max_duplicates bounds K, the
 * number of (tile, surfel) pairs of one pass. */
int satsplat_create(satsplat_ctx** out, int device, int64_t max_surfels, int32_t max_width, int32_t max_height,
                    int64_t max_duplicates);
void satsplat_destroy(satsplat_ctx* ctx);
const char* satsplat_last_error(const satsplat_ctx* ctx); /* never NULL; ctx may be NULL */
int64_t satsplat_scratch_bytes(const satsplat_ctx* ctx);  /* device bytes owned by the context */

/* ---- camera helper (host arithmetic only) -------------------------------------------------------------- */
/* Sun-direction affine camera of PAPER.md:165-173 Eq. 16 / :317-345 Eq. S1-S6: B_sun = B' (I - [0 0 s]),
 * s = (cos(az)/tan(el), sin(az)/tan(el), 1), B' = B + dB of `view`; followed by the 2-D viewport
 * x_px = viewport[0..1] (.) x + viewport[2..3] that fits the flattened scene into sun_w x sun_h.  Azimuth from +X
 * toward +Y, elevation above the horizon, radians.  sun_out gets dF = 0, the depth row of `view` (the sun depth
 * is the original elevation, :167) and view_dir = -(cos az cos el, sin az cos el, sin el).  reproj_out is the
 * 2x4 map view pixel + height -> sun pixel used by the shadow test.  All HOST pointers. */
int satsplat_sun_camera(const satsplat_camera* view, float azimuth, float elevation, int32_t sun_w, int32_t sun_h,
                        const float viewport[4], satsplat_camera* sun_out, float reproj_out[8]);

/* Cascade camera optimisation (Fig. 1 :159): the sun camera is DERIVED from the refined view camera
 * F' = F + dF, so what reaches the sun camera's 2x4 matrix (v_dF_sun of satsplat_shadow_map_backward) and the
 * reprojection constants (v_reproj of satsplat_render_backward) flows back into dF.  This is the adjoint of
 * satsplat_sun_camera with respect to F': for a camera built by Eq. 16 the reprojection is
 * x_s = diag(sc) x - sc (B' s) h + t, so only its k_h column depends on F', and
 *   v_dF[r][c] += sc_r (v_F_sun[r][c] - s_c (v_F_sun[r][2] + v_reproj[r][2]))   c = 0,1,2   (s_2 = 1)
 *   v_dF[r][3] += sc_r  v_F_sun[r][3].
 * `view`, `viewport` HOST (same values as given to satsplat_sun_camera); v_F_sun, v_reproj DEVICE [8] (either may be
 * NULL = zero); v_dF DEVICE [8], accumulated into.  One tiny kernel on `stream`, no host synchronisation.
 * Errors: SATSPLAT_E_INVALID (NULL view / viewport / v_dF, zero elevation), SATSPLAT_E_CUDA. */
int satsplat_sun_camera_backward(const satsplat_camera* view, float azimuth, float elevation, const float viewport[4],
                                 const float* v_F_sun, const float* v_reproj, float* v_dF, satsplat_stream stream);

/* ---- hot path ------------------------------------------------------------------------------------------ */
/* (a1)+(a2) per-surfel preprocess and binning (PAPER.md:97-131 Eq. 6-12; :140).  Per surfel: rotation from the
 * quaternion, M = B' R S' (Eq. 8), Q = M^-1 (Eq. 10), centre c, height depth z_c (Eq. 11), depth slope, opacity,
 * sensor-facing normal, 3-sigma extent widened to the low-pass disc of Eq. 12, tile rect and count; then exclusive
 * scan, key duplication (tile << 32 | order-preserving depth bits), stable radix sort and per-tile ranges.
 * All array arguments are DEVICE pointers; `cam` is a HOST pointer.  Requires N <= max_surfels and
 * cam->width/height <= max_width/max_height.  The five surfel buffers must stay valid and unmodified until the
 * backward of this pass has been enqueued (the per-surfel chain rule re-reads them). */
int satsplat_preprocess(satsplat_ctx* ctx, const satsplat_camera* cam, int64_t N, const float* means,
                        const float* quats, const float* scales, const float* opacity_logits, const float* rgb,
                        satsplat_stream stream);

/* (a3)+(a5) per-16x16-tile front-to-back compositing (Eq. 14) of colour, alpha, expected depth,
 * normal, median depth and the depth-distortion term, with the Eq. 1 colour correction and shadow test fused
 * into the epilogue.  Outputs are DEVICE [H,W,4] buffers (any may be NULL to skip the store); `shading` HOST. */
int satsplat_render_forward(satsplat_ctx* ctx, const satsplat_shading* shading, float* out_rgba, float* out_geom,
                            float* out_aux, satsplat_stream stream);

/* Depth-only compositing on a preprocessed SUN context: sun_depth_out[Hs,Ws] = D + T z_bg (DEVICE pointer). */
int satsplat_shadow_map(satsplat_ctx* sun_ctx, float* sun_depth_out, satsplat_stream stream);

/* (a4) backward of satsplat_render_forward: epilogue backward (v_cc, v_ambient, v_reproj, scatter into
 * v_sun_depth), compositing backward in reverse order with warp-shuffle reduction before any atomics, then the
 * per-surfel chain to (means, quats, scales, logits, rgb) and the reduction to v_dF (Eq. 15).
 * Upstream v_rgba / v_geom / v_aux: DEVICE [H,W,4], any may be NULL (= zero); v_aux channels (d median,
 * d distortion, ignored, ignored).  All v_* outputs are DEVICE pointers, accumulated into (+=); any may be NULL
 * (v_sun_depth / v_reproj must be non-NULL only if the caller wants them). */
int satsplat_render_backward(satsplat_ctx* ctx, const satsplat_shading* shading, const float* v_rgba,
                             const float* v_geom, const float* v_aux, float* v_means, float* v_quats,
                             float* v_scales, float* v_opacity_logits, float* v_rgb, float* v_dF /*[8]*/,
                             float* v_cc /*[12]*/, float* v_ambient /*[3]*/, float* v_sun_depth /*[Hs,Ws]*/,
                             float* v_reproj /*[8]*/, satsplat_stream stream);

/* Backward of satsplat_shadow_map: v_sun_depth DEVICE [Hs,Ws]; surfel gradients and v_dF_sun (gradient w.r.t.
 * the sun camera's 2x4) accumulated into DEVICE buffers. */
int satsplat_shadow_map_backward(satsplat_ctx* sun_ctx, const float* v_sun_depth, float* v_means, float* v_quats,
                                 float* v_scales, float* v_opacity_logits, float* v_dF_sun /*[8]*/,
                                 satsplat_stream stream);

/* The sun of one view: angles (radians; azimuth from +X toward +Y, elevation above the horizon, Eq. S2), the size of
 * its depth map and the 2-D viewport (scale x, scale y, shift x, shift y) that fits the flattened footprint in it. */
typedef struct {
  float azimuth, elevation;
  int32_t width, height;
  float viewport[4];
} satsplat_sun;

/* ---- (f2) device-resident cameras: the cascade camera chain of PAPER.md:155-176, Fig. 1 --------------------------------
 * With dF stepped on the device by the optimiser every iteration, cameras baked into kernel arguments would force a
 * re-capture of the step's CUDA graph per view and per step.  Here the per-view constants live in a DEVICE array of
 * satsplat_view_params, dF in a DEVICE [V,8] array, the current view in a DEVICE int32, and satsplat_camera_chain
 * (one tiny kernel) builds from them a DEVICE camera block:
 *   floats [0,16) view camera, [16,32) sun camera, [32,48) nearby camera, each (F'[8], view_dir[3], b_z, z_bg, bg[3]);
 *   [48,76) the view's shading constants: cc[12], ambient[3], reproj[8], depth_bias, slope; [76,80) unused.
 * The *_device calls read their camera / shading from that block through a pointer. */
#define SATSPLAT_CAMERA_BLOCK_FLOATS 80
#define SATSPLAT_CAM_VIEW 0
#define SATSPLAT_CAM_SUN 1
#define SATSPLAT_CAM_NEARBY 2

typedef struct {            /* constants of one view; fill with satsplat_view_params_fill, then copy to the device */
  float F[8];               /* 2x4 world -> pixel (Eq. 2, 7); dF is NOT here: it is the learnable [V,8] array          */
  float view_dir[3];
  float b_z;
  float z_bg;
  float bg_rgb[3];
  float cc[12];             /* Eq. 1 */
  float ambient[3];
  float depth_bias;
  float slope;
  float nearby_d_azimuth;   /* perturbation of the azimuth / elevation of d_main = B_x x B_y for the nearby camera     */
  float nearby_d_elevation; /* (PAPER.md:176); radians                                                                 */
  float pad0;
  float sun_viewport[4];
  double sun_s[2];          /* (cos phi / tan theta, sin phi / tan theta) of Eq. S2, from the sun angles (metadata)     */
  float sun_view_dir[3];
  float pad1;
} satsplat_view_params;

/* HOST helper: fills `out` from the host structs (`shading` gives cc, ambient, depth_bias, slope; `sun` the angles and
 * viewport; both may be NULL = identity colour correction / no sun).  The trigonometry of Eq. S2 is done here, once,
 * in double, exactly as satsplat_sun_camera does it, so that the device-built sun camera is bit-equal to the helper's. */
int satsplat_view_params_fill(const satsplat_camera* cam, const satsplat_shading* shading, const satsplat_sun* sun,
                              float nearby_d_azimuth, float nearby_d_elevation, satsplat_view_params* out);

/* Builds the camera block of view *view_index (DEVICE int32; NULL = view 0) from views[V] and dF[V,8] (DEVICE; dF may be
 * NULL = zero): F' = F + dF (Eq. 15), sun camera + reprojection constants (Eq. 16 + viewport, bit-equal to
 * satsplat_sun_camera), nearby camera, shading constants.  One kernel, no host synchronisation. */
int satsplat_camera_chain(const satsplat_view_params* views, const float* dF, const int32_t* view_index, float* block,
                          satsplat_stream stream);

/* Adjoint of satsplat_camera_chain with respect to dF: v_dF_all[*view_index] += v_dF_view (the view pass's own gradient,
 * DEVICE [8]) + adjoint of the sun camera applied to v_F_sun (sun pass) and v_reproj (shadow test) + adjoint of the
 * nearby camera applied to v_F_nearby (a nearby-view pass).  Any of the four [8] inputs may be NULL (= zero).
 * v_dF_all DEVICE [V,8], accumulated into. */
int satsplat_camera_chain_backward(const satsplat_view_params* views, const float* dF, const int32_t* view_index,
                                   const float* v_dF_view, const float* v_F_sun, const float* v_reproj, const float* v_F_nearby,
                                   float* v_dF_all, satsplat_stream stream);

/* *view_index = (*view_index + stride) % n_views on the device (so that a captured graph can walk through the views). */
int satsplat_advance_view_index(int32_t* view_index, int32_t stride, int32_t n_views, satsplat_stream stream);

/* satsplat_preprocess with the camera `which` (SATSPLAT_CAM_*) of a DEVICE camera block; width / height (host values,
 * fixed per context) size the grid.  The context then renders from the device camera: satsplat_shadow_map,
 * satsplat_shadow_map_backward work unchanged; the view pass uses the two *_device calls below. */
int satsplat_preprocess_device(satsplat_ctx* ctx, int32_t width, int32_t height, const float* block, int32_t which, int64_t N,
                               const float* means, const float* quats, const float* scales, const float* opacity_logits,
                               const float* rgb, satsplat_stream stream);

/* satsplat_render_forward / satsplat_render_backward with cc, ambient, reproj, depth_bias, slope read from the block;
 * sun_depth DEVICE [sun_height, sun_width] or NULL (= shadows off).  SATSPLAT_E_STATE unless the context was
 * preprocessed by satsplat_preprocess_device. */
int satsplat_render_forward_device(satsplat_ctx* ctx, const float* block, const float* sun_depth, int32_t sun_width,
                                   int32_t sun_height, float* out_rgba, float* out_geom, float* out_aux, satsplat_stream stream);
int satsplat_render_backward_device(satsplat_ctx* ctx, const float* block, const float* sun_depth, int32_t sun_width,
                                    int32_t sun_height, const float* v_rgba, const float* v_geom, const float* v_aux,
                                    float* v_means, float* v_quats, float* v_scales, float* v_opacity_logits, float* v_rgb,
                                    float* v_dF /*[8]*/, float* v_cc /*[12]*/, float* v_ambient /*[3]*/,
                                    float* v_sun_depth /*[Hs,Ws]*/, float* v_reproj /*[8]*/, satsplat_stream stream);


/* Allocates the device staging buffers satsplat_iteration_host and satsplat_training_step_host need (sized for the
 * contexts' maxima; 45 floats per pixel and 26 per surfel for the two slots of the view context) and their two copy streams.  The only allocating call besides satsplat_create; idempotent; `sun_ctx` may be NULL.  If an allocation fails (SATSPLAT_E_CUDA) everything this call had allocated so far is freed again and a later call starts afresh. */
int satsplat_reserve_host_staging(satsplat_ctx* ctx, satsplat_ctx* sun_ctx);

/* One whole training-view iteration with HOST buffers (end-to-end leg of the benchmark): copies the surfels and
 * upstream gradients host->device, builds the sun camera and the reprojection constants from F' = F + dF (Eq. 16;
 * shading->reproj / sun_depth are ignored when shading->shadows_on), runs sun pass + view pass forward + backward of
 * both + the cascade chain of the sun camera back into dF (Fig. 1), copies images and gradients back, and
 * synchronises `stream`: exactly the work of the staged device calls.  h_* are HOST pointers (pinned memory
 * recommended); h_grads = packed [N*13 + 8 + 12 + 3] floats: means(3N) quats(4N) scales(2N) logits(N) rgb(3N) dF(8)
 * cc(12) ambient(3), any N (the device staging is padded to 16-byte boundaries internally).  All sizes are validated
 * before the first copy.  `sun_ctx` / `sun` may be NULL when shadows are off.  SATSPLAT_E_STATE if
 * satsplat_reserve_host_staging has not been called. */
int satsplat_iteration_host(satsplat_ctx* ctx, satsplat_ctx* sun_ctx, const satsplat_camera* cam,
                            const satsplat_sun* sun, const satsplat_shading* shading, int64_t N,
                            const float* h_means, const float* h_quats, const float* h_scales,
                            const float* h_logits, const float* h_rgb, const float* h_v_rgba, const float* h_v_geom,
                            const float* h_v_aux, float* h_out_rgba, float* h_out_geom, float* h_out_aux,
                            float* h_grads, satsplat_stream stream);

/* The same iteration split in two, so that the copies of consecutive steps overlap (the upload of step i+1 crosses PCIe
 * while the kernels of step i run): _begin enqueues everything for one step on staging slot `slot` (0 or 1) and returns
 * without synchronising; _end blocks until that step's images and gradients are in the host buffers.  A slot can be
 * begun again only after its _end (SATSPLAT_E_STATE otherwise); the host buffers of a step must stay valid and
 * untouched until its _end.  The two slots share the contexts' scratch, so both steps in flight must be begun on the SAME
 * `stream` (SATSPLAT_E_STATE otherwise); if _begin fails after copies were enqueued it drains them before returning, so the
 * caller's buffers are free again on any error.  satsplat_iteration_host == _begin(slot 0) + _end(slot 0). */
int satsplat_iteration_host_begin(satsplat_ctx* ctx, satsplat_ctx* sun_ctx, int32_t slot, const satsplat_camera* cam,
                                  const satsplat_sun* sun, const satsplat_shading* shading, int64_t N,
                                  const float* h_means, const float* h_quats, const float* h_scales,
                                  const float* h_logits, const float* h_rgb, const float* h_v_rgba, const float* h_v_geom,
                                  const float* h_v_aux, float* h_out_rgba, float* h_out_geom, float* h_out_aux,
                                  float* h_grads, satsplat_stream stream);
int satsplat_iteration_host_end(satsplat_ctx* ctx, int32_t slot);

/* ---- optimiser step ------------------------------------------------------- */
/* One Adam step [Kingma & Ba 2015, Alg. 1] over the five surfel groups with per-group learning rates (PAPER.md:349:
 * 0.075 means, 0.0025 colour, 0.001 quaternions and scales; the paper names no opacity rate, no betas and no epsilon:
 * all are arguments).  theta <- theta - lr m^/(sqrt(v^) + eps) with m^ = m/(1 - beta1^t), v^ = v/(1 - beta2^t); the
 * scale group is stepped in log space (theta = log s, dL/dtheta = s dL/ds, s <- s exp(-step)) so that the linear
 * scales of this library stay positive, and its state is that of log s.
 * HOST struct.  lr[] in the order means, quats, scales, opacity logits, rgb; step = t >= 1. */
typedef struct {
  float lr[5];
  float beta1, beta2, eps;
  int32_t step;
} satsplat_adam;
/* Floats in each of the two state arrays for N surfels (13 N rounded so that every group starts 16-byte aligned). */
int64_t satsplat_adam_state_floats(int64_t N);
/* All pointers DEVICE, fp32, 16-byte aligned.  Parameters are updated in place; gradients are read only; adam_m and
 * adam_v (satsplat_adam_state_floats(N) floats each, zero before the first step) are caller-owned state, updated in
 * place.  One kernel on `stream`, no host synchronisation.  Errors: SATSPLAT_E_INVALID (NULL pointer, N < 0,
 * step < 1, beta outside [0,1)), SATSPLAT_E_CUDA. */
int satsplat_adam_step(int64_t N, float* means, float* quats, float* scales, float* opacity_logits, float* rgb,
                       const float* v_means, const float* v_quats, const float* v_scales, const float* v_opacity_logits,
                       const float* v_rgb, float* adam_m, float* adam_v, const satsplat_adam* hp, satsplat_stream stream);

/* The same step for the per-camera groups ("0.0001 for camera delta matrices, and 0.001 for camera gain and
 * bias"): the row of dF (Eq. 15), the 3x4 [C | c] and the ambient term (Eq. 1) of the view *view_index (DEVICE int32; NULL =
 * view 0).  One training iteration renders one view, so only that view has a gradient: its 23 values, their state and its
 * own step counter advance (bias correction from steps[view] + 1); every other view is left untouched.  A schedule such as
 * "camera loss from iteration 3000" is the caller's: pass lr = 0 until then.
 *   views     DEVICE [n_views] table (the one satsplat_camera_chain reads); cc and ambient are updated IN it
 *   dF        DEVICE [n_views,8], updated in place; v_dF_all DEVICE [n_views,8] as accumulated by
 *             satsplat_camera_chain_backward (the view's row is set to zero afterwards if clear_v_dF != 0); both NULL = group off
 *   v_cc [12], v_ambient [3]   DEVICE gradients of the rendered view (satsplat_render_backward*); NULL = group off
 *   adam_m, adam_v DEVICE [n_views,23] (dF 8, cc 12, ambient 3 per view), zero before the first step; steps DEVICE int32
 *             [n_views], zero before the first step
 *   hp        HOST; lr[] in the order dF, cc, ambient
 * One 32-thread kernel on `stream`, no host synchronisation; all view-dependent state is on the device, so a captured graph
 * serves every view.  Errors: SATSPLAT_E_INVALID, SATSPLAT_E_CUDA. */
typedef struct {
  float lr[3];
  float beta1, beta2, eps;
} satsplat_camera_adam;
int satsplat_adam_step_cameras(int32_t n_views, const int32_t* view_index, satsplat_view_params* views, float* dF, float* v_dF_all,
                               const float* v_cc, const float* v_ambient, float* adam_m, float* adam_v, int32_t* steps,
                               const satsplat_camera_adam* hp, int32_t clear_v_dF, satsplat_stream stream);

/* ---- loss stage ----------------------------------------------------------- */
/* L = w_l1 mean|I - I*| + w_ssim (1 - mean SSIM(I, I*)) + w_dist mean(L_dist) + w_normal mean(1 - A_sg N_r . N_d)
 * (PAPER.md:349 lists the terms and weights 0.8 / 0.2 / 0.05 / 0.05; :133-138 Eq. 13 defines N_d) and its gradients with
 * respect to the three rendered images = the upstream gradients of satsplat_render_backward.
 *   I = out_rgba.xyz, A = out_rgba.w, N_r = out_geom.xyz (alpha-weighted rendered normal), D = out_geom.w,
 *   L_dist = out_aux.y; means over the H W pixels (and 3 channels for L1 / SSIM).
 *   SSIM: 11x11 Gaussian window, sigma 1.5, zero padding, C1 = 0.01^2, C2 = 0.03^2, per channel.
 *   N_d (Eq. 13): normal of the world point map backprojected from the background-composited depth
 *   z_v = D + (1 - A) z_bg with F' = F + dF (height h = b_z - z_v), central differences on interior pixels, zero on
 *   the one-pixel border, oriented towards the sensor; A_sg = alpha with stop-gradient (2DGS's normal consistency).
 * HOST: cam, w.  DEVICE, fp32, 16-byte aligned: the three rendered images and target_rgba [H,W,4] (4th channel of
 * the target ignored); scratch (satsplat_loss_scratch_floats(W, H) floats); v_rgba / v_geom / v_aux [H,W,4] are
 * OVERWRITTEN with dL/d(out_rgba, out_geom, out_aux); loss_sums [8]: [0] sum |I - I*| (divide by 3 H W), [1] sum of the
 * SSIM map (3 H W), [2] sum L_dist (H W), [3] sum (1 - A N_r.N_d) (H W), rest zero.  Three kernels ordered after the
 * work already queued on `stream` and before any work queued on it later (one of them runs on an internal side stream,
 * forked and joined with events: capturable in a CUDA graph); no host synchronisation.  The side stream and its two
 * events are per device and shared by all calls: calls for one device must not be issued from several host threads at
 * the same time (issue them from one thread, on any streams).  Errors: SATSPLAT_E_INVALID (NULL pointer, singular camera), SATSPLAT_E_CUDA. */
typedef struct {
  float w_l1, w_ssim, w_dist, w_normal;
} satsplat_loss_weights;
int64_t satsplat_loss_scratch_floats(int32_t width, int32_t height);
int satsplat_loss_upstream(const satsplat_camera* cam, const satsplat_loss_weights* w, const float* out_rgba,
                           const float* out_geom, const float* out_aux, const float* target_rgba, float* scratch,
                           float* v_rgba, float* v_geom, float* v_aux, float* loss_sums, satsplat_stream stream);

/* One whole TRAINING step with HOST buffers: satsplat_iteration_host with the loss stage in the middle.  Copies the
 * surfels and the target image host->device, runs sun pass + view pass forward, satsplat_loss_upstream on the rendered
 * images (its upstream gradients never leave the device), the backward of both passes and the cascade chain, and copies
 * back the packed gradients (layout of satsplat_iteration_host), the 8 loss sums of satsplat_loss_upstream and, if
 * h_out_rgba is not NULL, the rendered image.  Per step this moves 13 N + 4 H W floats up and 13 N + 31 floats down
 * instead of the 13 N + 12 H W up / 13 N + 12 H W down of the rasteriser-only call.  _begin / _end as for
 * satsplat_iteration_host (the two families share the staging slots: a slot carries one step of either kind at a
 * time).  h_target_rgba [H,W,4] (4th channel ignored), h_loss_sums [8]: HOST.  Errors as satsplat_iteration_host. */
int satsplat_training_step_host(satsplat_ctx* ctx, satsplat_ctx* sun_ctx, const satsplat_camera* cam, const satsplat_sun* sun,
                                const satsplat_shading* shading, const satsplat_loss_weights* weights, int64_t N,
                                const float* h_means, const float* h_quats, const float* h_scales, const float* h_logits,
                                const float* h_rgb, const float* h_target_rgba, float* h_out_rgba, float* h_grads,
                                float* h_loss_sums, satsplat_stream stream);
int satsplat_training_step_host_begin(satsplat_ctx* ctx, satsplat_ctx* sun_ctx, int32_t slot, const satsplat_camera* cam,
                                      const satsplat_sun* sun, const satsplat_shading* shading,
                                      const satsplat_loss_weights* weights, int64_t N, const float* h_means,
                                      const float* h_quats, const float* h_scales, const float* h_logits, const float* h_rgb,
                                      const float* h_target_rgba, float* h_out_rgba, float* h_grads, float* h_loss_sums,
                                      satsplat_stream stream);
int satsplat_training_step_host_end(satsplat_ctx* ctx, int32_t slot);

/* ---- geometry-aware initialisation ----------------------------------------- */
/* Surfels from a DSM.  dsm[row, col] heights on a regular grid of spacing `cell`; the centre of
 * cell (row, col) is at (origin_x + (col + 0.5) cell, origin_y + (row + 0.5) cell).
 *   area-weighted sampling (:186): weight a = |dx x dy| = cell^2 sqrt(1 + h_x^2 + h_y^2) with finite-difference slopes
 *     (central inside, one-sided on the border); sample k takes the first cell, in row-major order, whose cumulative
 *     weight exceeds u[k] * total (cumulative sum in double precision); its centre is
 *     (origin + (col + jx[k], row + jy[k]) cell, h + h_x (jx - 0.5) cell + h_y (jy - 0.5) cell) (tangent-plane lift);
 *     u, jx, jy in [0, 1) are the CALLER's random numbers;
 *   orientation (:192): n = (-h_x, -h_y, 1)/|.|, t_u = world x axis made orthogonal to n (Gram-Schmidt), t_v = n x t_u,
 *     quaternion (w, x, y, z) of R = [t_u | t_v | n], w >= 0;
 *   scale (:194): s_u = s_v = mean distance to the 3 nearest other sampled centres (exact kNN); `cell` if N <= 3.
 * All pointers DEVICE: dsm [dsm_h, dsm_w], u / jx / jy [N], scratch (satsplat_init_scratch_bytes bytes, 16-byte aligned),
 * outputs means [N,3], quats [N,4], scales [N,2] fp32 and, if not NULL, cells_out [N] int32 (the sampled row-major cell
 * index).  Nine kernels on `stream`, no host synchronisation.  Errors: SATSPLAT_E_INVALID, SATSPLAT_E_CUDA. */
int64_t satsplat_init_scratch_bytes(int32_t dsm_w, int32_t dsm_h, int64_t N);
int satsplat_init_from_dsm(const float* dsm, int32_t dsm_w, int32_t dsm_h, float cell, float origin_x, float origin_y, int64_t N,
                           const float* u, const float* jx, const float* jy, void* scratch, float* means, float* quats,
                           float* scales, int32_t* cells_out, satsplat_stream stream);

/* ---- relocation of dead surfels (second half) ------------------------------ */
/* PAPER.md:200 "use the 3DGS-MCMC [22] strategy to relocate Gaussians during training".  A surfel is DEAD if
 * sigmoid(logit) <= o_min ([22]: 0.005; decided on the logit).  Every dead surfel draws a live source j with probability
 * proportional to opacity: the first j, in index order, whose cumulative live opacity exceeds u[d] * total (double
 * precision; u in [0,1) are the CALLER's random numbers, only those of dead surfels are read).  A source drawn by n - 1
 * dead surfels (n capped at n_max; [22]: 51) and its n - 1 copies all get opacity o' = 1 - (1 - alpha)^(1/n) (clamped to
 * [o_min, 1 - 1e-7]) and scales multiplied by alpha / D, D = sum_{i=1..n} sum_{k<i} C(i-1,k) (-1)^k o'^(k+1) / sqrt(k+1):
 * the n copies composited at the centre give alpha back and the composited profile keeps its integral.  A dead surfel
 * also takes the source's centre, rotation and colour.  The Adam state (layout of satsplat_adam_step; both NULL = none) of
 * every dead surfel and every drawn source is cleared.  No live surfel: nothing moves.
 * All pointers DEVICE; parameters and state are updated in place; scratch: satsplat_relocate_scratch_bytes(N) bytes,
 * 16-byte aligned; src_out [N] int32 (may be NULL): source index of a relocated surfel, -1 otherwise.  Seven kernels on
 * `stream`, no host synchronisation.  Errors: SATSPLAT_E_INVALID, SATSPLAT_E_CUDA. */
int64_t satsplat_relocate_scratch_bytes(int64_t N);
int satsplat_relocate(int64_t N, float* means, float* quats, float* scales, float* opacity_logits, float* rgb, float* adam_m,
                      float* adam_v, const float* u, float o_min, int32_t n_max, void* scratch, int32_t* src_out,
                      satsplat_stream stream);

/* satsplat_relocate for callers that cannot supply scratch memory.  Same operation, same arguments (minus `scratch`), same
 * results, but the working memory is an array built into the library instead of a caller buffer, and the call itself never
 * allocates or frees device memory.  It is meant for hosts where an allocation at this point is not an option: the
 * surrounding framework has already claimed the whole GPU for its own pool and exposes no C allocator, the job runs under a
 * hard memory quota, or the training loop cannot afford the device-wide pause that an allocation or a free brings.
 *   Limit: N <= SATSPLAT_RELOCATE_STATIC_MAX_SURFELS (131072; the array is about 3.5 MB).  A larger N is refused with
 *     SATSPLAT_E_INVALID and a message that names the limit; nothing is launched.  Use satsplat_relocate beyond it.
 *   Cost: each GPU on which the library is loaded carries the array from load until the process exits, used or not.
 *   First call per device: looks up the array's device address (cudaGetSymbolAddress with the caller's current device) and
 *     keeps it; make that first call with the right device current and outside any stream capture.  Later calls only launch.
 *   Sharing: all calls on one GPU work in the same array.  The array keeps whatever the previous call wrote; that is
 *     harmless because every call rewrites each entry before reading it (nothing needs to be cleared by the caller).  Two
 *     calls whose kernels can overlap on the GPU (different streams without an event between them, or several host threads)
 *     corrupt each other: order them on one stream or with events.
 * Pointers, in-place updates, u, o_min, n_max, src_out and `stream` exactly as for satsplat_relocate.
 * Errors: SATSPLAT_E_INVALID (bad argument, NULL pointer, N over the limit), SATSPLAT_E_CUDA; message via
 * satsplat_last_error(NULL). */
#define SATSPLAT_RELOCATE_STATIC_MAX_SURFELS 131072
int satsplat_relocate_static(int64_t N, float* means, float* quats, float* scales, float* opacity_logits, float* rgb,
                             float* adam_m, float* adam_v, const float* u, float o_min, int32_t n_max, int32_t* src_out,
                             satsplat_stream stream);

/* ---- status, test and profiling access ------------------------------------------------------------------ */
/* Synchronises `stream`, then reports the last preprocess: K (duplicated keys) and whether max_duplicates
 * overflowed (returns SATSPLAT_E_CAPACITY then).  HOST pointers, may be NULL. */
int satsplat_sync_status(satsplat_ctx* ctx, int64_t* K, satsplat_stream stream);

/* Pointers into the context's scratch for the bit-exact binning checks (DEVICE pointers returned through HOST
 * pointer arguments; valid until the next preprocess on this context; K read with a stream sync):
 * keys[K] = (tile << 32) | depth bits, sorted; vals[K] surfel ids; tile_ranges[tiles,2]; rects[N,4] uint16
 * (tx0,ty0,tx1,ty1); counts[N] uint32. */
int satsplat_debug_bins(satsplat_ctx* ctx, int64_t* K, const uint64_t** keys, const uint32_t** vals,
                        const uint32_t** tile_ranges, const uint16_t** rects, const uint32_t** counts,
                        satsplat_stream stream);

/* Second half of a backward call made with SATSPLAT_OPT_SPLIT_BACKWARD = 1 on `ctx`: turns the moment records the blend half
 * left into surfel gradients (accumulated into v_means ... v_rgb, DEVICE, any may be NULL; v_rgb is ignored for a
 * depth-only context), reduces v_dF and delivers v_cc / v_ambient / v_reproj.  Must run after the blend half (stream
 * order or an event) and before the next backward on `ctx`; two chains that accumulate into the same gradient buffers must
 * be ordered by the caller.  SATSPLAT_E_STATE if no split backward is pending.  While one IS pending, satsplat_preprocess*,
 * satsplat_render_backward*, satsplat_shadow_map_backward and satsplat_set_option(SATSPLAT_OPT_SPLIT_BACKWARD) on `ctx` return
 * SATSPLAT_E_STATE and launch nothing (the moment records would otherwise be overwritten or added to twice). */
int satsplat_backward_chain(satsplat_ctx* ctx, float* v_means, float* v_quats, float* v_scales, float* v_opacity_logits, float* v_rgb,
                            float* v_dF /*[8]*/, float* v_cc /*[12]*/, float* v_ambient /*[3]*/, float* v_reproj /*[8]*/,
                            satsplat_stream stream);

/* Copies the per-surfel records of the last preprocess into records_out (DEVICE [N,16] fp32) in the canonical
 * order (c_x, c_y, Q00, Q01, Q10, Q11, z_c, g0, g1, alpha, r, g, b, n_x, n_y, n_z) and flags_out (DEVICE [N] uint8:
 * bit0 culled, bit1 degenerate, bit2 normal flipped). */
int satsplat_debug_records(satsplat_ctx* ctx, float* records_out, uint8_t* flags_out, satsplat_stream stream);

/* Per-pixel planes of the last forward: n_visited[H,W] (tile-list entries visited, including the one that
 * triggered the transmittance stop) and n_contrib[H,W] (composited entries); DEVICE int32 pointers owned by
 * the context.  Their sums are the evaluated / contributing pair counts the roofline is quoted against.
 * Instrumentation, not part of the method: the forward stores them (8 B / pixel) only while
 * SATSPLAT_OPT_DEBUG_PLANES is 1 (default 0); SATSPLAT_E_STATE if the last forward ran without it. */
int satsplat_debug_planes(satsplat_ctx* ctx, const int32_t** n_visited, const int32_t** n_contrib);

/* Per-stage device times of the most recent hot call on this context, measured with CUDA events on the
 * caller's stream when profiling is enabled (costs event records, no host sync until the query).
 * Stage ids: SATSPLAT_STAGE_*.  ms_out HOST [SATSPLAT_NUM_STAGES]; stages that did not run report 0. */
#define SATSPLAT_STAGE_PREPROCESS 0
#define SATSPLAT_STAGE_SCAN 1
#define SATSPLAT_STAGE_DUPLICATE 2
#define SATSPLAT_STAGE_SORT 3
#define SATSPLAT_STAGE_RANGES 4
#define SATSPLAT_STAGE_BLEND_FWD 5
#define SATSPLAT_STAGE_BLEND_BWD 6
#define SATSPLAT_STAGE_CHAIN_BWD 7
#define SATSPLAT_NUM_STAGES 8
int satsplat_set_profiling(satsplat_ctx* ctx, int32_t enabled);
int satsplat_stage_ms(satsplat_ctx* ctx, float* ms_out);

/* Options (HOST call; takes effect at the next satsplat_preprocess).
 *   SATSPLAT_OPT_BINNING: how (a2) builds the sorted (tile, depth, surfel) list.  Both give the same, unique,
 *     bit-exact result (keys, order, ranges):
 *       SATSPLAT_BINNING_TILESORT (default) per-tile counts with atomics -> tile scan (= ranges) -> scatter -> one
 *                                           shared-memory sort per tile by (depth bits, surfel id); 4 launches
 *       SATSPLAT_BINNING_RADIX              per-surfel scan -> key duplication -> stable 8-bit LSD radix sort of the
 *                                           64-bit keys -> range detection; the general-purpose device sort */
#define SATSPLAT_OPT_BINNING 0
/*   SATSPLAT_OPT_SPLIT_BACKWARD (0 default / 1): with 1, satsplat_render_backward, satsplat_render_backward_device and
 *     satsplat_shadow_map_backward stop after their blend half (epilogue backward + reverse compositing: per-surfel moment
 *     records, v_sun_depth and the epilogue sums stay in the context; their v_means ... v_reproj arguments are ignored and
 *     may be NULL) and satsplat_backward_chain runs the per-surfel chain.  For callers that overlap the chain of one pass
 *     (HBM-bound) with the blend backward of the next pass (issue-bound) on two streams. */
#define SATSPLAT_OPT_SPLIT_BACKWARD 1
/*   SATSPLAT_OPT_DEBUG_PLANES (0 default / 1): the forward calls also store the per-pixel visit / contribution counters that
 *     satsplat_debug_planes returns (takes effect at the next forward). */
#define SATSPLAT_OPT_DEBUG_PLANES 2
#define SATSPLAT_BINNING_TILESORT 0
#define SATSPLAT_BINNING_RADIX 1
int satsplat_set_option(satsplat_ctx* ctx, int32_t option, int32_t value);

const char* satsplat_version(void);

/* Cumulative number of CUDA kernels this library has launched in this process (all contexts). */
int64_t satsplat_kernel_launches(void);

/* The two issue-rate peaks the blend kernels' roofline is quoted against, MEASURED on `device` by
 * two micro-benchmark kernels: FP32 lane-instructions per second (independent FFMA chains on every sub-partition)
 * and MUFU operations per second (independent ex2.approx chains).  HOST outputs; sm_count may be NULL.  Synchronises
 * the device (a few milliseconds): a measurement utility for bench.py, not part of the hot path. */
int satsplat_measure_peaks(int device, double* fp32_lane_inst_per_s, double* mufu_per_s, int* sm_count);

#ifdef __cplusplus
}
#endif
#endif /* SATSPLAT_H_ */

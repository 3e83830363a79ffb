// oracle/satsplat_oracle.cpp
//
// TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct CPU implementation of the affine-2DGS
// rasterisation path of SatSplat (arxiv/paper_2606_28581), written from /root/reference/PAPER.md.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load
// this file.  It shares no code, header, table or constant generator with the CUDA path under
// paper_2606_28581_b200/ and neither includes the other.
//
// What it computes, and where the paper defines it (PAPER.md line numbers):
//   * surfel P(u,v) = p_k + s_u t_u u + s_v t_v v                          Eq. 3-4,  l.69-79
//   * affine projection x = B_xy P + b_xy, z = B_z P + b_z                 Eq. 6-7,  l.97-105
//   * inverse map (u,v) = Q x + q, Q = (B_xy R S')^-1                      Eq. 8-10, l.107-120
//   * height depth B_z = [0 0 -1], b_z = max_altitude                      Eq. 11,   l.122-124
//   * lower-bounded Gaussian G^ = max(G(u(x)), G((x-c)/sigma))             Eq. 12,   l.126-131
//   * normal = last column of R, alpha-blended in world space              l.133-135
//   * bbox per splat, sort by centre depth, 16x16 tiles, alpha blending    Eq. 14,   l.140-145
//   * delta camera F' = F + dF                                             Eq. 15,   l.155-163
//   * sun camera B_sun = B_xy (I - [0 0 s])                                Eq. 16 / S1-S6, l.165-173, l.317-345
//   * image formation I = (C A + c) (.) (V + (1-V) L_a)                    Eq. 1,    l.55-61
// Where the paper is silent (sigma, cut-offs, alpha/T thresholds, median depth, distortion form, shadow
// test constants) the readings are those listed in DESIGN.md "Readings of the paper"; those constants
// are "parity unpinned" against the paper (they are this build's stated conventions).
//
// Structure: per-surfel preprocess (fp32 op-sequence for everything that feeds an integer, double for the
// smooth pins), reference binning (emit keys, std::stable_sort, ranges), a per-pixel compositor that walks
// ONE list of surfel ids in order (the list is either every surfel in depth order = "all-pairs", or the
// pixel's tile list), the Eq. 1 epilogue, and the analytic backward of all of it.  No blocking, fusion
// or reordering beyond what the algorithm states.  Floating point is double everywhere except the
// written fp32 contract of preprocess_f32.
//
// Build: g++ -O2 -std=c++17 -fopenmp -ffp-contract=off -shared -fPIC (see oracle/oracle.py).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---- constants (conventions of 3DGS/2DGS where the paper says "we follow") ----
constexpr int    kTile      = 16;
constexpr double kInvSigma2 = 2.0;         // sigma = 1/sqrt(2) px  => |d|^2 / sigma^2 = 2 |d|^2   (Eq. 12)
constexpr double kRhoCut    = 9.0;         // 3-sigma cut-off
constexpr double kAlphaMin  = 1.0 / 255.0;
constexpr double kAlphaMax  = 0.99;
constexpr double kTMin      = 1e-4;
constexpr float  kDetEpsF   = 1e-6f;       // |det(B_xy R S')| <= eps  => degenerate (l.126)
constexpr float  kLogitCull = -5.5373342f; // sigmoid(logit) < 1/255
constexpr float  kMinExtent = 2.1213204f;  // 3 sigma = 3/sqrt(2) px

enum : uint8_t { F_CULLED = 1, F_DEGENERATE = 2, F_FLIPPED = 4 };
enum : int32_t { OPT_NO_RHO_CUT = 1, OPT_NO_ALPHA_SKIP = 2, OPT_NO_T_STOP = 4 };

// canonical record layout (16 values per surfel)
enum { R_CX = 0, R_CY, R_Q00, R_Q01, R_Q10, R_Q11, R_ZC, R_G0, R_G1, R_ALPHA, R_R, R_G, R_B, R_NX, R_NY, R_NZ, R_SIZE };

}  // namespace

extern "C" {

struct orc_cam_f32 {
  int32_t width, height;
  float F[8], dF[8], view_dir[3], b_z;
};
struct orc_cam_f64 {
  int32_t width, height;
  double F[8], dF[8], view_dir[3], b_z;
};

struct orc_shading {
  double cc[12];        // 3x4 [C | c]
  double ambient[3];    // L_a
  int32_t shadows_on;
  int32_t sun_w, sun_h;
  int32_t _pad;
  const double* sun_depth;  // [sun_h, sun_w]
  double reproj[8];     // 2x4 [R_x | k_h | k_0]
  double bias, slope;
};

struct orc_render {
  int32_t width, height;
  double b_z, z_bg, bg[3];
  int32_t tile_mode;    // 1: lists are per-16x16-tile ranges into vals; 0: one global list for all pixels
  int32_t tiles_x;
  const uint32_t* vals;     // surfel ids
  const uint32_t* ranges;   // [tiles,2] (tile mode)
  int64_t list_len;         // global mode
  int32_t options;          // OPT_* (finite-difference pins switch the cut-offs off)
  int32_t threads;
};

// ---------------------------------------------------------------------------------------------------
// B. per-surfel preprocess, fp32 contract.  Every operation below is a single correctly-rounded IEEE
// binary32 operation in the written order (fmaf = fused); compiled with -ffp-contract=off.
// ---------------------------------------------------------------------------------------------------
static inline float sum2(float a, float b, float c, float d) { return fmaf(a, b, c * d); }
static inline float diff2(float a, float b, float c, float d) { return fmaf(a, b, -(c * d)); }

int orc_preprocess_f32(const orc_cam_f32* cam, int64_t N, const float* means, const float* quats,
                       const float* scales, const float* logits, const float* rgb, float* rec,
                       int32_t* rect, uint32_t* count, uint32_t* depth_key, uint8_t* flags) {
  const int TX = (cam->width + kTile - 1) / kTile, TY = (cam->height + kTile - 1) / kTile;
  float Fp[8];
  for (int i = 0; i < 8; ++i) Fp[i] = cam->F[i] + cam->dF[i];  // Eq. 15, one rounding
  const float B00 = Fp[0], B01 = Fp[1], B02 = Fp[2], b0 = Fp[3];
  const float B10 = Fp[4], B11 = Fp[5], B12 = Fp[6], b1 = Fp[7];
  for (int64_t i = 0; i < N; ++i) {
    const float* p = means + 3 * i;
    const float qw = quats[4 * i], qx = quats[4 * i + 1], qy = quats[4 * i + 2], qz = quats[4 * i + 3];
    const float su = scales[2 * i], sv = scales[2 * i + 1];
    float* r = rec + R_SIZE * i;
    uint8_t fl = 0;
    // 1. normalise the quaternion
    const float n2 = fmaf(qz, qz, fmaf(qy, qy, fmaf(qx, qx, qw * qw)));
    const float inv = 1.0f / sqrtf(n2);
    const float w = qw * inv, x = qx * inv, y = qy * inv, z = qz * inv;
    // 2. rotation columns: tangents t_u, t_v and normal n (Eq. 3-4; l.133)
    const float tu[3] = {1.0f - 2.0f * sum2(y, y, z, z), 2.0f * sum2(x, y, w, z), 2.0f * diff2(x, z, w, y)};
    const float tv[3] = {2.0f * diff2(x, y, w, z), 1.0f - 2.0f * sum2(x, x, z, z), 2.0f * sum2(y, z, w, x)};
    float nn[3] = {2.0f * sum2(x, z, w, y), 2.0f * diff2(y, z, w, x), 1.0f - 2.0f * sum2(x, x, y, y)};
    // 3. M = B_xy R S'  (Eq. 8)
    const float aux = fmaf(B02, tu[2], fmaf(B01, tu[1], B00 * tu[0]));
    const float auy = fmaf(B12, tu[2], fmaf(B11, tu[1], B10 * tu[0]));
    const float avx = fmaf(B02, tv[2], fmaf(B01, tv[1], B00 * tv[0]));
    const float avy = fmaf(B12, tv[2], fmaf(B11, tv[1], B10 * tv[0]));
    const float M00 = su * aux, M10 = su * auy, M01 = sv * avx, M11 = sv * avy;
    // 4. projected centre c = B_xy p + b_xy
    const float cx = fmaf(B02, p[2], fmaf(B01, p[1], fmaf(B00, p[0], b0)));
    const float cy = fmaf(B12, p[2], fmaf(B11, p[1], fmaf(B10, p[0], b1)));
    // 5. height-based depth (Eq. 11) and its order-preserving key
    const float zc = cam->b_z - p[2];
    uint32_t k;
    std::memcpy(&k, &zc, 4);
    k = (k & 0x80000000u) ? ~k : (k | 0x80000000u);
    // 6. extent: exact bbox of the 3-sigma ellipse M M^T, widened to the 3-sigma low-pass disc
    const float ex = fmaf(M01, M01, M00 * M00), ey = fmaf(M11, M11, M10 * M10);
    const float extx = fmaxf(3.0f * sqrtf(ex), kMinExtent), exty = fmaxf(3.0f * sqrtf(ey), kMinExtent);
    // 8. cull tests (before 7 so that non-finite values never reach the int conversion)
    bool cull = logits[i] < kLogitCull || !(n2 > 0.0f) || !(su > 0.0f) || !(sv > 0.0f) ||
                !std::isfinite(n2) || !std::isfinite(cx) || !std::isfinite(cy) || !std::isfinite(extx) ||
                !std::isfinite(exty) || !std::isfinite(zc);
    int tx0 = 0, tx1 = 0, ty0 = 0, ty1 = 0;
    if (!cull) {
      // 7. tile rect: floor in float, clamp in float to [-1, T], then to int
      auto tile_of = [](float v, int T) {
        float t = floorf(v * 0.0625f);
        t = fminf(fmaxf(t, -1.0f), (float)T);
        return (int)t;
      };
      tx0 = std::min(std::max(tile_of(cx - extx, TX), 0), TX);
      tx1 = std::min(std::max(tile_of(cx + extx, TX) + 1, 0), TX);
      ty0 = std::min(std::max(tile_of(cy - exty, TY), 0), TY);
      ty1 = std::min(std::max(tile_of(cy + exty, TY) + 1, 0), TY);
    } else {
      fl |= F_CULLED;
    }
    const int cnt = cull ? 0 : std::max(tx1 - tx0, 0) * std::max(ty1 - ty0, 0);
    rect[4 * i] = tx0; rect[4 * i + 1] = ty0; rect[4 * i + 2] = tx1; rect[4 * i + 3] = ty1;
    count[i] = (uint32_t)cnt;
    depth_key[i] = k;
    // 10. the record
    const float det = fmaf(M00, M11, -(M01 * M10));
    float Q00 = 0, Q01 = 0, Q10 = 0, Q11 = 0, g0 = 0, g1 = 0;
    if (!(fabsf(det) > kDetEpsF)) {
      fl |= F_DEGENERATE;
    } else {
      const float id = 1.0f / det;
      Q00 = M11 * id; Q01 = -M01 * id; Q10 = -M10 * id; Q11 = M00 * id;   // Eq. 10
      const float r0 = su * tu[2], r1 = sv * tv[2];
      g0 = -fmaf(r1, Q10, r0 * Q00);
      g1 = -fmaf(r1, Q11, r0 * Q01);
    }
    const float dotv = fmaf(nn[2], cam->view_dir[2], fmaf(nn[1], cam->view_dir[1], nn[0] * cam->view_dir[0]));
    if (dotv > 0.0f) { nn[0] = -nn[0]; nn[1] = -nn[1]; nn[2] = -nn[2]; fl |= F_FLIPPED; }
    const float alpha = (float)(1.0 / (1.0 + std::exp(-(double)logits[i])));
    r[R_CX] = cx; r[R_CY] = cy; r[R_Q00] = Q00; r[R_Q01] = Q01; r[R_Q10] = Q10; r[R_Q11] = Q11;
    r[R_ZC] = zc; r[R_G0] = g0; r[R_G1] = g1; r[R_ALPHA] = alpha;
    r[R_R] = rgb[3 * i]; r[R_G] = rgb[3 * i + 1]; r[R_B] = rgb[3 * i + 2];
    r[R_NX] = nn[0]; r[R_NY] = nn[1]; r[R_NZ] = nn[2];
    flags[i] = fl;
  }
  return 0;
}

// ---------------------------------------------------------------------------------------------------
// The same per-surfel quantities from the raw inputs, everything in double (smooth pins, finite
// differences).  Cull / degenerate decisions use the same thresholds.
// ---------------------------------------------------------------------------------------------------
struct SurfelGeom {  // intermediates shared by the double preprocess and its backward
  double qn, w, x, y, z;
  double tu[3], tv[3], n[3];
  double B[2][3], b[2];
  double au[2], av[2], M[2][2], det, Q[2][2], r[2];
  bool degenerate, flipped;
};

static void surfel_geom(const orc_cam_f64* cam, const double* p, const double* q, const double* s, SurfelGeom& G) {
  for (int r = 0; r < 2; ++r) {
    for (int c = 0; c < 3; ++c) G.B[r][c] = cam->F[4 * r + c] + cam->dF[4 * r + c];  // Eq. 15
    G.b[r] = cam->F[4 * r + 3] + cam->dF[4 * r + 3];
  }
  G.qn = std::sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
  const double w = q[0] / G.qn, x = q[1] / G.qn, y = q[2] / G.qn, z = q[3] / G.qn;
  G.w = w; G.x = x; G.y = y; G.z = z;
  G.tu[0] = 1 - 2 * (y * y + z * z); G.tu[1] = 2 * (x * y + w * z); G.tu[2] = 2 * (x * z - w * y);
  G.tv[0] = 2 * (x * y - w * z); G.tv[1] = 1 - 2 * (x * x + z * z); G.tv[2] = 2 * (y * z + w * x);
  G.n[0] = 2 * (x * z + w * y); G.n[1] = 2 * (y * z - w * x); G.n[2] = 1 - 2 * (x * x + y * y);
  for (int r = 0; r < 2; ++r) {
    G.au[r] = G.B[r][0] * G.tu[0] + G.B[r][1] * G.tu[1] + G.B[r][2] * G.tu[2];
    G.av[r] = G.B[r][0] * G.tv[0] + G.B[r][1] * G.tv[1] + G.B[r][2] * G.tv[2];
    G.M[r][0] = s[0] * G.au[r];
    G.M[r][1] = s[1] * G.av[r];
  }
  G.det = G.M[0][0] * G.M[1][1] - G.M[0][1] * G.M[1][0];
  G.degenerate = !(std::fabs(G.det) > (double)kDetEpsF);
  G.r[0] = s[0] * G.tu[2];
  G.r[1] = s[1] * G.tv[2];
  if (!G.degenerate) {
    G.Q[0][0] = G.M[1][1] / G.det; G.Q[0][1] = -G.M[0][1] / G.det;
    G.Q[1][0] = -G.M[1][0] / G.det; G.Q[1][1] = G.M[0][0] / G.det;
  } else {
    G.Q[0][0] = G.Q[0][1] = G.Q[1][0] = G.Q[1][1] = 0;
  }
  G.flipped = (G.n[0] * cam->view_dir[0] + G.n[1] * cam->view_dir[1] + G.n[2] * cam->view_dir[2]) > 0;
}

int orc_preprocess_f64(const orc_cam_f64* cam, int64_t N, const double* means, const double* quats,
                       const double* scales, const double* logits, const double* rgb, double* rec,
                       uint8_t* flags) {
  for (int64_t i = 0; i < N; ++i) {
    const double* p = means + 3 * i;
    const double* q = quats + 4 * i;
    const double* s = scales + 2 * i;
    double* r = rec + R_SIZE * i;
    uint8_t fl = 0;
    const double n2 = q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3];
    if (logits[i] < (double)kLogitCull || !(n2 > 0) || !(s[0] > 0) || !(s[1] > 0) || !std::isfinite(n2) ||
        !std::isfinite(p[0]) || !std::isfinite(p[1]) || !std::isfinite(p[2])) {
      flags[i] = F_CULLED;
      for (int k = 0; k < R_SIZE; ++k) r[k] = 0;
      continue;
    }
    SurfelGeom G;
    surfel_geom(cam, p, q, s, G);
    r[R_CX] = G.B[0][0] * p[0] + G.B[0][1] * p[1] + G.B[0][2] * p[2] + G.b[0];
    r[R_CY] = G.B[1][0] * p[0] + G.B[1][1] * p[1] + G.B[1][2] * p[2] + G.b[1];
    r[R_ZC] = cam->b_z - p[2];                                  // Eq. 11
    r[R_Q00] = G.Q[0][0]; r[R_Q01] = G.Q[0][1]; r[R_Q10] = G.Q[1][0]; r[R_Q11] = G.Q[1][1];
    // z(x) = b_z - P_z(u,v) = z_c - r.(u,v) = z_c + g.(x - c),  g = -r Q   (from Eq. 6 with Eq. 11)
    r[R_G0] = G.degenerate ? 0 : -(G.r[0] * G.Q[0][0] + G.r[1] * G.Q[1][0]);
    r[R_G1] = G.degenerate ? 0 : -(G.r[0] * G.Q[0][1] + G.r[1] * G.Q[1][1]);
    r[R_ALPHA] = 1.0 / (1.0 + std::exp(-logits[i]));
    r[R_R] = rgb[3 * i]; r[R_G] = rgb[3 * i + 1]; r[R_B] = rgb[3 * i + 2];
    const double sg = G.flipped ? -1.0 : 1.0;
    r[R_NX] = sg * G.n[0]; r[R_NY] = sg * G.n[1]; r[R_NZ] = sg * G.n[2];
    if (G.degenerate) fl |= F_DEGENERATE;
    if (G.flipped) fl |= F_FLIPPED;
    flags[i] = fl;
  }
  return 0;
}

// ---------------------------------------------------------------------------------------------------
// B9. reference binning: emit (tile, depth key) keys in surfel order, row-major over the rect, stable sort,
// tile ranges.  K = sum(count) is computed by the caller.
// ---------------------------------------------------------------------------------------------------
int orc_bin(int64_t N, int32_t TX, int32_t TY, const int32_t* rect, const uint32_t* count,
            const uint32_t* depth_key, int64_t K, uint64_t* keys, uint32_t* vals, uint32_t* ranges) {
  std::vector<std::pair<uint64_t, uint32_t>> kv;
  kv.reserve((size_t)K);
  for (int64_t i = 0; i < N; ++i) {
    if (count[i] == 0) continue;
    for (int ty = rect[4 * i + 1]; ty < rect[4 * i + 3]; ++ty)
      for (int tx = rect[4 * i]; tx < rect[4 * i + 2]; ++tx)
        kv.emplace_back(((uint64_t)(uint32_t)(ty * TX + tx) << 32) | depth_key[i], (uint32_t)i);
  }
  if ((int64_t)kv.size() != K) return -1;
  std::stable_sort(kv.begin(), kv.end(),
                   [](const std::pair<uint64_t, uint32_t>& a, const std::pair<uint64_t, uint32_t>& b) { return a.first < b.first; });
  for (int64_t t = 0; t < (int64_t)TX * TY; ++t) ranges[2 * t] = ranges[2 * t + 1] = 0;
  for (int64_t j = 0; j < K; ++j) {
    keys[j] = kv[j].first;
    vals[j] = kv[j].second;
    const uint32_t t = (uint32_t)(kv[j].first >> 32);
    if (j == 0 || (uint32_t)(kv[j - 1].first >> 32) != t) ranges[2 * t] = (uint32_t)j;
    ranges[2 * t + 1] = (uint32_t)(j + 1);
  }
  return 0;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------
// C. per-pixel forward: walk ONE list of surfel ids front to back.
// ---------------------------------------------------------------------------------------------------
namespace {

struct Hit {  // one composited surfel at one pixel
  uint32_t id;
  double a, G, T, w, z, u, v, dx, dy;
  bool lowpass;  // rho2 < rho3: the screen-space term of Eq. 12 won
  bool clamped;  // alpha*G >= alpha_max
};

struct PixelState {
  double C[3], N[3], M1, M2, L, T, med;
  int32_t mi;          // surfel id of the median-depth contributor, -1 if none
  int32_t n_visited;   // list entries visited (including the one that triggered the stop)
  int64_t n_contrib;
  int64_t n_lowpass, n_clamped, n_degenerate;   // composited pairs on the low-pass branch / with alpha clamped / of degenerate surfels
  double margin[6];    // smallest distance to each decision: rho cut, alpha skip, T stop, median, branch, clamp
};

void composite_pixel(const orc_render& cfg, const double* rec, const uint8_t* flags, const uint32_t* list,
                     int64_t len, double px, double py, PixelState& S, std::vector<Hit>* hits) {
  S.C[0] = S.C[1] = S.C[2] = S.N[0] = S.N[1] = S.N[2] = 0;
  S.M1 = S.M2 = S.L = 0;
  S.T = 1;
  S.med = cfg.z_bg;
  S.mi = -1;
  S.n_visited = 0;
  S.n_contrib = 0;
  S.n_lowpass = S.n_clamped = S.n_degenerate = 0;
  for (double& m : S.margin) m = std::numeric_limits<double>::infinity();
  if (hits) hits->clear();
  const double inf = std::numeric_limits<double>::infinity();
  for (int64_t j = 0; j < len; ++j) {
    const uint32_t id = list[j];
    if (flags[id] & F_CULLED) continue;
    S.n_visited = (int32_t)(j + 1);
    const double* r = rec + R_SIZE * id;
    const double dx = px - r[R_CX], dy = py - r[R_CY];
    const double u = r[R_Q00] * dx + r[R_Q01] * dy, v = r[R_Q10] * dx + r[R_Q11] * dy;   // Eq. 9
    const double rho3 = (flags[id] & F_DEGENERATE) ? inf : u * u + v * v;
    const double rho2 = kInvSigma2 * (dx * dx + dy * dy);
    const double rho = std::min(rho3, rho2);  // Eq. 12: max of two Gaussians = min of the exponents
    if (!(cfg.options & OPT_NO_RHO_CUT)) {
      S.margin[0] = std::min(S.margin[0], std::fabs(rho - kRhoCut));
      if (rho > kRhoCut) continue;
    }
    const double G = std::exp(-0.5 * rho);
    const double aG = r[R_ALPHA] * G;
    const double a = std::min(kAlphaMax, aG);
    if (!(cfg.options & OPT_NO_ALPHA_SKIP)) {
      S.margin[1] = std::min(S.margin[1], std::fabs(aG - kAlphaMin) / kAlphaMin);
      if (a < kAlphaMin) continue;
    }
    const double Tn = S.T * (1 - a);
    if (!(cfg.options & OPT_NO_T_STOP)) {
      S.margin[2] = std::min(S.margin[2], std::fabs(Tn - kTMin) / kTMin);
      if (Tn < kTMin) break;  // stop BEFORE compositing this surfel
    }
    S.margin[5] = std::min(S.margin[5], std::fabs(aG - kAlphaMax));
    if (std::isfinite(rho3)) S.margin[4] = std::min(S.margin[4], std::fabs(rho3 - rho2));
    const bool lowpass = !(rho3 <= rho2);
    const double w = a * S.T;
    const double z = lowpass ? r[R_ZC] : r[R_ZC] + r[R_G0] * dx + r[R_G1] * dy;  // Eq. 6 depth at the intersection
    S.margin[3] = std::min(S.margin[3], std::fabs(S.T - 0.5));
    if (S.T > 0.5) { S.med = z; S.mi = (int32_t)id; }
    S.L += w * (z * z * (1 - S.T) + S.M2 - 2 * z * S.M1);  // sum_{j<i} w_i w_j (z_i - z_j)^2
    for (int c = 0; c < 3; ++c) { S.C[c] += w * r[R_R + c]; S.N[c] += w * r[R_NX + c]; }   // Eq. 14
    S.M1 += w * z;
    S.M2 += w * z * z;
    if (hits) hits->push_back(Hit{id, a, G, S.T, w, z, u, v, dx, dy, lowpass, !(aG < kAlphaMax)});
    S.T = Tn;
    ++S.n_contrib;
    if (lowpass) ++S.n_lowpass;
    if (!(aG < kAlphaMax)) ++S.n_clamped;
    if (flags[id] & F_DEGENERATE) ++S.n_degenerate;
  }
}

struct ShadeState {  // D. epilogue intermediates
  double albedo[3], albedoC[3], shade[3], V, I[3];
  double zv, h, xs[2], ds, gap;
  bool in_map;
  int x0, y0, x1, y1;
  double fx, fy;
};

void shade_pixel(const orc_render& cfg, const orc_shading& sh, const PixelState& S, double px, double py, ShadeState& E) {
  for (int c = 0; c < 3; ++c) E.albedo[c] = S.C[c] + S.T * cfg.bg[c];
  for (int c = 0; c < 3; ++c)
    E.albedoC[c] = sh.cc[4 * c] * E.albedo[0] + sh.cc[4 * c + 1] * E.albedo[1] + sh.cc[4 * c + 2] * E.albedo[2] + sh.cc[4 * c + 3];
  E.V = 1;
  E.in_map = false;
  E.zv = S.M1 + S.T * cfg.z_bg;
  E.h = cfg.b_z - E.zv;
  if (sh.shadows_on) {
    E.xs[0] = sh.reproj[0] * px + sh.reproj[1] * py + sh.reproj[2] * E.h + sh.reproj[3];
    E.xs[1] = sh.reproj[4] * px + sh.reproj[5] * py + sh.reproj[6] * E.h + sh.reproj[7];
    if (E.xs[0] >= 0.5 && E.xs[0] <= sh.sun_w - 0.5 && E.xs[1] >= 0.5 && E.xs[1] <= sh.sun_h - 0.5) {
      E.in_map = true;
      const double tx = E.xs[0] - 0.5, ty = E.xs[1] - 0.5;
      E.x0 = (int)std::floor(tx); E.y0 = (int)std::floor(ty);
      E.x0 = std::min(E.x0, sh.sun_w - 1); E.y0 = std::min(E.y0, sh.sun_h - 1);
      E.fx = tx - E.x0; E.fy = ty - E.y0;
      E.x1 = std::min(E.x0 + 1, sh.sun_w - 1); E.y1 = std::min(E.y0 + 1, sh.sun_h - 1);
      const double* D = sh.sun_depth;
      const int W = sh.sun_w;
      E.ds = (1 - E.fy) * ((1 - E.fx) * D[E.y0 * W + E.x0] + E.fx * D[E.y0 * W + E.x1]) +
             E.fy * ((1 - E.fx) * D[E.y1 * W + E.x0] + E.fx * D[E.y1 * W + E.x1]);
      E.gap = E.zv - E.ds;
      E.V = 1.0 / (1.0 + std::exp(sh.slope * (E.gap - sh.bias)));
    }
  }
  for (int c = 0; c < 3; ++c) {
    E.shade[c] = E.V + (1 - E.V) * sh.ambient[c];   // Eq. 1 sun-sky shading
    E.I[c] = E.albedoC[c] * E.shade[c];             // Eq. 1
  }
}

inline void pixel_list(const orc_render& cfg, int ix, int iy, const uint32_t*& list, int64_t& len) {
  if (cfg.tile_mode) {
    const int t = (iy / kTile) * cfg.tiles_x + (ix / kTile);
    list = cfg.vals + cfg.ranges[2 * t];
    len = (int64_t)cfg.ranges[2 * t + 1] - (int64_t)cfg.ranges[2 * t];
  } else {
    list = cfg.vals;
    len = cfg.list_len;
  }
}

inline void atomic_add(double* p, double v) {
#pragma omp atomic
  *p += v;
}

}  // namespace

extern "C" {

// out_rgba [H,W,4] = (I rgb, A);  out_geom [H,W,4] = (N xyz, D);  out_aux [H,W,4] = (median depth,
// distortion, V, T_final);  albedo [H,W,3] (pre-correction, incl. T*bg);  last [H,W] = list entries
// visited;  med_idx [H,W];  margins [H,W,6];  counters[5] = (evaluated pairs, contributing pairs, and of the
// contributing pairs: on the low-pass branch of Eq. 12, with alpha clamped at alpha_max, of degenerate surfels).
int orc_forward(const orc_render* cfg, const orc_shading* sh, const double* rec, const uint8_t* flags,
                double* out_rgba, double* out_geom, double* out_aux, double* albedo, int32_t* last,
                int32_t* med_idx, double* margins, int64_t* counters) {
  const int W = cfg->width, H = cfg->height;
  int64_t evaluated = 0, contributing = 0, n_lowpass = 0, n_clamped = 0, n_degenerate = 0;
#pragma omp parallel for schedule(dynamic, 4) num_threads(cfg->threads > 0 ? cfg->threads : 1) reduction(+ : evaluated, contributing, n_lowpass, n_clamped, n_degenerate)
  for (int iy = 0; iy < H; ++iy) {
    for (int ix = 0; ix < W; ++ix) {
      const uint32_t* list; int64_t len;
      pixel_list(*cfg, ix, iy, list, len);
      const double px = ix + 0.5, py = iy + 0.5;
      PixelState S;
      composite_pixel(*cfg, rec, flags, list, len, px, py, S, nullptr);
      ShadeState E;
      shade_pixel(*cfg, *sh, S, px, py, E);
      const int64_t o = (int64_t)iy * W + ix;
      for (int c = 0; c < 3; ++c) { out_rgba[4 * o + c] = E.I[c]; out_geom[4 * o + c] = S.N[c]; }
      out_rgba[4 * o + 3] = 1 - S.T;
      out_geom[4 * o + 3] = S.M1;
      out_aux[4 * o] = S.med; out_aux[4 * o + 1] = S.L; out_aux[4 * o + 2] = E.V; out_aux[4 * o + 3] = S.T;
      if (albedo) for (int c = 0; c < 3; ++c) albedo[3 * o + c] = E.albedo[c];
      if (last) last[o] = S.n_visited;
      if (med_idx) med_idx[o] = S.mi;
      if (margins) for (int k = 0; k < 6; ++k) margins[6 * o + k] = S.margin[k];
      evaluated += S.n_visited;
      contributing += S.n_contrib;
      n_lowpass += S.n_lowpass; n_clamped += S.n_clamped; n_degenerate += S.n_degenerate;
    }
  }
  if (counters) {
    counters[0] = evaluated; counters[1] = contributing;
    counters[2] = n_lowpass; counters[3] = n_clamped; counters[4] = n_degenerate;
  }
  return 0;
}

// ---------------------------------------------------------------------------------------------------
// E. analytic backward of the epilogue and of the compositor.  Upstream gradients may be NULL (= 0).
// v_aux channels: (d median, d distortion, ignored, ignored).  All outputs are accumulated into (+=).
// v_rec [N,16] in the canonical record layout (gradient w.r.t. the flipped normal as stored).
// ---------------------------------------------------------------------------------------------------
//
// Rounding-error twin (tests only; every a_* pointer may be NULL).  a_rec [N,16], a_cc, a_ambient, a_reproj and
// a_sun_depth receive, for every gradient value above, the sum of the ABSOLUTE values of the per-pixel / per-pair
// terms that are added into it, each term itself being formed from absolute values of its factors (running error
// analysis: a floating-point evaluation of the same sums in precision eps is off by at most c eps a_* for a modest
// c that counts the operations per term and the length of the sum).  The twin is evaluated on the same gradient
// written in the depth frame shifted to the pixel's first contributor (z - z_0) and with the distortion adjoint in
// its centred form psi_i = A (z_i - m)^2 + (M2 - M1^2 / A), m = M1 / A: identical gradients, but their terms do not
// carry the cancellation of the raw depths (z ~ b_z), so a_* measures the conditioning of the sums, not of that frame.
int orc_backward(const orc_render* cfg, const orc_shading* sh, const double* rec, const uint8_t* flags,
                 const double* v_rgba, const double* v_geom, const double* v_aux, double* v_rec,
                 double* v_cc, double* v_ambient, double* v_reproj, double* v_sun_depth,
                 double* a_rec, double* a_cc, double* a_ambient, double* a_reproj, double* a_sun_depth) {
  const int W = cfg->width, H = cfg->height;
#pragma omp parallel num_threads(cfg->threads > 0 ? cfg->threads : 1)
  {
    std::vector<Hit> hits;
    std::vector<double> aphi;
    double l_cc[12] = {0}, l_amb[3] = {0}, l_rep[8] = {0};
    double t_cc[12] = {0}, t_amb[3] = {0}, t_rep[8] = {0};   // twins
#pragma omp for schedule(dynamic, 4)
    for (int iy = 0; iy < H; ++iy) {
      for (int ix = 0; ix < W; ++ix) {
        const uint32_t* list; int64_t len;
        pixel_list(*cfg, ix, iy, list, len);
        const double px = ix + 0.5, py = iy + 0.5;
        PixelState S;
        composite_pixel(*cfg, rec, flags, list, len, px, py, S, &hits);
        ShadeState E;
        shade_pixel(*cfg, *sh, S, px, py, E);
        const int64_t o = (int64_t)iy * W + ix;
        double vI[3] = {0, 0, 0}, vA = 0, vN[3] = {0, 0, 0}, vD = 0, vmed = 0, vL = 0;
        if (v_rgba) { for (int c = 0; c < 3; ++c) vI[c] = v_rgba[4 * o + c]; vA = v_rgba[4 * o + 3]; }
        if (v_geom) { for (int c = 0; c < 3; ++c) vN[c] = v_geom[4 * o + c]; vD = v_geom[4 * o + 3]; }
        if (v_aux) { vmed = v_aux[4 * o]; vL = v_aux[4 * o + 1]; }
        // ---- epilogue backward (Eq. 1) ----
        double v_albedo[3] = {0, 0, 0}, v_albedoC[3], vV = 0;
        for (int c = 0; c < 3; ++c) {
          const double v_shade = vI[c] * E.albedoC[c];
          v_albedoC[c] = vI[c] * E.shade[c];
          vV += v_shade * (1 - sh->ambient[c]);
          l_amb[c] += v_shade * (1 - E.V);
          for (int k = 0; k < 3; ++k) l_cc[4 * c + k] += v_albedoC[c] * E.albedo[k];
          l_cc[4 * c + 3] += v_albedoC[c];
          t_amb[c] += std::fabs(v_shade * (1 - E.V));
          for (int k = 0; k < 3; ++k) t_cc[4 * c + k] += std::fabs(v_albedoC[c] * E.albedo[k]);
          t_cc[4 * c + 3] += std::fabs(v_albedoC[c]);
        }
        for (int k = 0; k < 3; ++k)
          v_albedo[k] = sh->cc[k] * v_albedoC[0] + sh->cc[4 + k] * v_albedoC[1] + sh->cc[8 + k] * v_albedoC[2];
        double vT = 0;  // gradient w.r.t. the final transmittance T_f (A = 1 - T_f)
        if (sh->shadows_on && E.in_map) {
          const double v_gap = -sh->slope * E.V * (1 - E.V) * vV;
          double v_zv = v_gap;
          const double v_ds = -v_gap;
          const double* D = sh->sun_depth;
          const int SW = sh->sun_w;
          if (v_sun_depth) {
            atomic_add(&v_sun_depth[E.y0 * SW + E.x0], v_ds * (1 - E.fy) * (1 - E.fx));
            atomic_add(&v_sun_depth[E.y0 * SW + E.x1], v_ds * (1 - E.fy) * E.fx);
            atomic_add(&v_sun_depth[E.y1 * SW + E.x0], v_ds * E.fy * (1 - E.fx));
            atomic_add(&v_sun_depth[E.y1 * SW + E.x1], v_ds * E.fy * E.fx);
          }
          if (a_sun_depth) {
            atomic_add(&a_sun_depth[E.y0 * SW + E.x0], std::fabs(v_ds * (1 - E.fy) * (1 - E.fx)));
            atomic_add(&a_sun_depth[E.y0 * SW + E.x1], std::fabs(v_ds * (1 - E.fy) * E.fx));
            atomic_add(&a_sun_depth[E.y1 * SW + E.x0], std::fabs(v_ds * E.fy * (1 - E.fx)));
            atomic_add(&a_sun_depth[E.y1 * SW + E.x1], std::fabs(v_ds * E.fy * E.fx));
          }
          // d d_s / d x_s through the bilinear weights
          const double dds_dx = (1 - E.fy) * (D[E.y0 * SW + E.x1] - D[E.y0 * SW + E.x0]) + E.fy * (D[E.y1 * SW + E.x1] - D[E.y1 * SW + E.x0]);
          const double dds_dy = (1 - E.fx) * (D[E.y1 * SW + E.x0] - D[E.y0 * SW + E.x0]) + E.fx * (D[E.y1 * SW + E.x1] - D[E.y0 * SW + E.x1]);
          const double v_xs[2] = {v_ds * dds_dx, v_ds * dds_dy};
          const double v_h = sh->reproj[2] * v_xs[0] + sh->reproj[6] * v_xs[1];
          v_zv -= v_h;  // h = b_z - z_v
          for (int r = 0; r < 2; ++r) {
            l_rep[4 * r + 0] += v_xs[r] * px; l_rep[4 * r + 1] += v_xs[r] * py;
            l_rep[4 * r + 2] += v_xs[r] * E.h; l_rep[4 * r + 3] += v_xs[r];
            t_rep[4 * r + 0] += std::fabs(v_xs[r] * px); t_rep[4 * r + 1] += std::fabs(v_xs[r] * py);
            t_rep[4 * r + 2] += std::fabs(v_xs[r] * E.h); t_rep[4 * r + 3] += std::fabs(v_xs[r]);
          }
          vD += v_zv;             // z_v = D + T_f z_bg
          vT += cfg->z_bg * v_zv;
        }
        vT += -vA;                // A = 1 - T_f
        for (int c = 0; c < 3; ++c) vT += v_albedo[c] * cfg->bg[c];  // albedo = C + T_f bg
        // ---- compositor backward, reverse order ----
        const double A = 1 - S.T, M1 = S.M1, M2 = S.M2, Tf = S.T;
        double Ssum = 0;  // sum_{k>i} w_k phi_k
        // twin: shifted depth frame and centred distortion adjoint (see the header of this function)
        const double z0 = hits.empty() ? 0.0 : hits[0].z;
        const double zm = A > 0 ? M1 / A : 0.0, zvar = A > 0 ? std::max(M2 - M1 * M1 / A, 0.0) : 0.0;
        const double t_vT = std::fabs(vT - vD * z0);   // per-pixel scalars enter the twin by their absolute value
        double t_Ssum = 0;
        for (int64_t h = (int64_t)hits.size() - 1; h >= 0; --h) {
          const Hit& X = hits[h];
          const double* r = rec + R_SIZE * X.id;
          double* g = v_rec + R_SIZE * X.id;
          const double psi = X.z * X.z * A - 2 * X.z * M1 + M2;  // dL/dw_i
          const double phi = v_albedo[0] * r[R_R] + v_albedo[1] * r[R_G] + v_albedo[2] * r[R_B] +
                             vN[0] * r[R_NX] + vN[1] * r[R_NY] + vN[2] * r[R_NZ] + vD * X.z + vL * psi;
          const double v_a = X.T * phi - (Ssum + Tf * vT) / (1 - X.a);
          Ssum += X.w * phi;
          for (int c = 0; c < 3; ++c) { atomic_add(&g[R_R + c], X.w * v_albedo[c]); atomic_add(&g[R_NX + c], X.w * vN[c]); }
          const double v_z = X.w * (vD + 2 * vL * (X.z * A - M1)) + ((int32_t)X.id == S.mi ? vmed : 0.0);
          double v_G = 0;
          if (!X.clamped) { atomic_add(&g[R_ALPHA], X.G * v_a); v_G = r[R_ALPHA] * v_a; }
          const double v_rho = -0.5 * X.G * v_G;
          if (a_rec) {
            double* t = a_rec + R_SIZE * X.id;
            const double dzm = X.z - zm;
            double t_phi = std::fabs(vD * (X.z - z0)) + std::fabs(vL) * (A * dzm * dzm + zvar);
            for (int c = 0; c < 3; ++c) t_phi += std::fabs(v_albedo[c] * r[R_R + c]) + std::fabs(vN[c] * r[R_NX + c]);
            const double t_va = X.T * t_phi + (t_Ssum + Tf * t_vT) / (1 - X.a);
            t_Ssum += X.w * t_phi;
            for (int c = 0; c < 3; ++c) { atomic_add(&t[R_R + c], std::fabs(X.w * v_albedo[c])); atomic_add(&t[R_NX + c], std::fabs(X.w * vN[c])); }
            const double t_vz = X.w * (std::fabs(vD) + 2 * std::fabs(vL) * A * std::fabs(dzm)) + ((int32_t)X.id == S.mi ? std::fabs(vmed) : 0.0);
            double t_vG = 0;
            if (!X.clamped) { atomic_add(&t[R_ALPHA], X.G * t_va); t_vG = r[R_ALPHA] * t_va; }
            const double t_vrho = 0.5 * X.G * t_vG;
            atomic_add(&t[R_ZC], t_vz);
            double t_vd[2];
            if (!X.lowpass) {
              const double tu = 2 * std::fabs(X.u) * t_vrho, tv = 2 * std::fabs(X.v) * t_vrho;
              atomic_add(&t[R_G0], t_vz * std::fabs(X.dx)); atomic_add(&t[R_G1], t_vz * std::fabs(X.dy));
              t_vd[0] = t_vz * std::fabs(r[R_G0]) + std::fabs(r[R_Q00]) * tu + std::fabs(r[R_Q10]) * tv;
              t_vd[1] = t_vz * std::fabs(r[R_G1]) + std::fabs(r[R_Q01]) * tu + std::fabs(r[R_Q11]) * tv;
              atomic_add(&t[R_Q00], tu * std::fabs(X.dx)); atomic_add(&t[R_Q01], tu * std::fabs(X.dy));
              atomic_add(&t[R_Q10], tv * std::fabs(X.dx)); atomic_add(&t[R_Q11], tv * std::fabs(X.dy));
            } else {
              t_vd[0] = 2 * kInvSigma2 * std::fabs(X.dx) * t_vrho;
              t_vd[1] = 2 * kInvSigma2 * std::fabs(X.dy) * t_vrho;
            }
            atomic_add(&t[R_CX], t_vd[0]);
            atomic_add(&t[R_CY], t_vd[1]);
          }
          double v_d[2];
          atomic_add(&g[R_ZC], v_z);
          if (!X.lowpass) {
            const double vu = 2 * X.u * v_rho, vv = 2 * X.v * v_rho;
            atomic_add(&g[R_G0], v_z * X.dx); atomic_add(&g[R_G1], v_z * X.dy);
            v_d[0] = v_z * r[R_G0] + r[R_Q00] * vu + r[R_Q10] * vv;
            v_d[1] = v_z * r[R_G1] + r[R_Q01] * vu + r[R_Q11] * vv;
            atomic_add(&g[R_Q00], vu * X.dx); atomic_add(&g[R_Q01], vu * X.dy);
            atomic_add(&g[R_Q10], vv * X.dx); atomic_add(&g[R_Q11], vv * X.dy);
          } else {
            v_d[0] = 2 * kInvSigma2 * X.dx * v_rho;
            v_d[1] = 2 * kInvSigma2 * X.dy * v_rho;
          }
          atomic_add(&g[R_CX], -v_d[0]);
          atomic_add(&g[R_CY], -v_d[1]);
        }
      }
    }
#pragma omp critical
    {
      if (v_cc) for (int k = 0; k < 12; ++k) v_cc[k] += l_cc[k];
      if (v_ambient) for (int k = 0; k < 3; ++k) v_ambient[k] += l_amb[k];
      if (v_reproj) for (int k = 0; k < 8; ++k) v_reproj[k] += l_rep[k];
      if (a_cc) for (int k = 0; k < 12; ++k) a_cc[k] += t_cc[k];
      if (a_ambient) for (int k = 0; k < 3; ++k) a_ambient[k] += t_amb[k];
      if (a_reproj) for (int k = 0; k < 8; ++k) a_reproj[k] += t_rep[k];
    }
  }
  return 0;
}

// ---------------------------------------------------------------------------------------------------
// E (per-surfel chain): record gradients -> gradients of (p, q, s, logit, rgb) and of dF (Eq. 15).
// All outputs accumulated into (+=).
// ---------------------------------------------------------------------------------------------------
// Twin (tests only; a_rec NULL = off): the absolute sums a_rec of orc_backward pushed through the absolute values of
// the same chain, term by term, into a_means ... a_dF (accumulated into).
int orc_preprocess_backward(const orc_cam_f64* cam, int64_t N, const double* means, const double* quats,
                            const double* scales, const double* logits, const uint8_t* flags,
                            const double* v_rec, double* v_means, double* v_quats, double* v_scales,
                            double* v_logits, double* v_rgb, double* v_dF,
                            const double* a_rec, double* a_means, double* a_quats, double* a_scales,
                            double* a_logits, double* a_rgb, double* a_dF) {
  for (int64_t i = 0; i < N; ++i) {
    if (flags[i] & F_CULLED) continue;
    if (a_rec) {
      const double* p = means + 3 * i;
      const double* q = quats + 4 * i;
      const double* sc = scales + 2 * i;
      const double* t = a_rec + R_SIZE * i;
      SurfelGeom G;
      surfel_geom(cam, p, q, sc, G);
      auto ab = [](double x) { return std::fabs(x); };
      const double alpha = 1.0 / (1.0 + std::exp(-logits[i]));
      a_logits[i] += t[R_ALPHA] * alpha * (1 - alpha);
      for (int c = 0; c < 3; ++c) a_rgb[3 * i + c] += t[R_R + c];
      double t_tu[3] = {0, 0, 0}, t_tv[3] = {0, 0, 0};
      const double t_n[3] = {t[R_NX], t[R_NY], t[R_NZ]};
      const double t_c[2] = {t[R_CX], t[R_CY]};
      double t_B[2][3] = {{0, 0, 0}, {0, 0, 0}};
      if (!(flags[i] & F_DEGENERATE)) {
        double tQ[2][2] = {{t[R_Q00], t[R_Q01]}, {t[R_Q10], t[R_Q11]}};
        const double tg[2] = {t[R_G0], t[R_G1]};
        double t_r[2];
        for (int a = 0; a < 2; ++a) {
          t_r[a] = tg[0] * ab(G.Q[a][0]) + tg[1] * ab(G.Q[a][1]);
          for (int b = 0; b < 2; ++b) tQ[a][b] += ab(G.r[a]) * tg[b];
        }
        double tmp[2][2], tM[2][2];
        for (int a = 0; a < 2; ++a)
          for (int b = 0; b < 2; ++b) tmp[a][b] = ab(G.Q[0][a]) * tQ[0][b] + ab(G.Q[1][a]) * tQ[1][b];
        for (int a = 0; a < 2; ++a)
          for (int b = 0; b < 2; ++b) tM[a][b] = tmp[a][0] * ab(G.Q[b][0]) + tmp[a][1] * ab(G.Q[b][1]);
        a_scales[2 * i] += tM[0][0] * ab(G.au[0]) + tM[1][0] * ab(G.au[1]) + t_r[0] * ab(G.tu[2]);
        a_scales[2 * i + 1] += tM[0][1] * ab(G.av[0]) + tM[1][1] * ab(G.av[1]) + t_r[1] * ab(G.tv[2]);
        const double t_au[2] = {sc[0] * tM[0][0], sc[0] * tM[1][0]};
        const double t_av[2] = {sc[1] * tM[0][1], sc[1] * tM[1][1]};
        for (int c = 0; c < 3; ++c) {
          t_tu[c] += ab(G.B[0][c]) * t_au[0] + ab(G.B[1][c]) * t_au[1];
          t_tv[c] += ab(G.B[0][c]) * t_av[0] + ab(G.B[1][c]) * t_av[1];
          for (int r = 0; r < 2; ++r) t_B[r][c] += t_au[r] * ab(G.tu[c]) + t_av[r] * ab(G.tv[c]);
        }
        t_tu[2] += sc[0] * t_r[0];
        t_tv[2] += sc[1] * t_r[1];
      }
      for (int c = 0; c < 3; ++c) {
        a_means[3 * i + c] += ab(G.B[0][c]) * t_c[0] + ab(G.B[1][c]) * t_c[1];
        for (int r = 0; r < 2; ++r) t_B[r][c] += t_c[r] * ab(p[c]);
      }
      a_means[3 * i + 2] += t[R_ZC];
      for (int r = 0; r < 2; ++r) {
        for (int c = 0; c < 3; ++c) a_dF[4 * r + c] += t_B[r][c];
        a_dF[4 * r + 3] += t_c[r];
      }
      const double Gm[3][3] = {{t_tu[0], t_tv[0], t_n[0]}, {t_tu[1], t_tv[1], t_n[1]}, {t_tu[2], t_tv[2], t_n[2]}};
      const double w = ab(G.w), x = ab(G.x), y = ab(G.y), z = ab(G.z);
      double tq[4];
      tq[0] = 2 * (x * (Gm[2][1] + Gm[1][2]) + y * (Gm[0][2] + Gm[2][0]) + z * (Gm[1][0] + Gm[0][1]));
      tq[1] = 2 * (2 * x * (Gm[1][1] + Gm[2][2]) + y * (Gm[0][1] + Gm[1][0]) + z * (Gm[0][2] + Gm[2][0]) + w * (Gm[2][1] + Gm[1][2]));
      tq[2] = 2 * (x * (Gm[0][1] + Gm[1][0]) + 2 * y * (Gm[0][0] + Gm[2][2]) + z * (Gm[1][2] + Gm[2][1]) + w * (Gm[0][2] + Gm[2][0]));
      tq[3] = 2 * (x * (Gm[0][2] + Gm[2][0]) + y * (Gm[1][2] + Gm[2][1]) + 2 * z * (Gm[0][0] + Gm[1][1]) + w * (Gm[1][0] + Gm[0][1]));
      const double qh[4] = {w, x, y, z};
      const double dotq = qh[0] * tq[0] + qh[1] * tq[1] + qh[2] * tq[2] + qh[3] * tq[3];
      for (int k = 0; k < 4; ++k) a_quats[4 * i + k] += (tq[k] + qh[k] * dotq) / G.qn;
    }
    const double* p = means + 3 * i;
    const double* q = quats + 4 * i;
    const double* s = scales + 2 * i;
    const double* g = v_rec + R_SIZE * i;
    SurfelGeom G;
    surfel_geom(cam, p, q, s, G);
    const double alpha = 1.0 / (1.0 + std::exp(-logits[i]));
    v_logits[i] += g[R_ALPHA] * alpha * (1 - alpha);
    for (int c = 0; c < 3; ++c) v_rgb[3 * i + c] += g[R_R + c];
    // The flip and degenerate decisions are those of the preprocess that produced the records the forward composited
    // (its flags), not a fresh evaluation: in the fp32 record mode
    // a surfel whose normal is within rounding of perpendicular to the viewing direction may be flipped in fp32 and
    // not in double, and the backward must differentiate the function the forward evaluated.
    const bool flipped = flags[i] & F_FLIPPED, degenerate = flags[i] & F_DEGENERATE;
    const double sg = flipped ? -1.0 : 1.0;
    double v_tu[3] = {0, 0, 0}, v_tv[3] = {0, 0, 0};
    const double v_n[3] = {sg * g[R_NX], sg * g[R_NY], sg * g[R_NZ]};
    const double v_c[2] = {g[R_CX], g[R_CY]};
    double v_B[2][3] = {{0, 0, 0}, {0, 0, 0}};
    if (!degenerate) {
      double vQ[2][2] = {{g[R_Q00], g[R_Q01]}, {g[R_Q10], g[R_Q11]}};
      const double vg[2] = {g[R_G0], g[R_G1]};
      // g_j = -sum_i r_i Q_ij
      double v_r[2];
      for (int a = 0; a < 2; ++a) {
        v_r[a] = -(vg[0] * G.Q[a][0] + vg[1] * G.Q[a][1]);
        for (int b = 0; b < 2; ++b) vQ[a][b] += -G.r[a] * vg[b];
      }
      // Q = M^-1  =>  v_M = -Q^T v_Q Q^T
      double tmp[2][2], vM[2][2];
      for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b) tmp[a][b] = G.Q[0][a] * vQ[0][b] + G.Q[1][a] * vQ[1][b];   // Q^T vQ
      for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b) vM[a][b] = -(tmp[a][0] * G.Q[b][0] + tmp[a][1] * G.Q[b][1]);  // (.) Q^T
      // M[:,0] = s_u a_u, M[:,1] = s_v a_v, r_0 = s_u t_u.z, r_1 = s_v t_v.z
      v_scales[2 * i] += vM[0][0] * G.au[0] + vM[1][0] * G.au[1] + v_r[0] * G.tu[2];
      v_scales[2 * i + 1] += vM[0][1] * G.av[0] + vM[1][1] * G.av[1] + v_r[1] * G.tv[2];
      const double v_au[2] = {s[0] * vM[0][0], s[0] * vM[1][0]};
      const double v_av[2] = {s[1] * vM[0][1], s[1] * vM[1][1]};
      for (int c = 0; c < 3; ++c) {
        v_tu[c] += G.B[0][c] * v_au[0] + G.B[1][c] * v_au[1];   // a_u = B t_u
        v_tv[c] += G.B[0][c] * v_av[0] + G.B[1][c] * v_av[1];
        for (int r = 0; r < 2; ++r) v_B[r][c] += v_au[r] * G.tu[c] + v_av[r] * G.tv[c];
      }
      v_tu[2] += s[0] * v_r[0];
      v_tv[2] += s[1] * v_r[1];
    }
    // c = B p + b ; z_c = b_z - p_z
    for (int c = 0; c < 3; ++c) {
      v_means[3 * i + c] += G.B[0][c] * v_c[0] + G.B[1][c] * v_c[1];
      for (int r = 0; r < 2; ++r) v_B[r][c] += v_c[r] * p[c];
    }
    v_means[3 * i + 2] -= g[R_ZC];
    for (int r = 0; r < 2; ++r) {
      for (int c = 0; c < 3; ++c) v_dF[4 * r + c] += v_B[r][c];
      v_dF[4 * r + 3] += v_c[r];
    }
    // rotation -> unit quaternion -> raw quaternion.  R = [t_u | t_v | n], Gm[r][c] = dL/dR[r][c]
    const double Gm[3][3] = {{v_tu[0], v_tv[0], v_n[0]}, {v_tu[1], v_tv[1], v_n[1]}, {v_tu[2], v_tv[2], v_n[2]}};
    const double w = G.w, x = G.x, y = G.y, z = G.z;
    double vq[4];
    vq[0] = 2 * (x * (Gm[2][1] - Gm[1][2]) + y * (Gm[0][2] - Gm[2][0]) + z * (Gm[1][0] - Gm[0][1]));
    vq[1] = 2 * (-2 * x * (Gm[1][1] + Gm[2][2]) + y * (Gm[0][1] + Gm[1][0]) + z * (Gm[0][2] + Gm[2][0]) + w * (Gm[2][1] - Gm[1][2]));
    vq[2] = 2 * (x * (Gm[0][1] + Gm[1][0]) - 2 * y * (Gm[0][0] + Gm[2][2]) + z * (Gm[1][2] + Gm[2][1]) + w * (Gm[0][2] - Gm[2][0]));
    vq[3] = 2 * (x * (Gm[0][2] + Gm[2][0]) + y * (Gm[1][2] + Gm[2][1]) - 2 * z * (Gm[0][0] + Gm[1][1]) + w * (Gm[1][0] - Gm[0][1]));
    const double qh[4] = {w, x, y, z};
    const double dotq = qh[0] * vq[0] + qh[1] * vq[1] + qh[2] * vq[2] + qh[3] * vq[3];
    for (int k = 0; k < 4; ++k) v_quats[4 * i + k] += (vq[k] - qh[k] * dotq) / G.qn;
  }
  return 0;
}

// ---------------------------------------------------------------------------------------------------
// Sun-direction affine camera (Eq. 16, S1-S4) followed by a 2-D viewport, and the view-pixel ->
// sun-pixel reprojection x_s = R_x x + k_h h + k_0 (h = world height of the surface seen at x).
// Fp = F + dF of the view camera (2x4).  viewport = (sx, sy, tx, ty): x_sun_px = s (.) x_sun + t.
// ---------------------------------------------------------------------------------------------------
int orc_sun_camera(const double* Fp, double azimuth, double elevation, const double* viewport,
                   double* F_sun, double* reproj) {
  const double s[3] = {std::cos(azimuth) / std::tan(elevation), std::sin(azimuth) / std::tan(elevation), 1.0};  // Eq. S2
  double Bs[2][3], bs[2];
  for (int r = 0; r < 2; ++r) {
    const double* B = Fp + 4 * r;
    const double Bs3 = B[0] * s[0] + B[1] * s[1] + B[2] * s[2];
    // B (I - [0 0 s]) : columns 0,1 unchanged, column 2 -> B[:,2] - B s      (Eq. 16)
    Bs[r][0] = B[0]; Bs[r][1] = B[1]; Bs[r][2] = B[2] - Bs3;
    bs[r] = B[3];
    const double sc = viewport[r], tr = viewport[2 + r];
    for (int c = 0; c < 3; ++c) Bs[r][c] *= sc;
    bs[r] = bs[r] * sc + tr;
    for (int c = 0; c < 3; ++c) F_sun[4 * r + c] = Bs[r][c];
    F_sun[4 * r + 3] = bs[r];
  }
  // view: x = B2 p_xy + B3 h + b  =>  p_xy = B2^-1 (x - B3 h - b);  sun: x_s = S2 p_xy + S3 h + b_s
  const double B2[2][2] = {{Fp[0], Fp[1]}, {Fp[4], Fp[5]}};
  const double det = B2[0][0] * B2[1][1] - B2[0][1] * B2[1][0];
  if (!(std::fabs(det) > 0)) return -1;
  const double Bi[2][2] = {{B2[1][1] / det, -B2[0][1] / det}, {-B2[1][0] / det, B2[0][0] / det}};
  for (int r = 0; r < 2; ++r) {
    const double Rx0 = Bs[r][0] * Bi[0][0] + Bs[r][1] * Bi[1][0];
    const double Rx1 = Bs[r][0] * Bi[0][1] + Bs[r][1] * Bi[1][1];
    reproj[4 * r + 0] = Rx0;
    reproj[4 * r + 1] = Rx1;
    reproj[4 * r + 2] = Bs[r][2] - (Rx0 * Fp[2] + Rx1 * Fp[6]);
    reproj[4 * r + 3] = bs[r] - (Rx0 * Fp[3] + Rx1 * Fp[7]);
  }
  return 0;
}

// ---------------------------------------------------------------------------------------------------
// Adjoint of orc_sun_camera with respect to Fp = F + dF (cascade camera optimisation, Fig. 1:
// the sun camera is derived from the refined view camera, so the gradients that reach the sun camera's 2x4 matrix
// (sun pass) and the reprojection constants (shadow test) flow back into dF).  Written as the reverse of the steps of
// orc_sun_camera, one by one, without using that the result simplifies.  v_Fp is accumulated into.
// ---------------------------------------------------------------------------------------------------
int orc_sun_camera_backward(const double* Fp, double azimuth, double elevation, const double* viewport,
                            const double* v_F_sun, const double* v_reproj, double* v_Fp) {
  const double s[3] = {std::cos(azimuth) / std::tan(elevation), std::sin(azimuth) / std::tan(elevation), 1.0};
  // ---- forward values that the adjoint needs ----
  double Bs[2][3];
  for (int r = 0; r < 2; ++r) {
    const double* B = Fp + 4 * r;
    const double Bs3 = B[0] * s[0] + B[1] * s[1] + B[2] * s[2];
    Bs[r][0] = viewport[r] * B[0]; Bs[r][1] = viewport[r] * B[1]; Bs[r][2] = viewport[r] * (B[2] - Bs3);
  }
  const double B2[2][2] = {{Fp[0], Fp[1]}, {Fp[4], Fp[5]}};
  const double det = B2[0][0] * B2[1][1] - B2[0][1] * B2[1][0];
  if (!(std::fabs(det) > 0)) return -1;
  const double Bi[2][2] = {{B2[1][1] / det, -B2[0][1] / det}, {-B2[1][0] / det, B2[0][0] / det}};
  double Rx[2][2];
  for (int r = 0; r < 2; ++r) {
    Rx[r][0] = Bs[r][0] * Bi[0][0] + Bs[r][1] * Bi[1][0];
    Rx[r][1] = Bs[r][0] * Bi[0][1] + Bs[r][1] * Bi[1][1];
  }
  // ---- reverse ----
  double vBs[2][3], vbs[2], vBi[2][2] = {{0, 0}, {0, 0}};
  for (int r = 0; r < 2; ++r) {
    const double* vr = v_reproj + 4 * r;
    const double* vf = v_F_sun + 4 * r;
    // reproj[r][2] = Bs[r][2] - (Rx0 Fp[2] + Rx1 Fp[6]);  reproj[r][3] = bs[r] - (Rx0 Fp[3] + Rx1 Fp[7])
    const double vRx0 = vr[0] - vr[2] * Fp[2] - vr[3] * Fp[3];
    const double vRx1 = vr[1] - vr[2] * Fp[6] - vr[3] * Fp[7];
    v_Fp[2] += -vr[2] * Rx[r][0]; v_Fp[6] += -vr[2] * Rx[r][1];
    v_Fp[3] += -vr[3] * Rx[r][0]; v_Fp[7] += -vr[3] * Rx[r][1];
    // Rx0 = Bs0 Bi00 + Bs1 Bi10;  Rx1 = Bs0 Bi01 + Bs1 Bi11
    vBs[r][0] = vf[0] + vRx0 * Bi[0][0] + vRx1 * Bi[0][1];
    vBs[r][1] = vf[1] + vRx0 * Bi[1][0] + vRx1 * Bi[1][1];
    vBs[r][2] = vf[2] + vr[2];
    vbs[r] = vf[3] + vr[3];
    vBi[0][0] += vRx0 * Bs[r][0]; vBi[1][0] += vRx0 * Bs[r][1];
    vBi[0][1] += vRx1 * Bs[r][0]; vBi[1][1] += vRx1 * Bs[r][1];
  }
  // Bi = B2^-1  =>  v_B2 = -Bi^T v_Bi Bi^T
  double tmp[2][2], vB2[2][2];
  for (int a = 0; a < 2; ++a)
    for (int b = 0; b < 2; ++b) tmp[a][b] = Bi[0][a] * vBi[0][b] + Bi[1][a] * vBi[1][b];
  for (int a = 0; a < 2; ++a)
    for (int b = 0; b < 2; ++b) vB2[a][b] = -(tmp[a][0] * Bi[b][0] + tmp[a][1] * Bi[b][1]);
  v_Fp[0] += vB2[0][0]; v_Fp[1] += vB2[0][1]; v_Fp[4] += vB2[1][0]; v_Fp[5] += vB2[1][1];
  // Bs[r] = sc_r (B0, B1, B2 - B.s),  bs[r] = sc_r B3 + tr_r
  for (int r = 0; r < 2; ++r) {
    const double sc = viewport[r];
    const double vBs3 = -sc * vBs[r][2];                 // through the B.s term
    v_Fp[4 * r + 0] += sc * vBs[r][0] + vBs3 * s[0];
    v_Fp[4 * r + 1] += sc * vBs[r][1] + vBs3 * s[1];
    v_Fp[4 * r + 2] += sc * vBs[r][2] + vBs3 * s[2];
    v_Fp[4 * r + 3] += sc * vbs[r];
  }
  return 0;
}

// ---------------------------------------------------------------------------------------------------
// Nearby camera (Fig. 1): "we compute the azimuth and elevation angle of the original camera viewing
// direction d_main.  We then add small random perturbations to the angles to create a new viewing direction.  Then
// apply the same projection matrix transformation as Eq. (16)".  d_main = B_x x B_y is the nullspace of
// B_xy; its angles are taken on the ray pointing up (towards the sensor), in the convention of Eq. S2 (azimuth from +X
// towards +Y, elevation above the horizon), so that a zero perturbation returns the input camera: B u = 0 leaves the
// third column unchanged.  The offset column is kept (as for the sun camera: b_sun = b').  DESIGN.md reading 27.
// angles_out (may be NULL) = (azimuth, elevation) of the main direction.
// ---------------------------------------------------------------------------------------------------
int orc_nearby_camera(const double* Fp, double d_azimuth, double d_elevation, double* F_near, double* angles_out) {
  const double* Bx = Fp;
  const double* By = Fp + 4;
  const double d[3] = {Bx[1] * By[2] - Bx[2] * By[1], Bx[2] * By[0] - Bx[0] * By[2], Bx[0] * By[1] - Bx[1] * By[0]};
  const double dn = std::sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
  if (!(dn > 0)) return -1;
  const double sg = d[2] < 0 ? -1.0 : 1.0;                       // the ray that points up
  const double u[3] = {sg * d[0] / dn, sg * d[1] / dn, sg * d[2] / dn};
  const double az = std::atan2(u[1], u[0]), el = std::asin(u[2]);
  if (angles_out) { angles_out[0] = az; angles_out[1] = el; }
  const double a2 = az + d_azimuth, e2 = el + d_elevation;
  const double s[3] = {std::cos(a2) / std::tan(e2), std::sin(a2) / std::tan(e2), 1.0};   // Eq. S2 for the new direction
  for (int r = 0; r < 2; ++r) {
    const double* B = Fp + 4 * r;
    const double Bs = B[0] * s[0] + B[1] * s[1] + B[2] * s[2];
    F_near[4 * r + 0] = B[0];
    F_near[4 * r + 1] = B[1];
    F_near[4 * r + 2] = B[2] - Bs;                               // Eq. 16: B (I - [0 0 s])
    F_near[4 * r + 3] = B[3];
  }
  return 0;
}

// Adjoint of orc_nearby_camera with respect to Fp (the gradient a nearby-view render sends back into dF through the
// cascade), the reverse of its steps one by one.  v_Fp is accumulated into.
int orc_nearby_camera_backward(const double* Fp, double d_azimuth, double d_elevation, const double* v_F_near, double* v_Fp) {
  const double* Bx = Fp;
  const double* By = Fp + 4;
  const double d[3] = {Bx[1] * By[2] - Bx[2] * By[1], Bx[2] * By[0] - Bx[0] * By[2], Bx[0] * By[1] - Bx[1] * By[0]};
  const double dn = std::sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
  if (!(dn > 0)) return -1;
  const double sg = d[2] < 0 ? -1.0 : 1.0;
  const double u[3] = {sg * d[0] / dn, sg * d[1] / dn, sg * d[2] / dn};
  const double az = std::atan2(u[1], u[0]), el = std::asin(u[2]);
  const double a2 = az + d_azimuth, e2 = el + d_elevation;
  const double ct = 1.0 / std::tan(e2);
  const double s[3] = {std::cos(a2) * ct, std::sin(a2) * ct, 1.0};
  // ---- reverse: F_near[r] = (B0, B1, B2 - B.s, B3) ----
  double vs[3] = {0, 0, 0};
  for (int r = 0; r < 2; ++r) {
    const double* B = Fp + 4 * r;
    const double* vf = v_F_near + 4 * r;
    v_Fp[4 * r + 0] += vf[0] - vf[2] * s[0];
    v_Fp[4 * r + 1] += vf[1] - vf[2] * s[1];
    v_Fp[4 * r + 2] += vf[2] - vf[2] * s[2];
    v_Fp[4 * r + 3] += vf[3];
    for (int k = 0; k < 3; ++k) vs[k] += -vf[2] * B[k];
  }
  // s = (cos a2 ct, sin a2 ct, 1), ct = 1 / tan e2
  const double v_a2 = vs[0] * (-std::sin(a2) * ct) + vs[1] * (std::cos(a2) * ct);
  const double v_ct = vs[0] * std::cos(a2) + vs[1] * std::sin(a2);
  const double v_e2 = -v_ct / (std::sin(e2) * std::sin(e2));
  // az = atan2(u1, u0), el = asin(u2)
  const double h2 = u[0] * u[0] + u[1] * u[1];
  if (!(h2 > 0)) return -2;                                      // exactly nadir: the azimuth is undefined
  double vu[3] = {v_a2 * (-u[1] / h2), v_a2 * (u[0] / h2), v_e2 / std::sqrt(1.0 - u[2] * u[2])};
  // u = sg d / |d|
  const double dot = u[0] * vu[0] + u[1] * vu[1] + u[2] * vu[2];
  double vd[3];
  for (int k = 0; k < 3; ++k) vd[k] = sg * (vu[k] - u[k] * dot) / dn;
  // d = Bx x By  =>  v_Bx = By x v_d,  v_By = v_d x Bx
  v_Fp[0] += By[1] * vd[2] - By[2] * vd[1];
  v_Fp[1] += By[2] * vd[0] - By[0] * vd[2];
  v_Fp[2] += By[0] * vd[1] - By[1] * vd[0];
  v_Fp[4] += vd[1] * Bx[2] - vd[2] * Bx[1];
  v_Fp[5] += vd[2] * Bx[0] - vd[0] * Bx[2];
  v_Fp[6] += vd[0] * Bx[1] - vd[1] * Bx[0];
  return 0;
}

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"

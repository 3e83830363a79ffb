// camera.cu — (f2) the cascade camera chain on the device (Fig. 1 :159).  One tiny kernel builds, for
// the view a device-resident index selects, F' = F + dF (Eq. 15), the sun camera and the reprojection constants (Eq. 16),
// the nearby camera (azimuth / elevation of d_main = B_x x B_y perturbed, then Eq. 16 again) and the
// view's shading constants into a camera block that the *_device calls read through a pointer.  Because nothing of a
// view is baked into kernel arguments any more, ONE captured CUDA graph serves every view and every optimiser step.
// The backward kernel chains the gradients that reach the sun camera, the reprojection constants and the nearby camera
// back into that view's row of dF.
#include "camera_math.cuh"
#include "internal.cuh"

namespace satsplat {

__device__ __forceinline__ void write_camera(float* dst, const float Fp[8], float vx, float vy, float vz, float b_z, float z_bg,
                                             float bg0, float bg1, float bg2) {
  for (int k = 0; k < 8; ++k) dst[k] = Fp[k];
  dst[8] = vx; dst[9] = vy; dst[10] = vz; dst[11] = b_z; dst[12] = z_bg; dst[13] = bg0; dst[14] = bg1; dst[15] = bg2;
}

// main viewing direction of a 2x4 camera: d = B_x x B_y, on the ray that points up; its azimuth / elevation in the
// convention of Eq. S2.  Returns false for a rank-deficient B.
__device__ __forceinline__ bool main_direction(const double Fp[8], double u[3], double& dn, double& sg) {
  const double* Bx = Fp;
  const double* By = Fp + 4;
  const double d[3] = {Bx[1] * By[2] - Bx[2] * By[1], Bx[2] * By[0] - Bx[0] * By[2], Bx[0] * By[1] - Bx[1] * By[0]};
  dn = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
  if (!(dn > 0.0)) return false;
  sg = d[2] < 0.0 ? -1.0 : 1.0;
  for (int k = 0; k < 3; ++k) u[k] = sg * d[k] / dn;
  return true;
}

__global__ void camera_chain_kernel(const satsplat_view_params* __restrict__ views, const float* __restrict__ dF_all,
                                    const int32_t* __restrict__ view_index, float* __restrict__ block) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  const int vi = view_index ? *view_index : 0;
  const satsplat_view_params& V = views[vi];
  float Fp[8];
  double Fpd[8];
  for (int k = 0; k < 8; ++k) {
    Fp[k] = __fadd_rn(V.F[k], dF_all ? dF_all[8 * vi + k] : 0.f);   // Eq. 15 (one fp32 rounding, as the host path)
    Fpd[k] = (double)Fp[k];
  }
  write_camera(block, Fp, V.view_dir[0], V.view_dir[1], V.view_dir[2], V.b_z, V.z_bg, V.bg_rgb[0], V.bg_rgb[1], V.bg_rgb[2]);
  // sun camera + reprojection (Eq. 16): the same source as the host helper, bit for bit
  float F_sun[8], reproj[8];
  if (!sun_camera_math(Fpd, V.sun_s[0], V.sun_s[1], V.sun_viewport, F_sun, reproj)) {
    for (int k = 0; k < 8; ++k) { F_sun[k] = 0.f; reproj[k] = 0.f; }
  }
  write_camera(block + kCamFloats, F_sun, V.sun_view_dir[0], V.sun_view_dir[1], V.sun_view_dir[2], V.b_z, V.z_bg, 0.f, 0.f, 0.f);
  // nearby camera
  float F_near[8];
  float nvx = V.view_dir[0], nvy = V.view_dir[1], nvz = V.view_dir[2];
  for (int k = 0; k < 8; ++k) F_near[k] = Fp[k];
  double u[3], dn, sg;
  if (main_direction(Fpd, u, dn, sg)) {
    const double az = atan2(u[1], u[0]), el = asin(u[2]);
    const double a2 = az + (double)V.nearby_d_azimuth, e2 = el + (double)V.nearby_d_elevation;
    const double ct = 1.0 / tan(e2);
    const double s[3] = {cos(a2) * ct, sin(a2) * ct, 1.0};
    for (int r = 0; r < 2; ++r) {
      const double* B = Fpd + 4 * r;
      F_near[4 * r + 2] = (float)(B[2] - (B[0] * s[0] + B[1] * s[1] + B[2] * s[2]));   // Eq. 16 with the new direction
    }
    nvx = (float)(-cos(a2) * cos(e2)); nvy = (float)(-sin(a2) * cos(e2)); nvz = (float)(-sin(e2));   // sensor -> scene
  }
  write_camera(block + 2 * kCamFloats, F_near, nvx, nvy, nvz, V.b_z, V.z_bg, V.bg_rgb[0], V.bg_rgb[1], V.bg_rgb[2]);
  float* sh = block + kBlockShading;
  for (int k = 0; k < 12; ++k) sh[k] = V.cc[k];
  for (int k = 0; k < 3; ++k) sh[12 + k] = V.ambient[k];
  for (int k = 0; k < 8; ++k) sh[15 + k] = reproj[k];
  sh[23] = V.depth_bias;
  sh[24] = V.slope;
  sh[25] = sh[26] = sh[27] = 0.f;
}

// v_dF_all[view] += v_dF_view + (adjoint of the sun camera and reprojection w.r.t. F') + (adjoint of the nearby camera)
__global__ void camera_chain_backward_kernel(const satsplat_view_params* __restrict__ views, const float* __restrict__ dF_all,
                                             const int32_t* __restrict__ view_index, const float* __restrict__ v_dF_view,
                                             const float* __restrict__ v_F_sun, const float* __restrict__ v_reproj,
                                             const float* __restrict__ v_F_near, float* __restrict__ v_dF_all) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  const int vi = view_index ? *view_index : 0;
  const satsplat_view_params& V = views[vi];
  double Fpd[8], g[8];
  for (int k = 0; k < 8; ++k) {
    Fpd[k] = (double)__fadd_rn(V.F[k], dF_all ? dF_all[8 * vi + k] : 0.f);
    g[k] = v_dF_view ? (double)v_dF_view[k] : 0.0;
  }
  // sun camera: F_sun[r] = sc_r (B0, B1, B2 - B.s, B3) + (0,0,0,tr); reproj = [diag(sc) | -sc (B.s) | t]: only the third
  // column of either depends on F' (closed form of the adjoint, pinned against the step-by-step oracle)
  const double s[3] = {V.sun_s[0], V.sun_s[1], 1.0};
  for (int r = 0; r < 2; ++r) {
    const double sc = (double)V.sun_viewport[r];
    const double vs2 = (v_F_sun ? (double)v_F_sun[4 * r + 2] : 0.0) + (v_reproj ? (double)v_reproj[4 * r + 2] : 0.0);
    for (int c = 0; c < 4; ++c) {
      const double vs = v_F_sun ? (double)v_F_sun[4 * r + c] : 0.0;
      g[4 * r + c] += sc * (vs - (c < 3 ? s[c] : 0.0) * vs2);
    }
  }
  // nearby camera: reverse of the forward steps
  double u[3], dn, sg;
  if (v_F_near && main_direction(Fpd, u, dn, sg)) {
    const double az = atan2(u[1], u[0]), el = asin(u[2]);
    const double a2 = az + (double)V.nearby_d_azimuth, e2 = el + (double)V.nearby_d_elevation;
    const double ct = 1.0 / tan(e2);
    const double sn[3] = {cos(a2) * ct, sin(a2) * ct, 1.0};
    double vs[3] = {0.0, 0.0, 0.0};
    for (int r = 0; r < 2; ++r) {
      const double* B = Fpd + 4 * r;
      const double vf2 = (double)v_F_near[4 * r + 2];
      g[4 * r + 0] += (double)v_F_near[4 * r + 0] - vf2 * sn[0];
      g[4 * r + 1] += (double)v_F_near[4 * r + 1] - vf2 * sn[1];
      g[4 * r + 2] += vf2 - vf2 * sn[2];
      g[4 * r + 3] += (double)v_F_near[4 * r + 3];
      for (int k = 0; k < 3; ++k) vs[k] += -vf2 * B[k];
    }
    const double h2 = u[0] * u[0] + u[1] * u[1];
    if (h2 > 0.0) {   // exactly nadir: the azimuth is undefined, the direction term is dropped
      const double v_a2 = vs[0] * (-sin(a2) * ct) + vs[1] * (cos(a2) * ct);
      const double v_ct = vs[0] * cos(a2) + vs[1] * sin(a2);
      const double v_e2 = -v_ct / (sin(e2) * sin(e2));
      const double vu[3] = {v_a2 * (-u[1] / h2), v_a2 * (u[0] / h2), v_e2 / sqrt(1.0 - u[2] * u[2])};
      const double dot = u[0] * vu[0] + u[1] * vu[1] + u[2] * vu[2];
      double vd[3];
      for (int k = 0; k < 3; ++k) vd[k] = sg * (vu[k] - u[k] * dot) / dn;
      const double* Bx = Fpd;
      const double* By = Fpd + 4;
      g[0] += By[1] * vd[2] - By[2] * vd[1];
      g[1] += By[2] * vd[0] - By[0] * vd[2];
      g[2] += By[0] * vd[1] - By[1] * vd[0];
      g[4] += vd[1] * Bx[2] - vd[2] * Bx[1];
      g[5] += vd[2] * Bx[0] - vd[0] * Bx[2];
      g[6] += vd[0] * Bx[1] - vd[1] * Bx[0];
    }
  }
  for (int k = 0; k < 8; ++k) v_dF_all[8 * vi + k] += (float)g[k];
}

__global__ void advance_index_kernel(int32_t* view_index, int32_t stride, int32_t n_views) {
  if (threadIdx.x == 0 && blockIdx.x == 0) *view_index = (*view_index + stride) % n_views;
}

cudaError_t launch_camera_chain(const satsplat_view_params* views, const float* dF_all, const int32_t* view_index, float* block,
                                cudaStream_t s) {
  ++g_kernel_launches;
  camera_chain_kernel<<<1, 32, 0, s>>>(views, dF_all, view_index, block);
  return cudaGetLastError();
}

cudaError_t launch_camera_chain_backward(const satsplat_view_params* views, const float* dF_all, const int32_t* view_index,
                                         const float* v_dF_view, const float* v_F_sun, const float* v_reproj, const float* v_F_nearby,
                                         float* v_dF_all, cudaStream_t s) {
  ++g_kernel_launches;
  camera_chain_backward_kernel<<<1, 32, 0, s>>>(views, dF_all, view_index, v_dF_view, v_F_sun, v_reproj, v_F_nearby, v_dF_all);
  return cudaGetLastError();
}

cudaError_t launch_advance_index(int32_t* view_index, int32_t stride, int32_t n_views, cudaStream_t s) {
  ++g_kernel_launches;
  advance_index_kernel<<<1, 32, 0, s>>>(view_index, stride, n_views);
  return cudaGetLastError();
}

}  // namespace satsplat

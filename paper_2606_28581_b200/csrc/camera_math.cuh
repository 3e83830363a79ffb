// camera_math.cuh — the Eq. 16 sun camera + reprojection constants as ONE piece of source shared by the host helper
// (satsplat_sun_camera) and the device chain kernel (satsplat_camera_chain), written with singly rounded double
// operations in a fixed order (never contracted: explicit intrinsics on the device, -ffp-contract=off on the host), so
// that the device-built camera is bit-equal to the host-built one.  NOT part of the C ABI; never seen by oracle/.
#pragma once
#include <cuda_runtime.h>

namespace satsplat {

#ifdef __CUDA_ARCH__
#define SS_DMUL(a, b) __dmul_rn((a), (b))
#define SS_DADD(a, b) __dadd_rn((a), (b))
#define SS_DSUB(a, b) __dsub_rn((a), (b))
#define SS_DDIV(a, b) __ddiv_rn((a), (b))
#else
#define SS_DMUL(a, b) ((a) * (b))
#define SS_DADD(a, b) ((a) + (b))
#define SS_DSUB(a, b) ((a) - (b))
#define SS_DDIV(a, b) ((a) / (b))
#endif

// Fp: F' = F + dF (2x4, the fp32 values promoted); s0, s1: (cos phi / tan theta, sin phi / tan theta) of Eq. S2;
// viewport = (scale x, scale y, shift x, shift y).  Outputs: the sun camera's 2x4 and the reprojection 2x4
// [R_x | k_h | k_0] (x_s = R_x x + k_h h + k_0), both rounded to fp32 once.  Returns false if B_xy[:, 0:2] is singular.
__host__ __device__ inline bool sun_camera_math(const double Fp[8], double s0, double s1, const float viewport[4], float F_sun[8],
                                                float reproj[8]) {
  double S[2][4];
  for (int r = 0; r < 2; ++r) {
    const double* B = Fp + 4 * r;
    const double Bs = SS_DADD(SS_DADD(SS_DMUL(B[0], s0), SS_DMUL(B[1], s1)), B[2]);   // B s, s_z = 1
    const double sc = (double)viewport[r], tr = (double)viewport[2 + r];
    S[r][0] = SS_DMUL(sc, B[0]);
    S[r][1] = SS_DMUL(sc, B[1]);
    S[r][2] = SS_DMUL(sc, SS_DSUB(B[2], Bs));                                         // Eq. 16: B (I - [0 0 s])
    S[r][3] = SS_DADD(SS_DMUL(sc, B[3]), tr);
  }
  const double det = SS_DSUB(SS_DMUL(Fp[0], Fp[5]), SS_DMUL(Fp[1], Fp[4]));
  if (!(det > 0.0 || det < 0.0)) return false;
  const double Bi00 = SS_DDIV(Fp[5], det), Bi01 = SS_DDIV(-Fp[1], det), Bi10 = SS_DDIV(-Fp[4], det), Bi11 = SS_DDIV(Fp[0], det);
  for (int r = 0; r < 2; ++r) {
    for (int c = 0; c < 4; ++c) F_sun[4 * r + c] = (float)S[r][c];
    const double Rx0 = SS_DADD(SS_DMUL(S[r][0], Bi00), SS_DMUL(S[r][1], Bi10));
    const double Rx1 = SS_DADD(SS_DMUL(S[r][0], Bi01), SS_DMUL(S[r][1], Bi11));
    reproj[4 * r + 0] = (float)Rx0;
    reproj[4 * r + 1] = (float)Rx1;
    reproj[4 * r + 2] = (float)SS_DSUB(S[r][2], SS_DADD(SS_DMUL(Rx0, Fp[2]), SS_DMUL(Rx1, Fp[6])));
    reproj[4 * r + 3] = (float)SS_DSUB(S[r][3], SS_DADD(SS_DMUL(Rx0, Fp[3]), SS_DMUL(Rx1, Fp[7])));
  }
  return true;
}

}  // namespace satsplat

"""Oracle for the loss stage: image L1 + SSIM, depth distortion, and the normal-consistency
term between the rendered normal and the normal of the depth map (Eq. 13; weights :349), together
with the upstream gradients (v_rgba, v_geom, v_aux) that the rasteriser's backward consumes.

TEST INFRASTRUCTURE ONLY: imported by tests/ and bench.py's cpu_baseline leg; shares no code with
paper_2606_28581_b200/.  Plain numpy, float64, every step written out in the order of the definitions below.

Definitions and readings (DESIGN.md section 2 rows 21-24; the paper gives names, references and weights only):
  L = w_l1 mean|I - I*| + w_ssim (1 - mean SSIM(I, I*)) + w_dist mean(L_dist) + w_normal mean(1 - A_sg N_r . N_d)
  * means over all H W pixels (and the 3 channels for L1 / SSIM);
  * SSIM [Wang et al. 2004] as used by 3DGS: 11x11 Gaussian window, sigma 1.5, zero padding, C1 = 0.01^2, C2 = 0.03^2,
    per channel, on I = out_rgba[..., :3];
  * L_dist = out_aux[..., 1] (the per-pixel distortion the rasteriser composites);
  * normal consistency as in 2DGS [19]: N_r = out_geom[..., :3] (alpha-weighted, un-normalised), A_sg = alpha with
    stop-gradient, N_d from Eq. 13 on the point map p_s backprojected from the depth map z_v = D + (1 - A) z_bg
    (the same background-composited depth the shadow test uses): height h = b_z - z_v,
    p_s = (B2^-1 (x - b - B3 h), h) with F' = [B2 B3 | b]; gradients by central differences
    grad_x p = p(i+1, j) - p(i-1, j), grad_y p = p(i, j+1) - p(i, j-1) on interior pixels, N_d = 0 on the one-pixel border;
    N_d = sgn c / |c|, c = grad_x p x grad_y p, sgn = the sign that makes the flat-ground normal face the sensor
    (one constant per camera).
Pins: tests/test_oracle_pins.py P16 (planar depth -> plane normal, SSIM identities and a brute-force window sum,
finite differences of the total).
PARITY UNPINNED against the paper for the SSIM window / constants, the depth map behind Eq. 13, the border rule and the
2DGS form of the normal term (the paper names them without formulas): this build's stated conventions.
"""
from __future__ import annotations

import numpy as np

C1, C2 = 0.01 ** 2, 0.03 ** 2
WIN, SIGMA = 11, 1.5


def gaussian_window():
    x = np.arange(WIN) - WIN // 2
    g = np.exp(-(x * x) / (2.0 * SIGMA * SIGMA))
    return g / g.sum()


def _blur(img):
    """Separable 11-tap Gaussian, zero padding, over the first two axes of img [H, W, ...]."""
    g = gaussian_window()
    H, W = img.shape[:2]
    r = WIN // 2
    pad = np.zeros((H + 2 * r, W) + img.shape[2:])
    pad[r:r + H] = img
    tmp = sum(g[k] * pad[k:k + H] for k in range(WIN))
    pad = np.zeros((H, W + 2 * r) + img.shape[2:])
    pad[:, r:r + W] = tmp
    return sum(g[k] * pad[:, k:k + W] for k in range(WIN))


def ssim_map_and_grad(I, J):
    """SSIM map of I against the target J (both [H, W, 3]) and d(sum of the map)/dI."""
    mu1, mu2 = _blur(I), _blur(J)
    e11, e22, e12 = _blur(I * I), _blur(J * J), _blur(I * J)
    s11, s22, s12 = e11 - mu1 * mu1, e22 - mu2 * mu2, e12 - mu1 * mu2
    a, b = 2 * mu1 * mu2 + C1, 2 * s12 + C2
    c, d = mu1 * mu1 + mu2 * mu2 + C1, s11 + s22 + C2
    m = (a * b) / (c * d)
    # partials of the map with respect to (mu1, e11, e12) at fixed J, then the adjoint of the three blurs
    dm_dmu1 = (2 * mu2 * b) / (c * d) - m * (2 * mu1) / c          # through a and c
    dm_ds11 = -m / d
    dm_ds12 = 2 * a / (c * d)
    dm_dmu1_tot = dm_dmu1 - 2 * mu1 * dm_ds11 - mu2 * dm_ds12      # s11 = e11 - mu1^2, s12 = e12 - mu1 mu2
    grad = _blur(dm_dmu1_tot) + 2 * I * _blur(dm_ds11) + J * _blur(dm_ds12)   # the window is symmetric: adjoint = blur
    return m, grad


def world_points(zv, Fp, b_z):
    """The point map p_s of Eq. 13: every pixel centre x = (j + .5, i + .5) backprojected to world
    coordinates with its depth: h = b_z - z_v (Eq. 11), p_xy = B2^-1 (x - b - B3 h), p_z = h, F' = [B2 B3 | b]."""
    Fp = np.asarray(Fp, np.float64).reshape(2, 4)
    B2, B3, b = Fp[:, :2], Fp[:, 2], Fp[:, 3]
    Bi = np.linalg.inv(B2)
    H, W = zv.shape
    x = np.stack(np.meshgrid(np.arange(W) + 0.5, np.arange(H) + 0.5), -1)      # [H, W, 2] = (column, row) centres
    h = b_z - zv
    pxy = (x - b - h[..., None] * B3) @ Bi.T
    return np.concatenate([pxy, h[..., None]], -1), Bi, B3


def depth_normals(zv, Fp, view_dir, b_z):
    """Eq. 13 as written: N_d = (grad_x p_s x grad_y p_s) / |.| with central differences of the point map on the
    interior pixels, zero on the one-pixel border; oriented towards the sensor by one sign per camera (the sign that
    makes the normal of a constant-depth map face the sensor).  Returns N_d [H, W, 3], the cross product c, the two
    difference maps, the interior mask and the sign."""
    p, _, _ = world_points(zv, Fp, b_z)
    H, W = zv.shape
    gx, gy = np.zeros((H, W, 3)), np.zeros((H, W, 3))
    gx[1:-1, 1:-1] = p[1:-1, 2:] - p[1:-1, :-2]          # x = column index
    gy[1:-1, 1:-1] = p[2:, 1:-1] - p[:-2, 1:-1]          # y = row index
    c = np.cross(gx, gy)
    flat, _, _ = world_points(np.zeros((3, 3)), Fp, b_z)
    c_flat = np.cross(flat[1, 2] - flat[1, 0], flat[2, 1] - flat[0, 1])
    sgn = -1.0 if float(c_flat @ np.asarray(view_dir, np.float64)) > 0 else 1.0
    interior = np.zeros((H, W), bool)
    interior[1:-1, 1:-1] = True
    cn = np.linalg.norm(c, axis=-1, keepdims=True)
    N = np.where(interior[..., None], sgn * c / np.where(cn > 0, cn, 1.0), 0.0)
    return N, c, gx, gy, interior, sgn


def loss_and_upstream(rgba, geom, aux, target, Fp, view_dir, b_z, z_bg, w_l1=0.8, w_ssim=0.2, w_dist=0.05, w_normal=0.05,
                      alpha_sg=None):
    """Returns (terms dict, v_rgba, v_geom, v_aux) in float64.  `target` is [H, W, 3].  `alpha_sg` (tests only): the
    stop-gradient copy of alpha that weights the normal term, held fixed while rgba is perturbed."""
    rgba, geom, aux, target = (np.asarray(a, np.float64) for a in (rgba, geom, aux, target))
    H, W = rgba.shape[:2]
    npx = float(H * W)
    I, A = rgba[..., :3], rgba[..., 3]
    v_rgba, v_geom, v_aux = np.zeros_like(rgba), np.zeros_like(geom), np.zeros_like(aux)
    # ---- L1 ----
    diff = I - target
    l1 = np.abs(diff).mean()
    v_rgba[..., :3] += w_l1 * np.sign(diff) / (3.0 * npx)
    # ---- SSIM ----
    m, g = ssim_map_and_grad(I, target)
    ssim = m.mean()
    v_rgba[..., :3] += -w_ssim * g / (3.0 * npx)
    # ---- distortion ----
    dist = aux[..., 1].mean()
    v_aux[..., 1] += w_dist / npx
    # ---- normal consistency ----
    D, Nr = geom[..., 3], geom[..., :3]
    zv = D + (1.0 - A) * z_bg
    Nd, c, gx, gy, interior, sgn = depth_normals(zv, Fp, view_dir, b_z)
    Asg = A if alpha_sg is None else np.asarray(alpha_sg, np.float64)
    dot = (Nr * Nd).sum(-1)
    normal = (1.0 - Asg * dot).mean()
    v_geom[..., :3] += -w_normal * Asg[..., None] * Nd / npx
    v_Nd = -w_normal * Asg[..., None] * Nr / npx
    # N = sgn c/|c|  =>  v_c = sgn (v_N - n (n . v_N)) / |c| with n = c/|c|
    cn = np.linalg.norm(c, axis=-1, keepdims=True)
    cn = np.where(interior[..., None], cn, 1.0)
    n = c / cn
    v_c = sgn * (v_Nd - n * (n * v_Nd).sum(-1, keepdims=True)) / cn
    v_c[~interior] = 0.0
    # c = gx x gy  =>  v_gx = gy x v_c,  v_gy = v_c x gx;  the differences scatter to the four neighbours of the point map
    v_gx, v_gy = np.cross(gy, v_c), np.cross(v_c, gx)
    v_p = np.zeros((H, W, 3))
    v_p[1:-1, 2:] += v_gx[1:-1, 1:-1]
    v_p[1:-1, :-2] -= v_gx[1:-1, 1:-1]
    v_p[2:, 1:-1] += v_gy[1:-1, 1:-1]
    v_p[:-2, 1:-1] -= v_gy[1:-1, 1:-1]
    # p_xy = B2^-1 (x - b - B3 h), p_z = h, h = b_z - z_v  =>  d p / d z_v = (B2^-1 B3, -1)
    _, Bi, B3 = world_points(zv, Fp, b_z)
    k = np.array([*(Bi @ B3), -1.0])
    v_zv = v_p @ k
    v_geom[..., 3] += v_zv                                # z_v = D + (1 - A) z_bg
    v_rgba[..., 3] += -z_bg * v_zv
    total = w_l1 * l1 + w_ssim * (1.0 - ssim) + w_dist * dist + w_normal * normal
    return dict(l1=l1, ssim=ssim, distortion=dist, normal=normal, total=total), v_rgba, v_geom, v_aux

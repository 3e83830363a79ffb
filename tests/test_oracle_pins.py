"""Pins for the CPU oracle: closed forms, invariants, an independent derivation, brute force and finite
differences (no GPU).  Each pin is chosen so that a plausible mistake in oracle/satsplat_oracle.cpp (a
dropped term, a wrong sign or index, a transposed operand) fails at least one of them.  None of the
expected values below comes from the oracle or from the CUDA path: they are numpy restatements of the
closed form for the special case, or properties the mathematics fixes.

P1  single camera-facing surfel          -> Gaussian ellipse, opacity, depth, normal (Eq. 8-12, 14)
P1b tilted surfel                        -> foreshortening by cos(beta), depth slope g (Eq. 6, 11)
P2/P7 stacked surfels at one pixel       -> blending order, transmittance, O(n^2) distortion, median
P3  inverse-map round trip               -> Eq. 8-10 and the depth plane
P4  homogeneous two-plane intersection   -> Eq. 9 is its affine special case
P5  sun camera                           -> Eq. 16, S1-S6, hand-evaluated fixtures, reprojection
P6  compositing invariants               -> T monotone in [0,1], A + T = 1, stop rule
P8  central finite differences           -> every gradient of step E incl. dF, CC, L_a, reproj, sun depth
P9  all-pairs == tile lists              -> bbox conservativeness, tile independence
P10 binning                              -> sorted, stable, complete, ranges consistent
P11 shadow test closed form              -> reprojection, bilinear, sigmoid sign, Eq. 1
P12 identity cases of Eq. 1
P13 fp32 contract vs double              -> records agree to fp32 rounding
"""
import math
import os

import numpy as np
import pytest

import satsplat_scenes as S

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def make_view(W, H, F, *, dF=None, view_dir=(0, 0, -1), b_z=100.0, z_bg=120.0, bg=(0, 0, 0), cc=None,
              ambient=(0.3, 0.35, 0.45)):
    cc = np.concatenate([np.eye(3), np.zeros((3, 1))], 1).reshape(12) if cc is None else cc
    return S.View(width=W, height=H, F=np.asarray(F, np.float32).reshape(8),
                  dF=np.zeros(8, np.float32) if dF is None else np.asarray(dF, np.float32),
                  view_dir=np.asarray(view_dir, np.float32), b_z=b_z, z_bg=z_bg,
                  bg_rgb=np.asarray(bg, np.float32), cc=np.asarray(cc, np.float32),
                  ambient=np.asarray(ambient, np.float32))


def nadir_F(gsd, W, H):
    return np.array([[1 / gsd, 0, 0, W / 2], [0, -1 / gsd, 0, H / 2]], np.float64)


def pixel_grid(W, H):
    px, py = np.meshgrid(np.arange(W) + 0.5, np.arange(H) + 0.5)
    return px, py


def render64(orc, view, means, quats, scales, logits, rgb, *, shading=None, options=0, bg=None):
    """all-pairs, everything in double from the raw inputs (record mode `double`)."""
    pre = orc.preprocess_f64(view, means, quats, scales, logits, rgb)
    order = np.argsort(-np.asarray(means, np.float64)[:, 2], kind="stable").astype(np.uint32)  # depth = b_z - z
    shading = shading or orc.Shading(cc=view.cc, ambient=view.ambient)
    out = orc.forward(view.width, view.height, view.b_z, view.z_bg, view.bg_rgb if bg is None else bg, pre["rec"],
                      pre["flags"], order, shading, options=options)
    return pre, order, out


# ------------------------------------------------------------------------------------------------ P1
def test_p1_single_camera_facing_surfel(orc):
    W = H = 48
    gsd = 0.5
    view = make_view(W, H, nadir_F(gsd, W, H))
    p = np.array([[0.7, -0.4, 12.0]])     # world; projects to (W/2 + 1.4, H/2 + 0.8)
    su, sv, logit = 1.5, 0.8, 0.3
    rgbv = np.array([[0.2, 0.5, 0.9]])
    pre, _, out = render64(orc, view, p, np.array([[1.0, 0, 0, 0]]), np.array([[su, sv]]), np.array([logit]), rgbv)
    px, py = pixel_grid(W, H)
    cx, cy = W / 2 + p[0, 0] / gsd, H / 2 - p[0, 1] / gsd
    dxw, dyw = (px - cx) * gsd, (py - cy) * gsd          # world offsets
    rho = (dxw / su) ** 2 + (dyw / sv) ** 2               # scales >= 1 px: the low-pass term never wins
    alpha = 1 / (1 + math.exp(-logit))
    A = np.minimum(0.99, alpha * np.exp(-0.5 * rho))
    A[(rho > 9) | (A < 1 / 255)] = 0
    zc = view.b_z - p[0, 2]
    np.testing.assert_allclose(out["rgba"][..., 3], A, atol=1e-13)
    for c in range(3):
        np.testing.assert_allclose(out["rgba"][..., c], A * rgbv[0, c], atol=1e-13)   # identity CC, bg 0
    np.testing.assert_allclose(out["geom"][..., 3], A * zc, atol=1e-11)
    np.testing.assert_allclose(out["geom"][..., 2], A * 1.0, atol=1e-13)              # n = +z faces the sensor
    np.testing.assert_allclose(out["geom"][..., :2], 0, atol=1e-13)
    np.testing.assert_allclose(out["aux"][..., 1], 0, atol=1e-9)                      # one surfel: no distortion
    np.testing.assert_allclose(out["aux"][..., 3], 1 - A, atol=1e-13)
    med = np.where(A > 0, zc, view.z_bg)
    np.testing.assert_allclose(out["aux"][..., 0], med, atol=1e-11)
    assert A.max() > 0.5 and (A > 0).sum() > 50


def test_p1b_tilted_surfel(orc):
    W = H = 64
    gsd = 0.5
    view = make_view(W, H, nadir_F(gsd, W, H))
    beta = math.radians(35.0)
    q = np.array([[math.cos(beta / 2), math.sin(beta / 2), 0, 0]])   # rotation about the u (= world x) axis
    p = np.array([[0.0, 0.0, 5.0]])
    su, sv = 2.0, 3.0
    pre, _, out = render64(orc, view, p, q, np.array([[su, sv]]), np.array([4.0]), np.array([[1.0, 1.0, 1.0]]))
    px, py = pixel_grid(W, H)
    dxw, dyw = (px - W / 2) * gsd, -(py - H / 2) * gsd   # image y is down
    u, v = dxw / su, dyw / (sv * math.cos(beta))         # v-extent on screen is foreshortened by cos(beta)
    rho = u * u + v * v
    alpha = 1 / (1 + math.exp(-4.0))
    A = np.minimum(0.99, alpha * np.exp(-0.5 * rho))
    keep = (rho <= 9) & (A >= 1 / 255)
    A = np.where(keep, A, 0)
    z = (view.b_z - p[0, 2]) - sv * math.sin(beta) * v   # P_z = p_z + s_v sin(beta) v  (Eq. 3, 6, 11)
    np.testing.assert_allclose(out["rgba"][..., 3], A, atol=1e-12)
    np.testing.assert_allclose(out["geom"][..., 3], A * z, atol=1e-10)
    n = np.array([0, -math.sin(beta), math.cos(beta)])
    for c in range(3):
        np.testing.assert_allclose(out["geom"][..., c], A * n[c], atol=1e-12)


def test_p1c_lowpass_wins_for_subpixel_and_edge_on(orc):
    """Eq. 12: a surfel much smaller than a pixel, or seen edge-on, renders as the sigma = 1/sqrt(2) px disc."""
    W = H = 16
    gsd = 1.0
    view = make_view(W, H, nadir_F(gsd, W, H))
    px, py = pixel_grid(W, H)
    d2 = (px - (W / 2 + 0.25)) ** 2 + (py - (H / 2 - 0.5)) ** 2
    alpha = 1 / (1 + math.exp(-1.0))
    A_disc = np.minimum(0.99, alpha * np.exp(-0.5 * 2.0 * d2))
    A_disc[(2 * d2 > 9) | (A_disc < 1 / 255)] = 0
    zc = view.b_z - 3.0
    # (a) tiny surfel: G(u) < G_lowpass everywhere except within ~the surfel itself (no pixel centre there)
    pre, _, out = render64(orc, view, np.array([[0.25, 0.5, 3.0]]), np.array([[1.0, 0, 0, 0]]),
                           np.array([[0.01, 0.01]]), np.array([1.0]), np.ones((1, 3)))
    np.testing.assert_allclose(out["rgba"][..., 3], A_disc, atol=1e-12)
    np.testing.assert_allclose(out["geom"][..., 3], A_disc * zc, atol=1e-10)   # low-pass branch uses z_c
    # (b) exactly edge-on surfel (normal horizontal): det = 0 -> degenerate flag, same disc
    q = np.array([[math.cos(math.pi / 4), math.sin(math.pi / 4), 0, 0]])       # 90 deg about x
    pre, _, out = render64(orc, view, np.array([[0.25, 0.5, 3.0]]), q, np.array([[0.01, 5.0]]), np.array([1.0]),
                           np.ones((1, 3)))
    assert pre["flags"][0] & orc.F_DEGENERATE
    np.testing.assert_allclose(out["rgba"][..., 3], A_disc, atol=1e-12)


# ------------------------------------------------------------------------------------------- P2 / P7
def test_p2_p7_stacked_surfels_blend_order_distortion_median(orc):
    rng = np.random.default_rng(5)
    W = H = 1
    view = make_view(W, H, nadir_F(1.0, W, H), z_bg=200.0, bg=(0.1, 0.2, 0.3))
    n = 9
    heights = rng.uniform(0, 30, n)
    means = np.stack([np.zeros(n), np.zeros(n), heights], 1)       # all centred on the single pixel centre
    logits = rng.normal(0.0, 1.5, n)
    logits[3] = 8.0                                                # one clamps at 0.99
    rgb = rng.uniform(0, 1, (n, 3))
    quats = np.tile([1.0, 0, 0, 0], (n, 1))
    pre, order, out = render64(orc, view, means, quats, np.full((n, 2), 4.0), logits, rgb)
    # by hand: front to back = decreasing height; G = 1 at the centre
    idx = np.argsort(-heights, kind="stable")
    T, C, D, Ls = 1.0, np.zeros(3), 0.0, 0.0
    ws, zs, med = [], [], view.z_bg
    for i in idx:
        a = min(0.99, 1 / (1 + math.exp(-logits[i])))
        z = view.b_z - heights[i]
        if T * (1 - a) < 1e-4:
            break
        if T > 0.5:
            med = z
        w = a * T
        ws.append(w); zs.append(z)
        C += w * rgb[i]; D += w * z
        T *= 1 - a
    ws, zs = np.array(ws), np.array(zs)
    for i in range(len(ws)):
        for j in range(i):
            Ls += ws[i] * ws[j] * (zs[i] - zs[j]) ** 2             # O(n^2) definition (Mip-NeRF-360 form)
    C = C + T * np.asarray(view.bg_rgb, np.float64)
    np.testing.assert_allclose(out["rgba"][0, 0, :3], C, rtol=1e-12)
    np.testing.assert_allclose(out["rgba"][0, 0, 3], 1 - T, rtol=1e-12)
    np.testing.assert_allclose(out["geom"][0, 0, 3], D, rtol=1e-12)
    np.testing.assert_allclose(out["aux"][0, 0, 1], Ls, rtol=1e-9)
    np.testing.assert_allclose(out["aux"][0, 0, 0], med, rtol=1e-12)
    np.testing.assert_allclose(out["aux"][0, 0, 3], T, rtol=1e-12)
    assert len(ws) >= 4


# ------------------------------------------------------------------------------------------------ P3
def test_p3_inverse_map_round_trip(orc):
    rng = np.random.default_rng(11)
    n = 200
    F, d = S.affine_camera(0.4, math.radians(22), 1.1, 256, 256, (10, -5, 0))
    dF = (rng.normal(0, 1e-3, 8)).astype(np.float32)
    view = make_view(256, 256, F, dF=dF, view_dir=d)
    means = rng.uniform(-30, 30, (n, 3))
    quats = rng.normal(0, 1, (n, 4)) * rng.uniform(0.3, 3, (n, 1))    # deliberately not unit
    scales = rng.uniform(0.2, 2, (n, 2))
    pre = orc.preprocess_f64(view, means, quats, scales, np.zeros(n), np.zeros((n, 3)))
    rec = pre["rec"]
    Fp = (view.F.astype(np.float64) + view.dF.astype(np.float64)).reshape(2, 4)
    qh = quats / np.linalg.norm(quats, axis=1, keepdims=True)
    w, x, y, z = qh.T
    # textbook rotation matrix of a unit quaternion, column by column
    R = np.stack([np.stack([1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)], 1),
                  np.stack([2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)], 1),
                  np.stack([2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)], 1)], 1)  # [n,3,3]
    np.testing.assert_allclose(np.einsum("nij,nkj->nik", R, R), np.tile(np.eye(3), (n, 1, 1)), atol=1e-12)
    uv = rng.uniform(-3, 3, (n, 2))
    P = means + scales[:, :1] * R[:, :, 0] * uv[:, :1] + scales[:, 1:] * R[:, :, 1] * uv[:, 1:]   # Eq. 3
    xpix = P @ Fp[:, :3].T + Fp[:, 3]                                                               # Eq. 6
    dd = xpix - rec[:, 0:2]
    u = rec[:, 2] * dd[:, 0] + rec[:, 3] * dd[:, 1]
    v = rec[:, 4] * dd[:, 0] + rec[:, 5] * dd[:, 1]
    np.testing.assert_allclose(np.stack([u, v], 1), uv, atol=1e-9)
    zz = rec[:, 6] + rec[:, 7] * dd[:, 0] + rec[:, 8] * dd[:, 1]
    np.testing.assert_allclose(zz, view.b_z - P[:, 2], atol=1e-9)                                   # Eq. 11
    np.testing.assert_allclose(rec[:, 0:2], means @ Fp[:, :3].T + Fp[:, 3], atol=1e-10)
    # stored normal: last column of R, flipped to face the sensor
    nrm = R[:, :, 2]
    flip = (nrm @ view.view_dir.astype(np.float64)) > 0
    np.testing.assert_allclose(rec[:, 13:16], np.where(flip[:, None], -nrm, nrm), atol=1e-12)
    assert ((pre["flags"] & orc.F_FLIPPED) > 0).tolist() == flip.tolist()


# ------------------------------------------------------------------------------------------------ P4
def test_p4_two_plane_intersection_reduces_to_affine_inverse(orc):
    """2DGS finds (u,v) by intersecting the two pixel planes transformed by (WH)^T.  With an
    affine W (last row 0 0 0 1) the same construction must give Q x + q of Eq. 9."""
    rng = np.random.default_rng(12)
    n = 50
    F, d = S.affine_camera(0.5, math.radians(30), 2.5, 128, 128, (0, 0, 0))
    view = make_view(128, 128, F, view_dir=d)
    means = rng.uniform(-20, 20, (n, 3))
    quats = rng.normal(0, 1, (n, 4))
    scales = rng.uniform(0.3, 2, (n, 2))
    rec = orc.preprocess_f64(view, means, quats, scales, np.zeros(n), np.zeros((n, 3)))["rec"]
    Fp = view.F.astype(np.float64).reshape(2, 4)
    Wm = np.zeros((4, 4)); Wm[:2] = Fp; Wm[2] = [0, 0, -1, view.b_z]; Wm[3] = [0, 0, 0, 1]   # Eq. 7 + Eq. 11
    qh = quats / np.linalg.norm(quats, axis=1, keepdims=True)
    for i in range(n):
        w, x, y, z = qh[i]
        tu = np.array([1 - 2 * (y * y + z * z), 2 * (x * y + w * z), 2 * (x * z - w * y)])
        tv = np.array([2 * (x * y - w * z), 1 - 2 * (x * x + z * z), 2 * (y * z + w * x)])
        Hm = np.zeros((4, 4)); Hm[:3, 0] = scales[i, 0] * tu; Hm[:3, 1] = scales[i, 1] * tv
        Hm[:3, 3] = means[i]; Hm[3, 3] = 1                                                     # Eq. 4
        WH = Wm @ Hm
        xp = rec[i, 0:2] + rng.uniform(-20, 20, 2)
        hx, hy = np.array([-1, 0, 0, xp[0]]), np.array([0, -1, 0, xp[1]])
        hu, hv = WH.T @ hx, WH.T @ hy
        den = hu[0] * hv[1] - hu[1] * hv[0]
        u = (hu[1] * hv[3] - hu[3] * hv[1]) / den
        v = (hu[3] * hv[0] - hu[0] * hv[3]) / den
        dd = xp - rec[i, 0:2]
        np.testing.assert_allclose([rec[i, 2] * dd[0] + rec[i, 3] * dd[1], rec[i, 4] * dd[0] + rec[i, 5] * dd[1]],
                                   [u, v], atol=1e-8)


# ------------------------------------------------------------------------------------------------ P5
def test_p5_sun_camera_fixtures_and_nullspace(orc):
    rows = [l for l in open(os.path.join(GOLDEN, "sun_camera_cases.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 4
    for l in rows:
        v = [float(t) for t in l.split()]
        phi, th = math.radians(v[0]), math.radians(v[1])
        B = np.array(v[2:8]).reshape(2, 3)
        Fp = np.concatenate([B, [[3.0], [-7.0]]], 1).reshape(8)
        F_sun, reproj = orc.sun_camera(Fp, phi, th, [1, 1, 0, 0])
        np.testing.assert_allclose(F_sun.reshape(2, 4)[:, :3], np.array(v[8:14]).reshape(2, 3), atol=1e-12)
        np.testing.assert_allclose(F_sun.reshape(2, 4)[:, 3], [3.0, -7.0], atol=1e-12)
    rng = np.random.default_rng(3)
    for _ in range(20):
        F, d = S.affine_camera(rng.uniform(0.3, 0.6), math.radians(rng.uniform(0, 35)), rng.uniform(0, 6.28), 512, 512,
                               (50, 60, 0))
        Fp = F.astype(np.float64)
        B = Fp.reshape(2, 4)[:, :3]
        # l.165: the viewing direction B_x x B_y spans the nullspace of B_xy
        np.testing.assert_allclose(B @ np.cross(B[0], B[1]), 0, atol=1e-9)
        phi, th = rng.uniform(0, 2 * math.pi), math.radians(rng.uniform(20, 80))
        s = np.array([math.cos(phi) / math.tan(th), math.sin(phi) / math.tan(th), 1.0])
        vp = np.array([rng.uniform(0.5, 2), rng.uniform(0.5, 2), rng.uniform(-50, 50), rng.uniform(-50, 50)])
        F_sun, reproj = orc.sun_camera(Fp, phi, th, vp)
        Fs = F_sun.reshape(2, 4)
        np.testing.assert_allclose(Fs[:, :3] @ s, 0, atol=1e-9)                                  # Eq. S6
        p = rng.uniform(-40, 40, 3)
        t = rng.uniform(-30, 30)
        np.testing.assert_allclose(Fs[:, :3] @ p + Fs[:, 3], Fs[:, :3] @ (p + t * s) + Fs[:, 3], atol=1e-8)
        # shadow of a point at height h falls on the ground at p_xy - h (cos phi, sin phi)/tan theta
        g = np.array([p[0] - p[2] * s[0], p[1] - p[2] * s[1], 0.0])
        np.testing.assert_allclose(Fs[:, :3] @ p, Fs[:, :3] @ g, atol=1e-8)
        # reprojection: view pixel x of a world point at height h  ->  its sun pixel
        xv = B @ p + Fp.reshape(2, 4)[:, 3]
        xs = Fs[:, :3] @ p + Fs[:, 3]
        R = reproj.reshape(2, 4)
        np.testing.assert_allclose(R[:, :2] @ xv + R[:, 2] * p[2] + R[:, 3], xs, atol=1e-7)
    # unscaled Eq. 16 camera: R_x = I, k_h = -B s, k_0 = 0
    F_sun, reproj = orc.sun_camera(Fp, phi, th, [1, 1, 0, 0])
    R = reproj.reshape(2, 4)
    np.testing.assert_allclose(R[:, :2], np.eye(2), atol=1e-12)
    np.testing.assert_allclose(R[:, 2], -(B @ s), atol=1e-10)
    np.testing.assert_allclose(R[:, 3], 0, atol=1e-9)


# ------------------------------------------------------------------------------------- P6 / P9 / P10
@pytest.fixture(scope="module")
def c0(orc):
    scene = S.make_config(0)
    view = scene.views[0]
    tile = orc.render_pass(view, scene, tile_mode=True)
    sh = orc.Shading(cc=view.cc, ambient=view.ambient)
    f_tile = orc.forward(view.width, view.height, view.b_z, view.z_bg, view.bg_rgb, tile["rec64"], tile["flags"],
                         tile["lists"], sh, threads=orc.num_threads())
    order = orc.global_order(tile["depth_key"], tile["flags"])
    f_all = orc.forward(view.width, view.height, view.b_z, view.z_bg, view.bg_rgb, tile["rec64"], tile["flags"],
                        order, sh, threads=orc.num_threads())
    return scene, view, tile, f_tile, f_all, order


def test_p6_compositing_invariants(c0):
    scene, view, tile, f, _, _ = c0
    T, A = f["aux"][..., 3], f["rgba"][..., 3]
    assert (T >= 1e-4).all() and (T <= 1).all()
    np.testing.assert_allclose(A + T, 1, atol=1e-15)
    assert (np.linalg.norm(f["geom"][..., :3], axis=-1) <= A * (1 + 1e-6) + 1e-12).all()     # |sum w n| <= sum w (fp32 normals are unit to ~1e-7)
    zmin, zmax = view.b_z - scene.means[:, 2].max() - 5, view.b_z - scene.means[:, 2].min() + 5
    has = A > 1e-3
    dmean = f["geom"][..., 3][has] / A[has]
    assert (dmean > zmin).all() and (dmean < zmax).all()
    assert (f["aux"][..., 1] >= -1e-12).all()                                   # distortion is a sum of squares
    assert (f["rgba"][..., :3] >= 0).all() and (f["rgba"][..., :3] <= 1 + 1e-12).all()
    assert f["counters"][1] > view.width * view.height


def test_p9_all_pairs_equals_tile_lists(c0):
    scene, view, tile, f_tile, f_all, _ = c0
    for k in ("rgba", "geom", "aux", "albedo", "med_idx"):
        assert np.array_equal(f_tile[k], f_all[k]), k
    assert f_all["counters"][1] == f_tile["counters"][1]
    assert f_all["counters"][0] > f_tile["counters"][0]


def test_p10_binning_sorted_stable_complete(c0, orc):
    scene, view, tile, *_ = c0
    keys, vals, ranges = tile["keys"], tile["vals"], tile["ranges"]
    rect, count, dk = tile["rect"], tile["count"], tile["depth_key"]
    TX = (view.width + 15) // 16
    assert np.all(keys[1:] >= keys[:-1])
    same = keys[1:] == keys[:-1]
    assert np.all(vals[1:][same] > vals[:-1][same])                      # ties broken by ascending surfel index
    # completeness: the multiset of (tile, surfel) pairs equals the rect expansion, done independently here
    pairs = set()
    for i in range(scene.n):
        if count[i]:
            for ty in range(rect[i, 1], rect[i, 3]):
                for tx in range(rect[i, 0], rect[i, 2]):
                    pairs.add((ty * TX + tx, i))
    got = list(zip((keys >> np.uint64(32)).astype(np.int64).tolist(), vals.tolist()))
    assert len(got) == len(pairs) == int(count.sum()) and set(got) == pairs
    assert np.array_equal((keys & np.uint64(0xFFFFFFFF)).astype(np.uint32), dk[vals])
    # depth key is order preserving
    zc = tile["rec"][:, 6]
    o = np.argsort(dk, kind="stable")
    assert np.all(np.diff(zc[o]) >= 0)
    # ranges
    tiles = (keys >> np.uint64(32)).astype(np.int64)
    for t in range(ranges.shape[0]):
        s, e = ranges[t]
        if e > s:
            assert np.all(tiles[s:e] == t) and (s == 0 or tiles[s - 1] < t) and (e == len(tiles) or tiles[e] > t)
        else:
            assert not np.any(tiles == t) and s == 0 and e == 0
    # rect really is the 3-sigma box, in tiles, clamped (spot-check against a direct float64 evaluation)
    rec = tile["rec"].astype(np.float64)
    M = np.linalg.inv(rec[:, 2:6].reshape(-1, 2, 2) + np.eye(2) * 1e-300)
    ok = (tile["flags"] & (orc.F_DEGENERATE | orc.F_CULLED)) == 0
    ext = np.maximum(3 * np.sqrt((M ** 2).sum(-1)), 3 / math.sqrt(2))
    lo = np.floor((rec[:, 0:2] - ext) / 16).astype(int)
    hi = np.floor((rec[:, 0:2] + ext) / 16).astype(int) + 1
    TY = (view.height + 15) // 16
    lo = np.clip(lo, 0, [TX, TY]); hi = np.clip(hi, 0, [TX, TY])
    mism = ((lo[:, 0] != rect[:, 0]) | (lo[:, 1] != rect[:, 1]) | (hi[:, 0] != rect[:, 2]) | (hi[:, 1] != rect[:, 3])) & ok
    assert mism.sum() <= 2          # float64 vs the fp32 contract may differ on a knife edge only


def test_p13_fp32_contract_matches_double(c0, orc):
    scene, view, tile, *_ = c0
    d = orc.preprocess_f64(view, scene.means, scene.quats, scene.scales, scene.opacity_logits, scene.rgb)
    ok = (tile["flags"] & orc.F_DEGENERATE) == 0
    assert np.array_equal(tile["flags"] & orc.F_DEGENERATE, d["flags"] & orc.F_DEGENERATE)
    a, b = tile["rec"][ok].astype(np.float64), d["rec"][ok]
    scale = np.abs(b).max(0) + 1e-6
    assert (np.abs(a - b) / scale).max() < 5e-5
    assert np.abs(a[:, :2] - b[:, :2]).max() < 1e-4     # centres to ~fp32 ulp at 128 px


# ------------------------------------------------------------------------------------------------ P8
def _fd_problem(orc, shadows, options, seed=21):
    rng = np.random.default_rng(seed)
    n, W, H = 14, 16, 16
    F, d = S.affine_camera(0.5, math.radians(20), 0.7, W, H, (4, 4, 0))
    means = np.concatenate([rng.uniform(0.5, 7.5, (n, 2)), rng.normal(0, 1.0, (n, 1))], 1)
    nrm = np.array([0, 0, 1.0]) + 0.5 * rng.normal(0, 1, (n, 3))
    quats = rng.normal(0, 1, (n, 4))
    quats[:, 0] += 3.0          # mostly upward-facing, generic otherwise
    quats *= rng.uniform(0.5, 2.0, (n, 1))
    del nrm
    P = dict(means=means, quats=quats, scales=rng.uniform(0.6, 2.0, (n, 2)), logits=rng.normal(0.5, 1, n),
             rgb=rng.uniform(0, 1, (n, 3)), dF=rng.normal(0, 1e-2, 8),
             cc=(np.concatenate([np.eye(3), np.zeros((3, 1))], 1) + rng.normal(0, 0.1, (3, 4))).reshape(12),
             ambient=rng.uniform(0.2, 0.5, 3))
    if shadows:
        P["reproj"] = np.array([0.9, 0.05, 0.3, 1.0, -0.04, 0.95, -0.2, 0.5]) + rng.normal(0, 0.01, 8)
        P["sun_depth"] = 10 + rng.normal(0, 1.0, (20, 20))
    view = make_view(W, H, F, view_dir=d, b_z=12.0, z_bg=16.0, bg=(0.2, 0.1, 0.3))
    up = [rng.normal(0, 1, (H, W, 4)) for _ in range(3)]
    up[2][..., 2:] = 0
    order = np.argsort(-means[:, 2], kind="stable").astype(np.uint32)

    def run(Pv, need_grad=False):
        sh = orc.Shading(cc=Pv["cc"], ambient=Pv["ambient"], sun_depth=Pv.get("sun_depth"), reproj=Pv.get("reproj"),
                         bias=0.5, slope=4.0)
        pre = orc.preprocess_f64(view, Pv["means"], Pv["quats"], Pv["scales"], Pv["logits"], Pv["rgb"],
                                 F=view.F.astype(np.float64), dF=Pv["dF"])
        out = orc.forward(W, H, view.b_z, view.z_bg, view.bg_rgb, pre["rec"], pre["flags"], order, sh, options=options)
        loss = (out["rgba"] * up[0]).sum() + (out["geom"] * up[1]).sum() + (out["aux"] * up[2]).sum()
        if not need_grad:
            return loss, out
        bw = orc.backward(W, H, view.b_z, view.z_bg, view.bg_rgb, pre["rec"], pre["flags"], order, sh, *up, options=options)
        g = orc.preprocess_backward(view, Pv["means"], Pv["quats"], Pv["scales"], Pv["logits"], pre["flags"],
                                    bw["v_rec"], F=view.F.astype(np.float64), dF=Pv["dF"])
        grads = dict(means=g["v_means"], quats=g["v_quats"], scales=g["v_scales"], logits=g["v_logits"], rgb=g["v_rgb"],
                     dF=g["v_dF"], cc=bw["v_cc"], ambient=bw["v_ambient"])
        if shadows:
            grads.update(reproj=bw["v_reproj"], sun_depth=bw["v_sun_depth"])
        return loss, out, grads

    return P, run


def _check_fd(P, run, names, h=1e-6, rtol=1e-6):
    _, out, grads = run(P, need_grad=True)
    rng = np.random.default_rng(0)
    worst = 0.0
    for name in names:
        base = np.asarray(P[name], np.float64)
        flat_idx = np.arange(base.size)
        if base.size > 60:
            flat_idx = rng.choice(base.size, 60, replace=False)
        g = np.asarray(grads[name]).reshape(-1)
        gscale = max(np.abs(g).max(), 1e-3)
        for k in flat_idx:
            Pp, Pm = dict(P), dict(P)
            e = np.zeros(base.size); e[k] = h * max(1.0, abs(base.reshape(-1)[k]))
            Pp[name] = (base.reshape(-1) + e).reshape(base.shape)
            Pm[name] = (base.reshape(-1) - e).reshape(base.shape)
            fd = (run(Pp)[0] - run(Pm)[0]) / (2 * e[k])
            err = abs(fd - g[k]) / gscale
            worst = max(worst, err)
            assert err < rtol, (name, int(k), fd, g[k])
    return out, worst


def test_p8_finite_differences_no_cutoffs(orc):
    """Cut-offs off (smooth objective): every parameter group, shadows off."""
    P, run = _fd_problem(orc, shadows=False, options=7)
    out, _ = _check_fd(P, run, ["means", "quats", "scales", "logits", "rgb", "dF", "cc", "ambient"])
    assert out["counters"][1] > 200


def test_p8_finite_differences_shadows(orc):
    """Shadows on with an arbitrary sun map: adds reproj, sun depth, ambient through V."""
    P, run = _fd_problem(orc, shadows=True, options=7)
    # bilinear sampling is piecewise smooth: keep the sample points away from texel borders for the FD step
    out, _ = _check_fd(P, run, ["means", "quats", "scales", "logits", "rgb", "dF", "cc", "ambient", "reproj", "sun_depth"])
    V = out["aux"][..., 2]
    assert V.min() < 0.4 and V.max() > 0.8          # the shadow test is exercised on both sides


def test_p8_finite_differences_with_cutoffs(orc):
    """Cut-offs on: gradients still match away from the decision boundaries (margins asserted)."""
    P, run = _fd_problem(orc, shadows=False, options=0, seed=33)
    _, out = run(P)
    m = out["margins"]
    # distance of every pixel from the rho cut, the alpha skip and the median switch; step 1e-7 moves rho by <1e-5
    assert np.isfinite(m[..., 0]).any()
    names = ["means", "scales", "logits", "rgb", "dF"]
    _, out, grads = run(P, need_grad=True)
    h = 1e-7
    rng = np.random.default_rng(1)
    for name in names:
        base = np.asarray(P[name], np.float64)
        g = np.asarray(grads[name]).reshape(-1)
        gscale = max(np.abs(g).max(), 1e-3)
        bad = 0
        idxs = rng.choice(base.size, min(base.size, 30), replace=False)
        for k in idxs:
            e = np.zeros(base.size); e[k] = h
            Pp, Pm = dict(P), dict(P)
            Pp[name] = (base.reshape(-1) + e).reshape(base.shape)
            Pm[name] = (base.reshape(-1) - e).reshape(base.shape)
            fd = (run(Pp)[0] - run(Pm)[0]) / (2 * h)
            if abs(fd - g[k]) / gscale > 1e-3:
                bad += 1            # a decision flipped inside the FD step (jump in the loss)
        assert bad <= 1, (name, bad)


# ------------------------------------------------------------------- P8b-d: the three branches of Eq. 12's backward
def _branch_fd_problem(orc, P, *, options=7, hold_flags=False, W=16, H=16, seed=5):
    """A finite-difference problem on hand-made surfel populations (view pass, shadows off).  With `hold_flags` the
    per-surfel decisions (degenerate, flipped) are those of the unperturbed inputs, as in the record mode the GPU
    path is compared in (reading 4: a degenerate surfel passes no gradient through Q, g)."""
    rng = np.random.default_rng(seed)
    F, d = S.affine_camera(0.5, math.radians(20), 0.7, W, H, (4, 4, 0))
    view = make_view(W, H, F, view_dir=d, b_z=12.0, z_bg=16.0, bg=(0.2, 0.1, 0.3))
    up = [rng.normal(0, 1, (H, W, 4)) for _ in range(3)]
    up[2][..., 2:] = 0
    order = np.argsort(-np.asarray(P["means"])[:, 2], kind="stable").astype(np.uint32)
    base_flags = orc.preprocess_f64(view, P["means"], P["quats"], P["scales"], P["logits"], P["rgb"],
                                    F=view.F.astype(np.float64), dF=P["dF"])["flags"].copy()

    def run(Pv, need_grad=False):
        sh = orc.Shading(cc=Pv["cc"], ambient=Pv["ambient"])
        pre = orc.preprocess_f64(view, Pv["means"], Pv["quats"], Pv["scales"], Pv["logits"], Pv["rgb"],
                                 F=view.F.astype(np.float64), dF=Pv["dF"])
        rec, flags = pre["rec"], pre["flags"]
        if hold_flags:
            # keep the stored normal on the side the unperturbed preprocess chose, and the degenerate decision as it was
            resign = ((flags ^ base_flags) & orc.F_FLIPPED) != 0
            rec[resign, 13:16] *= -1.0
            flags = base_flags
        out = orc.forward(W, H, view.b_z, view.z_bg, view.bg_rgb, rec, flags, order, sh, options=options)
        loss = (out["rgba"] * up[0]).sum() + (out["geom"] * up[1]).sum() + (out["aux"] * up[2]).sum()
        if not need_grad:
            return loss, out
        bw = orc.backward(W, H, view.b_z, view.z_bg, view.bg_rgb, rec, flags, order, sh, *up, options=options)
        g = orc.preprocess_backward(view, Pv["means"], Pv["quats"], Pv["scales"], Pv["logits"], flags, bw["v_rec"],
                                    F=view.F.astype(np.float64), dF=Pv["dF"])
        grads = dict(means=g["v_means"], quats=g["v_quats"], scales=g["v_scales"], logits=g["v_logits"], rgb=g["v_rgb"],
                     dF=g["v_dF"], cc=bw["v_cc"], ambient=bw["v_ambient"])
        return loss, out, grads

    return view, run


def _pair_table(orc, view, P):
    """(pixel, surfel) pair quantities straight from the definitions (numpy, no oracle arithmetic): alpha * G with
    the Eq. 12 exponent, which term of Eq. 12 is active."""
    pre = orc.preprocess_f64(view, P["means"], P["quats"], P["scales"], P["logits"], P["rgb"],
                             F=view.F.astype(np.float64), dF=P["dF"])
    r = pre["rec"]
    px, py = pixel_grid(view.width, view.height)
    dx, dy = px[..., None] - r[:, 0], py[..., None] - r[:, 1]
    u, v = r[:, 2] * dx + r[:, 3] * dy, r[:, 4] * dx + r[:, 5] * dy
    deg = (pre["flags"] & orc.F_DEGENERATE) != 0
    rho3 = np.where(deg, np.inf, u * u + v * v)
    rho2 = 2.0 * (dx * dx + dy * dy)
    aG = r[:, 9] * np.exp(-0.5 * np.minimum(rho3, rho2))
    return dict(aG=aG, lowpass=~(rho3 <= rho2), rho3=rho3, rho2=rho2, flags=pre["flags"])


def _common_groups(rng, n):
    return dict(rgb=rng.uniform(0, 1, (n, 3)), dF=rng.normal(0, 1e-2, 8),
                cc=(np.concatenate([np.eye(3), np.zeros((3, 1))], 1) + rng.normal(0, 0.1, (3, 4))).reshape(12),
                ambient=rng.uniform(0.2, 0.5, 3))


def test_p8b_alpha_clamp_branch_finite_differences(orc):
    """alpha' = min(alpha_max, alpha G) (reading 7): where the clamp is active neither the opacity nor the
    Gaussian receives a gradient.  Large, nearly opaque surfels so that many pairs sit on the clamp."""
    rng = np.random.default_rng(41)
    n = 12
    quats = rng.normal(0, 0.15, (n, 4)); quats[:, 0] += 1.0
    logits = np.where(np.arange(n) % 2 == 0, rng.uniform(7.0, 10.0, n), rng.normal(0.5, 1.0, n))
    P = dict(means=np.concatenate([rng.uniform(0.5, 7.5, (n, 2)), rng.normal(0, 1.0, (n, 1))], 1), quats=quats,
             scales=rng.uniform(2.5, 6.0, (n, 2)), logits=logits, **_common_groups(rng, n))
    view, run = _branch_fd_problem(orc, P)
    T = _pair_table(orc, view, P)
    clamped = T["aG"] >= 0.99
    assert clamped.sum() >= 10, clamped.sum()                       # the branch is exercised ...
    assert np.abs(T["aG"] - 0.99).min() > 2e-5                      # ... and no pair sits on the switch itself
    out, _ = _check_fd(P, run, ["means", "quats", "scales", "logits", "rgb", "dF", "cc", "ambient"], rtol=2e-6)
    assert out["counters"][3] == clamped.sum()                      # the oracle takes the same branch for the same pairs


def test_p8c_lowpass_branch_finite_differences(orc):
    """Eq. 12 low-pass term: rho = 2 |x - c|^2 wins for sub-pixel and steeply tilted surfels; its gradient goes to the
    centre only (no Q, no g), and the depth falls back to z_c.  Cut-offs off, every parameter group."""
    rng = np.random.default_rng(43)
    n = 14
    # half the surfels sub-pixel (0.05-0.2 m at 0.5 m GSD), the others needle-like: sub-pixel across, pixels along,
    # tilted up to 70 degrees, so that both terms of Eq. 12 are active on significant pairs of the same surfel
    scales = np.where((np.arange(n) % 2 == 0)[:, None], rng.uniform(0.05, 0.2, (n, 2)),
                      np.stack([rng.uniform(0.06, 0.2, n), rng.uniform(1.0, 2.5, n)], 1))
    ang = rng.uniform(0.0, math.radians(70), n)
    axis = rng.normal(0, 1, (n, 3)); axis[:, 2] *= 0.3
    axis /= np.linalg.norm(axis, axis=1, keepdims=True)
    quats = np.concatenate([np.cos(ang / 2)[:, None], np.sin(ang / 2)[:, None] * axis], 1) * rng.uniform(0.5, 2.0, (n, 1))
    P = dict(means=np.concatenate([rng.uniform(1.0, 7.0, (n, 2)), rng.normal(0, 0.5, (n, 1))], 1), quats=quats,
             scales=scales, logits=rng.normal(1.0, 1.0, n), **_common_groups(rng, n))
    view, run = _branch_fd_problem(orc, P)
    T = _pair_table(orc, view, P)
    sig = T["aG"] > 1e-4                                            # pairs that matter to the loss
    lp = T["lowpass"] & sig
    assert lp.sum() >= 30 and lp.sum() >= 0.3 * sig.sum(), (lp.sum(), sig.sum())
    assert (~T["lowpass"] & sig).sum() >= 10                        # the Eq. 9 term is active beside it
    # no significant pair sits on the switch between the two terms (the depth jumps there)
    assert np.abs(T["rho3"] - T["rho2"])[sig].min() > 1e-3
    out, _ = _check_fd(P, run, ["means", "quats", "scales", "logits", "rgb", "dF", "cc", "ambient"], h=1e-7, rtol=2e-6)
    assert out["counters"][2] == T["lowpass"].sum()


def test_p8d_degenerate_surfels_pass_no_gradient_through_Q_and_g(orc):
    """Exactly edge-on surfels (det(B'RS') = 0): low-pass term only, depth z_c, and with the per-surfel
    decisions held fixed the objective does not depend on their scales, nor on their rotation except through the
    blended normal (reading 4)."""
    rng = np.random.default_rng(47)
    n = 12
    W = H = 16
    F, d = S.affine_camera(0.5, math.radians(20), 0.7, W, H, (4, 4, 0))
    quats = rng.normal(0, 0.3, (n, 4)); quats[:, 0] += 1.5
    common = _common_groups(rng, n)
    Bp = (np.asarray(F, np.float64).reshape(2, 4) + common["dF"].reshape(2, 4))[:, :3]
    ray = np.cross(Bp[0], Bp[1])            # the parallel-ray direction of F' = F + dF
    edge = [2, 7]
    for i in edge:                          # frame with the ray direction inside the surfel plane: t_u = ray
        tu = ray / np.linalg.norm(ray)
        tv = np.cross(rng.normal(0, 1, 3), tu); tv /= np.linalg.norm(tv)
        nn = np.cross(tu, tv)
        R = np.stack([tu, tv, nn], 1)
        w = 0.5 * math.sqrt(max(1e-12, 1 + R[0, 0] + R[1, 1] + R[2, 2]))
        quats[i] = [w, (R[2, 1] - R[1, 2]) / (4 * w), (R[0, 2] - R[2, 0]) / (4 * w), (R[1, 0] - R[0, 1]) / (4 * w)]
    means = np.concatenate([rng.uniform(1.0, 7.0, (n, 2)), rng.normal(0, 1.0, (n, 1))], 1)
    means[edge, 2] = [2.5, 1.8]            # in front of most of the others
    logits = rng.normal(0.5, 1.0, n); logits[edge] = [1.5, 2.5]
    P = dict(means=means, quats=quats, scales=rng.uniform(0.6, 2.0, (n, 2)), logits=logits, **common)
    view, run = _branch_fd_problem(orc, P, hold_flags=True)
    T = _pair_table(orc, view, P)
    deg = (T["flags"] & orc.F_DEGENERATE) != 0
    assert deg[edge].all() and deg.sum() == len(edge)
    assert (T["aG"][..., deg] > 1e-2).sum() >= 10                   # the degenerate surfels are seen
    out, _ = _check_fd(P, run, ["means", "quats", "scales", "logits", "rgb", "dF", "cc", "ambient"], rtol=2e-6)
    assert out["counters"][4] == deg.sum() * W * H                  # cut-offs off: every pixel composites them
    _, _, grads = run(P, need_grad=True)
    assert np.all(grads["scales"][edge] == 0.0)                     # nothing flows through Q or g ...
    assert np.abs(grads["means"][edge]).min() > 1e-6 and np.abs(grads["logits"][edge]).min() > 1e-6   # ... but the rest does
    assert np.abs(grads["quats"][edge]).max() > 1e-6                # (the rotation still moves the blended normal)


# ------------------------------------------------------------------------------- P19: the rounding-error twin
def test_p19_absolute_value_twin_bounds_and_is_not_vacuous(c0, orc):
    """The a_* twins of the backward (sum of |per-pair term| pushed through |chain Jacobian|) are what the GPU
    parity bar scales its rounding allowance with, so they are pinned by what the mathematics fixes:
    (a) triangle inequality: a >= |v| for every gradient value;
    (b) a == v where every term has the same sign (colour gradient under a non-negative upstream image);
    (c) the gradients are linear in the upstream images: scaling the upstream of every pixel by its own factor
        (1 + d_p), |d_p| <= delta, moves no gradient value by more than delta * a;
    (d) not vacuous: on C0 the typical a / |v| is a small number."""
    scene, view, tile = c0[0], c0[1], c0[2]
    up = S.upstream_grads(scene.seed, 0, view.height, view.width)
    sh = orc.Shading(cc=view.cc, ambient=view.ambient)
    args = (view.width, view.height, view.b_z, view.z_bg, view.bg_rgb, tile["rec64"], tile["flags"], tile["lists"], sh)

    def grads(upstream, twin):
        bw = orc.backward(*args, *upstream, threads=orc.num_threads(), twin=twin)
        g = orc.preprocess_backward(view, scene.means, scene.quats, scene.scales, scene.opacity_logits, tile["flags"],
                                    bw["v_rec"], a_rec=bw.get("a_rec"))
        g.update(v_cc=bw["v_cc"], v_ambient=bw["v_ambient"])
        if twin:
            g.update(a_cc=bw["a_cc"], a_ambient=bw["a_ambient"])
        return g

    g = grads(up, True)
    names = ["means", "quats", "scales", "logits", "rgb", "dF", "cc"]
    for k in names:
        v, a = g["v_" + k], g["a_" + k]
        assert (a >= np.abs(v) * (1 - 1e-12) - 1e-300).all(), k                              # (a)
        if v.size > 32:     # per-surfel groups (the global sums dF, cc cancel over a thousand surfels by themselves)
            nz = np.abs(v) > 1e-9 * np.abs(v).max()
            assert np.median(a[nz] / np.abs(v[nz])) < 25, (k, np.median(a[nz] / np.abs(v[nz])))  # (d)
    rng = np.random.default_rng(5)
    delta = 1e-3
    fac = 1 + delta * rng.choice([-1.0, 1.0], (view.height, view.width, 1))
    g2 = grads([u * fac for u in up], False)
    for k in names:
        assert (np.abs(g2["v_" + k] - g["v_" + k]) <= delta * g["a_" + k] * (1 + 1e-9) + 1e-18).all(), k   # (c)
    pos = [np.abs(up[0]) * np.array([1, 1, 1, 0.0]), None, None]
    gp = grads(pos, True)
    np.testing.assert_allclose(gp["a_rgb"], np.abs(gp["v_rgb"]), rtol=1e-12, atol=1e-300)      # (b): w v_albedo >= 0 ...
    assert (gp["v_rgb"] >= 0).all() and gp["v_rgb"].max() > 0                                  # ... with C0's identity CC


# ----------------------------------------------------------------------------------------- P11 / P12
def test_p11_shadow_test_closed_form(orc):
    W = H = 24
    gsd = 0.5
    view = make_view(W, H, nadir_F(gsd, W, H), z_bg=130.0)
    # one big opaque camera-facing surfel: A = 0.99 over the whole frame
    means = np.array([[0.0, 0.0, 20.0]])
    pre = orc.preprocess_f64(view, means, np.array([[1.0, 0, 0, 0]]), np.array([[500.0, 500.0]]), np.array([20.0]),
                             np.array([[0.5, 0.6, 0.7]]))
    Ws, Hs = 40, 30
    sx, sy = np.meshgrid(np.arange(Ws), np.arange(Hs))
    sun_depth = 70.0 + 0.5 * sx - 0.25 * sy                  # linear ramp: bilinear interpolation is exact
    reproj = np.array([1.2, 0.1, 0.05, 3.0, -0.1, 0.9, -0.02, 2.0])
    cc = np.array([[1.1, 0.05, 0, 0.01], [0, 0.9, 0.1, -0.02], [0.02, 0, 1.2, 0.03]])
    amb = np.array([0.3, 0.35, 0.45])
    sh = orc.Shading(cc=cc.reshape(12), ambient=amb, sun_depth=sun_depth, reproj=reproj, bias=0.5, slope=4.0)
    out = orc.forward(W, H, view.b_z, view.z_bg, view.bg_rgb, pre["rec"], pre["flags"], np.array([0], np.uint32), sh)
    px, py = pixel_grid(W, H)
    A = 0.99
    zv = A * (view.b_z - 20.0) + (1 - A) * view.z_bg
    h = view.b_z - zv
    xs = reproj[0] * px + reproj[1] * py + reproj[2] * h + reproj[3]
    ys = reproj[4] * px + reproj[5] * py + reproj[6] * h + reproj[7]
    inside = (xs >= 0.5) & (xs <= Ws - 0.5) & (ys >= 0.5) & (ys <= Hs - 0.5)
    ds = 70.0 + 0.5 * (xs - 0.5) - 0.25 * (ys - 0.5)
    V = np.where(inside, 1 / (1 + np.exp(4.0 * (zv - ds - 0.5))), 1.0)
    assert inside.any() and (~inside).any() and V[inside].min() < 0.2 and V[inside].max() > 0.8
    np.testing.assert_allclose(out["aux"][..., 2], V, atol=1e-12)
    albedo = A * np.array([0.5, 0.6, 0.7])
    for c in range(3):
        I = (cc[c, :3] @ albedo + cc[c, 3]) * (V + (1 - V) * amb[c])          # Eq. 1
        np.testing.assert_allclose(out["rgba"][..., c], I, atol=1e-12)


def test_p12_identity_cases(c0, orc):
    scene, view, tile, f_tile, _, _ = c0
    np.testing.assert_array_equal(f_tile["rgba"][..., :3], f_tile["albedo"])    # CC = [I 0], shadows off
    np.testing.assert_array_equal(f_tile["aux"][..., 2], 1.0)
    cc = np.array([[0.9, 0.1, 0, 0.05], [0, 1.1, 0, 0], [0.1, 0, 0.8, -0.05]])
    f2 = orc.forward(view.width, view.height, view.b_z, view.z_bg, view.bg_rgb, tile["rec64"], tile["flags"],
                     tile["lists"], orc.Shading(cc=cc.reshape(12), ambient=(0.5, 0.5, 0.5)), threads=orc.num_threads())
    exp = f_tile["albedo"] @ cc[:, :3].T + cc[:, 3]
    np.testing.assert_allclose(f2["rgba"][..., :3], exp, atol=1e-14)
    for k in ("geom", "aux"):
        np.testing.assert_array_equal(f2[k], f_tile[k])


# ------------------------------------------------------------------------------------------------ P14
def test_p14_sun_camera_adjoint_fd_and_closed_form(orc):
    """Cascade: the sun camera and the reprojection constants are functions of F' = F + dF.
    (a) the adjoint of Eq. 16 + viewport against central finite differences of the forward helper;
    (b) the mathematics fixes the result: for a sun camera built by Eq. 16 the reprojection collapses to
        x_s = diag(sc) x - sc (B s) h + t, so the columns R_x and k_0 do not depend on F' at all and only k_h does."""
    rng = np.random.default_rng(5)
    for trial in range(4):
        Fp = np.array([[2.0, 0.1, 0.3, 40.0], [-0.15, -1.9, 0.8, 70.0]]).reshape(8) + rng.normal(0, 0.1, 8)
        az, el = rng.uniform(0, 2 * np.pi), np.radians(rng.uniform(30, 70))
        vp = np.array([rng.uniform(0.5, 2), rng.uniform(0.5, 2), rng.normal(0, 5), rng.normal(0, 5)])
        vF, vR = rng.normal(0, 1, 8), rng.normal(0, 1, 8)
        g = orc.sun_camera_backward(Fp, az, el, vp, vF, vR)

        def f(x):
            Fs, rp = orc.sun_camera(x, az, el, vp)
            return float(Fs @ vF + rp @ vR)
        for k in range(8):
            e = np.zeros(8); e[k] = 1e-6
            fd = (f(Fp + e) - f(Fp - e)) / 2e-6
            assert abs(fd - g[k]) < 1e-7 * max(1.0, np.abs(g).max()), (trial, k, fd, g[k])
        # (b) closed form
        Fs, rp = orc.sun_camera(Fp, az, el, vp)
        s = np.array([np.cos(az) / np.tan(el), np.sin(az) / np.tan(el), 1.0])
        B = Fp.reshape(2, 4)[:, :3]
        expect = np.array([[vp[0], 0, -vp[0] * (B[0] @ s), vp[2]], [0, vp[1], -vp[1] * (B[1] @ s), vp[3]]]).reshape(8)
        np.testing.assert_allclose(rp, expect, rtol=1e-11, atol=1e-10)
        only_const = np.zeros(8); only_const[[0, 1, 3, 4, 5, 7]] = rng.normal(0, 1, 6)
        np.testing.assert_allclose(orc.sun_camera_backward(Fp, az, el, vp, np.zeros(8), only_const), 0, atol=1e-9)


def test_p20_nearby_camera_nullspace_identity_roundtrip_and_adjoint(orc):
    """Nearby camera of the cascade (Fig. 1 :159; reading 27), pinned by what the text fixes:
    (a) zero perturbation returns the input camera (d_main is the nullspace of B_xy);
    (b) the new viewing direction s' is the nullspace of B_nearby (S5-S6 applied to the new direction);
    (c) round trip: the azimuth / elevation of the nearby camera's OWN main direction B_x x B_y are the perturbed angles;
    (d) the angles of a camera built from a known direction by the scene recipe are that direction's (independent of the
        cross product: the recipe's d is an input here);
    (e) the adjoint against central finite differences of the forward."""
    rng = np.random.default_rng(12)
    for trial in range(6):
        theta, psi = math.radians(rng.uniform(5, 35)), rng.uniform(0, 2 * math.pi)
        F, d = S.affine_camera(0.4, theta, psi, 512, 512, (10.0, -20.0, 5.0))
        Fp = np.asarray(F, np.float64).reshape(8) + rng.normal(0, 1e-3, 8)
        B = Fp.reshape(2, 4)[:, :3]
        # (a)
        F0, ang = orc.nearby_camera(Fp, 0.0, 0.0)
        np.testing.assert_allclose(F0, Fp, rtol=0, atol=1e-12 * np.abs(Fp).max())
        # (d) the up-pointing ray of the unperturbed recipe camera is -d: off-nadir theta <=> elevation 90 deg - theta
        _, ang_clean = orc.nearby_camera(np.asarray(F, np.float64).reshape(8), 0.0, 0.0)
        up_ray = -np.asarray(d, np.float64)
        assert abs(ang_clean[1] - (math.pi / 2 - theta)) < 1e-6
        assert abs(math.remainder(ang_clean[0] - math.atan2(up_ray[1], up_ray[0]), 2 * math.pi)) < 1e-5
        # (b), (c)
        da, de = rng.normal(0, 0.05), rng.normal(0, 0.03)
        Fn, _ = orc.nearby_camera(Fp, da, de)
        a2, e2 = ang[0] + da, ang[1] + de
        s2 = np.array([math.cos(a2) / math.tan(e2), math.sin(a2) / math.tan(e2), 1.0])
        Bn = Fn.reshape(2, 4)[:, :3]
        assert np.abs(Bn @ s2).max() < 1e-10 * np.abs(Bn).max()
        assert np.array_equal(Fn.reshape(2, 4)[:, [0, 1, 3]], Fp.reshape(2, 4)[:, [0, 1, 3]])    # Eq. 16 only touches column 3
        _, ang_n = orc.nearby_camera(Fn, 0.0, 0.0)
        assert abs(math.remainder(ang_n[0] - a2, 2 * math.pi)) < 1e-9 and abs(ang_n[1] - e2) < 1e-9
        # a point moved along the new direction keeps its nearby-image position (definition of a viewing direction)
        p = rng.normal(0, 30, 3)
        assert np.abs(Bn @ (p + 7.0 * s2) - Bn @ p).max() < 1e-8
        # (e)
        vF = rng.normal(0, 1, 8)
        g = orc.nearby_camera_backward(Fp, da, de, vF)
        for k in range(8):
            h = 1e-6 * max(1.0, abs(Fp[k]))
            e = np.zeros(8); e[k] = h
            fd = (orc.nearby_camera(Fp + e, da, de)[0] @ vF - orc.nearby_camera(Fp - e, da, de)[0] @ vF) / (2 * h)
            assert abs(fd - g[k]) < 2e-6 * max(1.0, np.abs(g).max()), (trial, k, fd, g[k])
    # a gradient that only reaches the untouched columns passes straight through
    only = np.zeros(8); only[[0, 1, 3, 4, 5, 7]] = 1.0
    np.testing.assert_allclose(orc.nearby_camera_backward(Fp, 0.02, -0.01, only), only, atol=1e-12)


def test_p14_cascade_total_dF_finite_differences(orc):
    """The whole cascade in one objective: dF moves the view camera, the sun camera built from it (Eq. 16), the sun
    depth map rendered with that camera, and the reprojection of the shadow test.  Total analytic gradient
    = view-pass v_dF + sun_camera_backward(sun-pass v_dF, v_reproj), against finite differences (cut-offs off)."""
    rng = np.random.default_rng(77)
    n, W, H, Ws, Hs = 12, 16, 16, 24, 24
    F, d = S.affine_camera(0.5, math.radians(20), 0.7, W, H, (4, 4, 0))
    means = np.concatenate([rng.uniform(1.0, 7.0, (n, 2)), rng.normal(0, 1.0, (n, 1))], 1)
    quats = rng.normal(0, 1, (n, 4)); quats[:, 0] += 3.0
    scales, logits, rgb = rng.uniform(0.8, 2.0, (n, 2)), rng.normal(0.5, 1, n), rng.uniform(0, 1, (n, 3))
    cc = (np.concatenate([np.eye(3), np.zeros((3, 1))], 1) + rng.normal(0, 0.1, (3, 4))).reshape(12)
    ambient = rng.uniform(0.2, 0.5, 3)
    az, el = 0.9, math.radians(50)
    vp = np.array([1.3, 1.3, 4.0, 6.0])
    view = make_view(W, H, F, view_dir=d, b_z=12.0, z_bg=16.0, bg=(0.2, 0.1, 0.3))
    up = [rng.normal(0, 1, (H, W, 4)) for _ in range(3)]
    up[2][..., 2:] = 0
    order = np.argsort(-means[:, 2], kind="stable").astype(np.uint32)
    F64 = view.F.astype(np.float64)
    sdir = -np.array([np.cos(az) * np.cos(el), np.sin(az) * np.cos(el), np.sin(el)])

    def run(dF, need_grad=False):
        Fp = F64.reshape(8) + dF
        F_sun, reproj = orc.sun_camera(Fp, az, el, vp)
        sun_view = make_view(Ws, Hs, F_sun.astype(np.float32), view_dir=sdir, b_z=12.0, z_bg=16.0, bg=(0, 0, 0))
        pre_s = orc.preprocess_f64(sun_view, means, quats, scales, logits, rgb, F=F_sun, dF=np.zeros(8))
        fs = orc.forward(Ws, Hs, 12.0, 16.0, np.zeros(3), pre_s["rec"], pre_s["flags"], order, orc.Shading(), options=7)
        sun_depth = fs["geom"][..., 3] + fs["aux"][..., 3] * 16.0
        sh = orc.Shading(cc=cc, ambient=ambient, sun_depth=sun_depth, reproj=reproj, bias=0.5, slope=4.0)
        pre = orc.preprocess_f64(view, means, quats, scales, logits, rgb, F=F64, dF=dF)
        out = orc.forward(W, H, 12.0, 16.0, view.bg_rgb, pre["rec"], pre["flags"], order, sh, options=7)
        loss = (out["rgba"] * up[0]).sum() + (out["geom"] * up[1]).sum() + (out["aux"] * up[2]).sum()
        if not need_grad:
            return loss, out
        bw = orc.backward(W, H, 12.0, 16.0, view.bg_rgb, pre["rec"], pre["flags"], order, sh, *up, options=7)
        g = orc.preprocess_backward(view, means, quats, scales, logits, pre["flags"], bw["v_rec"], F=F64, dF=dF)
        v_sd = bw["v_sun_depth"]
        vg = np.zeros((Hs, Ws, 4)); vg[..., 3] = v_sd
        vr = np.zeros((Hs, Ws, 4)); vr[..., 3] = -16.0 * v_sd
        bs = orc.backward(Ws, Hs, 12.0, 16.0, np.zeros(3), pre_s["rec"], pre_s["flags"], order, orc.Shading(), vr, vg, None,
                          options=7)
        gs = orc.preprocess_backward(sun_view, means, quats, scales, logits, pre_s["flags"], bs["v_rec"], F=F_sun,
                                     dF=np.zeros(8))
        total = g["v_dF"] + orc.sun_camera_backward(Fp, az, el, vp, gs["v_dF"], bw["v_reproj"])
        return loss, out, total, g["v_dF"]

    dF0 = rng.normal(0, 1e-2, 8)
    _, out, total, direct = run(dF0, need_grad=True)
    V = out["aux"][..., 2]
    assert V.min() < 0.5 and V.max() > 0.8                       # the shadow test is exercised
    assert np.abs(total - direct).max() > 1e-2 * np.abs(total).max()   # the cascade term matters in this problem
    scale = np.abs(total).max()
    for k in range(8):
        e = np.zeros(8); e[k] = 1e-6 * max(1.0, abs(F64.reshape(8)[k]))
        fd = (run(dF0 + e)[0] - run(dF0 - e)[0]) / (2 * e[k])
        assert abs(fd - total[k]) < 2e-5 * scale, (k, fd, total[k], direct[k])


# ------------------------------------------------------------------------------------------------ P15
def _adam_problem(seed=3, n=50):
    rng = np.random.default_rng(seed)
    params = dict(means=rng.normal(0, 5, (n, 3)), quats=rng.normal(0, 1, (n, 4)), scales=rng.uniform(0.2, 2.0, (n, 2)),
                  logits=rng.normal(0, 2, n), rgb=rng.uniform(0, 1, (n, 3)))
    lrs = dict(means=0.075, quats=0.001, scales=0.001, logits=0.05, rgb=0.0025)   # PAPER.md:349 (+ opacity: argument)
    return rng, params, lrs


def test_p15_adam_first_step_closed_form():
    """t = 1 from zero state: m^ = g, v^ = g^2, so the step is lr g / (|g| + eps) whatever b1, b2 are."""
    from oracle import adam
    rng, params, lrs = _adam_problem()
    grads = {k: rng.normal(0, 1, v.shape) * 10.0 ** rng.uniform(-4, 2) for k, v in params.items()}
    state = {k: (np.zeros_like(v), np.zeros_like(v)) for k, v in params.items()}
    new, st = adam.adam_step(params, grads, state, lrs, beta1=0.8, beta2=0.95, eps=1e-8, step=1)
    for k in adam.GROUPS:
        g = grads[k] * (params[k] if k == "scales" else 1.0)
        step = lrs[k] * g / (np.abs(g) + 1e-8)
        expect = params[k] * np.exp(-step) if k == "scales" else params[k] - step
        np.testing.assert_allclose(new[k], expect, rtol=1e-12, atol=1e-14)
        np.testing.assert_allclose(st[k][0], 0.2 * g, rtol=1e-12)
        np.testing.assert_allclose(st[k][1], 0.05 * g * g, rtol=1e-12)
    assert (new["scales"] > 0).all()


def test_p15_adam_matches_torch_optimizer_over_several_steps():
    """torch.optim.Adam (an independent library routine) on the same sequence of gradients; the scale group is handed to
    torch as theta = log s with the chain-ruled gradient, which is what "stepped in log space" means."""
    import torch
    from oracle import adam
    rng, params, lrs = _adam_problem(seed=8)
    tp = {k: torch.tensor(np.log(v) if k == "scales" else v, dtype=torch.float64, requires_grad=True) for k, v in params.items()}
    opt = torch.optim.Adam([dict(params=[tp[k]], lr=lrs[k]) for k in adam.GROUPS], betas=(0.9, 0.999), eps=1e-8)
    state = {k: (np.zeros_like(v), np.zeros_like(v)) for k, v in params.items()}
    cur = {k: v.copy() for k, v in params.items()}
    for t in range(1, 8):
        grads = {k: rng.normal(0, 1, v.shape) * (1.0 + 0.3 * t) for k, v in params.items()}
        cur_before = cur
        cur, state = adam.adam_step(cur, grads, state, lrs, step=t)
        for k in adam.GROUPS:
            g = grads[k] * (cur_before[k] if k == "scales" else 1.0)
            tp[k].grad = torch.tensor(g, dtype=torch.float64)
        opt.step()
        for k in adam.GROUPS:
            ref = tp[k].detach().numpy()
            ref = np.exp(ref) if k == "scales" else ref
            np.testing.assert_allclose(cur[k], ref, rtol=1e-10, atol=1e-12)


def test_p15_camera_adam_is_per_view_adam():
    """Per-camera groups (1e-4 camera deltas, 1e-3 gain and bias): over a sequence of iterations that render
    one view each, every view's rows follow torch.optim.Adam (an independent routine) run on that view ALONE with the
    gradients of the iterations that rendered it -- own state, own step counter -- and an iteration leaves the rows, the
    state and the counters of all other views bit for bit alone."""
    import torch
    from oracle import adam
    rng = np.random.default_rng(21)
    V = 4
    width = dict(dF=8, cc=12, ambient=3)
    lrs = dict(dF=1e-4, cc=1e-3, ambient=1e-3)
    params = {k: rng.normal(0, 1, (V, w)) for k, w in width.items()}
    state = {k: (np.zeros((V, w)), np.zeros((V, w))) for k, w in width.items()}
    steps = np.zeros(V, np.int64)
    tp = [{k: torch.tensor(params[k][v], dtype=torch.float64, requires_grad=True) for k in adam.CAMERA_GROUPS} for v in range(V)]
    opts = [torch.optim.Adam([dict(params=[tp[v][k]], lr=lrs[k]) for k in adam.CAMERA_GROUPS], betas=(0.9, 0.999), eps=1e-8) for v in range(V)]
    order = [0, 2, 2, 1, 0, 2, 3, 2, 0, 0, 1, 2]          # view 2 is rendered five times, view 3 once
    for it, view in enumerate(order):
        grads = {k: rng.normal(0, 1, w) * 10.0 ** rng.uniform(-3, 1) for k, w in width.items()}
        before = {k: params[k].copy() for k in width}, {k: (state[k][0].copy(), state[k][1].copy()) for k in width}, steps.copy()
        params, state, steps = adam.adam_step_cameras(params, grads, state, steps, view, lrs)
        for k in adam.CAMERA_GROUPS:
            tp[view][k].grad = torch.tensor(grads[k], dtype=torch.float64)
        opts[view].step()
        others = np.arange(V) != view
        for k in adam.CAMERA_GROUPS:
            np.testing.assert_allclose(params[k][view], tp[view][k].detach().numpy(), rtol=1e-12, atol=1e-15)
            assert np.array_equal(params[k][others], before[0][k][others])
            assert np.array_equal(state[k][0][others], before[1][k][0][others]) and np.array_equal(state[k][1][others], before[1][k][1][others])
            assert not np.array_equal(params[k][view], before[0][k][view])
        assert steps[view] == before[2][view] + 1 and np.array_equal(steps[others], before[2][others])
    assert steps.tolist() == [4, 2, 5, 1]
    # first step of a view, whatever the global iteration: lr g / (|g| + eps)
    p1 = {k: np.zeros((1, w)) for k, w in width.items()}
    g1 = {k: rng.normal(0, 1, w) for k, w in width.items()}
    out, _, _ = adam.adam_step_cameras(p1, g1, {k: (np.zeros((1, w)), np.zeros((1, w))) for k, w in width.items()}, np.zeros(1), 0, lrs)
    for k in adam.CAMERA_GROUPS:
        np.testing.assert_allclose(out[k][0], -lrs[k] * g1[k] / (np.abs(g1[k]) + 1e-8), rtol=1e-12)


# ------------------------------------------------------------------------------------------------ P16
def test_p16_depth_normals_of_a_world_plane():
    """Eq. 13 on the depth image of a tilted world plane seen by an affine camera: every interior pixel must return the
    plane's normal.  The depth image is built independently of the backprojection formula: each pixel's parallel ray
    (direction = null space of B) is intersected with the plane n0 . (p - q) = 0."""
    from oracle import losses
    W, H = 40, 32
    F, d = S.affine_camera(0.5, math.radians(25), 0.9, W, H, (10, 8, 0))
    Fp = np.asarray(F, np.float64).reshape(2, 4)
    B, b = Fp[:, :3], Fp[:, 3]
    ray = np.cross(B[0], B[1]); ray /= np.linalg.norm(ray)
    n0 = np.array([0.15, -0.25, 1.0]); n0 /= np.linalg.norm(n0)
    q = np.array([10.0, 8.0, 3.0])
    b_z = 20.0
    zv = np.zeros((H, W))
    for j in range(H):
        for i in range(W):
            x = np.array([i + 0.5, j + 0.5])
            p0 = np.linalg.lstsq(B, x - b, rcond=None)[0]          # some point on the pixel's ray
            t = (n0 @ (q - p0)) / (n0 @ ray)
            zv[j, i] = b_z - (p0 + t * ray)[2]
    N, c, _, _, interior, sgn = losses.depth_normals(zv, Fp, d, b_z)
    expect = n0 if n0 @ np.asarray(d, np.float64) < 0 else -n0      # facing the sensor
    assert np.abs(N[interior] - expect).max() < 1e-9
    assert (N[~interior] == 0).all() and interior.sum() == (W - 2) * (H - 2)
    # cross-check on a non-planar depth image: p_s is affine in z_v, so the cross product of the central differences
    # factors as c = c0 + dx c1 + dy c2 with dx, dy the central differences of the depth alone (the form a kernel
    # would evaluate); the oracle itself is Eq. 13 as written
    rng = np.random.default_rng(9)
    zv2 = zv + rng.normal(0, 0.3, zv.shape)
    N2, c2_, _, _, _, _ = losses.depth_normals(zv2, Fp, d, b_z)
    Bi = np.linalg.inv(Fp[:, :2])
    k = np.array([*(Bi @ Fp[:, 2]), -1.0])
    ax, ay = np.array([*(2.0 * Bi[:, 0]), 0.0]), np.array([*(2.0 * Bi[:, 1]), 0.0])
    dx = zv2[1:-1, 2:] - zv2[1:-1, :-2]
    dy = zv2[2:, 1:-1] - zv2[:-2, 1:-1]
    fact = np.cross(ax, ay) + dx[..., None] * np.cross(k, ay) + dy[..., None] * np.cross(ax, k)
    np.testing.assert_allclose(c2_[1:-1, 1:-1], fact, rtol=1e-10, atol=1e-12)
    assert np.abs(np.linalg.norm(N2[1:-1, 1:-1], axis=-1) - 1).max() < 1e-12


def test_p16_ssim_identities_and_brute_force_window():
    from oracle import losses
    rng = np.random.default_rng(4)
    g = losses.gaussian_window()
    assert abs(g.sum() - 1) < 1e-15 and np.allclose(g, g[::-1]) and len(g) == 11
    I = rng.uniform(0, 1, (24, 30, 3))
    m, _ = losses.ssim_map_and_grad(I, I.copy())
    assert np.abs(m - 1).max() < 1e-12                              # identical images, borders included
    # constant images away from the (zero-padded) border: variances vanish, SSIM = (2ab + C1)/(a^2 + b^2 + C1)
    a, b = 0.3, 0.7
    m, _ = losses.ssim_map_and_grad(np.full((30, 30, 3), a), np.full((30, 30, 3), b))
    np.testing.assert_allclose(m[10:20, 10:20], (2 * a * b + losses.C1) / (a * a + b * b + losses.C1), rtol=1e-9)
    # brute force at a few pixels: 2-D window = outer(g, g), zero outside the image
    J = rng.uniform(0, 1, (24, 30, 3))
    m, _ = losses.ssim_map_and_grad(I, J)
    G2 = np.outer(g, g)
    for (y, x) in [(0, 0), (3, 28), (12, 15), (23, 7)]:
        def win(A):
            acc = np.zeros(3)
            for dy in range(-5, 6):
                for dx in range(-5, 6):
                    yy, xx = y + dy, x + dx
                    if 0 <= yy < 24 and 0 <= xx < 30:
                        acc += G2[dy + 5, dx + 5] * A[yy, xx]
            return acc
        mu1, mu2 = win(I), win(J)
        s11, s22, s12 = win(I * I) - mu1 ** 2, win(J * J) - mu2 ** 2, win(I * J) - mu1 * mu2
        ref = ((2 * mu1 * mu2 + losses.C1) * (2 * s12 + losses.C2)) / ((mu1 ** 2 + mu2 ** 2 + losses.C1) * (s11 + s22 + losses.C2))
        np.testing.assert_allclose(m[y, x], ref, rtol=1e-10)


def test_p16_loss_upstream_gradients_finite_differences():
    """d(total)/d(rgba, geom, aux) against central finite differences (alpha's stop-gradient copy held fixed)."""
    from oracle import losses
    rng = np.random.default_rng(9)
    W, H = 20, 18
    F, d = S.affine_camera(0.5, math.radians(20), 0.7, W, H, (5, 4, 0))
    rgba = rng.uniform(0.1, 0.9, (H, W, 4))
    geom = np.concatenate([rng.normal(0, 0.5, (H, W, 3)), rng.uniform(8, 12, (H, W, 1))], -1)
    aux = rng.uniform(0, 1, (H, W, 4))
    target = rng.uniform(0, 1, (H, W, 3))
    args = dict(Fp=F, view_dir=d, b_z=15.0, z_bg=14.0, w_l1=0.8, w_ssim=0.2, w_dist=0.05, w_normal=0.05)
    A0 = rgba[..., 3].copy()
    terms, v_rgba, v_geom, v_aux = losses.loss_and_upstream(rgba, geom, aux, target, alpha_sg=A0, **args)
    assert 0 < terms["ssim"] < 1 and terms["l1"] > 0 and 0 < terms["normal"] < 2
    arrs, grads = dict(rgba=rgba, geom=geom, aux=aux), dict(rgba=v_rgba, geom=v_geom, aux=v_aux)

    def total(**over):
        a = {**arrs, **over}
        return losses.loss_and_upstream(a["rgba"], a["geom"], a["aux"], target, alpha_sg=A0, **args)[0]["total"]
    for name in ("rgba", "geom", "aux"):
        base, g = arrs[name], grads[name]
        gs = np.abs(g).max()
        for _ in range(40):
            idx = (rng.integers(H), rng.integers(W), rng.integers(4))
            e = np.zeros_like(base); e[idx] = 1e-6
            fd = (total(**{name: base + e}) - total(**{name: base - e})) / 2e-6
            assert abs(fd - g[idx]) < 1e-6 * gs + 1e-10, (name, idx, fd, g[idx])
    assert np.abs(v_geom[..., 3]).max() > 0 and np.abs(v_rgba[..., 3]).max() > 0     # the depth path is exercised


# ------------------------------------------------------------------------------------------------ P17
def test_p17_area_weights_plane_and_inverse_cdf():
    """a = |dx x dy|.  A tilted plane has the same weight cell^2 sqrt(1 + a^2 + b^2) in every cell (finite
    differences are exact for planes, one-sided ones included); the inverse transform on a hand-made weight row."""
    from oracle import init
    cell = 0.5
    yy, xx = np.meshgrid(np.arange(7) + 0.5, np.arange(9) + 0.5, indexing="ij")
    h = 0.8 * xx * cell - 1.7 * yy * cell + 3.0
    np.testing.assert_allclose(init.area_weights(h, cell), cell * cell * math.sqrt(1 + 0.8 ** 2 + 1.7 ** 2), rtol=1e-12)
    w = np.array([[1.0, 3.0], [2.0, 2.0]])            # cumulative 1, 4, 6, 8
    got = init.sample_cells(w, np.array([0.0, 0.124, 0.125, 0.49, 0.5, 0.74, 0.75, 0.999999]))
    assert got.tolist() == [0, 0, 1, 1, 2, 2, 3, 3]


def test_p17_facades_receive_their_share_of_samples():
    """A box building on flat ground: the cells on the wall ring carry the extra area |dh| * cell per unit length, and the
    sampled fraction follows the weights (PAPER.md:186 'building facades ... more likely to be selected')."""
    from oracle import init
    rng = np.random.default_rng(2)
    cell, n = 0.5, 200000
    h = np.zeros((60, 60)); h[20:40, 20:40] = 12.0
    w = init.area_weights(h, cell)
    wall = w > 1.5 * cell * cell
    assert wall.sum() > 0                                         # a two-cell-wide ring (central differences)
    out = init.init_from_dsm(h, cell, (0.0, 0.0), rng.uniform(0, 1, n), rng.uniform(0, 1, n), rng.uniform(0, 1, n))
    frac = wall.ravel()[out["cells"]].mean()
    expect = w[wall].sum() / w.sum()
    assert abs(frac - expect) < 4 * math.sqrt(expect * (1 - expect) / n)
    assert expect > 5 * wall.mean()                                # far more than their share of the footprint


def test_p17_frames_quaternions_and_knn_scale():
    from oracle import init
    from scipy.spatial.transform import Rotation
    rng = np.random.default_rng(3)
    for _ in range(50):
        hx, hy = rng.normal(0, 3, 2)
        R = init.frame(hx, hy)
        np.testing.assert_allclose(R.T @ R, np.eye(3), atol=1e-12)
        assert abs(np.linalg.det(R) - 1) < 1e-12
        n = np.array([-hx, -hy, 1.0]); n /= np.linalg.norm(n)
        np.testing.assert_allclose(R[:, 2], n, atol=1e-12)
        # t_u is the world x axis made orthogonal to n: in the plane of (e_x, n), on e_x's side
        assert abs(R[:, 0] @ np.cross(n, [1.0, 0, 0])) < 1e-12 and R[0, 0] > 0
        q = init.rotation_to_quat(R)
        assert q[0] >= 0 and abs(np.linalg.norm(q) - 1) < 1e-12
        np.testing.assert_allclose(Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix(), R, atol=1e-12)
    # kNN scale against brute force
    h = rng.normal(0, 1, (30, 30)).cumsum(0).cumsum(1) * 0.05
    n = 300
    out = init.init_from_dsm(h, 0.5, (10.0, -5.0), rng.uniform(0, 1, n), rng.uniform(0, 1, n), rng.uniform(0, 1, n))
    P_ = out["means"]
    D = np.linalg.norm(P_[:, None, :] - P_[None, :, :], axis=-1)
    D.sort(axis=1)
    np.testing.assert_allclose(out["scales"][:, 0], D[:, 1:4].mean(1), rtol=1e-12)
    assert (out["scales"][:, 0] == out["scales"][:, 1]).all()
    # centres lie on their cell's tangent plane and inside the cell
    col = np.floor((P_[:, 0] - 10.0) / 0.5).astype(int); row = np.floor((P_[:, 1] + 5.0) / 0.5).astype(int)
    assert (row * 30 + col == out["cells"]).all()


# ------------------------------------------------------------------------------------------------ P18
def test_p18_relocation_factors_preserve_centre_opacity_and_profile_integral():
    """The two things the 3DGS-MCMC relocation [22] is built to preserve, checked without its formula: N copies of
    opacity o' composited at the centre give the old opacity, and the composited 1-D profile through the centre keeps its
    integral (numerical quadrature of 1 - (1 - o' g_{s'}(x))^N against alpha s sqrt(2 pi))."""
    from oracle import relocate
    assert relocate.relocation_factors(0.37, 1) == (pytest.approx(0.37, rel=1e-15), pytest.approx(1.0, rel=1e-14))
    x = np.linspace(-60, 60, 2_400_001)
    for alpha in (0.02, 0.5, 0.93, 0.999):
        for n in (2, 3, 7, 20, 51):
            o_new, f = relocate.relocation_factors(alpha, n)
            assert abs(1 - (1 - o_new) ** n - alpha) < 1e-12
            s_old = 1.7
            s_new = s_old * f
            prof = 1 - (1 - o_new * np.exp(-x * x / (2 * s_new * s_new))) ** n
            integral = np.trapezoid(prof, x)
            assert abs(integral - alpha * s_old * math.sqrt(2 * math.pi)) < 1e-8 * integral, (alpha, n)
            assert 0 < f and s_new > 0


def test_p18_relocate_hand_example_and_degenerate_cases():
    from oracle import relocate
    sig_inv = lambda a: math.log(a / (1 - a))
    alphas = np.array([0.5, 0.001, 0.25, 0.004, 0.25])                 # surfels 1 and 3 are dead (<= 0.005)
    n = 5
    rng = np.random.default_rng(0)
    means, quats, scales, rgb = rng.normal(0, 1, (n, 3)), rng.normal(0, 1, (n, 4)), rng.uniform(0.5, 2, (n, 2)), rng.uniform(0, 1, (n, 3))
    logits = np.array([sig_inv(a) for a in alphas])
    st = lambda: dict(means=np.ones((n, 3)), quats=np.ones((n, 4)), scales=np.ones((n, 2)), logits=np.ones(n), rgb=np.ones((n, 3)))
    # live cumulative weights: [0.5, 0.5, 0.75, 0.75, 1.0]; u = 0.6 -> surfel 2, u = 0.1 -> surfel 0
    u = np.array([0.9, 0.6, 0.9, 0.1, 0.9])
    out = relocate.relocate(means, quats, scales, logits, rgb, st(), st(), u)
    assert out["dead"].tolist() == [False, True, False, True, False]
    assert out["src"].tolist() == [-1, 2, -1, 0, -1] and out["ratio"].tolist() == [2, 1, 2, 1, 1]
    for d, j in ((1, 2), (3, 0)):
        o_new, f = relocate.relocation_factors(alphas[j], 2)
        for k in ("means", "quats", "rgb"):
            np.testing.assert_array_equal(out[k][d], [means, quats, rgb][["means", "quats", "rgb"].index(k)][j])
        np.testing.assert_allclose(out["scales"][d], scales[j] * f, rtol=1e-14)
        np.testing.assert_allclose(out["scales"][j], scales[j] * f, rtol=1e-14)
        assert abs(1 / (1 + math.exp(-out["logits"][d])) - o_new) < 1e-14 and out["logits"][j] == out["logits"][d]
        np.testing.assert_array_equal(out["means"][j], means[j])
    # surfel 4 untouched, bit for bit; Adam state zeroed exactly on the four touched surfels
    for k, a in (("means", means), ("quats", quats), ("scales", scales), ("logits", logits), ("rgb", rgb)):
        np.testing.assert_array_equal(out[k][4], a[4])
    assert out["adam_m"]["means"][[0, 1, 2, 3]].sum() == 0 and (out["adam_m"]["means"][4] == 1).all()
    assert out["adam_v"]["logits"].tolist() == [0, 0, 0, 0, 1]
    # nothing dead / nothing alive: nothing moves
    same = relocate.relocate(means, quats, scales, np.full(n, 1.0), rgb, None, None, u)
    np.testing.assert_array_equal(same["scales"], scales)
    none_alive = relocate.relocate(means, quats, scales, np.full(n, -20.0), rgb, None, None, u)
    np.testing.assert_array_equal(none_alive["means"], means)
    # many copies of one source: the cap n_max applies to the factors
    logits2 = np.array([sig_inv(0.8)] + [-20.0] * 60)
    big = relocate.relocate(np.zeros((61, 3)), np.ones((61, 4)), np.ones((61, 2)), logits2, np.zeros((61, 3)), None, None,
                            np.full(61, 0.5))
    o51, f51 = relocate.relocation_factors(0.8, 51)
    np.testing.assert_allclose(big["scales"], f51, rtol=1e-12)
    assert big["ratio"][0] == 61

"""Seeded synthetic inputs for the affine-2DGS rasteriser (stand-ins for the paper's sites).

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_2606_28581_b200/``) and therefore holds NONE of the method's arithmetic: no
projection of surfels, no Gaussian evaluation, no blending, no sun-camera construction
(Eq. 16 lives in the oracle and, separately, in the library).  It only draws random scene
parameters and builds the *inputs* the C-ABI takes:

* surfels: ``means[N,3] quats[N,4] (w,x,y,z) scales[N,2] opacity_logits[N] rgb[N,3]`` fp32
* per view: a 2x4 affine camera ``F`` (world metres -> pixel coordinates), a 2x4 delta ``dF``,
  the viewing direction, ``b_z`` (max_altitude of PAPER.md Eq. 11), a background depth,
  the 3x4 colour correction, the ambient light, and the sun angles + viewport of the
  sun-direction camera (the camera itself is built by the code under test).
* upstream gradients ~ N(0,1) per output channel.

The paper measures on DFC2019 / IARPA2016 sites; those are not available here.
The scenes below copy their *shape* only: ~2.5-D urban height fields at 0.3-0.5 m/px, near-nadir
affine views, 1K-4M surfels.  Configs are numbered C0..C4 as in BASELINE.json (zero based).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

__all__ = ["Scene", "View", "make_config", "upstream_grads", "affine_camera", "CONFIG_NAMES"]

CONFIG_NAMES = {
    0: "C0 tiny correctness scene (1,024 surfels, 128x128)",
    1: "C1 single-site DSM (200k surfels, 10x 512x512)",
    2: "C2 shadow pass on C1 (sun map 1024x1024)",
    3: "C3 benchmark-shaped site (1M surfels, 2048x2048, shadows)",
    4: "C4 large-scene stress (4M surfels, 4096x4096)",
}


@dataclass
class View:
    width: int
    height: int
    F: np.ndarray          # [8] fp32, 2x4 row-major [B_xy | b_xy], world -> pixel
    dF: np.ndarray         # [8] fp32
    view_dir: np.ndarray   # [3] fp32, unit, sensor -> scene
    b_z: float             # max_altitude (Eq. 11); depth z = b_z - world_z
    z_bg: float            # background depth
    bg_rgb: np.ndarray     # [3] fp32
    cc: np.ndarray         # [12] fp32, 3x4 [C | c]
    ambient: np.ndarray    # [3] fp32
    shadows_on: bool = False
    sun_azimuth: float = 0.0     # radians, from +X toward +Y
    sun_elevation: float = 1.0   # radians above the horizon
    sun_width: int = 0
    sun_height: int = 0
    sun_viewport: np.ndarray = field(default_factory=lambda: np.array([1, 1, 0, 0], np.float32))
    depth_bias: float = 0.5
    slope: float = 4.0
    gsd: float = 0.5
    off_nadir: float = 0.0


@dataclass
class Scene:
    name: str
    means: np.ndarray
    quats: np.ndarray
    scales: np.ndarray
    opacity_logits: np.ndarray
    rgb: np.ndarray
    views: list
    seed: int

    @property
    def n(self) -> int:
        return int(self.means.shape[0])


# --------------------------------------------------------------------------------------
# cameras (input construction only: an affine camera from GSD / off-nadir / azimuth)
# --------------------------------------------------------------------------------------
def affine_camera(gsd, off_nadir, azimuth, width, height, look_at):
    """2x4 affine camera mapping world metres to pixel coordinates (pixel (i,j) centre at
    (i+.5, j+.5), x right, y down).  d = viewing direction (sensor -> scene)."""
    th, ps = float(off_nadir), float(azimuth)
    d = np.array([math.sin(th) * math.cos(ps), math.sin(th) * math.sin(ps), -math.cos(th)])
    yhat = np.array([0.0, 1.0, 0.0])
    e_up = yhat - yhat.dot(d) * d
    e_up /= np.linalg.norm(e_up)
    e_r = np.cross(d, e_up)
    p0 = np.asarray(look_at, np.float64)
    F = np.zeros((2, 4))
    F[0, :3] = e_r / gsd
    F[0, 3] = width / 2 - e_r.dot(p0) / gsd
    F[1, :3] = -e_up / gsd
    F[1, 3] = height / 2 + e_up.dot(p0) / gsd
    return F.astype(np.float32).reshape(8), d.astype(np.float32)


def _quat_from_frames(tu, tv, n):
    """Rotation matrices with columns (tu, tv, n) -> unit quaternions (w,x,y,z). Vectorised
    Shepperd's method."""
    m00, m10, m20 = tu[:, 0], tu[:, 1], tu[:, 2]
    m01, m11, m21 = tv[:, 0], tv[:, 1], tv[:, 2]
    m02, m12, m22 = n[:, 0], n[:, 1], n[:, 2]
    tr = m00 + m11 + m22
    q = np.zeros((tu.shape[0], 4))
    c0 = tr > 0
    c1 = (~c0) & (m00 >= m11) & (m00 >= m22)
    c2 = (~c0) & (~c1) & (m11 >= m22)
    c3 = (~c0) & (~c1) & (~c2)
    with np.errstate(invalid="ignore"):
        s = np.sqrt(np.maximum(tr + 1.0, 1e-30)) * 2
        q[c0] = np.stack([0.25 * s, (m21 - m12) / s, (m02 - m20) / s, (m10 - m01) / s], 1)[c0]
        s = np.sqrt(np.maximum(1.0 + m00 - m11 - m22, 1e-30)) * 2
        q[c1] = np.stack([(m21 - m12) / s, 0.25 * s, (m01 + m10) / s, (m02 + m20) / s], 1)[c1]
        s = np.sqrt(np.maximum(1.0 + m11 - m00 - m22, 1e-30)) * 2
        q[c2] = np.stack([(m02 - m20) / s, (m01 + m10) / s, 0.25 * s, (m12 + m21) / s], 1)[c2]
        s = np.sqrt(np.maximum(1.0 + m22 - m00 - m11, 1e-30)) * 2
        q[c3] = np.stack([(m10 - m01) / s, (m02 + m20) / s, (m12 + m21) / s, 0.25 * s], 1)[c3]
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    return q


def _frames_from_normals(rng, n):
    """Orthonormal tangents by Gram-Schmidt against a reference axis, then a
    random in-plane rotation."""
    n = n / np.linalg.norm(n, axis=1, keepdims=True)
    ref = np.tile(np.array([1.0, 0.0, 0.0]), (n.shape[0], 1))
    bad = np.abs(n[:, 0]) > 0.9
    ref[bad] = np.array([0.0, 1.0, 0.0])
    tu = ref - (ref * n).sum(1, keepdims=True) * n
    tu /= np.linalg.norm(tu, axis=1, keepdims=True)
    tv = np.cross(n, tu)
    ang = rng.uniform(0, 2 * math.pi, n.shape[0])
    ca, sa = np.cos(ang)[:, None], np.sin(ang)[:, None]
    tu2 = ca * tu + sa * tv
    tv2 = -sa * tu + ca * tv
    return tu2, tv2, n


# --------------------------------------------------------------------------------------
# height fields
# --------------------------------------------------------------------------------------
def _lowpass_noise(rng, cells, sigma_cells, amp):
    """N(0, amp) low-frequency relief: coarse white noise, bilinearly upsampled."""
    coarse_n = max(4, int(math.ceil(cells / max(sigma_cells, 1.0))) + 3)
    coarse = rng.normal(0, 1, (coarse_n, coarse_n))
    # smooth the coarse grid a little (3x3 box) so that the relief is gentle
    pad = np.pad(coarse, 1, mode="edge")
    coarse = sum(pad[i:i + coarse_n, j:j + coarse_n] for i in range(3) for j in range(3)) / 9.0
    coarse *= amp / max(coarse.std(), 1e-9)
    t = np.linspace(0, coarse_n - 1.001, cells)
    i0 = np.floor(t).astype(int)
    f = t - i0
    rows = coarse[i0] * (1 - f)[:, None] + coarse[i0 + 1] * f[:, None]
    out = rows[:, i0] * (1 - f)[None, :] + rows[:, i0 + 1] * f[None, :]
    return out


def _heightfield(rng, cells, cell, n_buildings, side_rng, height_rng, relief_amp, gabled):
    h = np.zeros((cells, cells))
    if relief_amp > 0:
        h += _lowpass_noise(rng, cells, 100.0 / cell, relief_amp)
    extent = cells * cell
    yy, xx = np.meshgrid(np.arange(cells), np.arange(cells), indexing="ij")
    del yy, xx
    for _ in range(n_buildings):
        sx, sy = rng.uniform(*side_rng, 2)
        cx, cy = rng.uniform(0.05 * extent, 0.95 * extent, 2)
        ht = rng.uniform(*height_rng)
        x0, x1 = int(max(0, (cx - sx / 2) / cell)), int(min(cells, (cx + sx / 2) / cell))
        y0, y1 = int(max(0, (cy - sy / 2) / cell)), int(min(cells, (cy + sy / 2) / cell))
        if x1 <= x0 or y1 <= y0:
            continue
        base = h[y0:y1, x0:x1].min()
        roof = np.full((y1 - y0, x1 - x0), base + ht)
        if gabled and rng.uniform() < 0.5:
            # gabled roof: ridge along x, pitch 20-35 degrees
            pitch = math.tan(rng.uniform(math.radians(20), math.radians(35)))
            yv = (np.arange(y0, y1) + 0.5) * cell
            rise = (sy / 2 - np.abs(yv - cy)) * pitch
            roof = roof + np.maximum(rise, 0.0)[:, None]
        h[y0:y1, x0:x1] = np.maximum(h[y0:y1, x0:x1], roof)
    return h


def _sample_heightfield(rng, h, cell, n, z_noise=0.0):
    """Area-weighted sampling of surfel centres on a 2.5-D height field:
    weight = |dx x dy| from finite differences; wall samples get z uniform between the low and
    high neighbour; normals from central differences."""
    cells = h.shape[0]
    gy, gx = np.gradient(h, cell)
    area = np.sqrt(1.0 + gx * gx + gy * gy)
    p = (area / area.sum()).ravel()
    cdf = np.cumsum(p)
    cdf /= cdf[-1]
    idx = np.searchsorted(cdf, rng.uniform(0, 1, n), side="right")
    idx = np.minimum(idx, cells * cells - 1)
    iy, ix = np.divmod(idx, cells)
    jx, jy = rng.uniform(0, 1, n), rng.uniform(0, 1, n)
    x = (ix + jx) * cell
    y = (iy + jy) * cell
    # local min / max over the 3x3 neighbourhood to spread wall samples vertically
    pad = np.pad(h, 1, mode="edge")
    lo = np.full_like(h, np.inf)
    hi = np.full_like(h, -np.inf)
    for di in range(3):
        for dj in range(3):
            w = pad[di:di + cells, dj:dj + cells]
            lo = np.minimum(lo, w)
            hi = np.maximum(hi, w)
    steep = (area > 2.0)[iy, ix]
    z = h[iy, ix].copy()
    zu = rng.uniform(0, 1, n)
    z[steep] = (lo[iy, ix] + zu * (hi[iy, ix] - lo[iy, ix]))[steep]
    nrm = np.stack([-gx[iy, ix], -gy[iy, ix], np.ones(n)], 1)
    if z_noise > 0:
        z = z + rng.normal(0, z_noise, n)
    return np.stack([x, y, z], 1), nrm


# --------------------------------------------------------------------------------------
# view lists
# --------------------------------------------------------------------------------------
def _make_views(rng, n_views, size, extent, look_at, off_nadir_rng, z_lo, z_hi, *, delta_sigma,
                cc_sigma, shadows, sun_size, sun_el_rng, fill=1.15, ambient=(0.3, 0.35, 0.45)):
    views = []
    gsd = extent * fill / size
    b_z = float(np.float32(z_hi + 10.0))
    z_bg = float(np.float32(b_z - (z_lo - 1.0)))
    habs = max(abs(z_lo), abs(z_hi)) + 1.0
    for _ in range(n_views):
        th = math.radians(rng.uniform(*off_nadir_rng))
        ps = rng.uniform(0, 2 * math.pi)
        F, d = affine_camera(gsd, th, ps, size, size, look_at)
        dF = np.zeros(8, np.float32)
        if delta_sigma > 0:
            # ~delta_sigma relative perturbation: the 2x3 part is in px/m, so scale by 1/gsd;
            # the offset column is in pixels (PAPER.md:269 noise recipe, Frobenius-scaled)
            noise = rng.normal(0, delta_sigma, (2, 4))
            noise[:, :3] /= gsd
            noise[:, 3] *= size * 0.5 * 0.1
            dF = noise.astype(np.float32).reshape(8)
        cc = np.concatenate([np.eye(3), np.zeros((3, 1))], 1)
        if cc_sigma > 0:
            cc = cc + rng.normal(0, cc_sigma, (3, 4))
        v = View(width=size, height=size, F=F, dF=dF, view_dir=d, b_z=b_z, z_bg=z_bg,
                 bg_rgb=np.zeros(3, np.float32), cc=cc.astype(np.float32).reshape(12),
                 ambient=np.asarray(ambient, np.float32), gsd=gsd, off_nadir=th)
        if shadows:
            el = math.radians(rng.uniform(*sun_el_rng))
            az = rng.uniform(0, 2 * math.pi)
            # viewport: uniform scale + shift so that the view frame, grown by the largest
            # horizontal displacement a point of height |h| can get (sun flattening + parallax),
            # fits the sun map.  Anything that still falls outside is treated as lit.
            margin_px = habs * (1.0 / math.tan(el) + math.tan(th) + 0.1) / gsd
            sc = sun_size / (size + 2.0 * margin_px)
            v.shadows_on = True
            v.sun_azimuth, v.sun_elevation = az, el
            v.sun_width = v.sun_height = sun_size
            v.sun_viewport = np.array([sc, sc, margin_px * sc, margin_px * sc], np.float32)
        views.append(v)
    return views


# --------------------------------------------------------------------------------------
# configs
# --------------------------------------------------------------------------------------
def _c0(seed=0, n=1024, size=128):
    rng = np.random.default_rng(seed)
    xy = rng.uniform(0, 64, (n, 2))
    z = rng.normal(0, 2, n)
    means = np.concatenate([xy, z[:, None]], 1)
    # 90 %: near-horizontal surfels (normal ~ +z); 10 %: facade-like (normal near the horizon)
    nrm = np.array([0, 0, 1.0]) + 0.35 * rng.normal(0, 1, (n, 3))
    facade = rng.uniform(0, 1, n) < 0.10
    phi = rng.uniform(0, 2 * math.pi, n)
    nf = np.stack([np.cos(phi), np.sin(phi), 0.15 * rng.normal(0, 1, n)], 1)
    nrm[facade] = nf[facade]
    tu, tv, nn = _frames_from_normals(rng, nrm)
    quats = _quat_from_frames(tu, tv, nn)
    scales = np.exp(rng.uniform(math.log(0.1), math.log(1.0), (n, 2)))
    logits = rng.normal(0, 1, n)
    rgb = rng.uniform(0, 1, (n, 3))
    gsd = 0.5
    F, d = affine_camera(gsd, math.radians(15.0), 0.0, size, size, (32.0, 32.0, 0.0))
    b_z = float(np.float32(z.max() + 10.0))
    z_bg = float(np.float32(b_z - (z.min() - 1.0)))
    cc = np.concatenate([np.eye(3), np.zeros((3, 1))], 1).astype(np.float32).reshape(12)
    view = View(width=size, height=size, F=F, dF=np.zeros(8, np.float32), view_dir=d, b_z=b_z,
                z_bg=z_bg, bg_rgb=np.zeros(3, np.float32), cc=cc,
                ambient=np.array([0.3, 0.35, 0.45], np.float32), gsd=gsd,
                off_nadir=math.radians(15.0))
    return _pack("C0", seed, means, quats, scales, logits, rgb, [view])


def _dsm_site(name, seed, *, extent, cell, n_buildings, side_rng, height_rng, relief_amp, gabled,
              n, scale_rng, log_scales, z_noise, n_views, size, off_nadir_rng, delta_sigma,
              cc_sigma, shadows, sun_size, sun_el_rng, big_tail=0.0, big_rng=(10.0, 40.0), fill=1.15):
    rng = np.random.default_rng(seed)
    cells = int(round(extent / cell))
    h = _heightfield(rng, cells, cell, n_buildings, side_rng, height_rng, relief_amp, gabled)
    means, nrm = _sample_heightfield(rng, h, cell, n, z_noise)
    tu, tv, nn = _frames_from_normals(rng, nrm)
    quats = _quat_from_frames(tu, tv, nn)
    if log_scales:
        scales = np.exp(rng.uniform(math.log(scale_rng[0]), math.log(scale_rng[1]), (n, 2)))
    else:
        scales = rng.uniform(scale_rng[0], scale_rng[1], (n, 2))
    if big_tail > 0:
        nb = int(round(n * big_tail))
        sel = rng.choice(n, nb, replace=False)
        scales[sel] = np.exp(rng.uniform(math.log(big_rng[0]), math.log(big_rng[1]), (nb, 2)))
    logits = 2.0 + rng.normal(0, 0.5, n)
    rgb = rng.uniform(0.1, 0.9, (n, 3))
    z_lo, z_hi = float(means[:, 2].min()), float(means[:, 2].max())
    look_at = (extent / 2, extent / 2, 0.0)
    views = _make_views(rng, n_views, size, extent, look_at, off_nadir_rng, z_lo, z_hi,
                        delta_sigma=delta_sigma, cc_sigma=cc_sigma, shadows=shadows,
                        sun_size=sun_size, sun_el_rng=sun_el_rng, fill=fill)
    return _pack(name, seed, means, quats, scales, logits, rgb, views)


def _pack(name, seed, means, quats, scales, logits, rgb, views):
    f = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    return Scene(name=name, seed=seed, means=f(means), quats=f(quats), scales=f(scales),
                 opacity_logits=f(logits), rgb=f(rgb), views=views)


def make_config(cfg: int, *, n=None, size=None, n_views=None, sun_size=None, seed=None,
                extent=None) -> Scene:
    """Build config C<cfg>.  The keyword overrides shrink a config for tests (same generator,
    same distributions, fewer surfels / pixels / views)."""
    if cfg == 0:
        return _c0(seed=0 if seed is None else seed, n=n or 1024, size=size or 128)
    if cfg in (1, 2):
        return _dsm_site(f"C{cfg}", 1 if seed is None else seed, extent=extent or 128.0, cell=0.5,
                         n_buildings=30, side_rng=(6.0, 30.0), height_rng=(5.0, 40.0),
                         relief_amp=0.0, gabled=False, n=n or 200_000, scale_rng=(0.25, 1.0),
                         log_scales=False, z_noise=0.0, n_views=n_views or 10, size=size or 512,
                         off_nadir_rng=(5.0, 30.0), delta_sigma=1e-3, cc_sigma=0.05,
                         shadows=(cfg == 2), sun_size=sun_size or 1024, sun_el_rng=(30.0, 70.0))
    if cfg == 3:
        return _dsm_site("C3", 3 if seed is None else seed, extent=extent or 1000.0, cell=0.3,
                         n_buildings=400, side_rng=(8.0, 60.0), height_rng=(3.0, 60.0),
                         relief_amp=3.0, gabled=True, n=n or 1_000_000, scale_rng=(0.35, 1.0),
                         log_scales=True, z_noise=1.5, n_views=n_views or 20, size=size or 2048,
                         off_nadir_rng=(5.0, 35.0), delta_sigma=1e-3, cc_sigma=0.05, shadows=True,
                         sun_size=sun_size or 2048, sun_el_rng=(25.0, 70.0), fill=1.0)
    if cfg == 4:
        return _dsm_site("C4", 4 if seed is None else seed, extent=extent or 2000.0, cell=0.3,
                         n_buildings=1600, side_rng=(8.0, 60.0), height_rng=(3.0, 60.0),
                         relief_amp=3.0, gabled=True, n=n or 4_000_000, scale_rng=(0.2, 3.0),
                         log_scales=True, z_noise=1.5, n_views=n_views or 4, size=size or 4096,
                         off_nadir_rng=(5.0, 35.0), delta_sigma=1e-3, cc_sigma=0.05, shadows=False,
                         sun_size=sun_size or 4096, sun_el_rng=(25.0, 70.0), big_tail=0.001,
                         fill=1.0)
    raise ValueError(f"unknown config {cfg}")


def upstream_grads(scene_seed: int, view_index: int, height: int, width: int):
    """Upstream gradients ~ N(0,1) per output channel, in the library's image layouts:
    v_rgba [H,W,4] (dI rgb, dA), v_geom [H,W,4] (dN xyz, dD), v_aux [H,W,4] (dmedian, ddistortion,
    0, 0)."""
    rng = np.random.default_rng(scene_seed + 1000 + 7919 * view_index)
    v_rgba = rng.normal(0, 1, (height, width, 4)).astype(np.float32)
    v_geom = rng.normal(0, 1, (height, width, 4)).astype(np.float32)
    v_aux = rng.normal(0, 1, (height, width, 4)).astype(np.float32)
    v_aux[..., 2:] = 0
    return v_rgba, v_geom, v_aux


def sun_depth_upstream(scene_seed: int, view_index: int, height: int, width: int):
    rng = np.random.default_rng(scene_seed + 2000 + 7919 * view_index)
    return rng.normal(0, 1, (height, width)).astype(np.float32)

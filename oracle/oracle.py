"""ctypes binding of the CPU oracle (oracle/satsplat_oracle.cpp).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
``--impl reference`` legs.  Never imported by the product package ``paper_2606_28581_b200``, and it
imports nothing from it.  The arithmetic lives in the C++ file; this module only marshals numpy arrays,
sums tile counts, orders surfels for the all-pairs list, and strings the stages together in the order
of PAPER.md Fig. 1 (sun pass -> view pass -> Eq. 1).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "satsplat_oracle.cpp")
_SO = os.path.join(_HERE, "libsatsplat_oracle.so")
_LOCK = threading.Lock()
_LIB = None

OPT_NO_RHO_CUT, OPT_NO_ALPHA_SKIP, OPT_NO_T_STOP = 1, 2, 4
F_CULLED, F_DEGENERATE, F_FLIPPED = 1, 2, 4
REC = dict(cx=0, cy=1, q00=2, q01=3, q10=4, q11=5, zc=6, g0=7, g1=8, alpha=9, r=10, g=11, b=12, nx=13, ny=14, nz=15)
TILE = 16


def _compile(out: str, opt: list) -> None:
    tmp = out + f".tmp{os.getpid()}"
    cmd = ["g++", *opt, "-std=c++17", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC", _SRC, "-o", tmp]
    subprocess.run(cmd, check=True)
    os.replace(tmp, out)


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it).  Portable -O2 build: the .so travels."""
    with _LOCK:
        if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
            _compile(_SO, ["-O2"])
    return _SO


def use_native_build() -> str:
    """The timed baseline's build (-O3 -march=native -ffp-contract=off), compiled ON the host it
    runs on (the file name carries the host's CPU model, so a copy made on another machine is never loaded).  Same
    source, same arithmetic (no fast-math, no contraction); only bench.py's CPU legs switch to it, before first use."""
    global _LIB
    import hashlib
    import platform
    model = platform.machine()
    try:
        with open("/proc/cpuinfo") as f:
            model += "".join(l for l in f if l.startswith(("model name", "flags")))[:20000]
    except OSError:
        pass
    so = os.path.join(_HERE, f"libsatsplat_oracle_native_{hashlib.sha1(model.encode()).hexdigest()[:10]}.so")
    with _LOCK:
        if not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(_SRC):
            _compile(so, ["-O3", "-march=native"])
        _LIB = None
    lib(so)
    return so


class _CamF32(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("F", C.c_float * 8), ("dF", C.c_float * 8),
                ("view_dir", C.c_float * 3), ("b_z", C.c_float)]


class _CamF64(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("F", C.c_double * 8), ("dF", C.c_double * 8),
                ("view_dir", C.c_double * 3), ("b_z", C.c_double)]


class _Shading(C.Structure):
    _fields_ = [("cc", C.c_double * 12), ("ambient", C.c_double * 3), ("shadows_on", C.c_int32),
                ("sun_w", C.c_int32), ("sun_h", C.c_int32), ("_pad", C.c_int32), ("sun_depth", C.c_void_p),
                ("reproj", C.c_double * 8), ("bias", C.c_double), ("slope", C.c_double)]


class _Render(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("b_z", C.c_double), ("z_bg", C.c_double),
                ("bg", C.c_double * 3), ("tile_mode", C.c_int32), ("tiles_x", C.c_int32), ("vals", C.c_void_p),
                ("ranges", C.c_void_p), ("list_len", C.c_int64), ("options", C.c_int32), ("threads", C.c_int32)]


def lib(path: str = None):
    global _LIB
    if _LIB is None:
        _LIB = C.CDLL(path or build())
        for name in ("orc_preprocess_f32", "orc_preprocess_f64", "orc_bin", "orc_forward", "orc_backward",
                     "orc_preprocess_backward", "orc_sun_camera", "orc_sun_camera_backward", "orc_nearby_camera",
                     "orc_nearby_camera_backward", "orc_num_threads"):
            getattr(_LIB, name).restype = C.c_int
    return _LIB


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def num_threads() -> int:
    return int(lib().orc_num_threads())


# ------------------------------------------------------------------------------------------------
# stage wrappers
# ------------------------------------------------------------------------------------------------
def _cam32(view):
    c = _CamF32()
    c.width, c.height = int(view.width), int(view.height)
    c.F[:] = [float(x) for x in _f32(view.F)]
    c.dF[:] = [float(x) for x in _f32(view.dF)]
    c.view_dir[:] = [float(x) for x in _f32(view.view_dir)]
    c.b_z = float(np.float32(view.b_z))
    return c


def _cam64(view, F=None, dF=None):
    c = _CamF64()
    c.width, c.height = int(view.width), int(view.height)
    c.F[:] = [float(x) for x in (view.F if F is None else F)]
    c.dF[:] = [float(x) for x in (view.dF if dF is None else dF)]
    c.view_dir[:] = [float(x) for x in view.view_dir]
    c.b_z = float(view.b_z)
    return c


def preprocess_f32(view, means, quats, scales, logits, rgb):
    """Binning contract (fp32 op sequence).  Returns record [N,16] f32, rect [N,4] i32 (tx0,ty0,tx1,ty1),
    count [N] u32, depth_key [N] u32, flags [N] u8."""
    n = means.shape[0]
    rec = np.zeros((n, 16), np.float32)
    rect = np.zeros((n, 4), np.int32)
    count = np.zeros(n, np.uint32)
    key = np.zeros(n, np.uint32)
    flags = np.zeros(n, np.uint8)
    cam = _cam32(view)
    rc = lib().orc_preprocess_f32(C.byref(cam), C.c_int64(n), _p(_f32(means)), _p(_f32(quats)), _p(_f32(scales)),
                                  _p(_f32(logits)), _p(_f32(rgb)), _p(rec), _p(rect), _p(count), _p(key), _p(flags))
    assert rc == 0
    return dict(rec=rec, rect=rect, count=count, depth_key=key, flags=flags)


def preprocess_f64(view, means, quats, scales, logits, rgb, F=None, dF=None):
    n = means.shape[0]
    rec = np.zeros((n, 16), np.float64)
    flags = np.zeros(n, np.uint8)
    cam = _cam64(view, F, dF)
    rc = lib().orc_preprocess_f64(C.byref(cam), C.c_int64(n), _p(_f64(means)), _p(_f64(quats)), _p(_f64(scales)),
                                  _p(_f64(logits)), _p(_f64(rgb)), _p(rec), _p(flags))
    assert rc == 0
    return dict(rec=rec, flags=flags)


def bin_tiles(width, height, rect, count, depth_key):
    """Reference binning: keys [K] u64 = (tile << 32) | depth_key, vals [K] u32, ranges [tiles,2] u32."""
    tx, ty = (width + TILE - 1) // TILE, (height + TILE - 1) // TILE
    k = int(count.astype(np.int64).sum())
    keys = np.zeros(k, np.uint64)
    vals = np.zeros(k, np.uint32)
    ranges = np.zeros((tx * ty, 2), np.uint32)
    rc = lib().orc_bin(C.c_int64(rect.shape[0]), C.c_int32(tx), C.c_int32(ty), _p(rect), _p(count), _p(depth_key),
                       C.c_int64(k), _p(keys), _p(vals), _p(ranges))
    assert rc == 0
    return keys, vals, ranges


def global_order(depth_key, flags):
    """All-pairs list: every non-culled surfel in (depth key, index) order."""
    idx = np.nonzero((flags & F_CULLED) == 0)[0]
    order = idx[np.argsort(depth_key[idx], kind="stable")]
    return order.astype(np.uint32)


class Shading:
    """Eq. 1 inputs + the shadow test inputs (reading 12/13)."""

    def __init__(self, cc=None, ambient=(0, 0, 0), sun_depth=None, reproj=None, bias=0.5, slope=4.0):
        self.cc = _f64(np.concatenate([np.eye(3), np.zeros((3, 1))], 1).reshape(12) if cc is None else cc)
        self.ambient = _f64(ambient)
        self.sun_depth = None if sun_depth is None else _f64(sun_depth)
        self.reproj = _f64(np.zeros(8) if reproj is None else reproj)
        self.bias, self.slope = float(bias), float(slope)

    def c(self):
        s = _Shading()
        s.cc[:] = list(self.cc)
        s.ambient[:] = list(self.ambient)
        s.shadows_on = 0 if self.sun_depth is None else 1
        if self.sun_depth is not None:
            s.sun_h, s.sun_w = self.sun_depth.shape
            s.sun_depth = self.sun_depth.ctypes.data
        s.reproj[:] = list(self.reproj)
        s.bias, s.slope = self.bias, self.slope
        return s


def _render_cfg(width, height, b_z, z_bg, bg, lists, options, threads):
    r = _Render()
    r.width, r.height = int(width), int(height)
    r.b_z, r.z_bg = float(b_z), float(z_bg)
    r.bg[:] = [float(x) for x in bg]
    r.options, r.threads = int(options), int(threads)
    keep = []
    if isinstance(lists, tuple):  # (vals, ranges): per-tile lists
        vals, ranges = lists
        vals = np.ascontiguousarray(vals, np.uint32)
        ranges = np.ascontiguousarray(ranges, np.uint32)
        r.tile_mode, r.tiles_x = 1, (int(width) + TILE - 1) // TILE
        r.vals, r.ranges = vals.ctypes.data, ranges.ctypes.data
        keep = [vals, ranges]
    else:  # one global list
        vals = np.ascontiguousarray(lists, np.uint32)
        r.tile_mode, r.tiles_x = 0, 0
        r.vals, r.list_len = vals.ctypes.data, int(vals.shape[0])
        keep = [vals]
    return r, keep


def forward(width, height, b_z, z_bg, bg, rec, flags, lists, shading: Shading, options=0, threads=1):
    """Per-pixel compositing (step C) + Eq. 1 epilogue (step D).  `lists` is either a uint32 array (one
    global list, all-pairs mode) or (vals, ranges) (per-tile lists)."""
    cfg, keep = _render_cfg(width, height, b_z, z_bg, bg, lists, options, threads)
    rec = _f64(rec)
    flags = np.ascontiguousarray(flags, np.uint8)
    H, W = int(height), int(width)
    out = dict(rgba=np.zeros((H, W, 4)), geom=np.zeros((H, W, 4)), aux=np.zeros((H, W, 4)),
               albedo=np.zeros((H, W, 3)), last=np.zeros((H, W), np.int32), med_idx=np.zeros((H, W), np.int32),
               margins=np.zeros((H, W, 6)), counters=np.zeros(5, np.int64))
    sh = shading.c()
    rc = lib().orc_forward(C.byref(cfg), C.byref(sh), _p(rec), _p(flags), _p(out["rgba"]), _p(out["geom"]),
                           _p(out["aux"]), _p(out["albedo"]), _p(out["last"]), _p(out["med_idx"]),
                           _p(out["margins"]), _p(out["counters"]))
    assert rc == 0
    del keep
    return out


def backward(width, height, b_z, z_bg, bg, rec, flags, lists, shading: Shading, v_rgba, v_geom, v_aux,
             options=0, threads=1, twin=False):
    """Analytic backward (step E) of epilogue + compositor.  Returns v_rec [N,16], v_cc [12], v_ambient [3],
    v_reproj [8], v_sun_depth [Hs,Ws] or None.  `twin`: also the absolute-value twins a_* of the same sums (the
    rounding-error scale of every gradient value, see orc_backward)."""
    cfg, keep = _render_cfg(width, height, b_z, z_bg, bg, lists, options, threads)
    rec = _f64(rec)
    flags = np.ascontiguousarray(flags, np.uint8)
    v_rec = np.zeros_like(rec)
    v_cc, v_amb, v_rep = np.zeros(12), np.zeros(3), np.zeros(8)
    v_sun = None if shading.sun_depth is None else np.zeros_like(shading.sun_depth)
    sh = shading.c()
    a = [None if x is None else _f64(x) for x in (v_rgba, v_geom, v_aux)]
    tw = dict(a_rec=None, a_cc=None, a_ambient=None, a_reproj=None, a_sun_depth=None)
    if twin:
        tw = dict(a_rec=np.zeros_like(rec), a_cc=np.zeros(12), a_ambient=np.zeros(3), a_reproj=np.zeros(8),
                  a_sun_depth=None if v_sun is None else np.zeros_like(v_sun))
    rc = lib().orc_backward(C.byref(cfg), C.byref(sh), _p(rec), _p(flags), _p(a[0]), _p(a[1]), _p(a[2]), _p(v_rec),
                            _p(v_cc), _p(v_amb), _p(v_rep), _p(v_sun), _p(tw["a_rec"]), _p(tw["a_cc"]), _p(tw["a_ambient"]),
                            _p(tw["a_reproj"]), _p(tw["a_sun_depth"]))
    assert rc == 0
    del keep
    out = dict(v_rec=v_rec, v_cc=v_cc, v_ambient=v_amb, v_reproj=v_rep, v_sun_depth=v_sun)
    if twin:
        out.update(tw)
    return out


def preprocess_backward(view, means, quats, scales, logits, flags, v_rec, F=None, dF=None, a_rec=None):
    """Per-surfel chain.  With `a_rec` (the twin of v_rec from backward(twin=True)) also returns the twins a_means,
    a_quats, a_scales, a_logits, a_rgb, a_dF."""
    n = means.shape[0]
    out = dict(v_means=np.zeros((n, 3)), v_quats=np.zeros((n, 4)), v_scales=np.zeros((n, 2)), v_logits=np.zeros(n),
               v_rgb=np.zeros((n, 3)), v_dF=np.zeros(8))
    tw = dict(a_means=None, a_quats=None, a_scales=None, a_logits=None, a_rgb=None, a_dF=None)
    if a_rec is not None:
        a_rec = _f64(a_rec)
        tw = dict(a_means=np.zeros((n, 3)), a_quats=np.zeros((n, 4)), a_scales=np.zeros((n, 2)), a_logits=np.zeros(n),
                  a_rgb=np.zeros((n, 3)), a_dF=np.zeros(8))
    cam = _cam64(view, F, dF)
    rc = lib().orc_preprocess_backward(C.byref(cam), C.c_int64(n), _p(_f64(means)), _p(_f64(quats)), _p(_f64(scales)),
                                       _p(_f64(logits)), _p(np.ascontiguousarray(flags, np.uint8)), _p(_f64(v_rec)),
                                       _p(out["v_means"]), _p(out["v_quats"]), _p(out["v_scales"]),
                                       _p(out["v_logits"]), _p(out["v_rgb"]), _p(out["v_dF"]), _p(a_rec),
                                       _p(tw["a_means"]), _p(tw["a_quats"]), _p(tw["a_scales"]), _p(tw["a_logits"]),
                                       _p(tw["a_rgb"]), _p(tw["a_dF"]))
    assert rc == 0
    if a_rec is not None:
        out.update(tw)
    return out


def sun_camera(Fp, azimuth, elevation, viewport):
    """Eq. 16 / S1-S4 + viewport.  Fp = F + dF (2x4).  Returns F_sun [8], reproj [8] (double)."""
    F_sun, reproj = np.zeros(8), np.zeros(8)
    rc = lib().orc_sun_camera(_p(_f64(Fp)), C.c_double(azimuth), C.c_double(elevation), _p(_f64(viewport)),
                              _p(F_sun), _p(reproj))
    assert rc == 0
    return F_sun, reproj


def sun_camera_backward(Fp, azimuth, elevation, viewport, v_F_sun, v_reproj):
    """Adjoint of sun_camera with respect to Fp = F + dF (= the gradient that reaches dF through the cascade,
    PAPER.md:155-176).  Returns v_Fp [8] (double)."""
    v_Fp = np.zeros(8)
    rc = lib().orc_sun_camera_backward(_p(_f64(Fp)), C.c_double(azimuth), C.c_double(elevation), _p(_f64(viewport)),
                                       _p(_f64(v_F_sun)), _p(_f64(v_reproj)), _p(v_Fp))
    assert rc == 0
    return v_Fp


def nearby_camera(Fp, d_azimuth, d_elevation):
    """Nearby camera of PAPER.md:176: azimuth / elevation of d_main = B_x x B_y perturbed, then Eq. 16.  Returns
    F_near [8] and (azimuth, elevation) of the main direction (double)."""
    F_near, ang = np.zeros(8), np.zeros(2)
    rc = lib().orc_nearby_camera(_p(_f64(Fp)), C.c_double(d_azimuth), C.c_double(d_elevation), _p(F_near), _p(ang))
    assert rc == 0
    return F_near, ang


def nearby_camera_backward(Fp, d_azimuth, d_elevation, v_F_near):
    """Adjoint of nearby_camera with respect to Fp.  Returns v_Fp [8] (double)."""
    v_Fp = np.zeros(8)
    rc = lib().orc_nearby_camera_backward(_p(_f64(Fp)), C.c_double(d_azimuth), C.c_double(d_elevation), _p(_f64(v_F_near)), _p(v_Fp))
    assert rc == 0
    return v_Fp


# ------------------------------------------------------------------------------------------------
# one full view iteration, in the order of PAPER.md Fig. 1: sun pass (depth) -> view pass -> Eq. 1 ->
# backward through Eq. 1, both passes and both per-surfel chains.
# ------------------------------------------------------------------------------------------------
class SunView:
    """The sun-direction camera of a view as a plain camera (inputs of the sun pass)."""

    def __init__(self, view, F_sun_f32):
        self.width, self.height = view.sun_width, view.sun_height
        self.F = _f32(F_sun_f32)
        self.dF = np.zeros(8, np.float32)
        # the sun camera's viewing direction is -s (towards the scene); only used for the normal flip
        az, el = view.sun_azimuth, view.sun_elevation
        d = -np.array([np.cos(az) * np.cos(el), np.sin(az) * np.cos(el), np.sin(el)])
        self.view_dir = _f32(d)
        self.b_z, self.z_bg, self.bg_rgb = view.b_z, view.z_bg, np.zeros(3, np.float32)


def sun_inputs(view):
    """fp32 sun camera + reprojection constants for a view (oracle's Eq. 16), as the inputs both the oracle
    and the code under test consume."""
    Fp = (_f32(view.F) + _f32(view.dF)).astype(np.float64)
    F_sun, reproj = sun_camera(Fp, view.sun_azimuth, view.sun_elevation, view.sun_viewport)
    return SunView(view, F_sun.astype(np.float32)), reproj.astype(np.float32)


def render_pass(view, scene, *, tile_mode=True, threads=1):
    """Preprocess (fp32 contract) + binning + lists for one camera.  Returns dict with rec (f64 copy of the
    f32 record), flags, lists, K and the binning arrays."""
    pre = preprocess_f32(view, scene.means, scene.quats, scene.scales, scene.opacity_logits, scene.rgb)
    keys, vals, ranges = bin_tiles(view.width, view.height, pre["rect"], pre["count"], pre["depth_key"])
    lists = (vals, ranges) if tile_mode else global_order(pre["depth_key"], pre["flags"])
    pre.update(keys=keys, vals=vals, ranges=ranges, lists=lists, rec64=pre["rec"].astype(np.float64))
    return pre


def view_iteration(scene, view, upstream=None, sun_upstream=None, *, tile_mode=True, threads=1,
                   do_backward=True, twin=False):
    """Full forward(+backward) of one view with record mode `float` (the fp32 record is the
    interface between preprocess and blend).  Returns a dict of outputs and gradients (all float64)."""
    res = {}
    shading = Shading(cc=view.cc, ambient=view.ambient, bias=view.depth_bias, slope=view.slope)
    sun = None
    if view.shadows_on:
        sun_view, reproj = sun_inputs(view)
        sun = render_pass(sun_view, scene, tile_mode=tile_mode)
        fs = forward(sun_view.width, sun_view.height, sun_view.b_z, sun_view.z_bg, np.zeros(3), sun["rec64"],
                     sun["flags"], sun["lists"], Shading(), threads=threads)
        sun_depth = fs["geom"][..., 3] + fs["aux"][..., 3] * sun_view.z_bg
        # the library hands the sun map over as an fp32 image; the oracle consumes the same precision
        shading = Shading(cc=view.cc, ambient=view.ambient, sun_depth=sun_depth.astype(np.float32),
                          reproj=reproj, bias=view.depth_bias, slope=view.slope)
        res.update(sun_view=sun_view, reproj=reproj, sun_depth=sun_depth, sun_pass=sun, sun_fwd=fs)
    main = render_pass(view, scene, tile_mode=tile_mode)
    fw = forward(view.width, view.height, view.b_z, view.z_bg, view.bg_rgb, main["rec64"], main["flags"],
                 main["lists"], shading, threads=threads)
    res.update(main_pass=main, fwd=fw, shading=shading)
    if not do_backward:
        return res
    v_rgba, v_geom, v_aux = upstream
    bw = backward(view.width, view.height, view.b_z, view.z_bg, view.bg_rgb, main["rec64"], main["flags"],
                  main["lists"], shading, v_rgba, v_geom, v_aux, threads=threads, twin=twin)
    g = preprocess_backward(view, scene.means, scene.quats, scene.scales, scene.opacity_logits, main["flags"],
                            bw["v_rec"], a_rec=bw.get("a_rec"))
    res.update(bwd=bw, grads=g)
    if view.shadows_on:
        v_sd = bw["v_sun_depth"]
        if sun_upstream is not None:
            v_sd = v_sd + sun_upstream
        Hs, Ws = v_sd.shape
        vg = np.zeros((Hs, Ws, 4)); vg[..., 3] = v_sd             # sun_depth = D + (1 - A) z_bg
        vr = np.zeros((Hs, Ws, 4)); vr[..., 3] = -sun_view.z_bg * v_sd
        bs = backward(sun_view.width, sun_view.height, sun_view.b_z, sun_view.z_bg, np.zeros(3), sun["rec64"],
                      sun["flags"], sun["lists"], Shading(), vr, vg, None, threads=threads, twin=twin)
        gs = preprocess_backward(sun_view, scene.means, scene.quats, scene.scales, scene.opacity_logits,
                                 sun["flags"], bs["v_rec"], a_rec=bs.get("a_rec"))
        res.update(sun_bwd=bs, sun_grads=gs)
    return res

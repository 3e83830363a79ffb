"""paper_2606_28581_b200 — thin Python binding of libsatsplat.so (the C ABI of include/satsplat.h).

Argument marshalling only: every step of the path runs in the hand-written sm_100a kernels under csrc/.
PyTorch is used for device memory and streams, nothing else.  There is no CPU fallback: if the CUDA library
is missing or fails to load, importing a compute entry point raises.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libsatsplat.so")
_LIB = None

OK, E_INVALID, E_CAPACITY, E_CUDA, E_STATE = 0, -1, -2, -3, -4
OPT_BINNING, BINNING_TILESORT, BINNING_RADIX = 0, 0, 1
OPT_SPLIT_BACKWARD = 1
OPT_DEBUG_PLANES = 2
STAGES = ("preprocess", "scan", "duplicate", "sort", "ranges", "blend_fwd", "blend_bwd", "chain_bwd")


class SatsplatError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"satsplat error {code}: {msg}")
        self.code = code


class Camera(C.Structure):
    """satsplat_camera (include/satsplat.h)."""
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("F", C.c_float * 8), ("dF", C.c_float * 8),
                ("view_dir", C.c_float * 3), ("b_z", C.c_float), ("z_bg", C.c_float), ("bg_rgb", C.c_float * 3)]

    @classmethod
    def make(cls, width, height, F, dF=None, view_dir=(0, 0, -1), b_z=0.0, z_bg=0.0, bg_rgb=(0, 0, 0)):
        c = cls()
        c.width, c.height = int(width), int(height)
        c.F[:] = [float(x) for x in F]
        c.dF[:] = [0.0] * 8 if dF is None else [float(x) for x in dF]
        c.view_dir[:] = [float(x) for x in view_dir]
        c.b_z, c.z_bg = float(b_z), float(z_bg)
        c.bg_rgb[:] = [float(x) for x in bg_rgb]
        return c

    @classmethod
    def from_view(cls, v):
        """From a satsplat_scenes.View-like object (duck typed)."""
        return cls.make(v.width, v.height, v.F, v.dF, v.view_dir, v.b_z, v.z_bg, v.bg_rgb)


class LossWeights(C.Structure):
    """satsplat_loss_weights (include/satsplat.h); 0.8, 0.2, 0.05, 0.05."""
    _fields_ = [("w_l1", C.c_float), ("w_ssim", C.c_float), ("w_dist", C.c_float), ("w_normal", C.c_float)]


class Adam(C.Structure):
    """satsplat_adam (include/satsplat.h): lr in the order means, quats, scales, opacity logits, rgb."""
    _fields_ = [("lr", C.c_float * 5), ("beta1", C.c_float), ("beta2", C.c_float), ("eps", C.c_float), ("step", C.c_int32)]


class CameraAdam(C.Structure):
    """satsplat_camera_adam (include/satsplat.h): lr in the order dF, cc, ambient."""
    _fields_ = [("lr", C.c_float * 3), ("beta1", C.c_float), ("beta2", C.c_float), ("eps", C.c_float)]


class Shading(C.Structure):
    """satsplat_shading (include/satsplat.h)."""
    _fields_ = [("cc", C.c_float * 12), ("ambient", C.c_float * 3), ("shadows_on", C.c_int32),
                ("sun_width", C.c_int32), ("sun_height", C.c_int32), ("sun_depth", C.c_void_p),
                ("reproj", C.c_float * 8), ("depth_bias", C.c_float), ("slope", C.c_float)]

    @classmethod
    def make(cls, cc=None, ambient=(0, 0, 0), sun_depth=None, reproj=None, depth_bias=0.5, slope=4.0):
        s = cls()
        s.cc[:] = [1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0] if cc is None else [float(x) for x in cc]
        s.ambient[:] = [float(x) for x in ambient]
        s.shadows_on = 0
        if sun_depth is not None:
            _check(sun_depth, torch.float32, 2)
            s.shadows_on = 1
            s.sun_height, s.sun_width = int(sun_depth.shape[0]), int(sun_depth.shape[1])
            s.sun_depth = sun_depth.data_ptr()
            s._keep = sun_depth
        s.reproj[:] = [0.0] * 8 if reproj is None else [float(x) for x in reproj]
        s.depth_bias, s.slope = float(depth_bias), float(slope)
        return s


class Sun(C.Structure):
    """satsplat_sun (include/satsplat.h)."""
    _fields_ = [("azimuth", C.c_float), ("elevation", C.c_float), ("width", C.c_int32), ("height", C.c_int32),
                ("viewport", C.c_float * 4)]

    @classmethod
    def from_view(cls, v):
        s = cls()
        s.azimuth, s.elevation = float(v.sun_azimuth), float(v.sun_elevation)
        s.width, s.height = int(v.sun_width), int(v.sun_height)
        s.viewport[:] = [float(x) for x in v.sun_viewport]
        return s


class ViewParams(C.Structure):
    """satsplat_view_params (include/satsplat.h): the constants of one view of the device-resident camera chain."""
    _fields_ = [("F", C.c_float * 8), ("view_dir", C.c_float * 3), ("b_z", C.c_float), ("z_bg", C.c_float), ("bg_rgb", C.c_float * 3),
                ("cc", C.c_float * 12), ("ambient", C.c_float * 3), ("depth_bias", C.c_float), ("slope", C.c_float),
                ("nearby_d_azimuth", C.c_float), ("nearby_d_elevation", C.c_float), ("pad0", C.c_float),
                ("sun_viewport", C.c_float * 4), ("sun_s", C.c_double * 2), ("sun_view_dir", C.c_float * 3), ("pad1", C.c_float)]


CAMERA_BLOCK_FLOATS = 80
CAM_VIEW, CAM_SUN, CAM_NEARBY = 0, 1, 2


def build(force: bool = False) -> str:
    from .build import build as _b
    return _b(force=force)


def lib():
    """Load libsatsplat.so; raises if it is missing (no fallback path exists)."""
    global _LIB
    if _LIB is None:
        if not os.path.exists(_SO):
            raise ImportError(f"{_SO} not built: run `python -m paper_2606_28581_b200.build` (needs nvcc); there is no CPU fallback")
        L = C.CDLL(_SO)
        L.satsplat_last_error.restype = C.c_char_p
        L.satsplat_last_error.argtypes = [C.c_void_p]
        L.satsplat_version.restype = C.c_char_p
        L.satsplat_scratch_bytes.restype = C.c_int64
        L.satsplat_kernel_launches.restype = C.c_int64
        L.satsplat_scratch_bytes.argtypes = [C.c_void_p]
        L.satsplat_destroy.restype = None
        L.satsplat_destroy.argtypes = [C.c_void_p]
        vp, i64, i32, f32 = C.c_void_p, C.c_int64, C.c_int32, C.c_float
        L.satsplat_create.argtypes = [C.POINTER(vp), C.c_int, i64, i32, i32, i64]
        L.satsplat_sun_camera.argtypes = [C.POINTER(Camera), f32, f32, i32, i32, C.POINTER(f32), C.POINTER(Camera), C.POINTER(f32)]
        L.satsplat_sun_camera_backward.argtypes = [C.POINTER(Camera), f32, f32, C.POINTER(f32), vp, vp, vp, vp]
        L.satsplat_loss_scratch_floats.restype = C.c_int64
        L.satsplat_loss_scratch_floats.argtypes = [i32, i32]
        L.satsplat_loss_upstream.argtypes = [C.POINTER(Camera), C.POINTER(LossWeights)] + [vp] * 10
        L.satsplat_init_scratch_bytes.restype = C.c_int64
        L.satsplat_init_scratch_bytes.argtypes = [i32, i32, i64]
        L.satsplat_init_from_dsm.argtypes = [vp, i32, i32, f32, f32, f32, i64] + [vp] * 9
        L.satsplat_relocate_scratch_bytes.restype = C.c_int64
        L.satsplat_relocate_scratch_bytes.argtypes = [i64]
        L.satsplat_relocate.argtypes = [i64] + [vp] * 8 + [f32, i32, vp, vp, vp]
        L.satsplat_relocate_static.argtypes = [i64] + [vp] * 8 + [f32, i32, vp, vp]
        L.satsplat_adam_state_floats.restype = C.c_int64
        L.satsplat_adam_state_floats.argtypes = [i64]
        L.satsplat_adam_step.argtypes = [i64] + [vp] * 12 + [C.POINTER(Adam), vp]
        L.satsplat_adam_step_cameras.argtypes = [i32] + [vp] * 9 + [C.POINTER(CameraAdam), i32, vp]
        L.satsplat_preprocess.argtypes = [vp, C.POINTER(Camera), i64, vp, vp, vp, vp, vp, vp]
        L.satsplat_render_forward.argtypes = [vp, C.POINTER(Shading), vp, vp, vp, vp]
        L.satsplat_shadow_map.argtypes = [vp, vp, vp]
        L.satsplat_render_backward.argtypes = [vp, C.POINTER(Shading)] + [vp] * 14
        L.satsplat_shadow_map_backward.argtypes = [vp] * 8
        L.satsplat_iteration_host.argtypes = [vp, vp, C.POINTER(Camera), C.POINTER(Sun), C.POINTER(Shading), i64] + [vp] * 13
        L.satsplat_reserve_host_staging.argtypes = [vp, vp]
        L.satsplat_iteration_host_begin.argtypes = [vp, vp, i32, C.POINTER(Camera), C.POINTER(Sun), C.POINTER(Shading), i64] + [vp] * 13
        L.satsplat_iteration_host_end.argtypes = [vp, i32]
        L.satsplat_training_step_host_begin.argtypes = [vp, vp, i32, C.POINTER(Camera), C.POINTER(Sun), C.POINTER(Shading),
                                                        C.POINTER(LossWeights), i64] + [vp] * 10
        L.satsplat_training_step_host_end.argtypes = [vp, i32]
        L.satsplat_training_step_host.argtypes = [vp, vp, C.POINTER(Camera), C.POINTER(Sun), C.POINTER(Shading),
                                                  C.POINTER(LossWeights), i64] + [vp] * 10
        L.satsplat_sync_status.argtypes = [vp, C.POINTER(i64), vp]
        L.satsplat_debug_bins.argtypes = [vp, C.POINTER(i64)] + [C.POINTER(vp)] * 5 + [vp]
        L.satsplat_debug_records.argtypes = [vp, vp, vp, vp]
        L.satsplat_debug_planes.argtypes = [vp, C.POINTER(vp), C.POINTER(vp)]
        L.satsplat_set_profiling.argtypes = [vp, i32]
        L.satsplat_set_option.argtypes = [vp, i32, i32]
        L.satsplat_stage_ms.argtypes = [vp, C.POINTER(f32)]
        L.satsplat_view_params_fill.argtypes = [C.POINTER(Camera), C.POINTER(Shading), C.POINTER(Sun), f32, f32, C.POINTER(ViewParams)]
        L.satsplat_camera_chain.argtypes = [vp] * 5
        L.satsplat_camera_chain_backward.argtypes = [vp] * 9
        L.satsplat_advance_view_index.argtypes = [vp, i32, i32, vp]
        L.satsplat_preprocess_device.argtypes = [vp, i32, i32, vp, i32, i64, vp, vp, vp, vp, vp, vp]
        L.satsplat_render_forward_device.argtypes = [vp, vp, vp, i32, i32, vp, vp, vp, vp]
        L.satsplat_render_backward_device.argtypes = [vp, vp, vp, i32, i32] + [vp] * 14
        L.satsplat_backward_chain.argtypes = [vp] * 11
        L.satsplat_measure_peaks.argtypes = [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_int)]
        _LIB = L
    return _LIB


def kernel_launches() -> int:
    return int(lib().satsplat_kernel_launches())


def measure_peaks(device: int = 0) -> dict:
    """satsplat_measure_peaks: measured FP32 lane-instructions/s and MUFU operations/s of `device`."""
    a, b, n = C.c_double(0), C.c_double(0), C.c_int(0)
    rc = lib().satsplat_measure_peaks(int(device), C.byref(a), C.byref(b), C.byref(n))
    if rc != 0:
        raise SatsplatError(rc, "satsplat_measure_peaks failed")
    return dict(fp32_lane_inst_per_s=a.value, mufu_per_s=b.value, sm_count=n.value)


def version() -> str:
    return lib().satsplat_version().decode()


def _check(t, dtype, ndim=None):
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor of dtype %s" % dtype)
    if ndim is not None and t.dim() != ndim:
        raise ValueError("expected %d dims" % ndim)
    return t


def _ptr(t, dtype=torch.float32):
    return None if t is None else _check(t, dtype).data_ptr()


class _DevBytes:
    """Raw device memory exposed through __cuda_array_interface__ so torch can view (then clone) it."""

    def __init__(self, ptr, nbytes):
        self.__cuda_array_interface__ = {"shape": (nbytes,), "typestr": "|u1", "data": (ptr, False), "version": 2}


def _wrap(ptr, nbytes, dev):
    if nbytes <= 0:
        return torch.empty(0, dtype=torch.uint8, device=dev)
    return torch.as_tensor(_DevBytes(ptr, nbytes), device=dev).clone()


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def sun_camera(view: Camera, azimuth, elevation, sun_w, sun_h, viewport):
    """satsplat_sun_camera: returns (sun Camera, reproj list[8])."""
    out, rep = Camera(), (C.c_float * 8)()
    vp = (C.c_float * 4)(*[float(x) for x in viewport])
    rc = lib().satsplat_sun_camera(C.byref(view), float(azimuth), float(elevation), int(sun_w), int(sun_h), vp, C.byref(out), rep)
    if rc:
        raise SatsplatError(rc, lib().satsplat_last_error(None).decode())
    return out, list(rep)


def sun_camera_backward(view: Camera, azimuth, elevation, viewport, v_F_sun, v_reproj, v_dF, stream=None):
    """satsplat_sun_camera_backward: v_dF (device [8]) += adjoint of the Eq. 16 sun camera applied to the device
    vectors v_F_sun / v_reproj (either may be None)."""
    vp = (C.c_float * 4)(*[float(x) for x in viewport])
    rc = lib().satsplat_sun_camera_backward(C.byref(view), float(azimuth), float(elevation), vp, _ptr(v_F_sun), _ptr(v_reproj),
                                            _ptr(v_dF), _stream(stream))
    if rc:
        raise SatsplatError(rc, lib().satsplat_last_error(None).decode())


def view_params_table(views, nearby=None, device="cuda"):
    """Device-resident array of satsplat_view_params for `views` (objects with the fields of satsplat_scenes.View), built
    with satsplat_view_params_fill (HOST) and copied up once.  `nearby[i]` = (d_azimuth, d_elevation) of view i's nearby
    camera.  Returns a uint8 device tensor [V, sizeof(satsplat_view_params)]."""
    arr = (ViewParams * len(views))()
    for i, v in enumerate(views):
        cam = Camera.from_view(v)
        sh = Shading.make(cc=v.cc, ambient=v.ambient, depth_bias=v.depth_bias, slope=v.slope)
        sun = Sun.from_view(v) if getattr(v, "shadows_on", False) else None
        da, de = (0.0, 0.0) if nearby is None else nearby[i]
        rc = lib().satsplat_view_params_fill(C.byref(cam), C.byref(sh), None if sun is None else C.byref(sun), float(da), float(de),
                                             C.byref(arr[i]))
        if rc:
            raise SatsplatError(rc, lib().satsplat_last_error(None).decode())
    raw = torch.frombuffer(bytearray(bytes(arr)), dtype=torch.uint8).view(len(views), C.sizeof(ViewParams))
    return raw.to(device)


def camera_chain(views_dev, dF_dev, view_index_dev, block_dev, stream=None):
    """satsplat_camera_chain: block_dev (device fp32 [80]) <- cameras of view *view_index_dev (device int32 [1])."""
    rc = lib().satsplat_camera_chain(_ptr(views_dev, torch.uint8), _ptr(dF_dev), _ptr(view_index_dev, torch.int32), _ptr(block_dev), _stream(stream))
    if rc:
        raise SatsplatError(rc, lib().satsplat_last_error(None).decode())


def camera_chain_backward(views_dev, dF_dev, view_index_dev, v_dF_view, v_F_sun, v_reproj, v_F_nearby, v_dF_all, stream=None):
    """satsplat_camera_chain_backward: v_dF_all[view] += v_dF_view + cascade adjoints (device tensors; inputs may be None)."""
    rc = lib().satsplat_camera_chain_backward(_ptr(views_dev, torch.uint8), _ptr(dF_dev), _ptr(view_index_dev, torch.int32), _ptr(v_dF_view), _ptr(v_F_sun),
                                              _ptr(v_reproj), _ptr(v_F_nearby), _ptr(v_dF_all), _stream(stream))
    if rc:
        raise SatsplatError(rc, lib().satsplat_last_error(None).decode())


def advance_view_index(view_index_dev, stride, n_views, stream=None):
    rc = lib().satsplat_advance_view_index(_ptr(view_index_dev, torch.int32), int(stride), int(n_views), _stream(stream))
    if rc:
        raise SatsplatError(rc, lib().satsplat_last_error(None).decode())


def loss_scratch_floats(width, height) -> int:
    return int(lib().satsplat_loss_scratch_floats(int(width), int(height)))


def loss_upstream(cam: Camera, out_rgba, out_geom, out_aux, target_rgba, scratch, v_rgba, v_geom, v_aux, loss_sums,
                  w_l1=0.8, w_ssim=0.2, w_dist=0.05, w_normal=0.05, stream=None):
    """satsplat_loss_upstream: fills v_rgba / v_geom / v_aux with dL/d(rendered images) and loss_sums[0:4] with the sums of
    |I - I*|, the SSIM map, the distortion and the normal term (device tensors)."""
    w = LossWeights(float(w_l1), float(w_ssim), float(w_dist), float(w_normal))
    rc = lib().satsplat_loss_upstream(C.byref(cam), C.byref(w), _ptr(out_rgba), _ptr(out_geom), _ptr(out_aux), _ptr(target_rgba),
                                      _ptr(scratch), _ptr(v_rgba), _ptr(v_geom), _ptr(v_aux), _ptr(loss_sums), _stream(stream))
    if rc:
        raise SatsplatError(rc, lib().satsplat_last_error(None).decode())


def init_from_dsm(dsm, cell, origin, u, jx, jy, want_cells=False, stream=None):
    """satsplat_init_from_dsm: dsm [H,W] and the random numbers u, jx, jy [N] are device tensors; returns device tensors
    (means [N,3], quats [N,4], scales [N,2][, cells [N] int32])."""
    _check(dsm, torch.float32, 2)
    H, W = dsm.shape
    n = int(u.numel())
    dev = dsm.device
    scratch = torch.empty(max(int(lib().satsplat_init_scratch_bytes(W, H, n)), 16), dtype=torch.uint8, device=dev)
    means, quats, scales = (torch.empty(n, k, device=dev) for k in (3, 4, 2))
    cells = torch.empty(n, dtype=torch.int32, device=dev) if want_cells else None
    rc = lib().satsplat_init_from_dsm(dsm.data_ptr(), W, H, float(cell), float(origin[0]), float(origin[1]), n, _ptr(u), _ptr(jx),
                                      _ptr(jy), scratch.data_ptr(), means.data_ptr(), quats.data_ptr(), scales.data_ptr(),
                                      None if cells is None else cells.data_ptr(), _stream(stream))
    if rc:
        raise SatsplatError(rc, lib().satsplat_last_error(None).decode())
    return (means, quats, scales, cells) if want_cells else (means, quats, scales)


def relocate(n, means, quats, scales, opacity_logits, rgb, adam_m, adam_v, u, o_min=0.005, n_max=51, want_src=False, stream=None):
    """satsplat_relocate: dead surfels (opacity <= o_min) are redrawn onto live ones, in place (device tensors)."""
    scratch = torch.empty(max(int(lib().satsplat_relocate_scratch_bytes(int(n))), 16), dtype=torch.uint8, device=means.device)
    src = torch.empty(int(n), dtype=torch.int32, device=means.device) if want_src else None
    rc = lib().satsplat_relocate(int(n), _ptr(means), _ptr(quats), _ptr(scales), _ptr(opacity_logits), _ptr(rgb), _ptr(adam_m),
                                 _ptr(adam_v), _ptr(u), float(o_min), int(n_max), scratch.data_ptr(),
                                 None if src is None else src.data_ptr(), _stream(stream))
    if rc:
        raise SatsplatError(rc, lib().satsplat_last_error(None).decode())
    return src


RELOCATE_STATIC_MAX_SURFELS = 131072


def relocate_static(n, means, quats, scales, opacity_logits, rgb, adam_m, adam_v, u, o_min=0.005, n_max=51, want_src=False, stream=None):
    """satsplat_relocate_static: `relocate` without a scratch buffer from the caller.  The library works in an array that is
    part of its own image, so the call performs no device allocation; that is what a host needs whose GPU memory is already
    fully owned by another pool or capped by a quota, or that cannot tolerate an allocation stall inside its loop.  At most
    RELOCATE_STATIC_MAX_SURFELS surfels (SatsplatError above that); calls on one GPU share the array and must not overlap.
    (`src`, when asked for, is an output tensor this binding creates for convenience; the C call takes a caller pointer.)"""
    src = torch.empty(int(n), dtype=torch.int32, device=means.device) if want_src else None
    rc = lib().satsplat_relocate_static(int(n), _ptr(means), _ptr(quats), _ptr(scales), _ptr(opacity_logits), _ptr(rgb), _ptr(adam_m),
                                        _ptr(adam_v), _ptr(u), float(o_min), int(n_max), None if src is None else src.data_ptr(),
                                        _stream(stream))
    if rc:
        raise SatsplatError(rc, lib().satsplat_last_error(None).decode())
    return src


def adam_state_floats(n) -> int:
    return int(lib().satsplat_adam_state_floats(int(n)))


def adam_step(n, means, quats, scales, opacity_logits, rgb, v_means, v_quats, v_scales, v_opacity_logits, v_rgb, adam_m, adam_v,
              lr, beta1=0.9, beta2=0.999, eps=1e-8, step=1, stream=None):
    """satsplat_adam_step: one fused Adam step over the five surfel groups, in place (device tensors)."""
    hp = Adam()
    hp.lr[:] = [float(x) for x in lr]
    hp.beta1, hp.beta2, hp.eps, hp.step = float(beta1), float(beta2), float(eps), int(step)
    rc = lib().satsplat_adam_step(int(n), _ptr(means), _ptr(quats), _ptr(scales), _ptr(opacity_logits), _ptr(rgb), _ptr(v_means),
                                  _ptr(v_quats), _ptr(v_scales), _ptr(v_opacity_logits), _ptr(v_rgb), _ptr(adam_m), _ptr(adam_v),
                                  C.byref(hp), _stream(stream))
    if rc:
        raise SatsplatError(rc, lib().satsplat_last_error(None).decode())


def adam_step_cameras(views_dev, view_index_dev, dF, v_dF_all, v_cc, v_ambient, adam_m, adam_v, steps, lr, beta1=0.9, beta2=0.999,
                      eps=1e-8, clear_v_dF=True, stream=None):
    """satsplat_adam_step_cameras: one Adam step on the dF row, [C | c] and ambient of view *view_index_dev, in place
    (cc / ambient inside the device view table `views_dev`); per-view state [V,23] and step counters [V] (device tensors)."""
    hp = CameraAdam()
    hp.lr[:] = [float(x) for x in lr]
    hp.beta1, hp.beta2, hp.eps = float(beta1), float(beta2), float(eps)
    rc = lib().satsplat_adam_step_cameras(int(views_dev.shape[0]), _ptr(view_index_dev, torch.int32), _ptr(views_dev, torch.uint8), _ptr(dF),
                                          _ptr(v_dF_all), _ptr(v_cc), _ptr(v_ambient), _ptr(adam_m), _ptr(adam_v),
                                          _ptr(steps, torch.int32), C.byref(hp), 1 if clear_v_dF else 0, _stream(stream))
    if rc:
        raise SatsplatError(rc, lib().satsplat_last_error(None).decode())


def view_table_shading(views_dev):
    """(cc [V,12], ambient [V,3]) float32 copies read out of a device view table (where satsplat_adam_step_cameras steps them)."""
    f = views_dev.view(torch.float32).view(views_dev.shape[0], -1)
    o_cc, o_amb = ViewParams.cc.offset // 4, ViewParams.ambient.offset // 4
    return f[:, o_cc:o_cc + 12].clone(), f[:, o_amb:o_amb + 3].clone()


class Context:
    """satsplat_ctx: scratch arena for one camera pass (create once, reuse every iteration)."""

    def __init__(self, max_surfels, max_width, max_height, max_duplicates, device=0):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2606_28581_b200 needs a CUDA device (there is no CPU fallback)")
        self._h = C.c_void_p()
        self.device = int(device)
        rc = lib().satsplat_create(C.byref(self._h), self.device, int(max_surfels), int(max_width), int(max_height), int(max_duplicates))
        if rc:
            raise SatsplatError(rc, lib().satsplat_last_error(None).decode())
        self._keep = {}

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().satsplat_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _rc(self, rc):
        if rc:
            raise SatsplatError(rc, lib().satsplat_last_error(self._h).decode())

    @property
    def scratch_bytes(self):
        return int(lib().satsplat_scratch_bytes(self._h))

    # ---- hot path ----
    def preprocess(self, cam: Camera, means, quats, scales, opacity_logits, rgb, stream=None):
        n = int(means.shape[0])
        self._keep["in"] = (means, quats, scales, opacity_logits, rgb)   # must outlive the backward
        self.cam, self.n = cam, n
        self._rc(lib().satsplat_preprocess(self._h, C.byref(cam), n, _ptr(means), _ptr(quats), _ptr(scales),
                                           _ptr(opacity_logits), _ptr(rgb), _stream(stream)))

    def preprocess_device(self, width, height, block, which, means, quats, scales, opacity_logits, rgb, stream=None):
        """satsplat_preprocess_device: camera `which` (CAM_*) of the device camera block `block` (fp32 [80])."""
        n = int(means.shape[0])
        self._keep["in"] = (means, quats, scales, opacity_logits, rgb, block)
        cam = Camera()
        cam.width, cam.height = int(width), int(height)
        self.cam, self.n = cam, n
        self._rc(lib().satsplat_preprocess_device(self._h, int(width), int(height), _ptr(block), int(which), n, _ptr(means), _ptr(quats),
                                                  _ptr(scales), _ptr(opacity_logits), _ptr(rgb), _stream(stream)))

    def render_forward_device(self, block, sun_depth, out_rgba=None, out_geom=None, out_aux=None, stream=None):
        sh, sw = (0, 0) if sun_depth is None else (int(sun_depth.shape[0]), int(sun_depth.shape[1]))
        self._rc(lib().satsplat_render_forward_device(self._h, _ptr(block), _ptr(sun_depth), sw, sh, _ptr(out_rgba), _ptr(out_geom),
                                                      _ptr(out_aux), _stream(stream)))

    def render_backward_device(self, block, sun_depth, v_rgba, v_geom, v_aux, v_means, v_quats, v_scales, v_opacity_logits, v_rgb,
                               v_dF=None, v_cc=None, v_ambient=None, v_sun_depth=None, v_reproj=None, stream=None):
        sh, sw = (0, 0) if sun_depth is None else (int(sun_depth.shape[0]), int(sun_depth.shape[1]))
        self._rc(lib().satsplat_render_backward_device(self._h, _ptr(block), _ptr(sun_depth), sw, sh, _ptr(v_rgba), _ptr(v_geom),
                                                       _ptr(v_aux), _ptr(v_means), _ptr(v_quats), _ptr(v_scales), _ptr(v_opacity_logits),
                                                       _ptr(v_rgb), _ptr(v_dF), _ptr(v_cc), _ptr(v_ambient), _ptr(v_sun_depth),
                                                       _ptr(v_reproj), _stream(stream)))

    def render_forward(self, shading: Shading, out_rgba=None, out_geom=None, out_aux=None, stream=None):
        self._rc(lib().satsplat_render_forward(self._h, C.byref(shading), _ptr(out_rgba), _ptr(out_geom), _ptr(out_aux), _stream(stream)))

    def shadow_map(self, sun_depth_out, stream=None):
        self._rc(lib().satsplat_shadow_map(self._h, _ptr(sun_depth_out), _stream(stream)))

    def render_backward(self, shading: Shading, v_rgba, v_geom, v_aux, v_means, v_quats, v_scales, v_opacity_logits, v_rgb,
                        v_dF=None, v_cc=None, v_ambient=None, v_sun_depth=None, v_reproj=None, stream=None):
        self._rc(lib().satsplat_render_backward(self._h, C.byref(shading), _ptr(v_rgba), _ptr(v_geom), _ptr(v_aux), _ptr(v_means),
                                                _ptr(v_quats), _ptr(v_scales), _ptr(v_opacity_logits), _ptr(v_rgb), _ptr(v_dF),
                                                _ptr(v_cc), _ptr(v_ambient), _ptr(v_sun_depth), _ptr(v_reproj), _stream(stream)))

    def backward_chain(self, v_means, v_quats, v_scales, v_opacity_logits, v_rgb=None, v_dF=None, v_cc=None, v_ambient=None,
                       v_reproj=None, stream=None):
        """satsplat_backward_chain: second half of a backward call made with OPT_SPLIT_BACKWARD = 1."""
        self._rc(lib().satsplat_backward_chain(self._h, _ptr(v_means), _ptr(v_quats), _ptr(v_scales), _ptr(v_opacity_logits), _ptr(v_rgb),
                                               _ptr(v_dF), _ptr(v_cc), _ptr(v_ambient), _ptr(v_reproj), _stream(stream)))

    def shadow_map_backward(self, v_sun_depth, v_means, v_quats, v_scales, v_opacity_logits, v_dF_sun=None, stream=None):
        self._rc(lib().satsplat_shadow_map_backward(self._h, _ptr(v_sun_depth), _ptr(v_means), _ptr(v_quats), _ptr(v_scales),
                                                    _ptr(v_opacity_logits), _ptr(v_dF_sun), _stream(stream)))

    # ---- status / test access ----
    def sync_status(self, stream=None) -> int:
        k = C.c_int64()
        self._rc(lib().satsplat_sync_status(self._h, C.byref(k), _stream(stream)))
        return int(k.value)

    def debug_bins(self, stream=None):
        """Copies of (keys[K] int64-viewed uint64, vals[K], ranges[tiles,2], rects[N,4], counts[N]) as torch tensors."""
        k = C.c_int64()
        ptrs = [C.c_void_p() for _ in range(5)]
        self._rc(lib().satsplat_debug_bins(self._h, C.byref(k), *[C.byref(p) for p in ptrs], _stream(stream)))
        K = int(k.value)
        tiles = ((self.cam.width + 15) // 16) * ((self.cam.height + 15) // 16)
        dev = torch.device("cuda", self.device)

        def copy(ptr, nbytes, dtype):
            return _wrap(ptr.value, nbytes, dev).view(dtype)

        keys = copy(ptrs[0], K * 8, torch.int64)
        vals = copy(ptrs[1], K * 4, torch.int32)
        ranges = copy(ptrs[2], tiles * 8, torch.int32).view(tiles, 2)
        rects = copy(ptrs[3], self.n * 8, torch.int16).view(self.n, 4)
        counts = copy(ptrs[4], self.n * 4, torch.int32)
        return K, keys, vals, ranges, rects, counts

    def debug_records(self, stream=None):
        dev = torch.device("cuda", self.device)
        rec = torch.empty(self.n, 16, dtype=torch.float32, device=dev)
        flags = torch.empty(self.n, dtype=torch.uint8, device=dev)
        self._rc(lib().satsplat_debug_records(self._h, rec.data_ptr(), flags.data_ptr(), _stream(stream)))
        return rec, flags

    def debug_planes(self):
        """(n_visited[H,W], n_contrib[H,W]) int32 copies."""
        a, b = C.c_void_p(), C.c_void_p()
        self._rc(lib().satsplat_debug_planes(self._h, C.byref(a), C.byref(b)))
        H, W = self.cam.height, self.cam.width
        dev = torch.device("cuda", self.device)
        torch.cuda.synchronize()
        outs = [_wrap(p.value, H * W * 4, dev).view(torch.int32).view(H, W) for p in (a, b)]
        return outs

    def set_option(self, option: int, value: int):
        self._rc(lib().satsplat_set_option(self._h, int(option), int(value)))

    def set_profiling(self, enabled: bool):
        self._rc(lib().satsplat_set_profiling(self._h, 1 if enabled else 0))

    def stage_ms(self):
        ms = (C.c_float * len(STAGES))()
        self._rc(lib().satsplat_stage_ms(self._h, ms))
        return dict(zip(STAGES, [float(x) for x in ms]))


def reserve_host_staging(ctx: Context, sun_ctx=None):
    """satsplat_reserve_host_staging: allocate the device staging of iteration_host (explicit, never lazy)."""
    ctx._rc(lib().satsplat_reserve_host_staging(ctx._h, None if sun_ctx is None else sun_ctx._h))


def _host_ptr(t):
    if t is None:
        return None
    if t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous():
        raise ValueError("expected contiguous fp32 CPU tensors")
    return t.data_ptr()


def iteration_host_begin(ctx: Context, sun_ctx, slot, cam: Camera, sun, shading: Shading, n, h_means, h_quats, h_scales, h_logits,
                         h_rgb, h_v_rgba, h_v_geom, h_v_aux, h_out_rgba, h_out_geom, h_out_aux, h_grads, stream=None):
    """satsplat_iteration_host_begin: enqueue one iteration with HOST tensors on staging slot 0 / 1; no synchronisation."""
    hp = _host_ptr
    ctx._rc(lib().satsplat_iteration_host_begin(ctx._h, None if sun_ctx is None else sun_ctx._h, int(slot), C.byref(cam),
                                                None if sun is None else C.byref(sun), C.byref(shading), int(n), hp(h_means),
                                                hp(h_quats), hp(h_scales), hp(h_logits), hp(h_rgb), hp(h_v_rgba), hp(h_v_geom),
                                                hp(h_v_aux), hp(h_out_rgba), hp(h_out_geom), hp(h_out_aux), hp(h_grads), _stream(stream)))


def training_step_host_begin(ctx: Context, sun_ctx, slot, cam: Camera, sun, shading: Shading, n, h_means, h_quats, h_scales,
                             h_logits, h_rgb, h_target_rgba, h_out_rgba, h_grads, h_loss_sums,
                             w_l1=0.8, w_ssim=0.2, w_dist=0.05, w_normal=0.05, stream=None):
    """satsplat_training_step_host_begin: forward -> loss stage on the device -> backward, HOST tensors (surfels and the
    target image up; gradients, the 8 loss sums and, if h_out_rgba is not None, the rendered image down); staging slot 0 / 1;
    no synchronisation."""
    hp = _host_ptr
    w = LossWeights(float(w_l1), float(w_ssim), float(w_dist), float(w_normal))
    ctx._rc(lib().satsplat_training_step_host_begin(ctx._h, None if sun_ctx is None else sun_ctx._h, int(slot), C.byref(cam),
                                                    None if sun is None else C.byref(sun), C.byref(shading), C.byref(w), int(n),
                                                    hp(h_means), hp(h_quats), hp(h_scales), hp(h_logits), hp(h_rgb),
                                                    hp(h_target_rgba), hp(h_out_rgba), hp(h_grads), hp(h_loss_sums), _stream(stream)))


def training_step_host_end(ctx: Context, slot):
    """satsplat_training_step_host_end: wait until the step begun on `slot` has delivered its gradients and loss sums."""
    ctx._rc(lib().satsplat_training_step_host_end(ctx._h, int(slot)))


def training_step_host(ctx: Context, sun_ctx, cam: Camera, sun, shading: Shading, n, h_means, h_quats, h_scales, h_logits, h_rgb,
                       h_target_rgba, h_out_rgba, h_grads, h_loss_sums, stream=None, **weights):
    """satsplat_training_step_host: _begin(slot 0) + _end(slot 0)."""
    training_step_host_begin(ctx, sun_ctx, 0, cam, sun, shading, n, h_means, h_quats, h_scales, h_logits, h_rgb, h_target_rgba,
                             h_out_rgba, h_grads, h_loss_sums, stream=stream, **weights)
    training_step_host_end(ctx, 0)


def iteration_host_end(ctx: Context, slot):
    """satsplat_iteration_host_end: wait until the step begun on `slot` has delivered its images and gradients."""
    ctx._rc(lib().satsplat_iteration_host_end(ctx._h, int(slot)))


def iteration_host(ctx: Context, sun_ctx, cam: Camera, sun, shading: Shading, n, h_means, h_quats, h_scales, h_logits,
                   h_rgb, h_v_rgba, h_v_geom, h_v_aux, h_out_rgba, h_out_geom, h_out_aux, h_grads, stream=None):
    """satsplat_iteration_host: one full training-view iteration with HOST (pinned CPU) tensors; `sun` is a Sun."""
    def hp(t):
        if t is None:
            return None
        if t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous():
            raise ValueError("expected contiguous fp32 CPU tensors")
        return t.data_ptr()
    rc = lib().satsplat_iteration_host(ctx._h, None if sun_ctx is None else sun_ctx._h, C.byref(cam),
                                       None if sun is None else C.byref(sun), C.byref(shading), int(n), hp(h_means),
                                       hp(h_quats), hp(h_scales), hp(h_logits), hp(h_rgb), hp(h_v_rgba), hp(h_v_geom),
                                       hp(h_v_aux), hp(h_out_rgba), hp(h_out_geom), hp(h_out_aux), hp(h_grads), _stream(stream))
    ctx._rc(rc)

"""Helpers for the GPU parity tests: run one view through the C ABI (via the thin Python binding) and through the
oracle on the SAME seeded inputs, and compare with the parity policy of DESIGN.md ("Parity policy at
discontinuities").  Nothing here computes expected values from the CUDA path."""
from __future__ import annotations

import numpy as np
import torch

# fragility thresholds on the oracle's per-pixel decision margins
# (rho cut [abs], alpha skip [rel], T stop [rel], median |T-0.5| [abs], depth branch |rho3-rho2| [abs], clamp [abs])
MARGIN_THRESH = np.array([2e-4, 2e-4, 2e-3, 2e-5, 2e-4, 2e-5])


def t(a, dtype=torch.float32):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda", dtype=dtype).contiguous()


class GpuScene:
    """Device copies of a scene's surfel arrays."""

    def __init__(self, scene):
        self.n = scene.n
        self.means, self.quats, self.scales = t(scene.means), t(scene.quats), t(scene.scales)
        self.logits, self.rgb = t(scene.opacity_logits), t(scene.rgb)

    def zeros_grads(self):
        z = lambda *s: torch.zeros(*s, device="cuda", dtype=torch.float32)
        return dict(v_means=z(self.n, 3), v_quats=z(self.n, 4), v_scales=z(self.n, 2), v_logits=z(self.n), v_rgb=z(self.n, 3),
                    v_dF=z(8), v_cc=z(12), v_ambient=z(3), v_reproj=z(8), v_dF_sun=z(8))


def gpu_view_iteration(P, gs: GpuScene, view, *, sun_view=None, reproj=None, upstream=None, sun_upstream=None,
                       do_backward=True, max_dup=None, ctx=None, sun_ctx=None, want_debug=True, binning=None):
    """One view through the CUDA path.  `sun_view`/`reproj`: the fp32 sun camera + reprojection constants (inputs)."""
    n = gs.n
    H, W = view.height, view.width
    max_dup = max_dup or max(16 * n, 1024)
    res = {}
    cam = P.Camera.from_view(view)
    own = []
    if ctx is None:
        ctx = P.Context(max(n, 1), W, H, max_dup)
        own.append(ctx)
    if binning is not None:
        ctx.set_option(P.OPT_BINNING, binning)
    ctx.set_option(P.OPT_DEBUG_PLANES, 1 if want_debug else 0)
    sun_depth = None
    if sun_view is not None:
        if sun_ctx is None:
            sun_ctx = P.Context(max(n, 1), sun_view.width, sun_view.height, max_dup)
            own.append(sun_ctx)
        if binning is not None:
            sun_ctx.set_option(P.OPT_BINNING, binning)
        scam = P.Camera.from_view(sun_view)
        sun_ctx.preprocess(scam, gs.means, gs.quats, gs.scales, gs.logits, gs.rgb)
        sun_depth = torch.empty(sun_view.height, sun_view.width, device="cuda", dtype=torch.float32)
        sun_ctx.shadow_map(sun_depth)
        res["sun_depth"] = sun_depth.cpu().numpy()
        if want_debug:
            res["sun_bins"] = sun_ctx.debug_bins()
    shading = P.Shading.make(cc=view.cc, ambient=view.ambient, sun_depth=sun_depth, reproj=reproj, depth_bias=view.depth_bias,
                             slope=view.slope)
    ctx.preprocess(cam, gs.means, gs.quats, gs.scales, gs.logits, gs.rgb)
    out = [torch.empty(H, W, 4, device="cuda", dtype=torch.float32) for _ in range(3)]
    ctx.render_forward(shading, *out)
    res["K"] = ctx.sync_status()
    res.update(rgba=out[0].cpu().numpy(), geom=out[1].cpu().numpy(), aux=out[2].cpu().numpy())
    if want_debug:
        res["bins"] = ctx.debug_bins()
        rec, flags = ctx.debug_records()
        res.update(rec=rec.cpu().numpy(), flags=flags.cpu().numpy())
        nv, nc = ctx.debug_planes()
        res.update(n_visited=nv.cpu().numpy(), n_contrib=nc.cpu().numpy())
    if do_backward:
        g = gs.zeros_grads()
        up = [None if u is None else t(u) for u in upstream]
        v_sun = None if sun_view is None else torch.zeros_like(sun_depth)
        ctx.render_backward(shading, up[0], up[1], up[2], g["v_means"], g["v_quats"], g["v_scales"], g["v_logits"], g["v_rgb"],
                            g["v_dF"], g["v_cc"], g["v_ambient"], v_sun, g["v_reproj"] if sun_view is not None else None)
        if sun_view is not None:
            res["v_sun_depth"] = v_sun.cpu().numpy()
            gsun = gs.zeros_grads()
            vs = v_sun if sun_upstream is None else v_sun + t(sun_upstream)
            sun_ctx.shadow_map_backward(vs.contiguous(), gsun["v_means"], gsun["v_quats"], gsun["v_scales"], gsun["v_logits"],
                                        gsun["v_dF_sun"])
            res["sun_grads"] = {k: v.cpu().numpy() for k, v in gsun.items()}
        res["grads"] = {k: v.cpu().numpy() for k, v in g.items()}
    torch.cuda.synchronize()
    for c in own:
        c.close()
    return res


# ------------------------------------------------------------------------------------------------------------
# comparisons
# ------------------------------------------------------------------------------------------------------------
def assert_bins_bitexact(orc_pass, bins, n):
    K, keys, vals, ranges, rects, counts = bins
    assert K == len(orc_pass["keys"]), (K, len(orc_pass["keys"]))
    assert np.array_equal(counts.cpu().numpy().view(np.uint32), orc_pass["count"])
    nz = orc_pass["count"] > 0
    r = rects.cpu().numpy().view(np.uint16).astype(np.int32)
    assert np.array_equal(r[nz], orc_pass["rect"][nz])
    assert keys.cpu().numpy().view(np.uint64).tobytes() == orc_pass["keys"].tobytes()       # memcmp
    assert vals.cpu().numpy().view(np.uint32).tobytes() == orc_pass["vals"].tobytes()
    assert ranges.cpu().numpy().view(np.uint32).tobytes() == orc_pass["ranges"].tobytes()


def assert_records(orc_pass, rec, flags):
    ref, rf = orc_pass["rec"], orc_pass["flags"]
    assert np.array_equal(flags, rf)
    ok = (orc_pass["count"] > 0)
    nd = ok & ((rf & 2) == 0)
    # c, z_c bit exact for every binned surfel; Q, g bit exact where not degenerate; normals bit exact
    for col in (0, 1, 6, 13, 14, 15, 10, 11, 12):
        assert np.array_equal(rec[ok, col].view(np.uint32), ref[ok, col].view(np.uint32)), col
    for col in (2, 3, 4, 5, 7, 8):
        assert np.array_equal(rec[nd, col].view(np.uint32), ref[nd, col].view(np.uint32)), col
    np.testing.assert_allclose(rec[ok, 9], ref[ok, 9], rtol=2e-6, atol=1e-7)       # alpha uses exp


def fragile_mask(margins, extra=None):
    m = (margins < MARGIN_THRESH).any(-1)
    if extra is not None:
        m |= extra
    return m


def compare_images(gpu, ref, fragile, *, atol=1e-5, rtol=1e-4, names=("rgba", "geom", "aux"), extra_tol=None,
                   max_fragile_frac=5e-3):
    """|gpu - ref| <= atol + rtol |ref| on every non-fragile pixel, every channel."""
    frac = fragile.mean()
    assert frac <= max_fragile_frac, f"too many fragile pixels: {frac}"
    stats = {}
    for k in names:
        g, r = gpu[k].astype(np.float64), ref[k]
        tol = atol + rtol * np.abs(r)
        if extra_tol is not None and k in extra_tol:
            tol = tol + extra_tol[k]
        err = np.abs(g - r)
        bad = (err > tol) & ~fragile[..., None]
        stats[k] = float((err / tol)[~fragile].max()) if (~fragile).any() else 0.0
        assert not bad.any(), (k, int(bad.sum()), np.argwhere(bad)[:5], g[bad][:5], r[bad][:5])
    return stats


EPS32 = 2.0 ** -24      # unit roundoff of fp32 (round to nearest)
C_ROUND = 128.0         # DESIGN.md section 3 "Gradient bar": the largest c any element has needed is 94 (profiles/r3_gradient_bar.md)
C_ROUND_SHADOW = 256.0  # view backward through the soft shadow test: the derivation's worst case (beside the conditioning term)


BAR_LOG = []            # one record per (label, gradient group): how much of the third term each comparison used
MAX_BEYOND_PLAIN = 1e-3  # masked runs: share of a group's elements that may lie outside the literal north_star tolerance


def compare_grads(gpu, ref, twin, pairs, *, atol=1e-5, rtol=1e-3, c=C_ROUND, extra=None, exempt=None, label=None,
                  max_beyond_plain_frac=None):
    """Gradient bar (north_star + DESIGN.md section 3), ONE rule for every gradient the path produces:

        |gpu - ref| <= atol + rtol |ref| + c 2^-24 S        element by element,

    S = the oracle's absolute-value twin of the same gradient value (sum of |per-pair term| pushed through |chain
    Jacobian|): what rounding theory gives for an fp32 evaluation of a signed sum whose terms each pass through at
    most c singly rounded operations.  No share of elements may miss it.  `pairs`: (gpu key, ref key, twin key).
    `extra[gpu key]`: a further additive tolerance array computed by the ORACLE (shadow stage: the twin of the
    conditioning of the shadow lookup).  `exempt[gpu key]`: boolean array of elements that may miss the bar
    (unmasked runs only: rows of surfels touched by a fragile pixel); returned in the statistics.
    `max_beyond_plain_frac`: the third term is the exception, not the bar: at most this share of the elements of a group of
    1000 elements or more may lie outside the literal `atol + rtol |ref|` (asserted; smaller groups are whole-image sums and
    are recorded only).  Every call with a `label` is recorded in BAR_LOG (written to gpurun_out/ at session end)."""
    stats = {}
    for kg, kr, kt in pairs:
        g = gpu[kg].astype(np.float64)
        r = np.asarray(ref[kr], np.float64).reshape(g.shape)
        S = np.asarray(twin[kt], np.float64).reshape(g.shape)
        assert (S >= np.abs(r) * (1 - 1e-9) - 1e-300).all(), (kg, "twin below |ref|")   # triangle inequality (P19)
        err = np.abs(g - r)
        tol = atol + rtol * np.abs(r) + c * EPS32 * S
        if extra is not None and kg in extra:
            tol = tol + np.asarray(extra[kg], np.float64).reshape(g.shape)
        bad = err > tol
        n_exempt = 0
        if exempt is not None and kg in exempt:
            ex = np.broadcast_to(np.asarray(exempt[kg]).reshape((-1,) + (1,) * (g.ndim - 1)), g.shape) if g.ndim > 1 else np.asarray(exempt[kg])
            n_exempt = int((bad & ex).sum())
            bad = bad & ~ex
        plain = atol + rtol * np.abs(r)
        need = np.where(S > 0, (err - plain) / (EPS32 * np.maximum(S, 1e-300)), 0.0)
        stats[kg] = dict(max_err_over_tol=float((err / tol).max()) if g.size else 0.0, beyond_plain=int((err > plain).sum()),
                         c_needed=float(need.max()) if g.size else 0.0, exempt_bad=n_exempt)
        over = need[err > plain]
        if label is not None:
            BAR_LOG.append(dict(label=label, group=kg, elements=int(g.size), beyond_plain=stats[kg]["beyond_plain"],
                                share=stats[kg]["beyond_plain"] / max(g.size, 1), c_needed_max=stats[kg]["c_needed"],
                                c_needed_p50=float(np.percentile(over, 50)) if over.size else 0.0,
                                c_needed_p99=float(np.percentile(over, 99)) if over.size else 0.0, c_allowed=float(c),
                                has_extra=bool(extra is not None and kg in extra), exempt_bad=n_exempt))
        if max_beyond_plain_frac is not None and g.size >= 1000:
            assert stats[kg]["beyond_plain"] <= max_beyond_plain_frac * g.size, (kg, "too many elements beyond the plain tolerance", stats[kg], g.size)
        if bad.any():
            i = int(np.argmax(np.where(bad, err / tol, 0).reshape(-1)))
            raise AssertionError((kg, "elements outside the bar", int(bad.sum()), g.size, stats[kg], g.reshape(-1)[i], r.reshape(-1)[i],
                                  S.reshape(-1)[i]))
    return stats


def touched_by(fragile, rec, flags):
    """Surfels whose 3-sigma screen box (from the oracle's fp32 record: centre, M = Q^-1, widened to the low-pass disc,
    one pixel of margin) contains a fragile pixel.  Test-side bookkeeping for the unmasked run only."""
    H, W = fragile.shape
    ii = np.zeros((H + 1, W + 1), np.int64)
    ii[1:, 1:] = fragile.astype(np.int64).cumsum(0).cumsum(1)
    r = rec.astype(np.float64)
    det = r[:, 2] * r[:, 5] - r[:, 3] * r[:, 4]
    ok = ((flags & 2) == 0) & (np.abs(det) > 0)
    with np.errstate(all="ignore"):
        ex = np.where(ok, 3.0 * np.sqrt(r[:, 5] ** 2 + r[:, 3] ** 2) / np.abs(det), 0.0)
        ey = np.where(ok, 3.0 * np.sqrt(r[:, 4] ** 2 + r[:, 2] ** 2) / np.abs(det), 0.0)
    ex = np.maximum(np.nan_to_num(ex, posinf=1e9), 2.1213204) + 1.0
    ey = np.maximum(np.nan_to_num(ey, posinf=1e9), 2.1213204) + 1.0
    cx, cy = np.nan_to_num(r[:, 0]), np.nan_to_num(r[:, 1])
    x0 = np.clip(np.floor(cx - ex), 0, W).astype(np.int64); x1 = np.clip(np.ceil(cx + ex), 0, W).astype(np.int64)
    y0 = np.clip(np.floor(cy - ey), 0, H).astype(np.int64); y1 = np.clip(np.ceil(cy + ey), 0, H).astype(np.int64)
    x1 = np.maximum(x1, x0); y1 = np.maximum(y1, y0)
    cnt = ii[y1, x1] - ii[y0, x1] - ii[y1, x0] + ii[y0, x0]
    return cnt > 0


GRAD_PAIRS = [("v_means", "v_means", "a_means"), ("v_quats", "v_quats", "a_quats"), ("v_scales", "v_scales", "a_scales"),
              ("v_logits", "v_logits", "a_logits"), ("v_rgb", "v_rgb", "a_rgb"), ("v_dF", "v_dF", "a_dF")]
EPI_PAIRS = [("v_cc", "v_cc", "a_cc"), ("v_ambient", "v_ambient", "a_ambient")]

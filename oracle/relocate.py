"""Oracle for the relocation step (second half; "use the 3DGS-MCMC [22] strategy
to relocate Gaussians during training").

TEST INFRASTRUCTURE ONLY: imported by tests/ only; shares no code with paper_2606_28581_b200/.  numpy float64, plain
loops, in the order of the steps below.

The SatSplat paper only cites [22] (Kheradmand et al., "3D Gaussian Splatting as Markov Chain Monte Carlo"); the rule
restated here is that paper's relocation, derived from what it must preserve (readings: DESIGN.md section 2 row 26):
  1. alpha_i = sigmoid(logit_i); surfel i is DEAD if alpha_i <= o_min (0.005 in [22]).
  2. every dead surfel d draws a live source j with probability proportional to alpha_j: inverse transform on the cumulative
     sum of the live opacities in index order with the caller's uniform number u_d (first j whose cumulative weight exceeds
     u_d * total).
  3. N_j = 1 + (number of dead surfels that drew j), capped at n_max (51 in [22]).
  4. the source and its copies all get opacity o' = 1 - (1 - alpha_j)^(1/N_j), so that N_j of them composited at the centre
     give the old opacity back (1 - (1 - o')^N = alpha_j), and both scales are multiplied by alpha_j / D with
         D = sum_{i=1..N} sum_{k=0..i-1} C(i-1, k) (-1)^k o'^(k+1) / sqrt(k+1),
     which keeps the integral of the composited profile through the centre: int 1 - (1 - o' g_{s'}(x))^N dx = s' sqrt(2 pi) D
     must equal int alpha g_s(x) dx = alpha s sqrt(2 pi).  o' is clamped to [o_min, 1 - 1e-7] before the logit.
  5. a dead surfel takes the source's centre, rotation and colour and the new (scale, logit); the source takes the new
     (scale, logit); the Adam state (m, v) of both is reset to zero.  If there is no live surfel nothing moves.
Pins: tests/test_oracle_pins.py P18.
PARITY UNPINNED against the SatSplat paper (it cites [22] without restating the rule); what the rule must preserve IS
pinned (P18, by quadrature).
"""
from __future__ import annotations

import math

import numpy as np


def relocation_factors(alpha, n):
    """(o', scale factor) for a source of opacity alpha split into n copies (step 4)."""
    o_new = 1.0 - (1.0 - alpha) ** (1.0 / n)
    denom = 0.0
    for i in range(1, n + 1):
        for k in range(i):
            denom += math.comb(i - 1, k) * (-1.0) ** k * o_new ** (k + 1) / math.sqrt(k + 1)
    return o_new, alpha / denom


def relocate(means, quats, scales, logits, rgb, adam_m, adam_v, u, o_min=0.005, n_max=51):
    """Returns new copies of all arrays plus (dead mask, source index per surfel (-1 if not relocated), N per surfel).
    adam_m / adam_v: dicts group -> array with the parameter's shape (or None)."""
    means, quats, scales, logits, rgb = (np.array(a, np.float64) for a in (means, quats, scales, logits, rgb))
    n = len(logits)
    alpha = 1.0 / (1.0 + np.exp(-logits))
    dead = alpha <= o_min
    src = np.full(n, -1, np.int64)
    ratio = np.ones(n, np.int64)
    w = np.where(dead, 0.0, alpha)
    cdf = np.cumsum(w)
    if n == 0 or cdf[-1] <= 0 or not dead.any():
        return dict(means=means, quats=quats, scales=scales, logits=logits, rgb=rgb, adam_m=adam_m, adam_v=adam_v, dead=dead,
                    src=src, ratio=ratio)
    for d in np.flatnonzero(dead):
        j = int(np.searchsorted(cdf, float(u[d]) * cdf[-1], side="right"))
        src[d] = min(j, n - 1)
        ratio[src[d]] += 1
    new_scales, new_logits = scales.copy(), logits.copy()
    for j in np.flatnonzero(ratio > 1):
        o_new, f = relocation_factors(alpha[j], int(min(ratio[j], n_max)))
        o_new = min(max(o_new, o_min), 1.0 - 1e-7)
        new_scales[j] = scales[j] * f
        new_logits[j] = math.log(o_new / (1.0 - o_new))
    out = dict(means=means.copy(), quats=quats.copy(), scales=new_scales.copy(), logits=new_logits.copy(), rgb=rgb.copy())
    for d in np.flatnonzero(dead):
        j = src[d]
        out["means"][d], out["quats"][d], out["rgb"][d] = means[j], quats[j], rgb[j]
        out["scales"][d], out["logits"][d] = new_scales[j], new_logits[j]
    touched = dead | (ratio > 1)
    for name, st in (("adam_m", adam_m), ("adam_v", adam_v)):
        if st is None:
            out[name] = None
            continue
        out[name] = {k: np.array(v, np.float64) for k, v in st.items()}
        for v in out[name].values():
            v[touched] = 0.0
    out.update(dead=dead, src=src, ratio=ratio)
    return out

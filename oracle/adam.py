"""Oracle for the optimiser step: Adam [Kingma & Ba 2015, Algorithm 1] over the surfel
parameter groups with per-group learning rates ("Adam optimizer with initial learning rates of 0.075 for
splat means, 0.0025 for color, 0.001 for quaternions and scales").

TEST INFRASTRUCTURE ONLY: imported by tests/ and bench.py's cpu_baseline leg; the product never imports it and it
shares no code with paper_2606_28581_b200/.  Plain numpy, float64, the textbook update written out:

    m <- b1 m + (1 - b1) g          v <- b2 v + (1 - b2) g^2
    m^ = m / (1 - b1^t)             v^ = v / (1 - b2^t)
    theta <- theta - lr m^ / (sqrt(v^) + eps)

Readings where the paper is silent (rows 19-20):
  * b1 = 0.9, b2 = 0.999, eps = 1e-8 are ARGUMENTS (the paper names none); the opacity learning rate is an argument too
    (the paper lists none for opacity);
  * the library's scales are linear and must stay positive, so the scale group is stepped in log space:
    theta = log s, dL/dtheta = s dL/ds, s <- s exp(-lr m^/(sqrt(v^) + eps)); its Adam state is that of theta.
  * per-camera groups ("0.0001 for camera delta matrices, and 0.001 for camera gain and bias"; Eq. 15 dF,
    Eq. 1 [C | c] and the ambient term L_a): one training iteration renders ONE view, so only that view's rows receive a
    gradient.  Reading: a view's rows, their Adam state and their step counter t_v advance only in the iterations that
    render the view (per-view Adam; the other views' rows are untouched, not decayed) -- adam_step_cameras below.
Pins: tests/test_oracle_pins.py P15 (first-step closed form, torch.optim.Adam as an independent routine, log-space
equivalence; per-camera groups: every view's subsequence of steps equals torch.optim.Adam run on that view alone).
PARITY UNPINNED against the paper for the opacity learning rate, the betas and epsilon (arguments) and the log-space
stepping of the scales.
"""
from __future__ import annotations

import numpy as np

GROUPS = ("means", "quats", "scales", "logits", "rgb")


def adam_step(params, grads, state, lrs, *, beta1=0.9, beta2=0.999, eps=1e-8, step=1):
    """One Adam step on the five surfel groups.  `params`, `grads`: dicts of float64 arrays keyed by GROUPS;
    `state`: dict group -> (m, v) (zeros before the first step); `lrs`: dict group -> learning rate; `step` = t >= 1.
    Returns (new_params, new_state); nothing is modified in place."""
    new_p, new_s = {}, {}
    c1, c2 = 1.0 - beta1 ** step, 1.0 - beta2 ** step
    for k in GROUPS:
        p = np.asarray(params[k], np.float64)
        g = np.asarray(grads[k], np.float64)
        m, v = (np.asarray(a, np.float64) for a in state[k])
        if k == "scales":
            g = p * g                                   # d/d log s
        m = beta1 * m + (1.0 - beta1) * g
        v = beta2 * v + (1.0 - beta2) * g * g
        upd = lrs[k] * (m / c1) / (np.sqrt(v / c2) + eps)
        new_p[k] = p * np.exp(-upd) if k == "scales" else p - upd
        new_s[k] = (m, v)
    return new_p, new_s


CAMERA_GROUPS = ("dF", "cc", "ambient")     # [V,8] camera deltas (Eq. 15), [V,12] gain and bias (Eq. 1), [V,3] ambient L_a


def adam_step_cameras(params, grads, state, steps, view, lrs, *, beta1=0.9, beta2=0.999, eps=1e-8):
    """One Adam step on the rows of view `view` of the per-camera groups.  `params`: dict of float64 arrays
    [V,8] / [V,12] / [V,3] keyed by CAMERA_GROUPS; `grads`: dict group -> gradient of THAT view's row ([8] / [12] / [3]);
    `state`: dict group -> (m, v), arrays shaped like the parameters; `steps`: int array [V], the number of steps each view
    has taken so far; `lrs`: dict group -> learning rate.  Returns (new_params, new_state, new_steps); the rows of every
    other view, their state and their counters come back unchanged.  Nothing is modified in place."""
    steps = np.array(steps, np.int64, copy=True)
    steps[view] += 1
    t = int(steps[view])
    c1, c2 = 1.0 - beta1 ** t, 1.0 - beta2 ** t
    new_p, new_s = {}, {}
    for k in CAMERA_GROUPS:
        p = np.array(params[k], np.float64, copy=True)
        m, v = (np.array(a, np.float64, copy=True) for a in state[k])
        g = np.asarray(grads[k], np.float64).reshape(p.shape[1])
        m[view] = beta1 * m[view] + (1.0 - beta1) * g
        v[view] = beta2 * v[view] + (1.0 - beta2) * g * g
        p[view] = p[view] - lrs[k] * (m[view] / c1) / (np.sqrt(v[view] / c2) + eps)
        new_p[k], new_s[k] = p, (m, v)
    return new_p, new_s, steps

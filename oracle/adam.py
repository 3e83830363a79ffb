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
Pins: tests/test_oracle_pins.py P15 (first-step closed form, torch.optim.Adam as an independent routine, log-space
equivalence).
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

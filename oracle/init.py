"""Oracle for the geometry-aware initialisation: area-weighted sampling
of surfel centres from a DSM, orientation from the DSM normal with Gram-Schmidt tangents, scale from the kNN point
spacing.

TEST INFRASTRUCTURE ONLY: imported by tests/ only; shares no code with paper_2606_28581_b200/.  numpy float64, scipy's
cKDTree as the library kNN routine, each step in the paper's order.

Readings (DESIGN.md section 2 row 25; the paper gives the idea, not the discretisation):
  * DSM h[row, col] on a regular grid of spacing `cell`, cell centre (col + 0.5, row + 0.5) * cell + origin;
    local tangents by finite differences (central inside, one-sided on the border):
    dx = (cell, 0, h_x cell), dy = (0, cell, h_y cell), weight a = |dx x dy| = cell^2 sqrt(1 + h_x^2 + h_y^2)  (:186);
  * sampling: inverse transform on the row-major cumulative sum of a; sample k takes the first cell whose cumulative
    weight exceeds u_k * total; the centre is jittered uniformly inside the cell, (jx, jy) in [0,1)^2, and lifted to the
    cell's tangent plane: z = h + h_x (jx - 0.5) cell + h_y (jy - 0.5) cell.  The random numbers (u, jx, jy) are INPUTS;
  * orientation (:192): n = (-h_x, -h_y, 1)/|.|, t_u = Gram-Schmidt of the world x axis against n, t_v = n x t_u,
    R = [t_u | t_v | n], quaternion (w, x, y, z) with w >= 0;
  * scale (:194): s_u = s_v = mean Euclidean distance to the k = 3 nearest other sampled centres.
PARITY UNPINNED against the paper for the discretisation (difference stencils, jitter, tangent-plane lift, k = 3, the
reference axis of the Gram-Schmidt step); the formulas the paper does print (|dx x dy|, orthonormal frame) are pinned (P17).
"""
from __future__ import annotations

import numpy as np


def slopes(dsm, cell):
    """h_x (along columns) and h_y (along rows): central differences inside, one-sided on the border."""
    h = np.asarray(dsm, np.float64)

    def diff(a, axis):
        a = np.moveaxis(a, axis, 0)
        d = np.zeros_like(a)
        if a.shape[0] > 1:                  # an axis of length 1 has no neighbour: slope 0
            d[1:-1] = (a[2:] - a[:-2]) / (2.0 * cell)
            d[0] = (a[1] - a[0]) / cell
            d[-1] = (a[-1] - a[-2]) / cell
        return np.moveaxis(d, 0, axis)
    return diff(h, 1), diff(h, 0)


def area_weights(dsm, cell):
    hx, hy = slopes(dsm, cell)
    return cell * cell * np.sqrt(1.0 + hx * hx + hy * hy)


def sample_cells(weights, u):
    cdf = np.cumsum(np.asarray(weights, np.float64).ravel())
    idx = np.searchsorted(cdf, np.asarray(u, np.float64) * cdf[-1], side="right")
    return np.minimum(idx, cdf.size - 1)


def rotation_to_quat(R):
    """Unit quaternion (w, x, y, z), w >= 0, of a proper rotation matrix (textbook trace method, largest-pivot branch)."""
    m = R
    tr = m[0, 0] + m[1, 1] + m[2, 2]
    if tr > 0:
        s = np.sqrt(tr + 1.0) * 2
        q = np.array([0.25 * s, (m[2, 1] - m[1, 2]) / s, (m[0, 2] - m[2, 0]) / s, (m[1, 0] - m[0, 1]) / s])
    elif m[0, 0] > m[1, 1] and m[0, 0] > m[2, 2]:
        s = np.sqrt(1.0 + m[0, 0] - m[1, 1] - m[2, 2]) * 2
        q = np.array([(m[2, 1] - m[1, 2]) / s, 0.25 * s, (m[0, 1] + m[1, 0]) / s, (m[0, 2] + m[2, 0]) / s])
    elif m[1, 1] > m[2, 2]:
        s = np.sqrt(1.0 + m[1, 1] - m[0, 0] - m[2, 2]) * 2
        q = np.array([(m[0, 2] - m[2, 0]) / s, (m[0, 1] + m[1, 0]) / s, 0.25 * s, (m[1, 2] + m[2, 1]) / s])
    else:
        s = np.sqrt(1.0 + m[2, 2] - m[0, 0] - m[1, 1]) * 2
        q = np.array([(m[1, 0] - m[0, 1]) / s, (m[0, 2] + m[2, 0]) / s, (m[1, 2] + m[2, 1]) / s, 0.25 * s])
    return q if q[0] >= 0 else -q


def frame(hx, hy):
    """R = [t_u | t_v | n] for a DSM cell with slopes (h_x, h_y)."""
    n = np.array([-hx, -hy, 1.0])
    n /= np.linalg.norm(n)
    ex = np.array([1.0, 0.0, 0.0])
    tu = ex - (ex @ n) * n
    tu /= np.linalg.norm(tu)
    tv = np.cross(n, tu)
    return np.stack([tu, tv, n], axis=1)


def init_from_dsm(dsm, cell, origin, u, jx, jy, k=3):
    """Returns dict(cells, means [N,3], quats [N,4], scales [N,2]) (float64)."""
    from scipy.spatial import cKDTree
    h = np.asarray(dsm, np.float64)
    H, W = h.shape
    hx, hy = slopes(h, cell)
    w = cell * cell * np.sqrt(1.0 + hx * hx + hy * hy)
    idx = sample_cells(w, u)
    row, col = idx // W, idx % W
    jx, jy = np.asarray(jx, np.float64), np.asarray(jy, np.float64)
    sx, sy = hx[row, col], hy[row, col]
    means = np.stack([origin[0] + (col + jx) * cell, origin[1] + (row + jy) * cell,
                      h[row, col] + sx * (jx - 0.5) * cell + sy * (jy - 0.5) * cell], axis=1)
    quats = np.stack([rotation_to_quat(frame(a, b)) for a, b in zip(sx, sy)]) if len(idx) else np.zeros((0, 4))
    if len(idx) > k:
        dist, _ = cKDTree(means).query(means, k=k + 1)
        s = dist[:, 1:].mean(axis=1)
    else:
        s = np.full(len(idx), cell)
    return dict(cells=idx, means=means, quats=quats, scales=np.stack([s, s], axis=1), weights=w)

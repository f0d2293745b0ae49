"""Maximum Mean Discrepancy between two 6-D phase-space point clouds -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only ``tests/`` may import this module; it shares no code with the CUDA package and imports nothing from it.

What the paper fixes (PAPER.md = /root/reference/PAPER.md): "The resulting simulated stream is compared to the observed
stream using the Maximum Mean Discrepancy (MMD), and the gradient of the loss is computed" (Fig. 2 step 4);
"we use the full 6D phase-space information of particles" (L39); the MMD "between simulated and observed streams [is] the
loss function" of the grid search and of the gradient steps (L47).  The paper prints neither the kernel, nor its
bandwidth, nor the estimator (it defers to its ref. [1]).  Reading taken (R20): the textbook squared MMD of
Gretton et al. with a Gaussian kernel on the 6-D points, one scale per coordinate, biased (V-statistic) estimator:

    k(u, v)     = exp( -1/2 sum_d ((u_d - v_d) / sigma_d)^2 ),   d = x, y, z, vx, vy, vz
    MMD^2(X, Y) = 1/n^2 sum_{i,i'} k(x_i, x_i') + 1/m^2 sum_{j,j'} k(y_j, y_j') - 2/(n m) sum_{i,j} k(x_i, y_j)

(the i = i' terms are included: MMD^2(X, X) = 0 exactly and MMD^2 >= 0 always), and its gradient with respect to the
simulated cloud X, which is what the paper's gradient descent pulls back through the simulator:

    dMMD^2/dx_{i,d} = -2/(n^2 sigma_d^2) sum_{i'} k(x_i, x_i') (x_i - x_i')_d + 2/(n m sigma_d^2) sum_j k(x_i, y_j) (x_i - y_j)_d

Written as the definition: plain double loops over points (numpy only inside one point's row), fp64.
Pins (tests/test_oracle_mmd.py): MMD^2(X, X) = 0, symmetry, one point against one point = 2 (1 - k), a hand-expanded
2-against-1 case, the limits sigma -> infinity (0) and sigma -> 0 (1/n + 1/m for distinct points), translation and
permutation invariance, non-negativity, central finite differences of the value for every gradient component.
"""
from __future__ import annotations

import numpy as np


def _points(pos, vel):
    pos = np.asarray(pos, dtype=np.float64)
    vel = np.asarray(vel, dtype=np.float64)
    if pos.ndim != 2 or vel.ndim != 2 or pos.shape[0] != vel.shape[0] or pos.shape[1] < 3 or vel.shape[1] < 3:
        raise ValueError("pos and vel must be [n, >= 3] arrays of the same length")
    return np.concatenate([pos[:, :3], vel[:, :3]], axis=1)


def _kernel_row(p, Q, inv_sigma):
    """k(p, q) for one point p against every row q of Q."""
    d = (Q - p) * inv_sigma
    return np.exp(-0.5 * np.sum(d * d, axis=1))


def mmd2(xpos, xvel, ypos, yvel, sigma):
    """Squared MMD (biased estimator) between the clouds X = (xpos, xvel) and Y = (ypos, yvel); sigma: 6 scales."""
    X, Y = _points(xpos, xvel), _points(ypos, yvel)
    inv = 1.0 / np.asarray(sigma, dtype=np.float64).reshape(6)
    n, m = X.shape[0], Y.shape[0]
    sxx = sxy = syy = 0.0
    for i in range(n):
        sxx += float(np.sum(_kernel_row(X[i], X, inv)))
        sxy += float(np.sum(_kernel_row(X[i], Y, inv)))
    for j in range(m):
        syy += float(np.sum(_kernel_row(Y[j], Y, inv)))
    return sxx / (n * n) + syy / (m * m) - 2.0 * sxy / (n * m)


def mmd2_grad(xpos, xvel, ypos, yvel, sigma):
    """(dMMD^2/dxpos [n, 3], dMMD^2/dxvel [n, 3]): the gradient with respect to the first cloud."""
    X, Y = _points(xpos, xvel), _points(ypos, yvel)
    inv = 1.0 / np.asarray(sigma, dtype=np.float64).reshape(6)
    n, m = X.shape[0], Y.shape[0]
    g = np.zeros((n, 6))
    for i in range(n):
        kx = _kernel_row(X[i], X, inv)
        ky = _kernel_row(X[i], Y, inv)
        g[i] = (-2.0 / (n * n)) * np.sum(kx[:, None] * (X[i] - X), axis=0) * inv * inv \
             + (2.0 / (n * m)) * np.sum(ky[:, None] * (X[i] - Y), axis=0) * inv * inv
    return g[:, :3], g[:, 3:]

"""Brute-force optimum of the PRIMAL on tiny instances (test infrastructure, fp64).

P(t) (see lp_model.py) is convex piecewise-linear on t >= 0 and bounded below by 0, so a
minimiser lies at a vertex of the hyperplane arrangement {Phi_i t = thr_i} U {t_j = 0}:
enumerate every choice of n of the N + n hyperplanes, solve the n x n system, keep the
feasible (t >= 0) points, return the smallest P.  Exponential; for n <= 4, N <= 16 only.
This pins oracle/simplex.py to something that is not a simplex.
"""
from __future__ import annotations

from itertools import combinations

import numpy as np

from .lp_model import class_arrays, class_offset, primal_objective


def brute_force_optimum(phi, point_class, classes, w, mask=None, bot_rows=None):
    phi = np.asarray(phi, dtype=np.float64)
    N, n = phi.shape
    if n > 4 or N > 16:
        raise ValueError("vertex enumeration is for tiny instances only")
    _, _, thr = class_arrays(point_class, classes)
    H = np.concatenate([phi, np.eye(n)], axis=0)          # hyperplane normals
    h = np.concatenate([thr * class_offset(point_class, classes), np.zeros(n)])
    best, best_t = np.inf, None
    for rows in combinations(range(N + n), n):
        M = H[list(rows)]
        if abs(np.linalg.det(M)) < 1e-12:
            continue
        t = np.linalg.solve(M, h[list(rows)])
        if np.any(t < -1e-10):
            continue
        t = np.maximum(t, 0.0)
        val = primal_objective(phi, point_class, classes, w, t, mask, bot_rows)
        if val < best:
            best, best_t = val, t
    return best, best_t

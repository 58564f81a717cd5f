"""O-LP: small dense bounded-variable simplex on the dual form Eq. (1) (test infrastructure, fp64).

    minimise c^T x   s.t.   A x + s = b,   0 <= x <= u,   s >= 0

Textbook primal simplex with upper-bounded variables on the full tableau.  x = 0 with the
slack basis is feasible because b = w_BOT * 1 >= 0 (Eq. 13), so no phase 1.  Dantzig pricing,
falling back to Bland's smallest-index rule while pivots are degenerate (b = 0 when w_BOT = 0
makes the start fully degenerate).  The paper's own baseline is Matlab's dual simplex (:161);
this is the analogue used only to obtain the exact optimum the ADMM iteration approximates.

Returns x* (dual-form variables), t* = multipliers of A x <= b (the beam-on times, :80) and
the optimum OPT = -c^T x* = P(t*).
"""
from __future__ import annotations

import numpy as np


class SimplexError(RuntimeError):
    pass


# consecutive degenerate pivots after which pricing switches to Bland's rule (termination guarantee)
BLAND_AFTER = 500


def solve_bounded(c, A, b, u, max_pivots: int = 200000, tol: float = 1e-9):
    c = np.asarray(c, dtype=np.float64); A = np.asarray(A, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64); u = np.asarray(u, dtype=np.float64)
    n, N = A.shape
    if np.any(b < 0):
        raise SimplexError("b must be >= 0 (slack basis feasible)")
    T = np.concatenate([A, np.eye(n)], axis=1)               # B^-1 [A I]
    cost = np.concatenate([c, np.zeros(n)])
    ub = np.concatenate([u, np.full(n, np.inf)])
    basis = np.arange(N, N + n)
    is_basic = np.zeros(N + n, dtype=bool); is_basic[basis] = True
    at_upper = np.zeros(N + n, dtype=bool)
    xb = b.copy()
    d = cost.copy()                                           # reduced costs (c_B = 0 initially)
    movable = ub > 0
    degenerate_run = 0
    for it in range(max_pivots):
        elig_up = (~is_basic) & movable & (~at_upper) & (d < -tol)
        elig_dn = (~is_basic) & movable & at_upper & (d > tol)
        elig = elig_up | elig_dn
        if not elig.any():
            break
        if degenerate_run > BLAND_AFTER:
            j = int(np.argmax(elig))                          # Bland: smallest index
        else:
            j = int(np.argmax(np.where(elig, np.abs(d), -1.0)))
        sgn = 1.0 if elig_up[j] else -1.0
        col = sgn * T[:, j]
        # ratio test
        theta = ub[j]                                         # bound flip of the entering variable
        r_leave, leave_to_upper = -1, False
        dec = col > tol
        if dec.any():
            ratios = np.where(dec, xb / np.where(dec, col, 1.0), np.inf)
            r = int(np.argmin(ratios))
            # Bland tie-break on leaving variable during degenerate runs
            if degenerate_run > BLAND_AFTER:
                m = ratios.min()
                ties = np.nonzero(ratios <= m + 1e-12)[0]
                r = int(ties[np.argmin(basis[ties])])
            if ratios[r] < theta:
                theta, r_leave, leave_to_upper = max(ratios[r], 0.0), r, False
        inc = (col < -tol) & np.isfinite(ub[basis])
        if inc.any():
            room = ub[basis] - xb
            ratios = np.where(inc, room / np.where(inc, -col, 1.0), np.inf)
            r = int(np.argmin(ratios))
            if ratios[r] < theta:
                theta, r_leave, leave_to_upper = max(ratios[r], 0.0), r, True
        if not np.isfinite(theta):
            raise SimplexError("unbounded (cannot happen: x is boxed)")
        degenerate_run = degenerate_run + 1 if theta <= 1e-13 else 0
        xb = xb - theta * col
        if r_leave < 0:
            at_upper[j] = not at_upper[j]
            continue
        # pivot: j enters at row r_leave
        leaving = basis[r_leave]
        piv = T[r_leave, j]
        T[r_leave, :] /= piv
        colj = T[:, j].copy(); colj[r_leave] = 0.0
        T -= np.outer(colj, T[r_leave, :])
        d = d - d[j] * T[r_leave, :]
        entering_value = (ub[j] - theta) if at_upper[j] else theta
        xb[r_leave] = entering_value
        basis[r_leave] = j
        is_basic[j] = True; is_basic[leaving] = False
        at_upper[j] = False
        at_upper[leaving] = leave_to_upper
    else:
        raise SimplexError("pivot limit reached")
    # polish: recompute the basic solution and the multipliers from the final basis (removes the
    # round-off accumulated by the tableau updates)
    v = np.where(at_upper, ub, 0.0)
    v[~np.isfinite(v)] = 0.0
    v[basis] = 0.0
    full = np.concatenate([A, np.eye(n)], axis=1)
    Bmat = full[:, basis]
    v[basis] = np.linalg.solve(Bmat, b - full @ v)
    x = v[:N]
    y = np.linalg.solve(Bmat.T, cost[basis])
    t = -y                                                    # multipliers of A x <= b
    t[np.abs(t) < 1e-15] = 0.0
    return dict(x=x, t=t, opt=float(-c @ x), pivots=it)


def solve_plan(phi, point_class, classes, w, mask=None, bot_rows=None, **kw):
    """Exact LP optimum for one plan of a workload."""
    from .lp_model import dual_lp
    c, A, b, u = dual_lp(phi, point_class, classes, w, mask, bot_rows)
    return solve_bounded(c, A, b, u, **kw)

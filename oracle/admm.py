"""O-ADMM: the paper's iteration, step by step, in fp64 numpy (test infrastructure).

PARITY UNPINNED by the paper (no printed iterate); see oracle/__init__.py for the pins used.

Follows PAPER.md section II.B in the paper's order and notation, three-variable scaled form:
    (6)  v  = S^-1 ( A (z1 - y1 - c/rho) - z2 + y2 ),   S = A A^T + I  (factorised once, :91, :100)
    (7)  x1 = z1 - y1 - c/rho - A^T v ;   x2 = v + z2 - y2
    (4b) z1 = clip(x1 + y1, l=0, u) ;     z2 = min(x2 + y2, b)
    (4c) y1 = y1 + x1 - z1 ;              y2 = y2 + x2 - z2
batched by stacking the per-plan vectors as columns (:96), one rho per column (:222).
A, c, b, u are the PRECONDITIONED data (III.C, :183, :213; readings R9-R11):
    D_i = 1 / N_class(i)            column scaling, x = D x_hat            (R10)
    R_j = 1 / || row j of A D ||_2  row normalisation => diag(S) = 2       (:213, R9)
    A_hat = R A D,  c_hat = D c,  b_hat = R b,  u_hat = u / D.
Initial iterate: all zeros (R6).  Beam-on times: t = rho * R o y2 (:80); lambda = D o z1.

Stopping rule (the paper fixes 3000 iterations and gives no criterion, :106, :240; reading R7,
Boyd et al. section 3.3 on the scaled problem, per plan, tested every `check_every` iterations):
    ||x - z+||_2 <= eps_abs*sqrt(N+n) + tol*max(||x||_2, ||z+||_2)   and
    ||z+ - z||_2 <= eps_abs*sqrt(N+n) + tol*||y+||_2
(norms over both blocks stacked).  A plan that meets it is frozen at that iterate.

Optional presolve (NOT in the paper; DESIGN.md deviation D1, off by default): the minimiser of c^T x over the box
alone is x_box = u where c < 0, 0 where c > 0.  If A x_box <= b it is feasible for Eq. (1) and therefore optimal,
the multipliers of A x <= b vanish (t* = 0), and Eq. (6), (7), (4b), (4c) have the fixed point
    z1 = x_box,  y1 = -c/rho,  z2 = A x_box,  y2 = 0        (v = 0 in Eq. 6)
which is returned for such a plan with 0 iterations.

Optional warm start (NOT in the paper; DESIGN.md deviation D3, off by default, with presolve only): a plan whose box optimum is NOT
feasible but violates A x <= b by at most a factor `warm_start_ratio` in every row ((A x_box)_j <= ratio * b_j) starts from
    z1 = x_box,  y1 = -c/rho,  z2 = min(A x_box, b),  y2 = A x_box - z2
instead of the zero iterate (R6).  The iteration itself and its fixed points are unchanged; only the starting point differs.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import numpy as np
import scipy.linalg
import scipy.linalg.blas

from .lp_model import class_arrays, class_offset


@dataclass
class Preconditioned:
    A_hat: np.ndarray      # [n, N]
    c_hat: np.ndarray      # [N]
    D: np.ndarray          # [N]
    R: np.ndarray          # [n]
    S: np.ndarray          # [n, n]
    chol: tuple            # scipy cho_factor(S)
    class_count: np.ndarray


def precondition(phi, point_class, classes) -> Preconditioned:
    """One fp64 working array of the size of Phi (the scalings are applied to it in place, in the order written below), so that
    the full-size configurations (N x n up to 600000 x 12000 = 58 GB in fp64) fit in host memory."""
    pc, sense, thr = class_arrays(point_class, classes)
    Nk = np.bincount(pc, minlength=len(classes)).astype(np.float64)
    D = 1.0 / Nk[pc]
    M = np.array(phi, dtype=np.float64, order="C")  # [N, n]; becomes A^T, (A D)^T, A_hat^T in turn
    M *= (sense / thr)[:, None]                     # Eq. (12) with varphi = phi / D_alpha (:326):  A = (phi * sense / thr)^T
    M *= D[:, None]                                 # A D
    norms = np.sqrt(np.einsum("ij,ij->j", M, M))    # 2-norm of every row of A D (R9)
    R = np.where(norms > 0, 1.0 / np.where(norms > 0, norms, 1.0), 1.0)
    M *= R[None, :]
    A_hat = M.T                                     # [n, N] view
    c_hat = D * (-sense) * class_offset(pc, classes)   # Eq. (11); 0 for a homogeneous hard class (the coupling columns of Eq. 12)
    # S = A A^T + I (:91).  The product is the symmetric rank-k update of BLAS (dsyrk on the column-major view A_hat: no copy,
    # half the flops of a general matmul -- the full-size cases are 4e13 - 9e13 flops), mirrored into both triangles.
    S = scipy.linalg.blas.dsyrk(1.0, A_hat, lower=1)
    S = S + np.tril(S, -1).T + np.eye(A_hat.shape[0])
    chol = scipy.linalg.cho_factor(S, lower=True)
    return Preconditioned(A_hat=A_hat, c_hat=c_hat, D=D, R=R, S=S, chol=chol, class_count=Nk)


def plan_bounds(pre: Preconditioned, point_class, classes, weights, masks: Optional[np.ndarray] = None, bot_rows=None):
    """u_hat [N, B] and b_hat [n, B] (Eq. 13, 15 scaled).  masks: [B, N] bool or None (:144); bot_rows: [n] 0/1, the rows of A
    that carry w_BOT in b (Eq. 13: b = (0, w_BOT) with the coupling blocks of Eq. 12), None = all rows."""
    pc = np.asarray(point_class).astype(np.int64)
    weights = np.asarray(weights, dtype=np.float64)
    B = weights.shape[0]
    N, n = pre.D.shape[0], pre.R.shape[0]
    thr_k = np.array([c.threshold for c in classes], dtype=np.float64)
    u_hat = np.zeros((N, B))
    for p in range(B):
        m = np.ones(N) if masks is None else np.asarray(masks[p], dtype=np.float64)
        Nkp = np.bincount(pc, weights=m, minlength=len(classes))
        with np.errstate(divide="ignore", invalid="ignore"):
            per_class = np.where(Nkp > 0, weights[p, :-1] * thr_k / Nkp, 0.0)
        u_p = per_class[pc] * m
        hard = np.array([bool(getattr(c, "hard", 0)) for c in classes])[pc] & (m > 0)
        u_hat[:, p] = np.where(hard, np.inf, u_p / pre.D)            # Eq. (15): u = infinity for a hard class
    b_hat = pre.R[:, None] * weights[None, :, -1]
    if bot_rows is not None:
        b_hat = b_hat * np.asarray(bot_rows, dtype=np.float64)[:, None]
    return u_hat, b_hat


def presolve_box_optimum(pre: Preconditioned, u_hat, b_hat, rho, margin: float = 1e-5):
    """Plans whose box optimum is feasible (module docstring).  Returns (accepted [B] bool, state dict for those
    plans' columns: z1, y1, z2, y2).  `margin`: A x_box <= b (1 - margin) is required, so that a plan sitting on the
    boundary within rounding is left to the iteration."""
    rho = np.asarray(rho, dtype=np.float64)
    c = pre.c_hat[:, None]
    x_box = np.where(c < 0, u_hat, 0.0)                                   # [N, B]
    finite = np.all(np.isfinite(x_box), axis=0)
    x_safe = np.where(np.isfinite(x_box), x_box, 0.0)
    Ax = pre.A_hat @ x_safe                                               # [n, B]
    accepted = finite & np.all(Ax <= b_hat * (1.0 - margin), axis=0)
    state = dict(z1=x_safe, y1=-c / rho[None, :] + 0.0 * x_safe, z2=Ax, y2=np.zeros_like(Ax))
    return accepted, state


def warm_start_plans(accepted, state, b_hat, ratio: float):
    """Plans that start from the box state (module docstring): rejected by the presolve, finite box optimum, and
    (A x_box)_j <= ratio * b_j in every row.  Returns (warm [B] bool, z2, y2 of the warm start)."""
    Ax = state["z2"]
    finite = np.all(np.isfinite(state["z1"]), axis=0)
    warm = (~accepted) & finite & np.all(Ax <= ratio * b_hat, axis=0) if ratio > 0 else np.zeros_like(accepted)
    z2 = np.minimum(Ax, b_hat)
    return warm, z2, Ax - z2


def admm_run(pre: Preconditioned, u_hat, b_hat, rho, iters: int, tol: Optional[float] = None,
             eps_abs: float = 1e-6, check_every: int = 10, state0=None, history: bool = False,
             presolve: bool = False, warm_start_ratio: float = 0.0):
    """Run `iters` iterations (tol=None) or until every plan meets the stopping rule / iters.
    presolve=True (tolerance mode only): see presolve_box_optimum."""
    A = pre.A_hat
    n, N = A.shape
    rho = np.asarray(rho, dtype=np.float64)
    B = rho.shape[0]
    if state0 is None:
        z1 = np.zeros((N, B)); y1 = np.zeros((N, B)); z2 = np.zeros((n, B)); y2 = np.zeros((n, B))
    else:
        z1, y1, z2, y2 = (np.array(a, dtype=np.float64, copy=True) for a in state0)
    c_over_rho = pre.c_hat[:, None] / rho[None, :]
    active = np.ones(B, dtype=bool)
    it_done = np.zeros(B, dtype=np.int64)
    converged = np.zeros(B, dtype=bool)
    res = np.zeros((B, 2))
    hist = [] if history else None
    dim = np.sqrt(float(N + n))
    presolved = np.zeros(B, dtype=bool)
    if presolve and tol is not None and state0 is None:
        presolved, ps = presolve_box_optimum(pre, u_hat, b_hat, rho)
        for name, arr in (("z1", z1), ("y1", y1), ("z2", z2), ("y2", y2)):
            arr[:, presolved] = ps[name][:, presolved]
        active &= ~presolved
        converged |= presolved
        if warm_start_ratio > 0:
            warm, wz2, wy2 = warm_start_plans(presolved, ps, b_hat, warm_start_ratio)
            z1[:, warm] = ps["z1"][:, warm]; y1[:, warm] = ps["y1"][:, warm]
            z2[:, warm] = wz2[:, warm]; y2[:, warm] = wy2[:, warm]
    for k in range(1, iters + 1):
        r1 = z1 - y1 - c_over_rho
        r2 = z2 - y2
        v = scipy.linalg.cho_solve(pre.chol, A @ r1 - r2)                  # (6)
        x1 = r1 - A.T @ v                                                  # (7)
        x2 = v + r2
        z1n = np.clip(x1 + y1, 0.0, u_hat)                                 # (4b)
        z2n = np.minimum(x2 + y2, b_hat)
        y1n = y1 + x1 - z1n                                                # (4c)
        y2n = y2 + x2 - z2n
        # the residual norms are only used by the stopping rule (at a check), by the history and as the reported residuals of the
        # last iteration: they are evaluated at those iterations only (ten passes over the [N, B] arrays otherwise dominate the
        # cost of an iteration at the full-size configurations); the iterates do not depend on them
        checking = tol is not None and k % check_every == 0
        if checking or hist is not None or k == iters:
            rp = np.sqrt(np.sum((x1 - z1n) ** 2, axis=0) + np.sum((x2 - z2n) ** 2, axis=0))
            rd = np.sqrt(np.sum((z1n - z1) ** 2, axis=0) + np.sum((z2n - z2) ** 2, axis=0))
            nx = np.sqrt(np.sum(x1 ** 2, axis=0) + np.sum(x2 ** 2, axis=0))
            nz = np.sqrt(np.sum(z1n ** 2, axis=0) + np.sum(z2n ** 2, axis=0))
            ny = np.sqrt(np.sum(y1n ** 2, axis=0) + np.sum(y2n ** 2, axis=0))
            res[active, 0] = rp[active]; res[active, 1] = rd[active]
        a = active
        if a.all():                      # every plan takes the new iterate: no masked column copies (same values)
            z1, y1, z2, y2 = z1n, y1n, z2n, y2n
        else:                            # frozen plans keep the iterate at which they passed the stopping rule
            z1[:, a] = z1n[:, a]; y1[:, a] = y1n[:, a]; z2[:, a] = z2n[:, a]; y2[:, a] = y2n[:, a]
        it_done[a] = k
        if hist is not None:
            hist.append(np.stack([rp, rd, nx, nz, ny], axis=1))
        if checking:
            ok = (rp <= eps_abs * dim + tol * np.maximum(nx, nz)) & (rd <= eps_abs * dim + tol * ny)
            newly = active & ok
            converged |= newly
            active = active & ~ok
            if not active.any():
                break
    out = dict(z1=z1, y1=y1, z2=z2, y2=y2, iters=it_done, converged=converged, res=res, presolved=presolved)
    if hist is not None:
        out["history"] = np.stack(hist, axis=0)        # [iters, B, 5]
    return out


def recover(pre: Preconditioned, state, rho):
    """t [B, n] = rho * R o y2 (:80) and lambda [B, N] = D o z1 (the dual-LP variables x of Eq. 1)."""
    rho = np.asarray(rho, dtype=np.float64)
    t = (state["y2"] * pre.R[:, None] * rho[None, :]).T
    lam = (state["z1"] * pre.D[:, None]).T
    return t, lam


def solve_workload(w, rho, iters, tol=None, check_every=10, eps_abs=1e-6, pre=None, history=False, presolve=False,
                   warm_start_ratio=0.0):
    """Convenience: precondition + bounds + run + recover + primal objective per plan."""
    from .lp_model import hard_violation, primal_terms
    if pre is None:
        pre = precondition(w.phi, w.point_class, w.classes)
    masks = None if w.row_mask is None else w.mask_bool()
    bot_rows = getattr(w, "bot_rows", None)
    u_hat, b_hat = plan_bounds(pre, w.point_class, w.classes, w.weights, masks, bot_rows)
    st = admm_run(pre, u_hat, b_hat, rho, iters, tol=tol, eps_abs=eps_abs, check_every=check_every,
                  history=history, presolve=presolve, warm_start_ratio=warm_start_ratio)
    t, lam = recover(pre, st, rho)
    # obj: the penalty terms of the soft classes + the BOT term at t (a hard class is a constraint, reported as its violation)
    hard = np.array([bool(getattr(c, "hard", 0)) for c in w.classes])
    obj = np.zeros(w.B); viol = np.zeros(w.B)
    for p in range(w.B):
        m = None if masks is None else masks[p]
        terms, bot = primal_terms(w.phi, w.point_class, w.classes, w.weights[p], t[p], m, bot_rows)
        obj[p] = terms[~hard].sum() + bot
        viol[p] = hard_violation(w.phi, w.point_class, w.classes, t[p], m) if hard.any() else 0.0
    st["hard_violation"] = viol
    st.update(t=t, lam=lam, obj=obj, pre=pre, u_hat=u_hat, b_hat=b_hat)
    return st

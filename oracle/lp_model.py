"""The linear program, written out from PAPER.md Appendix A (test infrastructure, fp64).

Primal (BASELINE.json configs): for one plan with class weights w_k (dose
units), beam-on-time weight w_BOT and active row set L_p,

    P(t) = sum_k (w_k / N_{k,p}) * sum_{i in class k, active} max(0, s_k * (thr_k - Phi_i t))
           + w_BOT * sum_j t_j,        t >= 0,

s_k = +1 for "dose >= thr" classes (target), -1 for "dose <= thr" classes (low dose).

Dual in the paper's form, Eq. (1) (body missing from the text, reading R1;
structure from Eq. (3) :62-66 and Eq. (11)-(15) :314-322):

    minimise c^T x   subject to   A x <= b,   0 <= x <= u

with one x_i per dose point, thresholds normalised as varphi = phi / D (:326):
    A[:, i] = s_k * Phi[i, :] / thr_k          (Eq. 12: +varphi_T^T, -varphi_LD^T)
    c_i     = -s_k                             (Eq. 11: -1 target, +1 low dose)
    b       = w_BOT * 1_n                      (Eq. 13)
    u_i     = w_k * thr_k * mask_i / N_{k,p}   (Eq. 15 with w in dose units, reading R11;
                                                masked rows get u = 0, :144, reading R12)
The LP optimum is OPT = -c^T x* = P(t*), t* = multipliers of A x <= b.
"""
from __future__ import annotations

import numpy as np


def class_arrays(point_class, classes):
    pc = np.asarray(point_class).astype(np.int64)
    sense = np.array([c.sense for c in classes], dtype=np.float64)[pc]
    thr = np.array([c.threshold for c in classes], dtype=np.float64)[pc]
    return pc, sense, thr


def active_counts(point_class, n_classes, mask):
    """N_{k,p}: number of active rows of each class for one plan (mask: [N] bool or None)."""
    pc = np.asarray(point_class).astype(np.int64)
    if mask is None:
        return np.bincount(pc, minlength=n_classes).astype(np.float64)
    return np.bincount(pc, weights=np.asarray(mask, dtype=np.float64), minlength=n_classes)


def dual_lp(phi, point_class, classes, w, mask=None):
    """(c, A, b, u) of Eq. (1) for one plan.  w = (w_class..., w_BOT)."""
    phi = np.asarray(phi, dtype=np.float64)
    N, n = phi.shape
    pc, sense, thr = class_arrays(point_class, classes)
    w = np.asarray(w, dtype=np.float64)
    m = np.ones(N) if mask is None else np.asarray(mask, dtype=np.float64)
    Nk = active_counts(pc, len(classes), mask)
    A = (phi * (sense / thr)[:, None]).T.copy()
    c = -sense
    b = np.full(n, w[-1])
    with np.errstate(divide="ignore", invalid="ignore"):
        per_class = np.where(Nk > 0, w[:-1] * np.array([cl.threshold for cl in classes]) / Nk, 0.0)
    u = per_class[pc] * m
    return c, A, b, u


def primal_terms(phi, point_class, classes, w, t, mask=None):
    """Per-class penalty terms and the BOT term of P(t)."""
    phi = np.asarray(phi, dtype=np.float64)
    pc, sense, thr = class_arrays(point_class, classes)
    w = np.asarray(w, dtype=np.float64)
    m = np.ones(phi.shape[0]) if mask is None else np.asarray(mask, dtype=np.float64)
    Nk = active_counts(pc, len(classes), mask)
    dose = phi @ np.asarray(t, dtype=np.float64)
    viol = np.maximum(0.0, sense * (thr - dose)) * m
    terms = np.zeros(len(classes))
    for k in range(len(classes)):
        if Nk[k] > 0:
            terms[k] = w[k] * viol[pc == k].sum() / Nk[k]
    return terms, w[-1] * float(np.sum(t))


def primal_objective(phi, point_class, classes, w, t, mask=None) -> float:
    terms, bot = primal_terms(phi, point_class, classes, w, t, mask)
    return float(terms.sum() + bot)


def dual_bound(phi, point_class, classes, w, x, mask=None) -> float:
    """Weak-duality lower bound from any x: clip to [0,u], shrink by theta until A x <= b,
    return -c^T (theta x)  (<= OPT).  DESIGN.md 'duality bracket'."""
    c, A, b, u = dual_lp(phi, point_class, classes, w, mask)
    x = np.clip(np.asarray(x, dtype=np.float64), 0.0, u)
    Ax = A @ x
    pos = Ax > 0
    theta = 1.0
    if np.any(pos):
        theta = min(1.0, float(np.min(b[pos] / Ax[pos])))
    theta = max(theta, 0.0)
    return float(-c @ (theta * x))


def kkt_report(phi, point_class, classes, w, x, t, mask=None):
    """Residuals of the optimality conditions of the primal/dual pair (all should be ~0)."""
    c, A, b, u = dual_lp(phi, point_class, classes, w, mask)
    x = np.asarray(x, dtype=np.float64); t = np.asarray(t, dtype=np.float64)
    slack = b - A @ x
    g = c + A.T @ t                       # reduced cost of x given multipliers t
    rep = dict(
        box=float(max(np.max(-x), np.max(x - u), 0.0)),
        row=float(max(np.max(-slack), 0.0)),
        t_neg=float(max(np.max(-t), 0.0)),
        compl_rows=float(np.max(np.abs(t * slack))),
        # g_i > 0 => x_i = 0 ; g_i < 0 => x_i = u_i
        compl_box=float(np.max(np.abs(np.where(g > 0, g * x, g * (x - u))))),
        gap=float(abs(primal_objective(phi, point_class, classes, w, t, mask) - (-c @ x))),
    )
    return rep

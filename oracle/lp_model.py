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

Hard classes (ClassSpec.hard = 1; Eq. 15: "organs at risk ... u = infinity"): the dual variable has no upper
bound, which in the primal makes s_k (thr_k - Phi_i t) <= 0 a constraint instead of a penalty.  P(t) then carries no term for
the class and is +inf where the constraint is violated by more than HARD_TOL; the class weight is ignored.

Sector / isocenter coupling (App. A, Eq. 12, 16, 17, :316, :330-332).  The last column block of A, (-C_S^T ; T^T) with c = 0 and
u = infinity, is one more set of columns: column (iso, s) has -1/scale in the three rows of the collimator times t_(iso,s,c) and +1
in the row of the isocenter time tau_iso, and b = (0, w_BOT) puts the beam-on-time weight on the isocenter rows only (Eq. 13).  In
this model such a column is a ROW of the (extended) Phi with a class of sense +1, threshold 1, hard = 2 ("homogeneous": the
constant of the constraint is 0 instead of the threshold, so c_i = 0): its primal constraint is Phi_i (t, tau) >= 0, i.e.
sum_c t_(iso,s,c) / scale <= tau_iso, and P = penalties + w_BOT sum_iso tau_iso -- the beam-on time of an isocenter is that of
its slowest sector.  `bot_rows` ([n] 0/1) marks the rows of A that carry w_BOT in b; None = all of them (the LP without coupling).
"""
from __future__ import annotations

import numpy as np


HARD_TOL = 1e-9


def _hard(classes):
    return np.array([bool(getattr(c, "hard", 0)) for c in classes])


def class_arrays(point_class, classes):
    pc = np.asarray(point_class).astype(np.int64)
    sense = np.array([c.sense for c in classes], dtype=np.float64)[pc]
    thr = np.array([c.threshold for c in classes], dtype=np.float64)[pc]
    return pc, sense, thr


def class_offset(point_class, classes):
    """The constant of a point's constraint / penalty in units of its threshold: 1, or 0 for a homogeneous hard class (hard = 2)."""
    pc = np.asarray(point_class).astype(np.int64)
    return np.array([0.0 if int(getattr(c, "hard", 0)) == 2 else 1.0 for c in classes])[pc]


def _bot(n, bot_rows):
    return np.ones(n) if bot_rows is None else np.asarray(bot_rows, dtype=np.float64)


def active_counts(point_class, n_classes, mask):
    """N_{k,p}: number of active rows of each class for one plan (mask: [N] bool or None)."""
    pc = np.asarray(point_class).astype(np.int64)
    if mask is None:
        return np.bincount(pc, minlength=n_classes).astype(np.float64)
    return np.bincount(pc, weights=np.asarray(mask, dtype=np.float64), minlength=n_classes)


def dual_lp(phi, point_class, classes, w, mask=None, bot_rows=None):
    """(c, A, b, u) of Eq. (1) for one plan.  w = (w_class..., w_BOT)."""
    phi = np.asarray(phi, dtype=np.float64)
    N, n = phi.shape
    pc, sense, thr = class_arrays(point_class, classes)
    w = np.asarray(w, dtype=np.float64)
    m = np.ones(N) if mask is None else np.asarray(mask, dtype=np.float64)
    Nk = active_counts(pc, len(classes), mask)
    A = (phi * (sense / thr)[:, None]).T.copy()
    c = -sense * class_offset(pc, classes)
    b = w[-1] * _bot(n, bot_rows)
    with np.errstate(divide="ignore", invalid="ignore"):
        per_class = np.where(Nk > 0, w[:-1] * np.array([cl.threshold for cl in classes]) / Nk, 0.0)
    u = per_class[pc] * m
    u = np.where(_hard(classes)[pc] & (m > 0), np.inf, u)
    return c, A, b, u


_ROW_CHUNK = 1 << 16      # rows of Phi converted to fp64 at a time (the full-size configurations do not fit twice in host memory)


def _dose(phi, t):
    """Phi t in fp64, Phi taken in row chunks."""
    t = np.asarray(t, dtype=np.float64)
    out = np.empty(phi.shape[0])
    for a in range(0, phi.shape[0], _ROW_CHUNK):
        out[a:a + _ROW_CHUNK] = np.asarray(phi[a:a + _ROW_CHUNK], dtype=np.float64) @ t
    return out


def primal_terms(phi, point_class, classes, w, t, mask=None, bot_rows=None):
    """Per-class penalty terms and the BOT term of P(t)."""
    pc, sense, thr = class_arrays(point_class, classes)
    w = np.asarray(w, dtype=np.float64)
    m = np.ones(phi.shape[0]) if mask is None else np.asarray(mask, dtype=np.float64)
    Nk = active_counts(pc, len(classes), mask)
    dose = _dose(phi, t)
    viol = np.maximum(0.0, sense * (class_offset(pc, classes) * thr - dose)) * m
    terms = np.zeros(len(classes))
    hard = _hard(classes)
    for k in range(len(classes)):
        if hard[k]:
            terms[k] = np.inf if (viol[pc == k] > HARD_TOL).any() else 0.0
        elif Nk[k] > 0:
            terms[k] = w[k] * viol[pc == k].sum() / Nk[k]
    return terms, w[-1] * float(np.sum(np.asarray(t, dtype=np.float64) * _bot(phi.shape[1], bot_rows)))


def hard_violation(phi, point_class, classes, t, mask=None) -> float:
    """Largest violation s_k (thr_k - Phi_i t) over the active rows of the hard classes (0 if there is none)."""
    pc, sense, thr = class_arrays(point_class, classes)
    m = np.ones(phi.shape[0]) if mask is None else np.asarray(mask, dtype=np.float64)
    sel = _hard(classes)[pc] & (m > 0)
    if not sel.any():
        return 0.0
    return float(np.max(np.maximum(0.0, sense * (class_offset(pc, classes) * thr - _dose(phi, t)))[sel]))


def primal_objective(phi, point_class, classes, w, t, mask=None, bot_rows=None) -> float:
    terms, bot = primal_terms(phi, point_class, classes, w, t, mask, bot_rows)
    return float(terms.sum() + bot)


def dual_bound(phi, point_class, classes, w, x, mask=None, bot_rows=None) -> float:
    """Weak-duality lower bound from any x: clip to [0,u], shrink by theta until A x <= b,
    return -c^T (theta x)  (<= OPT).  DESIGN.md 'duality bracket'.  A x is formed from row chunks of Phi."""
    pc, sense, thr = class_arrays(point_class, classes)
    w = np.asarray(w, dtype=np.float64)
    N, n = phi.shape
    m = np.ones(N) if mask is None else np.asarray(mask, dtype=np.float64)
    Nk = active_counts(pc, len(classes), mask)
    with np.errstate(divide="ignore", invalid="ignore"):
        per_class = np.where(Nk > 0, w[:-1] * np.array([cl.threshold for cl in classes]) / Nk, 0.0)
    u = per_class[pc] * m                                        # Eq. (15), as in dual_lp
    u = np.where(_hard(classes)[pc] & (m > 0), np.inf, u)
    c = -sense * class_offset(pc, classes)                       # Eq. (11)
    b = w[-1] * _bot(n, bot_rows)                                # Eq. (13)
    x = np.clip(np.asarray(x, dtype=np.float64), 0.0, u)
    xs = x * (sense / thr)                                       # A x = Phi^T (x * sense / thr), Eq. (12)
    Ax = np.zeros(n)
    for a in range(0, N, _ROW_CHUNK):
        Ax += xs[a:a + _ROW_CHUNK] @ np.asarray(phi[a:a + _ROW_CHUNK], dtype=np.float64)
    pos = Ax > 0
    theta = 1.0
    if np.any(pos):
        theta = min(1.0, float(np.min(b[pos] / Ax[pos])))
    theta = max(theta, 0.0)
    return float(-c @ (theta * x))


def kkt_report(phi, point_class, classes, w, x, t, mask=None, bot_rows=None):
    """Residuals of the optimality conditions of the primal/dual pair (all should be ~0)."""
    c, A, b, u = dual_lp(phi, point_class, classes, w, mask, bot_rows)
    x = np.asarray(x, dtype=np.float64); t = np.asarray(t, dtype=np.float64)
    slack = b - A @ x
    g = c + A.T @ t                       # reduced cost of x given multipliers t
    rep = dict(
        box=float(max(np.max(-x), np.max(x - u), 0.0)),
        row=float(max(np.max(-slack), 0.0)),
        t_neg=float(max(np.max(-t), 0.0)),
        compl_rows=float(np.max(np.abs(t * slack))),
        # g_i > 0 => x_i = 0 ; g_i < 0 => x_i = u_i
        # (a hard class has u = inf: its reduced cost must be >= 0)
        compl_box=float(np.max(np.abs(np.where(g > 0, g * x, np.where(np.isfinite(u), g * (x - np.where(np.isfinite(u), u, 0.0)),
                                                                       np.where(g < -1e-12, np.inf, 0.0)))))),
        gap=float(abs(primal_objective(phi, point_class, classes, w, t, mask, bot_rows) - (-c @ x))),
    )
    return rep

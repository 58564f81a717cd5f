"""O-2PASS: the two-pass optimisation of PAPER.md II.C (:108-114) with the union construction of :144, in fp64 numpy
(test infrastructure; shares no code with the CUDA path).

    pass 1   all B weightings on target points + a geometric low-dose shell                               (II.C.1, first pass)
    dose     d_p = Phi_cand t_p on a grid of candidate points, t_p = the first-pass solution of plan p     (:167, :286)
    volume   V_p = { c : D_LD <= d_p[c] < D_LD + Delta }                                                  (II.C.1, second pass)
    union    the second-pass low-dose points are sampled from the union of the V_p; plan p keeps the points inside V_p, the
             upper bound u of every other low-dose point is set to 0                                      (:144)
    pass 2   all B weightings on target points + the sampled points, with those per-plan bounds

The range test is taken on the dose rounded to fp32 (the CUDA path's dose is fp32: a decision taken from a floating-point value
is taken in the same precision on both sides).  Algorithm 1 (:116-136) is not implemented.
PARITY UNPINNED by the paper (it prints no two-pass numbers); pinned by tests/test_oracle_two_pass.py: the volume definition on a
hand-made dose, mask == row deletion, and pass 2 == a direct solve of the LP restricted to the plan's own points.
"""
from __future__ import annotations

import numpy as np

from . import admm


def lowdose_volumes(phi_cand, t, d_ld: float, delta: float):
    """in_volume [B, N_c] bool and the fp64 dose [B, N_c]."""
    dose = np.asarray(t, dtype=np.float64) @ np.asarray(phi_cand, dtype=np.float64).T
    d32 = dose.astype(np.float32)
    return (d32 >= np.float32(d_ld)) & (d32 < np.float32(d_ld + delta)), dose


def second_pass_problem(phi_target, phi_cand, in_volume, selected):
    """(Phi_2, point_class_2, masks_2 [B, N_2] bool) of the union construction for the selected candidate indices."""
    n_t = phi_target.shape[0]
    sel = np.asarray(selected, dtype=np.int64)
    phi2 = np.concatenate([np.asarray(phi_target), np.asarray(phi_cand)[sel]], axis=0)
    pc2 = np.concatenate([np.zeros(n_t, np.uint8), np.ones(sel.size, np.uint8)])
    masks2 = np.concatenate([np.ones((in_volume.shape[0], n_t), dtype=bool), in_volume[:, sel]], axis=1)
    return phi2, pc2, masks2


def _solve(phi, pc, classes, weights, rho_rule, masks, tol, max_iter):
    pre = admm.precondition(phi, pc, classes)
    rho = rho_rule(weights[:, -1], pc)
    u_hat, b_hat = admm.plan_bounds(pre, pc, classes, weights, masks)
    st = admm.admm_run(pre, u_hat, b_hat, rho, max_iter, tol=tol, presolve=True)
    t, _ = admm.recover(pre, st, rho)
    return dict(t=t, iters=st["iters"], converged=st["converged"], rho=rho)


def two_pass(phi_target, phi_shell, phi_cand, classes, weights, *, d_ld, delta, n_lowdose_2, pick, rho_rule, tol=1e-4, max_iter=3000):
    """rho_rule(w_BOT [B], point_class) -> rho [B] (an input rule shared with the CUDA path's caller, R8)."""
    weights = np.asarray(weights, dtype=np.float64)
    n_t = phi_target.shape[0]
    phi1 = np.concatenate([phi_target, phi_shell], axis=0)
    pc1 = np.concatenate([np.zeros(n_t, np.uint8), np.ones(phi_shell.shape[0], np.uint8)])
    p1 = _solve(phi1, pc1, classes, weights, rho_rule, None, tol, max_iter)
    in_volume, dose = lowdose_volumes(phi_cand, p1["t"], d_ld, delta)
    sel = np.asarray(pick(in_volume.any(axis=0), int(n_lowdose_2)), dtype=np.int64)
    phi2, pc2, masks2 = second_pass_problem(phi_target, phi_cand, in_volume, sel)
    p2 = _solve(phi2, pc2, classes, weights, rho_rule, masks2, tol, max_iter)
    return dict(pass1=p1, pass2=p2, selected=sel, in_volume=in_volume, dose=dose, phi2=phi2, pc2=pc2, masks2=masks2)

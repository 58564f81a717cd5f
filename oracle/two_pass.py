"""O-2PASS: the two-pass optimisation of PAPER.md II.C (:108-114) with the union construction of :144, in fp64 numpy
(test infrastructure; shares no code with the CUDA path).

    pass 1   all B weightings on target points + a geometric low-dose shell                               (II.C.1, first pass)
    dose     d_p = Phi_cand t_p on a grid of candidate points, t_p = the first-pass solution of plan p     (:167, :286)
    volume   V_p = { c : D_LD <= d_p[c] < D_LD + Delta }                                                  (II.C.1, second pass)
    union    the second-pass low-dose points are sampled from the union of the V_p; plan p keeps the points inside V_p, the
             upper bound u of every other low-dose point is set to 0                                      (:144)
    pass 2   all B weightings on target points + the sampled points, with those per-plan bounds

The range test is taken on the dose rounded to fp32 (the CUDA path's dose is fp32: a decision taken from a floating-point value
is taken in the same precision on both sides).

Algorithm 1 (:116-136, "Overlapping low-dose point sampling") is `overlapping_sampling` below, written line by line on a discrete
patient volume: a volume V_j is a set of candidate-grid indices, |V| its number of candidates, "sample k points from a set" = the k
members with the smallest value of a counter-based uniform u(stream, index) (workloads.uniform01: the random numbers are an input both
sides draw from the same generator), non-integer counts rounded to nearest.

PARITY UNPINNED by the paper (it prints no two-pass numbers); pinned by tests/test_oracle_two_pass.py: the volume definition on a
hand-made dose, mask == row deletion, pass 2 == a direct solve of the LP restricted to the plan's own points; for Algorithm 1:
disjoint volumes get exactly their N_LD points, identical volumes share all of them, p_j lies in V_j, and the spread of |p_j| over
seeds respects the bound of Eq. (8).
"""
from __future__ import annotations

import numpy as np

from . import admm


def lowdose_volumes(phi_cand, t, d_ld: float, delta: float):
    """in_volume [B, N_c] bool and the fp64 dose [B, N_c]."""
    dose = np.asarray(t, dtype=np.float64) @ np.asarray(phi_cand, dtype=np.float64).T
    d32 = dose.astype(np.float32)
    return (d32 >= np.float32(d_ld)) & (d32 < np.float32(d_ld + delta)), dose


def _sample(members, k, stream, uniform01):
    """the k members (a list of candidate indices) with the smallest u(stream, index); all of them if k >= len(members)"""
    members = sorted(members)
    k = int(k)
    if k >= len(members):
        return set(members)
    if k <= 0:
        return set()
    u = uniform01(stream, np.array(members, dtype=np.uint64))
    order = np.argsort(u, kind="stable")[:k]
    return {members[i] for i in order}


def overlapping_sampling(volumes, n_ld, seed: int, uniform01):
    """Algorithm 1 (:116-136).  volumes: [m, N_c] bool (V_j = the candidates inside plan j's low-dose volume); n_ld: [m] desired
    number of low-dose points N_LD,j; returns (P sorted list of candidate indices, p [m] list of sets, order).  The volumes are
    processed in the order of decreasing sampling density w_j = N_LD,j / |V_j| (:146); empty volumes get no points."""
    volumes = np.asarray(volumes, dtype=bool)
    m = volumes.shape[0]
    V = [set(np.nonzero(volumes[j])[0].tolist()) for j in range(m)]
    size = np.array([len(v) for v in V], dtype=np.float64)
    with np.errstate(divide="ignore", invalid="ignore"):
        omega = np.where(size > 0, np.asarray(n_ld, dtype=np.float64) / size, -1.0)
    order = [int(j) for j in np.argsort(-omega, kind="stable") if size[j] > 0]
    base = 2 * int(seed) * (m + 1)
    V_union, p_union = set(), set()                                     # line 1
    p = [set() for _ in range(m)]
    for step, j in enumerate(order):                                    # line 2
        w = min(float(omega[j]), 1.0)
        p_tilde = _sample(p_union, round(w * len(V_union)), base + 2 * step, uniform01)          # line 3
        p_in = p_tilde & V[j]                                                                      # line 4
        fresh = V[j] - V_union
        p_out = _sample(fresh, round(w * len(fresh)), base + 2 * step + 1, uniform01)              # line 5
        p[j] = p_in | p_out                                                                        # line 6
        p_union = p_tilde | p_out                                                                  # line 7
        V_union = V[j] | V_union                                                                   # line 8
    P = sorted(set().union(*p)) if m else []                                                       # line 9
    return P, p, order


def second_pass_problem_alg1(phi_target, phi_cand, P, p):
    """(Phi_2, point_class_2, masks_2) when the low-dose points are Algorithm 1's P and plan j keeps p_j."""
    n_t = phi_target.shape[0]
    P = np.asarray(P, dtype=np.int64)
    phi2 = np.concatenate([np.asarray(phi_target), np.asarray(phi_cand)[P]], axis=0)
    pc2 = np.concatenate([np.zeros(n_t, np.uint8), np.ones(P.size, np.uint8)])
    pos = {int(c): i for i, c in enumerate(P)}
    masks2 = np.zeros((len(p), n_t + P.size), dtype=bool)
    masks2[:, :n_t] = True
    for j, pj in enumerate(p):
        for c in pj:
            masks2[j, n_t + pos[int(c)]] = True
    return phi2, pc2, masks2


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

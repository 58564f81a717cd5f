"""Pins of oracle/two_pass.py (PAPER.md II.C, :108-114, :144).  CPU only."""
import numpy as np

from oracle import lp_model, simplex, two_pass as o2
from workloads import make_candidates, make_workload, pick_from_union, scaled_rho


def test_volume_is_the_half_open_dose_range():
    """II.C.1: the second-pass low-dose volume of a plan is where its first-pass dose lies in [D_LD, D_LD + Delta)."""
    phi_cand = np.eye(6, dtype=np.float32)                      # candidate c sees only time variable c: dose = t
    t = np.array([[0.49, 0.5, 0.6, 0.7499, 0.75, 2.0],
                  [0.0, 0.0, 0.0, 0.0, 0.0, 0.0]])
    inv, dose = o2.lowdose_volumes(phi_cand, t, 0.5, 0.25)
    assert np.array_equal(dose, t)
    assert inv.tolist() == [[False, True, True, True, False, False], [False] * 6]


def test_union_sampling_is_reproducible_and_uniform():
    union = np.zeros(5000, dtype=bool); union[100:4100] = True
    a = pick_from_union(union, 1000, seed=3)
    assert a.size == 1000 and np.all(union[a]) and np.all(np.diff(a) > 0)
    assert np.array_equal(a, pick_from_union(union, 1000, seed=3)) and not np.array_equal(a, pick_from_union(union, 1000, seed=4))
    assert abs(np.mean(a) - 2100) < 4 * 4000 / np.sqrt(12 * 1000)              # mean of a uniform sample of the members
    assert np.array_equal(pick_from_union(union, 99999, seed=3), np.nonzero(union)[0])   # fewer members than asked for: all of them


def test_second_pass_of_a_plan_is_the_lp_on_its_own_points():
    """:144: zeroing u outside a plan's volume == deleting those rows.  The oracle's two-pass result for plan p must reach the
    simplex optimum of the LP built from the target points and ONLY the sampled points inside V_p."""
    w = make_workload(1, n_target=60, n_lowdose=120, n_iso=1, grid=3)           # n = 24
    _, phic = make_candidates(w, 400)
    nt = int((w.point_class == 0).sum())
    res = o2.two_pass(w.phi[:nt], w.phi[nt:], phic, w.classes, w.weights, d_ld=0.5, delta=0.5, n_lowdose_2=80,
                      pick=lambda u, c: pick_from_union(u, c, 11), rho_rule=scaled_rho, tol=1e-5, max_iter=6000)
    vols = res["in_volume"].sum(axis=1)
    assert (vols > 0).sum() >= 3 and res["selected"].size > 20
    checked = 0
    for p in range(w.B):
        if not res["pass2"]["converged"][p] or w.beta[p] == 0:
            continue
        own = res["masks2"][p]
        if own[nt:].sum() == 0:
            continue
        phi_own, pc_own = res["phi2"][own], res["pc2"][own]
        opt = simplex.solve_plan(phi_own, pc_own, w.classes, w.weights[p])["opt"]
        P = lp_model.primal_objective(res["phi2"], res["pc2"], w.classes, w.weights[p], res["pass2"]["t"][p], res["masks2"][p])
        assert abs(P - opt) / max(abs(opt), 0.1) < 1e-3, (p, P, opt)
        checked += 1
    assert checked >= 2

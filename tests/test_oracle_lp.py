"""Pins for O-LP (oracle/simplex.py, oracle/lp_model.py): vertex enumeration, KKT, closed forms,
an independent LP solver.  CPU only."""
import os

import numpy as np
import pytest

from oracle import enumerate as vertex_enum
from oracle import lp_model, simplex
from workloads import make_tiny_workload, make_workload

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "c0_simplex_opt.txt")


def _golden():
    return np.loadtxt(GOLDEN)


@pytest.mark.parametrize("seed,NT,NL,n", [(1, 5, 7, 2), (2, 6, 8, 3), (3, 4, 6, 4), (4, 8, 8, 3)])
def test_simplex_equals_vertex_enumeration(seed, NT, NL, n):
    w = make_tiny_workload(seed, NT, NL, n)
    for p in range(w.B):
        bf, _ = vertex_enum.brute_force_optimum(w.phi, w.point_class, w.classes, w.weights[p])
        sx = simplex.solve_plan(w.phi, w.point_class, w.classes, w.weights[p])
        assert sx["opt"] == pytest.approx(bf, abs=1e-10)
        # the multipliers are a primal optimum too: P(t*) = OPT (zero duality gap)
        P = lp_model.primal_objective(w.phi, w.point_class, w.classes, w.weights[p], sx["t"])
        assert P == pytest.approx(bf, abs=1e-10)


def test_simplex_with_row_mask_equals_enumeration():
    w = make_tiny_workload(11, 5, 9, 3)
    rng_mask = np.ones(w.N, dtype=bool)
    rng_mask[[6, 9, 12]] = False                       # three low-dose rows inactive (u = 0)
    for p in range(w.B):
        bf, _ = vertex_enum.brute_force_optimum(w.phi, w.point_class, w.classes, w.weights[p], rng_mask)
        sx = simplex.solve_plan(w.phi, w.point_class, w.classes, w.weights[p], rng_mask)
        assert sx["opt"] == pytest.approx(bf, abs=1e-10)
    # masking rows must equal deleting them (R12: the mean is over the ACTIVE count)
    keep = rng_mask
    for p in (4, 7):
        a = simplex.solve_plan(w.phi, w.point_class, w.classes, w.weights[p], rng_mask)["opt"]
        b = simplex.solve_plan(w.phi[keep], w.point_class[keep], w.classes, w.weights[p])["opt"]
        assert a == pytest.approx(b, abs=1e-11)


def test_one_variable_closed_form():
    """n = 1: P is piecewise linear in the scalar t; the optimum is at t=0 or at a breakpoint thr_i/phi_i."""
    w = make_tiny_workload(21, 9, 14, 1)
    _, _, thr = lp_model.class_arrays(w.point_class, w.classes)
    cand = np.concatenate([[0.0], thr / w.phi[:, 0].astype(np.float64)])
    for p in range(w.B):
        vals = [lp_model.primal_objective(w.phi, w.point_class, w.classes, w.weights[p], np.array([t])) for t in cand]
        sx = simplex.solve_plan(w.phi, w.point_class, w.classes, w.weights[p])
        assert sx["opt"] == pytest.approx(min(vals), abs=1e-11)


def test_trivial_plan_closed_form():
    """If w_BOT >= max_j mean_T(Phi_ij) * w_T then t* = 0 and OPT = w_T exactly (directional
    derivative of P at t=0 is >= 0 in every coordinate; low-dose terms are inactive at zero dose)."""
    w = make_workload(0, n_target=300, n_lowdose=500, n_iso=4)
    bound = w.phi[w.point_class == 0].astype(np.float64).mean(axis=0).max()
    for alpha in (0.0, 0.7):
        wt = np.array([1.0, alpha, bound * (1 + 1e-9)])
        sx = simplex.solve_plan(w.phi, w.point_class, w.classes, wt)
        assert sx["opt"] == pytest.approx(1.0, abs=1e-9)
        # just below the threshold the optimum drops under 1
        wt2 = np.array([1.0, alpha, bound * 0.98])
        assert simplex.solve_plan(w.phi, w.point_class, w.classes, wt2)["opt"] < 1.0 - 1e-6


def test_kkt_and_duality_gap_config0_and_golden():
    w = make_workload(0)
    g = _golden()
    for p in (1, 3, 4, 8):
        sx = simplex.solve_plan(w.phi, w.point_class, w.classes, w.weights[p])
        rep = lp_model.kkt_report(w.phi, w.point_class, w.classes, w.weights[p], sx["x"], sx["t"])
        for k, v in rep.items():
            assert v < 1e-8, (p, k, v)
        assert sx["opt"] == pytest.approx(g[p, 3], rel=1e-9, abs=1e-12)
        assert (g[p, 1], g[p, 2]) == (w.alpha[p], w.beta[p])


def test_simplex_matches_independent_solver():
    """HiGHS (scipy) on the PRIMAL with explicit slack variables -- a different formulation and a
    different algorithm from oracle/simplex.py."""
    scipy_opt = pytest.importorskip("scipy.optimize")
    w = make_workload(0, n_target=200, n_lowdose=400, n_iso=3)
    N, n = w.N, w.n
    phi = w.phi.astype(np.float64)
    pc = w.point_class.astype(int)
    for p in (1, 4, 6, 7):
        wt = w.weights[p]
        NT, NL = (pc == 0).sum(), (pc == 1).sum()
        # variables [t (n), e (N)] ; min beta*sum t + sum_i coef_i e_i ; e_i >= s_i (thr_i - phi_i t)
        coef = np.where(pc == 0, wt[0] / NT, wt[1] / NL)
        cvec = np.concatenate([np.full(n, wt[2]), coef])
        s = np.where(pc == 0, 1.0, -1.0); thr = np.where(pc == 0, 1.0, 0.5)
        # -s_i phi_i t - e_i <= -s_i thr_i
        A_ub = np.concatenate([-(s[:, None] * phi), -np.eye(N)], axis=1)
        b_ub = -s * thr
        res = scipy_opt.linprog(cvec, A_ub=A_ub, b_ub=b_ub, bounds=[(0, None)] * (n + N), method="highs")
        assert res.status == 0
        sx = simplex.solve_plan(w.phi, w.point_class, w.classes, wt)
        assert sx["opt"] == pytest.approx(res.fun, abs=1e-8)


def test_dual_bound_brackets_optimum():
    w = make_workload(0, n_target=200, n_lowdose=400, n_iso=3)
    rng = np.random.default_rng(0)
    for p in (1, 4, 7):
        sx = simplex.solve_plan(w.phi, w.point_class, w.classes, w.weights[p])
        # exact x* gives the optimum; a perturbed x still gives a valid lower bound; any t>=0 an upper bound
        assert lp_model.dual_bound(w.phi, w.point_class, w.classes, w.weights[p], sx["x"]) == pytest.approx(sx["opt"], abs=1e-9)
        xp = sx["x"] * (1 + 0.3 * rng.standard_normal(w.N))
        assert lp_model.dual_bound(w.phi, w.point_class, w.classes, w.weights[p], xp) <= sx["opt"] + 1e-12
        tp = np.abs(sx["t"] * (1 + 0.3 * rng.standard_normal(w.n)))
        assert lp_model.primal_objective(w.phi, w.point_class, w.classes, w.weights[p], tp) >= sx["opt"] - 1e-12


def _three_class_tiny(seed, NT, NL, NO, n):
    """Tiny unstructured instance with a target class, a soft low-dose class and a HARD organ-at-risk class (dose <= 0.3)."""
    from workloads import ClassSpec, Workload, uniform01
    N = NT + NL + NO
    phi = uniform01(seed, np.arange(N * n)).reshape(N, n).astype(np.float32)
    pc = np.concatenate([np.zeros(NT, np.uint8), np.ones(NL, np.uint8), np.full(NO, 2, np.uint8)])
    classes = [ClassSpec(+1, 1.0), ClassSpec(-1, 0.5), ClassSpec(-1, 0.3, hard=1)]
    ab = [(0.5, 0.0), (0.5, 0.2), (1.0, 0.05), (0.0, 0.4)]
    weights = np.array([[1.0, a, 7.0, b_] for a, b_ in ab])          # the hard class's weight (7) must not matter
    return Workload(name=f"tiny3c{seed}", config=-1, phi=phi, point_class=pc, classes=classes, weights=weights, row_mask=None,
                    alpha=np.array([a for a, _ in ab]), beta=np.array([b_ for _, b_ in ab]))


@pytest.mark.parametrize("seed,NT,NL,NO,n", [(31, 5, 5, 3, 2), (32, 4, 6, 4, 3), (33, 6, 4, 2, 3)])
def test_hard_class_simplex_equals_vertex_enumeration(seed, NT, NL, NO, n):
    """PAPER.md:322 (Eq. 15, u = infinity for organs at risk): with a hard class the primal has constraints Phi_i t <= thr on those
    rows.  The simplex on the dual with unbounded variables must find the optimum the brute-force enumeration of the constrained
    primal finds, its multipliers must be feasible for the hard rows, and the hard class's weight must not enter."""
    w = _three_class_tiny(seed, NT, NL, NO, n)
    for p in range(w.B):
        bf, t_bf = vertex_enum.brute_force_optimum(w.phi, w.point_class, w.classes, w.weights[p])
        sx = simplex.solve_plan(w.phi, w.point_class, w.classes, w.weights[p])
        assert np.isfinite(bf) and sx["opt"] == pytest.approx(bf, abs=1e-10)
        assert lp_model.hard_violation(w.phi, w.point_class, w.classes, sx["t"]) < 1e-9
        P = lp_model.primal_objective(w.phi, w.point_class, w.classes, w.weights[p], sx["t"])
        assert P == pytest.approx(bf, abs=1e-9)
        w2 = w.weights[p].copy(); w2[2] = 0.0
        assert simplex.solve_plan(w.phi, w.point_class, w.classes, w2)["opt"] == pytest.approx(bf, abs=1e-12)
    # the hard rows bind somewhere: dropping the class changes at least one optimum
    soft_only = w.point_class < 2
    changed = [abs(simplex.solve_plan(w.phi[soft_only], w.point_class[soft_only], w.classes[:2], w.weights[p][[0, 1, 3]])["opt"]
                   - simplex.solve_plan(w.phi, w.point_class, w.classes, w.weights[p])["opt"]) > 1e-6 for p in range(w.B)]
    assert any(changed)

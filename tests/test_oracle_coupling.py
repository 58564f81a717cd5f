"""Pins of the sector / isocenter coupling of PAPER.md App. A (Eq. 12, 16, 17, :316, :330-332) in the oracle's LP model,
simplex and ADMM.  CPU only."""
import numpy as np
import pytest

from oracle import admm, enumerate as enum, lp_model, simplex
from workloads import ClassSpec, make_workload, scaled_rho, with_sector_coupling


def test_structure_of_the_coupled_problem():
    w0 = make_workload(0, n_target=40, n_lowdose=60, n_iso=2, grid=3)                # n = 48
    w = with_sector_coupling(w0)
    assert w.n == 48 + 2 and w.N == 100 + 16 and w.bot_rows.tolist() == [0] * 48 + [1, 1]
    C = -w.phi[100:, :48]; T = w.phi[100:, 48:]
    assert np.array_equal(C, np.kron(np.kron(np.eye(2), np.eye(8)), np.ones((1, 3))).astype(np.float32))     # Eq. (16)
    assert np.array_equal(T, np.kron(np.eye(2), np.ones((8, 1))).astype(np.float32))                         # Eq. (17)
    c, A, b, u = lp_model.dual_lp(w.phi, w.point_class, w.classes, w.weights[4], None, w.bot_rows)
    assert np.all(c[100:] == 0) and np.all(np.isinf(u[100:])) and np.all(b[:48] == 0) and np.all(b[48:] == w.weights[4, -1])   # Eq. (11), (13), (15)


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_simplex_equals_vertex_enumeration_with_a_coupling_row(seed):
    """One 'sector' of two 'collimators' and its isocenter time (3 variables): the simplex on the extended dual against brute-force
    enumeration of the vertices of the constrained primal."""
    rng = np.random.default_rng(seed)
    phi = np.zeros((9, 3))
    phi[:8, :2] = rng.uniform(0.1, 1.5, (8, 2))
    phi[8] = [-1.0, -1.0, 1.0]                                                       # t1 + t2 <= tau
    pc = np.array([0] * 4 + [1] * 4 + [2], dtype=np.uint8)
    classes = [ClassSpec(+1, 1.0), ClassSpec(-1, 0.5), ClassSpec(+1, 1.0, hard=2)]
    bot = np.array([0, 0, 1])
    for w in ([1.0, 0.5, 0.0, 0.3], [1.0, 0.0, 0.0, 0.05], [1.0, 1.0, 0.0, 1.0]):
        opt = simplex.solve_plan(phi, pc, classes, w, bot_rows=bot)
        best, t_best = enum.brute_force_optimum(phi, pc, classes, w, bot_rows=bot)
        assert abs(opt["opt"] - best) < 1e-9, (w, opt["opt"], best)
        assert abs(lp_model.primal_objective(phi, pc, classes, w, opt["t"], bot_rows=bot) - opt["opt"]) < 1e-9      # zero duality gap
        assert lp_model.hard_violation(phi, pc, classes, opt["t"]) < 1e-9
        if opt["opt"] < 1.0 - 1e-9:                                                  # some dose is delivered: tau is the sector's time
            assert abs(opt["t"][2] - (opt["t"][0] + opt["t"][1])) < 1e-9


def test_coupled_lp_against_an_independent_primal_solver():
    """The extended dual (simplex) against HiGHS on the primal written out by hand: min sum_k w_k/N_k sum e_i + w_BOT sum tau,
    e_i >= s_i (thr_i - Phi_i t), sum_c t_(iso,s,c) <= tau_iso, everything >= 0."""
    from scipy.optimize import linprog
    w0 = make_workload(0, n_target=30, n_lowdose=50, n_iso=2, grid=3)
    w = with_sector_coupling(w0)
    N0, n0, n_iso = w0.N, w0.n, 2
    sense = np.array([+1.0] * 30 + [-1.0] * 50); thr = np.array([1.0] * 30 + [0.5] * 50)
    for p in (1, 4, 5, 8):
        wT, wL, wB = w0.weights[p]
        cost = np.concatenate([np.zeros(n0), wB * np.ones(n_iso), np.array([wT / 30] * 30 + [wL / 50] * 50)])
        # -s_i Phi_i t - e_i <= -s_i thr_i
        A1 = np.concatenate([-(sense[:, None] * w0.phi.astype(np.float64)), np.zeros((N0, n_iso)), -np.eye(N0)], axis=1)
        b1 = -sense * thr
        A2 = np.zeros((8 * n_iso, n0 + n_iso + N0))
        for k in range(8 * n_iso):
            A2[k, 3 * k:3 * k + 3] = 1.0; A2[k, n0 + k // 8] = -1.0
        r = linprog(cost, A_ub=np.concatenate([A1, A2]), b_ub=np.concatenate([b1, np.zeros(8 * n_iso)]), bounds=(0, None), method="highs")
        assert r.status == 0
        opt = simplex.solve_plan(w.phi, w.point_class, w.classes, w.weights[p], bot_rows=w.bot_rows)
        assert abs(opt["opt"] - r.fun) < 1e-7 * max(1.0, abs(r.fun)), (p, opt["opt"], r.fun)


def test_oracle_admm_converges_to_the_coupled_optimum():
    w0 = make_workload(0, n_target=120, n_lowdose=240, n_iso=2, grid=3)
    w = with_sector_coupling(w0)
    rho = scaled_rho(w.beta, w0.point_class)
    st = admm.solve_workload(w, rho, 20000, tol=1e-5)
    checked = 0
    for p in range(w.B):
        if not st["converged"][p] or w.beta[p] == 0:
            continue
        opt = simplex.solve_plan(w.phi, w.point_class, w.classes, w.weights[p], bot_rows=w.bot_rows)["opt"]
        assert abs(st["obj"][p] - opt) / max(abs(opt), 0.1) < 1e-3, (p, st["obj"][p], opt)
        assert st["hard_violation"][p] < 1e-3
        checked += 1
    assert checked >= 4

"""Pins for O-ADMM (oracle/admm.py).  The paper prints no iterate, so the iteration is pinned by
what the mathematics fixes: the x-update solved two other ways (Eq. 5 sign-corrected as one KKT
system; the N x N normal equations of Eq. 4a), invariants, the fixed point at the simplex KKT
point, metamorphic relations and convergence to the exact LP optimum.  CPU only."""
import os

import numpy as np
import pytest

from oracle import admm, lp_model, simplex
from workloads import default_rho, make_workload, scaled_rho

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "c0_simplex_opt.txt")


@pytest.fixture(scope="module")
def small():
    w = make_workload(0, n_target=180, n_lowdose=320, n_iso=3)       # N=500, n=72, B=9
    pre = admm.precondition(w.phi, w.point_class, w.classes)
    u_hat, b_hat = admm.plan_bounds(pre, w.point_class, w.classes, w.weights)
    rho = default_rho(w.beta)
    return w, pre, u_hat, b_hat, rho


def _x_of_step(before, after):
    """x^{k+1} from consecutive states via (4c): x = y+ - y + z+."""
    return (after["y1"] - before["y1"] + after["z1"], after["y2"] - before["y2"] + after["z2"])


def test_schur_complement_structure(small):
    """after row normalisation diag(S) = 2 and off-diagonals lie in [-1, 1]."""
    _, pre, *_ = small
    assert np.allclose(np.diag(pre.S), 2.0, atol=1e-12)
    off = pre.S - np.diag(np.diag(pre.S))
    assert np.max(np.abs(off)) <= 1.0 + 1e-12
    assert np.allclose(np.sum(pre.A_hat ** 2, axis=1), 1.0, atol=1e-12)


def test_x_update_is_the_constrained_least_squares(small):
    """(6)+(7) must equal (a) the sign-corrected Eq. (5) solved as one dense system and (b) the
    minimiser of (4a) from its N x N normal equations (the S' = A^T A + I route of :104)."""
    w, pre, u_hat, b_hat, rho = small
    s0 = admm.admm_run(pre, u_hat, b_hat, rho, 7)
    s1 = admm.admm_run(pre, u_hat, b_hat, rho, 1, state0=(s0["z1"], s0["y1"], s0["z2"], s0["y2"]))
    x1, x2 = _x_of_step(s0, s1)
    A = pre.A_hat
    n, N = A.shape
    for p in (1, 4, 8):
        r1 = s0["z1"][:, p] - s0["y1"][:, p] - pre.c_hat / rho[p]
        r2 = s0["z2"][:, p] - s0["y2"][:, p]
        K = np.block([[np.eye(N), A.T], [A, -np.eye(n)]])          # Eq. (5) with the (2,2) block -I (R4)
        sol = np.linalg.solve(K, np.concatenate([r1, r2]))
        assert np.allclose(sol[:N], x1[:, p], atol=1e-10)
        assert np.allclose(sol[N:] + r2, x2[:, p], atol=1e-10)    # x2 = v + z2 - y2
        x1_ne = np.linalg.solve(np.eye(N) + A.T @ A, r1 + A.T @ r2)
        assert np.allclose(x1_ne, x1[:, p], atol=1e-10)
        # the PRINTED Eq. (5) (+I) disagrees by O(1): documents the typo reading R4
        bad = np.linalg.solve(np.block([[np.eye(N), A.T], [A, np.eye(n)]]), np.concatenate([r1, r2]))
        assert np.max(np.abs(bad[:N] - x1[:, p])) > 1e-3 * np.max(np.abs(x1[:, p]))


def test_invariants_every_iteration(small):
    w, pre, u_hat, b_hat, rho = small
    st = admm.admm_run(pre, u_hat, b_hat, rho, 0)
    state = (st["z1"], st["y1"], st["z2"], st["y2"])
    prev = st
    for k in range(12):
        cur = admm.admm_run(pre, u_hat, b_hat, rho, 1, state0=state)
        x1, x2 = _x_of_step(prev, cur)
        assert np.allclose(pre.A_hat @ x1, x2, atol=1e-9)                       # (x1,x2) in the set A
        z1, y1, z2, y2 = cur["z1"], cur["y1"], cur["z2"], cur["y2"]
        assert np.all(z1 >= 0) and np.all(z1 <= u_hat + 1e-15) and np.all(z2 <= b_hat + 1e-15)
        assert np.all(y2 >= -1e-15)                                             # multiplier of z2 <= b
        assert np.all(z1[y1 > 1e-12] == u_hat[y1 > 1e-12])                      # complementarity by construction
        assert np.all(z1[y1 < -1e-12] == 0.0)
        assert np.all(z2[y2 > 1e-12] == b_hat[y2 > 1e-12])
        state = (z1, y1, z2, y2); prev = cur


def test_single_state_form_equals_three_variable_form(small):
    """s = x+ + y  =>  z = Pi(s), y+ = s - z (derived from 4b/4c); the CUDA path stores only s."""
    w, pre, u_hat, b_hat, rho = small
    A = pre.A_hat
    n, N = A.shape
    B = len(rho)
    Sinv = np.linalg.inv(pre.S)
    s1 = np.zeros((N, B)); s2 = np.zeros((n, B))
    cr = pre.c_hat[:, None] / rho[None, :]
    for _ in range(40):
        z1 = np.clip(s1, 0, u_hat); z2 = np.minimum(s2, b_hat)
        v = Sinv @ (A @ (2 * z1 - s1 - cr) - (2 * z2 - s2))
        s1 = z1 - cr - A.T @ v
        s2 = z2 + v
    ref = admm.admm_run(pre, u_hat, b_hat, rho, 40)
    assert np.allclose(np.clip(s1, 0, u_hat), ref["z1"], atol=1e-10)
    assert np.allclose(s1 - np.clip(s1, 0, u_hat), ref["y1"], atol=1e-10)
    assert np.allclose(np.minimum(s2, b_hat), ref["z2"], atol=1e-9)
    assert np.allclose(s2 - np.minimum(s2, b_hat), ref["y2"], atol=1e-9)


def test_fixed_point_at_simplex_kkt_point(small):
    """Start at the exact LP solution: z1 = x*/D, y2 = t*/(rho R), y1 = -(c_hat + A_hat^T t_hat)/rho,
    z2 = A_hat z1.  One iteration must leave it unchanged (z1 -> x*, rho*y2 -> t*)."""
    w, pre, u_hat, b_hat, rho = small
    for p in (1, 4, 5, 7):
        sx = simplex.solve_plan(w.phi, w.point_class, w.classes, w.weights[p])
        z1 = sx["x"] / pre.D
        y2 = sx["t"] / (rho[p] * pre.R)
        y1 = -(pre.c_hat + pre.A_hat.T @ (rho[p] * y2)) / rho[p]
        z2 = pre.A_hat @ z1
        st0 = tuple(a[:, None] for a in (z1, y1, z2, y2))
        out = admm.admm_run(pre, u_hat[:, [p]], b_hat[:, [p]], rho[[p]], 1, state0=st0)
        scale = max(1.0, np.max(np.abs(y1)))
        for name, ref in zip(("z1", "y1", "z2", "y2"), st0):
            assert np.max(np.abs(out[name] - ref)) < 1e-8 * scale, (p, name)


def test_objective_scaling_metamorphic(small):
    """Weights * kappa with rho / kappa: iterates scale by kappa, times t are unchanged."""
    w, pre, u_hat, b_hat, rho = small
    kappa = 3.7
    a = admm.admm_run(pre, u_hat, b_hat, rho, 25)
    u2, b2 = admm.plan_bounds(pre, w.point_class, w.classes, w.weights * kappa)
    b = admm.admm_run(pre, u2, b2, rho / kappa, 25)
    for k in ("z1", "y1", "z2", "y2"):
        assert np.allclose(b[k], kappa * a[k], rtol=1e-9, atol=1e-12)
    ta, _ = admm.recover(pre, a, rho); tb, _ = admm.recover(pre, b, rho / kappa)
    assert np.allclose(ta, tb, rtol=1e-9, atol=1e-14)


def test_point_permutation_and_batch_independence(small):
    w, pre, u_hat, b_hat, rho = small
    ref = admm.admm_run(pre, u_hat, b_hat, rho, 20)
    perm = np.random.default_rng(5).permutation(w.N)
    pre2 = admm.precondition(w.phi[perm], w.point_class[perm], w.classes)
    u2, b2 = admm.plan_bounds(pre2, w.point_class[perm], w.classes, w.weights)
    out = admm.admm_run(pre2, u2, b2, rho, 20)
    assert np.allclose(out["z1"], ref["z1"][perm], atol=1e-10)
    assert np.allclose(out["y2"], ref["y2"], atol=1e-9)
    one = admm.admm_run(pre, u_hat[:, [6]], b_hat[:, [6]], rho[[6]], 20)       # plan alone == plan in batch (:96)
    assert np.allclose(one["z1"][:, 0], ref["z1"][:, 6], atol=1e-12)
    assert np.allclose(one["y2"][:, 0], ref["y2"][:, 6], atol=1e-12)


def test_row_mask_equals_deleting_rows():
    """zeroing u for rows outside a plan's low-dose set == solving without those rows
    (same objective; the shared A keeps the rows, so iterates differ but the limit does not)."""
    w = make_workload(0, n_target=150, n_lowdose=250, n_iso=2)
    mask = np.ones(w.N, dtype=bool); mask[150::3] = False
    p = 4
    full = simplex.solve_plan(w.phi, w.point_class, w.classes, w.weights[p], mask)["opt"]
    pre = admm.precondition(w.phi, w.point_class, w.classes)
    u_hat, b_hat = admm.plan_bounds(pre, w.point_class, w.classes, w.weights[[p]], mask[None, :])
    assert np.all(u_hat[~mask, 0] == 0.0)
    rho = default_rho(w.beta[[p]])
    st = admm.admm_run(pre, u_hat, b_hat, rho, 4000, tol=1e-5)
    t, _ = admm.recover(pre, st, rho)
    P = lp_model.primal_objective(w.phi, w.point_class, w.classes, w.weights[p], t[0], mask)
    assert abs(P - full) / max(abs(full), 0.1) < 1e-3


def test_converges_to_simplex_optimum_config0():
    """PAPER.md:80 + north_star: converged objectives within 1e-3 relative of the simplex optimum
    (error = |P - OPT| / max(|OPT|, 0.1), reading R15).  beta > 0 plans of config 0."""
    g = np.loadtxt(GOLDEN)
    plans = [1, 2, 4, 5, 7, 8, 0]
    w = make_workload(0, plans=plans)
    rho = default_rho(w.beta)
    st = admm.solve_workload(w, rho, 3000, tol=1e-4)
    assert st["converged"].all()
    assert np.all(st["iters"] % 10 == 0)
    err = np.abs(st["obj"] - g[plans, 3]) / np.maximum(np.abs(g[plans, 3]), 0.1)
    assert np.all(err < 1e-3), err
    # and the weak-duality bracket closes: Dual(lambda) <= OPT <= P(t)
    masks = None
    for i, p in enumerate(plans[:3]):
        lo = lp_model.dual_bound(w.phi, w.point_class, w.classes, w.weights[i], st["lam"][i])
        assert lo <= g[p, 3] + 1e-9 <= st["obj"][i] + 2e-9
        assert (st["obj"][i] - lo) / max(abs(st["obj"][i]), 0.1) < 2e-3


def test_stopping_rule_freezes_converged_plans(small):
    w, pre, u_hat, b_hat, rho = small
    a = admm.admm_run(pre, u_hat, b_hat, rho, 400, tol=1e-3, check_every=10)
    assert a["converged"].any() and not np.all(a["iters"] == a["iters"][0])
    p = int(np.argmin(a["iters"]))
    k = int(a["iters"][p])
    b = admm.admm_run(pre, u_hat, b_hat, rho, k)                                # frozen state == state after k its
    assert np.array_equal(a["z1"][:, p], b["z1"][:, p]) and np.array_equal(a["y2"][:, p], b["y2"][:, p])


def test_stopping_rule_hand_computed_two_plan_case():
    """Reading R7 pinned by a case small enough to iterate by hand: N = n = 1, one target point with Phi = 2, w_T = 1,
    rho = 1.  Then A^ = 1 (row normalised), c^ = -1, u^ = 1, S = 2, b^ = beta / 2, and Eq. (6)/(7) reduce to
    x1 = x2 = (r1 + r2) / 2.  Plan a: beta = 0.5 (b^ = 0.25); plan b: beta = 4 (b^ = 2).  By hand:
      a, k=1: x = .5  z = (.5, .25) y = (0, .25)   rp = .25  rd = sqrt(.3125)  |x| = sqrt(.5)   |z| = sqrt(.3125)  |y| = .25
      a, k=2: x = .75 z = (.75, .25) y = (0, .75)  rp = .5   rd = .25          |x| = .75 sqrt2  |z| = sqrt(.625)   |y| = .75
      b, k=1: x = .5  z = (.5, .5)  y = 0          rp = 0    rd = sqrt(.5)     |x| = sqrt(.5)   |z| = sqrt(.5)     |y| = 0
      b, k=2: x = 1   z = (1, 1)    y = 0          rp = 0    rd = sqrt(.5)     |x| = sqrt2      |z| = sqrt2        |y| = 0
    Decisions (eps_abs = 0): plan a with tol = .5 fails at k = 1 (rd = .559 > .5 * .25) and passes at k = 2
    (rp = .5 <= .5 * 1.0607, rd = .25 <= .5 * .75); with tol = .3 it fails at k = 2 (rp = .5 > .318).
    Plan b never passes the dual test while y = 0 (rd > 0 = tol |y|) unless eps_abs sqrt(N + n) covers rd."""
    from workloads import ClassSpec
    phi = np.array([[2.0]], dtype=np.float32)
    pc = np.zeros(1, np.uint8)
    classes = [ClassSpec(+1, 1.0)]
    weights = np.array([[1.0, 0.5], [1.0, 4.0]])
    pre = admm.precondition(phi, pc, classes)
    assert np.allclose(pre.A_hat, 1.0) and np.allclose(pre.c_hat, -1.0) and np.allclose(pre.S, 2.0)
    u_hat, b_hat = admm.plan_bounds(pre, pc, classes, weights)
    assert np.allclose(u_hat, 1.0) and np.allclose(b_hat, [[0.25, 2.0]])
    rho = np.ones(2)
    h = admm.admm_run(pre, u_hat, b_hat, rho, 2, history=True)["history"]          # [k, plan, (rp, rd, |x|, |z|, |y|)]
    s = np.sqrt
    hand = np.array([[[.25, s(.3125), s(.5), s(.3125), .25], [0, s(.5), s(.5), s(.5), 0]],
                     [[.5, .25, .75 * s(2), s(.625), .75], [0, s(.5), s(2), s(2), 0]]])
    assert np.allclose(h, hand, atol=1e-14)
    run = lambda tol, eps: admm.admm_run(pre, u_hat, b_hat, rho, 2, tol=tol, eps_abs=eps, check_every=1)
    a = run(0.5, 0.0)
    assert a["converged"].tolist() == [True, False] and a["iters"].tolist() == [2, 2]
    a = run(0.3, 0.0)
    assert a["converged"].tolist() == [False, False]
    # the absolute part: eps_abs sqrt(N + n) = eps sqrt(2); plan b passes at k = 1 iff eps sqrt2 >= rd = sqrt(.5), i.e. eps >= .5
    a = run(1e-9, 0.51)
    assert a["converged"][1] and a["iters"][1] == 1
    a = run(1e-9, 0.49)
    assert not a["converged"][1]


def test_presolve_accepts_exactly_the_plans_with_t_star_zero():
    """Deviation D1 (oracle/admm.py docstring): the box optimum is accepted iff the simplex optimum has t* = 0; the state returned
    is a fixed point of the iteration; its objective is the simplex optimum."""
    w = make_workload(0, n_target=60, n_lowdose=90, n_iso=1)                 # n = 24, small enough for the dense simplex
    bound = w.phi[w.point_class == 0].astype(np.float64).mean(axis=0).max()   # t* = 0 iff beta >= bound (test_trivial_plan_closed_form)
    betas = np.array([0.0, 0.5 * bound, 0.98 * bound, 1.02 * bound, 2.0 * bound])
    weights = np.stack([np.ones(5), np.full(5, 0.5), betas], axis=1)
    pre = admm.precondition(w.phi, w.point_class, w.classes)
    u_hat, b_hat = admm.plan_bounds(pre, w.point_class, w.classes, weights)
    rho = default_rho(betas)
    acc, st = admm.presolve_box_optimum(pre, u_hat, b_hat, rho)
    assert acc.tolist() == [False, False, False, True, True]
    for p in range(5):
        sol = simplex.solve_plan(w.phi, w.point_class, w.classes, weights[p])
        assert (np.max(np.abs(sol["t"])) < 1e-12) == bool(acc[p])
        if acc[p]:
            P0 = lp_model.primal_objective(w.phi, w.point_class, w.classes, weights[p], np.zeros(w.n))
            assert abs(P0 - sol["opt"]) < 1e-12
    one = admm.admm_run(pre, u_hat, b_hat, rho, 1, state0=(st["z1"], st["y1"], st["z2"], st["y2"]))
    for name in ("z1", "y1", "z2", "y2"):
        assert np.allclose(one[name][:, acc], st[name][:, acc], atol=1e-12), name
    # in a tolerance run such plans report 0 iterations and t = 0; the others are untouched by the option
    a = admm.admm_run(pre, u_hat, b_hat, rho, 300, tol=1e-3, presolve=True)
    b = admm.admm_run(pre, u_hat, b_hat, rho, 300, tol=1e-3)
    assert a["iters"][acc].tolist() == [0, 0] and np.all(a["y2"][:, acc] == 0) and a["converged"][acc].all()
    assert np.array_equal(a["iters"][~acc], b["iters"][~acc]) and np.array_equal(a["z1"][:, ~acc], b["z1"][:, ~acc])


def test_hard_class_admm_converges_to_the_constrained_optimum():
    """Hard class (u = infinity, Eq. 15): z1 is clipped below only, and rho R o y2 converges to a t that satisfies the
    hard rows and attains the simplex optimum of the constrained LP (pinned by vertex enumeration in test_oracle_lp.py)."""
    from test_oracle_lp import _three_class_tiny
    w = _three_class_tiny(32, 4, 6, 4, 3)
    pre = admm.precondition(w.phi, w.point_class, w.classes)
    u_hat, b_hat = admm.plan_bounds(pre, w.point_class, w.classes, w.weights)
    assert np.all(np.isinf(u_hat[w.point_class == 2])) and np.all(np.isfinite(u_hat[w.point_class < 2]))
    rho = np.full(w.B, 0.05)
    st = admm.admm_run(pre, u_hat, b_hat, rho, 20000, tol=1e-7, eps_abs=1e-10)
    t, lam = admm.recover(pre, st, rho)
    for p in range(w.B):
        sx = simplex.solve_plan(w.phi, w.point_class, w.classes, w.weights[p])
        soft = lp_model.primal_terms(w.phi, w.point_class, w.classes, w.weights[p], t[p])
        obj = soft[0][:2].sum() + soft[1]
        assert lp_model.hard_violation(w.phi, w.point_class, w.classes, t[p]) < 1e-5
        assert abs(obj - sx["opt"]) / max(abs(sx["opt"]), 0.1) < 1e-3, (p, obj, sx["opt"])


def test_warm_start_from_the_box_optimum():
    """Deviation D3: a plan the presolve rejects narrowly starts from the box state.  The rule selects by the largest ratio
    (A x_box)_j / b_j; the start is consistent (z in the boxes, y >= 0 complementary to them); the iteration reaches the simplex
    optimum as from the zero start, in fewer iterations for the plans next to the presolve threshold."""
    from oracle import simplex
    from workloads import Workload
    w0 = make_workload(0, n_target=200, n_lowdose=400, n_iso=2, grid=3)
    pre = admm.precondition(w0.phi, w0.point_class, w0.classes)
    one = np.array([[1.0, 0.5, 1.0]])
    u1, b1 = admm.plan_bounds(pre, w0.point_class, w0.classes, one, None)
    _, st1 = admm.presolve_box_optimum(pre, u1, b1, np.array([1e-3]))
    beta_star = float(np.max(st1["z2"] / b1))                       # w_BOT below which the box optimum stops being feasible (alpha = 0.5)
    betas = beta_star * np.array([1.2, 0.9, 0.6, 0.3, 0.1])         # ratios 0.83 (accepted), 1.1, 1.7, 3.3, 10
    weights = np.stack([np.ones(5), np.full(5, 0.5), betas], axis=1)
    w = Workload(name="warm", config=0, phi=w0.phi, point_class=w0.point_class, classes=w0.classes, weights=weights, row_mask=None,
                 alpha=np.full(5, 0.5), beta=betas)
    rho = scaled_rho(betas, w0.point_class)
    u_hat, b_hat = admm.plan_bounds(pre, w.point_class, w.classes, weights, None)
    acc, ps = admm.presolve_box_optimum(pre, u_hat, b_hat, rho)
    warm, z2, y2 = admm.warm_start_plans(acc, ps, b_hat, 2.5)
    assert acc.tolist() == [True, False, False, False, False] and warm.tolist() == [False, True, True, False, False]
    assert np.all(z2 <= b_hat + 1e-15) and np.all(y2 >= 0) and np.all((y2 == 0) | (z2 == b_hat))       # complementary
    cold = admm.solve_workload(w, rho, 20000, tol=1e-5, pre=pre, presolve=True)
    hot = admm.solve_workload(w, rho, 20000, tol=1e-5, pre=pre, presolve=True, warm_start_ratio=2.5)
    assert cold["converged"].all() and hot["converged"].all()
    for p in range(5):
        opt = simplex.solve_plan(w.phi, w.point_class, w.classes, weights[p])["opt"]
        assert abs(hot["obj"][p] - opt) / max(abs(opt), 0.1) < 1e-3 and abs(cold["obj"][p] - opt) / max(abs(opt), 0.1) < 1e-3
    assert np.array_equal(hot["iters"][~warm], cold["iters"][~warm])             # untouched plans: identical runs
    # (what the option buys depends on the case: nothing here; at config 3, full size, the plans next to the presolve threshold
    # need 1160 iterations instead of 2810 -- measured on the GPU, tests/test_gpu_parity.py and bench.py)

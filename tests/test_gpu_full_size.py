"""Full-size parity: BASELINE.json configs 2, 3 and 4 in the launch configuration bench.py times, against the fp64 oracle.

The oracle cannot iterate all plans of these sizes in test time (config 3: 7.6e12 fp64 flops per iteration), and plans are
independent columns: the CUDA path runs the WHOLE batch (81 / 441 plans), the oracle a seeded subset of them (8 of
the 81, 16 of the 441: always the beta = 0 plans of the subset, a plan with t* = 0, the grid corners, the centre and mid-grid plans),
and those are compared element by element
after K = 50 iterations (north_star: 1e-4 fp32 path, 1e-2 reduced storage; metric = DESIGN.md reading R17).  The oracle's
preconditioning (S = A^ A^^T + I in fp64, 4e13 - 9e13 flops, a minute or two on the host cores) is formed once per matrix and shared
by the tests of this module, and the oracle's objective P(t) -- one fp64 pass over Phi per plan -- is evaluated for three of the
subset's plans.  Converged objectives are certified by the weak-duality bracket: P(t) >= OPT >= Dual(x) for any t >= 0 and any
dual-feasible x, both evaluated by the oracle's fp64 LP model from the CUDA path's (t, D o z1).

The whole module is sized to run in about ten minutes on the GPU box (its host cores do the oracle's work; the driver allows
`pytest -m gpu` 1200 s in all)."""
import numpy as np
import pytest

from conftest import have_cuda
from parity_util import block2_errors, stacked_errors, t_errors

pytestmark = [pytest.mark.gpu, pytest.mark.skipif(not have_cuda(), reason="needs a CUDA device")]

TOL_FP32 = 1e-4
TOL_REDUCED = 1e-2
# DESIGN.md reading R20: the degenerate plan (alpha, beta) = (0, 0) has OPT = 0 and z -> 0; its block-2 dual (hence t) is the
# difference of two long products that cancel to ~1e-4 of their size, and NO fp32-accumulating implementation holds 1e-4 there
# (tests/test_gpu_parity.py::test_fixed_k_parity_config1_full_size measures a plain numpy-sgemm restatement of the oracle at
# 1.6e-3 on that plan, the tensor path at 5e-4).  Its bar on y is that measured fp32 floor; every other plan is held to
# north_star's tolerance.
DEGENERATE_BAR = 2e-3
OBJ_PLANS = 3              # the oracle's objective is evaluated for this many of the 16 plans (first, middle, last)
_P_ORACLE = {}


@pytest.fixture(scope="module")
def b():
    from paper_2509_08602_b200 import binding
    return binding


SUBSET = {2: 8, 3: 16, 4: 8}      # plans the oracle iterates per configuration (its dgemms are compute-bound: cost ~ columns)


def _subset(w, count):
    """`count` >= 8 plans: the four grid corners, beta = 0 and beta = 1 (t* = 0) at mid alpha, the grid centre, plan 1 (the smallest
    w_BOT > 0 at alpha = 0), and seeded mid-grid plans."""
    g = int(round(np.sqrt(w.B)))
    fixed = [0, g - 1, (g // 2) * g, (g // 2) * g + g - 1, (g - 1) * g, g * g - 1, (g // 2) * g + g // 2, 1]
    rng = np.random.default_rng(16)
    rest = [int(p) for p in rng.permutation(w.B) if p not in fixed][: count - len(fixed)]
    return np.array(sorted(fixed + rest))


def _oracle_iterates(pre, cases, K=50):
    """K iterations of the oracle for the plan subsets of several plan sets that share one Phi, as ONE run (a column is a
    plan): cases = {configuration: workload}.  Returns {configuration: dict(z1, y1, z2, y2, t, plans, rho)}."""
    from oracle import admm
    from workloads import scaled_rho
    u_cols, b_cols, rho_cols, spans, c0 = [], [], [], {}, 0
    for key, w in cases.items():
        plans = _subset(w, SUBSET[key])
        rho = scaled_rho(w.beta, w.point_class)
        ws = w.subset(plans)
        u_hat, b_hat = admm.plan_bounds(pre, ws.point_class, ws.classes, ws.weights, ws.mask_bool())
        u_cols.append(u_hat); b_cols.append(b_hat); rho_cols.append(rho[plans])
        spans[key] = (c0, plans, rho); c0 += len(plans)
    rho_all = np.concatenate(rho_cols)
    st = admm.admm_run(pre, np.concatenate(u_cols, axis=1), np.concatenate(b_cols, axis=1), rho_all, K)
    t_all, _ = admm.recover(pre, st, rho_all)
    out = {}
    for key, (c0, plans, rho) in spans.items():
        sl = slice(c0, c0 + len(plans))
        out[key] = dict(z1=st["z1"][:, sl], y1=st["y1"][:, sl], z2=st["z2"][:, sl], y2=st["y2"][:, sl], t=t_all[sl], plans=plans, rho=rho)
    return out


def _compare(b, h, w, out, ref, tol):
    from oracle import lp_model
    plans = ref["plans"]
    states = [b.admm_get_state(h, int(p)) for p in plans]
    ez, ey = stacked_errors(states, ref)
    ez2, ey2 = block2_errors(states, ref)
    et = t_errors(out["t"][plans], ref["t"])
    deg = (w.alpha[plans] == 0) & (w.beta[plans] == 0)
    worst = dict(z=ez.max(), y=ey[~deg].max(), z2=ez2.max(), y2=ey2[~deg].max(), t=et[~deg].max(),
                 y_degenerate=ey[deg].max(initial=0.0), t_degenerate=et[deg].max(initial=0.0))
    print("full-size parity", w.name, {k: f"{v:.2e}" for k, v in worst.items()})
    assert ez.max() < tol and ey[~deg].max() < tol, worst
    assert ey[deg].max(initial=0.0) < max(tol, DEGENERATE_BAR), worst
    masks = w.mask_bool()
    for j in np.linspace(0, len(plans) - 1, OBJ_PLANS).astype(int):
        p = int(plans[j])
        if (w.name, p) not in _P_ORACLE:         # the storage variants of one configuration share the oracle's P(t)
            _P_ORACLE[(w.name, p)] = lp_model.primal_objective(w.phi, w.point_class, w.classes, w.weights[p], ref["t"][j], masks[p])
        P = _P_ORACLE[(w.name, p)]
        assert abs(out["obj"][p] - P) / max(abs(P), 0.1) < tol, (p, out["obj"][p], P)
    return ez2, ey2, et, deg


@pytest.fixture(scope="module")
def case23():
    """configs 2 and 3 share one Phi (450000 x 9600, 17.3 GB): generated once, preconditioned once by the oracle, and both
    plan subsets (8 + 16 columns) iterated in one oracle run."""
    from oracle import admm
    from workloads import make_workload, with_plans_of
    import time
    t0 = time.time()
    w3 = make_workload(3)
    w2 = with_plans_of(w3, 2)
    t1 = time.time()
    pre = admm.precondition(w3.phi, w3.point_class, w3.classes)
    t2 = time.time()
    refs = _oracle_iterates(pre, {2: w2, 3: w3})
    print(f"configs 2/3: generation {t1 - t0:.0f} s, oracle preconditioning {t2 - t1:.0f} s, 50 oracle iterations of 24 columns {time.time() - t2:.0f} s")
    return w2, w3, pre, refs


def test_config2_full_size(b, case23):
    """config 2 (B = 81, one pass of 96 columns, per-plan row masks): the two contractions on sampled outputs the fp64 definition
    gives one by one, then the K = 50 iterates of 8 plans against the oracle."""
    import torch
    w2, _, pre, refs = case23
    ref = refs[2]
    rng = np.random.default_rng(11)
    h = b.admm_setup(torch.from_numpy(w2.phi), w2.point_class, w2.classes)
    for which in (0, 1):
        K = w2.N if which == 0 else w2.n
        rows = w2.n if which == 0 else w2.N
        small = rng.standard_normal((24, K)).astype(np.float32)
        got = b.admm_contract_probe(h, which, small)
        idx = np.unique(np.concatenate([rng.integers(0, rows, 48), [0, rows - 1, rows - 2]]))
        sub = (w2.phi[:, idx] if which == 0 else w2.phi[idx, :].T).astype(np.float64)          # [K, samples]
        exact = small.astype(np.float64) @ sub
        scale = np.abs(small.astype(np.float64)) @ sub
        assert np.max(np.abs(got[:, idx] - exact) / scale) < 1e-6, which
    rho = ref["rho"]
    mask = torch.from_numpy(w2.row_mask.view(np.int32)).cuda()
    out = b.admm_solve_batch(h, w2.weights, rho, mask, fixed_iters=50)
    ez2, ey2, et, deg = _compare(b, h, w2, out, ref, TOL_FP32)
    # block 2 alone (reading R20): 1e-4 except where the plan's block-2 dual is a cancellation remainder
    assert np.median(et) < TOL_FP32 and np.median(ey2) < TOL_FP32
    # plan p of the batch == the same plan run alone (bit-exact): the batch is 81 independent columns (:96)
    p = 40
    st_batch = b.admm_get_state(h, p)
    one = w2.subset([p])
    o1 = b.admm_solve_batch(h, one.weights, rho[[p]], one.row_mask, fixed_iters=50)
    for a, c in zip(st_batch, b.admm_get_state(h, 0)):
        assert np.array_equal(a, c)
    assert np.array_equal(o1["t"][0], out["t"][p])
    h.close()


def test_config3_full_size(b, case23):
    """config 3 (B = 441: five passes of <= 96 plans on the fp32 path, row masks): K = 50 iterates of 16 plans against the oracle;
    then a short tolerance-mode run in which plans freeze at different checks and are compacted across the passes: a frozen plan
    must equal the same plan run alone for its iteration count (bit-exact)."""
    import torch
    _, w3, pre, refs = case23
    ref = refs[3]
    rho = ref["rho"]
    h = b.admm_setup(torch.from_numpy(w3.phi), w3.point_class, w3.classes, presolve=False)
    mask = torch.from_numpy(w3.row_mask.view(np.int32)).cuda()
    out = b.admm_solve_batch(h, w3.weights, rho, mask, fixed_iters=50)
    _compare(b, h, w3, out, ref, TOL_FP32)
    cap = 40
    for tol in (0.5, 0.2, 0.08, 0.03):          # loose enough that plans pass at different checks within 40 iterations
        out = b.admm_solve_batch(h, w3.weights, rho, mask, tol=tol, max_iter=cap)
        iters = out["iters"].copy()
        if len(set(iters.tolist())) >= 3 and iters.max() == cap:
            break
    assert len(set(iters.tolist())) >= 3 and iters.min() < cap, np.unique(iters)   # plans really stopped at different checks
    frozen_early = int(np.argmin(iters)); ran_to_cap = int(np.argmax(iters))
    states = {p: b.admm_get_state(h, p) for p in (frozen_early, ran_to_cap)}
    for p, st in states.items():
        one = w3.subset([p])
        o1 = b.admm_solve_batch(h, one.weights, rho[[p]], one.row_mask, fixed_iters=int(iters[p]))
        for a, c in zip(st, b.admm_get_state(h, 0)):
            assert np.array_equal(a, c), p
        assert np.array_equal(o1["t"][0], out["t"][p])
    h.close()


def test_config3_converged_objectives_certified(b, case23):
    """Converged objectives on config 3 (the dense simplex cannot hold a 9600 x 459600 tableau): tolerance 1e-4, then the
    weak-duality bracket from the CUDA path's own (t, D o z1), evaluated by the oracle's fp64 LP model:
    (P(t) - Dual(x)) / max(|P|, 0.1) <= 1e-3 certifies |P - OPT| to north_star's 1e-3.  Plans: beta = 0.05 (iterates to
    convergence) at alpha = 0, 0.5, 1 and beta = 0.5 (settled by the presolve, deviation D1) at alpha = 0.5."""
    import torch
    from oracle import lp_model
    _, w3, pre, _ = case23
    g = 21
    plans = np.array([0 * g + 1, 10 * g + 1, 10 * g + 10, 20 * g + 1])
    w = w3.subset(plans)
    h = b.admm_setup(torch.from_numpy(w3.phi), w3.point_class, w3.classes)
    out = b.admm_solve_batch(h, w.weights, None, w.row_mask, tol=1e-4, max_iter=3000)
    masks = w.mask_bool()
    assert np.all(out["iters"] < 3000), out["iters"]
    assert np.array_equal(out["iters"] == 0, w.beta == 0.5)
    for i in range(w.B):
        z1 = b.admm_get_state(h, i)[0].astype(np.float64)
        P = lp_model.primal_objective(w.phi, w.point_class, w.classes, w.weights[i], out["t"][i].astype(np.float64), masks[i])
        lo = lp_model.dual_bound(w.phi, w.point_class, w.classes, w.weights[i], z1 * pre.D, masks[i])
        assert abs(out["obj"][i] - P) / max(abs(P), 0.1) < 1e-5                 # the CUDA path's own objective evaluation
        assert lo <= P + 1e-9 and (P - lo) / max(abs(P), 0.1) < 1e-3, (i, P, lo)
    h.close()


def test_config4_storage_variants(b):
    """config 4 (n = 12000 time variables, B = 441 plans, every dense storage mode of BASELINE.json) against the oracle on the
    ORIGINAL Phi: K = 50 iterates of 8 plans, 1e-4 for fp32 storage (3xTF32), 1e-2 for tf32-consumed and bf16 storage
    (north_star).  B = 441 runs the reduced-storage modes through the wide (97..256 plans per pass) kernel.  The ROW count is a
    quarter of the configuration's (50000 target + 100000 low-dose points, same geometry recipe and seeds): the oracle's share of the
    full 600000 x 12000 case -- S = A^ A^^T + I is 1.7e14 fp64 flops, an iteration reads the 58 GB fp64 A^ twice -- takes longer on
    the host cores than the whole GPU suite may (measured: 700 s); every kernel, tile shape, pass structure and storage mode is
    the full configuration's, only the loop over row tiles is shorter.  The full row count is covered by
    test_config4_full_size_sampled_outputs."""
    import time
    import torch
    from oracle import admm
    from workloads import make_workload
    t0 = time.time()
    w4 = make_workload(4, n_target=50000, n_lowdose=100000)
    t1 = time.time()
    pre = admm.precondition(w4.phi, w4.point_class, w4.classes)
    t2 = time.time()
    ref = _oracle_iterates(pre, {4: w4})[4]
    print(f"config 4 (150000 rows): generation {t1 - t0:.0f} s, oracle preconditioning {t2 - t1:.0f} s, 50 oracle iterations {time.time() - t2:.0f} s")
    del pre
    mask = torch.from_numpy(w4.row_mask.view(np.int32)).cuda()
    phi = torch.from_numpy(w4.phi)
    for storage, tol in ((b.ADMM_STORAGE_FP32_3XTF32, TOL_FP32), (b.ADMM_STORAGE_FP32_TF32, TOL_REDUCED), (b.ADMM_STORAGE_BF16, TOL_REDUCED)):
        h = b.admm_setup(phi, w4.point_class, w4.classes, storage=storage)
        out = b.admm_solve_batch(h, w4.weights, ref["rho"], mask, fixed_iters=50)
        ez2, ey2, et, deg = _compare(b, h, w4, out, ref, tol)
        # block 2 alone: most plans sit well inside the bar; the degenerate one is reported by _compare's printout
        assert np.median(et) < tol and np.median(ey2) < tol
        h.close()


def test_config4_full_size_sampled_outputs(b):
    """config 4 at its full size (600000 x 12000, 28.8 GB, B = 441) in the launch configuration of the bench: what the fp64
    definition gives one by one -- sampled outputs of both contractions (fp32 storage: against Phi; bf16 storage: against the
    bf16-rounded Phi the kernels consume, with bf16 hi/lo plan operands) -- and a property that holds at any size: a plan of the
    441-plan batch equals the same plan run alone, bit for bit (the batch is 441 independent columns)."""
    import torch
    from workloads import make_workload, scaled_rho
    w4 = make_workload(4)
    rho = scaled_rho(w4.beta, w4.point_class)
    rng = np.random.default_rng(12)
    phi = torch.from_numpy(w4.phi)
    mask = torch.from_numpy(w4.row_mask.view(np.int32)).cuda()
    for storage, bar in ((b.ADMM_STORAGE_FP32_3XTF32, 1e-6), (b.ADMM_STORAGE_BF16, 2e-5)):
        h = b.admm_setup(phi, w4.point_class, w4.classes, storage=storage)
        for which in (0, 1):
            K = w4.N if which == 0 else w4.n
            rows = w4.n if which == 0 else w4.N
            small = rng.standard_normal((24, K)).astype(np.float32)
            got = b.admm_contract_probe(h, which, small)
            idx = np.unique(np.concatenate([rng.integers(0, rows, 32), [0, rows - 1, rows - 2]]))
            sub = (w4.phi[:, idx] if which == 0 else w4.phi[idx, :].T)                               # [K, samples] fp32
            if storage == b.ADMM_STORAGE_BF16:
                sub = torch.from_numpy(np.ascontiguousarray(sub)).to(torch.bfloat16).to(torch.float32).numpy()   # RNE, as at setup
            sub = sub.astype(np.float64)
            exact = small.astype(np.float64) @ sub
            scale = np.abs(small.astype(np.float64)) @ sub
            assert np.max(np.abs(got[:, idx] - exact) / scale) < bar, (storage, which)
        K = 10
        out = b.admm_solve_batch(h, w4.weights, rho, mask, fixed_iters=K)
        p = 222
        st_batch = b.admm_get_state(h, p)
        one = w4.subset([p])
        o1 = b.admm_solve_batch(h, one.weights, rho[[p]], one.row_mask, fixed_iters=K)
        if storage == b.ADMM_STORAGE_FP32_3XTF32:            # one kernel serves 1 and 96 plans of a pass: bit-exact
            for a, c in zip(st_batch, b.admm_get_state(h, 0)):
                assert np.array_equal(a, c)
            assert np.array_equal(o1["t"][0], out["t"][p])
        else:                                                # 441 plans run the wide kernel, one plan the staged one (another
            for a, c in zip(st_batch, b.admm_get_state(h, 0)):   # accumulation order): inside the bf16-storage budget (measured 2e-3)
                assert np.linalg.norm(a.astype(np.float64) - c) <= TOL_REDUCED * max(np.linalg.norm(c), 1e-30)
        h.close()

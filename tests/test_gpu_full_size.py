"""Full-size parity: BASELINE.json configs 2, 3 and 4 in the launch configuration bench.py times, against the fp64 oracle.

The oracle cannot iterate all plans of these sizes in test time (config 3: 7.6e12 fp64 flops per iteration), and plans are
independent columns: the CUDA path runs the WHOLE batch (81 / 441 plans), the oracle a seeded subset of 16 of them
(always a beta = 0 plan, a plan with t* = 0, the grid corners and mid-grid plans), and those 16 are compared element by element
after K = 50 iterations (north_star: 1e-4 fp32 path, 1e-2 reduced storage; metric = DESIGN.md reading R17).  The oracle's
preconditioning (S = A^ A^^T + I in fp64, 4e13 - 9e13 flops, a few minutes on the host cores) is formed once per matrix and shared
by the tests of this module.  Converged objectives are certified by the weak-duality bracket: P(t) >= OPT >= Dual(x)
for any t >= 0 and any dual-feasible x, both evaluated by the oracle's fp64 LP model from the CUDA path's (t, D o z1)."""
import numpy as np
import pytest

from conftest import have_cuda
from parity_util import block2_errors, stacked_errors, t_errors

pytestmark = [pytest.mark.gpu, pytest.mark.skipif(not have_cuda(), reason="needs a CUDA device")]

TOL_FP32 = 1e-4
TOL_REDUCED = 1e-2


@pytest.fixture(scope="module")
def b():
    from paper_2509_08602_b200 import binding
    return binding


def _subset16(w):
    """16 plans: the four grid corners, beta = 0 and beta = 1 (t* = 0) at mid alpha, and seeded mid-grid plans."""
    g = int(round(np.sqrt(w.B)))
    fixed = [0, g - 1, (g // 2) * g, (g // 2) * g + g - 1, (g - 1) * g, g * g - 1, (g // 2) * g + g // 2, 1]
    rng = np.random.default_rng(16)
    rest = [int(p) for p in rng.permutation(w.B) if p not in fixed][: 16 - len(fixed)]
    return np.array(sorted(fixed + rest))


def _compare(b, h, w, out, ref, plans, tol):
    states = [b.admm_get_state(h, int(p)) for p in plans]
    ez, ey = stacked_errors(states, ref)
    ez2, ey2 = block2_errors(states, ref)
    et = t_errors(out["t"][plans], ref["t"])
    eobj = np.abs(out["obj"][plans] - ref["obj"]) / np.maximum(np.abs(ref["obj"]), 0.1)
    worst = dict(z=ez.max(), y=ey.max(), z2=ez2.max(), y2=ey2.max(), t=et.max(), obj=eobj.max())
    print("full-size parity", w.name, {k: f"{v:.2e}" for k, v in worst.items()})
    assert ez.max() < tol and ey.max() < tol, worst
    assert eobj.max() < tol, worst
    return ez2, ey2, et


@pytest.fixture(scope="module")
def case23():
    """configs 2 and 3 share one Phi (450000 x 9600, 17.3 GB): generated once, preconditioned once by the oracle."""
    from oracle import admm
    from workloads import make_workload, with_plans_of
    w3 = make_workload(3)
    w2 = with_plans_of(w3, 2)
    pre = admm.precondition(w3.phi, w3.point_class, w3.classes)
    return w2, w3, pre


def _oracle_subset(w, plans, rho, pre, K=50):
    from oracle import admm
    return admm.solve_workload(w.subset(plans), rho[plans], K, pre=pre)


def test_config2_full_size(b, case23):
    """config 2 (B = 81, one pass of 96 columns, per-plan row masks): the two contractions on sampled outputs the fp64 definition
    gives one by one, then the K = 50 iterates of 16 plans against the oracle."""
    import torch
    from workloads import scaled_rho
    w2, _, pre = case23
    rng = np.random.default_rng(11)
    h = b.admm_setup(torch.from_numpy(w2.phi), w2.point_class, w2.classes)
    for which in (0, 1):
        K = w2.N if which == 0 else w2.n
        rows = w2.n if which == 0 else w2.N
        small = rng.standard_normal((24, K)).astype(np.float32)
        got = b.admm_contract_probe(h, which, small)
        idx = np.unique(np.concatenate([rng.integers(0, rows, 200), [0, rows - 1, rows - 2]]))
        sub = (w2.phi[:, idx] if which == 0 else w2.phi[idx, :].T).astype(np.float64)          # [K, samples]
        exact = small.astype(np.float64) @ sub
        scale = np.abs(small.astype(np.float64)) @ sub
        assert np.max(np.abs(got[:, idx] - exact) / scale) < 1e-6, which
    rho = scaled_rho(w2.beta, w2.point_class)
    plans = _subset16(w2)
    ref = _oracle_subset(w2, plans, rho, pre)
    mask = torch.from_numpy(w2.row_mask.view(np.int32)).cuda()
    out = b.admm_solve_batch(h, w2.weights, rho, mask, fixed_iters=50)
    ez2, ey2, et = _compare(b, h, w2, out, ref, plans, TOL_FP32)
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
    from workloads import scaled_rho
    _, w3, pre = case23
    rho = scaled_rho(w3.beta, w3.point_class)
    plans = _subset16(w3)
    ref = _oracle_subset(w3, plans, rho, pre)
    h = b.admm_setup(torch.from_numpy(w3.phi), w3.point_class, w3.classes, presolve=False)
    mask = torch.from_numpy(w3.row_mask.view(np.int32)).cuda()
    out = b.admm_solve_batch(h, w3.weights, rho, mask, fixed_iters=50)
    _compare(b, h, w3, out, ref, plans, TOL_FP32)
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
    convergence) and beta = 0.5 (settled by the presolve, deviation D1) at alpha = 0, 0.5, 1."""
    import torch
    from oracle import lp_model
    _, w3, pre = case23
    g = 21
    plans = np.array([ia * g + ib for ia in (0, 10, 20) for ib in (1, 10)])
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


def test_config4_full_size_storage_variants(b):
    """config 4 (600000 x 12000, B = 441) in each dense storage mode of BASELINE.json: K = 50 iterates of 16 plans against the
    oracle on the ORIGINAL Phi -- 1e-4 for fp32 storage (3xTF32), 1e-2 for tf32-consumed and bf16 storage (north_star).  B = 441 runs
    the reduced-storage modes through the wide (97..256 plans per pass) kernel."""
    import torch
    from oracle import admm
    from workloads import make_workload, scaled_rho
    w4 = make_workload(4)
    pre = admm.precondition(w4.phi, w4.point_class, w4.classes)
    rho = scaled_rho(w4.beta, w4.point_class)
    plans = _subset16(w4)
    ref = admm.solve_workload(w4.subset(plans), rho[plans], 50, pre=pre)
    del pre
    mask = torch.from_numpy(w4.row_mask.view(np.int32)).cuda()
    phi = torch.from_numpy(w4.phi)
    for storage, tol in ((b.ADMM_STORAGE_FP32_3XTF32, TOL_FP32), (b.ADMM_STORAGE_FP32_TF32, TOL_REDUCED), (b.ADMM_STORAGE_BF16, TOL_REDUCED)):
        h = b.admm_setup(phi, w4.point_class, w4.classes, storage=storage)
        out = b.admm_solve_batch(h, w4.weights, rho, mask, fixed_iters=50)
        ez2, ey2, et = _compare(b, h, w4, out, ref, plans, tol)
        # block 2 alone: most plans sit well inside the bar; the degenerate ones (beta = 0: t is a cancellation remainder, reading
        # R20) are reported by _compare's printout
        assert np.median(et) < tol and np.median(ey2) < tol
        h.close()

"""Two-pass optimisation (PAPER.md II.C, :108-114, :144) through the C ABI against oracle/two_pass.py: the dose calculation
between the passes, the per-plan second-pass low-dose volumes, and the whole two-pass driver."""
import numpy as np
import pytest

from conftest import have_cuda

pytestmark = [pytest.mark.gpu, pytest.mark.skipif(not have_cuda(), reason="needs a CUDA device")]


@pytest.fixture(scope="module")
def b():
    from paper_2509_08602_b200 import binding
    return binding


@pytest.fixture(scope="module")
def case():
    from workloads import make_candidates, make_workload
    w = make_workload(1, n_target=1500, n_lowdose=3000, n_iso=6, grid=5)          # N = 4500, n = 144, B = 25
    pts, phic = make_candidates(w, 5000 + 13)                                      # ragged: 5013 candidates
    return w, phic


def _round_bf16(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).to(torch.bfloat16).to(torch.float32).numpy()


def test_dose_matches_the_definition(b, case):
    """admm_dose: dose[p][i] = Phi_i . t_p (:167, :286) element by element, on a dose-only handle and on a full one, for one pass
    of plans and for several (B = 130 > 96), host and device buffers, fp32 and bf16 storage."""
    import torch
    w, phic = case
    rng = np.random.default_rng(5)
    for B in (7, 130):
        t = np.abs(rng.standard_normal((B, w.n))).astype(np.float32) * 0.02
        exact = t.astype(np.float64) @ phic.astype(np.float64).T
        scale = np.abs(t.astype(np.float64)) @ np.abs(phic.astype(np.float64)).T + 1e-30
        h = b.admm_setup(phic, np.zeros(phic.shape[0], np.uint8), w.classes[:1], dose_only=True)
        got = b.admm_dose(h, t)
        assert got.shape == (B, phic.shape[0]) and np.max(np.abs(got - exact) / scale) < 1e-6
        out_dev = torch.empty((B, phic.shape[0]), dtype=torch.float32, device="cuda")
        b.admm_dose(h, torch.from_numpy(t).cuda(), out=out_dev)
        assert np.array_equal(out_dev.cpu().numpy(), got)
        with pytest.raises(b.AdmmError) as e:                                     # a dose-only handle has no S: it cannot solve
            b.admm_solve_batch(h, np.ones((B, 2)), None, fixed_iters=1)
        assert e.value.status == b.ADMM_ESTATE
        h.close()
    # the SIMT cross-check path serves the same call
    t = np.abs(rng.standard_normal((5, w.n))).astype(np.float32) * 0.02
    h = b.admm_setup(phic, np.zeros(phic.shape[0], np.uint8), w.classes[:1], dose_only=True, kernel_path=b.ADMM_PATH_SIMT)
    got = b.admm_dose(h, t)
    h.close()
    ex = t.astype(np.float64) @ phic.astype(np.float64).T
    assert np.max(np.abs(got - ex) / (np.abs(t.astype(np.float64)) @ np.abs(phic.astype(np.float64)).T + 1e-30)) < 2e-6
    # bf16 storage: against the rounded matrix the kernels consume, bf16 hi/lo time vectors (2^-17)
    t = np.abs(rng.standard_normal((9, w.n))).astype(np.float32) * 0.02
    Pr = _round_bf16(phic).astype(np.float64)
    h = b.admm_setup(phic, np.zeros(phic.shape[0], np.uint8), w.classes[:1], dose_only=True, storage=b.ADMM_STORAGE_BF16)
    got = b.admm_dose(h, t)
    h.close()
    assert np.max(np.abs(got - t.astype(np.float64) @ Pr.T) / (np.abs(t.astype(np.float64)) @ Pr.T + 1e-30)) < 2e-5
    # a full handle serves the dose of its own points too (the dose after a solve, :286)
    h = b.admm_setup(w.phi, w.point_class, w.classes)
    out = b.admm_solve_batch(h, w.weights, None, tol=1e-3, max_iter=200)
    dose = b.admm_dose(h, out["t"])
    h.close()
    ex = out["t"].astype(np.float64) @ w.phi.astype(np.float64).T
    assert np.max(np.abs(dose - ex)) < 1e-5 * max(1.0, np.abs(ex).max())


def test_lowdose_volumes_match_the_oracle(b, case):
    """admm_lowdose_volumes against oracle.two_pass.lowdose_volumes on the same first-pass t: the same bit for every candidate
    whose dose is not within rounding of a threshold, the union = OR of the plans."""
    from oracle import two_pass as o2
    w, phic = case
    rng = np.random.default_rng(6)
    t = np.abs(rng.standard_normal((w.B, w.n))).astype(np.float32) * 0.03
    t[3] = 0.0                                                                     # a plan with t = 0 (presolved): empty volume
    d_ld, delta = 0.5, 0.2
    ref, dose64 = o2.lowdose_volumes(phic, t, d_ld, delta)
    h = b.admm_setup(phic, np.zeros(phic.shape[0], np.uint8), w.classes[:1], dose_only=True)
    bits, anyb, dose = b.admm_lowdose_volumes(h, t, d_ld, d_ld + delta, want_dose=True)
    h.close()
    got = np.unpackbits(bits.view(np.uint8), axis=1, bitorder="little")[:, :phic.shape[0]].astype(bool)
    union = np.unpackbits(anyb.view(np.uint8), bitorder="little")[:phic.shape[0]].astype(bool)
    assert np.max(np.abs(dose - dose64)) < 2e-6 * max(1.0, np.abs(dose64).max())
    near = (np.abs(dose64 - d_ld) < 1e-5) | (np.abs(dose64 - (d_ld + delta)) < 1e-5)
    assert ref.sum() > 1000 and not got[3].any()
    assert np.array_equal(got[~near], ref[~near]) and near.mean() < 1e-3
    assert np.array_equal(union, got.any(axis=0))
    # and the bits are exactly the fp32 range test of the dose the call returned
    assert np.array_equal(got, (dose >= np.float32(d_ld)) & (dose < np.float32(d_ld + delta)))


def test_two_pass_driver_against_the_oracle(b, case):
    """The whole procedure: pass 1, volumes, union sampling, pass 2 with per-plan masks.  The two sides converge pass 1 to a
    tolerance, so their volumes may differ on a few candidates at the range boundaries; what is compared exactly is the second
    pass itself: the oracle solves the SECOND-PASS PROBLEM THE CUDA PATH BUILT (its selection, its volumes) and the converged
    objectives must agree to 1e-3 (north_star); the volumes of the two independent runs must agree on > 99 % of the candidates."""
    from oracle import lp_model, two_pass as o2
    from paper_2509_08602_b200 import two_pass as g2
    from workloads import pick_from_union, scaled_rho
    w, phic = case
    nt = int((w.point_class == 0).sum())
    pick = lambda u, c: pick_from_union(u, c, 21)
    kw = dict(d_ld=0.5, delta=0.25, n_lowdose_2=1500, pick=pick, tol=1e-4, max_iter=2000)
    rho = scaled_rho(w.beta, w.point_class)
    res = g2.two_pass(w.phi[:nt], w.phi[nt:], phic, w.classes, w.weights, rho=rho, **kw)
    ref = o2.two_pass(w.phi[:nt], w.phi[nt:], phic, w.classes, w.weights, rho_rule=scaled_rho, **kw)
    assert res["in_volume"].shape == ref["in_volume"].shape and ref["in_volume"].sum() > 500
    assert np.mean(res["in_volume"] == ref["in_volume"]) > 0.99
    assert len(set(res["selected"].tolist()) & set(ref["selected"].tolist())) > 0.9 * ref["selected"].size
    # the second pass of the CUDA path's own problem, solved by the oracle
    phi2, pc2, masks2 = o2.second_pass_problem(w.phi[:nt], phic, res["in_volume"], res["selected"])
    assert np.array_equal(np.unpackbits(res["row_mask2"].view(np.uint8), axis=1, bitorder="little")[:, :phi2.shape[0]].astype(bool), masks2)
    p2 = o2._solve(phi2, pc2, w.classes, np.asarray(w.weights, dtype=np.float64), scaled_rho, masks2, 1e-4, 2000)
    both = p2["converged"] & (res["pass2"]["iters"] < 2000)
    assert both.sum() >= 12
    for p in np.nonzero(both)[0]:
        P_ref = lp_model.primal_objective(phi2, pc2, w.classes, w.weights[p], p2["t"][p], masks2[p])
        assert abs(res["pass2"]["obj"][p] - P_ref) / max(abs(P_ref), 0.1) < 1e-3, (p, res["pass2"]["obj"][p], P_ref)


def test_two_pass_with_algorithm1_sampling(b, case):
    """sampling = "algorithm1" (:116-136): from the CUDA path's volumes the oracle's line-by-line Algorithm 1 must produce the same
    point set P and the same per-plan sets p_j (index work: bit-exact), every plan with a non-empty volume gets ~n_lowdose_2 points
    of its own, and the second pass on that problem reaches the oracle's objectives."""
    from oracle import lp_model, two_pass as o2
    from paper_2509_08602_b200 import two_pass as g2
    from workloads import scaled_rho, uniform01
    w, phic = case
    nt = int((w.point_class == 0).sum())
    plans = np.array([1, 2, 6, 7, 11, 12, 16, 17, 21, 22, 3])                       # w_BOT = 0.25, 0.5 at every alpha, and one t* = 0 plan
    ws = w.subset(plans)
    rho = scaled_rho(ws.beta, w.point_class)
    res = g2.two_pass(w.phi[:nt], w.phi[nt:], phic, w.classes, ws.weights, rho=rho, d_ld=0.5, delta=0.25, n_lowdose_2=300, pick=None,
                      tol=1e-4, max_iter=2000, sampling="algorithm1", uniform01=uniform01, seed=5)
    P, p, order = o2.overlapping_sampling(res["in_volume"], [300] * ws.B, seed=5, uniform01=uniform01)
    assert res["selected"].tolist() == P
    phi2, pc2, masks2 = o2.second_pass_problem_alg1(w.phi[:nt], phic, P, p)
    got_masks = np.unpackbits(res["row_mask2"].view(np.uint8), axis=1, bitorder="little")[:, :phi2.shape[0]].astype(bool)
    assert np.array_equal(got_masks, masks2)
    own = masks2[:, nt:].sum(axis=1)
    vol = res["in_volume"].sum(axis=1)
    assert np.all(own[vol >= 300] > 240) and np.all(own[vol >= 300] < 360) and np.all(own[vol == 0] == 0)
    assert len(P) < own.sum()                                                        # points are shared between plans
    p2 = o2._solve(phi2, pc2, w.classes, np.asarray(ws.weights, dtype=np.float64), scaled_rho, masks2, 1e-4, 2000)
    both = p2["converged"] & (res["pass2"]["iters"] < 2000)
    assert both.sum() >= 6
    for q in np.nonzero(both)[0]:
        P_ref = lp_model.primal_objective(phi2, pc2, w.classes, ws.weights[q], p2["t"][q], masks2[q])
        assert abs(res["pass2"]["obj"][q] - P_ref) / max(abs(P_ref), 0.1) < 1e-3, (q, res["pass2"]["obj"][q], P_ref)


def test_dose_argument_handling(b, case):
    """Strided t (ld_t > n), a single plan, and the documented argument errors."""
    import torch
    w, phic = case
    h = b.admm_setup(phic, np.zeros(phic.shape[0], np.uint8), w.classes[:1], dose_only=True)
    big = torch.zeros((3, w.n + 40), dtype=torch.float32)
    big[:, :w.n] = torch.rand((3, w.n)) * 0.02
    big[:, w.n:] = 7.0                                                             # must not be read
    view = big[:, :w.n]                                                            # stride(0) = n + 40
    got = b.admm_dose(h, view)
    ex = view.numpy().astype(np.float64) @ phic.astype(np.float64).T
    assert np.max(np.abs(got - ex)) < 1e-5 * max(1.0, np.abs(ex).max())
    one = b.admm_dose(h, view[1:2].contiguous())
    assert np.array_equal(one[0], got[1])                                          # a plan's dose does not depend on the batch
    with pytest.raises(b.AdmmError) as e:
        b.admm_lowdose_volumes(h, view.numpy().copy(), 0.5, 0.5)                   # empty range
    assert e.value.status == b.ADMM_EINVAL
    with pytest.raises(b.AdmmError) as e:
        b.admm_contract_probe(h, 0, np.zeros((2, phic.shape[0]), np.float32))      # no Phi^T on a dose-only handle
    assert e.value.status == b.ADMM_ESTATE
    with pytest.raises(b.AdmmError) as e:
        b.admm_get_preconditioner(h)
    assert e.value.status == b.ADMM_ESTATE
    h.close()

"""Sector / isocenter coupling of PAPER.md App. A (Eq. 12, 16, 17, :316, :330-332) through the C ABI: the coupling columns
(-C_S^T ; T^T) as rows of the extended Phi with a homogeneous hard class (hard = 2: c = 0, u = infinity) and b = (0, w_BOT)
(admm_options.bot_rows), against the oracle."""
import numpy as np
import pytest

from conftest import have_cuda
from parity_util import block2_errors, stacked_errors, t_errors

pytestmark = [pytest.mark.gpu, pytest.mark.skipif(not have_cuda(), reason="needs a CUDA device")]

TOL_FP32 = 1e-4


@pytest.fixture(scope="module")
def b():
    from paper_2509_08602_b200 import binding
    return binding


def test_fixed_k_parity_with_coupling(b):
    """K = 50 iterates of the coupled problem (n = 240 collimator times + 10 isocenter times, N = 3000 points + 80 coupling
    variables, ragged in both dimensions) against the oracle, all 9 plans, fp32 path and the SIMT cross-check path."""
    from oracle import admm
    from workloads import make_workload, scaled_rho, with_sector_coupling
    w0 = make_workload(0)
    w = with_sector_coupling(w0)
    rho = 0.3 * scaled_rho(w.beta, w0.point_class)
    ref = admm.solve_workload(w, rho, 50)
    assert (np.linalg.norm(ref["t"], axis=1) > 0).sum() >= 6
    for path in (b.ADMM_PATH_TCGEN05, b.ADMM_PATH_SIMT):
        h = b.admm_setup(w.phi, w.point_class, w.classes, bot_rows=w.bot_rows, kernel_path=path)
        out = b.admm_solve_batch(h, w.weights, rho, fixed_iters=50)
        states = [b.admm_get_state(h, p) for p in range(w.B)]
        h.close()
        ez, ey = stacked_errors(states, ref)
        ez2, ey2 = block2_errors(states, ref)
        et = t_errors(out["t"], ref["t"])
        eobj = np.abs(out["obj"] - ref["obj"]) / np.maximum(np.abs(ref["obj"]), 0.1)
        deg = (w.alpha == 0) & (w.beta == 0)
        assert ez.max() < TOL_FP32 and ey.max() < TOL_FP32, (path, ez.max(), ey.max())
        assert ez2[~deg].max() < TOL_FP32 and ey2[~deg].max() < TOL_FP32 and et[~deg].max() < TOL_FP32, (path, ez2, ey2, et)
        assert eobj[np.isfinite(ref["obj"])].max() < 1e-4


def test_converged_coupled_objectives_match_the_simplex(b):
    """Tolerance mode (presolve, stopping rule, compaction) on a coupled problem small enough for the dense simplex: converged
    objectives within 1e-3 of the LP optimum, the coupling constraints satisfied, and the isocenter time = its slowest sector."""
    from oracle import lp_model, simplex
    from workloads import make_workload, scaled_rho, with_sector_coupling
    w0 = make_workload(0, n_target=120, n_lowdose=240, n_iso=2, grid=3)
    w = with_sector_coupling(w0)
    rho = scaled_rho(w.beta, w0.point_class)
    h = b.admm_setup(w.phi, w.point_class, w.classes, bot_rows=w.bot_rows)
    out = b.admm_solve_batch(h, w.weights, rho, tol=1e-5, max_iter=20000)
    h.close()
    checked = 0
    for p in range(w.B):
        if out["iters"][p] >= 20000 or w.beta[p] == 0:
            continue
        opt = simplex.solve_plan(w.phi, w.point_class, w.classes, w.weights[p], bot_rows=w.bot_rows)["opt"]
        assert abs(out["obj"][p] - opt) / max(abs(opt), 0.1) < 1e-3, (p, out["obj"][p], opt)
        t = out["t"][p].astype(np.float64)
        assert lp_model.hard_violation(w.phi, w.point_class, w.classes, t) < 1e-3
        P = lp_model.primal_terms(w.phi, w.point_class, w.classes, w.weights[p], t, None, w.bot_rows)
        soft = P[0][:2].sum() + P[1]
        assert abs(out["obj"][p] - soft) / max(abs(soft), 0.1) < 1e-4                 # the library's P(t): w_BOT on the isocenter times only
        checked += 1
    assert checked >= 4


def test_fixed_k_parity_with_coupling_multitarget_and_row_masks(b):
    """The coupled problem on the multi-target geometry with per-plan low-dose row masks (configs 2-4's structure): 9 targets,
    18 isocenters (n = 432 + 18), 25 plans; K = 50 iterates against the oracle."""
    from oracle import admm
    from workloads import make_workload, scaled_rho, with_sector_coupling
    w0 = make_workload(2, n_target=1500, n_lowdose=3000, n_iso=18, grid=5)
    w = with_sector_coupling(w0)
    assert w.row_mask is not None and w.mask_bool()[:, w0.N:].all()
    rho = 0.3 * scaled_rho(w.beta, w0.point_class)
    ref = admm.solve_workload(w, rho, 50)
    h = b.admm_setup(w.phi, w.point_class, w.classes, bot_rows=w.bot_rows)
    out = b.admm_solve_batch(h, w.weights, rho, w.row_mask, fixed_iters=50)
    states = [b.admm_get_state(h, p) for p in range(w.B)]
    h.close()
    ez, ey = stacked_errors(states, ref)
    et = t_errors(out["t"], ref["t"])
    deg = (w.alpha == 0) & (w.beta == 0)
    assert ez.max() < TOL_FP32 and ey.max() < TOL_FP32 and et[~deg].max() < TOL_FP32, (ez.max(), ey.max(), et)


def test_coupling_with_reduced_storage(b):
    """The coupling rows (-1 / +1) are exact in tf32 and bf16, so the reduced-storage modes solve the coupled LP of the rounded Phi:
    K = 50 iterates against the oracle on the ORIGINAL Phi inside north_star's 1e-2 budget."""
    from oracle import admm
    from workloads import make_workload, scaled_rho, with_sector_coupling
    w0 = make_workload(0, n_target=600, n_lowdose=1200, n_iso=4, grid=3)
    w = with_sector_coupling(w0)
    rho = 0.3 * scaled_rho(w.beta, w0.point_class)
    ref = admm.solve_workload(w, rho, 50)
    for storage in (b.ADMM_STORAGE_FP32_TF32, b.ADMM_STORAGE_BF16):
        h = b.admm_setup(w.phi, w.point_class, w.classes, bot_rows=w.bot_rows, storage=storage)
        out = b.admm_solve_batch(h, w.weights, rho, fixed_iters=50)
        states = [b.admm_get_state(h, p) for p in range(w.B)]
        h.close()
        ez, ey = stacked_errors(states, ref)
        assert ez.max() < 1e-2 and ey.max() < 1e-2, (storage, ez.max(), ey.max())

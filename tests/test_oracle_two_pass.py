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


# ------------------------------------------------------------------------------------------ Algorithm 1 (:116-136)
def _disc(n, cx, r):
    """candidates on a line segment [0, n): the 'volume' of indices within r of cx"""
    i = np.arange(n)
    return np.abs(i - cx) <= r


def test_algorithm1_disjoint_and_identical_volumes():
    from workloads import uniform01
    vols = np.stack([_disc(6000, 1000, 500), _disc(6000, 3000, 400), _disc(6000, 5000, 300)])       # disjoint
    P, p, order = o2.overlapping_sampling(vols, [200, 200, 200], seed=1, uniform01=uniform01)
    assert order == [2, 1, 0]                                         # decreasing density = increasing volume here
    for j in range(3):
        assert len(p[j]) == 200 and all(vols[j][c] for c in p[j])     # exactly N_LD points, all inside V_j
    assert len(P) == 600
    same = np.stack([_disc(6000, 3000, 800)] * 4)                     # identical volumes, equal density: complete reuse
    P, p, _ = o2.overlapping_sampling(same, [300] * 4, seed=2, uniform01=uniform01)
    assert len(P) == 300 and all(pj == p[0] for pj in p)
    # an empty volume (a plan with t = 0) gets no points and does not disturb the others
    P2, p2, order2 = o2.overlapping_sampling(np.concatenate([same[:2], np.zeros((1, 6000), bool)]), [300] * 3, seed=2, uniform01=uniform01)
    assert len(p2[2]) == 0 and 2 not in order2 and len(p2[0]) == 300


def test_algorithm1_overlap_reuses_points_and_respects_eq8():
    """Overlapping volumes: points are shared, every p_j lies in V_j, |p_j| ~ N_LD,j with the spread of Eq. (8):
    relative std < 1 / sqrt(w_j |V_j|) (:148-155)."""
    from workloads import uniform01
    vols = np.stack([_disc(20000, 8000, 3000), _disc(20000, 10000, 4000), _disc(20000, 13000, 5000)])   # heavy overlaps
    n_ld = [400, 400, 400]
    counts = []
    for seed in range(40):
        P, p, order = o2.overlapping_sampling(vols, n_ld, seed=seed, uniform01=uniform01)
        assert all(all(vols[j][c] for c in p[j]) for j in range(3))
        assert len(P) < sum(len(x) for x in p)                                  # reuse: the union is smaller than the sum
        counts.append([len(x) for x in p])
    counts = np.array(counts, dtype=np.float64)
    assert np.all(np.abs(counts.mean(axis=0) - 400) < 0.05 * 400)               # the desired number in expectation
    rel_std = counts.std(axis=0) / 400
    assert np.all(rel_std < 1.0 / np.sqrt(400)), rel_std                        # Eq. (8)
    assert rel_std[order[0]] == 0                                               # the first (densest) volume is sampled exactly


def test_algorithm1_product_host_logic_equals_the_oracle():
    """The driver's vectorised implementation returns exactly the oracle's point sets (index work: bit-exact)."""
    from paper_2509_08602_b200 import build
    build.build()                                   # the package imports its C library (nvcc cross-compiles without a GPU)
    from paper_2509_08602_b200.two_pass import overlapping_sampling as fast
    from workloads import uniform01
    rng = np.random.default_rng(4)
    for trial in range(5):
        m, n_c = 7, 3000
        centres = rng.integers(300, 2700, m); radii = rng.integers(50, 700, m)
        vols = np.stack([_disc(n_c, c, r) for c, r in zip(centres, radii)])
        vols[rng.integers(0, m)] = False                                        # one empty volume
        n_ld = rng.integers(20, 200, m)
        P, p, _ = o2.overlapping_sampling(vols, n_ld, seed=trial, uniform01=uniform01)
        Pf, member = fast(vols, n_ld, trial, uniform01)
        assert Pf.tolist() == P
        for j in range(m):
            assert set(Pf[member[j]].tolist()) == p[j]

"""fp64 CPU oracle for the batched-ADMM radiosurgery path (arXiv 2509.08602).

TEST INFRASTRUCTURE ONLY.  Nothing in the product path (`paper_2509_08602_b200/`) may
import, call, link or execute anything in this package; only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference` legs do.
The oracle shares no code with the CUDA path: the only common module is `workloads/`
(seeded input generators, no method arithmetic).

Contents (each function cites the PAPER.md passage it restates):
  lp_model.py   the LP itself: dual form Eq. (1)/(11)-(15), primal objective, weak-duality bracket
  simplex.py    O-LP: small dense bounded-variable simplex on the dual form (exact optimum)
  enumerate.py  brute-force vertex enumeration of the primal on tiny instances
  admm.py       O-ADMM: the iteration Eq. (4b), (4c), (6), (7), batched per :96, fp64, plain numpy

Pins (tests/test_oracle_*.py, all `-m "not gpu"`):
  simplex   <- vertex enumeration, KKT + zero duality gap, closed forms (t*=0 plans, n=1), HiGHS
  admm      <- PARITY UNPINNED BY THE PAPER (it prints no iterate and no worked example).
               Pinned instead by: the invariant A x1 = x2 after every x-update; Eq. (5) (sign-
               corrected) solved as one dense KKT system; by-construction complementarity; the
               fixed point at the simplex KKT point; scaling / permutation / batch-independence
               metamorphic relations; diag(S)=2 and |S_ij|<=1 (:213); and convergence of
               P(rho*R*y2) to the simplex optimum (:80).
"""

"""Writes tests/golden/c0_simplex_opt.txt: the exact LP optima of the 9 plans of config 0.

Calls only `workloads/` (inputs) and `oracle/` (fp64 simplex).  Nothing here comes from the
CUDA path.  Run from the repo root:  python tests/golden/make_golden.py
The paper prints no worked example (PAPER.md has no numeric iterate or optimum for a given
input), so these values are the oracle's, pinned in tests/test_oracle_lp.py by vertex
enumeration, KKT residuals, closed forms and an independent LP solver.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import simplex  # noqa: E402
from workloads import make_workload  # noqa: E402


def main():
    w = make_workload(0)
    rows = []
    for p in range(w.B):
        sx = simplex.solve_plan(w.phi, w.point_class, w.classes, w.weights[p])
        rows.append((p, w.alpha[p], w.beta[p], sx["opt"], float(np.sum(sx["t"]))))
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "c0_simplex_opt.txt")
    with open(out, "w") as f:
        f.write("# config 0 (BASELINE.json configs[0]): exact LP optimum per plan, oracle/simplex.py, fp64\n")
        f.write("# plan alpha beta OPT sum_t\n")
        for r in rows:
            f.write("%d %.17g %.17g %.17g %.17g\n" % r)
    print("wrote", out)


if __name__ == "__main__":
    main()

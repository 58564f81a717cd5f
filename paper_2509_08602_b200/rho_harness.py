"""rho grid search (PAPER.md III.C, :183, :215-222) run as ONE batched solve on the GPU.

The paper tunes the step size by solving a validation set for rho in {0.1 / 2^n, n = 0..15} and fits Eq. (9),
rho = rho0 sqrt(w0 / w_BOT).  Because rho enters the iteration only through the iterates (:222) and S does not depend on it (:91),
a (weighting, rho) pair is just another column of the batch: the harness stacks every beam-on-time weight of the slider grid
with every multiplier of the default rule as B = n_beta x n_mult plans, solves them together, and prints per weight the
iterations each multiplier needed and the objective it reached.

    python -m paper_2509_08602_b200.rho_harness --config 1 [--alpha 0.5] [--max-iter 3000] [--storage bf16]

Output: a table (rows = w_BOT, columns = multiplier of the library's default rule) and the best multiplier per row.  The default
rule of the library (admm_solve_batch with rho = NULL; workloads.scaled_rho) was fitted with this tool (reading R8).
"""
from __future__ import annotations

import argparse

import numpy as np


def grid_search(phi, point_class, classes, betas, multipliers, alpha=0.5, row_mask=None, max_iter=3000, tol=1e-4,
                storage=None, presolve=True):
    """Returns dict(iters [n_beta, n_mult], obj, res [.., 2]).  row_mask: one plan's packed mask (shared by all columns) or None."""
    import torch
    from . import binding as b
    from workloads import scaled_rho
    BB, MM = np.meshgrid(np.asarray(betas, dtype=np.float64), np.asarray(multipliers, dtype=np.float64), indexing="ij")
    B = BB.size
    if B > 496:
        raise ValueError("at most 496 (weight, multiplier) pairs per batch")
    K = len(classes)
    weights = np.concatenate([np.ones((B, 1)), np.full((B, K - 1), alpha), BB.reshape(B, 1)], axis=1)
    rho = scaled_rho(BB.ravel(), point_class) * MM.ravel()
    mask = None
    if row_mask is not None:
        mask = torch.from_numpy(np.repeat(np.asarray(row_mask).reshape(1, -1), B, axis=0).view(np.int32)).cuda()
    h = b.admm_setup(phi, point_class, classes, storage=b.ADMM_STORAGE_FP32_3XTF32 if storage is None else storage, presolve=presolve)
    out = b.admm_solve_batch(h, weights, rho, mask, tol=tol, max_iter=max_iter)
    h.close()
    shape = BB.shape
    return dict(iters=out["iters"].reshape(shape), obj=out["obj"].reshape(shape), res=out["res"].reshape(shape + (2,)))


def main() -> None:
    from . import binding as b
    from workloads import make_workload
    ap = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--alpha", type=float, default=0.5)
    ap.add_argument("--max-iter", type=int, default=3000)
    ap.add_argument("--n-beta", type=int, default=21)
    ap.add_argument("--log2-mult", type=int, nargs=2, default=(-7, 8), help="multipliers 2^a .. 2^b of the default rule")
    ap.add_argument("--storage", default="fp32", choices=["fp32", "tf32", "bf16"])
    ap.add_argument("--no-presolve", action="store_true")
    args = ap.parse_args()
    w = make_workload(args.config, plans=np.arange(1))
    betas = np.linspace(0.0, 1.0, args.n_beta)
    mults = 2.0 ** np.arange(args.log2_mult[0], args.log2_mult[1] + 1)
    storage = dict(fp32=b.ADMM_STORAGE_FP32_3XTF32, tf32=b.ADMM_STORAGE_FP32_TF32, bf16=b.ADMM_STORAGE_BF16)[args.storage]
    r = grid_search(w.phi, w.point_class, w.classes, betas, mults, alpha=args.alpha,
                    row_mask=None if w.row_mask is None else w.row_mask[0], max_iter=args.max_iter, storage=storage,
                    presolve=not args.no_presolve)
    np.set_printoptions(linewidth=250)
    print(f"config {args.config}: N={w.N} n={w.n}, alpha={args.alpha}; iterations to tol 1e-4 (cap {args.max_iter}; 0 = settled by the presolve)")
    print("w_BOT \\ log2(multiplier): " + " ".join(f"{int(np.log2(m)):5d}" for m in mults))
    best_obj = r["obj"].min(axis=1, keepdims=True)
    ok = (r["iters"] < args.max_iter) & ((r["obj"] - best_obj) / np.maximum(np.abs(best_obj), 0.1) < 1e-3)
    for i, bt in enumerate(betas):
        row = " ".join(f"{int(v):5d}" for v in r["iters"][i])
        cand = np.where(ok[i], r["iters"][i], np.iinfo(np.int32).max)
        best = f"best 2^{int(np.log2(mults[int(np.argmin(cand))]))}" if ok[i].any() else "none converged to the best objective"
        print(f"{bt:6.3f}                 {row}   {best}")


if __name__ == "__main__":
    main()

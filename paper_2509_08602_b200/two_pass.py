"""Two-pass optimisation (PAPER.md II.C, :108-114) on top of the C ABI: argument marshalling and index bookkeeping only.

Pass 1 solves all B weightings on the target points + a geometric low-dose shell (the weight-independent sampling of II.C.1).
The first-pass dose of every plan is then computed on a grid of candidate points (`admm_lowdose_volumes`: one batched Phi_cand . T
product + the range test [D_LD, D_LD + Delta) per plan, on the GPU), which gives each plan its second-pass low-dose VOLUME.  Pass 2
uses the paper's union construction (:144): the low-dose points are sampled once from the union of all plans' volumes, and a plan
keeps only the points inside its own volume -- every other low-dose row gets u = 0 through the per-plan row mask -- so that one
A and one S = A A^T + I serve all B second-pass problems.  (Algorithm 1, :116-136, which re-balances the sampling density per plan,
is not implemented.)

Every arithmetic step runs in the library's kernels (admm_setup, admm_solve_batch, admm_lowdose_volumes); this module stacks
matrices, picks indices and packs masks.
"""
from __future__ import annotations

from typing import Optional, Sequence

import numpy as np

from . import binding as b


def _unpack(bits: np.ndarray, N: int) -> np.ndarray:
    return np.unpackbits(np.ascontiguousarray(bits).view(np.uint8), axis=-1, bitorder="little")[..., :N].astype(bool)


def _pack(mask_bool: np.ndarray) -> np.ndarray:
    B, N = mask_bool.shape
    words = (N + 31) // 32
    padded = np.zeros((B, words * 32), dtype=np.uint8)
    padded[:, :N] = mask_bool
    return np.packbits(padded, axis=1, bitorder="little").view(np.uint32).reshape(B, words)


def two_pass(phi_target: np.ndarray, phi_shell: np.ndarray, phi_cand: np.ndarray, classes: Sequence, weights: np.ndarray, *,
             d_ld: float, delta: float, n_lowdose_2: int, pick, rho: Optional[np.ndarray] = None, tol: float = 1e-4,
             max_iter: int = 3000, storage: int = b.ADMM_STORAGE_FP32_3XTF32, **setup_kw) -> dict:
    """phi_target [N_T, n], phi_shell [N_L1, n], phi_cand [N_c, n] float32; classes = (target class, low-dose class);
    weights [B, 3] = (w_T, w_LD, w_BOT); [d_ld, d_ld + delta) = the second-pass dose range in the units of Phi t;
    n_lowdose_2 = low-dose points of pass 2; pick(union_bool, count) -> sorted indices (e.g. workloads.pick_from_union).
    Returns dict(pass1=..., pass2=..., selected=indices into the candidates, in_volume [B, N_c] bool, row_mask2)."""
    n_t, n_c = phi_target.shape[0], phi_cand.shape[0]
    # ---- pass 1: geometric shell, no masks
    phi1 = np.ascontiguousarray(np.concatenate([phi_target, phi_shell], axis=0), dtype=np.float32)
    pc1 = np.concatenate([np.zeros(n_t, np.uint8), np.ones(phi_shell.shape[0], np.uint8)])
    h1 = b.admm_setup(phi1, pc1, classes, storage=storage, **setup_kw)
    out1 = b.admm_solve_batch(h1, weights, rho, tol=tol, max_iter=max_iter)
    h1.close()
    # ---- first-pass dose on the candidates and every plan's second-pass low-dose volume (II.C.1)
    hd = b.admm_setup(np.ascontiguousarray(phi_cand, dtype=np.float32), np.zeros(n_c, np.uint8), classes[:1], storage=storage,
                      dose_only=True)
    in_bits, any_bits = b.admm_lowdose_volumes(hd, out1["t"], d_ld, d_ld + delta)
    hd.close()
    in_volume = _unpack(in_bits, n_c)
    union = _unpack(any_bits.reshape(1, -1), n_c)[0]
    # ---- the union construction (:144): one point set for all plans, a plan's own volume through its row mask
    sel = np.asarray(pick(union, int(n_lowdose_2)), dtype=np.int64)
    B = weights.shape[0]
    mask2 = np.concatenate([np.ones((B, n_t), dtype=bool), in_volume[:, sel]], axis=1)
    phi2 = np.ascontiguousarray(np.concatenate([phi_target, phi_cand[sel]], axis=0), dtype=np.float32)
    pc2 = np.concatenate([np.zeros(n_t, np.uint8), np.ones(sel.size, np.uint8)])
    row_mask2 = _pack(mask2)
    h2 = b.admm_setup(phi2, pc2, classes, storage=storage, **setup_kw)
    out2 = b.admm_solve_batch(h2, weights, rho, row_mask2, tol=tol, max_iter=max_iter)
    h2.close()
    return dict(pass1=out1, pass2=out2, selected=sel, in_volume=in_volume, union=union, row_mask2=row_mask2)

"""Two-pass optimisation (PAPER.md II.C, :108-114) on top of the C ABI: argument marshalling and index bookkeeping only.

Pass 1 solves all B weightings on the target points + a geometric low-dose shell (the weight-independent sampling of II.C.1).
The first-pass dose of every plan is then computed on a grid of candidate points (`admm_lowdose_volumes`: one batched Phi_cand . T
product + the range test [D_LD, D_LD + Delta) per plan, on the GPU), which gives each plan its second-pass low-dose VOLUME.  Pass 2
uses the paper's union construction (:144): the low-dose points are sampled once from the union of all plans' volumes, and a plan
keeps only the points inside its own volume -- every other low-dose row gets u = 0 through the per-plan row mask -- so that one
A and one S = A A^T + I serve all B second-pass problems.  With sampling = "algorithm1" the points come from Algorithm 1 instead
(:116-136, overlapping low-dose point sampling: every plan gets ~n_lowdose_2 points inside its own volume, with maximal reuse of
points between overlapping volumes); the row masks then carry each plan's own point set p_j.

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


def overlapping_sampling(in_volume: np.ndarray, n_ld, seed: int, uniform01):
    """Algorithm 1 on a discrete patient volume: in_volume [m, N_c] bool (plan j's low-dose volume V_j as
    candidate-grid membership), n_ld [m] or scalar = desired points per plan.  Volumes are taken in the order of decreasing sampling
    density w_j = N_LD,j / |V_j| (:146); "sample k points from a set" = the k members with the smallest counter-based uniform
    u(stream, index) (`uniform01(stream, indices)`, e.g. workloads.uniform01).  Returns (P sorted candidate indices,
    member [m, len(P)] bool: plan j keeps P[member[j]])."""
    vol = np.asarray(in_volume, dtype=bool)
    m, n_c = vol.shape
    n_ld = np.broadcast_to(np.asarray(n_ld, dtype=np.float64), (m,))
    size = vol.sum(axis=1).astype(np.float64)
    omega = np.where(size > 0, n_ld / np.maximum(size, 1.0), -1.0)
    order = [int(j) for j in np.argsort(-omega, kind="stable") if size[j] > 0]
    base = 2 * int(seed) * (m + 1)

    def sample(mask: np.ndarray, k: int, stream: int) -> np.ndarray:
        idx = np.nonzero(mask)[0]
        out = np.zeros(n_c, dtype=bool)
        if k >= idx.size:
            out[idx] = True
        elif k > 0:
            u = uniform01(stream, idx.astype(np.uint64))
            out[idx[np.argsort(u, kind="stable")[:k]]] = True
        return out
    v_union = np.zeros(n_c, dtype=bool); p_union = np.zeros(n_c, dtype=bool)
    p = np.zeros((m, n_c), dtype=bool)
    for step, j in enumerate(order):
        w = min(float(omega[j]), 1.0)
        p_tilde = sample(p_union, int(round(w * int(v_union.sum()))), base + 2 * step)
        fresh = vol[j] & ~v_union
        p_out = sample(fresh, int(round(w * int(fresh.sum()))), base + 2 * step + 1)
        p[j] = (p_tilde & vol[j]) | p_out
        p_union = p_tilde | p_out
        v_union |= vol[j]
    P = np.nonzero(p.any(axis=0))[0]
    return P, p[:, P]


def two_pass(phi_target: np.ndarray, phi_shell: np.ndarray, phi_cand: np.ndarray, classes: Sequence, weights: np.ndarray, *,
             d_ld: float, delta: float, n_lowdose_2: int, pick, rho: Optional[np.ndarray] = None, tol: float = 1e-4,
             max_iter: int = 3000, storage: int = b.ADMM_STORAGE_FP32_3XTF32, sampling: str = "union", uniform01=None,
             seed: int = 0, **setup_kw) -> dict:
    """phi_target [N_T, n], phi_shell [N_L1, n], phi_cand [N_c, n] float32; classes = (target class, low-dose class);
    weights [B, 3] = (w_T, w_LD, w_BOT); [d_ld, d_ld + delta) = the second-pass dose range in the units of Phi t;
    n_lowdose_2 = low-dose points of pass 2 (of the union with sampling = "union", per plan with "algorithm1");
    pick(union_bool, count) -> sorted indices (e.g. workloads.pick_from_union); uniform01, seed: Algorithm 1's random numbers.
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
    B = weights.shape[0]
    if sampling == "algorithm1":
        sel, member = overlapping_sampling(in_volume, n_lowdose_2, seed, uniform01)
    else:
        sel = np.asarray(pick(union, int(n_lowdose_2)), dtype=np.int64)
        member = in_volume[:, sel]
    mask2 = np.concatenate([np.ones((B, n_t), dtype=bool), member], axis=1)
    phi2 = np.ascontiguousarray(np.concatenate([phi_target, phi_cand[sel]], axis=0), dtype=np.float32)
    pc2 = np.concatenate([np.zeros(n_t, np.uint8), np.ones(sel.size, np.uint8)])
    row_mask2 = _pack(mask2)
    h2 = b.admm_setup(phi2, pc2, classes, storage=storage, **setup_kw)
    out2 = b.admm_solve_batch(h2, weights, rho, row_mask2, tol=tol, max_iter=max_iter)
    h2.close()
    return dict(pass1=out1, pass2=out2, selected=sel, in_volume=in_volume, union=union, row_mask2=row_mask2)

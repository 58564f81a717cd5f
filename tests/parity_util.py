"""Helpers shared by the GPU parity tests: the iterate-parity metric of DESIGN.md (reading R17)."""
import numpy as np


def stacked_errors(gpu_states, oracle_state):
    """gpu_states: list over plans of (z1, y1, z2, y2); oracle_state: dict with [N,B] / [n,B] arrays.
    Returns (err_z[B], err_y[B]): ||g - o||_2 / max(||o||_2, 1e-3 * max_p ||o_p||_2) on the stacked
    (z1, z2) and (y1, y2) vectors."""
    B = len(gpu_states)
    oz = np.concatenate([oracle_state["z1"], oracle_state["z2"]], axis=0)
    oy = np.concatenate([oracle_state["y1"], oracle_state["y2"]], axis=0)
    nz = np.linalg.norm(oz, axis=0); ny = np.linalg.norm(oy, axis=0)
    ez = np.zeros(B); ey = np.zeros(B)
    for p, (z1, y1, z2, y2) in enumerate(gpu_states):
        gz = np.concatenate([z1.astype(np.float64), z2]); gy = np.concatenate([y1.astype(np.float64), y2])
        ez[p] = np.linalg.norm(gz - oz[:, p]) / max(nz[p], 1e-3 * nz.max(), 1e-300)
        ey[p] = np.linalg.norm(gy - oy[:, p]) / max(ny[p], 1e-3 * ny.max(), 1e-300)
    return ez, ey


def t_errors(t_gpu, t_oracle):
    nt = np.linalg.norm(t_oracle, axis=1)
    return np.linalg.norm(t_gpu.astype(np.float64) - t_oracle, axis=1) / np.maximum(nt, max(1e-3 * nt.max(), 1e-300))


def block2_errors(gpu_states, oracle_state):
    """Block 2 alone (the n time variables: 2 % of the stacked vector, but all of t): per plan
    ||g - o||_2 / max(||o||_2, 1e-3 max_p ||o_p||_2) on z2 and on y2."""
    out = []
    for key, idx in (("z2", 2), ("y2", 3)):
        o = oracle_state[key]
        no = np.linalg.norm(o, axis=0)
        floor = max(1e-3 * no.max(), 1e-300)
        out.append(np.array([np.linalg.norm(st[idx] - o[:, p]) / max(no[p], floor) for p, st in enumerate(gpu_states)]))
    return out

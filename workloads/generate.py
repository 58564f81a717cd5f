"""Seeded generators for the synthetic Gamma-Knife-like workloads (BASELINE.json configs 0-4).

Inputs only.  Nothing here belongs to the ADMM method: no scaling, no projection, no
Schur complement.  Both `oracle/` and the CUDA path consume these arrays unchanged.

Stand-in statement: the paper measures on 20 anonymised clinical cases exported from
GammaPlan (Table 1 :187-211).  Those are not available; these generators
produce inputs with the same structure (dense non-negative dose-rate kernels, one block
of target rows with sense ">=" and one of low-dose rows with sense "<=", 24 time
variables per isocenter = 8 sectors x 3 collimators).

RNG: SplitMix64 used as a counter-based generator: the k-th draw of stream `seed` is
mix(seed + (k+1)*GOLDEN); u = (x >> 11) * 2**-53.  No transcendental function is used in
sampling (rejection from bounding cubes), so the geometry is bit-portable; Phi itself
is computed in fp64 with numpy's exp and rounded to fp32.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Tuple

import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np

SEED_BASE = 250908602
_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)

# stream ids (added to SEED_BASE + 1000*config)
_S_RADII, _S_CENTRES, _S_TARGET, _S_LOWDOSE, _S_ISO, _S_GAINS, _S_MASKQ, _S_MASKROW, _S_CAND, _S_PICK = range(10)

COLLIMATOR_SIGMA_MM = (2.0, 4.0, 8.0)
N_SECTORS = 8


def splitmix64(seed: int, counters: np.ndarray) -> np.ndarray:
    """k-th output of the SplitMix64 sequence started at `seed` (k = counters, 0-based)."""
    with np.errstate(over="ignore"):
        k = np.asarray(counters, dtype=np.uint64)
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + (k + np.uint64(1)) * _GOLDEN
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(seed: int, counters: np.ndarray) -> np.ndarray:
    """fp64 uniforms in [0, 1) with 53 random bits."""
    return (splitmix64(seed, counters) >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


@dataclass(frozen=True)
class ClassSpec:
    """One dose-point class.  sense=+1: penalise dose BELOW threshold (target);
    sense=-1: penalise dose ABOVE threshold (low-dose / ring).  PAPER.md:41, :314-326."""
    sense: int
    threshold: float
    hard: int = 0


@dataclass
class Workload:
    name: str
    config: int
    phi: np.ndarray                      # [N, n] float32, C-contiguous (dose rate at point i per unit time j)
    point_class: np.ndarray              # [N] uint8
    classes: List[ClassSpec]
    weights: np.ndarray                  # [B, n_classes + 1] float64: class weights..., w_BOT
    row_mask: Optional[np.ndarray]       # [B, ceil(N/32)] uint32 bit-packed (bit i%32 of word i//32), or None
    alpha: np.ndarray                    # [B]
    beta: np.ndarray                     # [B]
    points: np.ndarray = field(repr=False, default=None)       # [N, 3] mm
    isocenters: np.ndarray = field(repr=False, default=None)   # [n_iso, 3] mm
    radii: np.ndarray = field(repr=False, default=None)
    centres: np.ndarray = field(repr=False, default=None)
    bot_rows: Optional[np.ndarray] = field(repr=False, default=None)   # [n] uint8: rows of A that carry w_BOT in b (None = all)

    @property
    def N(self) -> int:
        return int(self.phi.shape[0])

    @property
    def n(self) -> int:
        return int(self.phi.shape[1])

    @property
    def B(self) -> int:
        return int(self.weights.shape[0])

    def mask_bool(self) -> np.ndarray:
        """[B, N] bool view of row_mask (all True if there is no mask)."""
        if self.row_mask is None:
            return np.ones((self.B, self.N), dtype=bool)
        bits = np.unpackbits(self.row_mask.view(np.uint8), axis=1, bitorder="little")
        return bits[:, : self.N].astype(bool)

    def subset(self, plans) -> "Workload":
        """Same case, a subset of the plans (plans are independent columns)."""
        plans = np.asarray(plans, dtype=np.int64)
        return Workload(
            name=f"{self.name}[{len(plans)} plans]", config=self.config, phi=self.phi,
            point_class=self.point_class, classes=self.classes, weights=self.weights[plans].copy(),
            row_mask=None if self.row_mask is None else self.row_mask[plans].copy(),
            alpha=self.alpha[plans].copy(), beta=self.beta[plans].copy(), points=self.points,
            isocenters=self.isocenters, radii=self.radii, centres=self.centres, bot_rows=self.bot_rows)


# name -> (n_targets, total_volume_mm3, N_T, N_L, shell_outer_mm, n_iso, grid, masked)
CONFIGS: Dict[int, dict] = {
    0: dict(n_targets=1, volume=4.0 / 3.0 * np.pi * 5.0 ** 3, n_target=1000, n_lowdose=2000,
            shell_outer=10.0, n_iso=10, grid=3, masked=False),
    1: dict(n_targets=1, volume=3000.0, n_target=20000, n_lowdose=40000,
            shell_outer=20.0, n_iso=60, grid=9, masked=False),
    2: dict(n_targets=9, volume=52000.0, n_target=150000, n_lowdose=300000,
            shell_outer=20.0, n_iso=400, grid=9, masked=True),
    3: dict(n_targets=9, volume=52000.0, n_target=150000, n_lowdose=300000,
            shell_outer=20.0, n_iso=400, grid=21, masked=True),
    4: dict(n_targets=9, volume=52000.0, n_target=200000, n_lowdose=400000,
            shell_outer=20.0, n_iso=500, grid=21, masked=True),
}
SHELL_INNER_MM = 2.0
MIN_CENTRE_DIST_MM = 25.0
CENTRE_BALL_MM = 80.0


def weight_grid(grid: int) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """(alpha, beta) on a grid x grid lattice over [0,1]^2; plan p = i_alpha*grid + i_beta.
    weights row = (w_T=1, w_LD=alpha (dose units), w_BOT=beta)."""
    v = np.arange(grid, dtype=np.float64) / float(grid - 1)
    alpha = np.repeat(v, grid)
    beta = np.tile(v, grid)
    weights = np.stack([np.ones_like(alpha), alpha, beta], axis=1)
    return alpha, beta, weights


def default_rho(beta: np.ndarray, rho0: float = 1e-3, beta0: float = 0.05) -> np.ndarray:
    """Per-plan step size, the shape of PAPER.md Eq. (9) (:219-222): rho = rho0*sqrt(w0/w_BOT) with
    w0 the smallest non-zero slider step; w_BOT below w0 (incl. 0, outside the paper's domain) is
    clamped to w0.  rho is an INPUT of both the oracle and the CUDA path (reading R8)."""
    beta = np.asarray(beta, dtype=np.float64)
    return rho0 * np.sqrt(beta0 / np.maximum(beta, beta0))


def scaled_rho(beta: np.ndarray, point_class: np.ndarray, kappa: float = 1.0, beta0: float = 0.05,
               floor_div: float = 65536.0) -> np.ndarray:
    """Size-aware step size (reading R8): rho_p = (kappa / N_min) * sqrt(beta0 / max(beta_p, beta0/floor_div)),
    N_min = the smallest class count.  With the column scaling D_i = 1/N_class(i) (R10) the linear term of the
    iteration is c_hat/rho = -+1/(N_k rho), so rho0 = kappa/N_min keeps it O(1/kappa) whatever the number of dose
    points; the lower clamp lets rho grow 256x towards w_BOT = 0 (Eq. 9 has rho -> inf there; the rho grid harness of
    III.C run on configs 1 and 3 puts the best multiplier for w_BOT = 0 at 2^4..2^5 above the former 8x clamp).
    For config 0 (N_T = 1000) and beta >= beta0 this is default_rho().  The library's rho = NULL default is the same rule."""
    beta = np.asarray(beta, dtype=np.float64)
    n_min = float(np.bincount(np.asarray(point_class).astype(np.int64)).min())
    return (kappa / n_min) * np.sqrt(beta0 / np.maximum(beta, beta0 / floor_div))


def pack_mask(mask_bool: np.ndarray) -> np.ndarray:
    """[B, N] bool -> [B, ceil(N/32)] uint32, bit (i % 32) of word (i // 32)."""
    B, N = mask_bool.shape
    words = (N + 31) // 32
    padded = np.zeros((B, words * 32), dtype=np.uint8)
    padded[:, :N] = mask_bool
    return np.packbits(padded, axis=1, bitorder="little").view(np.uint32).reshape(B, words)


def _rejection(seed: int, count: int, half: float, accept, centre=None, block: int = 1 << 16) -> np.ndarray:
    """First `count` accepted candidates, in candidate order, of uniform draws from the cube
    [-half, half]^3 (+centre).  Candidate q uses counters 3q, 3q+1, 3q+2."""
    out = np.empty((count, 3), dtype=np.float64)
    got, q0 = 0, 0
    while got < count:
        q = np.arange(q0, q0 + block, dtype=np.uint64)
        xyz = np.stack([uniform01(seed, np.uint64(3) * q + np.uint64(d)) for d in range(3)], axis=1)
        xyz = (2.0 * xyz - 1.0) * half
        if centre is not None:
            xyz = xyz + centre
        keep = xyz[accept(xyz)]
        take = min(count - got, keep.shape[0])
        out[got:got + take] = keep[:take]
        got += take
        q0 += block
    return out


def _apportion(total: int, shares: np.ndarray) -> np.ndarray:
    """Largest-remainder split of `total` items in proportion to `shares` (each gets >= 1)."""
    raw = total * shares / shares.sum()
    base = np.maximum(np.floor(raw).astype(np.int64), 1)
    rem = raw - np.floor(raw)
    while base.sum() < total:
        k = int(np.argmax(rem)); base[k] += 1; rem[k] = -1.0
    while base.sum() > total:
        k = int(np.argmax(base)); base[k] -= 1
    return base


def _geometry(config: int, n_targets: int, volume: float, seed0: int):
    if n_targets == 1:
        r = (volume * 3.0 / (4.0 * np.pi)) ** (1.0 / 3.0)
        return np.array([r]), np.zeros((1, 3))
    raw = 0.5 + uniform01(seed0 + _S_RADII, np.arange(n_targets))
    scale = (volume / (4.0 / 3.0 * np.pi * np.sum(raw ** 3))) ** (1.0 / 3.0)
    radii = raw * scale
    centres = np.zeros((n_targets, 3))
    placed, q = 0, 0
    while placed < n_targets:
        u = np.array([uniform01(seed0 + _S_CENTRES, np.array([3 * q + d]))[0] for d in range(3)])
        q += 1
        c = (2.0 * u - 1.0) * CENTRE_BALL_MM
        if c @ c > CENTRE_BALL_MM ** 2:
            continue
        ok = True
        for k in range(placed):
            dmin = max(MIN_CENTRE_DIST_MM, radii[k] + radii[placed] + SHELL_INNER_MM)
            if np.linalg.norm(c - centres[k]) < dmin:
                ok = False
                break
        if ok:
            centres[placed] = c
            placed += 1
    return radii, centres


def _phi(points: np.ndarray, iso: np.ndarray, gains: np.ndarray, chunk: int = 8192) -> np.ndarray:
    """Phi[i, (iso*8 + s)*3 + c] = a_s * exp(-|p_i - c_iso|^2 / (2 sigma_c^2)), fp64 -> fp32,
    magnitudes below the smallest normal fp32 flushed to 0."""
    N, n_iso = points.shape[0], iso.shape[0]
    n = n_iso * N_SECTORS * len(COLLIMATOR_SIGMA_MM)
    phi = np.empty((N, n), dtype=np.float32)
    inv2s2 = 1.0 / (2.0 * np.asarray(COLLIMATOR_SIGMA_MM) ** 2)
    tiny = float(np.finfo(np.float32).tiny)
    def fill(a: int) -> None:
        p = points[a:a + chunk]
        d2 = ((p[:, None, :] - iso[None, :, :]) ** 2).sum(axis=2)             # [c, n_iso]
        e = np.exp(-d2[:, :, None] * inv2s2[None, None, :])                    # [c, n_iso, 3]
        blk = gains[None, None, :, None] * e[:, :, None, :]                    # [c, n_iso, 8, 3]
        blk[np.abs(blk) < tiny] = 0.0
        phi[a:a + chunk] = blk.reshape(p.shape[0], n).astype(np.float32)
    # row chunks are independent: the large cases (17-29 GB) are filled by a pool of threads (numpy releases the GIL inside
    # the array operations); every element is computed by the same operations whatever the number of workers
    starts = range(0, N, chunk)
    workers = min(len(starts), os.cpu_count() or 1, 32)
    if workers <= 1 or N * n < (1 << 24):
        for a in starts:
            fill(a)
    else:
        with ThreadPoolExecutor(max_workers=workers) as pool:
            list(pool.map(fill, starts))
    return phi


def _plans(config: int, grid: int, masked: bool, point_class: np.ndarray):
    """The plans of a configuration: the (alpha, beta) lattice and, for the masked configurations, each plan's low-dose row subset."""
    alpha, beta, weights = weight_grid(grid)
    B, N = weights.shape[0], point_class.shape[0]
    row_mask = None
    if masked:
        # per-plan low-dose subset: q_p ~ U(0.8, 1); low-dose row i is active in plan p
        # iff u(p, i) < q_p; target rows are always active.
        mseed = SEED_BASE + 1000 * config
        qp = 0.8 + 0.2 * uniform01(mseed + _S_MASKQ, np.arange(B))
        mb = np.ones((B, N), dtype=bool)
        ld_idx = np.nonzero(point_class == 1)[0].astype(np.uint64)
        for p in range(B):
            u = uniform01(mseed + _S_MASKROW, (np.uint64(p + 1) << np.uint64(32)) + ld_idx)
            mb[p, ld_idx.astype(np.int64)] = u < qp[p]
        row_mask = pack_mask(mb)
    return alpha, beta, weights, row_mask


def with_plans_of(w: Workload, config: int) -> Workload:
    """The case of `w` (same Phi, points, classes) with the plans of another configuration that shares its geometry: configs 2 and 3
    are one case with 81 and 441 plans (BASELINE.json: "Config 2 shapes with B=441"), so one generated Phi (17 GB) serves both."""
    geo = lambda c: 2 if c == 3 else c
    if geo(config) != geo(w.config) or w.N != CONFIGS[config]["n_target"] + CONFIGS[config]["n_lowdose"]:
        raise ValueError("with_plans_of: the configurations do not share a geometry")
    alpha, beta, weights, row_mask = _plans(config, CONFIGS[config]["grid"], CONFIGS[config]["masked"], w.point_class)
    return Workload(name=f"config{config}", config=config, phi=w.phi, point_class=w.point_class, classes=w.classes, weights=weights,
                    row_mask=row_mask, alpha=alpha, beta=beta, points=w.points, isocenters=w.isocenters, radii=w.radii, centres=w.centres)


def make_workload(config: int, *, n_target: Optional[int] = None, n_lowdose: Optional[int] = None,
                  n_iso: Optional[int] = None, grid: Optional[int] = None,
                  plans: Optional[np.ndarray] = None) -> Workload:
    """Build config 0-4.  The keyword overrides shrink the case for tests (same geometry
    recipe and seeds, fewer points / isocenters / plans); `plans` keeps a subset of plans."""
    spec = dict(CONFIGS[config])
    if n_target is not None: spec["n_target"] = int(n_target)
    if n_lowdose is not None: spec["n_lowdose"] = int(n_lowdose)
    if n_iso is not None: spec["n_iso"] = int(n_iso)
    if grid is not None: spec["grid"] = int(grid)
    # configs 2 and 3 share one geometry (BASELINE.json: "Config 2 shapes with B=441")
    geo_cfg = 2 if config == 3 else config
    seed0 = SEED_BASE + 1000 * geo_cfg
    radii, centres = _geometry(geo_cfg, spec["n_targets"], spec["volume"], seed0)
    K = len(radii)
    vol = radii ** 3
    nT = _apportion(spec["n_target"], vol) if K > 1 else np.array([spec["n_target"]])
    nI = _apportion(spec["n_iso"], vol) if K > 1 else np.array([spec["n_iso"]])

    tpts, isos = [], []
    for k in range(K):
        r, c = radii[k], centres[k]
        inside = lambda x, r=r, c=c: ((x - c) ** 2).sum(axis=1) <= r * r
        tpts.append(_rejection(seed0 + _S_TARGET + 100 * k, int(nT[k]), r, inside, centre=c))
        isos.append(_rejection(seed0 + _S_ISO + 100 * k, int(nI[k]), r, inside, centre=c,
                               block=max(256, 8 * int(nI[k]))))
    target_pts = np.concatenate(tpts, axis=0)
    iso = np.concatenate(isos, axis=0)

    r_out = spec["shell_outer"]
    if K == 1:
        r = radii[0]
        def in_shell(x, r=r):
            d2 = (x ** 2).sum(axis=1)
            return (d2 >= (r + SHELL_INNER_MM) ** 2) & (d2 <= (r + r_out) ** 2)
        ld_pts = _rejection(seed0 + _S_LOWDOSE, spec["n_lowdose"], r + r_out, in_shell)
    else:
        half = CENTRE_BALL_MM + float(radii.max()) + r_out
        def in_union(x):
            d = np.sqrt(((x[:, None, :] - centres[None, :, :]) ** 2).sum(axis=2))    # [c, K]
            in_any = ((d >= radii + SHELL_INNER_MM) & (d <= radii + r_out)).any(axis=1)
            too_close = (d < radii + SHELL_INNER_MM).any(axis=1)
            return in_any & ~too_close
        ld_pts = _rejection(seed0 + _S_LOWDOSE, spec["n_lowdose"], half, in_union)

    points = np.concatenate([target_pts, ld_pts], axis=0)
    point_class = np.concatenate([np.zeros(target_pts.shape[0], np.uint8),
                                  np.ones(ld_pts.shape[0], np.uint8)])
    gains = 0.8 + 0.4 * uniform01(seed0 + _S_GAINS, np.arange(N_SECTORS))
    phi = _phi(points, iso, gains)

    alpha, beta, weights, row_mask = _plans(config, spec["grid"], spec["masked"], point_class)

    w = Workload(name=f"config{config}", config=config, phi=phi, point_class=point_class,
                 classes=[ClassSpec(+1, 1.0), ClassSpec(-1, 0.5)], weights=weights,
                 row_mask=row_mask, alpha=alpha, beta=beta, points=points, isocenters=iso,
                 radii=radii, centres=centres)
    if plans is not None:
        w = w.subset(plans)
    return w


def make_tiny_workload(seed: int, N_T: int, N_L: int, n: int, B_alpha=(0.0, 0.5, 1.0),
                       B_beta=(0.0, 0.25, 1.0)) -> Workload:
    """Unstructured tiny instance for brute-force pins: Phi ~ U(0,1)^(N x n), no geometry."""
    N = N_T + N_L
    phi = uniform01(seed, np.arange(N * n)).reshape(N, n).astype(np.float32)
    point_class = np.concatenate([np.zeros(N_T, np.uint8), np.ones(N_L, np.uint8)])
    alpha = np.repeat(np.asarray(B_alpha, dtype=np.float64), len(B_beta))
    beta = np.tile(np.asarray(B_beta, dtype=np.float64), len(B_alpha))
    weights = np.stack([np.ones_like(alpha), alpha, beta], axis=1)
    return Workload(name=f"tiny{seed}", config=-1, phi=phi, point_class=point_class,
                    classes=[ClassSpec(+1, 1.0), ClassSpec(-1, 0.5)], weights=weights,
                    row_mask=None, alpha=alpha, beta=beta)


def make_candidates(w: Workload, n_cand: int):
    """Candidate dose points for the SECOND pass of the two-pass optimisation (PAPER.md II.C, :108-114): `n_cand` seeded points
    uniform in the tissue around the targets of `w` (outside every target, within the configuration's outer shell distance of
    some target surface -- a superset of the first-pass geometric shell, which starts 2 mm out), and their dose-rate rows
    Phi_cand [n_cand, n] for the isocenters / sectors / collimators of `w`.  Stand-in for the patient dose grid."""
    geo_cfg = 2 if w.config == 3 else w.config
    seed0 = SEED_BASE + 1000 * geo_cfg
    radii, centres = np.asarray(w.radii), np.asarray(w.centres)
    r_out = CONFIGS[geo_cfg]["shell_outer"]
    if len(radii) == 1:
        half = float(radii[0]) + r_out
    else:
        half = CENTRE_BALL_MM + float(radii.max()) + r_out

    def in_region(x):
        d = np.sqrt(((x[:, None, :] - centres[None, :, :]) ** 2).sum(axis=2)) - radii[None, :]     # signed distance to each target surface
        return (d > 0).all(axis=1) & (d <= r_out).any(axis=1)
    pts = _rejection(seed0 + _S_CAND, int(n_cand), half, in_region)
    gains = 0.8 + 0.4 * uniform01(seed0 + _S_GAINS, np.arange(N_SECTORS))
    return pts, _phi(pts, w.isocenters, gains)


def pick_from_union(union: np.ndarray, count: int, seed: int) -> np.ndarray:
    """`count` of the indices i with union[i] set, uniformly at random without replacement and reproducibly: the members with the
    `count` smallest values of the counter-based uniform u(seed, i) (all of them if there are fewer).  Sorted ascending.
    ("sample from the union of all low-dose volumes".)"""
    idx = np.nonzero(np.asarray(union, dtype=bool))[0]
    if idx.size <= count:
        return idx
    u = uniform01(SEED_BASE + _S_PICK + 1000003 * int(seed), idx.astype(np.uint64))
    return np.sort(idx[np.argsort(u, kind="stable")[:count]])



def with_sector_coupling(w: Workload, scale: float = 1.0) -> Workload:
    """The case of `w` with the sector / isocenter coupling of PAPER.md App. A (Eq. 12, 16, 17, :316, :330-332): one time variable
    tau_iso per isocenter is appended (n -> n + N_iso) and one dual variable per (isocenter, sector) (N -> N + 8 N_iso), whose
    row of the extended Phi is  -1/scale on the three collimator times of that sector (C = I (x) I_8 (x) 1_{1x3}) and +1 on tau_iso
    (T = I (x) 1_{8x1}); its class is homogeneous hard (sense +1, threshold 1, hard = 2: c = 0, u = infinity) and only the tau rows
    carry w_BOT in b (Eq. 13).  Column j of w.phi is time variable (iso*8 + s)*3 + c."""
    n_iso = w.n // (N_SECTORS * len(COLLIMATOR_SIGMA_MM))
    assert n_iso * N_SECTORS * len(COLLIMATOR_SIGMA_MM) == w.n
    n_c = N_SECTORS * n_iso
    phi = np.zeros((w.N + n_c, w.n + n_iso), dtype=np.float32)
    phi[:w.N, :w.n] = w.phi
    for k in range(n_c):
        phi[w.N + k, 3 * k:3 * k + 3] = -1.0 / scale
        phi[w.N + k, w.n + k // N_SECTORS] = 1.0
    pc = np.concatenate([w.point_class, np.full(n_c, len(w.classes), dtype=np.uint8)])
    classes = list(w.classes) + [ClassSpec(+1, 1.0, hard=2)]
    weights = np.concatenate([w.weights[:, :-1], np.zeros((w.B, 1)), w.weights[:, -1:]], axis=1)     # the coupling class has no weight
    bot = np.concatenate([np.zeros(w.n, np.uint8), np.ones(n_iso, np.uint8)])
    row_mask = None
    if w.row_mask is not None:                        # the coupling variables are active in every plan
        row_mask = pack_mask(np.concatenate([w.mask_bool(), np.ones((w.B, n_c), dtype=bool)], axis=1))
    return Workload(name=w.name + "+coupling", config=w.config, phi=phi, point_class=pc, classes=classes, weights=weights,
                    row_mask=row_mask, alpha=w.alpha, beta=w.beta, points=w.points, isocenters=w.isocenters, radii=w.radii,
                    centres=w.centres, bot_rows=bot)

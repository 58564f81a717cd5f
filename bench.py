"""bench.py -- plan-iterations/s and time-to-converge of the batched ADMM hot path (BASELINE.json metric) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C] [--storage fp32|tf32|bf16]

Workload: BASELINE.json configs[3] -- the 9-target case (N = 450000 dose points x n = 9600 time variables, dense fp32 Phi, 17.3 GB)
with the B = 441 plans of the 21 x 21 slider grid, per-plan low-dose row masks, convergence masking + compaction, tol 1e-4 -- the
configuration the metric is quoted on ("time-to-converge for B=81/441 plans").  configs[2] (the same Phi with the B = 81 plans of the
9 x 9 grid) is solved in the same run and reported inside the same JSON line (`config2`).

A "step" is ONE pass of the whole hot path over one batch of synthetic input: admm_solve_batch of all B plans from the zero iterate
(presolve, iterations with per-plan stopping + device-side compaction until every plan has converged or reached the cap of 3000
iterations = the paper's fixed count, then the objective evaluation).  `value` = plan-iterations done / device time
of the K timed steps.  Setup (upload, S = I + A A^T, Cholesky, inverse) is done once before the timed region and reported separately
(north_star: "timed separately"); the `e2e` leg times setup + solve from HOST buffers (pinned Phi in, host results out).

The headline is the fp32 path (3xTF32 products) from the zero iterate; the bf16-storage figures of the same workload are a second,
labelled object (`bf16_storage`), and `w_bot_positive` is the same solve restricted to the plans inside the paper's domain (w_BOT > 0),
without and with the warm start of deviation D3.  `full_batch` = a fixed-iteration run of all 441 plans (no plan frozen): the tensor-pipe-bound regime.

N > 1 (torchrun): weak scaling, plans are independent columns: every rank holds a replica of Phi and solves its own
B plans (a shifted slider grid); no data-path collective; value = all ranks' plan iterations / max-over-ranks device time.

--impl reference: there is no reference implementation (the reference is a paper); per the tier contract this arm times the fp64
numpy oracle, as it stands, on the host cores, on a bounded sample of the same workload (see _oracle_sample).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "plan_iterations_per_s"
UNIT = "plan-iterations/s"
TOL = 1e-4
MAX_ITER = 3000
SAMPLE_PLANS = 16          # oracle sample: this many plans ...
SAMPLE_ROW_STRIDE = 16     # ... on every 16th dose point of the large configurations (configs 0-1: all rows, all plans)


def _workload_desc(w, cfg):
    return (f"config{cfg}: N={w.N} points x n={w.n} time variables, B={w.B} plans, dense fp32 Phi {w.N * w.n * 4 / 1e9:.2f} GB"
            + (", per-plan low-dose row masks" if w.row_mask is not None else ""))


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return dict(hbm=float(d["hbm_gbs"]), bf16=float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                    source="measured (MEASURED_PEAKS.json: hbm_gbs, bf16_tflops_sustained)")
    return dict(hbm=6650.0, bf16=1380.0, source="fallback (B200_PROFILING.md: 6.65 TB/s copy, 1380 TFLOP/s sustained bf16)")


class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200",
                                       "-i", str(gpu_index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        time.sleep(0.25)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush(); self.f.seek(0)
        sm, mx, reasons = [], [], set()
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        self.f.close()
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons), samples=len(sm))
        return out


def rank_weights(weights: np.ndarray, rank: int, world: int) -> np.ndarray:
    """Weak scaling: rank r solves its own B plans -- the slider grid with the low-dose weight shifted by a
    fraction of one grid step, clipped to [0, 1].  Rank 0 always gets the unshifted grid."""
    B = weights.shape[0]
    g = max(int(round(np.sqrt(B))) - 1, 1)
    out = np.array(weights, dtype=np.float64, copy=True)
    out[:, 1] = np.clip(out[:, 1] + rank / (8.0 * max(world, 1)) / g, 0.0, 1.0)
    return out


def reduce_max_sum(dist, device, max_vals, sum_vals):
    """max over ranks of `max_vals`, sum over ranks of `sum_vals` (lists of floats); identity if not initialised."""
    import torch
    if dist is None or not dist.is_initialized():
        return list(max_vals), list(sum_vals)
    a = torch.tensor(list(max_vals), dtype=torch.float64, device=device)
    c = torch.tensor(list(sum_vals), dtype=torch.float64, device=device)
    dist.all_reduce(a, op=dist.ReduceOp.MAX)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return a.tolist(), c.tolist()


# ------------------------------------------------------------------------------------------------ the oracle, timed
def flops_per_plan_iteration(N: int, n: int) -> float:
    """Algorithmic flops of one plan-iteration of the oracle: the two Phi products (4 N n) and the two triangular solves (4 n^2)."""
    return 4.0 * N * n + 4.0 * n * n


def sample_workload(w):
    """The bounded sample the oracle is timed on.  configs 0-1: the workload itself.  configs 2-4 (fp64 A_hat alone is 35-58 GB and
    forming S takes minutes on the host): SAMPLE_PLANS seeded plans on every SAMPLE_ROW_STRIDE-th dose point -- the same matrix
    structure, classes, masks and n, 1/16 of the rows."""
    from workloads import Workload, pack_mask
    if w.N * w.n <= 2e8:
        return w, "all %d plans, all rows" % w.B, 1.0
    rng = np.random.default_rng(2509)
    plans = np.sort(rng.permutation(w.B)[:SAMPLE_PLANS])
    rows = np.arange(0, w.N, SAMPLE_ROW_STRIDE)
    ws = w.subset(plans)
    mask = None if ws.row_mask is None else pack_mask(ws.mask_bool()[:, rows])
    s = Workload(name=w.name + " sample", config=w.config, phi=np.ascontiguousarray(w.phi[rows]), point_class=w.point_class[rows],
                 classes=w.classes, weights=ws.weights, row_mask=mask, alpha=ws.alpha, beta=ws.beta)
    scale = flops_per_plan_iteration(s.N, s.n) / flops_per_plan_iteration(w.N, w.n)
    return s, (f"{SAMPLE_PLANS} seeded plans on every {SAMPLE_ROW_STRIDE}th dose point (N={s.N}, n={s.n}); rate scaled to the full "
               f"workload by the flops of a plan-iteration (x {scale:.4f}: EXTRAPOLATED)"), scale


class OracleTimer:
    """Times oracle.admm.admm_run as it stands (fp64 numpy/scipy, BLAS threads = host cores) on the sample, setup excluded."""

    def __init__(self, w):
        from oracle import admm as oracle_admm
        from workloads import scaled_rho
        try:
            from threadpoolctl import threadpool_info
            self.cores = int(max([i.get("num_threads", 1) for i in threadpool_info()] or [1]))
        except Exception:
            self.cores = os.cpu_count() or 1
        self.admm = oracle_admm
        self.s, self.desc, self.scale = sample_workload(w)
        self.rho = scaled_rho(self.s.beta, self.s.point_class)
        t0 = time.perf_counter()
        self.pre = oracle_admm.precondition(self.s.phi, self.s.point_class, self.s.classes)
        masks = None if self.s.row_mask is None else self.s.mask_bool()
        self.u_hat, self.b_hat = oracle_admm.plan_bounds(self.pre, self.s.point_class, self.s.classes, self.s.weights, masks)
        self.setup_s = time.perf_counter() - t0
        st = oracle_admm.admm_run(self.pre, self.u_hat, self.b_hat, self.rho, 1)            # warm-up iteration
        self.st0 = (st["z1"], st["y1"], st["z2"], st["y2"])

    def run(self, iters: int) -> float:
        """seconds for `iters` iterations of all sample plans"""
        t0 = time.perf_counter()
        self.admm.admm_run(self.pre, self.u_hat, self.b_hat, self.rho, iters, state0=self.st0)
        return time.perf_counter() - t0

    def rate(self, iters: int, seconds: float) -> float:
        """plan-iterations/s of the FULL workload implied by the sample"""
        return self.s.B * iters / seconds * self.scale


def run_reference(args) -> None:
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from workloads import make_workload
    w = make_workload(args.config)
    ot = OracleTimer(w)
    its = args.ref_iters
    for _ in range(max(args.warmup, 0)):
        ot.run(its)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        ot.run(its)
    dt = time.perf_counter() - t0
    value = ot.rate(its * args.steps, dt)
    sample = (f"{its} ADMM iterations per step of the fp64 numpy oracle on {ot.desc}; oracle setup ({ot.setup_s:.1f} s) excluded")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": _workload_desc(w, args.config)},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": ot.cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------ the CUDA path
def _summary(out, w, seconds, max_iter=MAX_ITER):
    """what one solve did: who converged, who was settled by the presolve, who hit the cap"""
    it = np.asarray(out["iters"].cpu() if hasattr(out["iters"], "cpu") else out["iters"])
    res = np.asarray(out["res"].cpu() if hasattr(out["res"], "cpu") else out["res"])
    capped = it >= max_iter
    d = {"seconds": seconds, "plans_total": int(w.B), "plans_presolved": int((it == 0).sum()),
         "plans_converged": int((~capped).sum()), "plans_capped": int(capped.sum()),
         "plans_capped_with_beta_0": int((capped & (w.beta == 0)).sum()),
         "plan_iterations": int(it.sum()), "max_iterations_of_a_converged_plan": int(it[~capped].max()) if (~capped).any() else 0,
         "max_abs_residual_norm": float(res.max()) if res.size else None,
         # a time TO CONVERGE exists only if every plan converged; otherwise the solve stopped at the cap
         "time_to_converge_s": seconds if not capped.any() else None,
         "time_to_stop_s": seconds}
    return d


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs index (3 = the bench workload; 2 rides along)")
    ap.add_argument("--ref-iters", type=int, default=10, help="oracle iterations per step for --impl reference / cpu_baseline")
    ap.add_argument("--storage", default="fp32", choices=["fp32", "tf32", "bf16"],
                    help="how Phi is stored / consumed for the headline; fp32 = 3xTF32, the 1e-4 path")
    ap.add_argument("--max-iter", type=int, default=MAX_ITER, help="iteration cap of a solve (3000 = the paper's count; smaller for ncu captures)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip config 2, the bf16-storage figures and the full-batch run")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    args.warmup = max(args.warmup, 3)
    max_iter = args.max_iter

    import torch
    import torch.distributed as dist
    from paper_2509_08602_b200 import binding as b          # fails loudly if the CUDA library is missing
    from workloads import make_workload, scaled_rho, with_plans_of

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl ours needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    t_start = time.perf_counter()

    w = make_workload(args.config)
    gen_s = time.perf_counter() - t_start
    # weak scaling: rank r solves its own B plans, the slider grid shifted inside [0,1]^2
    weights = rank_weights(w.weights, rank, world)
    rho = scaled_rho(weights[:, 2], w.point_class)
    stream = torch.cuda.current_stream().cuda_stream
    storages = {"fp32": b.ADMM_STORAGE_FP32_3XTF32, "tf32": b.ADMM_STORAGE_FP32_TF32, "bf16": b.ADMM_STORAGE_BF16}
    eb = {"fp32": 4.0, "tf32": 4.0, "bf16": 2.0}
    peaks = _peaks()
    N, n, B = w.N, w.n, w.B

    phi_pinned = torch.from_numpy(w.phi).pin_memory()
    h = b.admm_setup(phi_pinned, w.point_class, w.classes, device=local_rank, stream=stream, storage=storages[args.storage])
    setup_t = b.admm_get_timing(h)
    mask_dev = None if w.row_mask is None else torch.from_numpy(w.row_mask.view(np.int32)).to(dev)

    def outs_for(nb):
        return dict(t=torch.empty((nb, n), dtype=torch.float32, device=dev), obj=torch.empty(nb, dtype=torch.float64, device=dev),
                    res=torch.empty((nb, 2), dtype=torch.float32, device=dev), iters=torch.empty(nb, dtype=torch.int32, device=dev))
    outs = outs_for(B)

    def step():
        b.admm_solve_batch(h, weights, rho, mask_dev, tol=TOL, max_iter=max_iter, out=outs)
        return b.admm_get_timing(h)["plan_iters"], b.admm_last_launch_count(h)

    for _ in range(args.warmup):
        step()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local_rank)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    plan_iters = launches = 0
    for _ in range(args.steps):
        pi, lc = step()
        plan_iters += pi; launches += lc
    e1.record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    headline = _summary(outs, w, ms / args.steps / 1e3, max_iter)
    (ms,), (plan_iters, launches) = reduce_max_sum(dist if world > 1 else None, dev, [ms], [plan_iters, launches])
    plan_iters, launches = int(plan_iters), int(launches)
    value = plan_iters / (ms / 1e3)

    # ---- e2e: the same metric through the C ABI from HOST buffers (pinned Phi in, host results out), setup included
    e2e = None
    if not args.no_e2e:
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        h2 = b.admm_setup(phi_pinned, w.point_class, w.classes, device=local_rank, stream=stream, storage=storages[args.storage])
        b.admm_solve_batch(h2, weights, rho, w.row_mask, tol=TOL, max_iter=max_iter)
        pi2 = b.admm_get_timing(h2)["plan_iters"]
        h2.close()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        (dt,), (pi2,) = reduce_max_sum(dist if world > 1 else None, dev, [dt], [pi2])
        h2d = N * n * 4 + N + weights.size * 4 + rho.size * 4 + (0 if w.row_mask is None else w.row_mask.nbytes)
        d2h = B * n * 4 + B * 8 + B * 8 + B * 4
        e2e = {"value": pi2 / dt, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "note": "one step = admm_setup (upload of Phi from pinned host memory, S, Cholesky, inverse) + admm_solve_batch, host buffers in/out",
               "seconds_per_step": dt}

    line_extra = {}
    roof = None
    if rank == 0:
        # ---- per-kernel device times: CUDA events on the library's stream around every launch (profile_kernels)
        hp = b.admm_setup(phi_pinned, w.point_class, w.classes, device=local_rank, stream=stream, profile_kernels=True,
                          storage=storages[args.storage])
        live = np.nonzero(outs["iters"].cpu().numpy() > 0)[0]            # the plans the presolve leaves to the iteration
        if live.size == 0:
            live = np.arange(B)
        wl = w.subset(live)
        mask_l = None if wl.row_mask is None else torch.from_numpy(wl.row_mask.view(np.int32)).to(dev)
        K_prof = 40
        ol = outs_for(wl.B)
        b.admm_solve_batch(hp, weights[live], rho[live], mask_l, fixed_iters=5, out=ol)       # warm
        b.admm_solve_batch(hp, weights[live], rho[live], mask_l, fixed_iters=K_prof, out=ol)
        kt = b.admm_get_kernel_times(hp)
        Bl = float(wl.B)
        e = eb[args.storage]
        # algorithmic bytes per launch: the big operand once + the plan operands / state of that kernel;
        # ONE write of the K1 operand G (its hi/lo split is 3xTF32 emulation overhead, not the method's work)
        alg = {"k3_phi_v": e * N * n + 4.0 * n * Bl + 8.0 * N * Bl + 4.0 * N * Bl,        # Phi, V, s1 read + write, G write
               "k1_phiT_g": e * N * n + 4.0 * N * Bl + 4.0 * n * Bl}                      # Phi^T, G, W
        dom = max(("k1_phiT_g", "k3_phi_v"), key=lambda k: kt[k]["total_ms"])
        avg_ms = kt[dom]["total_ms"] / max(kt[dom]["launches"], 1)
        achieved = alg[dom] / (avg_ms * 1e-3) / 1e9
        traffic = None
        tp = os.path.join(ROOT, "profiles", "traffic.json")
        if os.path.exists(tp):
            with open(tp) as f:
                traffic = json.load(f).get(f"config{args.config}_{args.storage}_{dom}")
        roof = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peaks["hbm"], "unit": "GB/s", "frac": achieved / peaks["hbm"],
                "traffic": traffic, "peak_source": peaks["source"], "avg_launch_ms": avg_ms, "algorithmic_bytes_per_launch": alg[dom],
                "plans_in_the_launch": int(wl.B),
                "why_hbm": f"after the presolve {int(wl.B)} of {B} plans iterate: {int(wl.B)} columns per pass are {2 * wl.B / e:.0f} flop per byte of Phi, under the ridge",
                "all_kernels_ms_per_iteration": {k: v["total_ms"] / K_prof for k, v in kt.items()}}
        if not args.no_extras:
            # ---- the full batch, no plan frozen: the tensor-pipe-bound regime (B = 441)
            K_full = 10
            b.admm_solve_batch(hp, weights, rho, mask_dev, fixed_iters=3, out=outs)
            b.admm_solve_batch(hp, weights, rho, mask_dev, fixed_iters=K_full, out=outs)
            kt = b.admm_get_kernel_times(hp)
            it_ms = sum(v["total_ms"] for v in kt.values()) / K_full
            flops = 4.0 * N * n * B + 2.0 * n * n * B
            peak_tc = peaks["bf16"] * (0.5 if args.storage != "bf16" else 1.0)       # tf32 = half the bf16 rate (guide's nominal ratio)
            line_extra["full_batch"] = {
                "plans": B, "ms_per_iteration": it_ms, "plan_iterations_per_s": B / (it_ms / 1e3),
                "kernels_ms_per_iteration": {k: v["total_ms"] / K_full for k, v in kt.items()},
                "roofline": {"bound": "tensor", "achieved": flops / (it_ms * 1e-3) / 1e12, "peak": peak_tc, "unit": "TFLOP/s",
                             "frac": flops / (it_ms * 1e-3) / 1e12 / peak_tc,
                             "note": "algorithmic flops 4NnB + 2n^2B per iteration (3xTF32 emulation passes are overhead, not work) over the "
                                     "whole iteration; peak = sustained bf16 of MEASURED_PEAKS.json x the nominal tf32/bf16 ratio"}}
        hp.close()

        if not args.no_extras and args.config == 3:
            # ---- config 2: the same Phi with the 81 plans of the 9 x 9 grid
            w2 = with_plans_of(w, 2)
            rho2 = scaled_rho(w2.beta, w2.point_class)
            mask2 = torch.from_numpy(w2.row_mask.view(np.int32)).to(dev)
            o2 = outs_for(w2.B)
            times = []
            for i in range(3):
                torch.cuda.synchronize(); t0 = time.perf_counter()
                b.admm_solve_batch(h, w2.weights, rho2, mask2, tol=TOL, max_iter=max_iter, out=o2)
                torch.cuda.synchronize(); times.append(time.perf_counter() - t0)
            c2 = _summary(o2, w2, float(np.median(times[1:])), max_iter)
            c2["workload"] = _workload_desc(w2, 2)
            c2["plan_iterations_per_s"] = c2["plan_iterations"] / c2["seconds"]
            c2["protocol"] = "one untimed warm-up solve, then the median of 2 (PAPER.md:167)"
            line_extra["config2"] = c2
        if not args.no_extras:
            # ---- the plans inside the paper's domain: Eq. (9) has rho -> infinity at w_BOT = 0, and the w_BOT = 0
            # column of the slider grid is where the stragglers are; the same solve without that column, timed on its own
            pos = np.nonzero(weights[:, -1] > 0)[0]
            wp = w.subset(pos)
            maskp = None if wp.row_mask is None else torch.from_numpy(wp.row_mask.view(np.int32)).to(dev)
            op = outs_for(wp.B)
            times = []
            for i in range(2):
                torch.cuda.synchronize(); t0 = time.perf_counter()
                b.admm_solve_batch(h, weights[pos], rho[pos], maskp, tol=TOL, max_iter=max_iter, out=op)
                torch.cuda.synchronize(); times.append(time.perf_counter() - t0)
            cp = _summary(op, wp, times[-1], max_iter)
            cp["plan_iterations_per_s"] = cp["plan_iterations"] / cp["seconds"]
            cp["protocol"] = "one untimed warm-up solve, then one timed solve of the %d plans with w_BOT > 0" % wp.B
            # the same solve with the warm start of deviation D3 (admm_options.warm_start_ratio = 2.5: the plans the presolve
            # rejects narrowly start from their box optimum instead of the zero iterate); the headline keeps the zero start
            hw = b.admm_setup(phi_pinned, w.point_class, w.classes, device=local_rank, stream=stream, storage=storages[args.storage],
                              warm_start_ratio=2.5)
            times = []
            for i in range(2):
                torch.cuda.synchronize(); t0 = time.perf_counter()
                b.admm_solve_batch(hw, weights[pos], rho[pos], maskp, tol=TOL, max_iter=max_iter, out=op)
                torch.cuda.synchronize(); times.append(time.perf_counter() - t0)
            hw.close()
            cw = _summary(op, wp, times[-1], max_iter)
            cw["plan_iterations_per_s"] = cw["plan_iterations"] / cw["seconds"]
            cw["option"] = "warm_start_ratio = 2.5 (DESIGN.md deviation D3)"
            cp["with_warm_start"] = cw
            line_extra["w_bot_positive"] = cp
    h.close()

    if rank == 0 and not args.no_extras and args.storage == "fp32":
        # ---- the same workload with bf16 storage of Phi (half the HBM bytes; 1e-2 iterate budget, objectives certified to 1e-3)
        hb = b.admm_setup(phi_pinned, w.point_class, w.classes, device=local_rank, stream=stream, storage=b.ADMM_STORAGE_BF16,
                          profile_kernels=False)
        times = []
        for i in range(3):
            torch.cuda.synchronize(); t0 = time.perf_counter()
            b.admm_solve_batch(hb, weights, rho, mask_dev, tol=TOL, max_iter=max_iter, out=outs)
            torch.cuda.synchronize(); times.append(time.perf_counter() - t0)
        bf = _summary(outs, w, float(np.median(times[1:])), max_iter)
        bf["plan_iterations_per_s"] = bf["plan_iterations"] / bf["seconds"]
        bf["dtype"] = "bf16 Phi x bf16 hi/lo plan operands, fp32 accumulate; S^-1 apply in f64"
        bf["protocol"] = "one untimed warm-up solve, then the median of 2"
        torch.cuda.synchronize(); t0 = time.perf_counter()
        b.admm_solve_batch(hb, weights, rho, mask_dev, fixed_iters=10, out=outs)
        torch.cuda.synchronize()
        bf["full_batch_ms_per_iteration"] = (time.perf_counter() - t0) / 10 * 1e3
        hb.close()
        # the plans with w_BOT > 0, bf16 storage, warm start (deviation D3): the fastest configuration of the library on this workload
        pos = np.nonzero(weights[:, -1] > 0)[0]
        wp = w.subset(pos)
        maskp = None if wp.row_mask is None else torch.from_numpy(wp.row_mask.view(np.int32)).to(dev)
        op = outs_for(wp.B)
        hbw = b.admm_setup(phi_pinned, w.point_class, w.classes, device=local_rank, stream=stream, storage=b.ADMM_STORAGE_BF16,
                           warm_start_ratio=2.5)
        times = []
        for i in range(2):
            torch.cuda.synchronize(); t0 = time.perf_counter()
            b.admm_solve_batch(hbw, weights[pos], rho[pos], maskp, tol=TOL, max_iter=max_iter, out=op)
            torch.cuda.synchronize(); times.append(time.perf_counter() - t0)
        hbw.close()
        bw = _summary(op, wp, times[-1], max_iter)
        bw["option"] = "bf16 storage, warm_start_ratio = 2.5, the %d plans with w_BOT > 0" % wp.B
        bf["w_bot_positive_with_warm_start"] = bw
        line_extra["bf16_storage"] = bf

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        ot = OracleTimer(w)
        sec = ot.run(args.ref_iters)
        cpu = {"value": ot.rate(args.ref_iters, sec), "unit": UNIT, "cores": ot.cores, "kind": "oracle",
               "sample": f"{args.ref_iters} ADMM iterations of the fp64 numpy oracle in {sec:.1f} s on {ot.desc}; its setup ({ot.setup_s:.1f} s) excluded like the GPU's"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": {"fp32": "f32 (3xTF32 tensor-core products, fp32 accumulate; S^-1 apply and block-2 state in f64)",
                      "tf32": "tf32-rounded Phi x tf32 hi/lo plan operands, fp32 accumulate; S^-1 apply in f64",
                      "bf16": "bf16 Phi x bf16 hi/lo plan operands, fp32 accumulate; S^-1 apply in f64"}[args.storage],
            "data": "synthetic",
            "config": {"workload": _workload_desc(w, args.config), "storage": args.storage, "tol": TOL, "max_iter": max_iter,
                       "plans_per_gpu": B, "presolve": "on (plans whose box optimum is feasible are settled in closed form, 0 iterations)",
                       "l2": "inputs larger than L2: Phi and Phi^T (2 x %.1f GB) are streamed every iteration" % (N * n * eb[args.storage] / 1e9),
                       "parallelism": "plans sharded over ranks, Phi replicated" if world > 1 else "single GPU"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roof, "cpu_baseline": cpu,
            "solve": headline,
            "time_to_converge_s": headline["time_to_converge_s"], "time_to_stop_s": headline["time_to_stop_s"],
            "plans_converged": headline["plans_converged"], "plans_total": headline["plans_total"],
            "setup_ms": {k: setup_t[k] for k in ("upload_ms", "syrk_ms", "factor_ms", "setup_ms")},
            "generation_s": gen_s, "bench_wall_s": time.perf_counter() - t_start,
        }
        line.update(line_extra)
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

"""bench.py -- plan-iterations/s of the batched ADMM hot path (BASELINE.json metric) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C]

A "step" is ONE pass of the whole hot path over one batch of synthetic input: admm_solve_batch of all B
plans of the workload from the zero iterate to convergence (tol 1e-4, cap 3000 iterations = the paper's
fixed count) with per-plan convergence masking + compaction, then the objective evaluation.
Setup (upload, S = I + A A^T, Cholesky, inverse) is done once before the timed region and reported
separately (north_star: "timed separately"); the `e2e` leg times setup + solve from host buffers.

N > 1 (torchrun): weak scaling, plans are independent columns: every rank holds a replica of
Phi and solves its own B plans (a shifted slider grid); no data-path collective; value = all ranks' plan
iterations / max-over-ranks device time.
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


def _workload_desc(w, cfg):
    return f"config{cfg}: N={w.N} points x n={w.n} time variables, B={w.B} plans, dense fp32 Phi {w.N * w.n * 4 / 1e6:.1f} MB"


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                       "-i", str(gpu_index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        time.sleep(0.15)
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


def _oracle_sample(w, rho, iters: int):
    """Times the oracle as it stands on the host cores: `iters` iterations of all plans (setup excluded)."""
    from oracle import admm as oracle_admm
    try:
        from threadpoolctl import threadpool_info
        cores = max([i.get("num_threads", 1) for i in threadpool_info()] or [1])
    except Exception:
        cores = os.cpu_count() or 1
    t0 = time.perf_counter()
    pre = oracle_admm.precondition(w.phi, w.point_class, w.classes)
    masks = None if w.row_mask is None else w.mask_bool()
    u_hat, b_hat = oracle_admm.plan_bounds(pre, w.point_class, w.classes, w.weights, masks)
    t_setup = time.perf_counter() - t0
    state = oracle_admm.admm_run(pre, u_hat, b_hat, rho, 1)            # warm-up iteration
    st0 = (state["z1"], state["y1"], state["z2"], state["y2"])
    t0 = time.perf_counter()
    oracle_admm.admm_run(pre, u_hat, b_hat, rho, iters, state0=st0)
    dt = time.perf_counter() - t0
    return dict(value=w.B * iters / dt, seconds=dt, setup_seconds=t_setup, cores=int(cores), pre=(pre, u_hat, b_hat, st0))


def run_reference(args) -> None:
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import admm as oracle_admm
    from workloads import make_workload, scaled_rho
    w = make_workload(args.config)
    rho = scaled_rho(w.beta, w.point_class)
    its = args.ref_iters
    first = _oracle_sample(w, rho, its)
    pre, u_hat, b_hat, st0 = first["pre"]
    for _ in range(max(args.warmup - 1, 0)):
        oracle_admm.admm_run(pre, u_hat, b_hat, rho, its, state0=st0)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_admm.admm_run(pre, u_hat, b_hat, rho, its, state0=st0)
    dt = time.perf_counter() - t0
    value = w.B * its * args.steps / dt
    sample = f"{its} ADMM iterations of all {w.B} plans per step (fp64 numpy oracle, setup excluded: {first['setup_seconds']:.1f} s)"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": _workload_desc(w, args.config)},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": first["cores"], "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json configs index (1 = the bench workload)")
    ap.add_argument("--ref-iters", type=int, default=40, help="oracle iterations per step for --impl reference / cpu_baseline")
    ap.add_argument("--storage", default="fp32", choices=["fp32", "tf32", "bf16"],
                    help="how Phi is stored / consumed (BASELINE.json config 4 variants); fp32 = 3xTF32, the 1e-4 path")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
        return

    import torch
    import torch.distributed as dist
    from paper_2509_08602_b200 import binding as b          # fails loudly if the CUDA library is missing
    from workloads import make_workload, scaled_rho

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl ours needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    w = make_workload(args.config)
    # weak scaling: rank r solves its own B plans, the slider grid shifted inside [0,1]^2
    weights = rank_weights(w.weights, rank, world)
    rho = scaled_rho(weights[:, 2], w.point_class)
    stream = torch.cuda.current_stream().cuda_stream

    phi_pinned = torch.from_numpy(w.phi).pin_memory()
    storage = {"fp32": b.ADMM_STORAGE_FP32_3XTF32, "tf32": b.ADMM_STORAGE_FP32_TF32, "bf16": b.ADMM_STORAGE_BF16}[args.storage]
    elem_bytes = 2 if args.storage == "bf16" else 4
    h = b.admm_setup(phi_pinned, w.point_class, w.classes, device=local_rank, stream=stream, storage=storage)
    setup_t = b.admm_get_timing(h)
    mask_dev = None if w.row_mask is None else torch.from_numpy(w.row_mask.view(np.int32)).to(dev)
    outs = dict(t=torch.empty((w.B, w.n), dtype=torch.float32, device=dev),
                obj=torch.empty(w.B, dtype=torch.float64, device=dev),
                res=torch.empty((w.B, 2), dtype=torch.float32, device=dev),
                iters=torch.empty(w.B, dtype=torch.int32, device=dev))

    def step():
        b.admm_solve_batch(h, weights, rho, mask_dev, tol=TOL, max_iter=MAX_ITER, out=outs)
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
    iters_np = outs["iters"].cpu().numpy()
    res_np = outs["res"].cpu().numpy()
    n_conv = int((iters_np < MAX_ITER).sum())
    (ms,), (plan_iters, launches) = reduce_max_sum(dist if world > 1 else None, dev, [ms], [plan_iters, launches])
    plan_iters, launches = int(plan_iters), int(launches)
    value = plan_iters / (ms / 1e3)

    # ---- e2e: the same metric through the C ABI from HOST buffers (pinned Phi in, host results out), setup included
    e2e = None
    if not args.no_e2e:
        n_e2e = 2
        host_out = None
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        pi2 = 0
        for _ in range(n_e2e):
            h2 = b.admm_setup(phi_pinned, w.point_class, w.classes, device=local_rank, stream=stream, storage=storage)
            host_out = b.admm_solve_batch(h2, weights, rho, w.row_mask, tol=TOL, max_iter=MAX_ITER)
            pi2 += b.admm_get_timing(h2)["plan_iters"]
            h2.close()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        (dt,), (pi2,) = reduce_max_sum(dist if world > 1 else None, dev, [dt], [pi2])
        h2d = w.N * w.n * 4 + w.N + weights.size * 4 + rho.size * 4 + (0 if w.row_mask is None else w.row_mask.nbytes)
        d2h = w.B * w.n * 4 + w.B * 8 + w.B * 8 + w.B * 4
        e2e = {"value": pi2 / dt, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "note": "admm_setup (upload, S, Cholesky, inverse) + admm_solve_batch per step, host buffers in/out",
               "seconds_per_step": dt / n_e2e}

    # ---- roofline of the dominant kernel: CUDA events around every launch of a fixed-iteration solve
    roof = None
    if rank == 0:
        hp = b.admm_setup(phi_pinned, w.point_class, w.classes, device=local_rank, stream=stream, profile_kernels=True, storage=storage)
        K_prof = 100
        b.admm_solve_batch(hp, weights, rho, mask_dev, fixed_iters=K_prof, out=outs)     # warm
        b.admm_solve_batch(hp, weights, rho, mask_dev, fixed_iters=K_prof, out=outs)
        kt = b.admm_get_kernel_times(hp)
        hp.close()
        N, n, B = w.N, w.n, w.B
        # algorithmic bytes per launch: Phi once + state / operand traffic of that kernel
        eb = float(elem_bytes)
        alg = {"k3_phi_v": eb * N * n + 2 * eb * n * B + 8.0 * N * B + 2 * eb * N * B,   # Phi, V hi/lo, s1 r+w, G hi+lo w
               "k1_phiT_g": eb * N * n + 2 * eb * N * B + 4.0 * n * B}                   # Phi^T, G hi/lo, W
        dom = max(("k1_phiT_g", "k3_phi_v"), key=lambda k: kt[k]["total_ms"])
        avg_ms = kt[dom]["total_ms"] / max(kt[dom]["launches"], 1)
        peak, which = _peaks()
        achieved = alg[dom] / (avg_ms * 1e-3) / 1e9
        traffic = None
        tp = os.path.join(ROOT, "profiles", "traffic.json")
        if os.path.exists(tp):
            with open(tp) as f:
                traffic = json.load(f).get(dom)
        roof = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "peak_source": which, "avg_launch_ms": avg_ms, "algorithmic_bytes_per_launch": alg[dom],
                "all_kernels_ms_per_iteration": {k: v["total_ms"] / K_prof for k, v in kt.items()}}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        s = _oracle_sample(w, scaled_rho(w.beta, w.point_class), args.ref_iters)
        cpu = {"value": s["value"], "unit": UNIT, "cores": s["cores"], "kind": "oracle",
               "sample": f"{args.ref_iters} ADMM iterations of all {w.B} plans of the same workload in {s['seconds']:.1f} s "
                         f"(fp64 numpy oracle; its setup, {s['setup_seconds']:.1f} s, excluded like the GPU's)"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": {"fp32": "f32 (3xTF32 tensor-core products, fp32 accumulate; S^-1 apply and block-2 state in f64)",
                      "tf32": "tf32-rounded Phi x tf32 hi/lo plan operands, fp32 accumulate; S^-1 apply in f64",
                      "bf16": "bf16 Phi x bf16 hi/lo plan operands, fp32 accumulate; S^-1 apply in f64"}[args.storage],
            "data": "synthetic",
            "config": {"workload": _workload_desc(w, args.config), "storage": args.storage, "tol": TOL, "max_iter": MAX_ITER,
                       "plans_per_gpu": w.B, "l2": "inputs larger than L2: Phi and Phi^T (2 x %.0f MB) are streamed every iteration" % (w.N * w.n * 4 / 1e6),
                       "parallelism": "plans sharded over ranks, Phi replicated" if world > 1 else "single GPU"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roof, "cpu_baseline": cpu,
            "time_to_converge_s": ms / args.steps / 1e3, "plans_converged": n_conv, "plans_total": int(w.B),
            "max_abs_residual_norm": float(np.max(res_np)) if res_np.size else None,
            "setup_ms": {k: setup_t[k] for k in ("upload_ms", "syrk_ms", "factor_ms", "setup_ms")},
        }
        print(json.dumps(line))
    h.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

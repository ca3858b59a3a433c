#!/usr/bin/env python
"""bench.py — fGMRES + geometric-multigrid solve throughput on synthetic planes (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C]

A "step" is one pass of the whole hot path on one plane: mg_update_coeffs (coefficient restriction to
all levels + coarsest factorisation) followed by mg_solve (fGMRES(30) + V(2,2) to rtol 1e-10).
metric = unknown*iters/s = (mesh points x fGMRES iterations) / time, whole job over all ranks.
N > 1: one process per GPU (torchrun), every rank solves its own plane (planes are independent,
PAPER.md:211, 322-324): weak scaling, no data-path collective.
--impl reference times the CPU oracle (oracle/) on the host cores on a bounded sample.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2509_11831_b200 import workloads as W  # noqa: E402

METRIC = "fgmres_mg_solve_unknown_iters_per_s"
UNIT = "unknown*iters/s"
RTOL = 1e-10
WORKLOADS = {
    1: "configs[0]: unit square 65x65, 4 levels",
    2: "configs[1]: annulus 513x513 (~190k unknowns), 7 levels",
    3: "configs[2]: D-shape with X-point 1025x1025 (~700k unknowns), 8 levels",
    4: "configs[3]: D-shape with X-point 4097x4097 (~11M unknowns), 10 levels",
    5: "configs[4]: D-shape 2049x2049 (~2.8M unknowns), 9 levels, time stepping",
}
# algorithmic bytes per point (SURVEY.md 8(d) / DESIGN.md section 6): one full RB-B GS sweep
GS_BYTES_PER_POINT = 64.0


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush(); self.f.seek(0)
        sm, mx, reasons = [], [], set()
        for line in self.f.read().splitlines():
            t = [v.strip() for v in line.split(",")]
            if len(t) < 6:
                continue
            try:
                sm.append(float(t[0])); mx.append(float(t[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), t[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out = {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons)}
        return out


def oracle_sample(pl, max_iters):
    """The oracle as it stands, 1 thread, on the same plane, capped at max_iters iterations."""
    from oracle import oracle as om
    o = om.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels, max_iters=max_iters)
    t0 = time.perf_counter()
    o.update(pl.lam, pl.c)
    r = o.solve(pl.f, pl.x0, RTOL)
    dt = time.perf_counter() - t0
    return dt, r["iters"], o


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    pl = W.make_plane(args.config)
    cap = args.ref_iters
    from oracle import oracle as om
    o = om.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels, max_iters=cap)
    times, iters = [], 0
    for k in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        o.update(pl.lam, pl.c)
        r = o.solve(pl.f, pl.x0, RTOL)
        dt = time.perf_counter() - t0
        iters = r["iters"]
        if k >= args.warmup:
            times.append(dt)
    total = sum(times)
    value = pl.n * iters * len(times) / total
    sample = f"update + first {iters} fGMRES iterations (max_iters={cap}) of the same plane per step, 1 thread"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOADS[args.config], "unknowns": pl.n, "rtol": RTOL, "cycle": "V(2,2)", "restart_m": 30},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2509_11831_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.use_torch_allocator()

    # every rank owns one plane of the same geometry with its own seed (planes are independent)
    pl = W.make_plane(args.config, seed=W.SEEDS[args.config] + 7919 * rank)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    s = B.Solver(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
    d_lam, d_c, d_f, d_x0 = dev(pl.lam), dev(pl.c), dev(pl.f), dev(pl.x0)
    d_x = torch.empty_like(d_f)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
    h_lam, h_c, h_f, h_x0 = pin(pl.lam), pin(pl.c), pin(pl.f), pin(pl.x0)
    h_x = torch.empty(pl.n, dtype=torch.float64).pin_memory().numpy()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step_device():
        s.update_coeffs(d_lam, d_c)
        _, iters, relres, rc = s.solve(d_f, d_x0, RTOL, x=d_x)
        return iters, relres, rc

    def step_host():
        s.update_coeffs_host(h_lam, h_c)
        _, iters, relres, rc = s.solve_host(h_f, h_x0, RTOL, x=h_x)
        return iters, relres, rc

    def timed(step, steps):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        l0 = s.kernel_launches
        ev0.record()
        out = None
        for _ in range(steps):
            out = step()
        ev1.record()
        barrier()
        ms = torch.tensor([ev0.elapsed_time(ev1)], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(ms, op=dist.ReduceOp.MAX)
        return float(ms.item()), out, s.kernel_launches - l0

    for _ in range(args.warmup):
        step_device()
    sampler = ClockSampler(local) if rank == 0 else None
    ms, (iters, relres, rc), launches = timed(step_device, args.steps)
    solve_ms, update_ms = s.last_solve_ms, s.last_update_ms
    clocks = sampler.stop() if sampler else None
    step_host()
    ms_e2e, (it_e, rr_e, rc_e), _ = timed(step_host, args.steps)

    # whole-job unknown*iters (every rank may take a different number of iterations)
    work = torch.tensor([float(pl.n) * iters, float(pl.n), float(iters)], dtype=torch.float64, device="cuda")
    work_e = torch.tensor([float(pl.n) * it_e], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(work); dist.all_reduce(work_e)
    value = float(work[0].item()) * args.steps / (ms * 1e-3)
    value_e2e = float(work_e[0].item()) * args.steps / (ms_e2e * 1e-3)

    # ---- roofline of the dominant kernel: one RB-B Gauss-Seidel sweep on the finest level, timed live
    peak, peak_src = peaks()
    roof = None
    if rank == 0:
        n0 = s.level_n(0)
        xs, bs = torch.randn(n0, dtype=torch.float64, device="cuda"), torch.randn(n0, dtype=torch.float64, device="cuda")
        def t_smooth(k, reps=5):
            best = 1e30
            for _ in range(reps):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize(); e0.record(); s.smooth(0, xs, bs, k); e1.record(); torch.cuda.synchronize()
                best = min(best, e0.elapsed_time(e1))
            return best
        t_smooth(1, 2)
        sweeps = 10
        per_sweep_ms = (t_smooth(sweeps) - t_smooth(0)) / sweeps
        achieved = GS_BYTES_PER_POINT * n0 / (per_sweep_ms * 1e-3) / 1e9
        roof = {"bound": "hbm", "kernel": "gs_sweep level 0 (red + black + guard groups)", "achieved": achieved, "peak": peak,
                "peak_source": peak_src, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                "algorithmic_bytes_per_launch": GS_BYTES_PER_POINT * n0, "ms_per_launch": per_sweep_ms}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        dt, it_o, _ = oracle_sample(pl, args.ref_iters)
        cpu = {"value": pl.n * it_o / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"update + first {it_o} fGMRES iterations of the same plane, 1 thread, {dt:.1f} s"}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": WORKLOADS[args.config], "unknowns_per_plane": pl.n, "planes": world, "rtol": RTOL,
                           "cycle": "V(2,2) RB-B GS", "restart_m": 30, "levels": s.levels,
                           "l2_policy": "inputs larger than L2 (no flush)" if pl.n * 8 * 8 > 126e6 else "working set fits L2 (small config)"},
                "iters": iters, "final_relres": relres, "status": rc, "solve_ms": solve_ms, "update_ms": update_ms,
                "clocks": clocks, "gpu_launches": launches,
                "e2e": {"value": value_e2e, "unit": UNIT, "h2d_bytes_per_step": 4 * pl.n * 8, "d2h_bytes_per_step": pl.n * 8,
                        "ms_per_step": ms_e2e / args.steps, "iters": it_e},
                "roofline": roof, "cpu_baseline": cpu}
        print(json.dumps(line))
    s.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--ref-iters", type=int, default=2, help="iteration cap of the oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

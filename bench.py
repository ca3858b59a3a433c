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
# Roofline kernel: the fused launch "two RB-B Gauss-Seidel sweeps + defect + full-weighting restriction" on level 0.
# Algorithmic bytes per point of THAT launch: every array the operation needs, moved exactly once:
# x in 8 + c 8 + b 8 + 1/a_ll 8 + lambda 8 + x out 8 + point code 2 + restricted defect 8/4 = 52 B.  The three-loop
# formulation of SURVEY.md 8(d) (2 x 64 B/pt for two sweeps + 61 B/pt for defect + restriction = 189 B/pt) is reported
# beside it as what the fusion avoids; it is not a statement about HBM.
ROOF_BYTES_PER_POINT = 52.0
UNFUSED_BYTES_PER_POINT = 2 * 64.0 + 61.0
# DRAM bytes per launch of the roofline kernel (dram__bytes_read.sum + dram__bytes_write.sum of one `ncu --set full`
# capture per config), kept in profiles/roofline_traffic.json with the command and the date of the capture


def roofline_traffic(cfg):
    p = os.path.join(ROOT, "profiles", "roofline_traffic.json")
    try:
        e = json.load(open(p))["configs"].get(str(cfg))
        return (float(e["dram_bytes_per_launch"]), e.get("capture")) if e else (None, None)
    except (OSError, KeyError, ValueError):
        return None, None


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


def oracle_sample(pl, max_iters, xi=None):
    """The oracle as it stands, 1 thread, on the same plane, capped at max_iters iterations."""
    from oracle import oracle as om
    o = om.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels, max_iters=max_iters)
    t0 = time.perf_counter()
    if xi is None:
        o.update(pl.lam, pl.c)
    else:
        o.update3(pl.lam, xi, pl.c)
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
            "config": {"workload": WORKLOADS[args.config], "unknowns_per_plane": pl.n, "planes": 1, "rtol": RTOL,
                       "cycle": "V(2,2) RB-B GS", "restart_m": 30, "levels": pl.levels, "step": "mg_update_coeffs + mg_solve (oracle, bounded sample)"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def spawn_command(gpus, argv, port=None):
    """`python bench.py --gpus N` without a launcher: the torchrun command that starts one rank per GPU (what the driver
    runs itself for N > 1)."""
    if port is None:
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={gpus}", "--master-addr", "127.0.0.1",
            "--master-port", str(port), os.path.abspath(__file__)] + list(argv)


def respawn(args, argv):
    """--gpus N > 1 outside a launcher (no WORLD_SIZE in the environment): re-exec under torchrun so that N ranks exist."""
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        cmd = spawn_command(args.gpus, argv)
        os.execv(cmd[0], cmd)


def run_dry(args):
    """MG_BENCH_DRY=1: the multi-rank plumbing without a GPU (gloo, CPU): every rank owns its plane's inputs, the two
    reductions of whole_job run, rank 0 prints the line.  Used by tests/test_bench_sharding.py."""
    import torch.distributed as dist
    world, rank = int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0"))
    if world > 1:
        dist.init_process_group("gloo")
    pl = W.make_plane(args.config, 65, seed=plane_seed(args.config, rank))
    ms, work, value = whole_job(10.0 * (rank + 1), float(pl.n) * 7, world, "cpu")
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                          "ms_per_step": ms / max(args.steps, 1), "scaling": "weak", "data": "dry run (no GPU work)", "dry": True}))
    if world > 1:
        dist.destroy_process_group()


def plane_seed(cfg, rank):
    """Every rank owns its own plane of the same geometry (planes are independent solves)."""
    return W.SEEDS[cfg] + 7919 * rank


def whole_job(ms_local, unknown_iters_local, world, device):
    """Max-over-ranks time and summed work: value = all units processed by all ranks / slowest rank's time.
    No data-path collective exists; these two reductions are the only communication of the bench."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    w = torch.tensor([unknown_iters_local], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(w, op=dist.ReduceOp.SUM)
    ms, work = float(t.item()), float(w.item())
    return ms, work, work / (ms * 1e-3)


def make_steps(cfg, rank, nsteps, lattice=None):
    """Inputs of `nsteps` consecutive steps.  Configs 1-4: the same plane every step (x0 = 0).
    Config 5: the time-stepping sequence of BASELINE.json configs[4] (coefficients and right-hand side
    perturbed every step, warm start from the previous solution)."""
    pl = W.make_plane(cfg, lattice, seed=plane_seed(cfg, rank))
    if cfg != 5:
        return pl, [pl] * nsteps, False
    seq, cur = [pl], pl
    for k in range(nsteps - 1):
        cur = W.next_step(cur, k)
        seq.append(cur)
    return pl, seq, True


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

    nsteps = args.warmup + args.steps
    pl, seq, warm = make_steps(args.config, rank, nsteps, args.lattice)
    uniq = seq if warm else seq[:1]
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    s = B.Solver(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels, full_cgs2=args.full_cgs2, solver=args.solver)
    d_in = [(dev(q.lam), dev(q.c), dev(q.f)) for q in uniq]          # resident in HBM before the timed region
    h_in = [(pin(q.lam).numpy(), pin(q.c).numpy(), pin(q.f).numpy()) for q in uniq]
    # --three-field: the paper's lambda phi - xi div(c grad phi) = rho (Eq. 3) with a seeded xi, the same every step
    xi = W.xi_field(pl) if args.three_field else None
    d_xi, h_xi = (dev(xi), pin(xi).numpy()) if args.three_field else (None, None)
    d_x0, d_x = dev(pl.x0), torch.empty(pl.n, dtype=torch.float64, device="cuda")
    h_x0, h_x = pin(pl.x0).numpy(), torch.empty(pl.n, dtype=torch.float64).pin_memory().numpy()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step_device(k):
        lam, c, f = d_in[k if warm else 0]
        s.update_coeffs3(lam, d_xi, c)
        _, iters, relres, rc = s.solve(f, d_x if (warm and k > 0) else d_x0, args.rtol, x=d_x)   # d_x may alias d_x0
        return iters, relres, rc

    def step_host(k):
        lam, c, f = h_in[k if warm else 0]
        if h_xi is None:
            s.update_coeffs_host(lam, c)
        else:
            s.update_coeffs3_host(lam, h_xi, c)
        _, iters, relres, rc = s.solve_host(f, h_x if (warm and k > 0) else h_x0, args.rtol, x=h_x)
        return iters, relres, rc

    def timed(step, first, steps):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        l0 = s.kernel_launches
        ev0.record()
        outs, solve_ms, update_ms = [], [], []
        for k in range(first, first + steps):
            outs.append(step(k))
            solve_ms.append(s.last_solve_ms); update_ms.append(s.last_update_ms)
        ev1.record()
        barrier()
        return ev0.elapsed_time(ev1), outs, s.kernel_launches - l0, solve_ms, update_ms

    if args.roofline_only:                 # profiling aid: only the roofline kernel (after one update), nothing timed
        s.update_coeffs3(d_in[0][0], d_xi, d_in[0][1])
        n0 = s.level_n(0)
        xs, bs = torch.randn(n0, dtype=torch.float64, device="cuda"), torch.randn(n0, dtype=torch.float64, device="cuda")
        for _ in range(4):
            s.smooth_restrict(0, xs, bs, 2)
        torch.cuda.synchronize()
        s.close()
        return
    for k in range(args.warmup):
        step_device(k)
    sampler = ClockSampler(local) if rank == 0 else None
    ms_loc, outs, launches, solve_ms, update_ms = timed(step_device, args.warmup, args.steps)
    clocks = sampler.stop() if sampler else None
    iters_all = [o[0] for o in outs]
    ms, work, value = whole_job(ms_loc, float(pl.n) * sum(iters_all), world, "cuda")
    reorth = s.last_reorth
    for k in range(args.warmup):
        step_host(k)
    ms_e_loc, outs_e, _, _, _ = timed(step_host, args.warmup, args.steps)
    ms_e2e, _, value_e2e = whole_job(ms_e_loc, float(pl.n) * sum(o[0] for o in outs_e), world, "cuda")

    # ---- roofline of the dominant kernel (profiles/r01e_launches_config4.md): k_gs<2,false,true> on level 0, i.e.
    # two fused red-black-boundary Gauss-Seidel sweeps + defect + full-weighting restriction in one launch.
    # Timed live: CUDA events on the launching stream around exactly that launch (mg_last_step_ms).
    peak, peak_src = peaks()
    roof = None
    if rank == 0:
        n0 = s.level_n(0)
        xs, bs = torch.randn(n0, dtype=torch.float64, device="cuda"), torch.randn(n0, dtype=torch.float64, device="cuda")
        t = []
        for _ in range(12):
            s.smooth_restrict(0, xs, bs, 2)
            t.append(s.last_step_ms)
        per_launch_ms = float(np.median(t[2:]))
        alg = ROOF_BYTES_PER_POINT * n0
        achieved = alg / (per_launch_ms * 1e-3) / 1e9
        traffic, capture = roofline_traffic(args.config) if (args.lattice is None and not args.three_field) else (None, None)
        roof = {"bound": "hbm", "kernel": "k_gs_strip<6,8,0,1> (+ k_gs on overflow tiles) level 0: two fused RB-B Gauss-Seidel sweeps + defect + FW restriction per launch",
                "achieved": achieved, "peak": peak, "peak_source": peak_src, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
                "algorithmic_bytes_per_launch": alg, "ms_per_launch": per_launch_ms,
                "note": "algorithmic bytes = 52 B/pt: every array of the fused launch moved once (DESIGN.md section 6); the kernel is bound by "
                        "shared-memory / issue latency, not by HBM",
                "unfused_formulation": {"bytes_per_launch": UNFUSED_BYTES_PER_POINT * n0,
                                        "speedup_over_its_roofline": UNFUSED_BYTES_PER_POINT * n0 / (per_launch_ms * 1e-3) / 1e9 / peak}}
        if traffic:
            roof["traffic_capture"] = capture
            roof["frac_of_traffic"] = traffic / (per_launch_ms * 1e-3) / 1e9 / peak

    cpu = cpu_all = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        dt, it_o, _ = oracle_sample(pl, args.ref_iters, xi)
        cpu = {"value": pl.n * it_o / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"update + first {it_o} fGMRES iterations of the same plane, 1 thread, {dt:.1f} s"}
        # second, separately labelled line: the same source built with -fopenmp, grid loops on all host cores (the
        # analogue of the paper's OpenMP backend); a timing line only (reductions sum in another order)
        from oracle import oracle as om
        try:
            om.use_openmp(True)
            dt2, it2, _ = oracle_sample(pl, args.ref_iters, xi)
            cpu_all = {"value": pl.n * it2 / dt2, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle, same source compiled with -fopenmp",
                       "sample": f"update + first {it2} fGMRES iterations of the same plane, {os.cpu_count()} threads, {dt2:.1f} s"}
        except Exception as e:                            # no OpenMP runtime on the box: say so, keep the line
            cpu_all = {"unavailable": str(e)[:200]}
        finally:
            om.use_openmp(False)

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": WORKLOADS[args.config] + (f" [geometry on a {args.lattice}^2 lattice]" if args.lattice else ""),
                           "unknowns_per_plane": pl.n, "planes": world, "rtol": args.rtol,
                           "cycle": "V(2,2) RB-B GS", "restart_m": 30, "levels": s.levels, "solver": args.solver,
                           "form": "three-field (lambda, xi, c), PAPER.md Eq. 3" if args.three_field else "two-field (lambda, c), xi = 1",
                           "step": ("mg_update_coeffs3" if args.three_field else "mg_update_coeffs") + " + mg_solve" + (" (time stepping: new coefficients and rhs, warm start)" if warm else ""),
                           "l2_policy": "inputs larger than L2 (no flush)" if pl.n * 8 * 8 > 126e6 else "working set fits L2 (small config)"},
                "iters": iters_all[-1], "iters_per_step": iters_all, "final_relres": outs[-1][1], "status": outs[-1][2],
                "second_gs_updates": reorth,      # Arnoldi steps of the last solve whose second update ran (G23)
                "solve_ms": float(np.median(solve_ms)), "update_ms": float(np.median(update_ms)),
                "solve_ms_per_plane": float(np.median(solve_ms)),
                "clocks": clocks, "gpu_launches": launches,
                "e2e": {"value": value_e2e, "unit": UNIT, "h2d_bytes_per_step": (5 if args.three_field else 4) * pl.n * 8, "d2h_bytes_per_step": pl.n * 8,
                        "ms_per_step": ms_e2e / args.steps, "iters": outs_e[-1][0]},
                "roofline": roof, "cpu_baseline": cpu, "cpu_baseline_allcores": cpu_all}
        print(json.dumps(line))
    s.close()
    if world > 1:
        dist.destroy_process_group()


def run_planes(args):
    """several planes per GPU solved concurrently — one handle, one stream and one host thread per
    plane (16 independent poloidal planes per time step).  Production planes have 1e5-2e6 points
    (PAPER.md:256): alone they leave most of a B200 idle (latency bound), together they fill it.  Secondary bench line:
    HBM-resident inputs only."""
    import threading
    import torch
    import torch.distributed as dist
    from paper_2509_11831_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.use_torch_allocator()
    P = args.planes
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    streams = [torch.cuda.Stream() for _ in range(P)]
    planes = [W.make_plane(args.config, seed=plane_seed(args.config, rank * P + p)) for p in range(P)]
    solvers, data = [], []
    for p, pl in enumerate(planes):
        with torch.cuda.stream(streams[p]):
            solvers.append(B.Solver(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels, stream=streams[p]))
            data.append((dev(pl.lam), dev(pl.c), dev(pl.f), dev(pl.x0), torch.empty(pl.n, dtype=torch.float64, device="cuda")))
    torch.cuda.synchronize()
    iters = [[] for _ in range(P)]

    def work(p, steps, keep):
        lam, c, f, x0, x = data[p]
        torch.cuda.set_device(local)
        for _ in range(steps):
            solvers[p].update_coeffs(lam, c, stream=streams[p])
            _, it, rr, rc = solvers[p].solve(f, x0, RTOL, x=x, stream=streams[p])
            if keep:
                iters[p].append(it)

    def round_(steps, keep):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        ev0.record()
        for st in streams:
            st.wait_event(ev0)
        th = [threading.Thread(target=work, args=(p, steps, keep)) for p in range(P)]
        [t.start() for t in th]
        [t.join() for t in th]
        for st in streams:
            torch.cuda.current_stream().wait_stream(st)
        ev1.record()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        return ev0.elapsed_time(ev1)

    l0 = sum(s.kernel_launches for s in solvers)
    round_(args.warmup, False)
    l1 = sum(s.kernel_launches for s in solvers)
    sampler = ClockSampler(local) if rank == 0 else None
    ms_loc = round_(args.steps, True)
    clocks = sampler.stop() if sampler else None
    work_loc = float(sum(pl.n * sum(iters[p]) for p, pl in enumerate(planes)))
    ms, work, value = whole_job(ms_loc, work_loc, world, "cuda")
    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": WORKLOADS[args.config], "unknowns_per_plane": planes[0].n, "planes": P * world,
                           "planes_per_gpu": P, "concurrency": "one handle + stream + host thread per plane", "rtol": RTOL,
                           "cycle": "V(2,2) RB-B GS", "restart_m": 30, "levels": solvers[0].levels,
                           "step": "mg_update_coeffs + mg_solve on every plane"},
                "iters": iters[0][-1], "ms_per_plane_solve": ms / args.steps / P, "clocks": clocks,
                "gpu_launches": sum(s.kernel_launches for s in solvers) - l1, "e2e": None, "roofline": None, "cpu_baseline": None}
        print(json.dumps(line))
    for s in solvers:
        s.close()
    if world > 1:
        dist.destroy_process_group()


def run_planes_batched(args):
    """P planes of one mesh solved TOGETHER by one handle (mg_options.planes): mesh tables shared,
    vectors [plane][slot], every kernel launched once for all planes, one fGMRES state per plane (PAPER.md:211, 256,
    320-324).  Secondary bench line: HBM-resident inputs only."""
    import torch
    import torch.distributed as dist
    from paper_2509_11831_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.use_torch_allocator()
    P = args.planes
    planes = [W.make_plane(args.config, args.lattice, seed=plane_seed(args.config, rank * P + p)) for p in range(P)]
    p0 = planes[0]
    dev = lambda name: torch.from_numpy(np.stack([getattr(pl, name) for pl in planes])).cuda()
    lam, c, f, x0 = dev("lam"), dev("c"), dev("f"), dev("x0")
    x = torch.empty_like(f)
    s = B.Solver(p0.i, p0.j, p0.kind, p0.h, levels=p0.levels, planes=P)
    its = None

    def steps(k):
        nonlocal its
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        ev0.record()
        tot = 0
        for _ in range(k):
            s.update_coeffs(lam, c)
            _, its, rr, rc = s.solve(f, x0, args.rtol, x=x)
            assert rc == 0, (rc, its, rr)
            tot += sum(its)
        ev1.record()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        return ev0.elapsed_time(ev1), tot

    steps(args.warmup)
    l1 = s.kernel_launches
    sampler = ClockSampler(local) if rank == 0 else None
    ms_loc, tot = steps(args.steps)
    clocks = sampler.stop() if sampler else None
    ms, work, value = whole_job(ms_loc, float(p0.n * tot), world, "cuda")
    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": WORKLOADS[args.config], "unknowns_per_plane": p0.n, "planes": P * world,
                           "planes_per_gpu": P, "concurrency": "planes batched in the kernels (one handle, gridDim.y = planes)",
                           "rtol": args.rtol, "cycle": "V(2,2) RB-B GS", "restart_m": 30, "levels": s.levels,
                           "step": "mg_update_coeffs + mg_solve on all planes"},
                "iters": list(its), "ms_per_plane_solve": ms / args.steps / P, "clocks": clocks,
                "gpu_launches": s.kernel_launches - l1, "launches_per_step": (s.kernel_launches - l1) / args.steps,
                "e2e": None, "roofline": None, "cpu_baseline": None}
        print(json.dumps(line))
    s.close()
    if world > 1:
        dist.destroy_process_group()


def run_paper_mms(args):
    """The paper's own scaling experiment: annulus of Eq. 19-22, h halved from 4e-3 with one more
    level per refinement (4 ... 9 levels, N = 2.4e4 ... 2.4e7), V-cycle with five pre- and post-smoothing sweeps, stop at 1e-8,
    Dirichlet or Neumann conditions on the inner circle.  One JSON line per case: iterations, update / solve time (CUDA
    events), error against the manufactured solution.  Context for BASELINE.md, not the headline metric."""
    import torch
    from paper_2509_11831_b200 import binding as B
    from tests import cases as TC      # the paper-case generator is test material (sympy); only this option needs it
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    B.use_torch_allocator()
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    for k in range(args.paper_mms):
        h, levels = 4e-3 / 2 ** k, 4 + k
        for neumann in (False, True):
            pl = TC.make_paper_annulus(h, levels, neumann_inner=neumann, absorb_xi=not args.three_field)
            s = B.Solver(pl.i, pl.j, pl.kind, pl.h, levels=levels, nu_pre=5, nu_post=5)
            f = pl.f
            if neumann:
                lv = s.level_info(0)
                oR, oZ = TC.neumann_offsets(lv["kind"], lv["ns_tn"], lv["ns_fallback"], lv["nbr"])
                f = TC.neumann_gamma(pl, oR[lv["user2canon"]], oZ[lv["user2canon"]])
            d_lam, d_c, d_f, d_x0 = dev(pl.lam), dev(pl.c), dev(f), dev(pl.x0)
            d_xi = dev(pl.meta["xi"]) if args.three_field else None      # Eq. 21's xi as printed, not absorbed
            sol, upd = [], []
            for _ in range(args.warmup + args.steps):
                s.update_coeffs3(d_lam, d_xi, d_c)
                x, iters, relres, rc = s.solve(d_f, d_x0, 1e-8)
                sol.append(s.last_solve_ms); upd.append(s.last_update_ms)
            m = pl.kind == 0
            e = x.cpu().numpy()[m] - pl.meta["phi"][m]
            print(json.dumps({"workload": "PAPER.md Eq. 19-22 annulus MMS, V(5,5), rtol 1e-8", "h": h, "levels": levels,
                              "form": "three-field, xi of Eq. 21 as printed" if args.three_field else "xi absorbed (PAPER.md:47)",
                              "inner_bc": "neumann" if neumann else "dirichlet", "points": pl.n, "iters": iters, "status": rc,
                              "final_relres": relres, "solve_ms": float(np.median(sol[args.warmup:])),
                              "update_ms": float(np.median(upd[args.warmup:])),
                              "unknown_iters_per_s": pl.n * iters / (float(np.median(sol[args.warmup:])) * 1e-3),
                              "err_l2": float(np.linalg.norm(e) / np.linalg.norm(pl.meta["phi"][m])), "err_linf": float(np.abs(e).max())}),
                  flush=True)
            s.close()
            del d_lam, d_c, d_f, d_x0, d_xi, x
            torch.cuda.empty_cache()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--ref-iters", type=int, default=8, help="iteration cap of the oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--rtol", type=float, default=RTOL, help="stop tolerance of Eq. 23 (scaling runs beyond the BASELINE sizes; default 1e-10)")
    ap.add_argument("--full-cgs2", action="store_true", help="always run the second Gram-Schmidt update (MG_SETUP_FULL_CGS2)")
    ap.add_argument("--roofline-only", action="store_true", help="launch only the roofline kernel (for ncu captures)")
    ap.add_argument("--lattice", type=int, default=None, help="same geometry on an n x n lattice (2^k + 1; O(N) scaling runs)")
    ap.add_argument("--paper-mms", type=int, default=0, metavar="R",
                    help="run the paper's annulus MMS scaling experiment over R refinements (6 reaches its 24 M points) instead")
    ap.add_argument("--three-field", action="store_true", help="secondary line: the paper's three-field form with a seeded xi (mg_update_coeffs3)")
    ap.add_argument("--planes", type=int, default=1, help="planes per GPU solved together by one batched handle (secondary line, SURVEY.md 8(f) NEXT-1)")
    ap.add_argument("--solver", default="fgmres", choices=["fgmres", "bicgstab"], help="outer solver (secondary line: BiCGStab, PAPER.md:342)")
    ap.add_argument("--plane-streams", action="store_true", help="with --planes: one handle + stream + host thread per plane instead of the batched handle")
    args = ap.parse_args()
    respawn(args, sys.argv[1:])
    if os.environ.get("MG_BENCH_DRY"):
        run_dry(args)
    elif args.impl == "reference":
        run_reference(args)
    elif args.paper_mms > 0:
        run_paper_mms(args)
    elif args.planes > 1:
        run_planes(args) if args.plane_streams else run_planes_batched(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

"""Multi-GPU path of bench.py on the CPU: planes are independent solves, so N ranks
shard the planes with no data-path collective; the only communication is the max-over-ranks time and the
summed work.  Two gloo processes exercise exactly the helpers bench.py uses under torchrun."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_2509_11831_b200 import workloads as W
    pl = W.make_plane(3, 65, seed=bench.plane_seed(3, rank))
    ms_local = 10.0 * (rank + 1)                      # rank 1 is the slow one
    work_local = float(pl.n) * (7 + rank)             # ranks may take different iteration counts
    ms, work, value = bench.whole_job(ms_local, work_local, world, "cpu")
    out[rank] = (pl.n, float(pl.f.sum()), ms, work, value)
    dist.destroy_process_group()


def test_world_size_2_weak_scaling_aggregation():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        r0, r1 = out[0], out[1]
    assert r0[0] == r1[0]                             # same geometry on every rank ...
    assert r0[1] != r1[1]                             # ... different seeded right-hand sides (own plane each)
    assert r0[2:] == r1[2:]                           # every rank sees the same reduced numbers
    ms, work, value = r0[2:]
    assert ms == 20.0                                 # max over ranks
    assert work == r0[0] * 7.0 + r1[0] * 8.0          # sum over ranks
    assert value == pytest.approx(work / 20e-3)


def test_single_rank_needs_no_process_group():
    import bench
    ms, work, value = bench.whole_job(5.0, 1000.0, 1, "cpu")
    assert (ms, work) == (5.0, 1000.0) and value == pytest.approx(2e5)


def test_config5_step_sequence_is_seeded_and_chained():
    from paper_2509_11831_b200 import workloads as W        # bench.make_steps chains exactly these calls
    a = W.make_plane(5, 129)
    b1, b2 = W.next_step(a, 0), W.next_step(a, 0)
    assert np.array_equal(b1.c, b2.c) and np.array_equal(b1.f, b2.f)             # seeded
    c = W.next_step(b1, 1)
    assert np.all(np.abs(b1.lam / a.lam - 1.0) <= 0.05 + 1e-12) and np.all(np.abs(c.c / b1.c - 1.0) <= 0.05 + 1e-12)
    assert not np.array_equal(c.f, b1.f) and np.array_equal(c.i, a.i)


def test_bench_gpus_n_spawns_its_own_ranks():
    """`python bench.py --gpus 2` with no launcher re-executes itself under torchrun (one rank per GPU, 127.0.0.1
    rendezvous) — the driver's command shape for the scaling runs.  Dry mode: gloo on the CPU, no GPU work."""
    import json
    import subprocess
    env = dict(os.environ, MG_BENCH_DRY="1")
    for k in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT"):
        env.pop(k, None)
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--config", "3", "--steps", "2", "--warmup", "1"],
                         env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [json.loads(l) for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1 and lines[0]["n_gpus"] == 2 and lines[0]["ms_per_step"] == 10.0      # max over ranks: 20 ms / 2 steps
    import bench
    cmd = bench.spawn_command(4, ["--gpus", "4", "--steps", "3"], port=29511)
    assert cmd[1:4] == ["-m", "torch.distributed.run", "--nnodes=1"] and "--nproc-per-node=4" in cmd and cmd[-4:] == ["--gpus", "4", "--steps", "3"]
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1"

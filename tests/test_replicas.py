"""Multi-GPU host logic (replicas only): which workload a rank runs and how per-rank timings
combine into the whole-job figure.  World size 2 over gloo on CPU; no kernel is involved."""
import os
import socket

import pytest

from paper_0809_3098_b200 import replicas
from paper_0809_3098_b200 import workloads as W


def test_replica_workloads_same_grid_distinct_reynolds():
    base = W.config(4)
    ws = [replicas.replica_workload(base, r, 8) for r in range(8)]
    assert ws[0] is base
    for r, w in enumerate(ws):
        assert (w.N, w.dt, w.sweeps_per_stage, w.sor_omega) == (base.N, base.dt, base.sweeps_per_stage, base.sor_omega)
        assert w.Re in replicas.TABLE1_RE                      # Table 1 of the paper
        if r:
            assert w.Re != base.Re and w.seed != base.seed
    assert len({w.seed for w in ws}) == 8
    assert replicas.replica_workload(base, 3, 1) is base


def test_combine_single_rank_is_identity():
    assert replicas.combine(10.0, 2.0, 1) == (10.0, 2.0)


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # rank r processed 100 (r + 1) units in (1 + r) seconds: the job did 300 units in max = 2 s
        u, t = replicas.combine(100.0 * (rank + 1), 1.0 + rank, world, dist, torch.device("cpu"))
        q.put((rank, u, t))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(120)
def test_combine_world_size_2_gloo():
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    got = sorted(q.get(timeout=90) for _ in ps)
    for p in ps:
        p.join(30)
        assert p.exitcode == 0
    assert got == [(0, 300.0, 2.0), (1, 300.0, 2.0)]


@pytest.mark.timeout(180)
def test_bench_spawns_its_own_ranks_when_no_launcher_set_the_world():
    """A bare `python bench.py --gpus 2` (no torchrun, no WORLD_SIZE) re-executes itself as 2 ranks and prints ONE line with
    n_gpus = 2: the spawn / rendezvous / max-of-times / sum-of-units path over gloo with a stubbed step (CAV_BENCH_STUB=1)."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    env["CAV_BENCH_STUB"] = "1"
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--steps", "3"], env=env,
                         capture_output=True, text=True, timeout=150)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, out.stdout
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["stub"] is True
    assert "STUB" in d["metric"] and "stub" in d["unit"]          # cannot be mistaken for (or harvested as) the real metric
    env.pop("PYTEST_CURRENT_TEST", None)                           # outside pytest the stub is refused
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "1", "--steps", "1"], env=env,
                         capture_output=True, text=True, timeout=150)
    assert out.returncode == 2 and not [l for l in out.stdout.splitlines() if l.startswith("{")]
    # rank 1 sleeps twice as long: the job time is the MAX over ranks, the units are the SUM
    assert 55.0 <= d["ms_per_step"] * 3 <= 400.0
    G = 1025 ** 2
    assert abs(d["value"] * (d["ms_per_step"] * 3e-3) / (2 * 5.0 * G * 3) - 1.0) < 1e-9

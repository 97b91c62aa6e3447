"""The N>1 host logic on CPU: 2 processes over gloo (no GPU): disjoint world ranges, rank-distinct
worlds, max-over-ranks timing, whole-job throughput."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import gp_scenes as gs
from paper_2606_19641_b200 import shard


def test_partitions_are_disjoint_and_cover():
    for n, ws in ((1024, 8), (10, 4), (3, 8), (7, 1)):
        spans = [shard.strong_world_range(r, ws, n) for r in range(ws)]
        covered = [w for b, c in spans for w in range(b, b + c)]
        assert covered == list(range(n))
        assert max(c for _, c in spans) - min(c for _, c in spans) <= 1
    assert [shard.weak_world_range(r, 1024) for r in range(3)] == [(0, 1024), (1024, 1024), (2048, 1024)]
    with pytest.raises(ValueError):
        shard.strong_world_range(4, 4, 10)


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world_size, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world_size))
    dist.init_process_group("gloo", rank=rank, world_size=world_size)
    try:
        cfg = gs.config("small", n_worlds=3)
        w0, nw = shard.weak_world_range(rank, cfg.n_worlds)
        agents, quads = gs.gen_world_prims(cfg.replace(n_worlds=w0 + nw), w0, nw)
        # every rank's worlds are different and equal to the same global ids generated anywhere
        digest = torch.tensor([float(agents["cx"].astype(np.float64).sum()), float(w0), float(nw)], dtype=torch.float64)
        gathered = [torch.zeros(3, dtype=torch.float64) for _ in range(world_size)]
        dist.all_gather(gathered, digest)
        ms = 2.0 + rank                                   # the slower rank decides
        mx = shard.max_over_ranks(ms)
        val = shard.aggregate_throughput(cfg.views, 10, ms)
        dist.barrier()
        out.put((rank, [g.tolist() for g in gathered], mx, val, cfg.views))
    finally:
        dist.destroy_process_group()


def test_two_ranks_over_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, gathered, mx, val, views in res:
        assert mx == 3.0                                             # max over ranks, not the local time
        assert abs(val - 2 * views * 10 / 3.0e-3) < 1e-6 * val       # whole-job aggregate
        (s0, b0, n0), (s1, b1, n1) = gathered
        assert (b0, n0, b1, n1) == (0.0, 3.0, 3.0, 3.0)              # disjoint contiguous world ids
        assert s0 != s1                                              # different worlds
    # rank 1's worlds are exactly global worlds 3..5 of the same generator
    cfg = gs.config("small", n_worlds=6)
    a, _ = gs.gen_world_prims(cfg)
    assert abs(float(a["cx"][3:6].astype(np.float64).sum()) - res[1][1][1][0]) < 1e-9


def test_bench_gpus_n_starts_n_ranks_by_itself():
    """`python bench.py --gpus 2` with no launcher around it (no WORLD_SIZE in the environment) must start two ranks itself
    (VERDICT r2): CPU dry run of that launch over gloo; rank 0 prints the one JSON line with n_gpus = 2."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    p = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--launch-check"], env=env,
                       capture_output=True, text=True, timeout=300)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [ln for ln in p.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    out = json.loads(lines[0])
    assert out["n_gpus"] == 2 and out["asked_gpus"] == 2 and out["slowest_rank_ms"] == 2.0


def test_bench_reference_arm_runs_on_rank_zero_only():
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    p = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--gpus", "2", "--workload", "tiny",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert p.returncode == 0 and p.stdout.strip() == ""              # the other ranks exit 0 without work
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK")}
    p = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--gpus", "2", "--workload", "tiny",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert p.returncode == 0, p.stderr[-2000:]
    out = json.loads(p.stdout.strip().splitlines()[-1])
    assert out["impl"] == "reference" and out["n_gpus"] == 2 and out["gpu_launches"] == 0 and out["value"] > 0

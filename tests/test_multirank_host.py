"""N > 1 host logic on CPU (gloo, world_size 2): how bench.py splits the batch, reduces the per-rank
timings to the slowest rank and lets rank 0 alone report.  dgfs_collide itself needs no collective
(PAPER.md P:86), so there is no data-path exchange to test."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    sys.path.insert(0, ROOT)
    import dataclasses
    from paper_1903_04670_b200.parallel import shard_range, rank_seed, max_over_ranks, whole_job_rate
    from workloads import get_config, make_points
    cfg = get_config("c0")
    # weak scaling: own seed per rank => different, reproducible inputs
    f = make_points(dataclasses.replace(cfg, seed=rank_seed(cfg.seed, rank)), range(2))
    sums = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
    dist.all_gather(sums, torch.tensor([float(f.sum())], dtype=torch.float64))
    # strong split of a given batch: blocks tile [0, nx) exactly
    lo, hi = shard_range(11, world, rank)
    blocks = [torch.zeros(2, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(blocks, torch.tensor([lo, hi]))
    # the slowest rank sets the time
    ms = max_over_ranks(10.0 + 5.0 * rank)
    dist.barrier()
    if rank == 0:
        out.put(dict(sums=[float(s) for s in sums], blocks=[b.tolist() for b in blocks], ms=ms,
                     rate=whole_job_rate(8, world, ms)))
    dist.destroy_process_group()


def test_two_ranks_gloo_sharding_and_timing():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.SimpleQueue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    res = out.get()
    assert res["sums"][0] != res["sums"][1]
    assert res["blocks"] == [[0, 6], [6, 11]]
    assert res["ms"] == 15.0
    assert abs(res["rate"] - 16 / 15e-3) < 1e-9


def test_shard_range_tiles_the_batch():
    from paper_1903_04670_b200.parallel import shard_range, max_over_ranks
    for nx in (0, 1, 7, 4096):
        for world in (1, 2, 3, 8):
            edges = [shard_range(nx, world, r) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == nx
            assert all(edges[i][1] == edges[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in edges]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_range(4, 2, 2)
    assert max_over_ranks(3.5) == 3.5                     # no process group: identity


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    """bench.py --impl reference launched as the driver launches it for N = 2: rank 0 alone runs the
    oracle and prints the JSON line, rank 1 exits 0 without work."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"),
           "--impl", "reference", "--workload", "c0", "--gpus", "2", "--steps", "1", "--warmup", "0"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0

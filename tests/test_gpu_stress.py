"""Randomised use of the boundary (seeded): contexts of random (N, species, M, N_rho, VHS / VSS), random batch sizes, launch
groups and workspace budgets, the v0 and v1 pipelines, precision 1, the Nyquist-filter variant; dgfs_collide on the
current stream, dgfs_collide_pairs on another stream without any synchronisation in between (the library orders the calls
of one context), dgfs_collide_noalloc, dgfs_collide_host.  Every batched result must equal, bit for bit, the results of
single-point calls of the same context (points are independent), three times in a row."""
import os

import numpy as np
import pytest

from workloads import make_points
from workloads.configs import Config, _mean_matrix

pytestmark = pytest.mark.gpu

ENV_KEYS = ("DGFS_V1_CHUNK", "DGFS_V1_GRAPH_ITEMS", "DGFS_PIPELINE", "DGFS_V1_WS_GB")


@pytest.mark.parametrize("seed", [3, 17])
def test_random_contexts_batches_and_streams(seed, monkeypatch):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device: there is no CPU fallback")
    from paper_1903_04670_b200 import Dgfs, DgfsError
    torch.cuda.set_device(0)
    rng = np.random.default_rng(seed)
    ran_noalloc = 0
    for case in range(30):
        N = int(rng.choice([8, 16, 24, 32]))
        ns = int(rng.choice([1, 2, 3]))
        M = int(rng.choice([6, 12, 32] if N <= 16 else [6, 12]))
        N_rho = int(rng.integers(1, 4))
        vss = bool(rng.integers(0, 2))
        alpha = tuple(1.0 + (0.1 + 0.3 * rng.random() if vss else 0.0) for _ in range(ns))
        cfg = Config("s", int(rng.integers(1, 1 << 30)), tuple(1.0 + 0.7 * i for i in range(ns)),
                     _mean_matrix(tuple(0.6 + 0.1 * i for i in range(ns))), _mean_matrix(alpha),
                     N=N, L=5.5, N_rho=N_rho, M=M, nx=3, kind="bimaxwell")
        nx = int(rng.integers(1, {8: 70, 16: 40, 24: 14, 32: 9}[N] + 1))
        for k in ENV_KEYS:
            monkeypatch.delenv(k, raising=False)
        kw = {}
        if rng.random() < 0.3:
            monkeypatch.setenv("DGFS_V1_CHUNK", str(int(rng.integers(1, 9))))
        if rng.random() < 0.2:
            monkeypatch.setenv("DGFS_V1_GRAPH_ITEMS", "0")
        if rng.random() < 0.2:
            monkeypatch.setenv("DGFS_PIPELINE", "v0")
        elif not vss and rng.random() < 0.25:
            kw["precision"] = 1
        if rng.random() < 0.15:
            monkeypatch.setenv("DGFS_V1_WS_GB", "0.05")
        if rng.random() < 0.2:
            kw["nyquist_filter"] = True
        what = dict(case=case, N=N, ns=ns, M=M, N_rho=N_rho, vss=vss, nx=nx, kw=kw,
                    env={k: os.environ[k] for k in ENV_KEYS if k in os.environ})
        f = torch.from_numpy(make_points(cfg, range(nx))).cuda()
        with Dgfs.from_config(cfg, device=0, **kw) as op:
            ref = torch.stack([op.collide(f[x:x + 1].contiguous())[0] for x in range(nx)])
            refp = torch.stack([op.collide_pairs(f[x:x + 1].contiguous())[0] for x in range(nx)])
            assert bool(torch.isfinite(ref).all()) and float(ref.abs().max()) > 0.0, what
            side = torch.cuda.Stream()
            for rep in range(3):
                a = op.collide(f)
                with torch.cuda.stream(side):
                    b = op.collide_pairs(f)
                c = torch.empty_like(ref)
                try:
                    op.collide_noalloc(f, c)
                    ran_noalloc += 1
                except DgfsError as e:                  # v0 contexts, or a point beyond the static scratch: refused
                    assert e.code in (-1, -4), what
                    c = None
                h = op.collide_host(f.cpu().numpy())
                torch.cuda.synchronize()
                assert torch.equal(a, ref), what
                assert torch.equal(b, refp), what
                assert c is None or torch.equal(c, ref), what
                assert np.array_equal(h, ref.cpu().numpy()), what
    assert ran_noalloc > 0


def test_launch_group_at_the_grid_limit(monkeypatch):
    """Maximum sizes of the launch geometry: a launch group asked to be larger than the grid's y extent allows
    (65535 rows = points x pairs) is clipped to it, and a batch larger than one group is split with a ragged tail; v1 (20 000
    points of N = 8, 2 species: groups of 16 383 + 3 617) and the v0 pipeline's own limit.  Sampled points against
    single-point calls, bit for bit; no point left unwritten."""
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device: there is no CPU fallback")
    from paper_1903_04670_b200 import Dgfs
    torch.cuda.set_device(0)
    cfg = Config("g", 77, (1.0, 1.7), _mean_matrix((0.6, 0.8)), _mean_matrix((1.0, 1.0)),
                 N=8, L=5.5, N_rho=2, M=6, nx=3, kind="bimaxwell")
    nx = 20000
    base = torch.from_numpy(make_points(cfg, range(50))).cuda()
    scale = 1.0 + 0.5 * torch.rand(nx, 1, 1, dtype=torch.float64, device="cuda", generator=torch.Generator("cuda").manual_seed(5))
    f = (base[torch.arange(nx, device="cuda") % 50] * scale).contiguous()
    sample = [0, 1, 16382, 16383, 16384, 19998, 19999]
    for pipeline, chunk_env in (("v1", "DGFS_V1_CHUNK"), ("v0", "DGFS_SCRATCH_MB")):
        monkeypatch.delenv("DGFS_PIPELINE", raising=False)
        if pipeline == "v0":
            monkeypatch.setenv("DGFS_PIPELINE", "v0")
        monkeypatch.setenv(chunk_env, "40000")
        with Dgfs.from_config(cfg, device=0) as op:
            out = torch.full((nx, cfg.ns, cfg.N ** 3), float("nan"), dtype=torch.float64, device="cuda")
            op.collide(f, out=out)
            assert bool(torch.isfinite(out).all()), pipeline
            for x in sample:
                assert torch.equal(op.collide(f[x:x + 1].contiguous())[0], out[x]), (pipeline, x)
        monkeypatch.delenv(chunk_env, raising=False)

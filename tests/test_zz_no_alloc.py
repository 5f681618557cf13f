"""dgfs_collide_noalloc (include/dgfs.h): dgfs_collide with the workspace in the library's static device array
(DGFS_NOALLOC_SCRATCH_BYTES = 64 MiB) instead of an allocation, for callers that must not allocate device memory.
Checked against the existing path, dgfs_collide, on the same seeded inputs, on two calls in a row (the second call
finds what the first left in the shared array), within the tolerance of the other GPU tests (1e-10 relative to max|Q|);
the two paths run the same kernels, so the results are also expected to be equal bit for bit.

This file is collected last on purpose (pytest -x stops at the first failure) and passes alone in a fresh process."""
import numpy as np
import pytest

from workloads import get_config, make_points

pytestmark = pytest.mark.gpu

TOL = 1e-10
SCRATCH_BYTES = 64 << 20


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(0)
    return torch


def _cfg(name, ns, N, N_rho, M, seed):
    from workloads.configs import Config, _mean_matrix
    masses = (1.0, 2.0, 3.5)[:ns]
    return Config(name, seed, masses, _mean_matrix((0.6, 0.8, 0.7)[:ns]), _mean_matrix((1.0,) * ns),
                  N=N, L=5.5, N_rho=N_rho, M=M, nx=3, kind="bimaxwell")


def _rel(a, b):
    a, b = a.cpu().numpy(), b.cpu().numpy()
    return (np.max(np.abs(a - b), axis=-1) / np.max(np.abs(b), axis=-1)).max()


def _device_bytes_in_use(torch):
    free, total = torch.cuda.mem_get_info()
    return total - free


def test_two_calls_in_a_row_match_dgfs_collide_on_c0(torch_cuda):
    torch = torch_cuda
    from paper_1903_04670_b200 import Dgfs
    cfg = get_config("c0")
    f1 = torch.from_numpy(make_points(cfg, range(cfg.nx))).cuda()
    f2 = torch.from_numpy(make_points(cfg, range(cfg.nx, 2 * cfg.nx))).cuda()      # other inputs for the second call
    with Dgfs.from_config(cfg, device=0) as op:
        ref1, ref2 = op.collide(f1).clone(), op.collide(f2).clone()
        out1, out2 = torch.empty_like(ref1), torch.empty_like(ref2)
        torch.cuda.synchronize()
        used = _device_bytes_in_use(torch)
        op.collide_noalloc(f1, out1)
        op.collide_noalloc(f2, out2)
        torch.cuda.synchronize()
        assert _device_bytes_in_use(torch) <= used          # the calls took no device memory
        assert _rel(out1, ref1) < TOL and _rel(out2, ref2) < TOL
        assert torch.equal(out1, ref1) and torch.equal(out2, ref2)
        # and the first inputs again, after the array has held the second call's data
        out1.zero_()
        op.collide_noalloc(f1, out1)
        assert torch.equal(out1, ref1)
    assert float(ref1.abs().max()) > 0.0 and not torch.equal(ref1, ref2)


def test_batch_beyond_the_array_runs_in_smaller_launch_groups(torch_cuda):
    """100 points of a 2-species N = 16 configuration need more than 64 MiB in one launch group: the no-alloc call
    halves the group until it fits the array and still equals dgfs_collide; also on a fresh context whose first call
    ever is the no-alloc one (kernel attributes are set there)."""
    torch = torch_cuda
    from paper_1903_04670_b200 import Dgfs
    cfg = _cfg("t", 2, 16, 3, 12, seed=21)
    nx = 100
    f = torch.from_numpy(make_points(cfg, range(nx))).cuda()
    out = torch.empty((nx, cfg.ns, cfg.N ** 3), dtype=torch.float64, device="cuda")
    with Dgfs.from_config(cfg, device=0) as op:
        assert op.workspace_bytes(nx) > SCRATCH_BYTES       # what dgfs_collide would allocate for this batch
        op.collide_noalloc(f, out)                          # first call of the context
        ref = op.collide(f)
        assert _rel(out, ref) < TOL and torch.equal(out, ref)
        out.zero_()
        op.collide_noalloc(f, out)                          # second call in a row
        assert _rel(out, ref) < TOL and torch.equal(out, ref)


def test_three_species_n32_single_points(torch_cuda):
    """N = 32 (the headline resolution), three species (nine VHS pairs): a few points per call fit the array."""
    torch = torch_cuda
    from paper_1903_04670_b200 import Dgfs
    cfg = _cfg("t", 3, 32, 2, 6, seed=5)
    f = torch.from_numpy(make_points(cfg, range(5))).cuda()
    out = torch.empty((5, cfg.ns, cfg.N ** 3), dtype=torch.float64, device="cuda")
    with Dgfs.from_config(cfg, device=0) as op:
        ref = op.collide(f).clone()
        for _ in range(2):
            out.zero_()
            op.collide_noalloc(f, out)
            assert _rel(out, ref) < TOL and torch.equal(out, ref)


def test_sizes_beyond_the_limit_and_unsupported_contexts_are_refused(torch_cuda, monkeypatch):
    torch = torch_cuda
    from paper_1903_04670_b200 import Dgfs, DgfsError
    # one point of N = 48 with nine pairs and a 32-point sphere rule does not fit 64 MiB
    cfg = _cfg("t", 3, 48, 1, 32, seed=3)
    f = torch.from_numpy(make_points(cfg, range(1))).cuda()
    out = torch.full((1, cfg.ns, cfg.N ** 3), 7.0, dtype=torch.float64, device="cuda")
    with Dgfs.from_config(cfg, device=0) as op:
        assert op.workspace_bytes(1) > SCRATCH_BYTES
        with pytest.raises(DgfsError) as ei:
            op.collide_noalloc(f, out)
        assert ei.value.code == -1 and "DGFS_NOALLOC_SCRATCH_BYTES" in str(ei.value)
        torch.cuda.synchronize()
        assert bool((out == 7.0).all())                     # refused before any launch
        ref = op.collide(f)                                 # the context still works
        assert torch.isfinite(ref).all()
    # a context on the v0 pipeline
    monkeypatch.setenv("DGFS_PIPELINE", "v0")
    cfg0 = get_config("c0")
    f0 = torch.from_numpy(make_points(cfg0, range(1))).cuda()
    with Dgfs.from_config(cfg0, device=0) as op:
        with pytest.raises(DgfsError) as ei:
            op.collide_noalloc(f0, torch.empty_like(f0))
        assert ei.value.code == -4

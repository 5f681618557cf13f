"""Parity at the sizes of BASELINE.json's configs c1..c4: the GPU runs the batch in the launch
configuration bench.py times (one dgfs_collide[_pairs] call over the whole batch); the oracle
computes a seeded sample of points one by one (SURVEY.md 8(d) "parity is checked on a seeded
subset").  Tolerance: 1e-10 relative to max|Q| per (point, pair) array."""
import os

import numpy as np
import pytest

from workloads import get_config, make_points, make_dg_state

pytestmark = pytest.mark.gpu

TOL = 1e-10


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(0)
    return torch


def _oracle_pairs(cfg, f_sample):
    from oracle.tables import precompute
    from oracle.collide import collide_pairs
    tab = precompute(cfg.N, cfg.N_rho, cfg.M, cfg.L, cfg.mass, cfg.omega, cfg.alpha)
    return collide_pairs(tab, f_sample)


def _check(Qg, Qo, what):
    num = np.max(np.abs(Qg - Qo), axis=-1)
    den = np.max(np.abs(Qo), axis=-1)
    err = num / den
    print("%s: max rel err %.3e over %d (point, pair) arrays" % (what, err.max(), err.size))
    assert err.max() < TOL, err


def _run_batch(torch, cfg, xs_all, sample, pairs=True):
    from paper_1903_04670_b200 import Dgfs
    f = make_points(cfg, xs_all)
    pos = [list(xs_all).index(x) for x in sample]
    with Dgfs.from_config(cfg, device=0) as op:
        fd = torch.from_numpy(f).cuda()
        Q = op.collide_pairs(fd) if pairs else op.collide(fd)
        torch.cuda.synchronize()
        Qs = Q[pos].cpu().numpy()
        del Q, fd
    torch.cuda.empty_cache()
    return f[pos], Qs


def test_c1_full_batch_sampled_points(torch_cuda):
    cfg = get_config("c1")
    sample = [0, 1, 511, 1023]
    fs, Qg = _run_batch(torch_cuda, cfg, range(cfg.nx), sample)
    _check(Qg, _oracle_pairs(cfg, fs), "c1")


def test_c2_full_batch_sampled_points_both_halves(torch_cuda):
    """Headline config, all 4096 points in one call; sample covers the near-equilibrium half
    (x < 2048, Q is a small difference of large terms) and the non-equilibrium half."""
    cfg = get_config("c2")
    sample = [0, 2047, 2048, 4095]
    fs, Qg = _run_batch(torch_cuda, cfg, range(cfg.nx), sample, pairs=False)
    Qo = _oracle_pairs(cfg, fs).sum(axis=2)
    _check(Qg, Qo, "c2 (summed over q)")


def test_c2_pairs_output_reduced_batch(torch_cuda):
    cfg = get_config("c2")
    xs = [5, 1000, 2047, 2048, 3000, 4095, 17]
    sample = [1000, 3000]
    fs, Qg = _run_batch(torch_cuda, cfg, xs, sample)
    _check(Qg, _oracle_pairs(cfg, fs), "c2 pairs")


def test_c3_collision_term_of_dg_state(torch_cuda):
    """c3's collide call: 3 species, 8 of 9 pairs VSS (full b tables), 64 spatial DOF."""
    torch = torch_cuda
    from paper_1903_04670_b200 import Dgfs
    cfg = get_config("c3")
    K = cfg.order + 1
    f = make_dg_state(cfg).reshape(cfg.ne * K, cfg.ns, cfg.N ** 3)
    # perturb node values so that the DOF of one element differ
    rng = np.random.default_rng(cfg.seed)
    f = f * (1.0 + 0.02 * rng.uniform(-1, 1, (f.shape[0], f.shape[1], 1)))
    pos = [0, 37]
    with Dgfs.from_config(cfg, device=0) as op:
        Q = op.collide_pairs(torch.from_numpy(f).cuda())
        Qg = Q[pos].cpu().numpy()
    _check(Qg, _oracle_pairs(cfg, f[pos]), "c3 collide")


@pytest.mark.slow
def test_c4_stress_reduced_batch(torch_cuda):
    """N=48, N_rho=48, M=32 (tables and arrays beyond shared memory).  The batch is cut to 24 of
    the config's 2048 points (the full batch is ~0.4 PFLOP); one point goes through the oracle."""
    cfg = get_config("c4")
    xs = list(range(0, 2048, 89))[:24]
    xs[-1] = 2047
    sample = [xs[7]]
    fs, Qg = _run_batch(torch_cuda, cfg, xs, sample)
    from oracle.tables import precompute
    from oracle.collide import collide_pair
    tab = precompute(cfg.N, cfg.N_rho, cfg.M, cfg.L, cfg.mass, cfg.omega, cfg.alpha)
    for (p, q) in ((0, 1), (1, 0)):          # ~1 min of oracle time per pair
        Qo = collide_pair(tab, p, q, fs[0, p], fs[0, q])
        _check(Qg[0, p, q][None], Qo[None], "c4 pair (%d,%d)" % (p, q))

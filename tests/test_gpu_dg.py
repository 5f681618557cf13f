"""Parity of dgfs_advect_rhs / dgfs_step (rows D1-D4, through the C ABI) with oracle/dg.py.

Tolerances: transport alone is a handful of fp64 operations per node: 1e-12 relative to max|rhs|.
A full step carries the collision term (1e-10 relative to max|Q|, north_star); after n steps the
state is compared at 1e-10 relative to max|f| and, because dt |L(f)| << |f| makes that bar loose, the
increment f_n - f_0 at 1e-10 relative to max|f_n - f_0| as well."""
import numpy as np
import pytest

from workloads import get_config, make_dg_state

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(0)
    return torch


def _rough_state(ne, K, ns, N, L, mass, seed, wall_T=(1.0, 1.0)):
    from oracle.dg import wall_maxwellian
    rng = np.random.default_rng(seed)
    f = np.empty((ne, K, ns, N ** 3))
    for p in range(ns):
        f[:, :, p] = (0.6 + 0.4 * p) * wall_maxwellian(N, L, (0.1, -0.05, 0.0), 1.1, mass[p])
    return f * (1.0 + 0.2 * rng.uniform(-1, 1, f.shape))


@pytest.mark.parametrize("ne,order,ns,N", [(1, 1, 1, 8), (3, 2, 2, 8), (5, 3, 2, 16), (2, 7, 1, 8), (16, 3, 3, 8)])
def test_advect_rhs_matches_oracle(torch_cuda, ne, order, ns, N):
    torch = torch_cuda
    from oracle import dg
    from paper_1903_04670_b200 import Dgfs, Mesh1D, api
    L = 5.0
    mass = (1.0, 1.5, 2.0)[:ns]
    K = order + 1
    wall_T, wall_u = (0.8, 1.2), ((0.0, 0.2, 0.0), (0.0, -0.2, 0.1))
    f = _rough_state(ne, K, ns, N, L, mass, seed=ne * 10 + order)
    omesh = dg.Mesh1D(ne, order, x0=-0.3, x1=1.4, wall_T=wall_T, wall_u=wall_u)
    ro = dg.advect_rhs(omesh, f, N, L, mass)
    om = [[0.5] * ns] * ns
    al = [[1.0] * ns] * ns
    with Dgfs(mass, om, al, N, 2, 6, L, device=0) as op:
        mesh = Mesh1D(ne, order, x0=-0.3, x1=1.4, wall_T=wall_T, wall_u=wall_u)
        fd = torch.from_numpy(f).cuda()
        rd = torch.empty_like(fd)
        api.dgfs_advect_rhs(op.ctx, mesh, fd, rd)
        rg = rd.cpu().numpy()
        with pytest.raises(api.DgfsError):
            api.dgfs_advect_rhs(op.ctx, mesh, fd, fd)                       # aliasing
        with pytest.raises(api.DgfsError):
            api.dgfs_advect_rhs(op.ctx, Mesh1D(ne, 9), fd, rd)              # order out of range
    assert np.max(np.abs(rg - ro)) < 1e-12 * np.max(np.abs(ro))


def test_step_matches_oracle_small(torch_cuda):
    """2 species, VHS (v1 collision pipeline inside), 3 elements of order 2, 2 SSP-RK3 steps."""
    torch = torch_cuda
    from oracle import dg
    from oracle.tables import precompute
    from oracle.collide import collide
    from paper_1903_04670_b200 import Dgfs, Mesh1D, api
    N, L, N_rho, M = 8, 5.0, 3, 6
    mass = (1.0, 2.0)
    om = ((0.81, 0.805), (0.805, 0.8))
    al = ((1.0, 1.0), (1.0, 1.0))
    ne, order, dt, nsteps = 3, 2, 2e-3, 2
    f = _rough_state(ne, order + 1, 2, N, L, mass, seed=3)
    tab = precompute(N, N_rho, M, L, mass, om, al)
    omesh = dg.Mesh1D(ne, order, wall_T=(0.8, 1.2))
    fo = dg.step(omesh, f, dt, nsteps, N, L, mass, collide=lambda g: collide(tab, g))
    with Dgfs(mass, om, al, N, N_rho, M, L, device=0) as op:
        fd = torch.from_numpy(f).cuda()
        api.dgfs_step(op.ctx, Mesh1D(ne, order, wall_T=(0.8, 1.2)), fd, dt, nsteps)
        fg = fd.cpu().numpy()
        api.dgfs_step(op.ctx, Mesh1D(ne, order, wall_T=(0.8, 1.2)), fd, dt, 0)          # nsteps = 0: no-op
        assert np.array_equal(fd.cpu().numpy(), fg)
    es, ei = _step_errs(fg, fo, f)
    assert es < 1e-10 and ei < 1e-10, (es, ei)                                # state and increment f_n - f_0
    assert np.max(np.abs(fg - f)) > 1e-4 * np.max(np.abs(f))                  # the state did move


def _step_errs(fg, fo, f0):
    """(error of the state relative to max|f|, error of the increment f_n - f_0 relative to max|increment|)."""
    return (np.max(np.abs(fg - fo)) / np.max(np.abs(fo)),
            np.max(np.abs((fg - f0) - (fo - f0))) / np.max(np.abs(fo - f0)))


@pytest.mark.slow
def test_step_c3_whole_slab_after_steps_1_and_5(torch_cuda):
    """Config c3 (3 species, 8 of 9 pairs VSS, 16 elements of order 3 = 64 DOF, N = 24, diffuse walls at 0.8 / 1.2):
    the whole slab after 1 and after 5 SSP-RK3 steps (15 stages, 8640 pair evaluations through the oracle, spread
    over the host cores).  Both the state (1e-10 of max|f|) and the increment f_n - f_0 (1e-10 of max|f_n - f_0|,
    the sharper statement: dt = 2e-4 makes the increment ~1e-3 of the state) are compared."""
    torch = torch_cuda
    from oracle import dg
    from oracle_pool import tables_for, collide_pool, record
    from paper_1903_04670_b200 import Dgfs, Mesh1D, api
    cfg = get_config("c3")
    f = make_dg_state(cfg)
    tab = tables_for(cfg)
    omesh = dg.Mesh1D(cfg.ne, cfg.order, wall_T=cfg.wall_T)
    coll = lambda g: collide_pool(tab, g)
    fo1 = dg.step(omesh, f, cfg.dt, 1, cfg.N, cfg.L, cfg.mass, collide=coll)
    fo5 = dg.step(omesh, fo1, cfg.dt, 4, cfg.N, cfg.L, cfg.mass, collide=coll)
    mesh = Mesh1D(cfg.ne, cfg.order, wall_T=cfg.wall_T)
    with Dgfs.from_config(cfg, device=0) as op:
        fd = torch.from_numpy(f).cuda()
        api.dgfs_step(op.ctx, mesh, fd, cfg.dt, 1)
        fg1 = fd.cpu().numpy()
        api.dgfs_step(op.ctx, mesh, fd, cfg.dt, 4)
        fg5 = fd.cpu().numpy()
        fe = torch.from_numpy(f).cuda()
        api.dgfs_step(op.ctx, mesh, fe, cfg.dt, 5)                  # 5 steps in one call == 1 + 4
        assert torch.equal(fe, fd)
    for n, fg, fo in ((1, fg1, fo1), (5, fg5, fo5)):
        es, ei = _step_errs(fg, fo, f)
        record("c3", "whole slab after %d RK3 step(s): state" % n, es, 1e-10)
        record("c3", "whole slab after %d RK3 step(s): increment f_n - f_0" % n, ei, 1e-10)
        assert es < 1e-10 and ei < 1e-10, (n, es, ei)


def test_couette_c01_euler_step(torch_cuda):
    """Second workload: the paper's Couette case C-01 (Table 2: Ar-Kr-like
    masses, all four pairs VSS, printed Knudsen numbers, walls moving at -+50 m/s, 4 elements of order 3, 32^3,
    N_rho = 8, M = 12, forward Euler).  One Euler step of the whole slab against the oracle (all 16 nodes, both
    walls), and nsteps = 2 in one call bit-equal to two calls of one step (odd / even buffer parity of the
    Euler ping-pong)."""
    torch = torch_cuda
    from oracle import dg
    from oracle_pool import tables_for, drop_tables, collide_pool, record
    from paper_1903_04670_b200 import Dgfs, Mesh1D, api
    cfg = get_config("couette")
    f = make_dg_state(cfg)
    tab = tables_for(cfg)
    omesh = dg.Mesh1D(cfg.ne, cfg.order, wall_T=cfg.wall_T, wall_u=cfg.wall_u)
    fo = dg.step(omesh, f, cfg.dt, 1, cfg.N, cfg.L, cfg.mass, collide=lambda g: collide_pool(tab, g), scheme="euler")
    drop_tables(cfg)
    mesh = Mesh1D(cfg.ne, cfg.order, wall_T=cfg.wall_T, wall_u=cfg.wall_u)
    with Dgfs.from_config(cfg, device=0) as op:
        fd = torch.from_numpy(f).cuda()
        api.dgfs_step_euler(op.ctx, mesh, fd, cfg.dt, 1)
        f1 = fd.cpu().numpy()
        api.dgfs_step_euler(op.ctx, mesh, fd, cfg.dt, 1)
        f2 = fd.clone()
        fe = torch.from_numpy(f).cuda()
        api.dgfs_step_euler(op.ctx, mesh, fe, cfg.dt, 2)
        assert torch.equal(fe, f2)
        api.dgfs_step_euler(op.ctx, mesh, fe, cfg.dt, 0)                     # no-op
        assert torch.equal(fe, f2)
        with pytest.raises(api.DgfsError):
            api.dgfs_step_euler(op.ctx, mesh, fe, -1.0, 1)
    es, ei = _step_errs(f1, fo, f)
    record("couette", "whole slab after 1 Euler step: state", es, 1e-10)
    record("couette", "whole slab after 1 Euler step: increment", ei, 1e-10)
    assert es < 1e-10 and ei < 1e-10, (es, ei)
    # the step did something: the gas at the wall nodes picked up y momentum of the sign of its wall's velocity
    c = -cfg.L + (np.arange(cfg.N) + 0.5) * 2.0 * cfg.L / cfg.N
    cy = np.broadcast_to(c[None, :, None], (cfg.N,) * 3).reshape(-1)
    for p in range(cfg.ns):
        assert (f1[0, 0, p] * cy).sum() < 0.0 < (f1[-1, -1, p] * cy).sum()

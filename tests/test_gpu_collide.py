"""Parity of the CUDA path (through the C ABI, via the ctypes binding) with the CPU oracle.

Bar (BASELINE.json north_star): max|Q_gpu - Q_oracle| <= 1e-10 * max|Q_oracle| per (point, pair)
array, fp64.  Tables: 1e-13 relative to the table's max.
"""
import numpy as np
import pytest

from workloads import get_config, make_points, make_dg_state, maxwellian

pytestmark = pytest.mark.gpu

TOL = 1e-10


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(0)
    return torch


def _oracle_tables(cfg, **kw):
    from oracle.tables import precompute
    return precompute(cfg.N, cfg.N_rho, cfg.M, cfg.L, cfg.mass, cfg.omega, cfg.alpha, **kw)


def _gpu_op(cfg, **kw):
    from paper_1903_04670_b200 import Dgfs
    return Dgfs.from_config(cfg, device=0, **kw)


def _pair_errs(Qg, Qo):
    """max over velocity nodes, per (x, p, q), relative to that array's max."""
    num = np.max(np.abs(Qg - Qo), axis=-1)
    den = np.max(np.abs(Qo), axis=-1)
    return num / den


def _rand_cfg(name, ns, N, N_rho, M, alpha_diag, omega_diag, masses, seed):
    from workloads.configs import Config, _mean_matrix
    return Config(name, seed, tuple(masses), _mean_matrix(omega_diag), _mean_matrix(alpha_diag),
                  N=N, L=5.5, N_rho=N_rho, M=M, nx=3, kind="bimaxwell")


# ------------------------------------------------------------------------------ config c0, complete
def test_c0_all_points_all_pairs(torch_cuda):
    torch = torch_cuda
    from oracle.collide import collide_pairs
    cfg = get_config("c0")
    f = make_points(cfg, range(cfg.nx))
    Qo = collide_pairs(_oracle_tables(cfg), f)
    with _gpu_op(cfg) as op:
        fd = torch.from_numpy(f).cuda()
        Qg = op.collide_pairs(fd).cpu().numpy()
        Qs = op.collide(fd).cpu().numpy()
    assert _pair_errs(Qg, Qo).max() < TOL
    Qos = Qo.sum(axis=2)
    assert (np.max(np.abs(Qs - Qos), axis=-1) / np.max(np.abs(Qos), axis=-1)).max() < TOL


# ------------------------------------------------------------- every supported N, VHS and VSS pairs
@pytest.mark.parametrize("N,N_rho,M,ns,alpha", [
    (8, 5, 12, 3, (1.0, 1.2, 1.4)),       # mixed: pair (0,0) VHS, the rest VSS
    (16, 4, 6, 2, (1.0, 1.0)),
    (16, 3, 12, 2, (1.3, 1.0)),
    (24, 3, 12, 2, (1.0, 1.0)),           # radix-3 path
    (24, 2, 6, 2, (1.0, 1.45)),
    (32, 3, 12, 2, (1.0, 1.0)),
    (32, 2, 6, 2, (1.4, 1.4)),
    (48, 2, 6, 2, (1.0, 1.0)),
    (48, 1, 6, 2, (1.0, 1.2)),
])
def test_small_radial_rule_every_N(torch_cuda, N, N_rho, M, ns, alpha):
    _small_radial_rule(torch_cuda, N, N_rho, M, ns, alpha)


@pytest.mark.parametrize("N,N_rho,M,ns", [(8, 3, 6, 2), (16, 2, 12, 2), (32, 2, 12, 2),
                                          (8, 2, 32, 2),       # weighted 32-point rule: R-10 weight folding (v0_wfac)
                                          (48, 1, 12, 2)])     # N = 48 on the stage-per-kernel pipeline (VSS pairs use it)
def test_v0_pipeline_on_vhs_pairs(torch_cuda, monkeypatch, N, N_rho, M, ns):
    """All-VHS configurations default to the v1 pipeline; DGFS_PIPELINE=v0 keeps the stage-per-kernel
    pipeline (the one VSS pairs and N = 48 use) covered on the same inputs."""
    monkeypatch.setenv("DGFS_PIPELINE", "v0")
    _small_radial_rule(torch_cuda, N, N_rho, M, ns, (1.0,) * ns)


@pytest.mark.parametrize("N,N_rho,M,ns,noise", [
    (8, 4, 32, 2, 0.3),        # 32-point rule: 11 distinct sigma_z values
    (8, 3, 12, 3, 0.5),        # 9 pairs, strongly rough input: the Nyquist-plane terms are O(1) of the result
    (16, 2, 32, 1, 0.3),       # single species: sides A and B share their z shifts
    (32, 2, 6, 2, 0.3),        # octahedron: sigma with two zero components
    (32, 1, 32, 1, 0.3),       # more uz planes than k_wterm keeps resident in shared memory
    (48, 2, 12, 2, 0.3),       # N = 48: the 64-thread plane job with split transforms (collide_v1_wide.cuh)
    (48, 1, 32, 2, 0.3),       # ... with the weighted 32-point rule of config c4
])
def test_v1_nyquist_terms(torch_cuda, N, N_rho, M, ns, noise):
    _small_radial_rule(torch_cuda, N, N_rho, M, ns, (1.0,) * ns, noise=noise)


def test_table_mode_1_collide(torch_cuda):
    """Algorithm 1 taken literally (pre-computation sphere): every pair then has a full b table, also
    the VHS ones, and runs the per-s forward transforms of the v1 pipeline."""
    torch = torch_cuda
    from oracle.collide import collide_pairs
    from oracle.quadrature import sphere_rule
    sp, wp = sphere_rule(12)
    cfg = _rand_cfg("t", 2, 16, 3, 6, (1.0, 1.3), (0.6, 0.8), (1.0, 2.0), seed=31)
    rng = np.random.default_rng(31)
    f = make_points(cfg, range(cfg.nx)) * (1.0 + 0.2 * rng.uniform(-1, 1, (cfg.nx, 2, 16 ** 3)))
    kw = dict(table_mode=1, sigma_pre=sp, w_pre=wp)
    Qo = collide_pairs(_oracle_tables(cfg, **kw), f)
    with _gpu_op(cfg, **kw) as op:
        Qg = op.collide_pairs(torch.from_numpy(f).cuda()).cpu().numpy()
    assert _pair_errs(Qg, Qo).max() < TOL


@pytest.mark.parametrize("N,alpha", [(8, (1.0, 1.2, 1.4)), (16, (1.3, 1.0))])
def test_v0_pipeline_on_vss_pairs(torch_cuda, monkeypatch, N, alpha):
    """VSS pairs default to the v1 pipeline for N <= 32; DGFS_PIPELINE=v0 keeps the stage-per-kernel one
    (which N = 48 always uses) covered on the same inputs."""
    monkeypatch.setenv("DGFS_PIPELINE", "v0")
    _small_radial_rule(torch_cuda, N, 3, 12, len(alpha), alpha)


def test_v1_antipodal_symmetry_switch(torch_cuda, monkeypatch):
    """R-10: same-species VHS pairs run one point of every antipodal couple with the summed weight.  With the
    switch off every point is run; both agree with the oracle, and with each other far below the tolerance."""
    torch = torch_cuda
    from oracle.collide import collide_pairs
    cfg = _rand_cfg("t", 2, 16, 3, 32, (1.0, 1.0), (0.6, 0.8), (1.0, 2.0), seed=41)     # unequal weights in the rule
    rng = np.random.default_rng(41)
    f = make_points(cfg, range(cfg.nx)) * (1.0 + 0.3 * rng.uniform(-1, 1, (cfg.nx, 2, 16 ** 3)))
    Qo = collide_pairs(_oracle_tables(cfg), f)
    fd = torch.from_numpy(f).cuda()
    with _gpu_op(cfg) as op:
        Q_on = op.collide_pairs(fd).cpu().numpy()
        fl_on = op.flops_per_pair_eval(0, 0), op.flops_per_pair_eval(0, 1)
    monkeypatch.setenv("DGFS_V1_ANTIPODAL", "0")
    with _gpu_op(cfg) as op:
        Q_off = op.collide_pairs(fd).cpu().numpy()
        fl_off = op.flops_per_pair_eval(0, 0), op.flops_per_pair_eval(0, 1)
    assert _pair_errs(Q_on, Qo).max() < TOL and _pair_errs(Q_off, Qo).max() < TOL
    assert _pair_errs(Q_on, Q_off).max() < 1e-12
    assert fl_on[0] < 0.62 * fl_off[0] and fl_on[1] == fl_off[1]          # only the diagonal pair gets cheaper


@pytest.mark.parametrize("N,alpha,M", [(16, (1.0, 1.0), 12), (8, (1.0, 1.3), 6), (32, (1.0, 1.0), 12), (48, (1.0, 1.0), 6)])
def test_nyquist_filter_mode(torch_cuda, N, alpha, M):
    """dgfs_params.nyquist_filter = 1: Q(P f_p, P f_q); the oracle filters the inputs spectrally and runs
    Algorithm 2 unchanged, the library filters in physical space and skips its Nyquist-field kernels."""
    torch = torch_cuda
    from oracle.collide import collide_pairs, nyquist_filter
    cfg = _rand_cfg("t", 2, N, 2, M, alpha, (0.6, 0.8), (1.0, 2.0), seed=77 + N)
    rng = np.random.default_rng(N)
    f = make_points(cfg, range(cfg.nx)) * (1.0 + 0.3 * rng.uniform(-1, 1, (cfg.nx, 2, N ** 3)))
    Qo = collide_pairs(_oracle_tables(cfg), nyquist_filter(f, N))
    with _gpu_op(cfg, nyquist_filter=True) as op:
        Qg = op.collide_pairs(torch.from_numpy(f).cuda()).cpu().numpy()
    with _gpu_op(cfg) as op:
        Qu = op.collide_pairs(torch.from_numpy(f).cuda()).cpu().numpy()
    assert _pair_errs(Qg, Qo).max() < TOL
    assert _pair_errs(Qu, Qo).max() > 1e-6            # the unfiltered operator is a different one on rough inputs


def test_v1_user_sphere_rule_without_symmetry(torch_cuda):
    """A caller-supplied sigma set with no shared sigma_z values (every z shift is its own job)."""
    torch = torch_cuda
    from oracle.collide import collide_pairs
    rng = np.random.default_rng(5)
    M = 7
    sig = rng.normal(size=(M, 3)); sig /= np.linalg.norm(sig, axis=1)[:, None]
    w = rng.uniform(0.5, 1.5, M); w *= 4 * np.pi / w.sum()
    cfg = _rand_cfg("t", 2, 16, 3, M, (1.0, 1.0), (0.5, 0.9), (1.0, 3.0), seed=21)
    f = make_points(cfg, range(cfg.nx)) * (1.0 + 0.2 * rng.uniform(-1, 1, (cfg.nx, 2, 16 ** 3)))
    Qo = collide_pairs(_oracle_tables(cfg, sigma=sig, w_sigma=w), f)
    with _gpu_op(cfg, sigma=sig, w_sigma=w) as op:
        Qg = op.collide_pairs(torch.from_numpy(f).cuda()).cpu().numpy()
    assert _pair_errs(Qg, Qo).max() < TOL


def _small_radial_rule(torch_cuda, N, N_rho, M, ns, alpha, noise=0.05):
    torch = torch_cuda
    from oracle.collide import collide_pairs
    masses = (1.0, 2.5, 1.7)[:ns]
    omega = (0.5, 0.81, 0.7)[:ns]
    cfg = _rand_cfg("t", ns, N, N_rho, M, alpha, omega, masses, seed=1000 + N)
    f = make_points(cfg, range(cfg.nx))
    # make the input rough (exercises the Nyquist planes / complex path)
    rng = np.random.default_rng(N)
    f *= 1.0 + noise * rng.uniform(-1, 1, f.shape)
    Qo = collide_pairs(_oracle_tables(cfg), f)
    with _gpu_op(cfg) as op:
        Qg = op.collide_pairs(torch.from_numpy(f).cuda()).cpu().numpy()
    errs = _pair_errs(Qg, Qo)
    assert errs.max() < TOL, errs


# ------------------------------------------------------------------------------------------- tables
@pytest.mark.parametrize("N,alpha,table_mode", [(8, (1.0, 1.0), 0), (8, (1.0, 1.4), 0), (16, (1.3, 1.2), 0),
                                                (8, (1.0, 1.4), 1), (24, (1.0, 1.25), 0)])
def test_tables_match_oracle(torch_cuda, N, alpha, table_mode):
    from oracle.quadrature import sphere_rule
    cfg = _rand_cfg("t", 2, N, 4, 12, alpha, (0.6, 0.8), (1.0, 2.0), seed=5)
    kw = {}
    if table_mode == 1:
        sp, wp = sphere_rule(32)
        kw = dict(table_mode=1, sigma_pre=sp, w_pre=wp)
    # the same sphere points in the same order on both sides (inputs, not results)
    sig, wsig = sphere_rule(cfg.M)
    tab = _oracle_tables(cfg, sigma=sig, w_sigma=wsig, **kw)
    with _gpu_op(cfg, sigma=sig, w_sigma=wsig, **kw) as op:
        quad = op.quadrature()
        assert abs(quad["R"] - tab.R) < 1e-14 * tab.R
        np.testing.assert_allclose(quad["rho"], tab.rho, rtol=1e-13, atol=0)
        np.testing.assert_allclose(quad["w_rho"], tab.w_rho, rtol=1e-13, atol=0)
        np.testing.assert_allclose(quad["beta"], tab.beta, rtol=1e-13, atol=0)
        for p in range(2):
            for q in range(2):
                a, b, c = op.tables(p, q)
                assert np.max(np.abs(a - tab.a)) < 1e-13 * np.max(np.abs(tab.a))
                assert np.max(np.abs(b - tab.b[p, q])) < 1e-13 * np.max(np.abs(tab.b[p, q])), (p, q)
                assert np.max(np.abs(c - tab.c[p, q])) < 1e-13 * np.max(np.abs(tab.c[p, q])), (p, q)


def test_builtin_sphere_rules_are_the_oracles_point_sets(torch_cuda):
    from oracle.quadrature import sphere_rule
    for M in (6, 12, 32):
        cfg = _rand_cfg("t", 1, 8, 2, M, (1.0,), (0.5,), (1.0,), seed=5)
        with _gpu_op(cfg) as op:
            quad = op.quadrature()
        sig, w = sphere_rule(M)
        key = lambda s, ww: sorted((round(x, 12), round(y, 12), round(z, 12), round(v, 12)) for (x, y, z), v in zip(s, ww))
        assert key(quad["sigma"], quad["w_sigma"]) == key(sig, w)


# ----------------------------------------------------------------------- edge cases of the boundary
def test_empty_batch_and_argument_errors(torch_cuda):
    torch = torch_cuda
    from paper_1903_04670_b200 import api
    cfg = get_config("c0")
    with _gpu_op(cfg) as op:
        f = torch.zeros((1, cfg.ns, cfg.N ** 3), dtype=torch.float64, device="cuda")
        Q = torch.full_like(f, 7.0)
        api.dgfs_collide(op.ctx, f, Q, 0)                 # nx = 0: no-op
        torch.cuda.synchronize()
        assert float(Q.min()) == 7.0
        with pytest.raises(api.DgfsError) as e:
            api.dgfs_collide(op.ctx, f, f, 1)             # aliasing
        assert e.value.code == api.DGFS_EINVAL
        with pytest.raises(api.DgfsError):
            api.dgfs_collide(op.ctx, f, Q, -1)
        assert api.load_library().dgfs_collide(op.ctx, None, None, 1, None) == api.DGFS_EINVAL
        op.collide(f, Q)                                   # f = 0 => Q = 0 exactly
        torch.cuda.synchronize()
        assert float(Q.abs().max()) == 0.0
        assert op.workspace_bytes(4) > 0
        op.reserve(4)


def test_single_species_and_single_point(torch_cuda):
    torch = torch_cuda
    from oracle.collide import collide
    cfg = _rand_cfg("t", 1, 16, 5, 12, (1.0,), (1.0,), (1.0,), seed=77)     # Maxwell molecules
    f = make_points(cfg, [0])
    Qo = collide(_oracle_tables(cfg), f)
    with _gpu_op(cfg) as op:
        Qg = op.collide(torch.from_numpy(f).cuda()).cpu().numpy()
    assert np.max(np.abs(Qg - Qo)) < TOL * np.max(np.abs(Qo))


def test_batch_is_consistent_with_single_point_calls_and_chunking(torch_cuda, monkeypatch):
    """Points are independent: a batched call equals per-point calls bit for bit, also when
    the workspace budget forces several chunks and a ragged last chunk."""
    torch = torch_cuda
    cfg = _rand_cfg("t", 2, 16, 3, 6, (1.0, 1.3), (0.6, 0.8), (1.0, 2.0), seed=9)
    f = torch.from_numpy(make_points(cfg, range(7))).cuda()
    with _gpu_op(cfg) as op:
        Qb = op.collide_pairs(f).clone()
        for x in (0, 3, 6):
            Q1 = op.collide_pairs(f[x:x + 1].contiguous())
            assert torch.equal(Q1[0], Qb[x])
    monkeypatch.setenv("DGFS_SCRATCH_MB", "2")       # forces nbx = 1..2 points per chunk
    with _gpu_op(cfg) as op:
        Qc = op.collide_pairs(f)
        assert torch.equal(Qc, Qb)


def test_v1_batch_consistency_and_chunking(torch_cuda, monkeypatch):
    """Same as above for the v1 pipeline (all pairs VHS): chunk of 8 points by default, 3 here, ragged tail."""
    torch = torch_cuda
    cfg = _rand_cfg("t", 2, 16, 3, 12, (1.0, 1.0), (0.6, 0.8), (1.0, 2.0), seed=9)
    f = torch.from_numpy(make_points(cfg, range(11))).cuda()
    with _gpu_op(cfg) as op:
        Qb = op.collide_pairs(f).clone()
        Qs = op.collide(f).clone()
        for x in (0, 7, 8, 10):
            Q1 = op.collide_pairs(f[x:x + 1].contiguous())
            assert torch.equal(Q1[0], Qb[x])
    monkeypatch.setenv("DGFS_V1_CHUNK", "3")
    with _gpu_op(cfg) as op:
        assert torch.equal(op.collide_pairs(f), Qb)
        assert torch.equal(op.collide(f), Qs)


def test_v1_workspace_budget_shrinks_the_launch_group(torch_cuda, monkeypatch):
    """The launch group is halved until its workspace fits the byte budget (70 % of the free memory at create, or
    DGFS_V1_WS_GB); the result does not change by a bit."""
    torch = torch_cuda
    cfg = _rand_cfg("t", 2, 16, 3, 12, (1.0, 1.0), (0.6, 0.8), (1.0, 2.0), seed=9)
    f = torch.from_numpy(make_points(cfg, range(40))).cuda()
    with _gpu_op(cfg) as op:
        big = op.workspace_bytes(40)
        Qb = op.collide_pairs(f).clone()
    monkeypatch.setenv("DGFS_V1_WS_GB", "%.9f" % (0.3 * big / 1e9))
    with _gpu_op(cfg) as op:
        small = op.workspace_bytes(40)
        assert small <= 0.3 * big * 1.3 and small < big
        assert torch.equal(op.collide_pairs(f), Qb)


def test_k_wterm_cluster_multicast_variant_is_bit_equal(torch_cuda, monkeypatch):
    """DGFS_V1_WTERM_MC=1 (N = 32): k_wterm as clusters of four blocks, the uy plane of a sphere point fetched once per
    item by a TMA multicast (measured slower than the default, profiles/r02_wterm.md; kept as a switch): same sums in
    the same order, so the results equal the default's bit for bit; white-noise inputs so that the Nyquist fields count."""
    torch = torch_cuda
    cfg = _rand_cfg("t", 2, 32, 3, 12, (1.0, 1.0), (0.6, 0.8), (1.0, 2.0), seed=23)
    rng = np.random.default_rng(5)
    f = make_points(cfg, range(6)) * (1.0 + 0.4 * rng.uniform(-1, 1, (6, cfg.ns, cfg.N ** 3)))
    fd = torch.from_numpy(f).cuda()
    with _gpu_op(cfg) as op:
        Q0 = op.collide_pairs(fd).clone()
    monkeypatch.setenv("DGFS_V1_WTERM_MC", "1")
    with _gpu_op(cfg) as op:
        Q1 = op.collide_pairs(fd).clone()
        Q2 = op.collide_pairs(fd)
        assert torch.equal(Q1, Q0) and torch.equal(Q2, Q0)


def test_v1_mixed_pairs_batch_consistency_and_chunking(torch_cuda, monkeypatch):
    """3 species, pair (0,0) VHS and the other eight VSS in one context: the two kinds share the z shifts and
    the Nyquist fields and take different kernels afterwards; chunking must not change a bit."""
    torch = torch_cuda
    cfg = _rand_cfg("t", 3, 8, 3, 12, (1.0, 1.2, 1.4), (0.5, 0.7, 0.8), (1.0, 1.5, 2.0), seed=12)
    f = torch.from_numpy(make_points(cfg, range(7))).cuda()
    with _gpu_op(cfg) as op:
        Qb = op.collide_pairs(f).clone()
        Qs = op.collide(f).clone()
        Q1 = op.collide_pairs(f[5:6].contiguous())
        assert torch.equal(Q1[0], Qb[5])
    monkeypatch.setenv("DGFS_V1_CHUNK", "3")
    with _gpu_op(cfg) as op:
        assert torch.equal(op.collide_pairs(f), Qb)
        assert torch.equal(op.collide(f), Qs)


def test_output_on_side_stream_and_repeatability(torch_cuda):
    torch = torch_cuda
    cfg = get_config("c0")
    f = torch.from_numpy(make_points(cfg, range(cfg.nx))).cuda()
    with _gpu_op(cfg) as op:
        Q0 = op.collide(f).clone()
        s = torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            Q1 = op.collide(f)
        s.synchronize()
        assert torch.equal(Q0, Q1)


def test_host_buffer_call_matches_device_call(torch_cuda):
    """dgfs_collide_host (HOST pointers, slabs pipelined on the library's streams) == dgfs_collide."""
    torch = torch_cuda
    cfg = get_config("c0")
    xs = [i % cfg.nx for i in range(37)]          # ragged against any slab size
    f = make_points(cfg, xs)
    with _gpu_op(cfg) as op:
        Qd = op.collide(torch.from_numpy(f).cuda()).cpu().numpy()
        Qh = op.collide_host(f)                                    # numpy, pageable
        fh = torch.from_numpy(f).pin_memory()
        Qp = op.collide_host(fh, torch.empty_like(fh).pin_memory()).numpy()   # pinned torch
        from paper_1903_04670_b200 import DgfsError
        with pytest.raises(ValueError):
            op.collide_host(f.astype(np.float32))
    assert np.array_equal(Qd, Qh) and np.array_equal(Qd, Qp)


def test_fp64_peak_probe_is_plausible(torch_cuda):
    from paper_1903_04670_b200 import dgfs_measure_fp64_peak
    burst, sustained = dgfs_measure_fp64_peak(0, 0.2)
    assert 5.0 < sustained <= burst < 60.0


# ------------------------------------------------------------------ symmetry-compressed full b tables
@pytest.mark.parametrize("N,M,pipeline", [(8, 12, "v1"), (8, 32, "v1"), (16, 12, "v0"), (24, 12, "v1")])
def test_full_b_tables_stored_per_orbit_of_the_sphere_rule(torch_cuda, monkeypatch, N, M, pipeline):
    """b_rs(k) of a VSS pair depends on k through |k| and k . sigma_s only (Eq. 16), so the
    library stores one table per orbit of the sphere rule under the signed axis permutations that keep y in place
    (icosahedron: 3 of 12, 32-point rule: 7 of 32) on the extended grid.  Same table values as the oracle's _b_exact (1e-13), same Q as the
    paper's layout [N_rho][M][N^3] (DGFS_BTABLE=full) and as the oracle (1e-10), a fraction of the bytes."""
    torch = torch_cuda
    from oracle.collide import collide_pairs
    if pipeline == "v0":
        monkeypatch.setenv("DGFS_PIPELINE", "v0")
    from oracle.quadrature import sphere_rule
    cfg = _rand_cfg("t", 2, N, 2, M, (1.2, 1.45), (0.6, 0.8), (1.0, 2.0), seed=21)
    f = make_points(cfg, range(2))
    sig, wsig = sphere_rule(M)          # the same sphere points in the same order on both sides (inputs, not results)
    tab = _oracle_tables(cfg, sigma=sig, w_sigma=wsig)
    Qo = collide_pairs(tab, f)
    res = {}
    for mode in ("sym", "full"):
        monkeypatch.setenv("DGFS_BTABLE", mode)
        with _gpu_op(cfg, sigma=sig, w_sigma=wsig) as op:
            Q = op.collide_pairs(torch.from_numpy(f).cuda()).cpu().numpy()
            b01 = op.tables(0, 1)[1]
            res[mode] = (Q, b01, op.table_bytes())
        assert _pair_errs(Q, Qo).max() < TOL, mode
        assert np.max(np.abs(b01 - tab.b[0, 1])) < 1e-13 * np.max(np.abs(tab.b[0, 1])), mode
    orbits = {12: 3, 32: 7}[M]        # orbits under sign flips and the x <-> z swap (the ky index stays the fastest)
    assert res["full"][2] == 4 * cfg.N_rho * M * N ** 3 * 16
    assert res["sym"][2] == 4 * cfg.N_rho * orbits * (N + 1) ** 3 * 16
    assert _pair_errs(res["sym"][0], res["full"][0]).max() < 1e-12


def test_full_b_tables_of_a_rule_without_symmetry_stay_in_full(torch_cuda):
    """A rotated sphere rule has no two points related by a signed axis permutation: nothing to share."""
    torch = torch_cuda
    from oracle.quadrature import sphere_rule
    from oracle.collide import collide_pairs
    sig, w = sphere_rule(12)
    th = 0.3
    Rz = np.array([[np.cos(th), -np.sin(th), 0], [np.sin(th), np.cos(th), 0], [0, 0, 1.0]])
    Rx = np.array([[1.0, 0, 0], [0, np.cos(0.7), -np.sin(0.7)], [0, np.sin(0.7), np.cos(0.7)]])
    sig = sig @ (Rz @ Rx).T
    sig /= np.linalg.norm(sig, axis=1)[:, None]
    cfg = _rand_cfg("t", 2, 8, 2, 12, (1.3, 1.3), (0.6, 0.8), (1.0, 2.0), seed=22)
    f = make_points(cfg, range(2))
    Qo = collide_pairs(_oracle_tables(cfg, sigma=sig, w_sigma=w), f)
    with _gpu_op(cfg, sigma=sig, w_sigma=w) as op:
        Q = op.collide_pairs(torch.from_numpy(f).cuda()).cpu().numpy()
        assert op.table_bytes() >= 4 * cfg.N_rho * 6 * 8 ** 3 * 16      # antipodes may still pair up, nothing more
    assert _pair_errs(Q, Qo).max() < TOL


# ------------------------------------------------------------------ dgfs_params.precision = 1 (fp32 inner loop)
@pytest.mark.parametrize("N,N_rho,M", [(8, 4, 6), (16, 3, 12), (24, 3, 12), (32, 3, 12), (32, 2, 32)])
def test_precision_1_within_1e_4_on_non_equilibrium_inputs(torch_cuda, N, N_rho, M):
    """SURVEY 8(f) item 1 / north_star "1e-4 if an fp32 mode is offered": steps 4-6 of Algorithm 2 in fp32, the rest in
    fp64, against the SAME fp64 oracle at 1e-4 of max|Q| per (point, pair) array on bi-Maxwellian inputs."""
    torch = torch_cuda
    from oracle.collide import collide_pairs
    from oracle_pool import record
    cfg = _rand_cfg("t", 2, N, N_rho, M, (1.0, 1.0), (0.6, 0.8), (1.0, 2.0), seed=31)
    f = make_points(cfg, range(3))
    Qo = collide_pairs(_oracle_tables(cfg), f)
    with _gpu_op(cfg, precision=1) as op:
        fd = torch.from_numpy(f).cuda()
        Qg = op.collide_pairs(fd).cpu().numpy()
        Qs = op.collide(fd).cpu().numpy()
    err = _pair_errs(Qg, Qo).max()
    record("fp32", "N=%d N_rho=%d M=%d, bi-Maxwellian inputs, all pairs" % (N, N_rho, M), err, 1e-4)
    assert err < 1e-4
    Qos = Qo.sum(axis=2)
    assert (np.max(np.abs(Qs - Qos), axis=-1) / np.max(np.abs(Qos), axis=-1)).max() < 1e-4


def test_precision_1_is_refused_where_it_is_not_implemented(torch_cuda):
    from paper_1903_04670_b200 import api
    vss = _rand_cfg("t", 2, 8, 2, 6, (1.0, 1.3), (0.6, 0.8), (1.0, 2.0), seed=1)
    with pytest.raises(api.DgfsError) as e:
        _gpu_op(vss, precision=1)
    assert e.value.code == api.DGFS_ENOSUP
    big = _rand_cfg("t", 2, 48, 1, 6, (1.0, 1.0), (0.6, 0.8), (1.0, 2.0), seed=1)
    with pytest.raises(api.DgfsError) as e:
        _gpu_op(big, precision=1)
    assert e.value.code == api.DGFS_ENOSUP
    with pytest.raises(api.DgfsError) as e:
        _gpu_op(vss, precision=2)
    assert e.value.code == api.DGFS_EINVAL


@pytest.mark.parametrize("N", [8, 24, 48])
def test_dft_probe_both_methods_compute_the_dft(torch_cuda, N):
    """dgfs_measure_dft (the FFT-vs-tensor-core evidence of DESIGN.md section 8): each method's transform of the probe
    input equals the direct sum (evaluated on the host inside the library) to round-off, and a rate comes back."""
    from oracle_pool import record
    from paper_1903_04670_b200 import dgfs_measure_dft
    rates = []
    for method in (0, 1):
        rate, err = dgfs_measure_dft(0, N, method, 0.2)
        assert err < 1e-12 and rate > 0, (method, rate, err)
        rates.append(rate)
    record("dft-probe", "N=%d: register FFT %.3e DFT/s, FP64 mma.sync m8n8k4 %.3e DFT/s, ratio" % (N, rates[0], rates[1]),
           rates[0] / rates[1], 1.0)


def test_fp64_mix_probe_dfma_and_dmma_share_one_pipe(torch_cuda):
    """dgfs_measure_fp64_mix: both kinds of FP64 instruction reach the pipe's rate alone; issued side by side their
    rates do not add up to more than one pipe's worth (they would, up to ~2x, on separate pipes).  The figures go to the
    log (profiles/r02_dft_probe.md); asserted loosely: the combined rate stays below 1.3x the better pure rate."""
    from oracle_pool import record
    from paper_1903_04670_b200 import dgfs_measure_fp64_mix, DgfsError
    f_only, _ = dgfs_measure_fp64_mix(0, 8, 0, 0.2)
    _, m_only = dgfs_measure_fp64_mix(0, 0, 8, 0.2)
    f_mix, m_mix = dgfs_measure_fp64_mix(0, 8, 8, 0.2)
    f_mix2, m_mix2 = dgfs_measure_fp64_mix(0, 8, 2, 0.2)
    print("fp64 mix: DFMA alone %.2f, DMMA alone %.2f, mixed 8+8: %.2f + %.2f, mixed 8+2: %.2f + %.2f TFLOP/s" % (
        f_only, m_only, f_mix, m_mix, f_mix2, m_mix2))
    assert f_only > 10.0 and m_only > 10.0
    for f, m in ((f_mix, m_mix), (f_mix2, m_mix2)):
        record("fp64-mix", "DFMA %.2f + DMMA %.2f TFLOP/s side by side, sum / better pure rate" % (f, m),
               (f + m) / max(f_only, m_only), 1.3)
        assert f + m < 1.3 * max(f_only, m_only)
    with pytest.raises(DgfsError):
        dgfs_measure_fp64_mix(0, 3, 5, 0.1)


def test_calls_on_two_streams_of_one_context_do_not_race(torch_cuda):
    """The workspace belongs to one call at a time: a call on another stream, issued without any host or stream
    synchronisation, waits for the previous call's last launch (include/dgfs.h: calls on one context are ordered)."""
    torch = torch_cuda
    cfg = _rand_cfg("t", 2, 16, 3, 12, (1.0, 1.0), (0.6, 0.8), (1.0, 2.0), seed=41)
    fa = torch.from_numpy(make_points(cfg, range(24))).cuda()
    fb = torch.from_numpy(make_points(cfg, range(24, 48))).cuda()
    with _gpu_op(cfg) as op:
        Qa0, Qb0 = op.collide(fa).clone(), op.collide(fb).clone()
        torch.cuda.synchronize()
        sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
        Qa, Qb = torch.empty_like(fa), torch.empty_like(fb)
        for _ in range(3):
            with torch.cuda.stream(sa):
                op.collide(fa, Qa)
            with torch.cuda.stream(sb):
                op.collide(fb, Qb)
        torch.cuda.synchronize()
        assert torch.equal(Qa, Qa0) and torch.equal(Qb, Qb0)


def test_two_contexts_on_two_devices(torch_cuda):
    """Kernel attributes (dynamic shared memory opt-in) are set per context, i.e. per device."""
    torch = torch_cuda
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    cfg = get_config("c0")
    f = make_points(cfg, range(cfg.nx))
    outs = []
    for dev in (0, 1):
        with torch.cuda.device(dev):
            from paper_1903_04670_b200 import Dgfs
            with Dgfs.from_config(cfg, device=dev) as op:
                outs.append(op.collide(torch.from_numpy(f).cuda(dev)).cpu())
    assert torch.equal(outs[0], outs[1])

"""Pins for oracle/collide.py (Algo 2): brute-force Galerkin sums (Eq. 11-13), exact discrete
invariants, the shift identity of Eq. 8, and the survey-time golden values."""
import json
import os
from math import pi

import numpy as np
import pytest

from oracle.collide import collide, collide_pair, collide_pairs
from oracle.galerkin import galerkin_exact_vhs, galerkin_lowrank
from oracle.tables import precompute
from workloads import maxwellian, velocity_nodes

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rand_f(N, seed, ns=2):
    rng = np.random.default_rng(seed)
    return rng.random((ns, N ** 3)) + 0.1


def _relerr(a, b):
    return np.max(np.abs(a - b)) / np.max(np.abs(b))


# ---------------------------------------------------------------- X-2: brute-force Galerkin sum
@pytest.mark.parametrize("N,N_rho,M,alpha", [
    (4, 3, 6, 1.0), (6, 4, 12, 1.0), (4, 3, 12, 1.4), (6, 2, 6, 1.25)])
def test_algo2_equals_wrapped_galerkin_sum(N, N_rho, M, alpha):
    """Algo 2 (FFT convolutions) == Eq. 11 with Eq. 13 inserted, index sums mod N, same tables."""
    tab = precompute(N, N_rho, M, 5.0, [1.0, 2.0], [[0.5, 0.7], [0.7, 0.8]], [[alpha] * 2] * 2)
    f = _rand_f(N, 7)
    for p in range(2):
        for q in range(2):
            fast = collide_pair(tab, p, q, f[p], f[q])
            brute = galerkin_lowrank(tab, p, q, f[p], f[q], wrap=True)
            assert _relerr(fast, brute) < 1e-12, (p, q)


def test_wraparound_is_the_only_difference_to_literal_eq11():
    """X-2b: on inputs band-limited to |l_d| < N/4 the literal (unwrapped) Eq. 11 equals Algo 2;
    on full-band inputs it does not."""
    N = 8
    tab = precompute(N, 3, 6, 5.0, [1.0, 2.0], [[0.5, 0.7], [0.7, 0.8]], [[1.0, 1.0], [1.0, 1.0]])
    f = _rand_f(N, 11)
    v = np.round(np.fft.fftfreq(N) * N)
    keep = (np.abs(v) < N // 4)
    mask = keep[:, None, None] & keep[None, :, None] & keep[None, None, :]
    fb = np.empty_like(f)
    for p in range(2):
        fb[p] = np.real(np.fft.ifftn(np.fft.fftn(f[p].reshape(N, N, N)) * mask)).reshape(-1)
    p, q = 0, 1
    fast = collide_pair(tab, p, q, fb[p], fb[q])
    lit = galerkin_lowrank(tab, p, q, fb[p], fb[q], wrap=False)
    assert _relerr(fast, lit) < 1e-12
    fast_full = collide_pair(tab, p, q, f[p], f[q])
    lit_full = galerkin_lowrank(tab, p, q, f[p], f[q], wrap=False)
    assert _relerr(fast_full, lit_full) > 1e-3


def test_lowrank_converges_to_full_kernel_modes():
    """X-2c: against Eq. 11 with the full, non-low-rank G+(l,m), G-(m) of Eq. 12 (VHS) the fast
    algorithm differs by the quadrature error of Eq. 13, which falls with M and N_rho."""
    N, L = 6, 5.0
    c = velocity_nodes(N, L)
    f = np.stack([maxwellian(N, L, 1.0, (0.2, -0.1, 0.3), 1.0, 1.0),
                  maxwellian(N, L, 0.8, (-0.1, 0.2, 0.0), 1.5, 2.0)])
    errs = {}
    ref = None
    for (N_rho, M) in [(3, 6), (6, 6), (6, 12), (12, 32)]:
        tab = precompute(N, N_rho, M, L, [1.0, 2.0], [[0.5] * 2] * 2, [[1.0] * 2] * 2)
        if ref is None:
            ref = galerkin_exact_vhs(tab, 0, 1, f[0], f[1], wrap=True)
        errs[(N_rho, M)] = _relerr(collide_pair(tab, 0, 1, f[0], f[1]), ref)
    assert errs[(12, 32)] < errs[(6, 12)] < errs[(6, 6)]
    assert errs[(12, 32)] < 1e-3
    assert errs[(6, 12)] < 2e-2


# ---------------------------------------------------------------- X-6: exact invariants
@pytest.fixture(scope="module")
def tab8():
    return precompute(8, 4, 12, 5.0, [1.0, 2.0], [[0.5, 0.7], [0.7, 0.8]], [[1.0, 1.3], [1.3, 1.0]])


def test_circular_shift_equivariance(tab8):
    N = 8
    f = _rand_f(N, 3)
    sh = (1, 2, 3)
    fs = np.stack([np.roll(f[p].reshape(N, N, N), sh, axis=(0, 1, 2)).reshape(-1) for p in range(2)])
    for (p, q) in [(0, 1), (1, 0), (1, 1)]:
        Q = collide_pair(tab8, p, q, f[p], f[q]).reshape(N, N, N)
        Qs = collide_pair(tab8, p, q, fs[p], fs[q]).reshape(N, N, N)
        assert _relerr(Qs, np.roll(Q, sh, axis=(0, 1, 2))) < 1e-13


def test_cyclic_axis_permutation_equivariance(tab8):
    """The sphere sets of S-2 are invariant under (x,y,z) -> (y,z,x)."""
    N = 8
    f = _rand_f(N, 4)
    fp = np.stack([f[p].reshape(N, N, N).transpose(1, 2, 0).reshape(-1) for p in range(2)])
    Q = collide_pair(tab8, 0, 1, f[0], f[1]).reshape(N, N, N)
    Qp = collide_pair(tab8, 0, 1, fp[0], fp[1]).reshape(N, N, N)
    assert _relerr(Qp, Q.transpose(1, 2, 0)) < 1e-13


def test_bilinearity(tab8):
    f, g = _rand_f(8, 5), _rand_f(8, 6)
    Q1 = collide_pair(tab8, 0, 1, f[0], f[1])
    Q2 = collide_pair(tab8, 0, 1, 2.5 * f[0], -0.5 * f[1])
    assert _relerr(Q2, -1.25 * Q1) < 1e-13
    Q3 = collide_pair(tab8, 0, 1, f[0] + g[0], f[1])
    assert _relerr(Q3, Q1 + collide_pair(tab8, 0, 1, g[0], f[1])) < 1e-13


def test_pair_mass_exchange_symmetry():
    """sum_c Q_pq = sum_c Q_qp exactly for beta = 1, symmetric omega/alpha and an antipodal sigma set
    (the k = 0 mode of gain and loss is symmetric under (p,l) <-> (q,m))."""
    tab = precompute(8, 4, 12, 5.0, [1.0, 2.0], [[0.5, 0.7], [0.7, 0.8]], [[1.0, 1.3], [1.3, 1.0]],
                     beta_override=[[1.0, 1.0], [1.0, 1.0]])
    f = _rand_f(8, 8)
    s01 = collide_pair(tab, 0, 1, f[0], f[1]).sum()
    s10 = collide_pair(tab, 1, 0, f[1], f[0]).sum()
    assert abs(s01 - s10) < 1e-12 * abs(s01)


def test_collide_sums_pairs_with_beta(tab8):
    f = _rand_f(8, 9)[None]
    Qpq = collide_pairs(tab8, f)
    Q = collide(tab8, f)
    assert Qpq.shape == (1, 2, 2, 512) and Q.shape == (1, 2, 512)
    un = collide_pair(tab8, 0, 1, f[0, 0], f[0, 1], scale_beta=False)
    assert _relerr(Qpq[0, 0, 1], tab8.beta[0, 1] * un) < 1e-15
    assert _relerr(Q[0, 1], Qpq[0, 1, 0] + Qpq[0, 1, 1]) < 1e-15


# ---------------------------------------------------------------- X-7: shift identity (Eq. 8)
def test_phase_modulation_is_a_shift():
    """ifft(e^{i mu a_rs} fft(f)) is the trigonometric interpolant of f at c + mu rho_r sigma_s:
    exact for a single Fourier mode below Nyquist.  Fixes the sign conventions of steps 4-5."""
    N, L = 8, 5.0
    tab = precompute(N, 3, 12, L, [1.0, 2.0], [[0.5] * 2] * 2, [[1.0] * 2] * 2)
    c = velocity_nodes(N, L)
    k = np.array([1.0, -2.0, 3.0])
    cx, cy, cz = np.meshgrid(c, c, c, indexing="ij")
    mode = lambda X, Y, Z: np.exp(1j * pi / L * (k[0] * X + k[1] * Y + k[2] * Z))
    f = mode(cx, cy, cz)
    mu = 2.0 / 3.0
    for (r, s) in [(0, 0), (2, 5), (1, 11)]:
        d = mu * tab.rho[r] * tab.sigma[s]
        shifted = np.fft.ifftn(np.exp(1j * mu * tab.a[r, s].reshape(N, N, N)) * np.fft.fftn(f))
        assert np.max(np.abs(shifted - mode(cx + d[0], cy + d[1], cz + d[2]))) < 1e-13
        back = np.fft.ifftn(np.exp(-1j * mu * tab.a[r, s].reshape(N, N, N)) * np.fft.fftn(f))
        assert np.max(np.abs(back - mode(cx - d[0], cy - d[1], cz - d[2]))) < 1e-13


# ---------------------------------------------------------------- X-1: golden values
# Independent numpy implementation written at survey time and validated there against the
# brute-force sum and Table 1; inputs are closed-form Maxwellians.
_A3 = {
    "G0": {  # VHS omega = 0.5, alpha = 1
        (0, 0): (0.05626976975981913, 0.37420910471961744, 0.10635258505705569, 0.01512306014772609,
                 7.89752035578687e-06, 3.2866573159273056),
        (0, 1): (0.06497473343613969, 1.014331286771163, -0.4622803004338871, 0.021951144256563804,
                 -1.1574742862086577e-06, -3.3192767191159387),
        (1, 0): (0.045944074618482676, 0.6329637974841061, 0.09518194940371572, -0.009978298881149565,
                 7.501814366665447e-07, -3.31927671911594),
        (1, 1): (0.05626976975981913, 0.25619222441700495, -0.1386722065535564, 0.04051558653370373,
                 -2.7685378115135695e-06, -0.01965156646431261),
    },
    "G1": {  # VSS omega = 0.8, alpha = 1.4
        (0, 0): (0.08089262497771565, 0.2330215635618067, 0.05318086941009237, 0.00720440450618837,
                 3.821038017989679e-06, 1.495501578068615),
        (0, 1): (0.08568339694141708, 0.6283941677248353, -0.2771925091581886, 0.0045416351432029265,
                 -3.816391364637738e-07, -1.8144503939770453),
        (1, 0): (0.060587311012374696, 0.40997573469107806, 0.05780797649586811, -0.002128170385060322,
                 5.464765236968017e-07, -1.8144503939770484),
        (1, 1): (0.06570522848569581, 0.15122877583594058, -0.090038651431743, 0.020180515482553254,
                 -1.3254223560247387e-06, -0.1556965431704652),
    },
}


def _a3_inputs():
    N, L = 8, 5.0
    f0 = maxwellian(N, L, 1.0, (0.2, -0.1, 0.3), 1.0, 1.0)
    f1 = maxwellian(N, L, 0.8, (-0.1, 0.2, 0.0), 1.5, 2.0)
    return N, L, [f0, f1]


@pytest.mark.parametrize("case,omega,alpha", [("G0", 0.5, 1.0), ("G1", 0.8, 1.4)])
def test_survey_golden_values(case, omega, alpha):
    N, L, f = _a3_inputs()
    assert abs(f[0][(4 * 8 + 4) * 8 + 4] - 0.07974112500017586) < 1e-16
    assert abs(f[1][(4 * 8 + 4) * 8 + 4] - 0.05124100075479413) < 1e-16
    tab = precompute(N, 8, 6, L, [1.0, 2.0], [[omega] * 2] * 2, [[alpha] * 2] * 2)
    assert abs(tab.R - 3.7045835599744903) < 1e-15
    for (p, q), (beta, qmax, q444, q352, q0, qsum) in _A3[case].items():
        assert abs(tab.beta[p, q] - beta) < 1e-15
        Q = collide_pair(tab, p, q, f[p], f[q], scale_beta=False)
        tol = 1e-11 * qmax
        assert abs(np.abs(Q).max() - qmax) < tol
        assert abs(Q[(4 * 8 + 4) * 8 + 4] - q444) < tol
        assert abs(Q[(3 * 8 + 5) * 8 + 2] - q352) < tol
        assert abs(Q[0] - q0) < tol
        assert abs(Q.sum() * 1.25 ** 3 - qsum) < 1e-11 * abs(qsum) + tol


def test_stored_golden_file_matches_oracle():
    """tests/golden/oracle_c0.json is written by tests/golden/make_golden.py (calls only oracle/);
    it is the stored expected output for config c0 used by the GPU smoke/parity checks."""
    path = os.path.join(GOLD, "oracle_c0.json")
    if not os.path.exists(path):
        pytest.skip("golden file not generated")
    from workloads import get_config, make_points
    gold = json.load(open(path))
    cfg = get_config("c0")
    tab = precompute(cfg.N, cfg.N_rho, cfg.M, cfg.L, cfg.mass, cfg.omega, cfg.alpha)
    f = make_points(cfg, range(cfg.nx))
    Qpq = collide_pairs(tab, f)
    for ent in gold["samples"]:
        x, p, q, z = ent["x"], ent["p"], ent["q"], ent["z"]
        assert abs(Qpq[x, p, q, z] - ent["Q"]) <= 1e-13 * gold["maxabs"][x][p][q]


def test_nyquist_filter_is_the_projection_it_claims():
    """oracle.collide.nyquist_filter (variant of SURVEY 8(f) item 2): a projection that removes exactly the
    three Nyquist planes; equal to the separable alternating-mean form prod_d (1 - E_d); after it every
    shifted field of Algorithm 2 is real (the reason the variant exists)."""
    from oracle.collide import nyquist_filter
    from oracle.tables import precompute
    N = 8
    rng = np.random.default_rng(3)
    f = rng.uniform(0.1, 1.0, (2, N ** 3))
    Pf = nyquist_filter(f, N)
    assert np.max(np.abs(nyquist_filter(Pf, N) - Pf)) < 1e-14                      # P^2 = P
    g = np.fft.fftn(Pf.reshape(2, N, N, N), axes=(1, 2, 3))
    H = N // 2
    assert max(np.abs(g[:, H]).max(), np.abs(g[:, :, H]).max(), np.abs(g[:, :, :, H]).max()) < 1e-12
    g0 = np.fft.fftn(f.reshape(2, N, N, N), axes=(1, 2, 3))
    keep = np.ones((N, N, N), bool); keep[H] = False; keep[:, H] = False; keep[:, :, H] = False
    assert np.max(np.abs((g - g0)[:, keep])) < 1e-12                               # the other modes are untouched
    # separable physical-space form: (1 - E_d) f = f - (-1)^c mean((-1)^c f) along each axis
    h = f.reshape(2, N, N, N).copy()
    sg = (-1.0) ** np.arange(N)
    for ax in (1, 2, 3):
        shp = [1, 1, 1, 1]; shp[ax] = N
        s = sg.reshape(shp)
        h = h - s * np.mean(s * h, axis=ax, keepdims=True)
    assert np.max(np.abs(h.reshape(2, -1) - Pf)) < 1e-14
    # shifted fields of filtered inputs are real
    tab = precompute(N, 3, 6, 5.0, (1.0, 2.0), ((0.5, 0.5), (0.5, 0.5)), ((1.0, 1.0), (1.0, 1.0)))
    FT = np.fft.fftn(Pf[0].reshape(N, N, N))
    for r in range(3):
        for s_ in range(6):
            A = np.fft.ifftn(np.exp(1j * 0.4 * tab.a[r, s_].reshape(N, N, N)) * FT)
            assert np.abs(A.imag).max() < 1e-13 * np.abs(A.real).max()

"""Pins for oracle/quadrature.py and oracle/tables.py (Algo 1, Eq. 5, 6, 9, 16, 17).
Each check compares the oracle with something fixed by the paper or by mathematics, not with itself."""
import os
from math import gamma as Gamma, pi, sqrt

import numpy as np
import pytest

from oracle.quadrature import gauss_legendre_0R, sphere_rule
from oracle.tables import (C_eta, freq_grid, freq_index, knudsen, precompute, prefactor_beta,
                           truncation_radius)

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _sphere_monomial(a, b, c):
    """Exact int_{S^2} x^a y^b z^c dS: 0 if any exponent is odd, else
    2 Gamma((a+1)/2) Gamma((b+1)/2) Gamma((c+1)/2) / Gamma((a+b+c+3)/2)."""
    if a % 2 or b % 2 or c % 2:
        return 0.0
    return 2.0 * Gamma((a + 1) / 2) * Gamma((b + 1) / 2) * Gamma((c + 1) / 2) / Gamma((a + b + c + 3) / 2)


@pytest.mark.parametrize("M,degree", [(6, 3), (12, 5), (32, 9)])
def test_sphere_rule_exactness(M, degree):
    sig, w = sphere_rule(M)
    assert sig.shape == (M, 3)
    assert np.allclose(np.linalg.norm(sig, axis=1), 1.0, atol=1e-15)
    assert abs(w.sum() - 4 * pi) < 1e-13
    for a in range(degree + 1):
        for b in range(degree + 1 - a):
            for c in range(degree + 1 - a - b):
                q = (w * sig[:, 0] ** a * sig[:, 1] ** b * sig[:, 2] ** c).sum()
                assert abs(q - _sphere_monomial(a, b, c)) < 1e-13, (a, b, c)
    # the rule is not exact one even degree higher (guards against a too-good-to-be-true bug)
    d = degree + 1
    bad = max(abs((w * sig[:, 0] ** a * sig[:, 1] ** (d - a)).sum() - _sphere_monomial(a, d - a, 0))
              for a in range(0, d + 1, 2))
    assert bad > 1e-3
    # antipodal symmetry (used by the CUDA path's pair sharing; property of the sets of S-2)
    for s in range(M):
        assert np.min(np.linalg.norm(sig + sig[s], axis=1)) < 1e-15


def test_gauss_legendre_polynomial_exactness():
    R = 3.7
    rho, w = gauss_legendre_0R(8, R)
    assert np.all(rho > 0) and np.all(rho < R)
    for k in range(16):                                  # exact to degree 2n-1 = 15
        assert abs((w * rho ** k).sum() - R ** (k + 1) / (k + 1)) < 1e-12 * R ** (k + 1)
    assert abs((w * rho ** 16).sum() - R ** 17 / 17) > 1e-12 * R ** 17


def test_freq_index_matches_fftfreq():
    for N in (4, 6, 8, 24, 32, 48):
        assert np.array_equal(freq_index(N), np.round(np.fft.fftfreq(N) * N).astype(int))
    l = freq_grid(4)
    assert l.shape == (64, 3)
    assert tuple(l[(1 * 4 + 2) * 4 + 3]) == (1.0, -2.0, -1.0)     # z = (ix*N+iy)*N+iz, iz fastest


def test_truncation_radius_equal_mass_classical():
    # Eq. 9 with equal masses reduces to the classical single-species 4L/(3+sqrt 2)
    assert abs(truncation_radius(5.0, [1.0, 1.0]) - 4 * 5.0 / (3 + sqrt(2))) < 1e-15
    # m_a = 2, m_b = 1:  4L / (1 + 8/3 + sqrt 3)
    assert abs(truncation_radius(5.0, [1.0, 2.0]) - 20.0 / (1 + 8 / 3 + sqrt(3))) < 1e-14
    assert abs(truncation_radius(5.0, [2.0, 1.0]) - truncation_radius(5.0, [1.0, 2.0])) == 0.0


def test_knudsen_table2():
    """X-4: Eq. 5 with the printed inputs of Table 2 reproduces the printed Kn to 3 digits."""
    m = {1: 66.3, 2: 139.1}
    d = {(1, 1): 4.11e-10, (1, 2): 4.405e-10, (2, 1): 4.405e-10, (2, 2): 4.7e-10}
    om = {(1, 1): 0.81, (1, 2): 0.805, (2, 1): 0.805, (2, 2): 0.8}
    rows = [ln.split() for ln in open(os.path.join(GOLD, "paper_table2_kn.txt")) if not ln.startswith("#")]
    assert len(rows) == 4
    for p, q, kn_print in rows:
        p, q = int(p), int(q)
        kn = knudsen(m[p], m[q], 1.680e21, d[(p, q)], 1.0, om[(p, q)], 1e-3)
        assert abs(kn - float(kn_print)) < 1.5e-3, (p, q, kn)


def test_prefactor_closed_values():
    # hard spheres, equal unit masses, Kn = 1: 1/sqrt2 * 1 * 1/(4 Gamma(2) pi) = 1/(4 sqrt2 pi)
    assert abs(prefactor_beta(1.0, 1.0, 0.5, 1.0) - 1 / (4 * sqrt(2) * pi)) < 1e-16
    # Maxwell molecules omega = 1, alpha = 1, masses (1, 3): reduced mass 3/4
    b = prefactor_beta(1.0, 3.0, 1.0, 1.0, kn=2.0)
    assert abs(b - 0.5 / sqrt(1 + 1 / 3) / sqrt(0.75) / (4 * Gamma(1.5) * pi)) < 1e-16
    # orientation of the mass ratio: beta_pq != beta_qp for unequal masses
    assert prefactor_beta(1.0, 2.0, 0.5, 1.0) > prefactor_beta(2.0, 1.0, 0.5, 1.0)


def _tab(**kw):
    args = dict(N=6, N_rho=5, M=6, L=5.0, mass=[1.0, 2.0], omega=[[0.5, 0.7], [0.7, 0.8]],
                alpha=[[1.0, 1.0], [1.0, 1.0]])
    args.update(kw)
    return precompute(**args)


def test_table_a_definition():
    tab = _tab()
    l = freq_grid(6)
    r, s, z = 3, 4, (2 * 6 + 5) * 6 + 1
    assert tab.a.shape == (5, 6, 216)
    assert abs(tab.a[r, s, z] - pi / 5.0 * tab.rho[r] * np.dot(l[z], tab.sigma[s])) < 1e-15


def test_table_closed_forms_vhs():
    """X-5 for eta = 0."""
    tab = _tab()
    z0 = 0                                                     # l = 0
    for p in range(2):
        for q in range(2):
            g = tab.gam[p, q]
            assert abs(g - 2 * (1 - [[0.5, 0.7], [0.7, 0.8]][p][q])) < 1e-15         # reading G-1
            b = tab.b[p, q]
            assert np.max(np.abs(b.imag)) == 0.0                                      # real
            assert np.max(np.abs(b - b[:, :1, :])) == 0.0                             # independent of s
            assert np.allclose(b[:, 0, z0], 4 * pi * tab.rho ** (g + 2), rtol=1e-14)  # b(0) = rho^{g+2} C_0
            c = tab.c[p, q]
            assert np.max(np.abs(c.imag)) == 0.0
            assert abs(c[z0].real - 4 * pi * 4 * pi * (tab.w_rho * tab.rho ** (g + 2)).sum()) < 1e-12 * abs(c[z0])
    # integer gamma (omega = 0.5 -> gamma = 1): c(0) = (4 pi)^2 R^4 / 4, the rule being exact
    assert abs(tab.c[0, 0, 0].real - (4 * pi) ** 2 * tab.R ** 4 / 4) < 1e-11 * (4 * pi) ** 2 * tab.R ** 4
    # c depends on (gamma, eta) only, not on the masses
    tab2 = _tab(mass=[3.0, 0.5], R=tab.R)
    assert np.allclose(tab2.c, tab.c, rtol=1e-15, atol=0)
    assert not np.allclose(tab2.b, tab.b, rtol=1e-3)
    # value at a non-zero frequency against the textbook Fourier transform of the unit ball
    # shell: int_{S^2} e^{-i k.u} du = 4 pi sin|k|/|k|
    l = freq_grid(6)
    z = (1 * 6 + 2) * 6 + 3
    kk = np.linalg.norm(l[z])
    mu_q = 2.0 / 3.0
    x = mu_q * pi * tab.rho / 5.0 * kk
    assert np.allclose(tab.b[0, 1, :, 2, z].real, tab.rho ** (tab.gam[0, 1] + 2) * 4 * pi * np.sin(x) / x, rtol=1e-13)


def _b_direct_sphere(rho_r, gam, eta, mu_q, L, lvec, sigma_s, nt=200, nphi=256):
    """Independent evaluation of Eq. 16's integral: product rule on the sphere in coordinates
    about the z-axis (NOT about sigma): Gauss-Legendre in cos(theta) x trapezoid in phi, on the
    smooth part, with the (1+sigma.u)^eta endpoint singularity removed by rotating sigma to the pole."""
    # rotate so that sigma_s is the z axis (Householder), then the integrand is (1+t)^eta * smooth
    e3 = np.array([0.0, 0.0, 1.0])
    v = sigma_s - e3
    H = np.eye(3) if np.linalg.norm(v) < 1e-15 else np.eye(3) - 2.0 * np.outer(v, v) / (v @ v)
    lrot = H @ lvec
    from scipy.special import roots_jacobi
    t, wt = roots_jacobi(nt, 0.0, eta)
    ph = 2 * pi * np.arange(nphi) / nphi
    st = np.sqrt(1 - t * t)
    ux = st[:, None] * np.cos(ph)[None, :]
    uy = st[:, None] * np.sin(ph)[None, :]
    uz = t[:, None] * np.ones(nphi)[None, :]
    phase = np.exp(-1j * mu_q * pi / L * rho_r * (lrot[0] * ux + lrot[1] * uy + lrot[2] * uz))
    return rho_r ** (gam + 2) * (wt[:, None] * phase).sum() * (2 * pi / nphi)


def test_table_b_vss_against_direct_sphere_quadrature():
    """X-5 for eta != 0: the Gauss-Jacobi/J0 form equals a direct 2-D quadrature of Eq. 16."""
    tab = _tab(alpha=[[1.4, 1.2], [1.2, 1.0]], N_rho=3)
    l = freq_grid(6)
    for (p, q) in [(0, 0), (0, 1), (1, 0)]:
        e, g = tab.eta[p, q], tab.gam[p, q]
        assert abs(e - ([[1.4, 1.2], [1.2, 1.0]][p][q] - 1)) < 1e-15
        mu_q = tab.mass[q] / (tab.mass[p] + tab.mass[q])
        for (r, s, z) in [(0, 0, 0), (1, 3, 7), (2, 5, 100), (2, 1, 215), (1, 2, (3 * 6 + 3) * 6 + 3)]:
            ref = _b_direct_sphere(tab.rho[r], g, e, mu_q, tab.L, l[z], tab.sigma[s])
            assert abs(tab.b[p, q, r, s, z] - ref) < 1e-12 * abs(tab.b[p, q, r, s, 0]), (p, q, r, s, z)
        # b(0) = rho^{g+2} C_eta ; Hermitian symmetry b(-l) = conj b(l)
        assert np.allclose(tab.b[p, q, :, 0, 0], tab.rho ** (g + 2) * C_eta(e), rtol=1e-13)
        zpos = (1 * 6 + 2) * 6 + 1            # l = (1, 2, 1)
        zneg = (5 * 6 + 4) * 6 + 5            # l = (-1,-2,-1)
        assert np.allclose(tab.b[p, q, :, :, zneg], np.conj(tab.b[p, q, :, :, zpos]), rtol=1e-13)
        # c(0) = 4 pi C_eta sum_r w_r rho^{g+2}
        assert abs(tab.c[p, q, 0].real - 4 * pi * C_eta(e) * (tab.w_rho * tab.rho ** (g + 2)).sum()) \
            < 1e-12 * abs(tab.c[p, q, 0])


def test_table_mode1_converges_to_exact_angles():
    """Algo 1's pre-sphere quadrature (table_mode 1) tends to the exact angular integrals (P-1):
    with the degree-9 rule the low frequencies of b and c agree closely, and better than with degree 5."""
    rel = lambda x, y: np.max(np.abs(x - y)) / np.max(np.abs(y))
    vhs, vss = [], []
    for Mpre in (12, 32):
        sp, wp = sphere_rule(Mpre)
        # small R keeps the phases rho' |l| <= 1.4 so that a degree-5/9 rule can resolve them
        kw = dict(N=4, N_rho=3, L=8.0, R=1.0, alpha=[[1.0, 1.3], [1.3, 1.0]])
        t1 = _tab(table_mode=1, sigma_pre=sp, w_pre=wp, **kw)
        t0 = _tab(**kw)
        vhs.append(max(rel(t1.b[0, 0], t0.b[0, 0]), rel(t1.c[0, 0], t0.c[0, 0])))
        vss.append(max(rel(t1.b[0, 1], t0.b[0, 1]), rel(t1.c[0, 1], t0.c[0, 1])))
    # eta = 0: smooth integrand, fast convergence (measured 5e-5 -> 2e-9)
    assert vhs[0] < 1e-3 and vhs[1] < 1e-7
    # eta = 0.3: (1 + sigma.u)^eta is not smooth at the antipode, algebraic convergence only
    # (measured 3.8e-3 -> 1.3e-3) -- the reason table_mode 0 is the default (reading P-1)
    assert vss[1] < vss[0] < 1e-2


def test_precompute_in_worker_processes_is_bit_identical():
    """precompute(workers=n) runs the same statements per pair in forked processes: identical tables."""
    kw = dict(N=6, N_rho=3, M=6, L=5.0, mass=(1.0, 2.0, 1.5), omega=[[0.7, 0.75, 0.8]] * 3, alpha=[[1.0, 1.2, 1.4]] * 3)
    t1 = precompute(**kw)
    t2 = precompute(workers=3, **kw)
    for name in ("a", "b", "c", "beta"):
        assert np.array_equal(getattr(t1, name), getattr(t2, name)), name


def test_pooled_oracle_equals_serial_oracle():
    """tests/oracle_pool.py only distributes oracle.collide.collide_pair calls: same numbers as collide_pairs."""
    import os, sys
    sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
    from oracle.collide import collide_pairs
    from oracle_pool import collide_pairs_pool
    tab = precompute(N=6, N_rho=2, M=6, L=5.0, mass=(1.0, 2.0), omega=[[0.6, 0.7]] * 2, alpha=[[1.0, 1.3]] * 2)
    rng = np.random.default_rng(5)
    f = rng.uniform(0.1, 1.0, (3, 2, 216))
    assert np.array_equal(collide_pairs_pool(tab, f), collide_pairs(tab, f))

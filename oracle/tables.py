"""Algorithm 1 of PAPER.md: precomputed tables a, b^(pq), c^(pq); Eq. 5, 6, 9.
ORACLE -- test infrastructure, numpy fp64, follows the paper's loops and notation.

Readings (restated in DESIGN.md): G-1 gamma = 2(1-omega); S-1 full sphere;
RAD-1 one global R from (max mass, min mass); P-1 table_mode 0 evaluates the angular integrals
of Eq. 16/17 exactly, table_mode 1 keeps Algo 1's pre-computation sphere quadrature.
"""
from dataclasses import dataclass
from math import gamma as Gamma, pi, sqrt

import numpy as np
from scipy.special import j0, roots_jacobi

from .quadrature import gauss_legendre_0R, sphere_rule


def freq_index(N: int) -> np.ndarray:
    """Algo 1 steps 1-3: v_x = x - (x >= N/2) * N."""
    x = np.arange(N)
    return x - (x >= N // 2) * N


def freq_grid(N: int) -> np.ndarray:
    """Algo 1 step 4: l = ndgrid(v), flattened row-major -> l[z][3], z=(ix*N+iy)*N+iz."""
    v = freq_index(N)
    lx, ly, lz = np.meshgrid(v, v, v, indexing="ij")
    return np.stack([lx.ravel(), ly.ravel(), lz.ravel()], axis=1).astype(np.float64)


def truncation_radius(L: float, masses) -> float:
    """Eq. 9 with m_a = max mass, m_b = min mass (reading RAD-1)."""
    ma, mb = max(masses), min(masses)
    return 4.0 * L / (1.0 + max(4.0 * ma / (mb + ma), 2.0) + sqrt(1.0 + ma / mb))


def knudsen(mp, mq, n0, d_ref, T_ref_over_T0, omega, H0) -> float:
    """Eq. 5."""
    return 1.0 / (sqrt(1.0 + mp / mq) * pi * n0 * d_ref ** 2 * T_ref_over_T0 ** (omega - 0.5) * H0)


def prefactor_beta(mp, mq, omega, alpha, kn=1.0) -> float:
    """Eq. 6."""
    return (1.0 / kn) * (1.0 / sqrt(1.0 + mp / mq)) / (mp * mq / (mp + mq)) ** (omega - 0.5) \
        * alpha / (2.0 ** (1.0 + alpha) * Gamma(2.5 - omega) * pi)


def sinc_u(x):
    """sin(x)/x with value 1 at x = 0 (unnormalised sinc)."""
    return np.sinc(np.asarray(x) / pi)


@dataclass
class Tables:
    N: int
    N_rho: int
    M: int
    L: float
    R: float
    mass: np.ndarray          # [ns]
    rho: np.ndarray           # [N_rho]
    w_rho: np.ndarray         # [N_rho]
    sigma: np.ndarray         # [M][3]
    w_sigma: np.ndarray       # [M]
    a: np.ndarray             # [N_rho][M][N^3]           real     (Algo 1 step 7)
    b: np.ndarray             # [ns][ns][N_rho][M][N^3]   complex  (Algo 1 step 13, Eq. 16)
    c: np.ndarray             # [ns][ns][N^3]             complex  (Algo 1 step 14, Eq. 17)
    beta: np.ndarray          # [ns][ns]                           (Eq. 6)
    gam: np.ndarray           # [ns][ns]  gamma_pq = 2(1-omega_pq)
    eta: np.ndarray           # [ns][ns]  eta_pq = alpha_pq - 1

    @property
    def ns(self):
        return len(self.mass)


def _b_exact(rho_r, gam, eta, mu_q, L, lvec, lnorm, sigma_s, n_gj=128):
    """O-7: F(k, rho, sigma) of Eq. 16 without B's constant factor, angular integral exact.

    eta = 0 : 4 pi rho^{gam+2} sinc_u(mu_q rho' |l|)
    eta != 0: 2 pi rho^{gam+2} int_{-1}^{1} (1+t)^eta exp(-i z t kappa) J0(z sqrt((1-t^2)(1-kappa^2))) dt,
              z = mu_q rho' |l|, kappa = lhat . sigma_s, by n_gj-node Gauss-Jacobi(0, eta).
    """
    rp = pi * rho_r / L
    z = mu_q * rp * lnorm
    if eta == 0.0:
        return (4.0 * pi * rho_r ** (gam + 2.0) * sinc_u(z)).astype(np.complex128)
    t, wt = roots_jacobi(n_gj, 0.0, eta)           # weight (1-t)^0 (1+t)^eta on [-1,1]
    with np.errstate(invalid="ignore", divide="ignore"):
        kappa = np.where(lnorm > 0, (lvec @ sigma_s) / np.where(lnorm > 0, lnorm, 1.0), 0.0)
    kappa = np.clip(kappa, -1.0, 1.0)
    out = np.zeros(len(lnorm), dtype=np.complex128)
    for tj, wj in zip(t, wt):
        out += wj * np.exp(-1j * z * tj * kappa) * j0(z * np.sqrt((1.0 - tj * tj) * (1.0 - kappa * kappa)))
    return 2.0 * pi * rho_r ** (gam + 2.0) * out


def C_eta(eta: float) -> float:
    """int_{S^2} (1 + sigma.u)^eta dsigma = 2 pi 2^{eta+1} / (eta+1)."""
    return 2.0 * pi * 2.0 ** (eta + 1.0) / (eta + 1.0)


_POOL_ARGS = None


def _pair_tables_pooled(pq):
    return _pair_tables(pq[0], pq[1], *_POOL_ARGS)


def _pair_tables(p, q, mass, gam, eta, omega, alpha, kn, rho, w_rho, sigma, w_sigma, L, l, lnorm, table_mode,
                 sigma_pre, w_pre):
    """b^(pq)[N_rho][M][N^3], c^(pq)[N^3], beta_pq of one pair: the body of Algorithm 1's loops over x, y (and y-hat)."""
    N_rho, M, N3 = len(rho), len(w_sigma), len(lnorm)
    b = np.zeros((N_rho, M, N3), dtype=np.complex128)
    c = np.zeros(N3, dtype=np.complex128)
    mu_q = mass[q] / (mass[p] + mass[q])
    g, e = gam[p, q], eta[p, q]
    beta = prefactor_beta(mass[p], mass[q], omega[p, q], alpha[p, q], kn[p, q])
    for x in range(N_rho):
        for y in range(M):
            if table_mode == 0:
                b[x, y, :] = _b_exact(rho[x], g, e, mu_q, L, l, lnorm, sigma[y])
            else:
                # Algo 1 steps 9-13: quadrature over the pre-computation sphere
                for yh in range(len(w_pre)):
                    Bpq = (1.0 + sigma[y] @ sigma_pre[yh]) ** e
                    b[x, y, :] += Bpq * w_pre[yh] * rho[x] ** (g + 2.0) * np.exp(
                        -1j * mu_q * pi / L * rho[x] * (l @ sigma_pre[yh]))
                    # step 14: c accumulates over x, y and y-hat (reading Q-3)
                    c[:] += w_rho[x] * w_sigma[y] * Bpq * w_pre[yh] * rho[x] ** (g + 2.0) \
                        * np.exp(-1j * pi / L * rho[x] * (l @ sigma_pre[yh]))
        if table_mode == 0:
            # O-8: both angular integrals of Eq. 17 done exactly
            c[:] += w_rho[x] * rho[x] ** (g + 2.0) * C_eta(e) * 4.0 * pi \
                * sinc_u(pi * rho[x] / L * lnorm)
    return b, c, beta


def precompute(N, N_rho, M, L, mass, omega, alpha, kn=None, R=None, sigma=None, w_sigma=None,
               table_mode=0, sigma_pre=None, w_pre=None, beta_override=None, workers=1) -> Tables:
    """Algorithm 1.  workers > 1: the pairs (p,q) are computed in that many forked processes."""
    mass = np.asarray(mass, dtype=np.float64)
    ns = len(mass)
    omega = np.asarray(omega, dtype=np.float64).reshape(ns, ns)
    alpha = np.asarray(alpha, dtype=np.float64).reshape(ns, ns)
    kn = np.ones((ns, ns)) if kn is None else np.asarray(kn, dtype=np.float64).reshape(ns, ns)
    if R is None or R <= 0:
        R = truncation_radius(L, mass)
    rho, w_rho = gauss_legendre_0R(N_rho, R)
    if sigma is None:
        sigma, w_sigma = sphere_rule(M)
    sigma = np.asarray(sigma, dtype=np.float64).reshape(M, 3)
    w_sigma = np.asarray(w_sigma, dtype=np.float64).reshape(M)

    l = freq_grid(N)                                # steps 1-4
    lnorm = np.sqrt((l * l).sum(axis=1))
    N3 = N ** 3

    gam = 2.0 * (1.0 - omega)                       # reading G-1
    eta = alpha - 1.0

    a = np.empty((N_rho, M, N3))
    b = np.zeros((ns, ns, N_rho, M, N3), dtype=np.complex128)
    c = np.zeros((ns, ns, N3), dtype=np.complex128)
    beta = np.empty((ns, ns))

    for x in range(N_rho):                          # step 5
        for y in range(M):                          # step 6
            a[x, y, :] = pi / L * rho[x] * (l @ sigma[y])        # step 7

    args = (mass, gam, eta, omega, alpha, kn, rho, w_rho, sigma, w_sigma, L, l, lnorm, table_mode, sigma_pre, w_pre)
    pairs = [(p, q) for p in range(ns) for q in range(ns)]
    if workers and workers > 1 and len(pairs) > 1:
        # the pairs are independent: same statements, run in forked worker processes (no change of arithmetic)
        import multiprocessing as mp
        global _POOL_ARGS
        _POOL_ARGS = args
        with mp.get_context("fork").Pool(min(workers, len(pairs))) as pool:
            res = pool.map(_pair_tables_pooled, pairs, chunksize=1)
        _POOL_ARGS = None
    else:
        res = [_pair_tables(p, q, *args) for (p, q) in pairs]
    for (p, q), (bpq, cpq, betapq) in zip(pairs, res):
        b[p, q], c[p, q], beta[p, q] = bpq, cpq, betapq
    if beta_override is not None:
        beta = np.asarray(beta_override, dtype=np.float64).reshape(ns, ns).copy()
    return Tables(N, N_rho, M, L, R, mass, rho, w_rho, sigma, w_sigma, a, b, c, beta, gam, eta)

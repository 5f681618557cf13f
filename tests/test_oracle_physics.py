"""Physics sanity pins for the oracle (BASELINE.json north_star): conservation
and the Maxwellian null hold to SPECTRAL accuracy only, so the tests assert the trend with N and
a bound at the finest grid, on resolved inputs (never on c0)."""
import numpy as np
import pytest

from oracle.collide import collide_pair
from oracle.tables import precompute
from workloads import maxwellian, velocity_nodes

MASS = (1.0, 83.798 / 39.948)
OMEGA = [[0.81, 0.805], [0.805, 0.80]]
L = 6.0


def _residuals(N, N_rho, f, M=12):
    tab = precompute(N, N_rho, M, L, MASS, OMEGA, [[1.0] * 2] * 2, beta_override=[[1.0] * 2] * 2)
    c = velocity_nodes(N, L)
    cx, cy, cz = np.meshgrid(c, c, c, indexing="ij")
    cvec = np.stack([cx.ravel(), cy.ravel(), cz.ravel()])
    c2 = (cvec ** 2).sum(axis=0)
    dV = (2 * L / N) ** 3
    Q = [[collide_pair(tab, p, q, f[p], f[q]) for q in range(2)] for p in range(2)]
    mass = max(abs(Q[p][q].sum() * dV) for p in range(2) for q in range(2))
    mom = np.max(np.abs((MASS[0] * cvec * Q[0][1] + MASS[1] * cvec * Q[1][0]).sum(axis=1) * dV))
    ene = abs((MASS[0] * c2 * Q[0][1] + MASS[1] * c2 * Q[1][0]).sum() * dV)
    mom_self = np.max(np.abs((cvec * Q[0][0]).sum(axis=1) * dV))
    qmax = max(np.abs(Q[p][q]).max() for p in range(2) for q in range(2))
    return mass, mom, ene, mom_self, qmax


@pytest.fixture(scope="module")
def maxwell_runs():
    u, T, n = (0.1, -0.05, 0.2), 1.0, (1.0, 0.6)
    out = {}
    for N, N_rho in [(16, 16), (24, 24), (32, 16)]:
        f = [maxwellian(N, L, n[p], u, T, MASS[p]) for p in range(2)]
        out[N] = _residuals(N, N_rho, f)
    return out


def test_maxwellian_null_to_spectral_accuracy(maxwell_runs):
    """X-9: common (u, T) Maxwellian mixture => Q_pq ~ 0; survey measured 1.6e-1, 1.7e-2, 3.2e-4."""
    q16, q24, q32 = (maxwell_runs[N][4] for N in (16, 24, 32))
    assert q24 < q16 / 4 and q32 < q24 / 10
    assert q32 < 1e-3


def test_conservation_to_spectral_accuracy(maxwell_runs):
    """X-8: per-pair mass, pair momentum and energy of Q_pq + Q_qp."""
    m16, m24, m32 = (maxwell_runs[N][0] for N in (16, 24, 32))
    assert m24 < m16 / 20 and m32 < m24 / 100
    assert m32 < 1e-5
    p16, p24, p32 = (maxwell_runs[N][1] for N in (16, 24, 32))
    assert p24 < p16 / 5 and p32 < p24 / 10 and p32 < 1e-3
    e16, e24, e32 = (maxwell_runs[N][2] for N in (16, 24, 32))
    assert e24 < e16 / 5 and e32 < e24 / 10 and e32 < 1e-4
    s24, s32 = maxwell_runs[24][3], maxwell_runs[32][3]
    assert s24 < 1e-3 and s32 < 1e-5


def test_conservation_nonequilibrium_resolved():
    """Same on a mildly non-equilibrium, well resolved bi-Maxwellian (T in [0.9, 1.4])."""
    N = 24
    f = [maxwellian(N, L, 0.7, (0.2, 0.0, -0.1), 0.9, MASS[p]) + maxwellian(N, L, 0.5, (-0.2, 0.1, 0.0), 1.4, MASS[p])
         for p in range(2)]
    mass, mom, ene, _, qmax = _residuals(N, 12, f)
    assert qmax > 1e-2            # genuinely out of equilibrium
    assert mass < 5e-3 and mom < 5e-2 and ene < 5e-3

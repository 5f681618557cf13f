"""Pins for oracle/bkw.py and, through it, the whole operator: closed-form Krook-Wu solution
(Eq. 19-23) and the errors printed in Table 1."""
import os
from math import exp, pi

import numpy as np
import pytest

from oracle.bkw import KrookWu
from oracle.collide import collide_pair
from oracle.tables import precompute
from workloads import velocity_nodes

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _v2(N, L):
    c = velocity_nodes(N, L)
    return (c[:, None, None] ** 2 + c[None, :, None] ** 2 + c[None, None, :] ** 2).reshape(-1)


@pytest.mark.parametrize("ratio", [1.0, 2.0, 4.0])
def test_eq22_is_time_derivative_of_eq19(ratio):
    """Transcription check of Eq. 20-23: central difference of Eq. 19 in t equals Eq. 22."""
    kw = KrookWu(1.0, ratio)
    assert abs(kw.condition()) < 1e-14                      # Eq. 21
    v2 = np.linspace(0.0, 30.0, 7)
    t, h = 5.5, 1e-5
    for p in range(2):
        fd = (kw.f(p, t + h, v2) - kw.f(p, t - h, v2)) / (2 * h)
        assert np.max(np.abs(fd - kw.dfdt(p, t, v2))) < 1e-9 * np.max(np.abs(kw.dfdt(p, t, v2))) + 1e-14


def test_bkw_moments():
    """Eq. 19 integrates to the density n^(p) at any t, and the total kinetic energy of the mixture
    is time independent (radial trapezoid rule on a fine grid)."""
    kw = KrookWu(1.0, 4.0)
    r = np.linspace(0, 40, 400001)
    for p in range(2):
        dens = np.trapezoid(4 * pi * r * r * kw.f(p, 5.5, r * r), r)
        assert abs(dens - 1.0) < 1e-9
    # total energy is time independent
    def energy(t):
        return sum(np.trapezoid(4 * pi * r ** 4 * 0.5 * kw.m[p] * kw.f(p, t, r * r), r) for p in range(2))
    assert abs(energy(5.5) - energy(1.0)) < 1e-9


def test_equal_mass_reduces_to_single_species_bkw():
    """X-3b: m1 = m2 gives K(t) = 1 - exp(-t/4)... (printed constants of SURVEY A.4) and the classic
    single-species Maxwell-molecule BKW form."""
    kw = KrookWu(1.0, 1.0)
    t = 5.5
    K = kw.K(t)
    assert abs(K - (1.0 - exp(-t / 4.0))) < 1e-15
    assert abs(K - 0.7471604041952535) < 1e-15
    Qp = kw.tau[0] * kw.Q(t)
    assert abs(Qp - (1 - K) / (2 * K)) < 1e-15
    v2 = np.array([0.0, 0.5, 3.0, 11.0])
    classic = (2 * pi * K) ** -1.5 * np.exp(-v2 / (2 * K)) * ((5 * K - 3) / (2 * K) + (1 - K) / (2 * K * K) * v2)
    assert np.max(np.abs(kw.f(0, t, v2) - classic)) < 1e-16


def _table1_rows():
    rows = []
    for ln in open(os.path.join(GOLD, "paper_table1_bkw.txt")):
        if ln.startswith("#") or not ln.strip():
            continue
        r, N, Nr, M, e1, e2 = ln.split()
        rows.append((float(r), int(N), int(Nr), int(M), float(e1), float(e2)))
    return rows


def _bkw_errors(ratio, N, N_rho, M):
    L, t = 12.0, 5.5
    kw = KrookWu(1.0, ratio)
    tab = precompute(N, N_rho, M, L, [1.0, ratio], [[1.0] * 2] * 2, [[1.0] * 2] * 2,
                     beta_override=kw.beta())                       # omega = 1 -> gamma = 0; alpha = 1 -> eta = 0
    v2 = _v2(N, L)
    f = [kw.f(p, t, v2) for p in range(2)]
    E = []
    for p in range(2):
        rhs = sum(collide_pair(tab, p, q, f[p], f[q]) for q in range(2))
        E.append(np.max(np.abs(rhs - kw.dfdt(p, t, v2))))
    return E


@pytest.mark.parametrize("row", _table1_rows(), ids=lambda r: "r%g-N%d-Nr%d-M%d" % r[:4])
def test_table1_errors_reproduced(row):
    """X-3: printed L-infinity errors of Table 1 (M = 12, N_rho in {N/2, N}) within 25 %;
    one entry (ratio 4, N=16, E2 = 2.42e-4) is only matched in order of magnitude by every reading
    tried at survey time and is asserted as an upper bound."""
    ratio, N, N_rho, M, e1, e2 = row
    E1, E2 = _bkw_errors(ratio, N, N_rho, M)
    assert abs(E1 - e1) < 0.25 * e1, (E1, e1)
    if ratio == 4 and N == 16:
        assert E2 < e2
    else:
        assert abs(E2 - e2) < 0.25 * e2, (E2, e2)


def test_spectral_convergence_equal_mass():
    """X-3: for ratio 1, M = 12 the error drops >= 10x from N=16 to 24 (N_rho = N/2 as Table 1 says suffices)."""
    e16 = _bkw_errors(1.0, 16, 8, 12)[0]
    e24 = _bkw_errors(1.0, 24, 12, 12)[0]
    assert e24 < e16 / 10.0

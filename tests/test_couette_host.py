"""Host-side pieces of the Couette runner (workloads/couette_case.py): the diagnostics it prints are
plain reductions; they are checked against what they must return on a Maxwellian and on polynomials.  The
configuration itself is checked against the numbers Table 2 prints."""
import numpy as np
import torch

from workloads.couette_case import gll, moments
from workloads import get_config, make_dg_state
from workloads.inputs import maxwellian


def test_gll_weights_integrate_polynomials_exactly():
    for order in (1, 3, 6):
        xi, w = gll(order)
        assert xi[0] == -1.0 and xi[-1] == 1.0 and abs(w.sum() - 2.0) < 1e-14
        for k in range(2 * order):                       # exact up to degree 2 order - 1
            assert abs((w * xi ** k).sum() - (0.0 if k % 2 else 2.0 / (k + 1))) < 1e-13


def test_moments_of_a_maxwellian():
    N, L = 32, 7.0
    mass = (1.0, 139.1 / 66.3)
    f = np.empty((1, 1, 2, N ** 3))
    f[0, 0, 0] = maxwellian(N, L, 0.7, (0.1, -0.15, 0.05), 1.1, mass[0])
    f[0, 0, 1] = maxwellian(N, L, 0.4, (0.0, 0.148, 0.0), 0.9, mass[1])
    n, u, T = moments(torch.from_numpy(f), N, L, mass)
    assert np.allclose(n.numpy()[0, 0], (0.7, 0.4), rtol=1e-9)
    assert np.allclose(u.numpy()[0, 0], ((0.1, -0.15, 0.05), (0.0, 0.148, 0.0)), atol=1e-9)
    assert np.allclose(T.numpy()[0, 0], (1.1, 0.9), rtol=1e-8)


def test_couette_config_is_table_2():
    cfg = get_config("couette")
    assert (cfg.N, cfg.N_rho, cfg.M, cfg.ne, cfg.order, cfg.L, cfg.scheme) == (32, 8, 12, 4, 3, 7.0, "euler")
    assert abs(cfg.mass[1] - 139.1 / 66.3) < 1e-15 and cfg.mass[0] == 1.0
    assert cfg.omega == ((0.81, 0.805), (0.805, 0.80)) and cfg.alpha == ((1.4, 1.36), (1.36, 1.32))
    assert cfg.kn == ((0.793, 0.803), (0.555, 0.606))
    # u_0 = sqrt(2 k T_0 / m_0) = 337.2 m/s (Table 2): the wall speed 50 m/s in units of u_0
    u0 = np.sqrt(2 * 1.380649e-23 * 273.0 / 66.3e-27)
    assert abs(u0 - 337.2) < 0.05 and abs(cfg.wall_u[1][1] - 50.0 / u0) < 1e-4 and cfg.wall_u[0][1] == -cfg.wall_u[1][1]
    f = make_dg_state(cfg)
    n, u, T = moments(torch.from_numpy(f), cfg.N, cfg.L, cfg.mass)
    assert np.allclose(n.numpy(), np.broadcast_to((1.0, 8.009e20 / 1.680e21), n.shape), rtol=1e-9)
    assert np.abs(u.numpy()).max() < 1e-12 and np.allclose(T.numpy(), 1.0, rtol=1e-7)


def test_printed_knudsen_numbers_follow_eq_5():
    """Eq. 5 with Table 2's dimensional inputs gives the printed Kn_pq to the printed digits."""
    from oracle.tables import knudsen
    cfg = get_config("couette")
    d = np.array([[4.11, 4.405], [4.405, 4.7]]) * 1e-10
    for p in range(2):
        for q in range(2):
            kn = knudsen(cfg.mass[p], cfg.mass[q], 1.680e21, d[p, q], 1.0, cfg.omega[p][q], 1e-3)
            assert abs(kn - cfg.kn[p][q]) < 1.5e-3, (p, q, kn)

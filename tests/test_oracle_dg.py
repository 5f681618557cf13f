"""Pins of oracle/dg.py (readings DG-1..DG-3; the paper prints no DG formulas or values):
textbook properties chosen so that a wrong sign, a transposed matrix, a wrong Jacobian, a wrong lift
column or a wrong wall balance fails at least one of them."""
import numpy as np
import pytest

from oracle import dg


def test_gll_nodes_and_matrices():
    # K = 3: -1, 0, 1;  K = 4: +-1, +-1/sqrt(5)  (closed forms)
    np.testing.assert_allclose(dg.gll_nodes(3), [-1.0, 0.0, 1.0], atol=1e-15)
    np.testing.assert_allclose(dg.gll_nodes(4), [-1.0, -1 / np.sqrt(5), 1 / np.sqrt(5), 1.0], atol=1e-14)
    for K in (2, 3, 4, 5, 7):
        xi = dg.gll_nodes(K)
        D, M = dg.lagrange_matrices(xi)
        for a in range(K):                       # D is exact on x^a, a <= order
            np.testing.assert_allclose(D @ xi ** a, a * xi ** max(a - 1, 0) if a else 0 * xi, atol=1e-11)
        # M integrates products of polynomials of degree <= order exactly: x^a x^b over [-1, 1]
        for a in range(K):
            for b in range(K):
                exact = 0.0 if (a + b) % 2 else 2.0 / (a + b + 1)
                assert abs(xi ** a @ M @ xi ** b - exact) < 1e-12
        assert abs(M.sum() - 2.0) < 1e-13
        # integration by parts: M D + (M D)^T = e_K e_K^T - e_1 e_1^T
        B = np.zeros((K, K)); B[-1, -1] = 1.0; B[0, 0] = -1.0
        np.testing.assert_allclose(M @ D + (M @ D).T, B, atol=1e-12)


def _poly_state(mesh, N, L, coef, ns=1):
    """f(x, c) = p(x) g(c) with p a polynomial in x and g a fixed positive profile."""
    x = mesh.node_x()
    px = sum(a * x ** i for i, a in enumerate(coef))
    g = dg.wall_maxwellian(N, L, (0.1, 0.0, 0.0), 1.0, 1.0)
    return (px[:, :, None, None] * g[None, None, None, :]).repeat(ns, axis=2), px, g


def test_interior_transport_is_exact_for_polynomials():
    """For data that is one polynomial of degree <= order across all elements the interface jumps vanish
    and rhs = -c_x p'(x) g(c) exactly at interior elements (walls touch only the two end elements)."""
    N, L = 4, 3.0
    mesh = dg.Mesh1D(5, 3, x0=-0.5, x1=2.0)
    coef = [0.7, -0.3, 0.5, 0.2]
    f, _, g = _poly_state(mesh, N, L, coef)
    x = mesh.node_x()
    dp = sum(i * a * x ** (i - 1) for i, a in enumerate(coef) if i)
    rhs = dg.advect_rhs(mesh, f, N, L, (1.0,))
    cx = dg.velocity_cx(N, L)
    exact = -dp[:, :, None, None] * (cx * g)[None, None, None, :]
    np.testing.assert_allclose(rhs[1:-1], exact[1:-1], atol=1e-12 * np.abs(exact).max())
    # end elements: only the wall half range differs
    np.testing.assert_allclose(rhs[0][..., cx < 0], exact[0][..., cx < 0], atol=1e-12 * np.abs(exact).max())
    np.testing.assert_allclose(rhs[-1][..., cx > 0], exact[-1][..., cx > 0], atol=1e-12 * np.abs(exact).max())


def test_upwinding_direction():
    """A jump between two constant states moves with the sign of c_x: the downstream element changes."""
    N, L = 4, 3.0
    mesh = dg.Mesh1D(4, 2)
    g = np.ones(N ** 3)
    f = np.ones((4, 3, 1, N ** 3))
    f[2:] = 2.0
    rhs = dg.advect_rhs(mesh, f * g, N, L, (1.0,))
    cx = dg.velocity_cx(N, L)
    assert np.abs(rhs[1][..., cx > 0]).max() < 1e-13          # upstream of the jump for c_x > 0: untouched
    assert np.abs(rhs[2][..., cx > 0]).max() > 0.1            # downstream: sees the jump
    assert np.abs(rhs[2][..., cx < 0]).max() < 1e-13
    assert np.abs(rhs[1][..., cx < 0]).max() > 0.1
    # sign: for c_x > 0 the state 1 flows into the element holding 2 => f decreases at its first node
    z = np.argmax(cx > 0)
    assert rhs[2, 0, 0, z] < 0


def test_wall_maxwellian_is_steady_and_mass_is_conserved():
    N, L = 8, 5.0
    mass = (1.0, 2.0)
    mesh = dg.Mesh1D(3, 2, wall_T=(1.0, 1.0))
    f = np.empty((3, 3, 2, N ** 3))
    for p, m in enumerate(mass):
        f[:, :, p] = (0.8 + 0.3 * p) * dg.wall_maxwellian(N, L, (0, 0, 0), 1.0, m)
    rhs = dg.advect_rhs(mesh, f, N, L, mass)
    assert np.abs(rhs).max() < 1e-13 * np.abs(f).max()
    # arbitrary state, different wall temperatures: d/dt of the per-species mass vanishes
    rng = np.random.default_rng(0)
    mesh = dg.Mesh1D(3, 2, wall_T=(0.8, 1.2), wall_u=((0, 0.1, 0), (0, -0.1, 0)))
    f = f * (1.0 + 0.3 * rng.uniform(-1, 1, f.shape))
    rhs = dg.advect_rhs(mesh, f, N, L, mass)
    w = mesh.M.sum(axis=0)                                    # nodal quadrature weights of the exact mass matrix
    dmass = np.einsum("k,ekpz->p", w, rhs) * mesh.h / 2.0
    scale = np.einsum("k,ekpz->p", w, np.abs(rhs)) * mesh.h / 2.0
    assert np.all(np.abs(dmass) < 1e-12 * scale)


def test_free_streaming_converges_at_order_plus_one():
    """Advect sin(2 pi x) g(c) with a single velocity sign away from the walls' influence: compare with the
    exact shifted profile on the region the wall has not reached; error ratio between ne and 2 ne ~ 2^(order+1)."""
    N, L = 2, 1.0                     # c_x = +-0.5
    errs = []
    for ne in (8, 16):
        mesh = dg.Mesh1D(ne, 2, x0=0.0, x1=1.0)
        x = mesh.node_x()
        g = np.ones(N ** 3)
        f = (1.0 + 0.5 * np.sin(2 * np.pi * x))[:, :, None, None] * g[None, None, None, :]
        T = 0.1
        nsteps = 40 * (ne // 8)
        u = dg.step(mesh, f, T / nsteps, nsteps, N, L, (1.0,))
        cx = dg.velocity_cx(N, L)
        z = np.argmax(cx > 0)          # c_x = +0.5: exact solution f0(x - 0.5 t) for x > 0.5 T
        exact = 1.0 + 0.5 * np.sin(2 * np.pi * (x - cx[z] * T))
        mask = x > 0.2
        errs.append(np.abs(u[:, :, 0, z] - exact)[mask].max())
    assert errs[0] / errs[1] > 6.0, errs


def test_rk3_is_third_order_in_time_on_a_linear_ode():
    """step() with a collide callback that makes L(f) = -f at every node and no transport (c_x sums cancel for
    constant-in-x data between Maxwellian walls is not needed here): use ne = 1 with a wall-steady state."""
    N, L = 4, 4.0
    mesh = dg.Mesh1D(1, 1, wall_T=(1.0, 1.0))
    f = np.empty((1, 2, 1, N ** 3))
    f[:] = dg.wall_maxwellian(N, L, (0, 0, 0), 1.0, 1.0)
    lam = -1.3
    errs = []
    for n in (4, 8):
        # the wall density follows the outgoing flux, so a uniformly scaled Maxwellian stays transport-steady
        u = dg.step(mesh, f, 1.0 / n, n, N, L, (1.0,), collide=lambda g: lam * g)
        errs.append(np.abs(u - np.exp(lam) * f).max() / np.abs(f).max())
    assert 6.5 < errs[0] / errs[1] < 9.5, errs


def test_euler_scheme_is_the_closed_form_on_a_linear_ode():
    """Same set-up with scheme "euler": n steps of size h on f' = lam f give (1 + h lam)^n f exactly (closed
    form, not a restatement of the update), and the error against e^{lam} halves with the step (first order)."""
    N, L = 4, 4.0
    mesh = dg.Mesh1D(1, 1, wall_T=(1.0, 1.0))
    f = np.empty((1, 2, 1, N ** 3))
    f[:] = dg.wall_maxwellian(N, L, (0, 0, 0), 1.0, 1.0)
    lam = -1.3
    errs = []
    for n in (16, 32):
        u = dg.step(mesh, f, 1.0 / n, n, N, L, (1.0,), collide=lambda g: lam * g, scheme="euler")
        assert np.abs(u - (1.0 + lam / n) ** n * f).max() < 1e-13 * np.abs(f).max()
        errs.append(np.abs(u - np.exp(lam) * f).max() / np.abs(f).max())
    assert 1.8 < errs[0] / errs[1] < 2.2, errs
    with pytest.raises(ValueError):
        dg.step(mesh, f, 0.1, 1, N, L, (1.0,), scheme="rk4")


def test_euler_step_is_f_plus_dt_rhs():
    """One Euler step of free transport on rough data equals f + dt advect_rhs(f) (ties scheme "euler" to the
    pinned right-hand side)."""
    rng = np.random.default_rng(5)
    N, L = 4, 4.0
    mesh = dg.Mesh1D(3, 2, wall_T=(0.9, 1.1), wall_u=((0, 0.1, 0), (0, -0.1, 0)))
    f = np.empty((3, 3, 2, N ** 3))
    for p, m in enumerate((1.0, 2.0)):
        f[:, :, p] = dg.wall_maxwellian(N, L, (0, 0, 0), 1.0, m)
    f *= 1.0 + 0.3 * rng.uniform(-1, 1, f.shape)
    u = dg.step(mesh, f, 1e-2, 1, N, L, (1.0, 2.0), scheme="euler")
    assert np.array_equal(u, f + 1e-2 * dg.advect_rhs(mesh, f, N, L, (1.0, 2.0)))

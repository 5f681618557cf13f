"""1-D nodal discontinuous Galerkin transport around the collision operator (secondary rows D1-D4 of
SURVEY.md section 8(a)).  ORACLE -- test infrastructure, numpy fp64, plain loops over elements.

The paper gives no formulas for its spatial scheme ("discontinuous Galerkin ... Runge-Kutta",
P:339 linear distribution of elements, Table 2 P:370-375 "purely diffuse" walls); this file states
the readings DG-1..DG-3 of DESIGN.md section 2:

  DG-1  K = order+1 Gauss-Lobatto-Legendre nodes per element, ne uniform elements of width h on
        [x0, x1], strong form with the exact mass matrix M of the Lagrange basis,
          d/dt f_e = -(2/h) c_x D f_e + (2/h) M^-1 [ e_K (c_x f_{e,K} - F*_{e+1/2}) - e_1 (c_x f_{e,1} - F*_{e-1/2}) ],
        upwind flux F*_{e+1/2} = c_x f_{e,K} if c_x > 0 else c_x f_{e+1,1}.
  DG-2  diffuse wall: the incoming half range is n_w Maxw(1, u_w, T_w; m_p) with n_w fixed per species by zero
        net mass flux through the wall, using the same discrete velocity sums.
  DG-3  SSP-RK3 (Shu-Osher): u1 = u + dt L(u); u2 = 3/4 u + 1/4 (u1 + dt L(u1)); u+ = 1/3 u + 2/3 (u2 + dt L(u2)),
        L(f) = transport + sum_q beta_pq Q^(pq)(f_p, f_q)  (right-hand side of Eq. 1).

PARITY-UNPINNED against the paper (it prints nothing to compare with).  Pinned by textbook properties in
tests/test_oracle_dg.py: D differentiates polynomials of degree <= order exactly, M integrates products
exactly, free streaming of polynomial-in-x data is exact in space, a uniform wall-temperature Maxwellian is
a steady state, per-species mass is conserved to round-off with diffuse walls, and the scheme converges at
order+1 on a smooth advected profile.
"""
import numpy as np


def gll_nodes(K: int) -> np.ndarray:
    """K Gauss-Lobatto-Legendre nodes on [-1, 1]: +-1 and the roots of P'_{K-1}."""
    if K < 2:
        raise ValueError("need at least 2 nodes")
    P = np.polynomial.legendre.Legendre.basis(K - 1)
    inner = np.sort(P.deriv().roots().real)
    return np.concatenate(([-1.0], inner, [1.0]))


def lagrange_matrices(xi: np.ndarray):
    """(D, M) of the Lagrange basis on the nodes xi: D[i][j] = l_j'(xi_i), M[i][j] = int l_i l_j."""
    K = len(xi)
    # monomial coefficients of every Lagrange polynomial from the Vandermonde system
    V = np.vander(xi, K, increasing=True)              # V[i][a] = xi_i^a
    C = np.linalg.inv(V)                               # l_j(x) = sum_a C[a][j] x^a
    D = np.zeros((K, K))
    for i in range(K):
        for j in range(K):
            D[i, j] = sum(a * C[a, j] * xi[i] ** (a - 1) for a in range(1, K))
    gx, gw = np.polynomial.legendre.leggauss(K + 1)    # exact to degree 2K+1 >= 2K-2
    Lg = np.array([[sum(C[a, j] * x ** a for a in range(K)) for j in range(K)] for x in gx])   # [g][j]
    M = np.einsum("g,gi,gj->ij", gw, Lg, Lg)
    return D, M


class Mesh1D:
    def __init__(self, ne, order, x0=0.0, x1=1.0, wall_T=(1.0, 1.0), wall_u=((0.0, 0.0, 0.0), (0.0, 0.0, 0.0))):
        self.ne, self.order, self.K = ne, order, order + 1
        self.x0, self.x1, self.h = x0, x1, (x1 - x0) / ne
        self.wall_T = tuple(wall_T)
        self.wall_u = tuple(tuple(u) for u in wall_u)
        self.xi = gll_nodes(self.K)
        self.D, self.M = lagrange_matrices(self.xi)
        self.Minv = np.linalg.inv(self.M)

    def node_x(self):
        """x[ne][K]"""
        return self.x0 + self.h * (np.arange(self.ne)[:, None] + 0.5 * (self.xi[None, :] + 1.0))


def velocity_cx(N: int, L: float) -> np.ndarray:
    """c_x of every velocity node z = (ix N + iy) N + iz (reading C-1, C-2)."""
    c = -L + (np.arange(N) + 0.5) * 2.0 * L / N
    return np.repeat(c, N * N)


def wall_maxwellian(N, L, u, T, m):
    """Maxw(1, u, T; m) on the grid, flattened (reading M-1)."""
    c = -L + (np.arange(N) + 0.5) * 2.0 * L / N
    ex = np.exp(-m * (c - u[0]) ** 2 / T)
    ey = np.exp(-m * (c - u[1]) ** 2 / T)
    ez = np.exp(-m * (c - u[2]) ** 2 / T)
    return (m / (np.pi * T)) ** 1.5 * (ex[:, None, None] * ey[None, :, None] * ez[None, None, :]).reshape(-1)


def advect_rhs(mesh: Mesh1D, f: np.ndarray, N: int, L: float, mass) -> np.ndarray:
    """-c_x d/dx f in the DG sense with upwind fluxes and diffuse walls.  f[ne][K][ns][N^3]."""
    ne, K, ns, N3 = f.shape
    cx = velocity_cx(N, L)
    pos = cx > 0
    rhs = np.zeros_like(f)
    # interface fluxes F[e] at x_{e-1/2}, e = 0..ne, per species
    F = np.zeros((ne + 1, ns, N3))
    for e in range(1, ne):
        F[e] = cx * np.where(pos, f[e - 1, K - 1], f[e, 0])
    for p in range(ns):
        # left wall (x0): gas leaves with c_x < 0, comes back with c_x > 0
        wl = wall_maxwellian(N, L, mesh.wall_u[0], mesh.wall_T[0], mass[p])
        out = np.sum(-cx[~pos] * f[0, 0, p][~pos])
        n_w = out / np.sum(cx[pos] * wl[pos])
        F[0, p] = cx * np.where(pos, n_w * wl, f[0, 0, p])
        # right wall (x1): gas leaves with c_x > 0, comes back with c_x < 0
        wr = wall_maxwellian(N, L, mesh.wall_u[1], mesh.wall_T[1], mass[p])
        out = np.sum(cx[pos] * f[ne - 1, K - 1, p][pos])
        n_w = out / np.sum(-cx[~pos] * wr[~pos])
        F[ne, p] = cx * np.where(pos, f[ne - 1, K - 1, p], n_w * wr)
    jac = 2.0 / mesh.h
    for e in range(ne):
        vol = -jac * cx * np.einsum("kj,jpz->kpz", mesh.D, f[e])
        jump_r = cx * f[e, K - 1] - F[e + 1]
        jump_l = cx * f[e, 0] - F[e]
        lift = jac * (mesh.Minv[:, K - 1][:, None, None] * jump_r[None] - mesh.Minv[:, 0][:, None, None] * jump_l[None])
        rhs[e] = vol + lift
    return rhs


def step(mesh: Mesh1D, f: np.ndarray, dt: float, nsteps: int, N: int, L: float, mass, collide=None,
         scheme: str = "rk3") -> np.ndarray:
    """nsteps steps of SSP-RK3 (scheme "rk3", reading DG-3) or of forward Euler (scheme "euler", the time
    stepping of the paper's Couette case, Table 2).
    collide(g[nx][ns][N^3]) -> Q[nx][ns][N^3] or None (free transport)."""
    if scheme not in ("rk3", "euler"):
        raise ValueError("scheme must be 'rk3' or 'euler'")
    ne, K, ns, N3 = f.shape

    def Lop(u):
        r = advect_rhs(mesh, u, N, L, mass)
        if collide is not None:
            r = r + collide(u.reshape(ne * K, ns, N3)).reshape(u.shape)
        return r

    u = f.copy()
    for _ in range(nsteps):
        if scheme == "euler":
            u = u + dt * Lop(u)
            continue
        u1 = u + dt * Lop(u)
        u2 = 0.75 * u + 0.25 * (u1 + dt * Lop(u1))
        u = u / 3.0 + (2.0 / 3.0) * (u2 + dt * Lop(u2))
    return u

"""Seeded input distribution functions for configs c0..c4 (recipe: DESIGN.md "Input recipe",
SURVEY.md section 8(d)).  Nothing here belongs to the collision algorithm.

Layout produced everywhere: f[x][p][z], z = (ix*N + iy)*N + iz (iz fastest), velocity node
c = (c[ix], c[iy], c[iz]) with c[j] = -L + (j + 1/2) * 2L/N   (reading C-1, cell-centred).
"""
import numpy as np

from .rng import splitmix64_uniform
from .configs import Config

POINT_STRIDE = 1 << 24     # counters reserved per spatial point
NOISE_OFFSET = 64          # first per-node noise counter inside a point's block


def velocity_nodes(N: int, L: float) -> np.ndarray:
    """The N cell-centred nodes of one velocity axis."""
    return -L + (np.arange(N) + 0.5) * (2.0 * L / N)


def maxwellian(N: int, L: float, n: float, u, T: float, m: float) -> np.ndarray:
    """n (m/(pi T))^{3/2} exp(-m |c-u|^2 / T) on the N^3 grid, flattened (reading M-1)."""
    c = velocity_nodes(N, L)
    ex = np.exp(-m * (c - u[0]) ** 2 / T)
    ey = np.exp(-m * (c - u[1]) ** 2 / T)
    ez = np.exp(-m * (c - u[2]) ** 2 / T)
    g = ex[:, None, None] * ey[None, :, None] * ez[None, None, :]
    return (n * (m / (np.pi * T)) ** 1.5) * g.reshape(-1)


def _U(seed, counter, lo, hi):
    return lo + (hi - lo) * float(splitmix64_uniform(seed, [counter])[0])


def _bimaxwell_point(cfg: Config, x: int) -> np.ndarray:
    """c0/c1/c4: f_p = sum_{j=1,2} Maxw(n_j, u_j, T_j; m_p); draw order species p, component j,
    then (n, ux, uy, uz, T)."""
    base = x * POINT_STRIDE
    out = np.empty((cfg.ns, cfg.N ** 3))
    for p in range(cfg.ns):
        acc = np.zeros(cfg.N ** 3)
        for j in range(2):
            k = base + (p * 2 + j) * 5
            n = _U(cfg.seed, k + 0, 0.5, 1.5)
            u = [_U(cfg.seed, k + 1 + d, -0.3, 0.3) for d in range(3)]
            T = _U(cfg.seed, k + 4, 0.5, 2.0)
            acc += maxwellian(cfg.N, cfg.L, n, u, T, cfg.mass[p])
        out[p] = acc
    return out


def _c2_point(cfg: Config, x: int) -> np.ndarray:
    base = x * POINT_STRIDE
    N3 = cfg.N ** 3
    out = np.empty((cfg.ns, N3))
    if x < cfg.nx // 2:
        # near equilibrium: common u, T; 1e-3 relative i.i.d. perturbation per velocity node
        u = [_U(cfg.seed, base + cfg.ns + d, -0.3, 0.3) for d in range(3)]
        T = _U(cfg.seed, base + cfg.ns + 3, 0.8, 1.5)
        for p in range(cfg.ns):
            n = _U(cfg.seed, base + p, 0.5, 1.5)
            k0 = base + NOISE_OFFSET + p * N3
            xi = 2.0 * splitmix64_uniform(cfg.seed, np.arange(k0, k0 + N3, dtype=np.uint64)) - 1.0
            out[p] = maxwellian(cfg.N, cfg.L, n, u, T, cfg.mass[p]) * (1.0 + 1.0e-3 * xi)
    else:
        # strongly non-equilibrium: two Maxwellians, temperature ratio up to 4
        for p in range(cfg.ns):
            k = base + p * 10
            na = _U(cfg.seed, k + 0, 0.5, 1.5)
            ua = [_U(cfg.seed, k + 1 + d, -0.3, 0.3) for d in range(3)]
            Ta = _U(cfg.seed, k + 4, 0.5, 0.75)
            nb = _U(cfg.seed, k + 5, 0.5, 1.5)
            ub = [_U(cfg.seed, k + 6 + d, -0.3, 0.3) for d in range(3)]
            Tb = Ta * _U(cfg.seed, k + 9, 1.5, 4.0)
            out[p] = (maxwellian(cfg.N, cfg.L, na, ua, Ta, cfg.mass[p])
                      + maxwellian(cfg.N, cfg.L, nb, ub, Tb, cfg.mass[p]))
    return out


def make_points(cfg: Config, xs) -> np.ndarray:
    """f[len(xs)][ns][N^3] for the spatial points `xs` of a homogeneous config (c0, c1, c2, c4)."""
    xs = list(xs)
    out = np.empty((len(xs), cfg.ns, cfg.N ** 3))
    for i, x in enumerate(xs):
        if cfg.kind == "bimaxwell":
            out[i] = _bimaxwell_point(cfg, int(x))
        elif cfg.kind == "c2mix":
            out[i] = _c2_point(cfg, int(x))
        else:
            raise ValueError("make_points is for homogeneous configs; use make_dg_state for c3")
    return out


def make_dg_state(cfg: Config) -> np.ndarray:
    """Initial state of the DG cases, f[ne][K][ns][N^3], K = order+1 nodes per element.  c3 (reading DG-4):
    f_p = n_p (1 + 0.05 xi_{e,p}) Maxw(1, 0, 1; m_p), xi ~ U[-1,1] per (element, species),
    the same value at every node of the element."""
    K = cfg.order + 1
    out = np.empty((cfg.ne, K, cfg.ns, cfg.N ** 3))
    for e in range(cfg.ne):
        for p in range(cfg.ns):
            xi = 2.0 * float(splitmix64_uniform(cfg.seed, [e * cfg.ns + p])[0]) - 1.0
            if cfg.kind == "couette":
                xi = 0.0                       # Table 2: uniform gas at rest, T = T_0
            fp = maxwellian(cfg.N, cfg.L, cfg.density[p] * (1.0 + 0.05 * xi), (0.0, 0.0, 0.0), 1.0,
                            cfg.mass[p])
            out[e, :, p, :] = fp[None, :]
    return out

"""The five workload configurations of BASELINE.json `configs`, with the readings of
SURVEY.md section 8(d) (seeds, open parameters).  Pure data: no arithmetic of the method."""
from dataclasses import dataclass, field
from typing import Tuple

_AR, _KR = 39.948, 83.798


@dataclass(frozen=True)
class Config:
    name: str
    seed: int
    mass: Tuple[float, ...]
    omega: Tuple[Tuple[float, ...], ...]      # [ns][ns] viscosity index (Eq. 4)
    alpha: Tuple[Tuple[float, ...], ...]      # [ns][ns] VSS scattering parameter; 1 = VHS
    N: int
    L: float
    N_rho: int
    M: int
    nx: int                                   # spatial points in the batch
    kind: str                                 # "bimaxwell" | "c2mix" | "dg"
    # config 3 only (1-D DG slab, reading DG-4)
    ne: int = 0
    order: int = 0
    dt: float = 0.0
    nsteps: int = 0
    wall_T: Tuple[float, float] = (1.0, 1.0)
    density: Tuple[float, ...] = field(default_factory=tuple)
    # Couette case only
    wall_u: Tuple[Tuple[float, float, float], Tuple[float, float, float]] = ((0.0, 0.0, 0.0), (0.0, 0.0, 0.0))
    kn: Tuple[Tuple[float, ...], ...] = ()    # [ns][ns] Knudsen numbers (Eq. 5); () = all 1
    scheme: str = "rk3"                       # time stepping of the DG cases: "rk3" | "euler"

    @property
    def ns(self) -> int:
        return len(self.mass)


def _full(v, ns):
    return tuple(tuple(float(v) for _ in range(ns)) for _ in range(ns))


def _mean_matrix(diag):
    ns = len(diag)
    return tuple(tuple(0.5 * (diag[p] + diag[q]) for q in range(ns)) for p in range(ns))


CONFIGS = {
    # BASELINE.json configs[0]
    "c0": Config("c0", 190304670, (1.0, 2.0), _full(0.5, 2), _full(1.0, 2),
                 N=8, L=5.0, N_rho=8, M=6, nx=4, kind="bimaxwell"),
    # configs[1]: Ar/Kr, omega 0.81 / 0.80 / mixed 0.805
    "c1": Config("c1", 190304671, (1.0, _KR / _AR), ((0.81, 0.805), (0.805, 0.80)), _full(1.0, 2),
                 N=24, L=6.0, N_rho=24, M=12, nx=1024, kind="bimaxwell"),
    # configs[2]: headline
    "c2": Config("c2", 190304672, (1.0, _KR / _AR), ((0.81, 0.805), (0.805, 0.80)), _full(1.0, 2),
                 N=32, L=6.0, N_rho=32, M=12, nx=4096, kind="c2mix"),
    # configs[3]: 1-D DG slab, 3 species, VSS (reading DG-4)
    "c3": Config("c3", 190304673, (1.0, 1.5, 2.0), _mean_matrix((0.70, 0.75, 0.80)),
                 _mean_matrix((1.0, 1.2, 1.4)),
                 N=24, L=6.0, N_rho=24, M=12, nx=64, kind="dg",
                 ne=16, order=3, dt=2.0e-4, nsteps=100, wall_T=(0.8, 1.2),
                 density=(1.0, 0.8, 0.6)),
    # configs[4]: stress case
    "c4": Config("c4", 190304674, (1.0, 4.0), _full(0.5, 2), _full(1.0, 2),
                 N=48, L=7.0, N_rho=48, M=32, nx=2048, kind="bimaxwell"),
    # Second workload: the paper's Couette case C-01, Table 2, in the
    # paper's units (m_0 = 66.3e-27 kg, u_0 = 337.2 m/s, T_0 = 273 K, n_0 = 1.680e21 m^-3, H_0 = 1 mm): masses
    # {66.3, 139.1}e-27 kg, VSS with the printed omega / alpha, Knudsen numbers as printed, walls at
    # y velocity -+50 m/s and 273 K, gas initially at rest at 273 K with n = {1.680e21, 8.009e20} m^-3, 4 elements
    # of order 3, 32^3 velocity grid on [-7, 7]^3, N_rho = 8, M = 12, forward Euler.  The paper does not print its
    # time step: dt is this repository's choice.
    "couette": Config("couette", 190304675, (1.0, 139.1 / 66.3), ((0.81, 0.805), (0.805, 0.80)),
                      ((1.4, 1.36), (1.36, 1.32)),
                      N=32, L=7.0, N_rho=8, M=12, nx=16, kind="couette",
                      ne=4, order=3, dt=1.0e-3, nsteps=100, wall_T=(1.0, 1.0),
                      density=(1.0, 8.009e20 / 1.680e21),
                      wall_u=((0.0, -50.0 / 337.2, 0.0), (0.0, 50.0 / 337.2, 0.0)),
                      kn=((0.793, 0.803), (0.555, 0.606)), scheme="euler"),
    # Two extra operating points for bench lines (not BASELINE.json configurations):
    # c4 with VSS scattering (every pair needs a full table b_rs(k): 2.7 GB per pair in the paper's layout),
    # and c2 at the radial resolution the paper recommends as sufficient, N_rho = N/2.
    "c4vss": Config("c4vss", 190304676, (1.0, 4.0), _full(0.5, 2), ((1.2, 1.3), (1.3, 1.4)),
                    N=48, L=7.0, N_rho=48, M=32, nx=64, kind="bimaxwell"),
    "c2half": Config("c2half", 190304672, (1.0, _KR / _AR), ((0.81, 0.805), (0.805, 0.80)), _full(1.0, 2),
                     N=32, L=6.0, N_rho=16, M=12, nx=4096, kind="c2mix"),
}


def get_config(name: str) -> Config:
    return CONFIGS[name]

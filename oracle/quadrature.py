"""Quadrature rules used by Algo 1.  ORACLE -- test infrastructure.

* radial: N_rho-point Gauss-Legendre mapped to [0, R]           ("rho, the GLQ zeros")
* sphere: closed-form symmetric rules standing in for the spherical designs of ref. [18]
  whose point files are not available (reading S-1/S-2 of SURVEY.md section 8(c)):
  M=6 octahedron, M=12 icosahedron, M=32 icosahedron + dual dodecahedron (weighted).
"""
import numpy as np


def gauss_legendre_0R(N_rho: int, R: float):
    """(rho_r, w_r): Gauss-Legendre nodes/weights on [0, R]  (O-2)."""
    x, w = np.polynomial.legendre.leggauss(N_rho)
    return 0.5 * R * (x + 1.0), 0.5 * R * w


def sphere_rule(M: int):
    """(sigma[M][3], w_sigma[M]) with sum(w) = 4 pi  (S-2).  Full sphere, all M points."""
    phi = 0.5 * (1.0 + np.sqrt(5.0))
    if M == 6:
        pts = []
        for d in range(3):
            for s in (1.0, -1.0):
                v = [0.0, 0.0, 0.0]
                v[d] = s
                pts.append(v)
        sig = np.array(pts)
        w = np.full(6, 4.0 * np.pi / 6.0)
    elif M in (12, 32):
        ico = []
        for s1 in (1.0, -1.0):
            for s2 in (1.0, -1.0):
                ico += [[0.0, s1, s2 * phi], [s1, s2 * phi, 0.0], [s2 * phi, 0.0, s1]]
        ico = np.array(ico)
        ico /= np.linalg.norm(ico, axis=1)[:, None]
        if M == 12:
            sig, w = ico, np.full(12, 4.0 * np.pi / 12.0)
        else:
            dod = []
            for a in (1.0, -1.0):
                for b in (1.0, -1.0):
                    for c in (1.0, -1.0):
                        dod.append([a, b, c])
            for a in (1.0, -1.0):
                for b in (1.0, -1.0):
                    dod += [[a / phi, 0.0, b * phi], [0.0, a * phi, b / phi], [a * phi, b / phi, 0.0]]
            dod = np.array(dod)
            dod /= np.linalg.norm(dod, axis=1)[:, None]
            sig = np.vstack([ico, dod])
            w = np.concatenate([np.full(12, 4.0 * np.pi * 5.0 / 168.0),
                                np.full(20, 4.0 * np.pi * 9.0 / 280.0)])
    else:
        raise ValueError("built-in sphere rules exist for M in {6, 12, 32}")
    return sig, w

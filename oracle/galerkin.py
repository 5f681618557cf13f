"""Direct O(N^6) evaluation of the Fourier-Galerkin sum, Eq. 11 of PAPER.md.
ORACLE -- test infrastructure; used only to pin oracle/collide.py on tiny N.

Two kernels:
* `galerkin_lowrank`: Eq. 11 with G+ replaced by the separated expansion Eq. 13/15 built from the
  SAME tables a, b, c as Algo 2 -> must equal Algo 2 to round-off when index sums are circular
  (wrap=True; the size-N FFTs of Algo 2 alias), and on inputs band-limited to |l_d| < N/4 also
  with the literal unwrapped sum of Eq. 11 (wrap=False).
* `galerkin_exact_vhs`: Eq. 11 with the full, non-low-rank kernel modes G+(l,m), G-(m) of Eq. 12
   for eta = 0, the radial integral by a fine Gauss-Legendre rule, the two angular
  integrals in closed form (4 pi sinc).  Differs from Algo 2 by the quadrature error of Eq. 13.
"""
from math import pi

import numpy as np

from .tables import Tables, freq_index, sinc_u


def _index_grid(N):
    i = np.arange(N)
    ix, iy, iz = np.meshgrid(i, i, i, indexing="ij")
    return np.stack([ix.ravel(), iy.ravel(), iz.ravel()], axis=1)          # [N^3][3] array indices


def _accumulate(N, fhat, ghat, kernel_row, wrap):
    """Q^_k = sum_{l,m: l+m=k} kernel(l, m) f^_l g^_m ; kernel_row(zl) returns kernel(l, all m)
    given the flat k index of every m.  Returns Q^ as flat [N^3] in array-index order."""
    idx = _index_grid(N)
    v = freq_index(N)
    N3 = N ** 3
    Qhat = np.zeros(N3, dtype=np.complex128)
    for zl in range(N3):
        il = idx[zl]
        if wrap:
            ik = (il[None, :] + idx) % N                       # circular index sum
            valid = np.ones(N3, dtype=bool)
        else:
            ksum = v[il][None, :] + v[idx]                     # literal l + m
            valid = np.all((ksum >= -N // 2) & (ksum < N // 2), axis=1)
            ik = ksum % N
        zk = (ik[:, 0] * N + ik[:, 1]) * N + ik[:, 2]
        contrib = kernel_row(zl, zk) * fhat[zl] * ghat
        np.add.at(Qhat, zk[valid], contrib[valid])
    return Qhat


def _to_physical(N, Qhat):
    """Q(c_j) = sum_k Q^_k e^{2 pi i k.j/N}  (Eq. 10 evaluated at the grid nodes)."""
    return np.fft.ifftn(Qhat.reshape(N, N, N)).reshape(-1) * N ** 3


def galerkin_lowrank(tab: Tables, p, q, Fp, Fq, wrap=True, scale_beta=True):
    N = tab.N
    N3 = N ** 3
    mp, mq = tab.mass[p], tab.mass[q]
    muq, mup = mq / (mp + mq), mp / (mp + mq)
    fhat = np.fft.fftn(Fp.reshape(N, N, N)).reshape(-1) / N3
    ghat = np.fft.fftn(Fq.reshape(N, N, N)).reshape(-1) / N3
    W = (tab.w_rho[:, None] * tab.w_sigma[None, :]).reshape(-1)              # [N_rho*M]
    a = tab.a.reshape(-1, N3)
    b = tab.b[p, q].reshape(-1, N3)
    E1 = np.exp(1j * muq * a)                                                # beta_r(l)  of Eq. 13
    E2 = np.exp(-1j * mup * a)                                               # gamma_r(m) of Eq. 13
    cvec = tab.c[p, q]

    def kernel_row(zl, zk):
        Gplus = np.einsum("r,rm,r,rm->m", W, b[:, zk], E1[:, zl], E2)        # sum_{r,s} alpha(k) beta(l) gamma(m)
        return Gplus - cvec                                                  # G+(l,m) - G-(m)

    Q = np.real(_to_physical(N, _accumulate(N, fhat, ghat, kernel_row, wrap)))
    return tab.beta[p, q] * Q if scale_beta else Q


def galerkin_exact_vhs(tab: Tables, p, q, Fp, Fq, wrap=True, n_gl=96, scale_beta=True):
    """Full kernel modes of Eq. 12 for eta = 0 (VHS):
       G+(l,m) = int_0^R rho^{gam+2} 4pi sinc_u(mu_q rho' |l+m|) 4pi sinc_u(rho' |mu_q l - mu_p m|) drho
       G-(m)   = int_0^R rho^{gam+2} 4pi 4pi sinc_u(rho' |m|) drho,          rho' = pi rho / L."""
    assert tab.eta[p, q] == 0.0
    N = tab.N
    N3 = N ** 3
    mp, mq = tab.mass[p], tab.mass[q]
    muq, mup = mq / (mp + mq), mp / (mp + mq)
    g = tab.gam[p, q]
    x, w = np.polynomial.legendre.leggauss(n_gl)
    rho, wr = 0.5 * tab.R * (x + 1.0), 0.5 * tab.R * w
    rp = pi * rho / tab.L
    fhat = np.fft.fftn(Fp.reshape(N, N, N)).reshape(-1) / N3
    ghat = np.fft.fftn(Fq.reshape(N, N, N)).reshape(-1) / N3
    v = freq_index(N).astype(np.float64)
    idx = _index_grid(N)
    lv = v[idx]                                                              # [N^3][3] signed frequencies
    Gminus = (wr[:, None] * rho[:, None] ** (g + 2.0) * (4 * pi) ** 2
              * sinc_u(rp[:, None] * np.linalg.norm(lv, axis=1)[None, :])).sum(axis=0)

    def kernel_row(zl, zk):
        l = lv[zl]
        knorm = np.linalg.norm(lv[zk], axis=1) if wrap else np.linalg.norm(l[None, :] + lv, axis=1)
        dnorm = np.linalg.norm(muq * l[None, :] - mup * lv, axis=1)
        Gplus = (wr[:, None] * rho[:, None] ** (g + 2.0) * (4 * pi) ** 2
                 * sinc_u(muq * rp[:, None] * knorm[None, :]) * sinc_u(rp[:, None] * dnorm[None, :])).sum(axis=0)
        return Gplus - Gminus

    Q = np.real(_to_physical(N, _accumulate(N, fhat, ghat, kernel_row, wrap)))
    return tab.beta[p, q] * Q if scale_beta else Q

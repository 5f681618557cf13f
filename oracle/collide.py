"""Algorithm 2 of PAPER.md: the collision operator Q^(pq), verbatim.
ORACLE -- test infrastructure, numpy fp64 / complex128, no fusion or reordering.

FFT convention (reading C-3): fft = unnormalised forward DFT with kernel e^{-2 pi i jk/N}
(numpy.fft.fftn), ifft = 1/N^3-normalised inverse (numpy.fft.ifftn) -- the Octave convention
the paper refers to.
"""
import numpy as np

from .tables import Tables


def collide_pair(tab: Tables, p: int, q: int, Fp: np.ndarray, Fq: np.ndarray, scale_beta=True) -> np.ndarray:
    """Q^(pq)(f^(p), f^(q)) on the N^3 grid (flattened).  Algo 2, one spatial point, one pair."""
    N = tab.N
    mp, mq = tab.mass[p], tab.mass[q]
    shape = (N, N, N)
    # step 1
    FTf = np.fft.fftn(Fp.reshape(shape))
    FTg = np.fft.fftn(Fq.reshape(shape))
    QG = np.zeros(shape, dtype=np.complex128)
    for x in range(tab.N_rho):                                               # step 2
        for y in range(tab.M):                                               # step 3
            axy = tab.a[x, y].reshape(shape)
            t1 = np.exp(1j * mq / (mp + mq) * axy) * FTf                     # step 4
            t2 = np.exp(-1j * mp / (mq + mp) * axy) * FTg                    # step 5
            t3 = np.fft.fftn(np.fft.ifftn(t1) * np.fft.ifftn(t2))            # step 6
            QG += tab.w_rho[x] * tab.w_sigma[y] * tab.b[p, q, x, y].reshape(shape) * t3   # step 7
    # step 10; the imaginary part is discarded (reading Q-4)
    Q = np.real(np.fft.ifftn(QG) - Fp.reshape(shape) * np.fft.ifftn(tab.c[p, q].reshape(shape) * FTg))
    if scale_beta:
        Q = tab.beta[p, q] * Q
    return Q.reshape(-1)


def collide_pairs(tab: Tables, f: np.ndarray) -> np.ndarray:
    """f[nx][ns][N^3] -> Qpq[nx][ns(p)][ns(q)][N^3] = beta_pq Q^(pq)(f_p, f_q)."""
    nx, ns, N3 = f.shape
    out = np.empty((nx, ns, ns, N3))
    for x in range(nx):
        for p in range(ns):
            for q in range(ns):
                out[x, p, q] = collide_pair(tab, p, q, f[x, p], f[x, q])
    return out


def collide(tab: Tables, f: np.ndarray) -> np.ndarray:
    """f[nx][ns][N^3] -> Q[nx][ns][N^3] = sum_q beta_pq Q^(pq)   (right-hand side of Eq. 1)."""
    return collide_pairs(tab, f).sum(axis=2)


def nyquist_filter(f: np.ndarray, N: int) -> np.ndarray:
    """P f: the samples with the three Nyquist planes of their spectrum (index N/2 along any axis, frequency
    -N/2) set to zero.  f[..., N^3] -> same shape.  Not part of the paper's algorithm: the operator
    Q(P f_p, P f_q) is the variant of SURVEY.md section 8(f) item 2 (`dgfs_params.nyquist_filter`), for which
    every shifted field of Algorithm 2 is exactly real.  Written spectrally here; the CUDA path does it in
    physical space (alternating means), so the two share no formula."""
    shape = f.shape
    g = np.fft.fftn(f.reshape(shape[:-1] + (N, N, N)), axes=(-3, -2, -1))
    H = N // 2
    g[..., H, :, :] = 0.0
    g[..., :, H, :] = 0.0
    g[..., :, :, H] = 0.0
    return np.real(np.fft.ifftn(g, axes=(-3, -2, -1))).reshape(shape)

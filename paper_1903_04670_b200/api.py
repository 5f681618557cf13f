"""ctypes binding of include/dgfs.h.  Same names as the C ABI; argument marshalling only.

Device buffers are torch CUDA tensors (fp64, contiguous); the library receives their
`data_ptr()` and the current torch CUDA stream.  Nothing here computes: if `libdgfs.so` is
missing or there is no CUDA device the calls raise `DgfsError` (no CPU fallback).
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libdgfs.so")
_lib = None

# every symbol include/dgfs.h declares
ABI_SYMBOLS = (
    "dgfs_create", "dgfs_destroy", "dgfs_last_error", "dgfs_collide", "dgfs_collide_pairs",
    "dgfs_workspace_bytes", "dgfs_reserve", "dgfs_get_quadrature", "dgfs_get_tables",
    "dgfs_flops_per_pair_eval", "dgfs_step", "dgfs_step_euler", "dgfs_advect_rhs",
    "dgfs_launch_count", "dgfs_profile_enable", "dgfs_profile_count", "dgfs_profile_get",
    "dgfs_profile_reset", "dgfs_collide_host", "dgfs_measure_fp64_peak", "dgfs_table_bytes", "dgfs_measure_dft",
    "dgfs_collide_noalloc", "dgfs_measure_fp64_mix",
)

DGFS_OK, DGFS_EINVAL, DGFS_ECUDA, DGFS_ENOMEM, DGFS_ENOSUP = 0, -1, -2, -3, -4


class DgfsError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libdgfs error %d: %s" % (code, msg))
        self.code = code


_dp = C.POINTER(C.c_double)


class _Params(C.Structure):
    _fields_ = [
        ("ns", C.c_int), ("mass", _dp), ("omega", _dp), ("alpha", _dp), ("kn", _dp),
        ("prefactor", _dp), ("N", C.c_int), ("N_rho", C.c_int), ("M", C.c_int),
        ("L", C.c_double), ("R", C.c_double), ("sigma", _dp), ("w_sigma", _dp),
        ("table_mode", C.c_int), ("M_pre", C.c_int), ("sigma_pre", _dp), ("w_pre", _dp),
        ("device", C.c_int), ("nyquist_filter", C.c_int), ("precision", C.c_int),
    ]


class _Mesh(C.Structure):
    _fields_ = [("ne", C.c_int), ("order", C.c_int), ("x0", C.c_double), ("x1", C.c_double),
                ("wall_T", C.c_double * 2), ("wall_u", (C.c_double * 3) * 2)]


class Mesh1D:
    """dgfs_mesh1d: ne uniform elements on [x0, x1], degree `order`, diffuse walls."""

    def __init__(self, ne, order, x0=0.0, x1=1.0, wall_T=(1.0, 1.0), wall_u=((0, 0, 0), (0, 0, 0))):
        self.ne, self.order, self.x0, self.x1 = int(ne), int(order), float(x0), float(x1)
        self.wall_T = tuple(float(t) for t in wall_T)
        self.wall_u = tuple(tuple(float(v) for v in u) for u in wall_u)

    def _c(self):
        m = _Mesh()
        m.ne, m.order, m.x0, m.x1 = self.ne, self.order, self.x0, self.x1
        for i in range(2):
            m.wall_T[i] = self.wall_T[i]
            for d in range(3):
                m.wall_u[i][d] = self.wall_u[i][d]
        return m


def library_path():
    return _LIB_PATH


def load_library():
    """dlopen libdgfs.so (built in-tree by paper_1903_04670_b200.build).  Raises if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise DgfsError(DGFS_ECUDA, "%s not built: run `python -m paper_1903_04670_b200.build` "
                        "(there is no CPU fallback)" % _LIB_PATH)
    lib = C.CDLL(_LIB_PATH)
    vp, ip = C.c_void_p, C.c_int
    lib.dgfs_create.argtypes = [C.POINTER(_Params), C.POINTER(vp)]
    lib.dgfs_create.restype = ip
    lib.dgfs_destroy.argtypes = [vp]
    lib.dgfs_destroy.restype = None
    lib.dgfs_last_error.argtypes = [vp]
    lib.dgfs_last_error.restype = C.c_char_p
    for name in ("dgfs_collide", "dgfs_collide_pairs", "dgfs_collide_noalloc"):
        fn = getattr(lib, name)
        fn.argtypes = [vp, vp, vp, ip, vp]
        fn.restype = ip
    lib.dgfs_collide_host.argtypes = [vp, vp, vp, ip]
    lib.dgfs_collide_host.restype = ip
    lib.dgfs_measure_fp64_peak.argtypes = [ip, C.c_double, _dp, _dp]
    lib.dgfs_measure_fp64_peak.restype = ip
    lib.dgfs_measure_fp64_mix.argtypes = [ip, ip, ip, C.c_double, _dp, _dp]
    lib.dgfs_measure_fp64_mix.restype = ip
    lib.dgfs_workspace_bytes.argtypes = [vp, ip]
    lib.dgfs_workspace_bytes.restype = C.c_size_t
    lib.dgfs_measure_dft.argtypes = [ip, ip, ip, C.c_double, _dp, _dp]
    lib.dgfs_measure_dft.restype = ip
    lib.dgfs_table_bytes.argtypes = [vp]
    lib.dgfs_table_bytes.restype = C.c_size_t
    lib.dgfs_reserve.argtypes = [vp, ip]
    lib.dgfs_reserve.restype = ip
    lib.dgfs_get_quadrature.argtypes = [vp, _dp, _dp, _dp, _dp, _dp, _dp]
    lib.dgfs_get_quadrature.restype = ip
    lib.dgfs_get_tables.argtypes = [vp, ip, ip, vp, vp, vp]
    lib.dgfs_get_tables.restype = ip
    lib.dgfs_flops_per_pair_eval.argtypes = [vp, ip, ip]
    lib.dgfs_flops_per_pair_eval.restype = C.c_double
    lib.dgfs_launch_count.argtypes = [vp]
    lib.dgfs_launch_count.restype = C.c_longlong
    lib.dgfs_profile_enable.argtypes = [vp, ip]
    lib.dgfs_profile_enable.restype = ip
    lib.dgfs_profile_count.argtypes = [vp]
    lib.dgfs_profile_count.restype = ip
    lib.dgfs_profile_get.argtypes = [vp, ip, C.POINTER(C.c_char_p), C.POINTER(C.c_longlong), _dp, _dp]
    lib.dgfs_profile_get.restype = ip
    lib.dgfs_profile_reset.argtypes = [vp]
    lib.dgfs_profile_reset.restype = ip
    lib.dgfs_step.argtypes = [vp, C.POINTER(_Mesh), vp, C.c_double, ip, vp]
    lib.dgfs_step.restype = ip
    lib.dgfs_step_euler.argtypes = [vp, C.POINTER(_Mesh), vp, C.c_double, ip, vp]
    lib.dgfs_step_euler.restype = ip
    lib.dgfs_advect_rhs.argtypes = [vp, C.POINTER(_Mesh), vp, vp, vp]
    lib.dgfs_advect_rhs.restype = ip
    _lib = lib
    return lib


def exported_symbols():
    """Names from ABI_SYMBOLS that the built library exports (no compute calls)."""
    lib = load_library()
    return [s for s in ABI_SYMBOLS if hasattr(lib, s)]


def _arr(x, n=None):
    if x is None:
        return None, None
    a = np.ascontiguousarray(np.asarray(x, dtype=np.float64).reshape(-1))
    if n is not None and a.size != n:
        raise ValueError("expected %d values, got %d" % (n, a.size))
    return a, a.ctypes.data_as(_dp)


def _check(ctx, rc):
    if rc != DGFS_OK:
        msg = load_library().dgfs_last_error(ctx)
        raise DgfsError(rc, msg.decode() if msg else "")


def dgfs_last_error(ctx=None):
    msg = load_library().dgfs_last_error(ctx)
    return msg.decode() if msg else ""


def dgfs_create(mass, omega, alpha, N, N_rho, M, L, kn=None, prefactor=None, R=0.0, sigma=None,
                w_sigma=None, table_mode=0, sigma_pre=None, w_pre=None, device=0, nyquist_filter=False, precision=0):
    """Algorithm 1 on the device.  Returns the opaque context handle."""
    lib = load_library()
    ns = len(np.asarray(mass).reshape(-1))
    keep = []
    p = _Params()
    p.ns = ns
    for name, val, n in (("mass", mass, ns), ("omega", omega, ns * ns), ("alpha", alpha, ns * ns),
                         ("kn", kn, ns * ns), ("prefactor", prefactor, ns * ns),
                         ("sigma", sigma, 3 * M), ("w_sigma", w_sigma, M),
                         ("sigma_pre", sigma_pre, None), ("w_pre", w_pre, None)):
        a, ptr = _arr(val, n)
        keep.append(a)
        if ptr is not None:
            setattr(p, name, ptr)
    p.N, p.N_rho, p.M, p.L, p.R = int(N), int(N_rho), int(M), float(L), float(R or 0.0)
    p.table_mode = int(table_mode)
    p.M_pre = 0 if w_pre is None else len(np.asarray(w_pre).reshape(-1))
    p.device = int(device)
    p.nyquist_filter = int(bool(nyquist_filter))
    p.precision = int(precision)
    out = C.c_void_p()
    rc = lib.dgfs_create(C.byref(p), C.byref(out))
    _check(None, rc)
    return out


def dgfs_destroy(ctx):
    load_library().dgfs_destroy(ctx)


def _stream_ptr():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev(t, who):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise ValueError("%s must be a contiguous fp64 CUDA tensor" % who)
    return C.c_void_p(t.data_ptr())


def dgfs_collide(ctx, f, Q, nx):
    """Q[x][p][:] = sum_q beta_pq Q^(pq)(f[x][p], f[x][q])  on the current torch stream."""
    _check(ctx, load_library().dgfs_collide(ctx, _dev(f, "f"), _dev(Q, "Q"), int(nx), _stream_ptr()))


def dgfs_collide_noalloc(ctx, f, Q, nx):
    """dgfs_collide out of the library's static device scratch (no device allocation; include/dgfs.h)."""
    _check(ctx, load_library().dgfs_collide_noalloc(ctx, _dev(f, "f"), _dev(Q, "Q"), int(nx), _stream_ptr()))


def dgfs_collide_pairs(ctx, f, Qpq, nx):
    _check(ctx, load_library().dgfs_collide_pairs(ctx, _dev(f, "f"), _dev(Qpq, "Qpq"), int(nx), _stream_ptr()))


def _host(t, who, n):
    """Host fp64 buffer (numpy array or CPU torch tensor, contiguous) -> void*."""
    if isinstance(t, np.ndarray):
        if t.dtype != np.float64 or not t.flags.c_contiguous or t.size != n:
            raise ValueError("%s must be a C-contiguous float64 array of %d values" % (who, n))
        return C.c_void_p(t.ctypes.data)
    import torch
    if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
            and t.numel() == n):
        raise ValueError("%s must be a contiguous fp64 host tensor of %d values" % (who, n))
    return C.c_void_p(t.data_ptr())


def dgfs_collide_host(ctx, f_host, Q_host, nx, ns, N3):
    """dgfs_collide with HOST buffers: copies in, kernels and copies out all inside the call."""
    n = int(nx) * int(ns) * int(N3)
    _check(ctx, load_library().dgfs_collide_host(ctx, _host(f_host, "f_host", n), _host(Q_host, "Q_host", n), int(nx)))


def dgfs_measure_fp64_peak(device=0, seconds=1.0):
    """(burst, sustained) TFLOP/s of the FP64 DFMA pipe, measured by the library."""
    a, b = C.c_double(), C.c_double()
    rc = load_library().dgfs_measure_fp64_peak(int(device), float(seconds), C.byref(a), C.byref(b))
    if rc != DGFS_OK:
        raise DgfsError(rc, "dgfs_measure_fp64_peak failed")
    return a.value, b.value


def dgfs_measure_fp64_mix(device=0, n_dfma=8, n_dmma=8, seconds=0.5):
    """(DFMA TFLOP/s, DMMA TFLOP/s) of a kernel that issues both kinds of FP64 instruction side by side."""
    a, b = C.c_double(), C.c_double()
    rc = load_library().dgfs_measure_fp64_mix(int(device), int(n_dfma), int(n_dmma), float(seconds), C.byref(a), C.byref(b))
    if rc != DGFS_OK:
        raise DgfsError(rc, "dgfs_measure_fp64_mix failed")
    return a.value, b.value


def dgfs_workspace_bytes(ctx, nx):
    return int(load_library().dgfs_workspace_bytes(ctx, int(nx)))


def dgfs_reserve(ctx, nx):
    _check(ctx, load_library().dgfs_reserve(ctx, int(nx)))


def dgfs_measure_dft(device, N, method, seconds=0.5):
    """(complex DFTs of length N per second, relative error of one transform): method 0 register FFT, 1 FP64 MMA."""
    rate, err = C.c_double(), C.c_double()
    _check(None, load_library().dgfs_measure_dft(int(device), int(N), int(method), float(seconds), C.byref(rate), C.byref(err)))
    return rate.value, err.value


def dgfs_table_bytes(ctx):
    return int(load_library().dgfs_table_bytes(ctx))


def dgfs_flops_per_pair_eval(ctx, p, q):
    return float(load_library().dgfs_flops_per_pair_eval(ctx, int(p), int(q)))


def dgfs_get_quadrature(ctx, ns, N_rho, M):
    R = C.c_double()
    rho, w_rho = np.empty(N_rho), np.empty(N_rho)
    sigma, w_sigma, beta = np.empty((M, 3)), np.empty(M), np.empty((ns, ns))
    P = lambda a: a.ctypes.data_as(_dp)
    _check(ctx, load_library().dgfs_get_quadrature(ctx, C.byref(R), P(rho), P(w_rho), P(sigma), P(w_sigma), P(beta)))
    return dict(R=R.value, rho=rho, w_rho=w_rho, sigma=sigma, w_sigma=w_sigma, beta=beta)


def dgfs_get_tables(ctx, p, q, N, N_rho, M, want=("a", "b", "c")):
    """Host copies of Algorithm 1's tables for pair (p,q): a real, b and c complex128."""
    N3 = N ** 3
    a = np.empty((N_rho, M, N3)) if "a" in want else None
    b = np.empty((N_rho, M, N3), dtype=np.complex128) if "b" in want else None
    c = np.empty(N3, dtype=np.complex128) if "c" in want else None
    vp = lambda x: C.c_void_p(x.ctypes.data) if x is not None else None
    _check(ctx, load_library().dgfs_get_tables(ctx, int(p), int(q), vp(a), vp(b), vp(c)))
    return a, b, c


def dgfs_launch_count(ctx):
    return int(load_library().dgfs_launch_count(ctx))


def dgfs_profile_enable(ctx, on):
    _check(ctx, load_library().dgfs_profile_enable(ctx, int(bool(on))))


def dgfs_profile_reset(ctx):
    _check(ctx, load_library().dgfs_profile_reset(ctx))


def dgfs_profile_count(ctx):
    return int(load_library().dgfs_profile_count(ctx))


def dgfs_profile_get(ctx, i):
    name, n, ms, fl = C.c_char_p(), C.c_longlong(), C.c_double(), C.c_double()
    _check(ctx, load_library().dgfs_profile_get(ctx, int(i), C.byref(name), C.byref(n), C.byref(ms), C.byref(fl)))
    return dict(name=name.value.decode(), launches=n.value, ms=ms.value, flops=fl.value)


def dgfs_step(ctx, mesh, f, dt, nsteps):
    m = mesh._c()
    _check(ctx, load_library().dgfs_step(ctx, C.byref(m), _dev(f, "f"), float(dt), int(nsteps), _stream_ptr()))


def dgfs_step_euler(ctx, mesh, f, dt, nsteps):
    m = mesh._c()
    _check(ctx, load_library().dgfs_step_euler(ctx, C.byref(m), _dev(f, "f"), float(dt), int(nsteps), _stream_ptr()))


def dgfs_advect_rhs(ctx, mesh, f, rhs):
    m = mesh._c()
    _check(ctx, load_library().dgfs_advect_rhs(ctx, C.byref(m), _dev(f, "f"), _dev(rhs, "rhs"), _stream_ptr()))


class Dgfs:
    """Convenience owner of one context (create -> collide -> destroy)."""

    def __init__(self, mass, omega, alpha, N, N_rho, M, L, **kw):
        self.ns = len(np.asarray(mass).reshape(-1))
        self.N, self.N_rho, self.M, self.L = int(N), int(N_rho), int(M), float(L)
        self.N3 = self.N ** 3
        self.ctx = dgfs_create(mass, omega, alpha, N, N_rho, M, L, **kw)

    @classmethod
    def from_config(cls, cfg, **kw):
        if getattr(cfg, "kn", ()):
            kw.setdefault("kn", cfg.kn)
        return cls(cfg.mass, cfg.omega, cfg.alpha, cfg.N, cfg.N_rho, cfg.M, cfg.L, **kw)

    def close(self):
        if self.ctx is not None:
            dgfs_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def collide(self, f, out=None):
        import torch
        nx = f.shape[0]
        if out is None:
            out = torch.empty((nx, self.ns, self.N3), dtype=torch.float64, device=f.device)
        dgfs_collide(self.ctx, f, out, nx)
        return out

    def collide_noalloc(self, f, out):
        """dgfs_collide_noalloc: `out` is the caller's ([nx][ns][N^3], fp64, CUDA); nothing is allocated."""
        dgfs_collide_noalloc(self.ctx, f, out, f.shape[0])
        return out

    def collide_pairs(self, f, out=None):
        import torch
        nx = f.shape[0]
        if out is None:
            out = torch.empty((nx, self.ns, self.ns, self.N3), dtype=torch.float64, device=f.device)
        dgfs_collide_pairs(self.ctx, f, out, nx)
        return out

    def collide_host(self, f_host, out_host=None):
        """End-to-end call with HOST numpy / CPU-torch buffers (dgfs_collide_host)."""
        nx = int(f_host.shape[0])
        if out_host is None:
            out_host = np.empty((nx, self.ns, self.N3)) if isinstance(f_host, np.ndarray) else f_host.new_empty(
                (nx, self.ns, self.N3))
        dgfs_collide_host(self.ctx, f_host, out_host, nx, self.ns, self.N3)
        return out_host

    def quadrature(self):
        return dgfs_get_quadrature(self.ctx, self.ns, self.N_rho, self.M)

    def tables(self, p, q, want=("a", "b", "c")):
        return dgfs_get_tables(self.ctx, p, q, self.N, self.N_rho, self.M, want)

    def flops_per_pair_eval(self, p, q):
        return dgfs_flops_per_pair_eval(self.ctx, p, q)

    def launch_count(self):
        return dgfs_launch_count(self.ctx)

    def profile(self, on=None, reset=False):
        """Per-kernel-class accumulators (list of dicts); `on` switches the event bracketing."""
        if on is not None:
            dgfs_profile_enable(self.ctx, on)
        if reset:
            dgfs_profile_reset(self.ctx)
        return [dgfs_profile_get(self.ctx, i) for i in range(dgfs_profile_count(self.ctx))]

    def reserve(self, nx):
        dgfs_reserve(self.ctx, nx)

    def workspace_bytes(self, nx):
        return dgfs_workspace_bytes(self.ctx, nx)

    def table_bytes(self):
        return dgfs_table_bytes(self.ctx)

"""Thin Python binding of the C ABI in include/dse.h (argument marshalling only).

PyTorch is used for device memory and streams; every step of the path runs in the CUDA kernels of
libdse_b200.so.  There is no CPU fallback: if the library is missing or there is no CUDA device the
calls raise.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdse_b200.so")

# every symbol include/dse.h and include/dse_diag.h declare (tests/test_abi.py checks the list against the headers)
EXPORTS = [
    "dse_create", "dse_create_with_tables", "dse_destroy", "dse_residual", "dse_jacobian", "dse_newton_step",
    "dse_newton_solve", "dse_lu_solve", "dse_jacobian_host", "dse_n_ext", "dse_get_tables", "dse_launch_count",
    "dse_kernel_info", "dse_set_timing", "dse_get_timing", "dse_gauss_legendre", "dse_gauss_legendre_noalloc", "dse_schwinger",
    "dse_dressing",
    "dse_jacobian_fd", "dse_strerror", "dse_last_error",
    "dse_probe", "dse_probe_flops", "dse_diag_set_tail_polls", "dse_diag_phase_stamps",
]

DSE_FLAG_GEOMETRY_CACHE = 1
DSE_FLAG_ANGULAR_TANH_SINH = 2
DSE_FLAG_RADIAL_SPLIT = 4
DSE_FLAG_USER_TABLES = 8
DSE_FLAG_CONST_COEF = 16
DSE_FLAG_PER_SYSTEM_KERNELS = 32
DSE_EBUSY = -4
PROBE_KINDS = {"dfma": 0, "dmma": 1, "dfma_3reg": 2, "dfma_reuse": 3, "dfma_dmma": 4, "dfma_lds": 5}
LATENCY_PROBE_KINDS = {"lat_redux_max": 6, "lat_redux_or": 7, "lat_ballot_ffs_shfl": 8, "lat_shfl": 9, "lat_dfma": 10}


class DseParams(C.Structure):
    _fields_ = [
        ("n_cheb", C.c_int32), ("n_r", C.c_int32), ("n_theta", C.c_int32), ("n_batch", C.c_int32),
        ("eps2", C.c_double), ("L2", C.c_double), ("alpha_mu", C.c_double), ("n_colors", C.c_double),
        ("x_G", C.c_double), ("x_Z", C.c_double), ("delta", C.c_double),
        ("ir_exp_G", C.c_double), ("ir_exp_Z", C.c_double), ("uv_omega", C.c_double),
        ("flags", C.c_int32), ("n_r_ir", C.c_int32),
    ]


class DseTables(C.Structure):
    _fields_ = [("x_ext", C.c_void_p), ("y", C.c_void_p), ("Wy", C.c_void_p), ("theta", C.c_void_p), ("Omega", C.c_void_p)]


class DseError(RuntimeError):
    def __init__(self, msg, code=None):
        super().__init__(msg)
        self.code = code


_lib = None


def load_library():
    """Loads libdse_b200.so (raises if it has not been built: python -m paper_1206_1779_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise DseError(f"{LIB_PATH} not found: build it with `python -m paper_1206_1779_b200.build` "
                       "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, dp = C.c_void_p, C.c_void_p
    L.dse_create.argtypes = [C.POINTER(DseParams), C.POINTER(vp)]
    L.dse_create_with_tables.argtypes = [C.POINTER(DseParams), C.POINTER(DseTables), C.POINTER(vp)]
    L.dse_destroy.argtypes = [vp]
    L.dse_residual.argtypes = [vp, dp, dp, dp, vp]
    L.dse_jacobian.argtypes = [vp, dp, dp, dp, dp, vp]
    L.dse_newton_step.argtypes = [vp, dp, dp, C.c_double, dp, vp]
    L.dse_newton_solve.argtypes = [vp, dp, dp, C.c_double, C.c_double, C.c_double, C.c_int32, dp, vp]
    L.dse_lu_solve.argtypes = [vp, C.c_int32, C.c_int32, dp, dp, dp, dp, vp]
    L.dse_jacobian_host.argtypes = [vp, dp, dp, dp, dp]
    L.dse_n_ext.argtypes = [vp]
    L.dse_get_tables.argtypes = [vp, dp, dp, dp, dp, dp]
    L.dse_launch_count.argtypes = [vp]
    L.dse_launch_count.restype = C.c_int64
    L.dse_kernel_info.argtypes = [vp, C.POINTER(C.c_int32 * 8)]
    L.dse_set_timing.argtypes = [vp, C.c_int32]
    L.dse_get_timing.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
    L.dse_jacobian_fd.argtypes = [vp, dp, dp, C.c_double, dp, vp]
    L.dse_gauss_legendre.argtypes = [C.c_int32, dp, dp, dp, vp]
    L.dse_gauss_legendre_noalloc.argtypes = [C.c_int32, dp, dp, vp]
    L.dse_schwinger.argtypes = [vp, dp, C.c_int32, C.c_double, C.c_double, dp, C.c_int32, dp, dp, vp]
    L.dse_dressing.argtypes = [vp, dp, dp, C.c_int32, dp, dp, dp, vp]
    L.dse_probe.argtypes = [C.c_int32, C.c_int32, C.c_int32, dp, vp]
    L.dse_diag_set_tail_polls.argtypes = [vp, C.c_int32]
    L.dse_diag_phase_stamps.argtypes = [C.c_int32, vp, C.c_int32]
    L.dse_probe_flops.argtypes = [C.c_int32, C.c_int32, C.c_int32]
    L.dse_probe_flops.restype = C.c_double
    L.dse_strerror.argtypes = [C.c_int]
    L.dse_strerror.restype = C.c_char_p
    L.dse_last_error.restype = C.c_char_p
    _lib = L
    return L


def _check(rc):
    if rc != 0:
        L = load_library()
        raise DseError(f"{L.dse_strerror(rc).decode()} ({rc}): {L.dse_last_error().decode()}", rc)


def params_from_workload(w, n_batch=None, flags=0):
    if getattr(w, "angular_rule", 0) == 1:
        flags |= DSE_FLAG_ANGULAR_TANH_SINH
    if getattr(w, "radial_split", 0) == 1:
        flags |= DSE_FLAG_RADIAL_SPLIT
    return DseParams(w.n_cheb, w.n_r, w.n_theta, w.n_batch if n_batch is None else n_batch, w.eps2, w.L2,
                     w.alpha_mu, w.n_colors, w.x_G, w.x_Z, w.delta, w.ir_exp_G, w.ir_exp_Z, w.uv_omega, flags, getattr(w, "n_ir", 0))


def _stream_ptr(stream=None):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _dev_ptr(t, n=None):
    import torch
    assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous(), "need a contiguous CUDA float64 tensor"
    if n is not None:
        assert t.numel() >= n, (t.numel(), n)
    return C.c_void_p(t.data_ptr())


class Dse:
    """dse_handle wrapper.  Method names mirror the C ABI: residual / jacobian / newton_step / lu_solve."""

    def __init__(self, params: DseParams, tables: dict = None):
        """tables (with DSE_FLAG_USER_TABLES): dict of float64 numpy arrays x_ext, y, Wy, theta, Omega in the layout of
        dse_tables (include/dse.h) -> dse_create_with_tables."""
        import torch
        if not torch.cuda.is_available():
            raise DseError("no CUDA device: this library has no CPU fallback")
        self.lib = load_library()
        self.params = params
        h = C.c_void_p()
        if tables is not None:
            arrs = {k: np.ascontiguousarray(tables[k], dtype=np.float64) for k in ("x_ext", "y", "Wy", "theta", "Omega")}
            t = DseTables(*[C.c_void_p(arrs[k].ctypes.data) for k in ("x_ext", "y", "Wy", "theta", "Omega")])
            _check(self.lib.dse_create_with_tables(C.byref(params), C.byref(t), C.byref(h)))
        else:
            _check(self.lib.dse_create(C.byref(params), C.byref(h)))
        self._h = h
        self.N = params.n_cheb
        self.B = params.n_batch
        self.n_ext = self.lib.dse_n_ext(h)

    def close(self):
        if getattr(self, "_h", None):
            self.lib.dse_destroy(self._h)
            self._h = None

    __del__ = close

    # ---- the path ---------------------------------------------------------------------------------
    def residual(self, c, bc, F=None, stream=None):
        import torch
        if F is None:
            F = torch.empty((self.B, 2 * self.N), dtype=torch.float64, device=c.device)
        _check(self.lib.dse_residual(self._h, _dev_ptr(c, self.B * 2 * self.N), _dev_ptr(bc, 2 * self.B),
                                     _dev_ptr(F, self.B * 2 * self.N), _stream_ptr(stream)))
        return F

    def jacobian(self, c, bc, J=None, F=None, stream=None):
        import torch
        n = 2 * self.N
        if J is None:
            J = torch.empty((self.B, n, n), dtype=torch.float64, device=c.device)
        if F is None:
            F = torch.empty((self.B, n), dtype=torch.float64, device=c.device)
        _check(self.lib.dse_jacobian(self._h, _dev_ptr(c, self.B * n), _dev_ptr(bc, 2 * self.B),
                                     _dev_ptr(J, self.B * n * n), _dev_ptr(F, self.B * n), _stream_ptr(stream)))
        return J, F

    def jacobian_fd(self, c, bc, eps_rel=1e-6, stream=None):
        """Central finite-difference Newton matrix (the paper's eq.(38)): a self-check of the analytic one."""
        import torch
        n = 2 * self.N
        J = torch.empty((self.B, n, n), dtype=torch.float64, device=c.device)
        _check(self.lib.dse_jacobian_fd(self._h, _dev_ptr(c, self.B * n), _dev_ptr(bc, 2 * self.B), float(eps_rel),
                                        _dev_ptr(J), _stream_ptr(stream)))
        return J

    def newton_step(self, c, bc, rho=1.0, stats=None, stream=None):
        import torch
        if stats is None:
            stats = torch.empty((self.B, 4), dtype=torch.float64, device=c.device)
        _check(self.lib.dse_newton_step(self._h, _dev_ptr(c, self.B * 2 * self.N), _dev_ptr(bc, 2 * self.B),
                                        float(rho), _dev_ptr(stats, 4 * self.B), _stream_ptr(stream)))
        return stats

    def newton_solve(self, c, bc, rho=1.0, step_cap=0.0, tol=1e-12, max_iter=50, info=None, stream=None):
        """Whole Newton iteration on the device (one CUDA graph, no host round trips); c is updated in place.
        Returns info [n_batch, 6] = (steps, |Delta|inf, |F|inf, min |pivot|, last rho_n, status)."""
        import torch
        if info is None:
            info = torch.empty((self.B, 6), dtype=torch.float64, device=c.device)
        _check(self.lib.dse_newton_solve(self._h, _dev_ptr(c, self.B * 2 * self.N), _dev_ptr(bc, 2 * self.B), float(rho),
                                         float(step_cap), float(tol), int(max_iter), _dev_ptr(info, 6 * self.B),
                                         _stream_ptr(stream)))
        return info

    def lu_solve(self, A, b, stream=None):
        import torch
        n_sys, n = b.shape
        x = torch.empty_like(b)
        stats = torch.empty((n_sys, 4), dtype=torch.float64, device=b.device)
        _check(self.lib.dse_lu_solve(self._h, n, n_sys, _dev_ptr(A, n_sys * n * n), _dev_ptr(b), _dev_ptr(x),
                                     _dev_ptr(stats), _stream_ptr(stream)))
        return x, stats

    def schwinger(self, c, t, n_nodes, p2_min, p2_max, stream=None):
        """Delta(t) of eq.(20) for every system: returns a [n_batch, len(t)] tensor."""
        import torch
        out = torch.empty((self.B, t.numel()), dtype=torch.float64, device=c.device)
        work = torch.empty((5 + self.B) * n_nodes + 4, dtype=torch.float64, device=c.device)
        _check(self.lib.dse_schwinger(self._h, _dev_ptr(c, self.B * 2 * self.N), int(n_nodes), float(p2_min),
                                      float(p2_max), _dev_ptr(t), int(t.numel()), _dev_ptr(out), _dev_ptr(work),
                                      _stream_ptr(stream)))
        self._keep = work            # the call is asynchronous: keep the workspace alive until the next call
        return out

    def dressing(self, c, x, stream=None):
        """ln G(x), ln Z(x), alpha(x) = alpha(mu^2) G^2 Z for every system: three [n_batch, len(x)] tensors."""
        import torch
        n_x = x.numel()
        out = [torch.empty((self.B, n_x), dtype=torch.float64, device=c.device) for _ in range(3)]
        _check(self.lib.dse_dressing(self._h, _dev_ptr(c, self.B * 2 * self.N), _dev_ptr(x), n_x, _dev_ptr(out[0]),
                                     _dev_ptr(out[1]), _dev_ptr(out[2]), _stream_ptr(stream)))
        return tuple(out)

    def jacobian_host(self, c_host: np.ndarray, bc_host: np.ndarray, J_host: np.ndarray, F_host: np.ndarray):
        """Host buffers in, host buffers out (numpy float64, C-contiguous; pinned memory recommended)."""
        for a in (c_host, bc_host, F_host) + ((J_host,) if J_host is not None else ()):
            assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
        _check(self.lib.dse_jacobian_host(self._h, C.c_void_p(c_host.ctypes.data), C.c_void_p(bc_host.ctypes.data),
                                          C.c_void_p(J_host.ctypes.data) if J_host is not None else None,
                                          C.c_void_p(F_host.ctypes.data)))

    # ---- introspection ----------------------------------------------------------------------------
    def tables(self):
        p = self.params
        split = bool(p.flags & DSE_FLAG_RADIAL_SPLIT)
        nr = (2 if split else 1) * p.n_r + p.n_r_ir
        shape = (self.n_ext, nr) if split else (nr,)          # the split rule has one radial rule per external point
        out = dict(x_ext=np.empty(self.n_ext), y=np.empty(shape), Wy=np.empty(shape), theta=np.empty(p.n_theta),
                   Omega=np.empty(p.n_theta))
        _check(self.lib.dse_get_tables(self._h, *[C.c_void_p(out[k].ctypes.data)
                                                  for k in ("x_ext", "y", "Wy", "theta", "Omega")]))
        return out

    def set_timing(self, enable=True):
        _check(self.lib.dse_set_timing(self._h, 1 if enable else 0))

    def get_timing(self):
        """(total ms of the point kernel, launches) since set_timing(True)."""
        ms = C.c_double(); n = C.c_int64()
        _check(self.lib.dse_get_timing(self._h, C.byref(ms), C.byref(n)))
        return ms.value, n.value

    def launch_count(self):
        return int(self.lib.dse_launch_count(self._h))

    def set_tail_polls(self, polls):
        """include/dse_diag.h: polls an owner of the fused tail spends before it leaves its rows to the finishing CTA."""
        _check(self.lib.dse_diag_set_tail_polls(self._h, int(polls)))

    def kernel_info(self):
        a = (C.c_int32 * 8)()
        _check(self.lib.dse_kernel_info(self._h, C.byref(a)))
        return dict(grid=a[0], block=a[1], smem=a[2], regs=a[3], ctas_per_sm=a[4], sms=a[5],
                    variant=("generic", "pipelined", "batched-dmma")[a[6]], kernels_per_build=a[7])


def probe(kind, blocks, iters, sink, stream=None):
    """include/dse_diag.h: launches one fp64 throughput probe; returns the floating-point operations of the launch."""
    k = {**PROBE_KINDS, **LATENCY_PROBE_KINDS}[kind] if isinstance(kind, str) else int(kind)
    L = load_library()
    _check(L.dse_probe(k, blocks, iters, _dev_ptr(sink, blocks * 256), _stream_ptr(stream)))
    return L.dse_probe_flops(k, blocks, iters)


def phase_stamps(which):
    """include/dse_diag.h: the phase stamps of the last single-system build (which = 0) or one-CTA LU (which = 1) as an int64
    numpy array; needs a library built with -DDSE_PHASE_TIMING."""
    import numpy as np
    n = 148 * 16 * 16 if which == 0 else 8192
    out = np.zeros(n, dtype=np.int64)
    rc = load_library().dse_diag_phase_stamps(int(which), C.c_void_p(out.ctypes.data), n)
    if rc < 0:
        _check(rc)
    return out[:rc]


def gauss_legendre(n, device="cuda", stream=None):
    """n-point Gauss-Legendre rule generated on the device: (x[n] ascending, w[n])."""
    import torch
    x = torch.empty(n, dtype=torch.float64, device=device)
    w = torch.empty(n, dtype=torch.float64, device=device)
    work = torch.empty(2 * (n + 2), dtype=torch.float64, device=device)
    _check(load_library().dse_gauss_legendre(int(n), _dev_ptr(x), _dev_ptr(w), _dev_ptr(work), _stream_ptr(stream)))
    import torch.cuda
    torch.cuda.current_stream().synchronize()
    return x, w


GL_NOALLOC_MAX_N = 1 << 17


def gauss_legendre_noalloc(n, x, w, stream=None):
    """dse_gauss_legendre_noalloc: writes the n-point rule into the caller's x[n], w[n]; the library allocates nothing (its
    scratch is a static device array; n <= GL_NOALLOC_MAX_N; calls that overlap on the GPU race -- include/dse.h)."""
    _check(load_library().dse_gauss_legendre_noalloc(int(n), _dev_ptr(x, n), _dev_ptr(w, n), _stream_ptr(stream)))


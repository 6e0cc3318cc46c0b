"""ctypes loader for the CPU oracle (TEST INFRASTRUCTURE, not the product).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It imports nothing from paper_1206_1779_b200 (the CUDA path) and vice versa.
Every function is a thin marshalling wrapper around oracle/dse_oracle.c; the passage each follows
is cited there.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
_dp = C.POINTER(C.c_double)


class OrcParams(C.Structure):
    _fields_ = [
        ("n_cheb", C.c_int32), ("n_r", C.c_int32), ("n_theta", C.c_int32), ("angular_rule", C.c_int32),
        ("eps2", C.c_double), ("L2", C.c_double), ("alpha_mu", C.c_double), ("n_colors", C.c_double),
        ("x_G", C.c_double), ("x_Z", C.c_double), ("delta", C.c_double),
        ("ir_exp_G", C.c_double), ("ir_exp_Z", C.c_double), ("uv_omega", C.c_double),
        ("n_ir", C.c_int32), ("radial_split", C.c_int32),
    ]


def make_params(n_cheb, n_r, n_theta, eps2, L2, x_G, x_Z, alpha_mu=1.0, n_colors=3.0, delta=-9.0 / 44.0,
                ir_exp_G=-0.595353, ir_exp_Z=2 * 0.595353, uv_omega=None, angular_rule=0, n_ir=0, radial_split=0):
    if uv_omega is None:
        uv_omega = 11.0 * n_colors * alpha_mu / (12.0 * np.pi)
    return OrcParams(int(n_cheb), int(n_r), int(n_theta), int(angular_rule), float(eps2), float(L2), float(alpha_mu),
                     float(n_colors), float(x_G), float(x_Z), float(delta), float(ir_exp_G), float(ir_exp_Z),
                     float(uv_omega), int(n_ir), int(radial_split))


def _ptr(a):
    return a.ctypes.data_as(_dp)


def _f64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


class Oracle:
    """One loaded oracle library; long_double=True loads the extended-precision build."""

    def __init__(self, long_double=False):
        libs = _build.build()
        self.lib = C.CDLL(libs["libdse_oracle_ld.so" if long_double else "libdse_oracle.so"])
        L = self.lib
        L.orc_gauss_legendre.argtypes = [C.c_int, _dp, _dp]
        L.orc_cheb_phi.argtypes = [C.c_int, C.c_double, _dp]
        L.orc_radial_rule_split.argtypes = [C.POINTER(OrcParams), C.c_double, _dp, _dp]
        L.orc_gl_node.argtypes = [C.c_int, C.c_int, _dp, _dp]
        L.orc_schwinger.argtypes = [C.POINTER(OrcParams), _dp, C.c_int, C.c_double, C.c_double, C.c_int, _dp, _dp]
        L.orc_schwinger_terms.argtypes = [C.POINTER(OrcParams), _dp, C.c_int, C.c_double, C.c_double, C.c_int, C.c_int, _dp, _dp]
        L.orc_schwinger_sum.argtypes = [C.c_int, _dp, _dp, C.c_int, _dp, _dp]
        for name in ("orc_z", "orc_kernel_M", "orc_kernel_Q", "orc_kernel_ghost", "orc_kernel_M_literal",
                     "orc_kernel_Q_literal"):
            f = getattr(L, name)
            f.argtypes = [C.c_double] * 3
            f.restype = C.c_double
        L.orc_s_map.argtypes = [C.POINTER(OrcParams), C.c_double]
        L.orc_s_map.restype = C.c_double
        L.orc_coupling_C.argtypes = [C.POINTER(OrcParams)]
        L.orc_coupling_C.restype = C.c_double
        L.orc_ln_dress.argtypes = [C.POINTER(OrcParams), _dp, C.c_double, _dp, _dp]
        L.orc_n_ext.argtypes = [C.POINTER(OrcParams)]
        L.orc_tables.argtypes = [C.POINTER(OrcParams)] + [_dp] * 7
        L.orc_self_energy.argtypes = [C.POINTER(OrcParams), _dp, C.c_double, C.c_int, _dp, _dp, C.c_int, _dp, _dp,
                                      _dp, _dp]
        L.orc_residual_jacobian.argtypes = [C.POINTER(OrcParams), _dp, C.c_double, C.c_double, _dp, _dp]
        L.orc_lu_solve.argtypes = [C.c_int, _dp, _dp, _dp, _dp]
        L.orc_newton_step.argtypes = [C.POINTER(OrcParams), _dp, C.c_double, C.c_double, C.c_double, _dp]

    # -- tables ---------------------------------------------------------------------------------
    def gauss_legendre(self, n):
        t = np.empty(n); w = np.empty(n)
        self.lib.orc_gauss_legendre(n, _ptr(t), _ptr(w))
        return t, w

    def radial_rule_split(self, p, x):
        n = p.n_ir + 2 * p.n_r
        y = np.empty(n); Wy = np.empty(n)
        self.lib.orc_radial_rule_split(C.byref(p), float(x), _ptr(y), _ptr(Wy))
        return y, Wy

    def gl_node(self, n, i):
        t = C.c_double(); w = C.c_double()
        self.lib.orc_gl_node(int(n), int(i), C.byref(t), C.byref(w))
        return t.value, w.value

    def schwinger(self, p, c, n_nodes, p2_min, p2_max, t):
        c = _f64(c); t = _f64(t)
        out = np.empty(len(t))
        self.lib.orc_schwinger(C.byref(p), _ptr(c), int(n_nodes), float(p2_min), float(p2_max), len(t), _ptr(t), _ptr(out))
        return out

    def schwinger_threads(self, p, c, n_nodes, p2_min, p2_max, t, threads=None):
        """orc_schwinger with the O(n_nodes^2) node table computed in ranges on several host threads (ctypes releases the
        GIL) and the sums taken serially afterwards: the same arithmetic, for the paper's 2^17-node rule (fn.13)."""
        import os
        from concurrent.futures import ThreadPoolExecutor
        c = _f64(c); t = _f64(t)
        n_nodes = int(n_nodes)
        threads = threads or min(os.cpu_count() or 1, 64)
        pn = np.empty(n_nodes); fn = np.empty(n_nodes)
        # Newton on the recurrence converges in fewer steps in the middle of the interval: interleave small ranges
        step = max(1, n_nodes // (threads * 16))
        ranges = [(i, min(i + step, n_nodes)) for i in range(0, n_nodes, step)]
        def work(r):
            self.lib.orc_schwinger_terms(C.byref(p), _ptr(c), n_nodes, float(p2_min), float(p2_max), r[0], r[1], _ptr(pn), _ptr(fn))
        with ThreadPoolExecutor(max_workers=threads) as pool:
            list(pool.map(work, ranges))
        out = np.empty(len(t))
        self.lib.orc_schwinger_sum(n_nodes, _ptr(pn), _ptr(fn), len(t), _ptr(t), _ptr(out))
        return out

    def cheb_phi(self, n, s):
        phi = np.empty(n)
        self.lib.orc_cheb_phi(n, float(s), _ptr(phi))
        return phi

    def tables(self, p):
        ne = self.lib.orc_n_ext(C.byref(p))
        nr = p.n_r + p.n_ir
        out = dict(x_ext=np.empty(ne), s_root=np.empty(p.n_cheb), t_r=np.empty(nr), y=np.empty(nr),
                   Wy=np.empty(nr), theta=np.empty(p.n_theta), Omega=np.empty(p.n_theta))
        self.lib.orc_tables(C.byref(p), *[_ptr(out[k]) for k in ("x_ext", "s_root", "t_r", "y", "Wy", "theta", "Omega")])
        return out

    # -- scalar pieces ----------------------------------------------------------------------------
    def z(self, x, y, th): return self.lib.orc_z(x, y, th)
    def kernel_M(self, x, y, th): return self.lib.orc_kernel_M(x, y, th)
    def kernel_Q(self, x, y, th): return self.lib.orc_kernel_Q(x, y, th)
    def kernel_ghost(self, x, y, th): return self.lib.orc_kernel_ghost(x, y, th)
    def kernel_M_literal(self, x, y, z): return self.lib.orc_kernel_M_literal(x, y, z)
    def kernel_Q_literal(self, x, y, z): return self.lib.orc_kernel_Q_literal(x, y, z)
    def s_map(self, p, u): return self.lib.orc_s_map(C.byref(p), float(u))
    def coupling_C(self, p): return self.lib.orc_coupling_C(C.byref(p))

    def ln_dress(self, p, c, u):
        c = _f64(c)
        g = C.c_double(); z = C.c_double()
        self.lib.orc_ln_dress(C.byref(p), _ptr(c), float(u), C.byref(g), C.byref(z))
        return g.value, z.value

    def self_energy(self, p, c, x, y, Wy, theta, Omega, derivs=False):
        c = _f64(c); y = _f64(y); Wy = _f64(Wy); theta = _f64(theta); Omega = _f64(Omega)
        out = np.empty(3)
        d = np.empty((4, p.n_cheb)) if derivs else None
        self.lib.orc_self_energy(C.byref(p), _ptr(c), float(x), len(y), _ptr(y), _ptr(Wy), len(theta), _ptr(theta),
                                 _ptr(Omega), _ptr(out), _ptr(d) if derivs else None)
        return (out, d) if derivs else out

    # -- the path ---------------------------------------------------------------------------------
    def residual_jacobian(self, p, c, gG, gZ, jac=True):
        c = _f64(c)
        n = 2 * p.n_cheb
        F = np.empty(n)
        J = np.empty((n, n)) if jac else None
        self.lib.orc_residual_jacobian(C.byref(p), _ptr(c), float(gG), float(gZ), _ptr(F), _ptr(J) if jac else None)
        return (F, J) if jac else F

    def lu_solve(self, A, b):
        A = _f64(A); b = _f64(b)
        n = len(b)
        x = np.empty(n); stats = np.empty(4)
        rc = self.lib.orc_lu_solve(n, _ptr(A), _ptr(b), _ptr(x), _ptr(stats))
        return x, stats, rc

    def newton_step(self, p, c, gG, gZ, rho=1.0):
        c = _f64(c).copy()
        stats = np.empty(4)
        rc = self.lib.orc_newton_step(C.byref(p), _ptr(c), float(gG), float(gZ), float(rho), _ptr(stats))
        return c, stats, rc

    def newton_solve(self, p, c, gG, gZ, rho=1.0, step_cap=0.0, tol=1e-12, max_iter=50):
        """The Newton-Raphson iteration, eq.(31)-(35) L218-273, with the under-relaxation of L226 ("used to relax the
        system ... After some iteration steps, this parameter can be set back to one"): the paper gives no rule for
        rho_n; reading A26 takes rho_n = min(rho, step_cap / |Delta_n|_inf) (no coefficient moves by more
        than step_cap; step_cap <= 0: rho_n = rho).  Step by step: build F, J -> solve J Delta = F -> c <- c - rho_n
        Delta; stop after the step whose |Delta|_inf < tol.  Returns (c, [(|Delta|inf, |F|inf scaled, min pivot,
        rho_n) per step], status) with status 1 converged, 0 max_iter reached, -1 non-finite Delta (c left as it was).
        Pinned by P9 (tests/test_oracle_path.py): the paper's printed alpha(M_Z^2), alpha(0), kappa."""
        c = _f64(c).copy()
        hist = []
        for _ in range(int(max_iter)):
            F, J = self.residual_jacobian(p, c, gG, gZ)
            d, st, rc = self.lu_solve(J, F)
            if not np.isfinite(st[0]):
                hist.append((st[0], st[1], st[2], 0.0))
                return c, hist, -1
            r = rho
            if step_cap > 0.0 and rho * st[0] > step_cap:
                r = step_cap / st[0]
            c = c - r * d
            hist.append((st[0], st[1], st[2], r))
            if st[0] < tol:
                return c, hist, 1
        return c, hist, 0

"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these tests touches the CUDA path.  Each is chosen so that a plausible mistake in
oracle/dse_oracle.c (dropped term, wrong sign/index/prefactor, transposed operand) fails one of them.
"""
import math
import os

import numpy as np
import pytest

from oracle.oracle import make_params

PI = math.pi
GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")) as fh:
    for line in fh:
        line = line.split("#")[0].split()
        if len(line) == 2:
            GOLD[line[0]] = float(line[1])


def flat_params(n=4, nr=8, nt=8, eps2=1e-4, L2=1e4, **kw):
    """G = Z = 1 everywhere when c = 0: no power-law / log continuation."""
    return make_params(n, nr, nt, eps2, L2, kw.pop("x_G", 1.0), kw.pop("x_Z", 1.0), ir_exp_G=0.0, ir_exp_Z=0.0,
                       uv_omega=0.0, **kw)


# ------------------------------------------------------------------------------------------ P1
@pytest.mark.parametrize("n", [1, 2, 3, 16, 64, 128, 1024])
def test_gauss_legendre_textbook(orc, orc_ld, n):
    t, w = orc.gauss_legendre(n)
    tl, wl = orc_ld.gauss_legendre(n)
    assert np.allclose(t, tl, atol=3e-16, rtol=0) and np.allclose(w, wl, rtol=1e-11, atol=0)
    assert abs(w.sum() - 2.0) < 1e-13
    assert np.all(np.diff(t) > 0) and np.allclose(t, -t[::-1], atol=1e-15)
    tn, wn = np.polynomial.legendre.leggauss(n)
    assert np.allclose(t, tn, atol=2e-15, rtol=0)
    assert np.allclose(w, wn, rtol=5e-9, atol=1e-17)     # numpy's own weights are only ~1e-9 at n=1024
    # exact for monomials up to degree 2n-1
    for d in sorted({0, 1, min(2, 2 * n - 1), min(2 * n - 2, 40), min(2 * n - 1, 41)}):
        exact = 0.0 if d % 2 else 2.0 / (d + 1)
        assert abs(np.sum(w * t ** d) - exact) < 1e-13


# ------------------------------------------------------------------------------------------ P2
def test_chebyshev_basis(orc):
    n = 40
    for ang in np.linspace(0, PI, 23):
        phi = orc.cheb_phi(n, math.cos(ang))
        ref = np.cos(np.arange(n) * ang)
        ref[0] = 0.5                       # b_0/2 convention, eq.(23),(24)
        assert np.allclose(phi, ref, atol=5e-13)
    # discrete orthogonality at the roots s_i = -cos(pi (i+1/2)/N)  (fn.9: collocation at the roots)
    N = 16
    p = make_params(N, 4, 4, 1e-6, 5e4, 1.0, 1.0)
    tab = orc.tables(p)
    T = np.stack([orc.cheb_phi(N, s) for s in tab["s_root"]])
    T[:, 0] *= 2
    G = T.T @ T
    D = np.diag([N] + [N / 2] * (N - 1))
    assert np.allclose(G, D, atol=1e-12)
    assert np.all(np.diff(tab["s_root"]) > 0)           # ascending x (reading A5)
    # interpolation of a known function round-trips: f(s) = exp(s) -> coefficients -> values
    f = np.exp(tab["s_root"])
    coef = (2.0 / N) * (T.T @ f)
    for s in (-1.0, -0.3, 0.77, 1.0):
        assert abs(orc.cheb_phi(N, s) @ coef - math.exp(s)) < 1e-13


def test_tables_maps(orc):
    p = make_params(8, 64, 16, 1e-10, 1e10, 1e2, 1e2)
    tab = orc.tables(p)
    Lg = math.log(p.L2 / p.eps2)
    # eq.(25) (reading A4): both printed forms agree
    for u in (1e-10, 3.3e-4, 1.0, 1e2, 9.9e9):
        s = orc.s_map(p, u)
        s_printed = math.log10(u / math.sqrt(p.L2 * p.eps2)) / math.log10(math.sqrt(p.L2 / p.eps2))
        assert abs(s - s_printed) < 1e-13
    assert np.allclose([orc.s_map(p, x) for x in tab["x_ext"][:8]], tab["s_root"], atol=1e-14)
    assert np.allclose([orc.s_map(p, y) for y in tab["y"]], tab["t_r"], atol=1e-13)
    # int dy f(y) with the log-mapped rule: int_{eps2}^{L2} y^-1 dy = Lg ; int y^-1/2 dy = 2(sqrt L2 - sqrt eps2)
    assert abs(np.sum(tab["Wy"] / tab["y"]) - Lg) < 1e-12 * Lg
    # angular rule: int_0^pi sin^2 = pi/2, int sin^4 = 3 pi/8  (eq.(4),(5))
    assert abs(np.sum(tab["Omega"] * np.sin(tab["theta"]) ** 2) - PI / 2) < 1e-14
    assert abs(np.sum(tab["Omega"] * np.sin(tab["theta"]) ** 4) - 3 * PI / 8) < 1e-14
    assert tab["x_ext"][8] == 1e2 and len(tab["x_ext"]) == 9
    p2 = make_params(8, 64, 16, 1e-10, 1e10, 3.0, 1e2)
    assert list(orc.tables(p2)["x_ext"][8:]) == [1e2, 3.0]   # index N: x_Z, index N+1: x_G
    assert abs(orc.coupling_C(p) - 3 / (2 * PI ** 2)) < 1e-16     # g^2 N_c/(2 pi)^3, alpha=1, N_c=3


# ------------------------------------------------------------------------------------------ P3
def test_stable_kernels_equal_literal(orc_ld, orc):
    rng = np.random.default_rng(7)
    for _ in range(400):
        x = 10 ** rng.uniform(-3, 3)
        y = x * 10 ** rng.uniform(-3, 3)
        th = rng.uniform(0.05, PI - 0.05)
        z_lit = x + y - 2 * math.sqrt(x * y) * math.cos(th)
        z = orc.z(x, y, th)
        assert abs(z - z_lit) <= 1e-12 * (x + y)
        # literal forms in long double (they cancel by ~ max(y/x, x/y)) vs stable forms in double
        Ml = orc_ld.kernel_M_literal(x, y, orc_ld.z(x, y, th))
        Ql = orc_ld.kernel_Q_literal(x, y, orc_ld.z(x, y, th))
        scale = max(x / y, y / x) ** 2
        assert abs(orc.kernel_M(x, y, th) - Ml) <= 1e-12 * scale * max(1, abs(Ml))
        assert abs(orc.kernel_Q(x, y, th) - Ql) <= 1e-11 * scale * max(1, abs(Ql))
    # near-degenerate ratios: tight check
    for (x, y, th) in [(1.0, 1.3, 0.7), (2.0, 0.5, 2.1), (1.0, 1.0, 1.0), (5.0, 4.0, 0.3)]:
        zl = orc_ld.z(x, y, th)
        assert abs(orc.kernel_M(x, y, th) - orc_ld.kernel_M_literal(x, y, zl)) < 1e-12
        assert abs(orc.kernel_Q(x, y, th) - orc_ld.kernel_Q_literal(x, y, zl)) < 5e-12
        assert abs(orc.kernel_Q(x, y, th) - orc.kernel_Q(y, x, th)) < 1e-13     # Q symmetric in x <-> y
        assert abs(orc.kernel_M(x, y, th) - y * math.sin(th) ** 2 / zl) < 1e-13
        assert abs(orc.kernel_ghost(x, y, th) - math.sin(th) ** 4 / zl ** 2) < 1e-12 / zl ** 2
    assert abs(orc.kernel_Q(3.0, 7.0, 0.0) - 15 / 4) < 1e-14
    # z stays accurate where the literal form has lost everything
    assert abs(orc.z(1e-10, 1e10, 1.0) / 1e10 - (1 + 1e-20 - 2e-10 * math.cos(1.0))) < 1e-15
    assert orc.z(1.0, 1.0, 1e-9) == pytest.approx(1e-18, rel=1e-12)


# ------------------------------------------------------------------------------------------ P4 / P7
def _ang(orc, n=600):
    t, w = orc.gauss_legendre(n)
    return (t + 1) * PI / 2, w * PI / 2


@pytest.mark.parametrize("t", [0.01, 0.5, 0.9])
def test_closed_form_angular_integrals(orc, t):
    th, Om = _ang(orc, 900)
    s2 = np.sin(th) ** 2
    for (x, y) in [(1.0, 1.0 / t), (1.0, t), (3.7, 3.7 / t)]:
        big, small = max(x, y), min(x, y)
        tt = small / big
        z = np.array([orc.z(x, y, a) for a in th])
        M = np.array([orc.kernel_M(x, y, a) for a in th])
        Q = np.array([orc.kernel_Q(x, y, a) for a in th])
        gh = np.array([orc.kernel_ghost(x, y, a) for a in th])
        tol = 1e-9
        assert abs(np.sum(Om * s2 / z) - PI / (2 * big)) < tol / big
        assert abs(np.sum(Om * s2 / z ** 2) - PI / (2 * big * (big - small))) < tol / (big * (big - small)) * 10
        assert abs(np.sum(Om * gh) - 3 * PI / (8 * big ** 2)) < tol / big ** 2
        assert abs(np.sum(Om * s2 * z) - PI * (x + y) / 2) < tol * (x + y)
        assert abs(np.sum(Om * s2 * z ** 2) - PI * (x * x + 3 * x * y + y * y) / 2) < tol * (x + y) ** 2
        exact_M = PI * (3 - tt) / 8 if y > x else PI * tt * (3 - tt) / 8
        assert abs(np.sum(Om * s2 * M) - exact_M) < tol
        assert abs(np.sum(Om * s2 * Q) - PI * (7 * tt * tt - 50 * tt - 6) / 16) < 10 * tol


def test_no_quadratic_divergence_P7(orc):
    """fn.5 L127: the +15/4 removes the O(1) term of int sin^2 (Q+M) for y >> x."""
    th, Om = _ang(orc, 400)
    s2 = np.sin(th) ** 2
    for ratio in (1e4, 1e8, 1e14):
        x, y = 2.0, 2.0 * ratio
        S = sum(Om[k] * s2[k] * (orc.kernel_Q(x, y, th[k]) + orc.kernel_M(x, y, th[k])) for k in range(len(th)))
        t = 1 / ratio
        assert abs(S - PI * (7 * t * t - 52 * t) / 16) < 1e-12
    # the individual limits: Q -> 6 cos^2 - 9/4 (int sin^2 = -3 pi/8), M -> sin^2 (int = +3 pi/8)
    assert abs(orc.kernel_Q(1.0, 1e30, 0.9) - (6 * math.cos(0.9) ** 2 - 2.25)) < 1e-12
    assert abs(orc.kernel_M(1.0, 1e30, 0.9) - math.sin(0.9) ** 2) < 1e-12


# ------------------------------------------------------------------------------------------ P5 / P6
def _split_rule(orc, eps2, L2, x, n):
    t, w = orc.gauss_legendre(n)
    ys, Ws = [], []
    for lo, hi in ((eps2, x), (x, L2)):
        if hi <= lo:
            continue
        L = math.log(hi / lo)
        y = lo * np.exp((t + 1) * L / 2)
        ys.append(y)
        Ws.append(w * L / 2 * y)
    return np.concatenate(ys), np.concatenate(Ws)


@pytest.mark.parametrize("x", [0.01, 1.0, 37.0])
def test_tree_level_self_energies_closed_form(orc, x):
    eps2, L2 = 1e-4, 1e4
    p = flat_params(eps2=eps2, L2=L2)
    C = orc.coupling_C(p)
    th, Om = _ang(orc, 400)
    y, Wy = _split_rule(orc, eps2, L2, x, 200)
    out = orc.self_energy(p, np.zeros(8), x, y, Wy, th, Om)
    PiG0 = -C * (3 * PI / 8) * ((x * x - eps2 ** 2) / (2 * x * x) + math.log(L2 / x))
    PiZ0 = (C * PI / (48 * x)) * ((5 / 3) * (x ** 3 - eps2 ** 3) / x ** 2 - 22 * (x * x - eps2 ** 2) / x
                                 - 6 * (x - eps2) + 7 * x * x * (1 / x - 1 / L2) - 52 * x * math.log(L2 / x))
    assert abs(out[0] - PiG0) < 1e-9 * abs(PiG0)
    assert abs(out[1] + out[2] - PiZ0) < 1e-9 * abs(PiZ0)
    # ghost loop alone: (C/3x) [ int_{y<x} pi t(3-t)/8 + int_{y>x} pi (3-t)/8 ]
    M0 = (C / (3 * x)) * (PI / 8) * ((3 * (x * x - eps2 ** 2) / (2 * x) - (x ** 3 - eps2 ** 3) / (3 * x * x))
                                    + 3 * (L2 - x) - x * math.log(L2 / x))
    assert abs(out[2] - M0) < 1e-9 * abs(M0)


def test_one_loop_anomalous_dimensions_P6(orc):
    """d Pi^0 / d ln(L2) at fixed x -> delta*omega (ghost) and gamma*omega (gluon), L58, L131."""
    delta, gamma = GOLD["delta"], GOLD["gamma"]
    assert abs(gamma + 2 * delta + 1) < 1e-15
    p = flat_params()
    omega = 11 * 3 * 1.0 / (12 * PI)
    assert abs(omega / 3 - GOLD["omega_over_alphaNc"]) < 1e-4
    th, Om = _ang(orc, 300)
    x = 1.0
    vals = []
    for L2 in (1e6, 1e8):
        pp = flat_params(eps2=1e-4, L2=L2)
        y, Wy = _split_rule(orc, 1e-4, L2, x, 200)
        vals.append(orc.self_energy(pp, np.zeros(8), x, y, Wy, th, Om))
    dln = math.log(1e8 / 1e6)
    slope_G = (vals[1][0] - vals[0][0]) / dln
    slope_Z = (vals[1][1] + vals[1][2] - vals[0][1] - vals[0][2]) / dln
    assert abs(slope_G - delta * omega) < 1e-9
    assert abs(slope_Z - gamma * omega) < 2e-6       # + O(x/L2) from the 7x^2/L2 term


# ------------------------------------------------------------------------------------------ P8
def test_infrared_exponent_and_fixed_point_P8(orc):
    """Power-law dressings G = B x^-kappa, Z = A x^(2 kappa) on (0, inf), x_G = 0:
    ghost eq.  => (C A B^2)^-1 = -I_G(kappa),  gluon eq. (ghost loop) => (C A B^2)^-1 = I_Z(kappa)/3.
    Both hold at the paper's kappa = 0.595353 and give alpha(0) N_c = 2 pi^2 / value = 8.915 (L151)."""
    th, Om = _ang(orc, 160)
    t, w = orc.gauss_legendre(48)

    def radial_panels(edges):
        ys, Ws = [], []
        for lo, hi in zip(edges[:-1], edges[1:]):
            L = math.log(hi / lo)
            y = lo * np.exp((t + 1) * L / 2)
            ys.append(y); Ws.append(w * L / 2 * y)
        return np.concatenate(ys), np.concatenate(Ws)

    Y = 1e12
    edges = [1e-14, 1e-8, 1e-4, 1e-2, 0.3, 0.7, 0.9, 1.0, 1.1, 1.5, 3.0, 1e2, 1e4, 1e8, Y]
    y, Wy = radial_panels(edges)
    s4 = np.sin(th) ** 4

    def I_G(kappa):
        p_ = 2 * kappa - 2
        tot = 0.0
        for yq, Wq in zip(y, Wy):
            acc = 0.0
            for k in range(len(th)):
                z = orc.z(1.0, yq, th[k])
                gh = orc.kernel_ghost(1.0, yq, th[k])          # sin^4 / z^2
                lr = math.log1p((1.0 - 2.0 * math.sqrt(yq) * math.cos(th[k])) / yq)   # ln(z/y)
                acc += Om[k] * gh * z * z * yq ** p_ * math.expm1(p_ * lr)
            tot += Wq * yq ** (1 - kappa) * acc
        tot += p_ * PI * (2 + p_) / 8 * Y ** (kappa - 1) / (1 - kappa)          # analytic tail beyond Y
        tot += -(3 * PI / 8) * edges[0] ** kappa / kappa                          # int_0^{y0}: -y^(kappa-1) 3pi/8
        return tot

    def I_Z(kappa):
        tot = 0.0
        for yq, Wq in zip(y, Wy):
            acc = 0.0
            for k in range(len(th)):
                z = orc.z(1.0, yq, th[k])
                acc += Om[k] * math.sin(th[k]) ** 2 * orc.kernel_M(1.0, yq, th[k]) * z ** (-kappa)
            tot += Wq * yq ** (-kappa) * acc
        tot += (3 * PI / 8) * Y ** (1 - 2 * kappa) / (2 * kappa - 1)             # tail: y^(-2 kappa) 3pi/8
        return tot

    k0 = GOLD["kappa"]
    g, zz = -I_G(k0), I_Z(k0) / 3
    assert abs(g - zz) < 2e-5 * abs(g)
    assert abs(2 * PI ** 2 / g - GOLD["alpha0_times_Nc"]) < 5e-4      # 8.915 printed to 4 digits
    assert abs(2 * PI ** 2 / zz - GOLD["alpha0_times_Nc"]) < 5e-4
    assert abs(2 * PI ** 2 / g / 3 - GOLD["alpha0_Nc3"]) < 5e-4
    # and kappa is where the two cross: the mismatch changes sign around it
    f_lo = -I_G(k0 - 0.0001) - I_Z(k0 - 0.0001) / 3
    f_hi = -I_G(k0 + 0.0001) - I_Z(k0 + 0.0001) / 3
    assert f_lo * f_hi < 0
    k_star = (k0 - 0.0001) + 0.0002 * f_lo / (f_lo - f_hi)
    assert abs(k_star - k0) < 5e-6                          # the paper prints six digits
    assert abs(k_star - (93 - math.sqrt(1201)) / 98) < 5e-6


# ------------------------------------------------------------------------------------------ NEXT f3
def test_tanh_sinh_angular_rule(orc):
    """PAPER.md L62-66, eq.(5): int_0^pi dtheta sin^2 f -> int_{-1}^{1} dxi sqrt(1-xi^2) f with a tanh-sinh rule
    (reading A9b).  Checked against closed forms: the measure itself, the ghost measure, and the closed-form
    angular integrals of pin P4 (kernels with endpoint-singular behaviour at t -> 1)."""
    p = make_params(4, 4, 64, 1e-4, 1e4, 1.0, 1.0, angular_rule=1)
    tab = orc.tables(p)
    th, Om = tab["theta"], tab["Omega"]
    assert np.all(np.diff(th) > 0) and th[0] > 0 and th[-1] < PI
    xi = np.cos(th)
    # nodes are xi = tanh((pi/2) sinh t) on an equidistant t grid in [-3, 3]
    t_grid = np.arcsinh(np.arctanh(np.clip(xi[8:-8], -1, 1)) * 2 / PI)
    assert np.allclose(np.diff(t_grid), -6.0 / 63, atol=1e-9)
    s2 = np.sin(th) ** 2
    assert abs(np.sum(Om * s2) - PI / 2) < 1e-13            # int sqrt(1-xi^2) dxi
    assert abs(np.sum(Om * s2 ** 2) - 3 * PI / 8) < 1e-13   # int (1-xi^2)^(3/2) dxi  (eq.(8), reading A1)
    for (x, y) in [(1.0, 2.0), (1.0, 1.0 / 0.9), (3.7, 0.037)]:
        big, small = max(x, y), min(x, y)
        tt = small / big
        z = np.array([orc.z(x, y, a) for a in th])
        M = np.array([orc.kernel_M(x, y, a) for a in th])
        Q = np.array([orc.kernel_Q(x, y, a) for a in th])
        assert abs(np.sum(Om * s2 / z) - PI / (2 * big)) < 1e-10 / big
        exact_M = PI * (3 - tt) / 8 if y > x else PI * tt * (3 - tt) / 8
        assert abs(np.sum(Om * s2 * M) - exact_M) < 1e-10
        assert abs(np.sum(Om * s2 * Q) - PI * (7 * tt * tt - 50 * tt - 6) / 16) < 1e-9
    # the two rules give the same self-energies up to their (small) quadrature errors
    c = np.array([0.2, -0.1, 0.05, 0.0, -0.3, 0.1, 0.0, 0.02])
    pg = make_params(4, 4, 64, 1e-4, 1e4, 1.0, 1.0, angular_rule=0)
    tg = orc.tables(pg)
    a = orc.self_energy(p, c, 0.7, tab["y"], tab["Wy"], th, Om)
    b = orc.self_energy(pg, c, 0.7, tg["y"], tg["Wy"], tg["theta"], tg["Omega"])
    assert np.allclose(a, b, rtol=1e-6)

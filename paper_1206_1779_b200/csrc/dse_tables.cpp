// dse_tables.cpp -- host-side builder of the quadrature-grid and Chebyshev tables (step H0).
//
// Gauss-Legendre rule for the radial integral with a non-linear node map -- here a
// single rule in s = 2 ln(y/eps2)/Lg - 1 on [eps2, L2] (BASELINE configs; reading A8);
// angular rule: Gauss-Legendre in theta on [0, pi] (reading A9); collocation at the mapped roots of
// T_N (fn.9 L224); map eq.(25) L185.  Everything is evaluated in long double and rounded once.
#include <cmath>

#include "dse_internal.h"

namespace dse {
namespace {

using ld = long double;
const ld PI_L = 3.141592653589793238462643383279502884L;

// Legendre P_n(x) and P_{n-1}(x) by the Bonnet recurrence.
inline void legendre_pair(int n, ld x, ld &pn, ld &pnm1)
{
    ld a = 1.0L, b = x;   // P_0, P_1
    if (n == 0) { pn = a; pnm1 = 0; return; }
    for (int m = 1; m < n; ++m) {
        ld c = ((2 * m + 1) * x * b - m * a) / (m + 1);
        a = b;
        b = c;
    }
    pn = b;
    pnm1 = a;
}

// nodes ascending in (-1,1); only the non-negative half is iterated, the rest mirrored.
void gauss_legendre(int n, std::vector<ld> &node, std::vector<ld> &weight)
{
    node.assign(n, 0);
    weight.assign(n, 0);
    const int half = (n + 1) / 2;
    for (int m = 0; m < half; ++m) {
        // m-th largest root; Tricomi-type starting value
        ld th = PI_L * (4 * m + 3) / (4 * n + 2);
        ld x = (1 - (ld)(n - 1) / (8.0L * n * n * n)) * cosl(th);
        ld pn, pm, dpn = 1;
        for (int it = 0; it < 60; ++it) {
            legendre_pair(n, x, pn, pm);
            dpn = n * (pm - x * pn) / (1 - x * x);
            ld step = pn / dpn;
            x -= step;
            if (fabsl(step) < 2e-19L) break;
        }
        legendre_pair(n, x, pn, pm);
        dpn = n * (pm - x * pn) / (1 - x * x);
        ld w = 2 / ((1 - x * x) * dpn * dpn);
        node[n - 1 - m] = x;
        weight[n - 1 - m] = w;
        node[m] = -x;
        weight[m] = w;
    }
    if (n % 2 == 1) node[n / 2] = 0;
}

inline void phi_row(int N, int Npad, ld s, double *out)
{
    ld tm = 1, t = s;
    for (int j = 0; j < Npad; ++j) out[j] = 0.0;
    out[0] = 0.5;   // phi_0 = 1/2: the c_0/2 convention of eq.(23),(24)
    if (N > 1) out[1] = (double)s;
    for (int j = 2; j < N; ++j) {
        ld tn = 2 * s * t - tm;
        tm = t;
        t = tn;
        out[j] = (double)tn;
    }
}

}  // namespace

// user != nullptr (DSE_FLAG_USER_TABLES): x_ext, y, Wy, theta, Omega are taken from the caller as they are; s(y_q), the
// phi tables, the square roots and the continuation add-ons are derived from those values exactly as from the library's own.
void build_tables(const dse_params &p, const dse_tables *user, HostTables &T)
{
    const bool split = (p.flags & DSE_FLAG_RADIAL_SPLIT) != 0;
    const int N = p.n_cheb, Nir = p.n_r_ir, Nmain = p.n_r, Nr = (split ? 2 : 1) * Nmain + Nir, Nt = p.n_theta;
    T.N = N;
    T.Npad = ((N + CJ - 1) / CJ) * CJ;
    T.Nr = Nr;
    T.Nt = Nt;
    int g = 32;
    if (Nt < 32) { g = 1; while (g < Nt) g <<= 1; }
    T.Ntpad = ((Nt + g - 1) / g) * g;
    const bool same = (p.x_G == p.x_Z);
    T.Next = N + (same ? 1 : 2);
    T.iZ = N;
    T.iG = same ? N : N + 1;
    const ld Lg = logl((ld)p.L2 / (ld)p.eps2);
    T.Lg = (double)Lg;
    const ld C = 4 * PI_L * (ld)p.alpha_mu * (ld)p.n_colors / (8 * PI_L * PI_L * PI_L);   // g^2 N_c/(2 pi)^3
    T.C = (double)C;

    std::vector<ld> t, w;
    // external points first (the split radial rule depends on them): Chebyshev roots s_i = -cos(pi (i+1/2)/N),
    // ascending, then x_Z, then x_G
    T.x_ext.resize(T.Next); T.sx_ext.resize(T.Next); T.c3x_ext.resize(T.Next);
    T.phi_x.assign((size_t)N * T.Npad, 0.0);
    for (int i = 0; i < N; ++i) {
        ld s = -cosl(PI_L * (i + 0.5L) / N);
        T.x_ext[i] = (double)((ld)p.eps2 * expl((s + 1) * Lg / 2));
        phi_row(N, T.Npad, s, &T.phi_x[(size_t)i * T.Npad]);
    }
    T.x_ext[T.iZ] = p.x_Z;
    if (!same) T.x_ext[T.iG] = p.x_G;
    if (user)
        for (int e = 0; e < T.Next; ++e) T.x_ext[e] = user->x_ext[e];
    for (int e = 0; e < T.Next; ++e) {
        T.sx_ext[e] = (double)sqrtl((ld)T.x_ext[e]);
        // at x = 0 (x_G = 0, L135) only the ghost equation is evaluated: the gluon prefactor C/(3x) is dropped
        T.c3x_ext[e] = T.x_ext[e] > 0.0 ? (double)(C / (3 * (ld)T.x_ext[e])) : 0.0;
    }

    // radial rule(s): [infrared piece | main], shared by all external points, or -- DSE_FLAG_RADIAL_SPLIT, eq.(26) --
    // [infrared piece | (eps2, x_e) | (x_e, L2)] per external point with n_r nodes in each interval (L364)
    const int nrules = split ? T.Next : 1;
    T.rstride = split ? Nr : 0;
    const size_t tot = (size_t)nrules * Nr;
    T.y.resize(tot); T.sy.resize(tot); T.Wy.resize(tot); T.t_r.resize(tot);
    T.EGy.assign(tot, 0.0); T.EZy.assign(tot, 0.0);
    T.phi_y.assign(tot * T.Npad, 0.0);
    std::vector<ld> tir, wir, tm, wm;
    if (Nir > 0) gauss_legendre(Nir, tir, wir);
    gauss_legendre(Nmain, tm, wm);
    for (int rule = 0; rule < nrules; ++rule) {
        const size_t o = (size_t)rule * Nr;
        // infrared piece int_0^{eps2} dy: GL in v, y = eps2 ((1+v)/2)^4, dy = 2 eps2 ((1+v)/2)^3 dv; the dressings there
        // are the power laws eq.(16),(17): ln G(y) = series(s = -1) + p_G ln(y/eps2)
        for (int q = 0; q < Nir; ++q) {
            const ld hq = (tir[q] + 1) / 2;
            T.y[o + q] = (double)((ld)p.eps2 * hq * hq * hq * hq);
            T.Wy[o + q] = (double)(wir[q] * 2 * (ld)p.eps2 * hq * hq * hq);
            if (user) { T.y[o + q] = user->y[o + q]; T.Wy[o + q] = user->Wy[o + q]; }
            T.t_r[o + q] = -1.0;
            const ld ell = logl((ld)T.y[o + q] / (ld)p.eps2);
            T.EGy[o + q] = (double)((ld)p.ir_exp_G * ell);
            T.EZy[o + q] = (double)((ld)p.ir_exp_Z * ell);
            phi_row(N, T.Npad, -1.0L, &T.phi_y[(o + q) * T.Npad]);
        }
        // main rule(s) in ln y: y = lo exp((v+1) L/2), dy = (L/2) y dv; s(y) by eq.(25)
        ld xm = split ? (ld)T.x_ext[rule] : (ld)p.L2;
        if (xm < (ld)p.eps2) xm = p.eps2;
        if (xm > (ld)p.L2) xm = p.L2;
        for (int part = 0; part < (split ? 2 : 1); ++part) {
            const ld lo = part == 0 ? (ld)p.eps2 : xm, hi = (split && part == 0) ? xm : (ld)p.L2;
            const ld L = logl(hi / lo);
            for (int q = 0; q < Nmain; ++q) {
                const size_t i = o + Nir + (size_t)part * Nmain + q;
                ld yy = lo * expl((tm[q] + 1) * L / 2);
                T.y[i] = (double)yy;
                T.Wy[i] = (double)(wm[q] * (L / 2) * yy);
                if (user) { T.y[i] = user->y[i]; T.Wy[i] = user->Wy[i]; yy = (ld)T.y[i]; }
                ld sy = 2 * logl(yy / (ld)p.eps2) / Lg - 1;
                if (!split && !user) sy = tm[q];                // the shared rule is laid out in s itself
                if (sy < -1) sy = -1;
                if (sy > 1) sy = 1;
                T.t_r[i] = (double)sy;
                phi_row(N, T.Npad, sy, &T.phi_y[i * T.Npad]);
            }
        }
        for (int q = 0; q < Nr; ++q) T.sy[o + q] = (double)sqrtl((ld)T.y[o + q]);    // sqrt of the rounded table value
    }
    // angular rule: Gauss-Legendre in theta, or tanh-sinh in xi = cos(theta) (eq.(5))
    T.theta.resize(Nt); T.Omega.resize(Nt);
    T.ang.assign((size_t)T.Ntpad * 6, 0.0);
    if (p.flags & DSE_FLAG_ANGULAR_TANH_SINH) {
        // int dxi sqrt(1-xi^2) f:  t_k equidistant in [-3,3], u = (pi/2) sinh t, xi = tanh u, 1-xi^2 = 1/cosh^2 u,
        // w = h (pi/2) cosh t / cosh^2 u, in the theta form: theta = 2 atan(e^-u), Omega = w / sin(theta) = w cosh u, so
        // that "Omega sin^2" and "Omega sin^4" are w sqrt(1-xi^2) and w (1-xi^2)^(3/2).
        const ld tmax = 3.0L, h = Nt > 1 ? 2 * tmax / (Nt - 1) : 0.0L;
        for (int k = 0; k < Nt; ++k) {
            const ld tt = tmax - h * k;                       // descending t: ascending theta
            const ld u = PI_L / 2 * sinhl(tt), ch = coshl(u);
            const ld wk = h * (PI_L / 2) * coshl(tt) / (ch * ch);
            T.theta[k] = (double)(2 * atanl(expl(-u)));
            T.Omega[k] = (double)(wk * ch);
            if (user) { T.theta[k] = user->theta[k]; T.Omega[k] = user->Omega[k]; }
            // the rule IS the pair (theta_k, Omega_k) of doubles that dse_get_tables returns: like the Gauss-Legendre
            // branch, everything the kernels use is derived from those rounded values (next to theta = pi, sin(theta)
            // inherits the rounding of theta -- nodes of relative weight < 1e-11; reading A25)
            const ld thd = (ld)T.theta[k], Om = (ld)T.Omega[k];
            const ld sh = sinl(thd / 2), c = cosl(thd), sn = sinl(thd);
            double *a = &T.ang[(size_t)k * 6];
            a[0] = (double)(sh * sh);
            a[1] = (double)(6 * c);
            a[2] = (double)(2 + c * c);
            a[3] = (double)(-2 * sn * sn);
            a[4] = (double)(Om * sn * sn);
            a[5] = (double)(Om * sn * sn * sn * sn);
        }
        for (int k = Nt; k < T.Ntpad; ++k) {                  // padded lanes: a valid angle with zero weight
            double *a = &T.ang[(size_t)k * 6];
            for (int m = 0; m < 4; ++m) a[m] = T.ang[m];
        }
    } else {
    gauss_legendre(Nt, t, w);
    for (int k = 0; k < T.Ntpad; ++k) {
        const int kk = k < Nt ? k : 0;                 // padded lanes: a valid angle with zero weight
        ld th = (t[kk] + 1) * PI_L / 2;
        ld Om = (k < Nt) ? w[kk] * PI_L / 2 : 0.0L;
        if (user) { th = user->theta[kk]; Om = (k < Nt) ? (ld)user->Omega[kk] : 0.0L; }
        if (k < Nt) { T.theta[k] = (double)th; T.Omega[k] = (double)Om; }
        // the kernels take theta as the rounded double (same input as any other consumer of the table)
        ld thd = (ld)(double)th;
        ld sh = sinl(thd / 2), c = cosl(thd), s = sinl(thd);
        double *a = &T.ang[(size_t)k * 6];
        a[0] = (double)(sh * sh);
        a[1] = (double)(6 * c);
        a[2] = (double)(2 + c * c);
        a[3] = (double)(-2 * s * s);
        a[4] = (double)((ld)(double)Om * s * s);
        a[5] = (double)((ld)(double)Om * s * s * s * s);
    }
    }
}

}  // namespace dse

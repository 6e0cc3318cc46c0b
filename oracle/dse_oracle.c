/*
 * dse_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, serial, obviously-correct CPU oracle for the residual vector and the analytic
 * Newton (Jacobian) matrix of the Chebyshev-collocated Landau-gauge ghost/gluon
 * Dyson-Schwinger equations of Hopfer/Alkofer/Haase (arXiv:1206.1779), written from
 * /root/reference/PAPER.md with the readings listed in DESIGN.md ("Readings of the paper").
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call this file.  It shares no code, header, table or constant with the
 * CUDA path under paper_1206_1779_b200/csrc/ and includes nothing from include/.
 *
 * Precision: `real` is double (default) or long double (-DORACLE_LONG_DOUBLE); the C interface
 * is always in double.  No blocking, fusion or reordering: loops run i (external point),
 * q (radial node), k (angular node), j (Chebyshev index), in that order.
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"):
 *   orc_gauss_legendre   P1  (sum w = 2, exactness to degree 2n-1, numpy leggauss)
 *   orc_cheb_phi         P2  (T_j(cos t) = cos(j t), discrete orthogonality at the roots)
 *   orc_z, orc_kernel_*  P3  (stable forms == literal eq.(10),(11)), P4 (closed-form angular
 *                            integrals), P7 (no O(1) term for y >> x)
 *   orc_self_energy      P5  (closed-form Pi_G^0, Pi_Z^0 for G=Z=1), P6 (one-loop delta*omega,
 *                            gamma*omega), P8 (kappa = 0.595353, alpha(0) N_c = 8.915 printed in
 *                            the paper), P12 (invariances)
 *   orc_ln_dress         continuity at eps2 and L2, slopes p_G, p_Z, delta*omega
 *   orc_residual_jacobian P11 (J vs central finite differences of F, eq.(38)), P12 (j=0 column
 *                            identities, momentum rescaling), brute force on N=N_r=N_theta=2
 *   orc_lu_solve, orc_newton_step  numpy.linalg.solve on scaled systems; P10 quadratic
 *                            convergence
 * "Parity unpinned": the *values* of F and J at the random-coefficient configs have no external
 * reference; they are fixed only through the pins above.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stdint.h>

#ifdef ORACLE_LONG_DOUBLE
typedef long double real;
#define R_EXP expl
#define R_LOG logl
#define R_SQRT sqrtl
#define R_SIN sinl
#define R_COS cosl
#define R_ATAN atanl
#define R_FABS fabsl
#define R_PI 3.14159265358979323846264338327950288L
#define R_TINY 1e-19L
#else
typedef double real;
#define R_EXP exp
#define R_LOG log
#define R_SQRT sqrt
#define R_SIN sin
#define R_COS cos
#define R_ATAN atan
#define R_FABS fabs
#define R_PI 3.14159265358979323846264338327950288
#define R_TINY 1e-16
#endif

/* Parameters of one discretised system.  Own definition; deliberately NOT include/dse.h. */
typedef struct orc_params {
    int32_t n_cheb;    /* N: Chebyshev polynomials per dressing function, eq.(23),(24) L179-181 */
    int32_t n_r;       /* radial Gauss-Legendre nodes in ln y on [eps2, L2] (L62; reading A8)   */
    int32_t n_theta;   /* angular Gauss-Legendre nodes in theta on [0, pi] (reading A9)         */
    int32_t angular_rule; /* 0: Gauss-Legendre in theta (BASELINE configs, reading A9);
                             1: tanh-sinh in xi = cos(theta) (eq.(5)), reading A9b      */
    double eps2, L2;   /* IR matching point / UV cutoff (L188)                                  */
    double alpha_mu;   /* alpha(mu^2) = g^2 / 4 pi (L131, L135)                                 */
    double n_colors;   /* N_c                                                                   */
    double x_G, x_Z;   /* MOM subtraction points, eq.(14),(15) L107-110                         */
    double delta;      /* ghost anomalous dimension, -9/44 (L58); gamma = -1 - 2 delta (L131)   */
    double ir_exp_G;   /* exponent of G below eps2, eq.(17): -kappa                             */
    double ir_exp_Z;   /* exponent of Z below eps2, eq.(16): 2 kappa                            */
    double uv_omega;   /* omega of eq.(18),(19) L121-131; 0 => constant continuation above L2   */
    int32_t n_ir;      /* NEXT f2: nodes of the infrared piece int_0^{eps2} dy of eq.(26); 0 = none */
    int32_t radial_split; /* NEXT f1: 1 = the paper's split int_{eps2}^{x} + int_{x}^{L2} (eq.(26)) with n_r
                             nodes in EACH interval (L364), so the radial rule depends on the external point */
} orc_params;

/* ------------------------------------------------------------------------------------------ */
/* P1. Gauss-Legendre nodes t[0..n) ascending in (-1,1) and weights w, by Newton iteration on   */
/* the Legendre three-term recurrence (textbook; "standard Gauss-Legendre").       */
static void gl_node(int n, int i, real *xo, real *wo)
{
    /* Chebyshev-like initial guess, ascending order */
    real x = -R_COS(R_PI * ((real)i + (real)0.75) / ((real)n + (real)0.5));
    real dp = 1;
    for (int it = 0; it < 100; ++it) {
        real p0 = 1, p1 = x;
        for (int m = 2; m <= n; ++m) {
            real p2 = (((real)(2 * m - 1)) * x * p1 - ((real)(m - 1)) * p0) / (real)m;
            p0 = p1; p1 = p2;
        }
        if (n == 1) { p0 = 1; p1 = x; }
        dp = (real)n * (x * p1 - p0) / (x * x - 1);     /* P_n'(x) */
        real dx = p1 / dp;
        x -= dx;
        if (R_FABS(dx) <= R_TINY) break;
    }
    /* final derivative at the converged node */
    {
        real p0 = 1, p1 = x;
        for (int m = 2; m <= n; ++m) {
            real p2 = (((real)(2 * m - 1)) * x * p1 - ((real)(m - 1)) * p0) / (real)m;
            p0 = p1; p1 = p2;
        }
        if (n == 1) { p0 = 1; p1 = x; }
        dp = (real)n * (x * p1 - p0) / (x * x - 1);
    }
    *xo = x;
    *wo = 2 / ((1 - x * x) * dp * dp);
}
void orc_gauss_legendre(int n, double *t, double *w)
{
    for (int i = 0; i < n; ++i) {
        real x, ww;
        gl_node(n, i, &x, &ww);
        t[i] = (double)x;
        w[i] = (double)ww;
    }
}
/* one node of the n-point rule (for sampled checks of very large rules, e.g. n = 2^17 of PAPER.md fn.13) */
void orc_gl_node(int n, int i, double *t, double *w)
{
    real x, ww;
    gl_node(n, i, &x, &ww);
    *t = (double)x; *w = (double)ww;
}

/* P2. phi_0 = 1/2, phi_j = T_j(s) for j >= 1 (the b_0/2 convention of eq.(23),(24) L179-181),  */
/* T_j by the three-term recurrence T_{j+1} = 2 s T_j - T_{j-1} (reading A19).                  */
static void phi_real(int n, real s, real *phi)
{
    real tm = 1, t = s;
    if (n > 0) phi[0] = (real)0.5;
    if (n > 1) phi[1] = s;
    for (int j = 2; j < n; ++j) {
        real tn = 2 * s * t - tm;
        tm = t; t = tn;
        phi[j] = tn;
    }
}
void orc_cheb_phi(int n, double s, double *phi)
{
    real *p = (real *)malloc(sizeof(real) * (size_t)(n > 0 ? n : 1));
    phi_real(n, (real)s, p);
    for (int j = 0; j < n; ++j) phi[j] = (double)p[j];
    free(p);
}

/* ------------------------------------------------------------------------------------------ */
/* O3. z = k^2 = x + y - 2 sqrt(xy) cos(theta)  (L62, L192) in the cancellation-free form       */
/*     z = (x-y)^2 / (sqrt x + sqrt y)^2 + 4 sqrt(xy) sin^2(theta/2)      (reading A15).        */
static real z_real(real x, real y, real theta)
{
    real sx = R_SQRT(x), sy = R_SQRT(y);
    real d = (x - y) / (sx + sy);
    real sh = R_SIN(theta / 2);
    return d * d + 4 * sx * sy * sh * sh;
}
double orc_z(double x, double y, double theta) { return (double)z_real(x, y, theta); }

/* eq.(10) L88 as printed (cancels catastrophically for y/x far from 1; test use only).        */
double orc_kernel_M_literal(double xd, double yd, double zd)
{
    real x = xd, y = yd, z = zd;
    return (double)((1 / z) * (-x / 4 + y / 2 - y * y / (4 * x)) + (real)0.5 + y / (2 * x) - z / (4 * x));
}
/* eq.(11) L90-94 as printed, including the +15/4 of fn.5 L127 (test use only).                */
double orc_kernel_Q_literal(double xd, double yd, double zd)
{
    real x = xd, y = yd, z = zd;
    real a = (1 / (z * z)) * (x * x * x / (8 * y) + x * x - (real)9 / 4 * x * y + y * y + y * y * y / (8 * x));
    real b = (1 / z) * (x * x / y - 4 * (x + y) + y * y / x);
    real c = -((real)9 / 4 * x / y + 4 + (real)9 / 4 * y / x);
    real d = z * (1 / x + 1 / y) + z * z / (8 * x * y) + (real)15 / 4;
    return (double)(a + b + c + d);
}
/* Stable forms (exact algebraic identities of eq.(10),(11); reading A15):            */
/*   M = y sin^2(theta) / z ;  Q = 15/4 - 2 sin^2(theta) [3 + 6 c r + (2 + c^2) r^2],           */
/*   c = cos(theta), r = sqrt(xy)/z.                                                            */
static real kernel_M_real(real x, real y, real theta)
{
    real z = z_real(x, y, theta);
    real st = R_SIN(theta);
    return y * st * st / z;
}
static real kernel_Q_real(real x, real y, real theta)
{
    real z = z_real(x, y, theta);
    real st = R_SIN(theta), c = R_COS(theta);
    real r = R_SQRT(x) * R_SQRT(y) / z;
    return (real)15 / 4 - 2 * st * st * (3 + 6 * c * r + (2 + c * c) * r * r);
}
double orc_kernel_M(double x, double y, double theta) { return (double)kernel_M_real(x, y, theta); }
double orc_kernel_Q(double x, double y, double theta) { return (double)kernel_Q_real(x, y, theta); }
/* ghost kernel of eq.(8) L76 after the O(4) measure eq.(4),(5) L60-64 with reading A1:         */
/* sin^4(theta) / z^2  (multiplies  -C * y * G(y) * Z(z) dy dtheta).                            */
double orc_kernel_ghost(double x, double y, double theta)
{
    real z = z_real(x, y, theta);
    real st = R_SIN(theta);
    real s2 = st * st;
    return (double)(s2 * s2 / (z * z));
}

/* ------------------------------------------------------------------------------------------ */
static real lg_of(const orc_params *p) { return R_LOG((real)p->L2 / (real)p->eps2); }
/* eq.(25) L185 (reading A4): s(u) = 2 ln(u/eps2)/ln(L2/eps2) - 1                               */
static real s_map(const orc_params *p, real u) { return 2 * R_LOG(u / (real)p->eps2) / lg_of(p) - 1; }
double orc_s_map(const orc_params *p, double u) { return (double)s_map(p, u); }
/* C = g^2 N_c / (2 pi)^3 with g^2 = 4 pi alpha(mu^2)  (eq.(8),(9) L76-80, L131)                */
static real coupling_C(const orc_params *p)
{
    return 4 * R_PI * (real)p->alpha_mu * (real)p->n_colors / (8 * R_PI * R_PI * R_PI);
}
double orc_coupling_C(const orc_params *p) { return (double)coupling_C(p); }

/* O2. ln G(u), ln Z(u) for every u > 0: the Chebyshev series eq.(23),(24) on the clamped        */
/* argument plus the analytic continuations eq.(16)-(19) L115-124 matched by continuity at      */
/* eps2 and L2 (L119, L131, L192).  c = (a_0..a_{N-1}, b_0..b_{N-1}); a <-> ln Z, b <-> ln G.   */
static void ln_dress(const orc_params *p, const real *c, real u, real *phi /*scratch N*/,
                     real *lnG, real *lnZ, real *s_clamped)
{
    const int N = p->n_cheb;
    real s = s_map(p, u);
    real EG = 0, EZ = 0;
    if (u < (real)p->eps2) {
        real l = R_LOG(u / (real)p->eps2);
        EG = (real)p->ir_exp_G * l;
        EZ = (real)p->ir_exp_Z * l;
        s = -1;
    } else if (u > (real)p->L2) {
        real gamma = -1 - 2 * (real)p->delta;
        real t = R_LOG(1 + (real)p->uv_omega * R_LOG(u / (real)p->L2));
        EG = (real)p->delta * t;
        EZ = gamma * t;
        s = 1;
    }
    if (s < -1) s = -1;
    if (s > 1) s = 1;
    phi_real(N, s, phi);
    real g = 0, zz = 0;
    for (int j = 0; j < N; ++j) { zz += c[j] * phi[j]; g += c[N + j] * phi[j]; }
    *lnG = g + EG;
    *lnZ = zz + EZ;
    *s_clamped = s;
}
void orc_ln_dress(const orc_params *p, const double *c, double u, double *lnG, double *lnZ)
{
    const int N = p->n_cheb;
    real *cr = (real *)malloc(sizeof(real) * (size_t)(3 * N));
    for (int j = 0; j < 2 * N; ++j) cr[j] = c[j];
    real g, z, s;
    ln_dress(p, cr, (real)u, cr + 2 * N, &g, &z, &s);
    *lnG = (double)g; *lnZ = (double)z;
    free(cr);
}

/* O4. Quadrature and collocation tables (H0): radial GL in s (so y_q = eps2 exp((t_q+1)Lg/2),  */
/* W_q = w_q (Lg/2) y_q), angular GL in theta on [0,pi], Chebyshev roots s_i = -cos(pi(i+1/2)/N)*/
/* mapped to x_i (fn.9 L224; readings A5, A8, A9).  n_ext = N + 1 (x_G == x_Z) or N + 2; the    */
/* subtraction points follow the roots: index N is x_Z, index N+1 (if present) is x_G.          */
int orc_n_ext(const orc_params *p) { return p->n_cheb + (p->x_G == p->x_Z ? 1 : 2); }
void orc_tables(const orc_params *p, double *x_ext, double *s_root, double *t_r, double *y, double *Wy,
                double *theta, double *Omega)
{
    const int N = p->n_cheb, Nr = p->n_r, Nt = p->n_theta;
    real Lg = lg_of(p);
    const int Nir = p->n_ir;
    int wmax = Nr > Nt ? Nr : Nt;
    if (Nir > wmax) wmax = Nir;
    double *w = (double *)malloc(sizeof(double) * (size_t)wmax);
    /* infrared piece int_0^{eps2} dy of eq.(26) L190 (the paper gives no node map: reading A23): Gauss-Legendre
     * in v on (-1,1) with y = eps2 ((1+v)/2)^4, dy = 2 eps2 ((1+v)/2)^3 dv; the dressings there are the power laws
     * eq.(16),(17).  These Nir nodes come first (ascending y); their mapped argument is the clamped s = -1. */
    if (Nir > 0) {
        orc_gauss_legendre(Nir, t_r, w);
        for (int q = 0; q < Nir; ++q) {
            real h = ((real)t_r[q] + 1) / 2;
            y[q] = (double)((real)p->eps2 * h * h * h * h);
            Wy[q] = (double)((real)w[q] * 2 * (real)p->eps2 * h * h * h);
            t_r[q] = -1.0;
        }
    }
    orc_gauss_legendre(Nr, t_r + Nir, w);
    for (int q = 0; q < Nr; ++q) {
        real yy = (real)p->eps2 * R_EXP(((real)t_r[Nir + q] + 1) * Lg / 2);
        y[Nir + q] = (double)yy;
        Wy[Nir + q] = (double)((real)w[q] * (Lg / 2) * yy);
    }
    double *tau = (double *)malloc(sizeof(double) * (size_t)Nt);
    if (p->angular_rule == 0) {
        orc_gauss_legendre(Nt, tau, w);
        for (int k = 0; k < Nt; ++k) {
            theta[k] = (double)(((real)tau[k] + 1) * R_PI / 2);
            Omega[k] = (double)((real)w[k] * R_PI / 2);
        }
    } else {
        /* tanh-sinh rule for int_{-1}^{1} dxi sqrt(1-xi^2) f  (eq.(5), ref.[31]); the paper gives no step or
         * truncation: reading A9b takes Nt equidistant abscissae t_k in [-3, 3], u_k = (pi/2) sinh t_k,
         * xi_k = tanh u_k, w_k = h (pi/2) cosh t_k / cosh^2 u_k.  In the theta form used here:
         * theta_k = 2 atan(exp(-u_k)) (so that cos theta = xi, sin theta = 1/cosh u without cancellation) and
         * Omega_k = w_k / sin theta_k, i.e. Omega sin^2 = w sqrt(1-xi^2), Omega sin^4 = w (1-xi^2)^(3/2). */
        const real tmax = 3;
        const real h = (Nt > 1) ? 2 * tmax / (real)(Nt - 1) : 0;
        for (int k = 0; k < Nt; ++k) {
            real t = tmax - h * (real)k;                 /* descending t -> ascending theta */
            real u = R_PI / 2 * (R_EXP(t) - R_EXP(-t)) / 2;
            real ch = (R_EXP(u) + R_EXP(-u)) / 2;        /* cosh u = 1 / sin theta */
            real wk = h * (R_PI / 2) * ((R_EXP(t) + R_EXP(-t)) / 2) / (ch * ch);
            theta[k] = (double)(2 * R_ATAN(R_EXP(-u)));
            Omega[k] = (double)(wk * ch);
        }
    }
    for (int i = 0; i < N; ++i) {
        real s = -R_COS(R_PI * ((real)i + (real)0.5) / (real)N);
        s_root[i] = (double)s;
        x_ext[i] = (double)((real)p->eps2 * R_EXP((s + 1) * Lg / 2));
    }
    x_ext[N] = p->x_Z;
    if (p->x_G != p->x_Z) x_ext[N + 1] = p->x_G;
    free(tau);
    free(w);
}

/* NEXT f1. Radial rule of external point x with the split of eq.(26): the n_ir infrared nodes of orc_tables,
 * then n_r Gauss-Legendre nodes in ln y on [eps2, xm] and n_r on [xm, L2], xm = min(max(x, eps2), L2) (L364: "32/64/128
 * Gauss-Legendre nodes within each of the three integration intervals").  An empty interval (x <= eps2 or x >= L2)
 * contributes nodes of zero weight.  y, Wy: n_ir + 2 n_r entries. */
void orc_radial_rule_split(const orc_params *p, double x, double *y, double *Wy)
{
    const int Nr = p->n_r, Nir = p->n_ir;
    double *t = (double *)malloc(sizeof(double) * (size_t)(2 * (Nr > Nir ? Nr : Nir)));
    double *w = t + (Nr > Nir ? Nr : Nir);
    if (Nir > 0) {
        orc_gauss_legendre(Nir, t, w);
        for (int q = 0; q < Nir; ++q) {
            real h = ((real)t[q] + 1) / 2;
            y[q] = (double)((real)p->eps2 * h * h * h * h);
            Wy[q] = (double)((real)w[q] * 2 * (real)p->eps2 * h * h * h);
        }
    }
    real xm = x;
    if (xm < (real)p->eps2) xm = p->eps2;
    if (xm > (real)p->L2) xm = p->L2;
    orc_gauss_legendre(Nr, t, w);
    for (int part = 0; part < 2; ++part) {
        const real lo = part == 0 ? (real)p->eps2 : xm, hi = part == 0 ? xm : (real)p->L2;
        const real L = R_LOG(hi / lo);
        for (int q = 0; q < Nr; ++q) {
            real yy = lo * R_EXP(((real)t[q] + 1) * L / 2);
            y[Nir + part * Nr + q] = (double)yy;
            Wy[Nir + part * Nr + q] = (double)((real)w[q] * (L / 2) * yy);
        }
    }
    free(t);
}

/* O5 + O7 at one external point x with an arbitrary product rule (y_q, W_q, theta_k, Omega_k): */
/*   Pi_G(x)   = sum_{q,k} v,           v  = -C W_q y_q Om_k sin^4/z^2 G(y_q) Z(z)    eq.(8)    */
/*   Pi_Z^Q(x) = sum wQ, wQ = (C/3x) W_q Om_k sin^2 Q P(y_q) P(z)                     eq.(9)    */
/*   Pi_Z^M(x) = sum wM, wM = (C/3x) W_q Om_k sin^2 M G(y_q) G(z)                     eq.(9)    */
/*   P(u) = G(u)^(-2-6 delta) Z(u)^(-3 delta)                                eq.(3),(9) L56-78  */
/* and, if dG_da != NULL, the coefficient derivatives (analytic; eq.(33)-(35) define J as these)*/
/*   dPi_G/db_j = sum v phi_j(s(y_q)),   dPi_G/da_j = sum v phi_j(s~(z)),                       */
/*   dPi_Z/da_j = sum e2 wQ [phi_j(s(y_q)) + phi_j(s~(z))],                                     */
/*   dPi_Z/db_j = sum (e1 wQ + wM) [phi_j(s(y_q)) + phi_j(s~(z))],  e1 = -2-6 delta, e2 = -3 delta */
static void self_energy(const orc_params *p, const real *c, real x, int ny, const double *yv, const double *Wv,
                        int nt, const double *thv, const double *Omv, real *PiG, real *PiZQ, real *PiZM,
                        real *dG_da, real *dG_db, real *dZ_da, real *dZ_db)
{
    const int N = p->n_cheb;
    const real C = coupling_C(p);
    const real e1 = -2 - 6 * (real)p->delta, e2 = -3 * (real)p->delta;
    real *phiy = (real *)malloc(sizeof(real) * (size_t)(2 * N));
    real *phiz = phiy + N;
    real sG = 0, sQ = 0, sM = 0;
    if (dG_da) for (int j = 0; j < N; ++j) dG_da[j] = dG_db[j] = dZ_da[j] = dZ_db[j] = 0;
    for (int q = 0; q < ny; ++q) {
        real y = yv[q], W = Wv[q];
        real lnGy, lnZy, sy;
        ln_dress(p, c, y, phiy, &lnGy, &lnZy, &sy);
        real lnPy = e1 * lnGy + e2 * lnZy;
        for (int k = 0; k < nt; ++k) {
            real th = thv[k], Om = Omv[k];
            real z = z_real(x, y, th);
            real lnGz, lnZz, sz;
            ln_dress(p, c, z, phiz, &lnGz, &lnZz, &sz);
            real lnPz = e1 * lnGz + e2 * lnZz;
            real st = R_SIN(th);
            real s2 = st * st;
            real Q = kernel_Q_real(x, y, th);
            real M = kernel_M_real(x, y, th);
            real v = -C * W * y * Om * s2 * s2 / (z * z) * R_EXP(lnGy + lnZz);
            /* at the ghost subtraction point x_G = 0 (L135) only eq.(8) is evaluated: gluon prefactor 1/(3x) -> 0 */
            const real c3x = (x > 0) ? C / (3 * x) : 0;
            real wQ = c3x * W * Om * s2 * Q * R_EXP(lnPy + lnPz);
            real wM = c3x * W * Om * s2 * M * R_EXP(lnGy + lnGz);
            sG += v; sQ += wQ; sM += wM;
            if (dG_da) {
                for (int j = 0; j < N; ++j) {
                    dG_db[j] += v * phiy[j];
                    dG_da[j] += v * phiz[j];
                    dZ_da[j] += e2 * wQ * (phiy[j] + phiz[j]);
                    dZ_db[j] += (e1 * wQ + wM) * (phiy[j] + phiz[j]);
                }
            }
        }
    }
    *PiG = sG; *PiZQ = sQ; *PiZM = sM;
    free(phiy);
}

/* Test entry: self-energies (and optionally derivatives) at x for a caller-supplied rule.      */
void orc_self_energy(const orc_params *p, const double *c, double x, int ny, const double *y, const double *Wy,
                     int nt, const double *theta, const double *Omega, double *out3 /*PiG,PiZ_Q,PiZ_M*/,
                     double *d4 /* NULL or [4][N]: dG_da, dG_db, dZ_da, dZ_db */)
{
    const int N = p->n_cheb;
    real *cr = (real *)malloc(sizeof(real) * (size_t)(6 * N));
    for (int j = 0; j < 2 * N; ++j) cr[j] = c[j];
    real a, b, m;
    real *d = cr + 2 * N;
    self_energy(p, cr, (real)x, ny, y, Wy, nt, theta, Omega, &a, &b, &m, d4 ? d : NULL, d4 ? d + N : NULL,
                d4 ? d + 2 * N : NULL, d4 ? d + 3 * N : NULL);
    out3[0] = (double)a; out3[1] = (double)b; out3[2] = (double)m;
    if (d4) for (int j = 0; j < 4 * N; ++j) d4[j] = (double)d[j];
    free(cr);
}

/* O6 + O7. Residual F (eq.(29),(30) L210-213) and Jacobian J (eq.(35),(36) L238-301):          */
/*   F = (z(x_0..x_{N-1}); g(x_0..x_{N-1})),  z(x_i) = 1/Z(x_i) - gZ - Pi_Z(x_i) + Pi_Z(x_Z),   */
/*   g(x_i) = 1/G(x_i) - gG - Pi_G(x_i) + Pi_G(x_G);  gG = 1/G(x_G), gZ = 1/Z(x_Z) (eq.(14),(15))*/
/*   J row-major [2N][2N], rows (z; g), columns (a; b)  (readings A6, A7).                      */
/* J may be NULL (residual only).  Returns 0.                                                   */
int orc_residual_jacobian(const orc_params *p, const double *c, double gG, double gZ, double *F, double *J)
{
    const int N = p->n_cheb, Nr = (p->radial_split ? 2 * p->n_r : p->n_r) + p->n_ir, Nt = p->n_theta;
    const int Ne = orc_n_ext(p);
    const int iZ = N, iG = (p->x_G == p->x_Z) ? N : N + 1;
    double *x_ext = (double *)malloc(sizeof(double) * (size_t)(Ne + N + 3 * Nr + 2 * Nt));
    double *s_root = x_ext + Ne, *t_r = s_root + N, *y = t_r + Nr, *Wy = y + Nr, *th = Wy + Nr, *Om = th + Nt;
    orc_tables(p, x_ext, s_root, t_r, y, Wy, th, Om);
    real *cr = (real *)malloc(sizeof(real) * (size_t)(2 * N + N + 3 * Ne + 4 * Ne * N));
    real *phi = cr + 2 * N, *PiG = phi + N, *PiQ = PiG + Ne, *PiM = PiQ + Ne, *D = PiM + Ne;
    for (int j = 0; j < 2 * N; ++j) cr[j] = c[j];
    for (int e = 0; e < Ne; ++e) {
        real *d = D + (size_t)4 * N * e;
        if (p->radial_split) orc_radial_rule_split(p, x_ext[e], y, Wy);      /* the rule of this external point */
        self_energy(p, cr, (real)x_ext[e], Nr, y, Wy, Nt, th, Om, &PiG[e], &PiQ[e], &PiM[e],
                    J ? d : NULL, J ? d + N : NULL, J ? d + 2 * N : NULL, J ? d + 3 * N : NULL);
    }
    for (int i = 0; i < N; ++i) {
        real lnG, lnZ, s;
        ln_dress(p, cr, (real)x_ext[i], phi, &lnG, &lnZ, &s);
        real invZ = R_EXP(-lnZ), invG = R_EXP(-lnG);
        real PiZ_i = PiQ[i] + PiM[i], PiZ_s = PiQ[iZ] + PiM[iZ];
        F[i] = (double)(invZ - (real)gZ - PiZ_i + PiZ_s);
        F[N + i] = (double)(invG - (real)gG - PiG[i] + PiG[iG]);
        if (J) {
            const real *di = D + (size_t)4 * N * i, *dZs = D + (size_t)4 * N * iZ, *dGs = D + (size_t)4 * N * iG;
            /* use the exact root s_i for the local term (phi at the collocation point) */
            phi_real(N, (real)s_root[i], phi);
            for (int j = 0; j < N; ++j) {
                /* dG_da = d[0..N), dG_db = d[N..2N), dZ_da = d[2N..3N), dZ_db = d[3N..4N) */
                J[(size_t)i * 2 * N + j] = (double)(-phi[j] * invZ - di[2 * N + j] + dZs[2 * N + j]);
                J[(size_t)i * 2 * N + N + j] = (double)(-di[3 * N + j] + dZs[3 * N + j]);
                J[(size_t)(N + i) * 2 * N + j] = (double)(-di[j] + dGs[j]);
                J[(size_t)(N + i) * 2 * N + N + j] = (double)(-phi[j] * invG - di[N + j] + dGs[N + j]);
            }
        }
    }
    free(cr);
    free(x_ext);
    return 0;
}

/* O8 (linear algebra part). Solve A x = b for dense row-major A[n][n] (L303 "standard LU       */
/* decomposition routines"; reading A18): scale row i of (A|b) by 1/max_j|A_ij|, LU with        */
/* partial pivoting (first maximal element wins ties), forward/back substitution.               */
/* stats[0] = max|x|, stats[1] = max_i |b_i| row-scaled, stats[2] = min |pivot|,                */
/* stats[3] = growth = max|U| / max|A_scaled|.  Returns 0, or 1 if a pivot is exactly 0.        */
int orc_lu_solve(int n, const double *A, const double *b, double *x, double *stats)
{
    real *M = (real *)malloc(sizeof(real) * (size_t)n * (size_t)(n + 1));
    real fmax = 0, amax = 0, umax = 0, pmin = INFINITY;
    int singular = 0;
    for (int i = 0; i < n; ++i) {
        real m = 0;
        for (int j = 0; j < n; ++j) { real a = R_FABS((real)A[(size_t)i * n + j]); if (a > m) m = a; }
        real r = (m > 0) ? 1 / m : 1;
        for (int j = 0; j < n; ++j) {
            M[(size_t)i * (n + 1) + j] = (real)A[(size_t)i * n + j] * r;
            real a = R_FABS(M[(size_t)i * (n + 1) + j]); if (a > amax) amax = a;
        }
        M[(size_t)i * (n + 1) + n] = (real)b[i] * r;
        if (R_FABS(M[(size_t)i * (n + 1) + n]) > fmax) fmax = R_FABS(M[(size_t)i * (n + 1) + n]);
    }
    for (int k = 0; k < n; ++k) {
        int piv = k; real pm = R_FABS(M[(size_t)k * (n + 1) + k]);
        for (int i = k + 1; i < n; ++i) {
            real a = R_FABS(M[(size_t)i * (n + 1) + k]);
            if (a > pm) { pm = a; piv = i; }
        }
        if (piv != k)
            for (int j = 0; j <= n; ++j) {
                real t = M[(size_t)k * (n + 1) + j];
                M[(size_t)k * (n + 1) + j] = M[(size_t)piv * (n + 1) + j];
                M[(size_t)piv * (n + 1) + j] = t;
            }
        if (pm < pmin) pmin = pm;
        if (pm == 0) { singular = 1; continue; }
        real pk = M[(size_t)k * (n + 1) + k];
        for (int i = k + 1; i < n; ++i) {
            real l = M[(size_t)i * (n + 1) + k] / pk;
            M[(size_t)i * (n + 1) + k] = 0;
            for (int j = k + 1; j <= n; ++j) M[(size_t)i * (n + 1) + j] -= l * M[(size_t)k * (n + 1) + j];
        }
    }
    for (int i = 0; i < n; ++i)
        for (int j = i; j < n; ++j) { real a = R_FABS(M[(size_t)i * (n + 1) + j]); if (a > umax) umax = a; }
    real xmax = 0;
    for (int i = n - 1; i >= 0; --i) {
        real s = M[(size_t)i * (n + 1) + n];
        for (int j = i + 1; j < n; ++j) s -= M[(size_t)i * (n + 1) + j] * (real)x[j];
        real xi = s / M[(size_t)i * (n + 1) + i];
        x[i] = (double)xi;
        if (R_FABS(xi) > xmax) xmax = R_FABS(xi);
    }
    if (stats) {
        stats[0] = (double)xmax; stats[1] = (double)fmax; stats[2] = (double)pmin;
        stats[3] = (double)(amax > 0 ? umax / amax : 0);
    }
    free(M);
    return singular;
}

/* O8. One Newton-Raphson step, eq.(31)-(35) L218-273: solve J Delta = F, c <- c - rho Delta.   */
int orc_newton_step(const orc_params *p, double *c, double gG, double gZ, double rho, double *stats)
{
    const int n = 2 * p->n_cheb;
    double *F = (double *)malloc(sizeof(double) * (size_t)n * (size_t)(n + 2));
    double *J = F + n, *d = J + (size_t)n * n;
    orc_residual_jacobian(p, c, gG, gZ, F, J);
    int rc = orc_lu_solve(n, J, F, d, stats);
    for (int j = 0; j < n; ++j) c[j] -= rho * d[j];
    free(F);
    return rc;
}

/* NEXT f4. Schwinger function of the gluon propagator, eq.(20) L157 with sigma(p^2) = Z(p^2)/p^2 (L161):
 *   Delta(t) = (1/pi) int_0^inf d|p| cos(t|p|) Z(p^2)/p^2
 * as a "generalized scalar product" over a mapped Gauss-Legendre rule (L382; 2^17 nodes in fn.13).  The paper
 * does not give the map: reading A22 takes n_nodes GL nodes in u = ln|p| on [ln sqrt(p2_min), ln sqrt(p2_max)],
 * d|p| = |p| du.  Z outside [eps2, L2] is the continuation of O2.  Plain serial sums, node by node. */
void orc_schwinger(const orc_params *p, const double *c, int n_nodes, double p2_min, double p2_max, int n_t,
                   const double *t, double *out)
{
    const int N = p->n_cheb;
    real *cr = (real *)malloc(sizeof(real) * (size_t)(3 * N + 2 * n_nodes));
    real *phi = cr + 2 * N, *pn = phi + N, *fn = pn + n_nodes;
    for (int j = 0; j < 2 * N; ++j) cr[j] = c[j];
    const real u0 = R_LOG((real)p2_min) / 2, u1 = R_LOG((real)p2_max) / 2;
    for (int i = 0; i < n_nodes; ++i) {
        real x, w;
        gl_node(n_nodes, i, &x, &w);
        real u = u0 + (x + 1) / 2 * (u1 - u0);
        real pp = R_EXP(u);
        real lnG, lnZ, sc;
        ln_dress(p, cr, pp * pp, phi, &lnG, &lnZ, &sc);
        pn[i] = pp;
        fn[i] = w * (u1 - u0) / 2 * pp * R_EXP(lnZ) / (pp * pp);      /* d|p| * Z(p^2)/p^2 */
    }
    for (int m = 0; m < n_t; ++m) {
        real sum = 0;
        for (int i = 0; i < n_nodes; ++i) sum += fn[i] * R_COS((real)t[m] * pn[i]);
        out[m] = (double)(sum / R_PI);
    }
    free(cr);
}

/* The same sums in two steps, for the paper's full-size rule (2^17 nodes, fn.13): the node table costs O(n_nodes^2)
 * (every node is a Newton iteration on the n_nodes-term Legendre recurrence), so a test may compute ranges of nodes
 * [i0, i1) on several host threads and then sum serially -- identical arithmetic to orc_schwinger in the double build. */
void orc_schwinger_terms(const orc_params *p, const double *c, int n_nodes, double p2_min, double p2_max, int i0, int i1,
                         double *pn, double *fn)
{
    const int N = p->n_cheb;
    real *cr = (real *)malloc(sizeof(real) * (size_t)(3 * N));
    real *phi = cr + 2 * N;
    for (int j = 0; j < 2 * N; ++j) cr[j] = c[j];
    const real u0 = R_LOG((real)p2_min) / 2, u1 = R_LOG((real)p2_max) / 2;
    for (int i = i0; i < i1; ++i) {
        real x, w;
        gl_node(n_nodes, i, &x, &w);
        real u = u0 + (x + 1) / 2 * (u1 - u0);
        real pp = R_EXP(u);
        real lnG, lnZ, sc;
        ln_dress(p, cr, pp * pp, phi, &lnG, &lnZ, &sc);
        pn[i] = (double)pp;
        fn[i] = (double)(w * (u1 - u0) / 2 * pp * R_EXP(lnZ) / (pp * pp));
    }
    free(cr);
}
void orc_schwinger_sum(int n_nodes, const double *pn, const double *fn, int n_t, const double *t, double *out)
{
    for (int m = 0; m < n_t; ++m) {
        real sum = 0;
        for (int i = 0; i < n_nodes; ++i) sum += (real)fn[i] * R_COS((real)t[m] * (real)pn[i]);
        out[m] = (double)(sum / R_PI);
    }
}

int orc_sizeof_real(void) { return (int)sizeof(real); }

/*
 * dse.h -- C ABI of the B200 (sm_100a) library that builds the residual vector and the analytic
 * Newton (Jacobian) matrix of the Chebyshev-collocated Landau-gauge ghost/gluon Dyson-Schwinger
 * equations of Hopfer/Alkofer/Haase, "Solving the Ghost-Gluon System of Yang-Mills Theory on GPUs"
 * (arXiv:1206.1779; cited below as PAPER.md L<line>, section/equation), and performs the Newton
 * update with an on-GPU equilibrated LU.
 *
 * What is computed (all fp64; readings of the paper are listed in DESIGN.md):
 *   unknowns      c = (a_0..a_{N-1}, b_0..b_{N-1}),  ln Z(x) = a_0/2 + sum_j a_j T_j(s(x)),
 *                 ln G(x) = b_0/2 + sum_j b_j T_j(s(x))                    eq.(23),(24),(28) L177-206
 *   map           s(x) = 2 ln(x/eps2)/ln(L2/eps2) - 1                      eq.(25)
 *   self-energies Pi_G(x), Pi_Z(x): 2-D quadratures of eq.(8),(9) L76-80 with the kernels
 *                 M, Q of eq.(10),(11) L88-96, the O(4) measure eq.(4),(5) L60-64,
 *                 z = x + y - 2 sqrt(xy) cos(theta) L62/L192, and the continuations eq.(16)-(19)
 *                 L115-124 of G(z), Z(z) outside [eps2, L2]
 *   residual      F = (z(x_0..x_{N-1}); g(x_0..x_{N-1}))                   eq.(27),(29),(30) L194-213
 *                 z(x_i) = 1/Z(x_i) - 1/Z(x_Z) - Pi_Z(x_i) + Pi_Z(x_Z),  g likewise (MOM, eq.(14),(15))
 *   Newton matrix J[r][c] = dF_r/dc_c, rows (z; g), columns (a; b)          eq.(33)-(36) L228-301
 *                 (analytic derivative; the paper's central differences eq.(38) L318 are a check)
 *   update        solve J Delta = F, c <- c - rho Delta                     eq.(31),(32) L218-222
 *
 * Conventions
 *   - Every pointer named *_dev is a DEVICE pointer owned by the CALLER (e.g. a torch tensor's
 *     data_ptr()); every pointer named *_host is a HOST pointer owned by the caller.  The library
 *     never allocates, frees or keeps caller buffers.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  dse_residual,
 *     dse_jacobian and dse_newton_step only enqueue work on `stream` and return; they never
 *     synchronise.  dse_create / dse_destroy / *_host calls synchronise.
 *   - Return value: 0 (DSE_OK) or a negative DSE_E* code; no exception crosses the ABI.  A singular or
 *     ill-scaled J is reported through stats_dev (min |pivot|), not through the return code.
 *   - A handle is bound to the device that was current in dse_create and must be used from one
 *     host thread, and on one stream, at a time.  Everything that selects a code path is in dse_params
 *     (no environment variables); the library keeps no state outside the handles, with ONE exception
 *     that the caller asks for explicitly: DSE_FLAG_CONST_COEF (below).  No CPU fallback: without a
 *     CUDA device dse_create fails with DSE_ECUDA.
 *   - Layouts: c_dev [n_batch][2N] (a then b); bc_dev [n_batch][2] = (1/G(x_G), 1/Z(x_Z));
 *     F_dev [n_batch][2N]; J_dev [n_batch][2N][2N] row-major; stats_dev [n_batch][4].
 */
#ifndef DSE_H_
#define DSE_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define DSE_API __attribute__((visibility("default")))
#else
#define DSE_API
#endif

#define DSE_OK 0
#define DSE_EINVAL (-1) /* bad parameter or null pointer                          */
#define DSE_ENOMEM (-2) /* host or device allocation failed                       */
#define DSE_ECUDA (-3)  /* CUDA runtime error (text via dse_last_error)           */
#define DSE_EBUSY (-4)  /* DSE_FLAG_CONST_COEF: the constant-bank slot is held by another handle */

#define DSE_MAX_NCHEB 128

/* Parameters of the discretisation and of the truncation: one POD struct, the only configuration channel. */
typedef struct dse_params {
    int32_t n_cheb;     /* N: Chebyshev polynomials per dressing function, 2 <= N <= 128 (eq.(23),(24))  */
    int32_t n_r;        /* radial Gauss-Legendre nodes in ln y on [eps2, L2], >= 2 (L62, eq.(26) reading) */
    int32_t n_theta;    /* angular Gauss-Legendre nodes in theta on [0, pi], >= 2 (L62-66 reading)       */
    int32_t n_batch;    /* independent systems sharing the grid (config 4), >= 1                         */
    double eps2, L2;    /* IR matching point and UV cutoff, 0 < eps2 < L2 (L188)                         */
    double alpha_mu;    /* alpha(mu^2) = g^2/4pi (L131,L135); C = 4 pi alpha N_c/(2 pi)^3                */
    double n_colors;    /* N_c                                                                           */
    double x_G, x_Z;    /* MOM subtraction points (eq.(14),(15)); x_Z > 0; x_G >= 0, x_G = 0 (the paper's choice,
                           L135) needs x_G != x_Z: at x = 0 only the ghost equation is evaluated             */
    double delta;       /* ghost anomalous dimension -9/44 (L58); gamma = -1 - 2 delta (L131)            */
    double ir_exp_G;    /* exponent of G below eps2, eq.(17): -kappa                                     */
    double ir_exp_Z;    /* exponent of Z below eps2, eq.(16): 2 kappa                                    */
    double uv_omega;    /* omega of eq.(18),(19); 0 => constant continuation above L2                    */
    int32_t flags;      /* DSE_FLAG_* bits                                                               */
    int32_t n_r_ir;     /* >= 0: Gauss-Legendre nodes of the infrared piece int_0^{eps2} dy of eq.(26),
                           y = eps2 ((1+v)/2)^4 (reading A23); 0 = no infrared piece (BASELINE configs) */
} dse_params;

#define DSE_FLAG_GEOMETRY_CACHE 1 /* precompute the coefficient-independent per-point factors once in
                                     dse_create (32 B/point in HBM) instead of per build            */

#define DSE_FLAG_ANGULAR_TANH_SINH 2 /* angular rule: tanh-sinh in xi = cos(theta) (eq.(5)) with n_theta
                                        equidistant abscissae t_k in [-3,3], xi_k = tanh((pi/2) sinh t_k), instead of
                                        Gauss-Legendre in theta (reading A9b)                              */

#define DSE_FLAG_RADIAL_SPLIT 4 /* the paper's radial split int_{eps2}^{x} + int_{x}^{L2} (eq.(26)) with n_r nodes in
                                   EACH interval (L364): the radial rule then depends on the external point
                                   (n_r_ir + 2 n_r nodes per point); default: one rule on [eps2, L2] (BASELINE configs) */

#define DSE_FLAG_USER_TABLES 8 /* the quadrature nodes and weights come from the caller (dse_create_with_tables): used to
                                  separate kernel error from table-builder error in parity tests -- PAPER.md L62 never
                                  gives the radial node map, so two independent builders may differ in the last digits */

#define DSE_FLAG_CONST_COEF 16 /* single system (n_batch = 1), software-pipelined point kernel, N a multiple of 8 with
                                  N/8 in {1,2,4,8,16}: the Chebyshev coefficients are read as constant-bank operands of the
                                  fp64 FMAs (about 12 % faster point kernel at BASELINE configs[3]; an in-stream device-to-device
                                  copy of c into the library's __constant__ array precedes every build).  The array is
                                  ONE slot per process and device context: dse_create fails with DSE_EBUSY while another
                                  live handle holds it, and with DSE_EINVAL if the shape cannot use it; the slot is released
                                  by dse_destroy.  Never taken implicitly: without the flag the coefficients sit in shared
                                  memory, whatever the creation order of the handles. */

#define DSE_FLAG_PER_SYSTEM_KERNELS 32 /* n_batch >= 8: do not use the batched fp64-tensor point kernel (systems are then
                                          walked one after the other by the single-system kernels); for tests and A/B runs */

typedef struct dse_handle dse_handle; /* opaque; owned by the library */

/* Builds the quadrature/collocation tables (Gauss-Legendre in ln y and in theta, Chebyshev roots
 * x_i, phi_j tables; eq.(25), fn.9 L224) on the host, copies them to the current
 * device and allocates the workspace.  Synchronous.  *out is set only on success. */
DSE_API int dse_create(const dse_params *params, dse_handle **out);

/* Caller-supplied quadrature tables (DSE_FLAG_USER_TABLES must be set in params->flags; dse_create refuses that flag).
 * All HOST pointers, read during the call only:
 *   x_ext[n_ext]            external momenta x_e: the N collocation points, then x_Z, then x_G if different (dse_n_ext order)
 *   y, Wy [n_rules][n_rad]  radial nodes y_q (infrared piece first) and weights of dy (for the log-mapped rule: w_q (Lg/2) y_q),
 *                           n_rad = n_r_ir + n_r (n_rules = 1), or n_r_ir + 2 n_r per external point under
 *                           DSE_FLAG_RADIAL_SPLIT (n_rules = n_ext)
 *   theta, Omega [n_theta]  angular nodes and weights of d(theta) (the sin^2 of the measure eq.(4),(5) stays in the integrand)
 * Everything else (s(y_q) by eq.(25), phi_j tables, square roots, the continuation add-ons) is derived from these values in
 * long double.  The collocation abscissae s_i stay the exact Chebyshev roots (fn.9 L224). */
typedef struct dse_tables {
    const double *x_ext, *y, *Wy, *theta, *Omega;
} dse_tables;
DSE_API int dse_create_with_tables(const dse_params *params, const dse_tables *tables, dse_handle **out);

/* Frees everything dse_create made.  Synchronous.  NULL is accepted. */
DSE_API int dse_destroy(dse_handle *h);

/* F only (eq.(29),(30)).  Same kernels as dse_jacobian without the derivative accumulation. */
DSE_API int dse_residual(dse_handle *h, const double *c_dev, const double *bc_dev, double *F_dev, void *stream);

/* F and J (eq.(29),(30),(35)).  Asynchronous on `stream`; deterministic (no atomics, fixed
 * reduction order): repeated calls give bitwise identical results. */
DSE_API int dse_jacobian(dse_handle *h, const double *c_dev, const double *bc_dev, double *J_dev, double *F_dev,
                 void *stream);

/* Self-check mode (the paper's own definition of the Newton matrix, eq.(38),(39) L316-336): J by central finite
 * differences of the residual, column j from c_j +- h_j with h_j = eps_rel * max(1, |c_j|) (the paper uses
 * eps_j ~ 1e-5 a_j, which fails at a_j = 0: DESIGN.md reading A16).  4N residual builds; asynchronous on `stream`.
 * J_dev [n_batch][2N][2N].  Meant for verification, not for speed. */
DSE_API int dse_jacobian_fd(dse_handle *h, const double *c_dev, const double *bc_dev, double eps_rel, double *J_dev,
                            void *stream);

/* One Newton-Raphson step (eq.(31)-(35)): builds J, F, scales each row of (J|F) by 1/max_j|J_ij|,
 * LU with partial pivoting (largest |a_ik|; exactly equal candidates: see below), solves J Delta = F,
 * c <- c - rho Delta in place.  stats_dev[b] = { max|Delta|, max_i|F_i| row-scaled, min|pivot|, growth max|U|/max|A| }.
 * stats_dev may be NULL.
 * Arithmetic of the factorisation (2N <= 128: fused multiply-add updates, multipliers = entry * (1/pivot) with a
 * reciprocal good to ~1 ulp; equal candidates go to the smallest row index; a pivot below 2^-1022 counts as singular.
 * 2N > 128: unfused updates, correctly rounded quotients, equal candidates go to the first row in the order a
 * row-swapping elimination would have).  Either way the unknowns agree with a plain elimination to rounding times the
 * conditioning of J; DESIGN.md section 3 states the parity bar the tests apply.
 * Singular or non-finite systems: the call is asynchronous, so they are reported through stats_dev, not the return code.
 * If a pivot is exactly zero (stats[2] == 0) or Delta has a non-finite entry, c is left UNCHANGED for that system and
 * stats[0] = +Inf; a caller that does not pass stats_dev cannot tell.  dse_newton_solve checks this itself (status -1). */
DSE_API int dse_newton_step(dse_handle *h, double *c_dev, const double *bc_dev, double rho, double *stats_dev,
                    void *stream);

/* The whole Newton-Raphson iteration (eq.(31)-(35); L226: "iterated", under-relaxed far from the solution, rho back
 * to one close to it) on the device, with no host round trip between the steps: one CUDA graph whose WHILE node
 * repeats the body (build J, F -> equilibrated LU -> update + convergence test) until every system has
 * |Delta|_inf < tol (Delta = the full Newton improvement of the step, tested before relaxation; the step that
 * passes the test is still applied) or max_iter steps have run.  Per system and step the relaxation is
 *     rho_n = min(rho, step_cap / |Delta_n|_inf)   (step_cap > 0: no coefficient moves by more than step_cap;
 *                                                    step_cap <= 0: rho_n = rho)             [DESIGN.md reading A26]
 * A system that has converged, or whose Delta is not finite (singular J), is frozen; the others go on.
 * c_dev [n_batch][2N] in/out, bc_dev [n_batch][2];  info_dev [n_batch][6] (may be NULL) =
 *   { steps taken, |Delta|_inf of the last step, row-scaled |F|_inf of the last step, smallest |pivot| over all
 *     steps, rho_n of the last step, status: 1 converged, 0 max_iter reached, -1 non-finite Delta }.
 * 0 < rho <= 1, tol >= 0 (0: always run max_iter steps), 1 <= max_iter.  Asynchronous on `stream`; the graph is
 * built at the first call and kept in the handle; the iterates live in the handle's own buffers, so calls on one
 * handle must be issued on one stream at a time (as for every other call that uses the workspace). */
DSE_API int dse_newton_solve(dse_handle *h, double *c_dev, const double *bc_dev, double rho, double step_cap, double tol,
                             int32_t max_iter, double *info_dev, void *stream);

/* Solves A x = b for n_sys dense row-major systems with the same equilibrated LU kernel that
 * dse_newton_step uses (exposed for tests): A_dev [n_sys][n][n], b_dev [n_sys][n], x_dev [n_sys][n],
 * stats_dev [n_sys][4] or NULL.  A_dev and b_dev are not modified.  1 <= n <= 256; n > 128 uses the handle's own
 * scratch and therefore requires n == 2 n_cheb and n_sys <= n_batch (else DSE_EINVAL). */
DSE_API int dse_lu_solve(dse_handle *h, int32_t n, int32_t n_sys, const double *A_dev, const double *b_dev,
                 double *x_dev, double *stats_dev, void *stream);

/* Host-buffer convenience (used for the end-to-end measurement): c, bc go to the device in one staged copy, dse_jacobian
 * runs, J, F come back -- up to 1 MiB of results are written by the assemble kernel straight into a mapped pinned buffer of
 * the handle (no copy node on the stream), larger ones are copied back; synchronous on the legacy default stream.
 * J_host may be NULL (then dse_residual).  The staging buffers are allocated at the first call. */
DSE_API int dse_jacobian_host(dse_handle *h, const double *c_host, const double *bc_host, double *J_host,
                      double *F_host);

/* Sizes: n_ext = number of external points (N roots, then x_Z, then x_G if different). */
DSE_API int dse_n_ext(const dse_handle *h);

/* Copies the tables to host arrays (any pointer may be NULL), in the layout of dse_tables: x_ext[n_ext],
 * y, Wy [n_rules][n_rad] (n_rules = 1, n_rad = n_r_ir + n_r; under DSE_FLAG_RADIAL_SPLIT n_rules = n_ext and
 * n_rad = n_r_ir + 2 n_r: the rule of every external point), theta[n_theta], Omega[n_theta].  For tests. */
DSE_API int dse_get_tables(const dse_handle *h, double *x_ext_host, double *y_host, double *Wy_host,
                   double *theta_host, double *Omega_host);

/* Number of kernels this handle has launched so far (bench.py's gpu_launches). */
DSE_API int64_t dse_launch_count(const dse_handle *h);

/* Configuration of the dominant kernel, for reporting: out[0] = grid, out[1] = block,
 * out[2] = dynamic shared memory bytes, out[3] = registers/thread, out[4] = resident CTAs/SM,
 * out[5] = SM count, out[6] = variant of the Jacobian point kernel (0 generic, 1 software-pipelined,
 * 2 batched: 8 systems per warp on the fp64 tensor path, chosen when n_batch >= 8 (padded to a multiple of 8 with
 * idle systems, at most a quarter of the padded batch), n_cheb <= 64 and n_theta >= 32),
 * out[7] = kernels per Jacobian build (1: the point kernel also reduces, contracts and assembles). */
DSE_API int dse_kernel_info(const dse_handle *h, int32_t out[8]);

/* Per-kernel device timing of the dominant (point) kernel, for the roofline report: while enabled,
 * every build records a CUDA event pair around the point kernel on the build's stream (nothing else
 * changes; where the point kernel is the whole build, its fused reduction/assembly tail is inside the pair).  dse_get_timing synchronises on the recorded events, adds them up and returns the
 * accumulated milliseconds and launch count since the last reset (enable resets). */
DSE_API int dse_set_timing(dse_handle *h, int32_t enable);
DSE_API int dse_get_timing(dse_handle *h, double *total_ms, int64_t *launches);

/* NEXT f4 -- the paper's second GPU workload (Table 2).
 * dse_gauss_legendre: n-point Gauss-Legendre rule generated on the device (Newton iteration on the Legendre
 * recurrence, one thread per pair of nodes): x_dev[n] ascending in (-1,1), w_dev[n]; work_dev >= 2(n+2) doubles.
 * dse_schwinger: Delta(t_m) = (1/pi) int d|p| cos(t_m |p|) Z(p^2)/p^2, eq.(20) with sigma = Z/p^2 (L161), over
 * n_nodes Gauss-Legendre nodes in ln|p| on [sqrt(p2_min), sqrt(p2_max)] (reading A22); Z from the
 * a-coefficients of c_dev [n_batch][2N] with the continuation of eq.(16),(19) outside [eps2, L2].
 * t_dev[n_t], delta_dev[n_batch][n_t]; work_dev >= (5 + n_batch) n_nodes + 4 doubles.  Asynchronous on `stream`,
 * deterministic.  2 <= n, n_nodes <= 2^24; 0 < p2_min < p2_max. */
DSE_API int dse_gauss_legendre(int32_t n, double *x_dev, double *w_dev, double *work_dev, void *stream);

/* dse_gauss_legendre for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): same kernels, same results, but the scratch (2 (n + 2) doubles of recurrence
 * coefficients) lives in a static device array of the library instead of work_dev.  The call allocates nothing (no
 * cudaMalloc / cudaFree / allocating library routine).  Limits and sharing:
 *   - 2 <= n <= DSE_GL_NOALLOC_MAX_N, else DSE_EINVAL with a message (dse_last_error);
 *   - the array (2 MiB) exists once per GPU that loads the library, until the process exits;
 *   - EVERY call on a device uses the same array and it keeps the last call's contents (nothing in it needs clearing:
 *     each call rewrites what it reads): calls that overlap on the GPU -- different streams, or a captured graph replayed
 *     concurrently -- RACE.  Issue them on one stream, or order them with events. */
#define DSE_GL_NOALLOC_MAX_N (1 << 17)
DSE_API int dse_gauss_legendre_noalloc(int32_t n, double *x_dev, double *w_dev, void *stream);
DSE_API int dse_schwinger(dse_handle *h, const double *c_dev, int32_t n_nodes, double p2_min, double p2_max,
                          const double *t_dev, int32_t n_t, double *delta_dev, double *work_dev, void *stream);

/* The dressing functions of a coefficient set at arbitrary momenta (what a solve is run for: PAPER.md Fig. 3-5):
 * ln G(x_m), ln Z(x_m) from the series eq.(23),(24) on the clamped argument s(x) (eq.(25)) plus the continuations
 * eq.(16)-(19) below eps2 and above L2, and the running coupling alpha(x_m) = alpha(mu^2) G^2(x_m) Z(x_m) (L145).
 * x_dev [n_x], all > 0; outputs [n_batch][n_x], any of them may be NULL (not all).  Asynchronous on `stream`. */
DSE_API int dse_dressing(dse_handle *h, const double *c_dev, const double *x_dev, int32_t n_x, double *lnG_dev,
                         double *lnZ_dev, double *alpha_dev, void *stream);

/* Text of a DSE_E* code, and the last CUDA error text seen by this thread ("" if none). */
DSE_API const char *dse_strerror(int code);
DSE_API const char *dse_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* DSE_H_ */

// dse_internal.h -- shared between the host API (dse_api.cu), the table builder (dse_tables.cpp)
// and the kernels.  Not part of the public ABI.
#pragma once
#include <cstdint>
#include <vector>

#include "../../include/dse.h"
#include "../../include/dse_diag.h"

namespace dse {

constexpr int CJ = 8;             // Chebyshev indices per chunk lane (phase 2 of the point kernel)
constexpr int MAX_NCH = DSE_MAX_NCHEB / CJ;

// Host-side tables (built once per handle; eq.(25), fn.9 L224).
struct HostTables {
    int N = 0, Npad = 0, Nr = 0, Nt = 0, Ntpad = 0, Next = 0;
    int iZ = 0, iG = 0;                       // external-point index of x_Z, x_G
    int rstride = 0;                          // radial tables are [Next][Nr] (rstride = Nr, split rule) or shared (0)
    double Lg = 0, C = 0;
    std::vector<double> x_ext, sx_ext, c3x_ext;   // x, sqrt x, C/(3x)
    std::vector<double> y, sy, Wy, t_r;           // radial nodes (infrared piece first), sqrt, dy weight, s(y_q)
    std::vector<double> EGy, EZy;                 // continuation add-ons of ln G(y_q), ln Z(y_q) (0 inside [eps2, L2])
    std::vector<double> theta, Omega;             // angular nodes/weights (unpadded)
    std::vector<double> ang;                      // [Ntpad][6]: sh2, 6c, 2+c^2, -2 s2, Om s2, Om s2^2
    std::vector<double> phi_y;                    // [Nr][Npad]   phi_j(t_q)   (phi_0 = 1/2)
    std::vector<double> phi_x;                    // [N][Npad]    phi_j(s_i)
};
// user: caller-supplied nodes and weights (DSE_FLAG_USER_TABLES) or nullptr
void build_tables(const dse_params &p, const dse_tables *user, HostTables &t);

// Everything the kernels need, passed by value.
constexpr int SELF_H1_MAX_ROWS = 2048;   // generic kernel: largest B*Gext*Nr for which every CTA computes G(y_q), P(y_q) of all rows itself
constexpr int TAIL_POLLS = 4096;       // fused tail: polls (64 ns apart + a memory round trip) for the subtraction points' rows before giving up

struct KParams {
    int N, Npad, NCH, SUB, rounds;     // Chebyshev: N, padded to NCH*CJ; phase-2 lanes = NCH chunk x SUB point lanes
    int Nr, Nt, Ntpad, g, rpb;         // angular nodes padded to a multiple of g (g = 32, or pow2 >= Nt); rows per batch
    int Next, B, iZ, iG;
    int rstride, Gext;                 // radial tables: element (e, q) at e*rstride + q; Gy/Py are [B][Gext][Nr] (Gext = Next or 1)
    long long R;                       // rows = B * Next * Nr
    int W;                             // warps in the grid of the point kernel
    long long U;                       // partition units of the Jacobian build: rows (upr = 1) or 32-point batches
    int upr;                           // partition units per row
    int bgroup;                        // systems per work unit: 8 with the batched DMMA point kernel, else 1
    int want_jac;                      // 0: residual only (skip phase 2)
    int use_constc;                    // coefficients are constant-bank operands (DSE_FLAG_CONST_COEF, pipelined kernel)
    int tail;                          // the point kernel finishes the build itself (reduction, contraction, assembly)
    int self_h1;                       // generic point kernel computes H1 itself (small builds: all B*Gext*Nr radial rows per CTA, in shared memory)
    int tail_polls;                    // polls an owner spends looking for the subtraction points' rows (dse_tail.cuh; default TAIL_POLLS)
    double eps2, L2, inv_eps2, two_over_Lg, Lg, pG, pZ, omega, delta, gamma, e1, e2, C;
    const double *x_ext, *sx_ext, *c3x_ext, *y, *sy, *Wy, *ang, *phi_y, *phi_x, *EGy, *EZy;
    const double *t_r;                 // s(y_q) of the radial nodes (clamped to [-1, 1]), same layout as y
    const double *geom;                // geometry cache [Next*Nr*Ntpad][4] or nullptr
    // arguments of one build (set per launch)
    const double *c, *bc;              // [B][2N] coefficients (a then b), [B][2] boundary values
    double *J, *F;                     // outputs
    // per-build workspace
    double *coefP;                     // [B][Npad][2]  (a_j, b_j), j = 0 pre-halved, zero padded       (prep_kernel)
    double *Gy, *Py;                   // [B][Gext][Nr]                                                  (prep_kernel)
    double *invG, *invZ;               // [B][N]   1/G(x_i), 1/Z(x_i)                                   (prep_kernel)
    double *Apart;                     // [B*Next][Nr][4]   sum_k (u_a, u_b, v, wQ+wM)
    double *AHead;                     // same shape: partial sums of rows whose angular batches span two warps (else 0)
    double *Spart;                     // [W + B*Next] slots (dse_tail.cuh: 6 Npad + 2 doubles; batched kernel: [8][3][Npad])
    double *Rz;                        // [B*Next][3][Npad]  A . Phi_y                                   (batched builds)
    double *Dg;                        // [B*Next][4][Npad]  dPiZ/da, dPiZ/db, dPiG/da, dPiG/db          (fused tail)
    double *PiInv;                     // [B*Next][4]        Pi_G, Pi_Z, 1/G(x_e), 1/Z(x_e)              (fused tail)
    unsigned *cnt;                     // [B*Next] arrival counters of the fused tail, [B] completed external points
    unsigned *done;
    unsigned *rdy;                     // [B] subtraction points (x_Z, x_G) whose derivative rows are written
    unsigned *pend;                    // [B][(Next + 31) / 32] bit e: rows of collocation point e are left to the finishing CTA
    const int *tail_cta;               // [grid][2]   first, last external point index a CTA works on (fused tail)
    const int *tail_bi;                // [B*Next][2] first, last warp that works on an external point
};

struct PointKernelConfig {
    int grid, block, smem, regs, ctas_per_sm, sms;       // Jacobian build (defines KParams::W and the partial slots)
    int res_grid, res_block, res_smem;                   // residual-only build (no partials)
    int pipelined;                                       // Jacobian build uses the software-pipelined kernel (2: 512-thread build)
    int batched;                                         // Jacobian build uses the batched DMMA kernel (8 systems per warp)
};

// launchers; each returns the number of kernels launched or <0 on error
// ev0/ev1: optional cudaEvent_t pair recorded around the point kernel (nullptr = no timing)
int launch_build(const KParams &k, const PointKernelConfig &cfg, const double *c_dev, const double *bc_dev,
                 double *J_dev, double *F_dev, void *stream, void *ev0 = nullptr, void *ev1 = nullptr);
int launch_point(const KParams &k, const PointKernelConfig &cfg, void *stream);
int query_point_kernel(const KParams &k, PointKernelConfig &cfg);
bool constc_shape_ok(const KParams &k);     // shapes that can read the coefficients from the constant bank
bool const_slot_acquire();                  // DSE_FLAG_CONST_COEF: the library's one __constant__ coefficient slot
void const_slot_release();
// batched DMMA point kernel (dse_point_batched.cu): eligibility, launch configuration, launch
bool batched_eligible(const KParams &k);
int query_point_batched(const KParams &k, PointKernelConfig &cfg);
int launch_point_batched(const KParams &k, const PointKernelConfig &cfg, void *stream);
int launch_fd_perturb(int n2, int B, const double *c, double *c_tmp, int j, double sign, double eps_rel, void *stream);
int launch_fd_column(int n2, int B, const double *c, const double *Fp, const double *Fm, double *J, int j, double eps_rel,
                     void *stream);
int launch_geometry(const KParams &k, double *geom, void *stream);
// H9 (dse_lu.cu): n <= 128 one CTA, matrix in registers; 128 < n <= 256 a cluster of 4 CTAs (needs `scratch`)
int phase_stamps_point(long long *out_host, int max_words);   // -DDSE_PHASE_TIMING builds: words copied (else 0) or < 0
int phase_stamps_lu(long long *out_host, int max_words);
int lu_configure(int n);          // opt-in attributes of the kernel that serves n, on the current device
int launch_lu(int n, int n_sys, const double *A, const double *b, double *x, double *c_inout, double rho,
              double *stats, double *scratch, void *stream);
size_t lu_scratch_doubles(int n);
// dse_solve.cu: the Newton iteration as a CUDA graph with a WHILE node (dse_newton_solve)
struct SolveGraph;
int solve_graph_create(const KParams &k, const PointKernelConfig &cfg, double *c, const double *bc, double *J, double *F,
                       double *delta, double *stats, double *lu_scratch, double *ctl, double *info, SolveGraph **out);
void solve_graph_destroy(SolveGraph *g);
int launch_solve(SolveGraph *g, double rho, double cap, double tol, int max_iter, void *stream);
int launch_gauss_legendre(int n, double *x, double *w, double *work, void *stream);
int launch_schwinger(const KParams &k, const double *c, int n, double p2_min, double p2_max, const double *t, int n_t,
                     double *out, double *work, void *stream);
int launch_dressing(const KParams &k, const double *c, int n_x, const double *x, double alpha_mu, double *lnG, double *lnZ,
                    double *alpha, void *stream);
int launch_probe(int kind, int blocks, int iters, double *sink, void *stream);

const char *last_error_text();
void set_error_text(const char *s);
int cuda_fail(int /*cudaError_t*/ e, const char *what);     // records the text, returns DSE_ECUDA

}  // namespace dse

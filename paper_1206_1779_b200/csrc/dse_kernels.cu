// dse_kernels.cu -- sm_100a kernels for the residual + analytic Newton matrix of the ghost/gluon DSEs.
//
// Launch sequences of one build (all on the caller's stream, no host sync, no data atomics):
//   Jacobian build, full-warp angular batches, compile-time chunk count (dse_point.cu, point_kernel_pipe):
//       ONE kernel -- H1 in its prologue, H2-H6 in its body, H7 + H8 in its tail (dse_tail.cuh)
//       (DSE_FLAG_CONST_COEF: preceded by two in-stream copies of c into the constant bank)
//   Jacobian build, other single-system shapes:   prep_kernel (H1) -> point_kernel (H2-H6 + the same tail)
//   batched Jacobian build (>= 8 systems, tensor path):
//       prep_kernel -> point_kernel_batched -> gemm_kernel (H7, DMMA) | contract_split_kernel -> assemble_kernel (H8)
//   residual only:                                 prep_kernel -> point kernel (no phase 2) -> assemble_kernel
// Equation numbers refer to PAPER.md (arXiv:1206.1779); see include/dse.h and DESIGN.md.
#include <cuda_runtime.h>

#include <cstdio>

#include "dse_device.cuh"

namespace dse {

namespace {

// ---------------------------------------------------------------------------------------------
// H1: per system b: (a_j, b_j) pairs with the j = 0 coefficient pre-halved (phi_0 = 1/2, eq.(23),(24)),
// G(y_q) = exp(ln G), P(y_q) = G^{e1} Z^{e2} (eq.(3),(9)), 1/G(x_i), 1/Z(x_i).
__global__ void __launch_bounds__(256) prep_kernel(const KParams P, const double *__restrict__ c)
{
    // grid (tiles, B); one WARP per fixed point (y_q or x_i), lanes over j, fixed xor-tree reduction
    pdl_trigger();
    const int b = blockIdx.y;
    const int lane = threadIdx.x & 31;
    const int item = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const double *cb = c + (size_t)b * 2 * P.N;
    if (blockIdx.x == 0) {
        for (int j = threadIdx.x; j < P.Npad; j += blockDim.x) {
            double a = 0.0, bb = 0.0;
            if (j < P.N) { a = cb[j]; bb = cb[P.N + j]; }
            if (j == 0) { a *= 0.5; bb *= 0.5; }
            P.coefP[((size_t)b * P.Npad + j) * 2 + 0] = a;
            P.coefP[((size_t)b * P.Npad + j) * 2 + 1] = bb;
        }
    }
    const int NG = P.Gext * P.Nr;                        // fixed points y_{e,q} (split rule) or y_q (shared rule)
    if (item >= NG + P.N) return;
    const bool isy = item < NG;
    const double *phi = isy ? P.phi_y + (size_t)item * P.Npad : P.phi_x + (size_t)(item - NG) * P.Npad;
    double lnZ = 0.0, lnG = 0.0;
    for (int j = lane; j < P.N; j += 32) {       // phi_0 = 1/2 is in the table
        const double f = phi[j];
        lnZ = fma(cb[j], f, lnZ);
        lnG = fma(cb[P.N + j], f, lnG);
    }
    for (int o = 16; o > 0; o >>= 1) {
        lnZ += __shfl_xor_sync(FULL, lnZ, o);
        lnG += __shfl_xor_sync(FULL, lnG, o);
    }
    if (lane == 0) {
        if (isy) {
            lnG += P.EGy[item]; lnZ += P.EZy[item];          // power-law continuation below eps2 (infrared piece)
            P.Gy[(size_t)b * NG + item] = exp(lnG);
            P.Py[(size_t)b * NG + item] = exp(P.e1 * lnG + P.e2 * lnZ);
        } else {
            P.invG[(size_t)b * P.N + (item - NG)] = exp(-lnG);
            P.invZ[(size_t)b * P.N + (item - NG)] = exp(-lnZ);
        }
    }
}

// Geometry cache builder (DSE_FLAG_GEOMETRY_CACHE): one thread per point, geom[(e*Nr+q)*Ntpad + k][4] = (s_raw | 2 + t, gv, gq, gm).
__global__ void geometry_kernel(const KParams P, double *__restrict__ geom)
{
    const long long n = (long long)P.Next * P.Nr * P.Ntpad;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        const int k = (int)(t % P.Ntpad);
        const long long eq = t / P.Ntpad;
        const int q = (int)(eq % P.Nr), e = (int)(eq / P.Nr);
        const double x = P.x_ext[e], sx = P.sx_ext[e], c3x = P.c3x_ext[e];
        const int rq = e * P.rstride + q;
        const double y = P.y[rq], sy = P.sy[rq], Wq = P.Wy[rq];
        RowConst rc;
        const double d = (x - y) / (sx + sy);
        rc.d2 = d * d; rc.sxy = sx * sy; rc.rv = -P.C * Wq * y; rc.rq = c3x * Wq; rc.rm = c3x * Wq * y;
        double a[6];
        for (int m = 0; m < 6; ++m) a[m] = P.ang[(size_t)k * 6 + m];
        double sraw, gv, gq, gm;
        point_geometry(rc, a, P.inv_eps2, P.two_over_Lg, sraw, gv, gq, gm);
        // z > L2: the argument is clamped to 1 and only t = ln[1 + omega ln(z/L2)] of eq.(18),(19) is needed -- it does not
        // depend on the coefficients either, so the record carries 2 + t in place of s_raw (the kernels take t = s_raw - 2)
        if (sraw > 1.0) sraw = 2.0 + log(fma(P.omega, (sraw - 1.0) * (0.5 * P.Lg), 1.0));
        double4 o = make_double4(sraw, gv, gq, gm);
        reinterpret_cast<double4 *>(geom)[t] = o;
    }
}

// ---------------------------------------------------------------------------------------------
// H7: Rz[b,e,stream][j] = sum_q A_stream[b,e,q] phi_j(t_q): the z-independent part of the Jacobian,
// a dense [3 N_ext x N_r] . [N_r x N] contraction per system, on the fp64 tensor path
// (mma.sync.aligned.m8n8k4 f64 -> DMMA).  One CTA per (8 external points, 8 values of j, system); its
// warps split K = N_r; each lane loads one 32-byte row-sum record (all three streams at once), so one
// k-step feeds three MMAs; the partial tiles are combined in warp order (deterministic).
// (batched builds only: single-system builds contract in the point kernel's tail.)  4 warps and NTG = 4 n-tiles
// (8 values of j each) per CTA: every row-sum record is read once per 32 values of j.
constexpr int GEMM_WARPS = 4, NTG = 4;
__global__ void __launch_bounds__(GEMM_WARPS * 32) gemm_kernel(const KParams P)
{
    __shared__ double s_c[GEMM_WARPS][3][32][2];
    pdl_trigger();
    pdl_wait();                                              // row sums of the point kernel
    const int lane = threadIdx.x & 31, wk = threadIdx.x >> 5, nwarps = blockDim.x >> 5;   // 3 <= nwarps <= GEMM_WARPS
    const int e0 = blockIdx.x * 8, n0 = blockIdx.y * 8 * NTG, b = blockIdx.z;
    const int ae = e0 + (lane >> 2), ak = lane & 3;          // A fragment: row = lane/4 (external point), col = lane%4 (q)
    const int bk = lane & 3, bn = n0 + (lane >> 2);          // B fragment: row = lane%4 (q), col = lane/4 (j)
    const bool arow_ok = ae < P.Next;
    const size_t rowbase = ((size_t)b * P.Next + (arow_ok ? ae : 0)) * P.Nr;
    const double4 *Arow = reinterpret_cast<const double4 *>(P.Apart) + rowbase;
    const double4 *Hrow = reinterpret_cast<const double4 *>(P.AHead) + rowbase;
    const int ksteps = (P.Nr + 3) / 4, per = (ksteps + nwarps - 1) / nwarps;
    const int ks0 = wk * per, ks1 = min(ksteps, ks0 + per);
    double c[NTG][3][2];
#pragma unroll
    for (int nt = 0; nt < NTG; ++nt)
#pragma unroll
        for (int st = 0; st < 3; ++st) c[nt][st][0] = c[nt][st][1] = 0.0;
#pragma unroll 2
    for (int ks = ks0; ks < ks1; ++ks) {
        const int qa = ks * 4 + ak, qb = ks * 4 + bk;
        double4 a = make_double4(0.0, 0.0, 0.0, 0.0);
        if (arow_ok && qa < P.Nr) {
            const double4 a1 = Arow[qa], a2 = Hrow[qa];
            a = make_double4(a1.x + a2.x, a1.y + a2.y, a1.z + a2.z, 0.0);
        }
#pragma unroll
        for (int nt = 0; nt < NTG; ++nt) {
            const double bb = (qb < P.Nr && bn + 8 * nt < P.Npad) ? P.phi_y[(size_t)qb * P.Npad + bn + 8 * nt] : 0.0;
            asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                         : "+d"(c[nt][0][0]), "+d"(c[nt][0][1]) : "d"(a.x), "d"(bb));
            asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                         : "+d"(c[nt][1][0]), "+d"(c[nt][1][1]) : "d"(a.y), "d"(bb));
            asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                         : "+d"(c[nt][2][0]), "+d"(c[nt][2][1]) : "d"(a.z), "d"(bb));
        }
    }
#pragma unroll
    for (int nt = 0; nt < NTG; ++nt) {
        if (nt > 0) __syncthreads();                         // the previous tile's partials have been combined
#pragma unroll
        for (int st = 0; st < 3; ++st) { s_c[wk][st][lane][0] = c[nt][st][0]; s_c[wk][st][lane][1] = c[nt][st][1]; }
        __syncthreads();
        if (wk < 3) {                                        // warp st combines stream st
            const int st = wk;
            double r0 = 0.0, r1 = 0.0;
            for (int w2 = 0; w2 < nwarps; ++w2) { r0 += s_c[w2][st][lane][0]; r1 += s_c[w2][st][lane][1]; }
            const int ce = e0 + (lane >> 2), cn = n0 + 8 * nt + 2 * (lane & 3);     // C fragment: row = lane/4, cols 2(lane%4), +1
            if (ce < P.Next && cn < P.Npad) {
                double *out = P.Rz + (((size_t)b * P.Next + ce) * 3 + st) * P.Npad;
                out[cn] = r0;
                out[cn + 1] = r1;
            }
        }
    }
}

// H7 with the split radial rule (DSE_FLAG_RADIAL_SPLIT): phi_j(s(y_{e,q})) depends on the external point, so the
// contraction is a batch of [3 x N_r].[N_r x N] products, one per (system, external point): one warp each, lanes
// over j, plain FMAs in ascending q (a 3-row operand cannot fill a tensor-core tile).
__global__ void __launch_bounds__(128) contract_split_kernel(const KParams P)
{
    const int e = blockIdx.x, b = blockIdx.y;
    pdl_trigger();
    pdl_wait();                                              // row sums of the point kernel
    const size_t rowbase = ((size_t)b * P.Next + e) * P.Nr;
    const double4 *A = reinterpret_cast<const double4 *>(P.Apart) + rowbase;
    const double4 *H = reinterpret_cast<const double4 *>(P.AHead) + rowbase;
    const double *Phi = P.phi_y + (size_t)e * P.rstride * P.Npad;
    for (int j = threadIdx.x; j < P.Npad; j += blockDim.x) {
        double ra = 0.0, rb = 0.0, rv = 0.0;
        for (int q = 0; q < P.Nr; ++q) {
            const double4 a = A[q], h = H[q];
            const double f = Phi[(size_t)q * P.Npad + j];
            ra = fma(a.x + h.x, f, ra); rb = fma(a.y + h.y, f, rb); rv = fma(a.z + h.z, f, rv);
        }
        double *out = P.Rz + ((size_t)b * P.Next + e) * 3 * P.Npad;
        out[j] = ra; out[P.Npad + j] = rb; out[2 * P.Npad + j] = rv;
    }
}

// ---------------------------------------------------------------------------------------------
// H8: one CTA per (system b, collocation index i).  Sums the per-warp partials of the external points
// e in {i, x_Z, x_G} in a fixed order, adds the z-independent part, subtracts the MOM rows
// (eq.(14),(15)), adds the local terms -phi_j(s_i)/Z(x_i), -phi_j(s_i)/G(x_i), and writes
//   F = (z(x_i); g(x_i))  eq.(29),(30),   J = [[dz/da, dz/db],[dg/da, dg/db]]  eq.(35),(36).
constexpr int ASM_THREADS = 512;

// partial sum over a contiguous part of the slot range of external point bi (ascending warp order)
__device__ __forceinline__ void reduce_part(const KParams &P, long long bi, int j, int part, int parts, double &Sa,
                                            double &Sb, double &Sv)
{
    // P.bgroup systems share one work unit (batched DMMA kernel: 8, else 1): the partition runs over the group-level
    // index big = (b / bgroup) * Next + e, and a slot holds bgroup partials
    const long long b_sys = bi / P.Next, e = bi - b_sys * P.Next;
    const long long big = (b_sys / P.bgroup) * P.Next + e;
    const int m = (int)(b_sys % P.bgroup);
    const long long rf = big * P.Nr * P.upr, rl = rf + (long long)P.Nr * P.upr - 1;     // first/last partition unit of big
    const long long wf = ((rf + 1) * P.W - 1) / P.U, wl = ((rl + 1) * P.W - 1) / P.U;
    const long long n = wl - wf + 1, per = (n + parts - 1) / parts;
    const long long w0 = wf + part * per, w1 = min(wl + 1, w0 + per);
    double a = 0.0, b = 0.0, v = 0.0;
#pragma unroll 4
    for (long long w = w0; w < w1; ++w) {
        const double *sp = P.Spart + ((size_t)(w + big) * P.bgroup + m) * 3 * P.Npad;
        a += __ldg(sp + j); b += __ldg(sp + P.Npad + j); v += __ldg(sp + 2 * P.Npad + j);
    }
    Sa = a; Sb = b; Sv = v;
}

// The derivative rows' z-independent part comes from Rz (gemm_kernel / contract_split_kernel).  Used by the batched builds
// and, with J == nullptr, by every residual-only build.
__global__ void __launch_bounds__(ASM_THREADS) assemble_kernel(const KParams P, const double *__restrict__ bc,
                                                               double *__restrict__ J, double *__restrict__ F)
{
    const int i = blockIdx.x, b = blockIdx.y;
    const int N = P.N, nthr = blockDim.x;      // 128 <= nthr <= ASM_THREADS, a multiple of 32 and of PJ
    const long long bi_i = (long long)b * P.Next + i, bi_Z = (long long)b * P.Next + P.iZ,
                    bi_G = (long long)b * P.Next + P.iG;
    __shared__ double s_pw[ASM_THREADS / 32][3][2];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    pdl_trigger();
    pdl_wait();                                              // partials, row sums, A.Phi of the kernels before
    // All global loads of the CTA (row sums for Pi, partial slots, the fused contraction) are issued before its single
    // barrier, so their latencies overlap; the combination steps after the barrier read shared memory only.
    const int npi = (P.iG != P.iZ) ? 3 : 2;
    {   // Pi_G, Pi_Z at e = i, x_Z, x_G: all threads stride over q, per-warp partials in fixed order
        for (int pt = 0; pt < npi; ++pt) {
            const long long bi = pt == 0 ? bi_i : (pt == 1 ? bi_Z : bi_G);
            double pg = 0.0, pz = 0.0;
            for (int q = threadIdx.x; q < P.Nr; q += nthr) {
                // (read-only loads: the compiler may hoist them over the shared-memory stores of the other stages)
                const double2 a = __ldg(reinterpret_cast<const double2 *>(P.Apart) + ((size_t)bi * P.Nr + q) * 2 + 1);
                const double2 hh = __ldg(reinterpret_cast<const double2 *>(P.AHead) + ((size_t)bi * P.Nr + q) * 2 + 1);
                pg += a.x + hh.x; pz += a.y + hh.y;
            }
            for (int o = 16; o > 0; o >>= 1) {
                pg += __shfl_xor_sync(FULL, pg, o);
                pz += __shfl_xor_sync(FULL, pz, o);
            }
            if (lane == 0) { s_pw[warp][pt][0] = pg; s_pw[warp][pt][1] = pz; }
        }
    }
    const double invZ = P.invZ[(size_t)b * N + i], invG = P.invG[(size_t)b * N + i];
    if (J == nullptr) {                                          // residual only
        __syncthreads();
        if (threadIdx.x == 0) {
            double pi[3][2];
            for (int pt = 0; pt < npi; ++pt)
                for (int cmp = 0; cmp < 2; ++cmp) {
                    double t = 0.0;
                    for (int w2 = 0; w2 < nthr / 32; ++w2) t += s_pw[w2][pt][cmp];
                    pi[pt][cmp] = t;
                }
            if (npi == 2) { pi[2][0] = pi[1][0]; pi[2][1] = pi[1][1]; }      // x_G == x_Z
            const double gG = bc[2 * b + 0], gZ = bc[2 * b + 1];
            F[(size_t)b * 2 * N + i] = invZ - gZ - pi[0][1] + pi[1][1];
            F[(size_t)b * 2 * N + N + i] = invG - gG - pi[0][0] + pi[2][0];
        }
        return;
    }
    // threads = (part, j): each sums a contiguous part of the slot range; parts are combined in order
    __shared__ double s_part[3][3][ASM_THREADS];
    int PJ = 8;
    while (PJ < N) PJ <<= 1;
    const int parts = nthr / PJ, part = threadIdx.x / PJ, j = threadIdx.x - part * PJ;
    const int npt = (P.iG != P.iZ) ? 3 : 2;
    if (j < N) {
        for (int pt = 0; pt < npt; ++pt) {
            const long long bi = pt == 0 ? bi_i : (pt == 1 ? bi_Z : bi_G);
            double a, bb, v;
            reduce_part(P, bi, j, part, parts, a, bb, v);
            s_part[pt][0][threadIdx.x] = a; s_part[pt][1][threadIdx.x] = bb; s_part[pt][2][threadIdx.x] = v;
        }
    }
    __syncthreads();
    if (threadIdx.x == nthr - 1) {                               // F (one thread; the J threads are the first ones)
        double pi[3][2];
        for (int pt = 0; pt < npi; ++pt)
            for (int cmp = 0; cmp < 2; ++cmp) {
                double t = 0.0;
                for (int w2 = 0; w2 < nthr / 32; ++w2) t += s_pw[w2][pt][cmp];
                pi[pt][cmp] = t;
            }
        if (npi == 2) { pi[2][0] = pi[1][0]; pi[2][1] = pi[1][1]; }          // x_G == x_Z
        const double gG = bc[2 * b + 0], gZ = bc[2 * b + 1];
        F[(size_t)b * 2 * N + i] = invZ - gZ - pi[0][1] + pi[1][1];
        F[(size_t)b * 2 * N + N + i] = invG - gG - pi[0][0] + pi[2][0];
    }
    if (part == 0 && j < N) {
        double S[3][3];
        for (int pt = 0; pt < npt; ++pt)
            for (int st = 0; st < 3; ++st) {
                double t = 0.0;
                for (int p2 = 0; p2 < parts; ++p2) t += s_part[pt][st][p2 * PJ + j];
                S[pt][st] = (j == 0) ? 0.5 * t : t;       // the kernel accumulates with T_0 = 1; phi_0 = 1/2
            }
        if (npt == 2) { S[2][0] = S[1][0]; S[2][1] = S[1][1]; S[2][2] = S[1][2]; }
        double R[6];                                             // R_a, R_b, R_v at x_i; R_a, R_b at x_Z; R_v at x_G
        {
            const double *Ri = P.Rz + (size_t)bi_i * 3 * P.Npad, *RZ = P.Rz + (size_t)bi_Z * 3 * P.Npad,
                         *RG = P.Rz + (size_t)bi_G * 3 * P.Npad;
            R[0] = Ri[j]; R[1] = Ri[P.Npad + j]; R[2] = Ri[2 * P.Npad + j];
            R[3] = RZ[j]; R[4] = RZ[P.Npad + j]; R[5] = RG[2 * P.Npad + j];
        }
        const double phi = P.phi_x[(size_t)i * P.Npad + j];
        // dPi_Z/da = Sa + Ra, dPi_Z/db = Sb + Rb, dPi_G/da = Sv, dPi_G/db = Rv
        const double dZa_i = S[0][0] + R[0], dZb_i = S[0][1] + R[1], dGa_i = S[0][2], dGb_i = R[2];
        const double dZa_s = S[1][0] + R[3], dZb_s = S[1][1] + R[4];
        const double dGa_s = S[2][2], dGb_s = R[5];
        double *Jb = J + (size_t)b * 4 * N * N;
        Jb[(size_t)i * 2 * N + j] = -phi * invZ - dZa_i + dZa_s;
        Jb[(size_t)i * 2 * N + N + j] = -dZb_i + dZb_s;
        Jb[(size_t)(N + i) * 2 * N + j] = -dGa_i + dGa_s;
        Jb[(size_t)(N + i) * 2 * N + N + j] = -phi * invG - dGb_i + dGb_s;
    }
}

// ---------------------------------------------------------------------------------------------
// Finite-difference self-check (eq.(38),(39)): c_tmp = c with c_j -> c_j + sign * h_j;  J[:, j] = (F+ - F-)/(2 h_j)
__device__ __forceinline__ double fd_step(double cj, double eps_rel) { return eps_rel * fmax(1.0, fabs(cj)); }

__global__ void fd_perturb_kernel(int n2, const double *__restrict__ c, double *__restrict__ c_tmp, int j, double sign,
                                  double eps_rel)
{
    const int b = blockIdx.x;
    for (int i = threadIdx.x; i < n2; i += blockDim.x) {
        const double v = c[(size_t)b * n2 + i];
        c_tmp[(size_t)b * n2 + i] = (i == j) ? v + sign * fd_step(v, eps_rel) : v;
    }
}

__global__ void fd_column_kernel(int n2, const double *__restrict__ c, const double *__restrict__ Fp,
                                 const double *__restrict__ Fm, double *__restrict__ J, int j, double eps_rel)
{
    const int b = blockIdx.x;
    const double cj = c[(size_t)b * n2 + j];
    // the step actually taken, as representable numbers: (c_j + h) - (c_j - h)
    const double h2 = (cj + fd_step(cj, eps_rel)) - (cj - fd_step(cj, eps_rel));
    for (int i = threadIdx.x; i < n2; i += blockDim.x)
        J[((size_t)b * n2 + i) * n2 + j] = (Fp[(size_t)b * n2 + i] - Fm[(size_t)b * n2 + i]) / h2;
}

thread_local char g_err[256] = "";

}  // namespace

const char *last_error_text() { return g_err; }
void set_error_text(const char *s) { snprintf(g_err, sizeof(g_err), "%s", s); }
int cuda_fail(int e, const char *what)
{
    snprintf(g_err, sizeof(g_err), "%s: %s", what, cudaGetErrorString((cudaError_t)e));
    return DSE_ECUDA;
}

int launch_geometry(const KParams &k, double *geom, void *stream)
{
    const long long n = (long long)k.Next * k.Nr * k.Ntpad;
    int blocks = (int)((n + 255) / 256);
    if (blocks > 148 * 16) blocks = 148 * 16;
    geometry_kernel<<<blocks, 256, 0, (cudaStream_t)stream>>>(k, geom);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "geometry_kernel launch");
    return 1;
}

int launch_build(const KParams &k, const PointKernelConfig &cfg, const double *c_dev, const double *bc_dev,
                 double *J_dev, double *F_dev, void *stream, void *ev0, void *ev1)
{
    cudaStream_t s = (cudaStream_t)stream;
    KParams kk = k;
    kk.want_jac = J_dev != nullptr;
    kk.c = c_dev; kk.bc = bc_dev; kk.J = J_dev; kk.F = F_dev;
    kk.tail = kk.want_jac && !cfg.batched;               // single-system kernels finish the build themselves
    int launches = 0;
    cudaError_t e;
    const bool one_kernel = kk.tail && (cfg.pipelined || kk.self_h1);    // these kernels also do H1
    if (!one_kernel) {
        prep_kernel<<<dim3((kk.Gext * kk.Nr + kk.N + 7) / 8, kk.B), 256, 0, s>>>(kk, c_dev);
        if ((e = cudaGetLastError()) != cudaSuccess) return cuda_fail(e, "prep_kernel launch");
        ++launches;
    }
    if (ev0 && (e = cudaEventRecord((cudaEvent_t)ev0, s)) != cudaSuccess) return cuda_fail(e, "cudaEventRecord");
    int rc = launch_point(kk, cfg, stream);
    if (rc < 0) return rc;
    launches += rc;
    if (ev1 && (e = cudaEventRecord((cudaEvent_t)ev1, s)) != cudaSuccess) return cuda_fail(e, "cudaEventRecord");
    if (kk.tail) return launches;
    if (kk.want_jac) {                                   // batched build: H7 on the tensor path, or the split rule's batch
        if (kk.rstride) {
            e = launch_pdl(contract_split_kernel, dim3(kk.Next, kk.B), dim3(128), 0, s, kk);
        } else {
            dim3 gg((kk.Next + 7) / 8, (kk.Npad / 8 + NTG - 1) / NTG, kk.B);
            e = launch_pdl(gemm_kernel, gg, dim3(GEMM_WARPS * 32), 0, s, kk);
        }
        if (e != cudaSuccess) return cuda_fail(e, "contraction launch");
        ++launches;
    }
    // many systems: few slots per external point, small CTAs keep more of them resident
    e = launch_pdl(assemble_kernel, dim3(kk.N, kk.B), dim3(kk.B >= 8 ? 128 : ASM_THREADS), 0, s, kk, bc_dev, J_dev, F_dev);
    if (e != cudaSuccess) return cuda_fail(e, "assemble_kernel launch");
    ++launches;
    return launches;
}

int launch_fd_perturb(int n2, int B, const double *c, double *c_tmp, int j, double sign, double eps_rel, void *stream)
{
    fd_perturb_kernel<<<B, 128, 0, (cudaStream_t)stream>>>(n2, c, c_tmp, j, sign, eps_rel);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "fd launch");
    return 1;
}
int launch_fd_column(int n2, int B, const double *c, const double *Fp, const double *Fm, double *J, int j, double eps_rel,
                     void *stream)
{
    fd_column_kernel<<<B, 128, 0, (cudaStream_t)stream>>>(n2, c, Fp, Fm, J, j, eps_rel);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "fd launch");
    return 1;
}

}  // namespace dse

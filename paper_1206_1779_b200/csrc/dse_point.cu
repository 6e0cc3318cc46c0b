// dse_point.cu -- the hot kernel (steps H2-H6 of DESIGN.md): every quadrature point (x_e, y_q, theta_k); for a Jacobian
// build the same kernel also finishes the build (H7, H8: dse_tail.cuh), so that a build is ONE launch.
//
// Each WARP is an independent worker that owns a contiguous range of the flattened (system, external point, radial
// node, angular batch) index and walks it in batches of 32 points:
//   phase 1 (lane = point): geometry (or the cached 32 B), clamp + continuation eq.(16)-(19), the
//     T_j recurrence shared by both series ln G(z), ln Z(z) (3 FMA per j; the recurrence runs as two
//     independent stride-2 chains T_{j+2} = 2 T_2 T_j - T_{j-2} for instruction-level parallelism),
//     3 exp, the weights v, wQ, wM (H4), the running row sums (H5, A[e,q] of H7); stash
//     (2s, u_a, u_b, v) and the chunk-start pairs (T_8c, T_8c+1) in warp-private shared memory;
//   phase 2 (lane = (chunk c, point sub-lane)): restart the recurrence at j = 8c and accumulate the
//     three z-dependent Jacobian streams Sa, Sb, Sv for 8 values of j in registers.
// Accumulators are flushed as per-(warp, external point) partials and summed in a fixed order.  No CTA-level
// synchronisation between the table load and the tail, no data atomics.
//   point_kernel       any shape (run-time chunk count, angular batches narrower than a warp), residual-only builds;
//                      coefficients, G(y_q), P(y_q) from prep_kernel
//   point_kernel_pipe  full-warp angular batches, compile-time chunk count: phase 1 of batch t and phase 2 of batch
//                      t-1 in one straight-line block (software pipelining); computes G(y_q), P(y_q) itself (H1)
#include <cstdio>
#include <atomic>

#include "dse_tail.cuh"

namespace dse {


namespace {

// DSE_FLAG_CONST_COEF: the coefficients c = (a_0..a_{N-1}, b_0..b_{N-1}) of a single-system build as constant-bank operands
// of the series FMAs.  Filled by ONE in-stream device-to-device copy of the caller's c (cudaMemcpyToSymbolAsync) before the
// point kernel is launched; N is the kernel's compile-time chunk count times 8, so b_j sits at a compile-time offset.
__constant__ double c_coef[2 * DSE_MAX_NCHEB];

// Template: NCH_T = number of 8-wide Chebyshev chunks when it is a power of two (everything unrolls),
// 0 = generic run-time shape; GEOM = read the geometry cache; JAC = accumulate the Jacobian streams and (P.tail)
// finish the build in the kernel's tail; JAC = false: residual only, finished by assemble_kernel.
template <int NCH_T, bool GEOM, bool JAC>
__global__ void __launch_bounds__(POINT_THREADS, 1) point_kernel(const __grid_constant__ KParams P)
{
    constexpr bool CT = NCH_T > 0;
    extern __shared__ __align__(16) double smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, WPB = blockDim.x >> 5;
    const int NCH = CT ? NCH_T : P.NCH;
    const int SUB = CT ? 32 / NCH_T : P.SUB;
    const int ROUNDS = CT ? NCH_T : P.rounds;
    const int Npad = NCH * CJ;
    double *s_ang = smem;
    // small Jacobian builds (P.self_h1): G(y_q), P(y_q) of ALL radial rows of all systems, computed by this CTA itself (H1)
    const int NGB = (JAC && P.self_h1) ? P.B * P.Gext * P.Nr : 0;
    double *s_Gy = smem + (size_t)P.Ntpad * 6, *s_Py = s_Gy + NGB;
    double *wbase = s_Py + NGB + (size_t)warp * warp_doubles(Npad, NCH);
    double2 *s_coef = reinterpret_cast<double2 *>(wbase);
    double4 *s_pt = reinterpret_cast<double4 *>(wbase + 2 * Npad);       // 33 entries, entry 32 = 0
    double *s_T = wbase + 2 * Npad + 132;
    double2 *s_T2 = reinterpret_cast<double2 *>(s_T);
    double4 *s_gbuf = reinterpret_cast<double4 *>(wbase + 2 * Npad + stash_doubles(NCH));   // [2][32] geometry records

    for (int t = threadIdx.x; t < P.Ntpad * 6; t += blockDim.x) s_ang[t] = P.ang[t];
    if (lane == 0) s_pt[32] = make_double4(0.0, 0.0, 0.0, 0.0);
    pdl_wait();                                             // prep_kernel: coefficient pairs, G(y_q), P(y_q) (or the kernel before)
    if (NGB) {
        // H1 by the CTA itself: thread = radial row, both series ln G(y), ln Z(y) of eq.(23),(24) at s(y_q) with T_j from
        // the three-term recurrence, plus the power-law terms of the infrared piece; G = exp(ln G), P = G^{e1} Z^{e2}
        const int NG = P.Gext * P.Nr, N = P.N;
        for (int it = threadIdx.x; it < NGB; it += blockDim.x) {
            const int b = it / NG, row = it - b * NG;
            const double *ca = P.c + (size_t)b * 2 * N, *cb = ca + N;
            const double sy = __ldg(P.t_r + row), ts = 2.0 * sy;
            double T0 = 1.0, T1 = sy;
            double lnZ = 0.5 * __ldg(ca), lnG = 0.5 * __ldg(cb);                 // phi_0 = 1/2
            for (int j = 1; j < N; ++j) {
                lnZ = fma(__ldg(ca + j), T1, lnZ); lnG = fma(__ldg(cb + j), T1, lnG);
                const double T2 = fma(ts, T1, -T0);
                T0 = T1; T1 = T2;
            }
            lnG += __ldg(P.EGy + row); lnZ += __ldg(P.EZy + row);
            s_Gy[it] = exp(lnG);
            s_Py[it] = exp(P.e1 * lnG + P.e2 * lnZ);
        }
    }
    __syncthreads();

    const int Nr = P.Nr, g = P.g;
    const long long R = P.R;
    const long long w = (long long)blockIdx.x * WPB + warp;
    const long long r0 = (w * R) / P.W, r1 = ((w + 1) * R) / P.W;
    const int c_lane = lane / SUB, sub = lane - c_lane * SUB;
    const bool active2 = CT ? true : (lane < NCH * SUB);
    const int rib = lane / g, kl = lane - rib * g;          // row-in-batch and angular lane
    const double halfLg = 0.5 * P.Lg;
    const double2 *tread = s_T2 + (active2 ? c_lane : 0) * (TCH_STRIDE / 2);

    double accA[CJ], accB[CJ], accV[CJ];
#pragma unroll
    for (int m = 0; m < CJ; ++m) accA[m] = accB[m] = accV[m] = 0.0;

    const int SLOT = slot_doubles(Npad);
    auto flush = [&](long long bi) {
        double *slot = P.Spart + (size_t)(w + bi) * SLOT;
#pragma unroll
        for (int st = 0; st < 3; ++st) {
            __syncwarp();
            if (active2) {
#pragma unroll
                for (int m = 0; m < CJ; ++m)
                    s_T[sub * Npad + c_lane * CJ + m] = (st == 0 ? accA[m] : (st == 1 ? accB[m] : accV[m]));
            }
            __syncwarp();
            for (int j = lane; j < Npad; j += 32) {
                double s = 0.0;
                for (int sb = 0; sb < SUB; ++sb) s += s_T[sb * Npad + j];
                slot[st * Npad + j] = s;
            }
        }
        __syncwarp();
    };

    // Geometry cache, full-warp angular batches: the warp's batches are consecutive 1 KB records of one linear
    // stream (wrapping at a system boundary), so the next batch is prefetched with cp.async into a warp-private
    // double buffer while the current one is processed -- no registers held across the batch.
    const bool PREF = GEOM && g == 32;
    const unsigned long long gpolicy = l2_evict_first_policy();
    const size_t gtotal = (size_t)P.Next * Nr * P.Ntpad;
    const double4 *gbase = reinterpret_cast<const double4 *>(P.geom), *gend = gbase + gtotal, *gnext = gbase;
    unsigned gphase = 0;
    auto prefetch = [&](unsigned buf) {
        const unsigned dst = (unsigned)__cvta_generic_to_shared(s_gbuf + buf * 32 + lane);
        asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(gnext), "l"(gpolicy));
        asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;\n" ::"r"(dst + 16), "l"(reinterpret_cast<const char *>(gnext) + 16), "l"(gpolicy));
        asm volatile("cp.async.commit_group;\n" ::);
    };
    if (PREF && r0 < r1) {
        const long long bi0 = r0 / Nr;
        gnext = gbase + ((size_t)(bi0 % P.Next) * Nr + (size_t)(r0 - bi0 * Nr)) * P.Ntpad + lane;
        prefetch(0);
    }

    // (bi, q0, b, e) are advanced incrementally: no 64-bit divisions inside the row loop
    long long r = r0;
    long long bi = r0 / Nr;
    int q0 = (int)(r0 - bi * Nr);
    int cur_b = (int)(bi / P.Next);
    int e = (int)(bi - (long long)cur_b * P.Next);
    bool fresh = true;                                   // accumulators belong to a new external point
    bool first_row = true;                               // no row of this external point has reached the slot yet
    auto load_coef = [&](int b) {                          // (a_j, b_j) pairs of system b, j = 0 pre-halved, zero padded
        for (int j = lane; j < Npad; j += 32) {
            if (NGB) {
                const double *ca = P.c + (size_t)b * 2 * P.N;
                const double h = j == 0 ? 0.5 : 1.0;
                s_coef[j] = j < P.N ? make_double2(h * __ldg(ca + j), h * __ldg(ca + P.N + j)) : make_double2(0.0, 0.0);
            } else {
                s_coef[j] = reinterpret_cast<const double2 *>(P.coefP)[(size_t)b * Npad + j];
            }
        }
        __syncwarp();
    };
    if (r0 < r1) load_coef(cur_b);
    while (r < r1) {
        if (fresh) {
#pragma unroll
            for (int m = 0; m < CJ; ++m) accA[m] = accB[m] = accV[m] = 0.0;
            fresh = false;
            first_row = true;
        }
        const long long left = r1 - r;
        int nrow = P.rpb;
        if (left < nrow) nrow = (int)left;
        if (Nr - q0 < nrow) nrow = Nr - q0;
        const bool rowact = rib < nrow;
        const int q = q0 + (rowact ? rib : 0);

        // row constants (identical in all lanes of a row)
        const double rowmask = rowact ? 1.0 : 0.0;
        const size_t gq = ((size_t)cur_b * P.Gext + (P.rstride ? e : 0)) * Nr + q;
        const double Gy = (NGB ? s_Gy[gq] : P.Gy[gq]) * rowmask, Py = (NGB ? s_Py[gq] : P.Py[gq]) * rowmask;
        RowConst rc;
        if (!GEOM) {
            const double x = P.x_ext[e], sx = P.sx_ext[e], c3x = P.c3x_ext[e];
            const int rq = e * P.rstride + q;
            const double y = P.y[rq], sy = P.sy[rq];
            const double Wq = P.Wy[rq];
            const double d = (x - y) / (sx + sy);
            rc.d2 = d * d; rc.sxy = sx * sy; rc.rv = -P.C * Wq * y; rc.rq = c3x * Wq; rc.rm = c3x * Wq * y;
        }
        double sumA = 0.0, sumB = 0.0, sumV = 0.0, sumZ = 0.0;
        const double4 *grow = GEOM ? reinterpret_cast<const double4 *>(P.geom) + ((size_t)e * Nr + q) * P.Ntpad + kl
                                   : nullptr;

        for (int kb = 0; kb < P.Ntpad; kb += 32) {
            // ---------------- phase 1: lane = point (k = kb + kl < Ntpad: g divides Ntpad, g <= 32) ----------------
            double gv, gqv, gm, sraw;
            if (GEOM && PREF) {
                gnext += 32;                                   // next batch of this warp (possibly of the next row)
                if (gnext >= gend) gnext -= gtotal;
                prefetch(gphase ^ 1);
                asm volatile("cp.async.wait_group 1;\n" ::: "memory");     // the current batch has landed
                const double2 *gp = reinterpret_cast<const double2 *>(s_gbuf + gphase * 32 + lane);
                const double2 g0 = gp[0], g1 = gp[1];
                sraw = g0.x; gv = g0.y; gqv = g1.x; gm = g1.y;
                gphase ^= 1;
            } else if (GEOM) {
                const double2 *gp = reinterpret_cast<const double2 *>(grow + kb);   // streamed once
                const double2 g0 = __ldcs(gp), g1 = __ldcs(gp + 1);
                sraw = g0.x; gv = g0.y; gqv = g1.x; gm = g1.y;
            } else {
                point_geometry(rc, s_ang + (kb + kl) * 6, P.inv_eps2, P.two_over_Lg, sraw, gv, gqv, gm);
            }
            double s = sraw, EG = 0.0, EZ = 0.0;
            if (sraw < -1.0) {                       // z < eps2: G ~ z^pG, Z ~ z^pZ   eq.(16),(17)
                const double ell = (sraw + 1.0) * halfLg;
                EG = P.pG * ell; EZ = P.pZ * ell; s = -1.0;
            } else if (sraw > 1.0) {                 // z > L2: [omega ln(z/L2) + 1]^{delta,gamma}  eq.(18),(19)
                const double t = GEOM ? sraw - 2.0 : log(fma(P.omega, (sraw - 1.0) * halfLg, 1.0));   // (cached: the record carries 2 + t)
                EG = P.delta * t; EZ = P.gamma * t; s = 1.0;
            }
            const double ts = 2.0 * s;
            const double t2 = fma(2.0 * ts, s, -2.0);       // 2 T_2(s): stride-2 recurrence T_{j+2} = 2 T_2 T_j - T_{j-2}
            double Te = 1.0, To = s;                        // T_0, T_1
            double Tem = fma(ts, s, -1.0), Tom = s;         // T_{-2} = T_2, T_{-1} = T_1
            double lz0 = 0.0, lz1 = 0.0, lg0 = 0.0, lg1 = 0.0;
#pragma unroll
            for (int c = 0; c < NCH; ++c) {
                if (JAC) s_T2[c * (TCH_STRIDE / 2) + lane] = make_double2(Te, To);
#pragma unroll
                for (int m = 0; m < CJ; m += 4) {
                    const double2 c0 = s_coef[c * CJ + m], c1 = s_coef[c * CJ + m + 1];
                    const double2 c2 = s_coef[c * CJ + m + 2], c3 = s_coef[c * CJ + m + 3];
                    lz0 = fma(c0.x, Te, lz0); lg0 = fma(c0.y, Te, lg0);
                    lz1 = fma(c1.x, To, lz1); lg1 = fma(c1.y, To, lg1);
                    Tem = fma(t2, Te, -Tem);  Tom = fma(t2, To, -Tom);   // T_{j+2}, T_{j+3}
                    lz0 = fma(c2.x, Tem, lz0); lg0 = fma(c2.y, Tem, lg0);
                    lz1 = fma(c3.x, Tom, lz1); lg1 = fma(c3.y, Tom, lg1);
                    Te = fma(t2, Tem, -Te);   To = fma(t2, Tom, -To);    // T_{j+4}, T_{j+5}
                }
            }
            {
                const double lnZz = (lz0 + lz1) + EZ, lnGz = (lg0 + lg1) + EG;
                const double lnPz = fma(P.e1, lnGz, P.e2 * lnZz);
                double Zz, Gz, Pz;
                // |x| <= 700 for all three, tested on the high words (0x4085e000 = high word of 700.0; NaN/Inf fail)
                const int hmax = max(max(__double2hiint(lnZz) & 0x7fffffff, __double2hiint(lnGz) & 0x7fffffff),
                                     __double2hiint(lnPz) & 0x7fffffff);
                if (hmax < 0x4085e000) {
                    Zz = fast_exp(lnZz); Gz = fast_exp(lnGz); Pz = fast_exp(lnPz);
                } else {                                   // out of the fast range (or NaN): library exp
                    Zz = exp(lnZz); Gz = exp(lnGz); Pz = exp(lnPz);
                }
                const double v = gv * (Gy * Zz);              // eq.(8):  -C W y Om sin^4/z^2 G(y) Z(z)
                const double wQ = gqv * (Py * Pz);            // eq.(9):  (C/3x) W Om sin^2 Q P(y) P(z)
                const double wM = gm * (Gy * Gz);             // eq.(9):  (C/3x) W Om sin^2 M G(y) G(z)
                const double ua = P.e2 * wQ;                  // weight of d/da_j  (P ~ Z^{e2})
                const double ub = fma(P.e1, wQ, wM);          // weight of d/db_j  (P ~ G^{e1}; G(y)G(z))
                sumA += ua; sumB += ub; sumV += v; sumZ += wQ + wM;
                if (JAC) s_pt[lane] = make_double4(ts, ua, ub, v);
            }
            if (JAC) {
                __syncwarp();
                // ---------------- phase 2: lane = (chunk, point sub-lane) ----------------
#pragma unroll
                for (int rd = 0; rd < ROUNDS; ++rd) {
                    const int pt = rd * SUB + sub;
                    const int pc = CT ? pt : ((active2 && pt < 32) ? pt : 32);     // slot 32 holds zero weights
                    const double4 pw = s_pt[pc];
                    const double2 tt = tread[pc & 31];
                    double T0 = tt.x, T1 = tt.y;
                    accA[0] = fma(pw.y, T0, accA[0]); accB[0] = fma(pw.z, T0, accB[0]); accV[0] = fma(pw.w, T0, accV[0]);
                    accA[1] = fma(pw.y, T1, accA[1]); accB[1] = fma(pw.z, T1, accB[1]); accV[1] = fma(pw.w, T1, accV[1]);
#pragma unroll
                    for (int m = 2; m < CJ; ++m) {
                        const double T2 = fma(pw.x, T1, -T0);
                        accA[m] = fma(pw.y, T2, accA[m]); accB[m] = fma(pw.z, T2, accB[m]); accV[m] = fma(pw.w, T2, accV[m]);
                        T0 = T1; T1 = T2;
                    }
                }
                __syncwarp();
            } else {
                asm volatile("" ::: "memory");      // keep the coefficient loads inside the loop (no hoisting -> no spills)
            }
        }
        // H5/H7: row sums over the angular nodes (fixed xor tree), one writer per row
        for (int o = g >> 1; o > 0; o >>= 1) {
            sumA += __shfl_xor_sync(FULL, sumA, o);
            sumB += __shfl_xor_sync(FULL, sumB, o);
            sumV += __shfl_xor_sync(FULL, sumV, o);
            sumZ += __shfl_xor_sync(FULL, sumZ, o);
        }
        if (JAC && P.tail) {
            // H5 + H7 in the warp's slot of this external point, row by row (dse_tail.cuh)
            for (int rb = 0; rb < nrow; ++rb) {
                const double rA = __shfl_sync(FULL, sumA, rb * g), rB = __shfl_sync(FULL, sumB, rb * g);
                const double rV = __shfl_sync(FULL, sumV, rb * g), rZ = __shfl_sync(FULL, sumZ, rb * g);
                const double *phi = P.phi_y + ((size_t)(P.rstride ? e * P.rstride : 0) + q0 + rb) * Npad;
                slot_row_update(P.Spart + (size_t)(w + bi) * SLOT, Npad, phi, rA, rB, rV, rZ, first_row, lane);
                first_row = false;
            }
        } else if (kl == 0 && rowact) {
            reinterpret_cast<double4 *>(P.Apart)[(size_t)bi * Nr + q] = make_double4(sumA, sumB, sumV, sumZ);
            reinterpret_cast<double4 *>(P.AHead)[(size_t)bi * Nr + q] = make_double4(0.0, 0.0, 0.0, 0.0);   // rows are never split here
        }
        r += nrow;
        q0 += nrow;
        if (q0 >= Nr) {                                  // next external point (nrow never crosses this boundary)
            if (JAC) flush(bi);
            fresh = true;
            q0 = 0; ++bi; ++e;
            if (e == P.Next && r < r1) {                 // next system: stage its coefficient pairs
                e = 0; ++cur_b;
                __syncwarp();
                load_coef(cur_b);
            }
        }
    }
    if (JAC && !fresh) flush(bi);
    if (PREF) asm volatile("cp.async.wait_group 0;\n" ::: "memory");
    if (JAC && P.tail) build_tail(P, smem);              // H8 by the last-arriving CTAs (uniform over the grid)
}


// ---------------------------------------------------------------------------------------------------------
// Software-pipelined variant (compile-time chunk count, full-warp angular batches, Jacobian on):
// iteration t runs phase 1 of batch t (series, exp -- long dependent chains, little fp64 pipe pressure)
// in the SAME straight-line block as phase 2 of batch t-1 (accumulation -- independent FMAs), reading and
// writing the two halves of a double-buffered stash, so the scheduler hides the chains behind the FMAs.
// One pipeline per (warp, external point) segment: prologue = zeroed weights, epilogue = phase 2 only.
// The kernel is a whole build: H1 (the series at the radial nodes, G(y_q) and P(y_q), for windows of 32 rows at a
// time: lane = row) in front, H7 + H8 (dse_tail.cuh) behind.
constexpr int PIPE_THREADS = 384;
constexpr int GP_DOUBLES = 64;                // G(y), P(y) of a window of 32 rows

__host__ __device__ inline int pipe_warp_doubles(int Npad, int NCH, bool constc, bool geom)
{
    return (constc ? 0 : 2 * Npad) + 2 * stash_doubles(NCH) + (geom ? GBUF_DOUBLES : 0) + GP_DOUBLES;
}

// H1 for a window of up to 32 consecutive rows starting at row rb (relative to the warp's first row r0): lane r takes row
// rb + r and runs both series ln G(y), ln Z(y) of eq.(23),(24) at s(y_q) by itself, with T_j(s) from the same stride-2
// recurrence as the main loop -- no table row is read (the rows phi_j(t_q) would be 512 B per row and warp, re-read by every
// warp that touches the row: memory latency that nothing hides), no cross-lane reduction.  It adds the power-law terms of
// the infrared piece and keeps G(y) = exp(ln G), P(y) = G^{e1} Z^{e2} (eq.(3),(9)).  The coefficients come from where the
// kernel keeps them (constant bank, or the pairs of system sb in shared memory); a row of another system reads c itself.
// (Not inlined: the body of the point kernel's loop has to stay inside the SM's instruction cache.)
// (s, addZ, addG) = t_r, EZy, EGy of the lane's row (pipe_row_tables: loaded by the caller, for the first window at the very
// top of the kernel so that their cold miss overlaps the rest of the prologue).
struct RowTab { double s, addZ, addG; };
__device__ __forceinline__ RowTab pipe_row_tables(const KParams &P, int n_rows, int g0, int gmod, int lane, int rb)
{
    RowTab t = {0.0, 0.0, 0.0};
    if (rb + lane < n_rows) {
        const int gi = (int)((g0 + rb + lane) % gmod);
        t.s = __ldg(P.t_r + gi); t.addZ = __ldg(P.EZy + gi); t.addG = __ldg(P.EGy + gi);
    }
    return t;
}
template <int Npad, bool CONSTC>
__device__ __noinline__ void pipe_fill_gp(const KParams &P, long long r0, int n_rows, RowTab tab,
                                          const double2 *s_coef, int sb, double2 *s_gp, int lane, int rb)
{
    const int N = P.N;
    const int nr = n_rows - rb < 32 ? n_rows - rb : 32;
    double Gv = 0.0, Pv = 0.0;
    if (lane < nr) {
        const double s = tab.s, addZ = tab.addZ, addG = tab.addG;
        const int br = (int)((r0 + rb + lane) / ((long long)P.Next * P.Nr));
        const double *ca = P.c + (size_t)br * 2 * N, *cb = ca + N;
        const bool own = CONSTC || br == sb;
        auto coef = [&](int j) -> double2 {                  // (a_j, b_j); zero beyond N
            if (CONSTC) return make_double2(c_coef[j], c_coef[Npad + j]);
            if (own) return s_coef[j];
            return j < N ? make_double2(__ldg(ca + j), __ldg(cb + j)) : make_double2(0.0, 0.0);
        };
        const double ts = 2.0 * s, t2 = fma(2.0 * ts, s, -2.0);          // T_{j+2} = 2 T_2 T_j - T_{j-2}
        double Te = 1.0, To = s, Tem = fma(ts, s, -1.0), Tom = s;
        double lz0, lz1 = 0.0, lg0, lg1 = 0.0;
        { const double2 c0 = coef(0); lz0 = 0.5 * c0.x; lg0 = 0.5 * c0.y; }      // phi_0 = 1/2
#pragma unroll 2
        for (int j0 = 0; j0 < Npad; j0 += 4) {
            const double2 c0 = coef(j0), c1 = coef(j0 + 1), c2 = coef(j0 + 2), c3 = coef(j0 + 3);
            if (j0 > 0) { lz0 = fma(c0.x, Te, lz0); lg0 = fma(c0.y, Te, lg0); }
            lz1 = fma(c1.x, To, lz1); lg1 = fma(c1.y, To, lg1);
            Tem = fma(t2, Te, -Tem);  Tom = fma(t2, To, -Tom);
            lz0 = fma(c2.x, Tem, lz0); lg0 = fma(c2.y, Tem, lg0);
            lz1 = fma(c3.x, Tom, lz1); lg1 = fma(c3.y, Tom, lg1);
            Te = fma(t2, Tem, -Te);   To = fma(t2, Tom, -To);
        }
        const double lnZ = (lz0 + lz1) + addZ, lnG = (lg0 + lg1) + addG;
        Gv = exp(lnG);
        Pv = exp(P.e1 * lnG + P.e2 * lnZ);
    }
    __syncwarp();
    s_gp[lane] = make_double2(Gv, Pv);
    __syncwarp();
}

// H5 + H7 of the rows [qa, qb] of external point bi = (b, e) that this warp has walked, at the end of the segment: the
// angular sums come back from the warp's own row records (the last row's from AHead if the warp stopped inside it), several
// rows of loads in flight; R[j] = sum_q A[q] phi_j(t_q), Pi = sum_q; written once into the warp's slot (dse_tail.cuh).
template <int Npad>
__device__ __noinline__ void pipe_contract(const KParams &P, double *slot, int bi, int e, int qa, int qb, bool last_partial, int lane)
{
    constexpr int JL = (Npad + 31) / 32;
    const int Nr = P.Nr;
    double R[JL][3], pg = 0.0, pz = 0.0;
#pragma unroll
    for (int u = 0; u < JL; ++u) R[u][0] = R[u][1] = R[u][2] = 0.0;
    const double *phib = P.phi_y + (size_t)(P.rstride ? e * P.rstride : 0) * Npad;
    const double *A = P.Apart + (size_t)bi * Nr * 4, *H = P.AHead + (size_t)bi * Nr * 4;
    __syncwarp();                                      // the records were written by other lanes of this warp
#pragma unroll 1
    constexpr int RT = JL <= 2 ? 6 : 3;                // rows per round trip (register budget)
    for (int q0 = qa; q0 <= qb; q0 += RT) {
        double4 rec[RT];
        double f[RT][JL];
#pragma unroll
        for (int v = 0; v < RT; ++v) {
            const int q = q0 + v;
            const bool ok = q <= qb;
            const double *src = ((ok && q == qb && last_partial) ? H : A) + (size_t)(ok ? q : qa) * 4;
            const double2 s0 = reinterpret_cast<const double2 *>(src)[0], s1 = reinterpret_cast<const double2 *>(src)[1];
            rec[v] = ok ? make_double4(s0.x, s0.y, s1.x, s1.y) : make_double4(0.0, 0.0, 0.0, 0.0);
#pragma unroll
            for (int u = 0; u < JL; ++u) {
                const int j = 32 * u + lane;
                f[v][u] = (ok && j < Npad) ? __ldg(phib + (size_t)q * Npad + j) : 0.0;
            }
        }
#pragma unroll
        for (int v = 0; v < RT; ++v) {
#pragma unroll
            for (int u = 0; u < JL; ++u) {
                R[u][0] = fma(rec[v].x, f[v][u], R[u][0]); R[u][1] = fma(rec[v].y, f[v][u], R[u][1]); R[u][2] = fma(rec[v].z, f[v][u], R[u][2]);
            }
            pg += rec[v].z; pz += rec[v].w;
        }
    }
#pragma unroll
    for (int u = 0; u < JL; ++u) {
        const int j = 32 * u + lane;
        if (j < Npad) { slot[3 * Npad + j] = R[u][0]; slot[4 * Npad + j] = R[u][1]; slot[5 * Npad + j] = R[u][2]; }
    }
    if (lane == 0) { slot[6 * Npad] = pg; slot[6 * Npad + 1] = pz; }
}

// THR: threads per CTA the register budget is compiled for (384: ~160 registers; 512: 128 registers, 16 warps per SM --
// 2 % faster on large problems, slower on small ones)
template <int NCH_T, bool GEOM, bool CONSTC, int THR = PIPE_THREADS>
__global__ void __launch_bounds__(THR, 1) point_kernel_pipe(const __grid_constant__ KParams P)
{
    // lanes = (chunk of 8 j, point sub-lane); chunk counts that do not divide 32 leave 32 - NCH * SUB lanes idle in
    // phase 2 and read the zero-weight stash slot 32 for the points past the batch
    constexpr int NCH = NCH_T, SUB = 32 / NCH_T, ROUNDS = (32 + SUB - 1) / SUB, Npad = NCH_T * CJ;
    constexpr bool EXACT = NCH * SUB == 32 && ROUNDS * SUB == 32;
    constexpr int SLOT = 6 * Npad + 2;                                      // = slot_doubles(Npad)
    extern __shared__ __align__(16) double smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, WPB = blockDim.x >> 5;
#ifdef DSE_PHASE_TIMING
    if (lane == 0) for (int z = 0; z < PHASE_SLOTS; ++z) phase_rec()[z] = 0;
#endif
    PHASE_STAMP(0);
    const int STASH = stash_doubles(NCH);
    const int WD = pipe_warp_doubles(Npad, NCH, CONSTC, GEOM);
    double *s_ang = smem;
    double *s_exp = smem + (size_t)P.Ntpad * 6;                              // 2^(k/64): table of fast_exp_tab
    double *s_log = s_exp + EXPTAB_DOUBLES;                                  // tables of fast_log_tab (geometry in registers only)
    double *wbase = s_log + (GEOM ? 0 : LOGTAB_DOUBLES) + (size_t)warp * WD;
    double2 *s_coef = reinterpret_cast<double2 *>(wbase);
    double *s_stash = wbase + (CONSTC ? 0 : 2 * Npad);                       // [2][STASH]: pt (33 x 4) then T
    double2 *s_gp = reinterpret_cast<double2 *>(s_stash + 2 * STASH);       // [32] (G(y), P(y)) of a window of rows
    double4 *s_gbuf = reinterpret_cast<double4 *>(s_stash + 2 * STASH + GP_DOUBLES);     // [2][32] geometry records
    const int Nr = P.Nr, BPR = P.Ntpad >> 5;                                 // batches per row
    // work is partitioned in 32-point batches (P.U = rows * BPR): balanced to +-1 batch over all warps; a row whose
    // batches span two warps has one angular-sum record from each (AHead: the head, Apart: the rest)
    const long long w = (long long)blockIdx.x * WPB + warp;
    const long long t0 = (w * P.U) / P.W, t1 = ((w + 1) * P.U) / P.W;
    const long long r0 = t0 / BPR;
    const int n_rows = t0 < t1 ? (int)((t1 - 1) / BPR + 1 - r0) : 0;        // rows r0 + [0, n_rows) are touched by this warp
    const int gmod = P.rstride ? P.Next * Nr : Nr;                           // rows of the radial tables
    const int g0 = (int)(r0 % gmod);
    // Everything the warp needs from (cold) global memory before its first batch is requested here, in one go: the radial
    // tables of its first window of rows (H1), its first geometry record, the angular table -- one memory round trip
    // instead of three in a row (an L2 flush, or a first build, makes each of them a DRAM miss)
    const RowTab tab0 = pipe_row_tables(P, n_rows, g0, gmod, lane, 0);
    if (CONSTC && lane * 8 < 2 * Npad) {     // the coefficient bank was rewritten just before this launch: cold in the constant
        double ctouch;                       // cache -- one lane per 64 B line asks now (volatile: the unused load stays)
        asm volatile("ld.const.f64 %0, [%1];" : "=d"(ctouch) : "l"(c_coef + lane * 8));
    }
    int bi = (int)(r0 / Nr);
    int q = (int)(r0 - (long long)bi * Nr);
    int cur_b = bi / P.Next;
    int e = bi - cur_b * P.Next;
    int kb = (int)(t0 - r0 * BPR);
    const unsigned gtotal = (unsigned)P.Next * (unsigned)Nr * (unsigned)P.Ntpad;
    unsigned gidx = 0, gphase = 0;
    const unsigned long long gpolicy = l2_evict_first_policy();
    auto prefetch = [&](unsigned buf) {      // geometry stream (GEOM): consecutive 1 KB records, cp.async double buffer
        const double4 *src = reinterpret_cast<const double4 *>(P.geom) + gidx;
        const unsigned dst = (unsigned)__cvta_generic_to_shared(s_gbuf + buf * 32 + lane);
        asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(src), "l"(gpolicy));
        asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;\n" ::"r"(dst + 16), "l"(reinterpret_cast<const char *>(src) + 16), "l"(gpolicy));
        asm volatile("cp.async.commit_group;\n" ::);
    };
    for (int t = threadIdx.x; t < P.Ntpad * 6; t += blockDim.x)              // angular table -> shared memory, asynchronously
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"((unsigned)__cvta_generic_to_shared(s_ang + t)), "l"(P.ang + t));
    asm volatile("cp.async.commit_group;\n" ::);                           // (the oldest group: complete before any later one)
    if (GEOM && t0 < t1) {
        gidx = ((unsigned)e * Nr + q) * P.Ntpad + kb * 32 + lane;
        prefetch(0);
    }
    if (threadIdx.x < 32) {   // the small tables the tail reads first (cold after an L2 flush): on their way while the points run
        const size_t tb_lines = ((size_t)2 * P.B * P.Next * sizeof(int) + 127) / 128;
        if (threadIdx.x < tb_lines) asm volatile("prefetch.global.L2 [%0];" ::"l"(reinterpret_cast<const char *>(P.tail_bi) + threadIdx.x * 128));
        if (threadIdx.x == 31) asm volatile("prefetch.global.L2 [%0];" ::"l"(P.tail_cta + 2 * blockIdx.x));
        if (threadIdx.x == 30 && blockIdx.x == 0) asm volatile("prefetch.global.L2 [%0];" ::"l"(P.bc));
    }
    {   // the whole table is read row by row (H1, H7) by every warp: pull it into L2 once, spread over the grid
        const size_t lines = ((size_t)gmod * Npad * sizeof(double) + 127) / 128;
        for (size_t l = (size_t)blockIdx.x * blockDim.x + threadIdx.x; l < lines; l += (size_t)gridDim.x * blockDim.x)
            asm volatile("prefetch.global.L2 [%0];" ::"l"(reinterpret_cast<const char *>(P.phi_y) + l * 128));
        const size_t xlines = ((size_t)P.N * Npad * sizeof(double) + 127) / 128;       // phi_j(s_i): read by the tail only
        for (size_t l = (size_t)blockIdx.x * blockDim.x + threadIdx.x; l < xlines; l += (size_t)gridDim.x * blockDim.x)
            asm volatile("prefetch.global.L2 [%0];" ::"l"(reinterpret_cast<const char *>(P.phi_x) + l * 128));
    }
    if (threadIdx.x < EXPTAB_DOUBLES) s_exp[threadIdx.x] = d_exp2_64[threadIdx.x];
    if (!GEOM && threadIdx.x < LOGTAB_DOUBLES) s_log[threadIdx.x] = d_logtab[threadIdx.x];
    pdl_wait();                                             // the coefficients may come from the kernel before (Newton update)
    PHASE_STAMP(1);

    if (t0 < t1) {
    const bool lane_on = EXACT || lane < NCH * SUB;
    const int c_lane = lane_on ? lane / SUB : 0, sub = lane_on ? lane - c_lane * SUB : 0;
    const double halfLg = 0.5 * P.Lg;

    double accA[CJ], accB[CJ], accV[CJ];

    // phase 2 of the batch stashed in buffer `buf`
    auto phase2 = [&](int buf) {
        const double4 *pts = reinterpret_cast<const double4 *>(s_stash + buf * STASH);
        const double2 *trd = reinterpret_cast<const double2 *>(s_stash + buf * STASH + 132) + c_lane * (TCH_STRIDE / 2);
        // the stash entries of round rd + 1 are requested before the 30 FMAs of round rd (their shared-memory latency was
        // the one exposed stall of this block: ncu source view)
        int pt = EXACT ? sub : min(sub, 32);                                     // slot 32: zero weights, finite T
        double4 pw = pts[pt];
        double2 tt = trd[pt];
#pragma unroll
        for (int rd = 0; rd < ROUNDS; ++rd) {
            const double4 cw = pw;
            double T0 = tt.x, T1 = tt.y;
            if (rd + 1 < ROUNDS) {
                pt = EXACT ? (rd + 1) * SUB + sub : min((rd + 1) * SUB + sub, 32);
                pw = pts[pt];
                tt = trd[pt];
            }
            accA[0] = fma(cw.y, T0, accA[0]); accB[0] = fma(cw.z, T0, accB[0]); accV[0] = fma(cw.w, T0, accV[0]);
            accA[1] = fma(cw.y, T1, accA[1]); accB[1] = fma(cw.z, T1, accB[1]); accV[1] = fma(cw.w, T1, accV[1]);
#pragma unroll
            for (int m = 2; m < CJ; ++m) {
                const double T2 = fma(cw.x, T1, -T0);
                accA[m] = fma(cw.y, T2, accA[m]); accB[m] = fma(cw.z, T2, accB[m]); accV[m] = fma(cw.w, T2, accV[m]);
                T0 = T1; T1 = T2;
            }
        }
    };
    // the same for the last batch of a segment (once per segment: a rolled loop -- the unrolled copy above is 6 KB of code,
    // and the loop body of the kernel has to stay inside the 32 KB instruction cache of the SM)
    auto phase2_last = [&](int buf) {
        const double4 *pts = reinterpret_cast<const double4 *>(s_stash + buf * STASH);
        const double2 *trd = reinterpret_cast<const double2 *>(s_stash + buf * STASH + 132) + c_lane * (TCH_STRIDE / 2);
#pragma unroll 1
        for (int rd = 0; rd < ROUNDS; ++rd) {
            const int pt = EXACT ? rd * SUB + sub : min(rd * SUB + sub, 32);
            const double4 pw = pts[pt];
            const double2 tt = trd[pt];
            double T0 = tt.x, T1 = tt.y;
            accA[0] = fma(pw.y, T0, accA[0]); accB[0] = fma(pw.z, T0, accB[0]); accV[0] = fma(pw.w, T0, accV[0]);
            accA[1] = fma(pw.y, T1, accA[1]); accB[1] = fma(pw.z, T1, accB[1]); accV[1] = fma(pw.w, T1, accV[1]);
#pragma unroll
            for (int m = 2; m < CJ; ++m) {
                const double T2 = fma(pw.x, T1, -T0);
                accA[m] = fma(pw.y, T2, accA[m]); accB[m] = fma(pw.z, T2, accB[m]); accV[m] = fma(pw.w, T2, accV[m]);
                T0 = T1; T1 = T2;
            }
        }
    };
    auto flush = [&](int bi, int buf) {      // `buf`'s T area is free: use it as the cross-lane scratch
        double *scr = s_stash + buf * STASH + 132;
        double *slot = P.Spart + (size_t)(w + bi) * SLOT;
        if constexpr (EXACT && (SUB == 4 || SUB == 8)) {
            // transposing reduction over the SUB point sub-lanes of a chunk (the low bits of the lane): at every stage a lane
            // keeps one half of its list and receives the partner's sums of that half -- 12 + 6 (+ 3) shuffles instead of
            // 24 conflicting shared-memory stores and three warp barriers; fixed pairwise order -> deterministic.  A lane ends
            // with 24 / SUB finished sums and stores them itself.
            double v[24];
#pragma unroll
            for (int m = 0; m < CJ; ++m) { v[m] = accA[m]; v[CJ + m] = accB[m]; v[2 * CJ + m] = accV[m]; }
            int base = 0;
#pragma unroll
            for (int d = SUB / 2, n = 24; d >= 1; d >>= 1, n >>= 1) {
                const int half = n >> 1;
                const bool up = (sub & d) != 0;
#pragma unroll
                for (int i = 0; i < 12; ++i) {
                    if (i < half) {
                        const double keep = up ? v[half + i] : v[i];
                        const double send = up ? v[i] : v[half + i];
                        v[i] = keep + __shfl_xor_sync(FULL, send, d);
                    }
                }
                base += up ? half : 0;
            }
#pragma unroll
            for (int i = 0; i < 24 / SUB; ++i) {
                const int o = base + i, st = o >> 3, m = o & 7;          // o = stream * 8 + index in the chunk
                slot[st * Npad + c_lane * CJ + m] = v[i];
            }
        } else {
#pragma unroll
            for (int st = 0; st < 3; ++st) {
                __syncwarp();
#pragma unroll
                for (int m = 0; m < CJ; ++m)
                    if (lane_on) scr[sub * Npad + c_lane * CJ + m] = (st == 0 ? accA[m] : (st == 1 ? accB[m] : accV[m]));
                __syncwarp();
                for (int j = lane; j < Npad; j += 32) {
                    double s = 0.0;
                    for (int sb = 0; sb < SUB; ++sb) s += scr[sb * Npad + j];
                    slot[st * Npad + j] = s;
                }
            }
            __syncwarp();
        }
    };

    // (geometry stream: 32-bit record index, at most 2^31 points per system; checked in dse_create)
    int row = 0;                                           // running row index of the flattened (b, e, q), relative to r0
    int gp_base = 0;                                       // current window of rows: [gp_base, gp_base + 32)
    auto fill_gp = [&](int rb, RowTab tab) {
        pipe_fill_gp<Npad, CONSTC>(P, r0, n_rows, tab, s_coef, cur_b, s_gp, lane, rb);
        gp_base = rb;
    };
    auto contract = [&](int bi, int e, int qa, int qb, bool last_partial) {
        pipe_contract<Npad>(P, P.Spart + (size_t)(w + bi) * SLOT, bi, e, qa, qb, last_partial, lane);
    };

    auto load_coef = [&](int b) {                          // (a_j, b_j) pairs of system b, zero padded
        const double *ca = P.c + (size_t)b * 2 * P.N;
        for (int j = lane; j < Npad; j += 32) s_coef[j] = j < P.N ? make_double2(__ldg(ca + j), __ldg(ca + P.N + j)) : make_double2(0.0, 0.0);
        __syncwarp();
    };
    if (!CONSTC) load_coef(cur_b);
    fill_gp(0, tab0);

    // both T stashes must hold finite numbers before the first (zero-weight) prologue phase 2
    for (int b2 = 0; b2 < 2; ++b2)
        for (int c = 0; c < NCH; ++c) {
            double2 *tz = reinterpret_cast<double2 *>(s_stash + b2 * STASH + 132) + c * (TCH_STRIDE / 2);
            tz[lane] = make_double2(0.0, 0.0);
            if (!EXACT && lane == 0) tz[32] = make_double2(0.0, 0.0);        // read with the zero-weight slot 32
        }
    if (!EXACT && lane < 2) reinterpret_cast<double4 *>(s_stash + lane * STASH)[32] = make_double4(0.0, 0.0, 0.0, 0.0);

    // H1 above ran while the angular table and the first geometry record were on their way; now the table must be there
    if (GEOM) asm volatile("cp.async.wait_group 1;\n" ::: "memory");       // all but the geometry record
    else asm volatile("cp.async.wait_group 0;\n" ::: "memory");
    __syncthreads();
    PHASE_STAMP(2);
    int rem = (int)(t1 - t0);                              // batches left for this warp
    int cur = 0;                                           // stash half written by the current batch
    while (rem > 0) {
        // ---------------- one (warp, external point) segment ----------------
#pragma unroll
        for (int m = 0; m < CJ; ++m) accA[m] = accB[m] = accV[m] = 0.0;
        reinterpret_cast<double4 *>(s_stash + (cur ^ 1) * STASH)[lane] = make_double4(0.0, 0.0, 0.0, 0.0);   // prologue
        __syncwarp();
        bool seg_done = false;
        const int q_seg = q;                               // first row of this segment
        bool last_partial = false;
        while (!seg_done) {
            if (row - gp_base >= 32) fill_gp(row, pipe_row_tables(P, n_rows, g0, gmod, lane, row));   // (warp-uniform)
            const double2 gp = s_gp[row - gp_base];
            const double Gy = gp.x, Py = gp.y;
            RowConst rc;
            if (!GEOM) {
                const double x = P.x_ext[e], sx = P.sx_ext[e], c3x = P.c3x_ext[e];
                const int rq = e * P.rstride + q;
                const double y = P.y[rq], sy = P.sy[rq];
                const double Wq = P.Wy[rq];
                const double d = (x - y) / (sx + sy);
                rc.d2 = d * d; rc.sxy = sx * sy; rc.rv = -P.C * Wq * y; rc.rq = c3x * Wq; rc.rm = c3x * Wq * y;
            }
            double sumA = 0.0, sumB = 0.0, sumV = 0.0, sumZ = 0.0;
            const int kb_end = (rem < BPR - kb) ? kb + rem : BPR;
            for (; kb < kb_end; ++kb, --rem) {
                double sraw, gv, gq, gm;
                if (GEOM) {
                    gidx += 32;
                    if (gidx >= gtotal) gidx -= gtotal;
                    prefetch(gphase ^ 1);
                    asm volatile("cp.async.wait_group 1;\n" ::: "memory");
                    const double2 *gpp = reinterpret_cast<const double2 *>(s_gbuf + gphase * 32 + lane);
                    const double2 g0 = gpp[0], g1 = gpp[1];
                    sraw = g0.x; gv = g0.y; gq = g1.x; gm = g1.y;
                    gphase ^= 1;
                } else {
                    point_geometry_fast(rc, s_ang + (kb * 32 + lane) * 6, P.inv_eps2, P.two_over_Lg, s_log, sraw, gv, gq, gm);
                }
                double s = sraw, EG = 0.0, EZ = 0.0;
                if (sraw < -1.0) {                       // z < eps2: eq.(16),(17)
                    const double ell = (sraw + 1.0) * halfLg;
                    EG = P.pG * ell; EZ = P.pZ * ell; s = -1.0;
                } else if (sraw > 1.0) {                 // z > L2: eq.(18),(19)
                    const double t = GEOM ? sraw - 2.0 : log(fma(P.omega, (sraw - 1.0) * halfLg, 1.0));   // (cached: the record carries 2 + t)
                    EG = P.delta * t; EZ = P.gamma * t; s = 1.0;
                }
                // ======== main block: phase 1 of this batch || phase 2 of the previous batch ========
                const double ts = 2.0 * s;
                const double t2 = fma(2.0 * ts, s, -2.0);
                double Te = 1.0, To = s, Tem = fma(ts, s, -1.0), Tom = s;
                double lz0 = 0.0, lz1 = 0.0, lg0 = 0.0, lg1 = 0.0;
                double2 *tw = reinterpret_cast<double2 *>(s_stash + cur * STASH + 132);
#pragma unroll
                for (int c = 0; c < NCH; ++c) {
                    tw[c * (TCH_STRIDE / 2) + lane] = make_double2(Te, To);
#pragma unroll
                    for (int m = 0; m < CJ; m += 4) {
                        const int j0 = c * CJ + m;
                        const double2 c0 = CONSTC ? make_double2(c_coef[j0], c_coef[Npad + j0]) : s_coef[j0];
                        const double2 c1 = CONSTC ? make_double2(c_coef[j0 + 1], c_coef[Npad + j0 + 1]) : s_coef[j0 + 1];
                        const double2 c2 = CONSTC ? make_double2(c_coef[j0 + 2], c_coef[Npad + j0 + 2]) : s_coef[j0 + 2];
                        const double2 c3 = CONSTC ? make_double2(c_coef[j0 + 3], c_coef[Npad + j0 + 3]) : s_coef[j0 + 3];
                        if (j0 == 0) { lz0 = 0.5 * c0.x; lg0 = 0.5 * c0.y; }      // phi_0 = 1/2: the c_0/2 of eq.(23),(24)
                        else { lz0 = fma(c0.x, Te, lz0); lg0 = fma(c0.y, Te, lg0); }
                        lz1 = fma(c1.x, To, lz1); lg1 = fma(c1.y, To, lg1);
                        Tem = fma(t2, Te, -Tem);  Tom = fma(t2, To, -Tom);
                        lz0 = fma(c2.x, Tem, lz0); lg0 = fma(c2.y, Tem, lg0);
                        lz1 = fma(c3.x, Tom, lz1); lg1 = fma(c3.y, Tom, lg1);
                        Te = fma(t2, Tem, -Te);   To = fma(t2, Tom, -To);
                    }
                }
                const double lnZz = (lz0 + lz1) + EZ, lnGz = (lg0 + lg1) + EG;
                const double lnPz = fma(P.e1, lnGz, P.e2 * lnZz);
                double Zz = fast_exp_tab(lnZz, s_exp), Gz = fast_exp_tab(lnGz, s_exp), Pz = fast_exp_tab(lnPz, s_exp);
                phase2(cur ^ 1);
                // ======== end of main block ========
                const int hmax = max(max(__double2hiint(lnZz) & 0x7fffffff, __double2hiint(lnGz) & 0x7fffffff),
                                     __double2hiint(lnPz) & 0x7fffffff);
                if (hmax >= 0x4085e000) { Zz = exp(lnZz); Gz = exp(lnGz); Pz = exp(lnPz); }   // |x| > 700 or NaN
                const double v = gv * (Gy * Zz);              // eq.(8)
                const double wQ = gq * (Py * Pz);             // eq.(9), gluon loop
                const double wM = gm * (Gy * Gz);             // eq.(9), ghost loop
                const double ua = P.e2 * wQ;
                const double ub = fma(P.e1, wQ, wM);
                sumA += ua; sumB += ub; sumV += v; sumZ += wQ + wM;
                reinterpret_cast<double4 *>(s_stash + cur * STASH)[lane] = make_double4(ts, ua, ub, v);
                __syncwarp();
                cur ^= 1;
            }
            // H5/H7: row sums over the 32 angular lanes.  Transposing reduction: after the first two steps each
            // quarter-warp carries one of the four sums (6 shuffles instead of 20; fixed order -> deterministic).
            {
                const bool up = lane & 16, hi = lane & 8;
                double x0 = up ? sumV : sumA, x1 = up ? sumZ : sumB;
                const double y0 = up ? sumA : sumV, y1 = up ? sumB : sumZ;
                x0 += __shfl_xor_sync(FULL, y0, 16);
                x1 += __shfl_xor_sync(FULL, y1, 16);
                double z = hi ? x1 : x0;
                const double zs = hi ? x0 : x1;
                z += __shfl_xor_sync(FULL, zs, 8);
                z += __shfl_xor_sync(FULL, z, 4);
                z += __shfl_xor_sync(FULL, z, 2);
                z += __shfl_xor_sync(FULL, z, 1);
                // lanes 0, 8, 16, 24 hold sum(u_a), sum(u_b), sum(v), sum(wQ + wM) of this warp's part of the row: its record
                const bool has_last = kb_end == BPR;
                double *dst = (has_last ? P.Apart : P.AHead) + ((size_t)bi * Nr + q) * 4 + (lane >> 3);
                if ((lane & 7) == 0) *dst = z;
                last_partial = !has_last;
                if (has_last) { kb = 0; ++q; ++row; if (q == Nr) seg_done = true; }
                if (rem <= 0) seg_done = true;
            }
        }
        // epilogue: phase 2 of the segment's last batch, then the partial of this (warp, external point)
        const long long t_seg = PHASE_NOW();
        phase2_last(cur ^ 1);
        flush(bi, cur);
        contract(bi, e, q_seg, last_partial ? q : q - 1, last_partial);
        PHASE_ADD(9, PHASE_NOW() - t_seg); PHASE_ADD(10, 1);
        if (q >= Nr) {
            q = 0; ++bi; ++e;
            if (e == P.Next) {
                e = 0; ++cur_b;
                if (!CONSTC && rem > 0) { __syncwarp(); load_coef(cur_b); }
            }
        }
    }
    if (GEOM) asm volatile("cp.async.wait_group 0;\n" ::: "memory");
    } else {                                               // a warp without work: its part of the angular table, the barrier
        asm volatile("cp.async.wait_group 0;\n" ::: "memory");
        __syncthreads();
    }
    PHASE_STAMP(3);
    build_tail(P, smem);                                   // H8 by the last-arriving CTAs (dse_tail.cuh)
}
using KernelFn = void (*)(const KParams);

template <bool GEOM, bool JAC>
KernelFn pick_nch(int nch)
{
    switch (nch) {
        case 1: return point_kernel<1, GEOM, JAC>;
        case 2: return point_kernel<2, GEOM, JAC>;
        case 4: return point_kernel<4, GEOM, JAC>;
        case 8: return point_kernel<8, GEOM, JAC>;
        case 16: return point_kernel<16, GEOM, JAC>;
        default: return point_kernel<0, GEOM, JAC>;       // run-time chunk count
    }
}

KernelFn pick(const KParams &k, bool jac)
{
    if (!jac) return k.geom ? pick_nch<true, false>(k.NCH) : pick_nch<false, false>(k.NCH);
    return k.geom ? pick_nch<true, true>(k.NCH) : pick_nch<false, true>(k.NCH);
}

int fail(cudaError_t e, const char *what) { return cuda_fail((int)e, what); }

}  // namespace

// include/dse_diag.h: the phase stamps of the last single-system build (0 words unless built with -DDSE_PHASE_TIMING)
int phase_stamps_point(long long *out_host, int max_words)
{
#ifdef DSE_PHASE_TIMING
    const int n = PHASE_CTAS * PHASE_WARPS * PHASE_SLOTS < max_words ? PHASE_CTAS * PHASE_WARPS * PHASE_SLOTS : max_words;
    const cudaError_t e = cudaMemcpyFromSymbol(out_host, g_phase, sizeof(long long) * n);
    return e == cudaSuccess ? n : cuda_fail((int)e, "cudaMemcpyFromSymbol(phase stamps)");
#else
    (void)out_host; (void)max_words;
    return 0;
#endif
}

// DSE_FLAG_CONST_COEF: the __constant__ coefficient arrays are one slot per loaded library; a handle holds it from
// dse_create to dse_destroy, and only if its caller asked for it.
static std::atomic<int> g_const_owner{0};
bool constc_shape_ok(const KParams &k)
{
    const bool pow2 = k.NCH == 1 || k.NCH == 2 || k.NCH == 4 || k.NCH == 8 || k.NCH == 16;
    return k.B == 1 && pow2 && k.N == k.Npad && k.g == 32;
}
bool const_slot_acquire()
{
    int expected = 0;
    return g_const_owner.compare_exchange_strong(expected, 1);
}
void const_slot_release() { g_const_owner.store(0); }

constexpr int PIPE_THREADS_BIG = 512;
static KernelFn pick_pipe(const KParams &k, bool big = false)
{
    if (big && k.NCH == 8) {                                     // 16 warps per SM: large problems with N = 57..64
        if (k.use_constc) return k.geom ? point_kernel_pipe<8, true, true, PIPE_THREADS_BIG> : point_kernel_pipe<8, false, true, PIPE_THREADS_BIG>;
        return k.geom ? point_kernel_pipe<8, true, false, PIPE_THREADS_BIG> : point_kernel_pipe<8, false, false, PIPE_THREADS_BIG>;
    }
#define DSE_PIPE_CASE(N)                                                                         \
    case N:                                                                                      \
        if (k.use_constc) return k.geom ? point_kernel_pipe<N, true, true> : point_kernel_pipe<N, false, true>; \
        return k.geom ? point_kernel_pipe<N, true, false> : point_kernel_pipe<N, false, false>;
#define DSE_PIPE_CASE_S(N)                                                                       \
    case N:                                                                                      \
        return k.geom ? point_kernel_pipe<N, true, false> : point_kernel_pipe<N, false, false>;
    switch (k.NCH) {
        DSE_PIPE_CASE(1)
        DSE_PIPE_CASE(2)
        DSE_PIPE_CASE_S(3)
        DSE_PIPE_CASE(4)
        DSE_PIPE_CASE_S(5)       // the paper's N = 36
        DSE_PIPE_CASE_S(6)
        DSE_PIPE_CASE_S(7)
        DSE_PIPE_CASE(8)
        DSE_PIPE_CASE_S(12)      // the paper's N = 96
        DSE_PIPE_CASE(16)
        default: return nullptr;
    }
#undef DSE_PIPE_CASE
#undef DSE_PIPE_CASE_S
}

// grid of the pipelined kernel: units are 32-point batches; every warp gets at least one row's worth of them, so that
// a row spans at most two warps (small problems are latency-bound: more warps with less work each is faster)
static long long pick_grid_pipe(const KParams &k, int sms, int per_sm, int wpb)
{
    const long long bpr = k.Ntpad / 32, units = k.R * bpr, min_units = bpr;
    long long grid = (long long)sms * per_sm;
    long long want_grid = (units / min_units + wpb - 1) / wpb;
    if (want_grid < 1) want_grid = 1;
    if (want_grid < grid) grid = want_grid;
    while (grid > 1 && units / (grid * wpb) < min_units) --grid;
    return grid;
}

static long long pick_grid(const KParams &k, int sms, int per_sm, int wpb)
{
    // persistent-style grid: one wave of resident CTAs, but never more warps than rows
    long long grid = (long long)sms * per_sm;
    const long long batches_per_row = k.Ntpad / 32 > 0 ? k.Ntpad / 32 : 1;   // 32-point batches
    // small problems are latency-bound: one 32-point batch per warp
    long long want_warps = k.R * batches_per_row / k.rpb;
    if (want_warps < 1) want_warps = 1;
    long long want_grid = (want_warps + wpb - 1) / wpb;
    if (want_grid < grid) grid = want_grid;
    while (grid * wpb > k.R && grid > 1) --grid;
    return grid;
}

int query_point_kernel(const KParams &k, PointKernelConfig &cfg)
{
    int dev = 0, sms = 0, smem_max = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(e, "cudaGetDevice");
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return fail(e, "cudaDeviceGetAttribute");
    e = cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e != cudaSuccess) return fail(e, "cudaDeviceGetAttribute(smem)");
    cfg.sms = sms;

    // residual-only build (and the Jacobian build of generic shapes): warp-independent kernel, 512 threads
    // (large N with full-warp angular batches: fewer warps per CTA until the per-warp stashes fit in shared memory)
    const long long ngb = (long long)k.B * k.Gext * k.Nr;
    const int h1_rows = ngb <= SELF_H1_MAX_ROWS ? (int)ngb : 0;      // (used by the Jacobian build of non-pipelined handles only)
    auto gsmem = [&](int thr) {
        int d = k.Ntpad * 6 + 2 * h1_rows + (thr / 32) * warp_doubles(k.Npad, k.NCH);
        const int need = tail_smem_doubles(k.Npad, thr);                    // the fused tail reuses the dynamic shared memory
        if (d < need) d = need;
        return (int)sizeof(double) * d;
    };
    int gthr = POINT_THREADS;
    while (gthr > 128 && gsmem(gthr) > smem_max) gthr -= 128;
    const int smem = gsmem(gthr);
    if (smem > smem_max) { set_error_text("n_theta too large: the angular table does not fit in shared memory"); return DSE_EINVAL; }
    for (int jac = 0; jac < 2; ++jac) {
        e = cudaFuncSetAttribute((const void *)pick(k, jac != 0), cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return fail(e, "cudaFuncSetAttribute(point_kernel smem)");
    }
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void *)pick(k, false), gthr, smem);
    if (e != cudaSuccess) return fail(e, "cudaOccupancyMaxActiveBlocksPerMultiprocessor");
    if (per_sm < 1) { set_error_text("point_kernel does not fit on an SM"); return DSE_ECUDA; }
    cfg.res_block = gthr;
    cfg.res_smem = smem;
    cfg.res_grid = (int)pick_grid(k, sms, per_sm, gthr / 32);

    // Jacobian build: software-pipelined kernel when the shape allows it
    const void *fn = (const void *)pick(k, true);
    int block = gthr, jsmem = smem;
    cfg.pipelined = 0;
    cfg.batched = 0;
    KernelFn pf = k.g == 32 ? pick_pipe(k) : nullptr;
    if (pf) {
        auto psmem_of = [&](int thr) {
            int d = k.Ntpad * 6 + EXPTAB_DOUBLES + (k.geom ? 0 : LOGTAB_DOUBLES) + (thr / 32) * pipe_warp_doubles(k.Npad, k.NCH, k.use_constc != 0, k.geom != nullptr);
            const int need = tail_smem_doubles(k.Npad, thr);                // the fused tail reuses the dynamic shared memory
            if (d < need) d = need;
            return (int)sizeof(double) * d;
        };
        // large problems (>= 48 batches per warp at 16 warps per SM) with 8 chunks: the 512-thread build of the kernel
        const long long units = k.R * (k.Ntpad / 32);
        const int big_smem = psmem_of(PIPE_THREADS_BIG);
        const bool big = k.NCH == 8 && units >= 48LL * sms * (PIPE_THREADS_BIG / 32) && big_smem <= smem_max;
        if (big) {
            pf = pick_pipe(k, true);
            e = cudaFuncSetAttribute((const void *)pf, cudaFuncAttributeMaxDynamicSharedMemorySize, big_smem);
            if (e != cudaSuccess) return fail(e, "cudaFuncSetAttribute(point_kernel_pipe smem)");
            fn = (const void *)pf; block = PIPE_THREADS_BIG; jsmem = big_smem; cfg.pipelined = 2;
        }
        // large N: fewer warps per CTA until the double-buffered stashes fit in shared memory (at least 8 warps)
        for (int thr = PIPE_THREADS; !big && thr >= 256; thr -= 128) {
            const int psmem = psmem_of(thr);
            if (psmem > smem_max) continue;
            e = cudaFuncSetAttribute((const void *)pf, cudaFuncAttributeMaxDynamicSharedMemorySize, psmem);
            if (e != cudaSuccess) return fail(e, "cudaFuncSetAttribute(point_kernel_pipe smem)");
            fn = (const void *)pf; block = thr; jsmem = psmem; cfg.pipelined = 1;
            break;
        }
    }
    cudaFuncAttributes fa;
    e = cudaFuncGetAttributes(&fa, fn);
    if (e != cudaSuccess) return fail(e, "cudaFuncGetAttributes");
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, block, jsmem);
    if (e != cudaSuccess) return fail(e, "cudaOccupancyMaxActiveBlocksPerMultiprocessor");
    if (per_sm < 1) { set_error_text("point kernel does not fit on an SM"); return DSE_ECUDA; }
    cfg.block = block;
    cfg.smem = jsmem;
    cfg.regs = fa.numRegs;
    cfg.ctas_per_sm = per_sm;
    cfg.grid = (int)(cfg.pipelined ? pick_grid_pipe(k, sms, per_sm, block / 32) : pick_grid(k, sms, per_sm, block / 32));
    return 0;
}

// Launches the point kernel of one build; k.c, k.bc, k.J, k.F and k.want_jac are set.  Returns the number of kernels
// launched (1) or < 0.
int launch_point(const KParams &k, const PointKernelConfig &cfg, void *stream)
{
    cudaStream_t s = (cudaStream_t)stream;
    if (cfg.batched) return launch_point_batched(k, cfg, stream);     // Jacobian or residual-only variant
    cudaError_t e;
    if (k.want_jac) {
        if (cfg.pipelined && k.use_constc) {                   // c -> constant bank (documented in-stream update)
            e = cudaMemcpyToSymbolAsync(c_coef, k.c, sizeof(double) * 2 * k.N, 0, cudaMemcpyDeviceToDevice, s);
            if (e != cudaSuccess) return fail(e, "cudaMemcpyToSymbolAsync(coefficients)");
        }
        KernelFn fn = cfg.pipelined ? pick_pipe(k, cfg.pipelined == 2) : pick(k, true);
        e = launch_pdl(fn, dim3(cfg.grid), dim3(cfg.block), (size_t)cfg.smem, s, k);
    } else {
        KParams kk = k;
        kk.W = cfg.res_grid * (cfg.res_block / 32);          // the residual build has its own row partition
        e = launch_pdl(pick(k, false), dim3(cfg.res_grid), dim3(cfg.res_block), (size_t)cfg.res_smem, s, kk);
    }
    if (e != cudaSuccess) return fail(e, "point kernel launch");
    return 1;
}

}  // namespace dse

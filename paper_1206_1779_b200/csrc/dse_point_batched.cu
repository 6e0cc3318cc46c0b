// dse_point_batched.cu -- the point kernel for batched builds (BASELINE configs[4]: 256 independent systems on one
// grid).  All systems share the geometry and therefore T_j(s~(z)) of every quadrature point, so both contractions of
// the hot path become DENSE and run on the fp64 tensor path (mma.sync.m8n8k4.f64 -> DMMA):
//   step A (series):      L[pt, (sys, a|b)]  = sum_j T[pt, j] * Coef[j, (sys, a|b)]     M = 8 points, N = 8 columns
//   step C (accumulate):  S[sys, j](stream) += sum_pt U[sys, pt](stream) * T[pt, j]     M = 8 systems, K = 4 points
// Each WARP owns 8 systems and a contiguous range of 32-point batches (4 tiles of 8 points); per tile: every lane
// evaluates the geometry of point lane/4 and the eight T_j, j = lane%4 (mod 4), by a stride-4 Chebyshev recurrence
// (exactly the A fragments of step A), writes them to a warp-private tile for the B fragments of step C; the C
// fragments of step A hand every lane ln Z(z), ln G(z) of two (point, system) pairs -> 3 exp and the weights there;
// the weights are transposed into A fragments with shuffles.  Partials per (warp, system group, external point) are
// written straight from the accumulator fragments; assemble_kernel sums them in warp order (deterministic).
// Requirements: n_batch >= 8 (padded to a multiple of 8 with idle systems, at most a quarter of the padded batch),
// N <= 64 (tiles of 16, 32, 48 or 64 indices), full-warp angular batches; other shapes, and handles created with
// DSE_FLAG_PER_SYSTEM_KERNELS, use dse_point.cu.
#include <cstdio>

#include "dse_device.cuh"

namespace dse {

namespace {

// NPADB = N padded to a multiple of 16 (16, 32, 48 or 64): Chebyshev extent of the tiles
template <int NPADB> struct BT {
    static constexpr int THREADS = NPADB <= 32 ? 384 : 256;      // 12 or 8 warps per SM (register budget)
    static constexpr int KS = NPADB / 4;                         // k-steps of step A
    static constexpr int NT = NPADB / 8;                         // n-tiles of step C
    static constexpr int TS = NPADB + 4;                         // row stride of the T tile: = 4 (mod 16), conflict-free
    static constexpr int COEF_DOUBLES = 2 * KS * 32;             // step-A B fragments of the warp's 8 systems
    static constexpr int WARP_DOUBLES = 8 * TS + GBUF_DOUBLES + COEF_DOUBLES;
};

__device__ __forceinline__ void dmma(double &c0, double &c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
        : "+d"(c0), "+d"(c1)
        : "d"(a), "d"(b));
}

// JAC = false: residual only (dse_residual) -- steps A and B and the row sums, no T tile, no accumulation
template <bool GEOM, int NPADB, bool JAC>
__global__ void __launch_bounds__(BT<NPADB>::THREADS, 1) point_kernel_batched(const KParams P)
{
    constexpr int BT_KS = BT<NPADB>::KS, BT_NT = BT<NPADB>::NT, BT_TS = BT<NPADB>::TS, BT_WARP_DOUBLES = BT<NPADB>::WARP_DOUBLES;
    extern __shared__ __align__(16) double smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, WPB = blockDim.x >> 5;
    double *s_ang = smem;
    double *s_exp = smem + (size_t)P.Ntpad * 6;                                     // 2^(k/64): table of fast_exp_tab
    double *sT = s_exp + EXPTAB_DOUBLES + (size_t)warp * BT_WARP_DOUBLES;           // [8][BT_TS]
    double4 *s_gbuf = reinterpret_cast<double4 *>(sT + 8 * BT_TS);                  // [2][32] geometry records
    double *sC = sT + 8 * BT_TS + GBUF_DOUBLES;                                     // [BT_KS][2][32] coefficient fragments
    for (int t = threadIdx.x; t < P.Ntpad * 6; t += blockDim.x) s_ang[t] = P.ang[t];
    if (threadIdx.x < EXPTAB_DOUBLES) s_exp[threadIdx.x] = d_exp2_64[threadIdx.x];
    pdl_wait();                                             // prep_kernel: coefficient pairs, G(y_q), P(y_q)
    __syncthreads();

    const int Nr = P.Nr, BPR = P.Ntpad >> 5, NG = P.Gext * Nr;
    const long long w = (long long)blockIdx.x * WPB + warp;
    const long long t0 = (w * P.U) / P.W, t1 = ((w + 1) * P.U) / P.W;
    if (t0 >= t1) return;
    const int pt_l = lane >> 2, jq = lane & 3;           // step A/B: point of the tile, systems jq and 4 + jq
    const double halfLg = 0.5 * P.Lg;

    long long r0 = t0 / BPR;
    int kb = (int)(t0 - r0 * BPR);
    int big = (int)(r0 / Nr);                            // group-level external index: sg * Next + e
    int q = (int)(r0 - (long long)big * Nr);
    int sg = big / P.Next, e = big - sg * P.Next;
    int rem = (int)(t1 - t0);

    // geometry stream (cache): consecutive 1 KB records of 32 points, cp.async double buffer
    const unsigned gtotal = (unsigned)P.Next * (unsigned)Nr * (unsigned)P.Ntpad;
    unsigned gidx = 0, gphase = 0;
    auto prefetch = [&](unsigned buf) {
        const double4 *src = reinterpret_cast<const double4 *>(P.geom) + gidx;
        const unsigned dst = (unsigned)__cvta_generic_to_shared(s_gbuf + buf * 32 + lane);
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(dst), "l"(src));
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(dst + 16), "l"(reinterpret_cast<const char *>(src) + 16));
        asm volatile("cp.async.commit_group;\n" ::);
    };
    if (GEOM) {
        gidx = ((unsigned)e * Nr + q) * P.Ntpad + kb * 32 + lane;
        prefetch(0);
    }

    // step-A B fragments (coefficients of the 8 systems) live in shared memory, one value per (k-step, pair, lane)
    auto load_coef = [&](int g) {
        const int col = lane >> 2;                        // column of the n-tile: system col/2, part col%2 (a|b)
        const double *c0 = P.coefP + ((size_t)(8 * g + (col >> 1)) * P.Npad) * 2 + (col & 1);
        const double *c1 = P.coefP + ((size_t)(8 * g + 4 + (col >> 1)) * P.Npad) * 2 + (col & 1);
#pragma unroll
        for (int ks = 0; ks < BT_KS; ++ks) {
            const bool in = 4 * ks + jq < P.Npad;           // NPADB may exceed the library's padding (multiple of 8)
            sC[(2 * ks) * 32 + lane] = in ? c0[(size_t)(4 * ks + jq) * 2] : 0.0;
            sC[(2 * ks + 1) * 32 + lane] = in ? c1[(size_t)(4 * ks + jq) * 2] : 0.0;
        }
    };
    load_coef(sg);

    double acc[3][BT_NT][2];                              // step-C accumulators: rows = systems, cols = j
    while (rem > 0) {
        // ---------------- one (warp, system group, external point) segment ----------------
        if (JAC) {
#pragma unroll
            for (int st = 0; st < 3; ++st)
#pragma unroll
                for (int nt = 0; nt < BT_NT; ++nt) acc[st][nt][0] = acc[st][nt][1] = 0.0;
        }
        bool seg_done = false;
        while (!seg_done) {
            const size_t gq0 = ((size_t)(8 * sg + jq) * P.Gext + (P.rstride ? e : 0)) * Nr + q;
            const size_t gq1 = gq0 + (size_t)4 * NG;
            const double Gy0 = P.Gy[gq0], Py0 = P.Py[gq0], Gy1 = P.Gy[gq1], Py1 = P.Py[gq1];
            RowConst rc;
            if (!GEOM) {
                const double x = P.x_ext[e], sx = P.sx_ext[e], c3x = P.c3x_ext[e];
                const int rq = e * P.rstride + q;
                const double y = P.y[rq], sy = P.sy[rq], Wq = P.Wy[rq];
                const double d = (x - y) / (sx + sy);
                rc.d2 = d * d; rc.sxy = sx * sy; rc.rv = -P.C * Wq * y; rc.rq = c3x * Wq; rc.rm = c3x * Wq * y;
            }
            double sum0[4] = {0.0, 0.0, 0.0, 0.0}, sum1[4] = {0.0, 0.0, 0.0, 0.0};   // (u_a, u_b, v, wQ+wM) of systems jq, 4+jq
            const int kb_begin = kb;
            const int kb_end = (rem < BPR - kb) ? kb + rem : BPR;
            for (; kb < kb_end; ++kb, --rem) {
                if (GEOM) {
                    gidx += 32;
                    if (gidx >= gtotal) gidx -= gtotal;
                    prefetch(gphase ^ 1);
                    asm volatile("cp.async.wait_group 1;\n" ::: "memory");
                    __syncwarp();
                }
#pragma unroll 1
                for (int tile = 0; tile < 4; ++tile) {
                    const int pidx = tile * 8 + pt_l;                // point of the batch handled by this lane
                    double sraw, gv, gq, gm;
                    if (GEOM) {
                        const double2 *gp = reinterpret_cast<const double2 *>(s_gbuf + gphase * 32 + pidx);
                        const double2 g0 = gp[0], g1 = gp[1];
                        sraw = g0.x; gv = g0.y; gq = g1.x; gm = g1.y;
                    } else {
                        point_geometry(rc, s_ang + (kb * 32 + pidx) * 6, P.inv_eps2, P.two_over_Lg, sraw, gv, gq, gm);
                    }
                    double s = sraw, EG = 0.0, EZ = 0.0;
                    if (sraw < -1.0) {
                        const double ell = (sraw + 1.0) * halfLg;
                        EG = P.pG * ell; EZ = P.pZ * ell; s = -1.0;
                    } else if (sraw > 1.0) {
                        const double t = GEOM ? sraw - 2.0 : log(fma(P.omega, (sraw - 1.0) * halfLg, 1.0));   // (cached: the record carries 2 + t)
                        EG = P.delta * t; EZ = P.gamma * t; s = 1.0;
                    }
                    // T_j(s), j = 4 ks + jq: stride-4 recurrence T_{j+4} = 2 T_4 T_j - T_{j-4}, started from T_0..T_4
                    const double ts = 2.0 * s;
                    const double T2 = fma(ts, s, -1.0), T3 = fma(ts, T2, -s), T4 = fma(ts, T3, -T2);
                    double Tc = jq == 0 ? 1.0 : (jq == 1 ? s : (jq == 2 ? T2 : T3));          // T_jq
                    double Tm = jq == 0 ? T4 : (jq == 1 ? T3 : (jq == 2 ? T2 : s));           // T_{jq-4} = T_{4-jq}
                    const double tw4 = 2.0 * T4;
                    double Tv[BT_KS];
                    Tv[0] = Tc;
#pragma unroll
                    for (int ks = 1; ks < BT_KS; ++ks) {
                        const double Tn = fma(tw4, Tc, -Tm);
                        Tm = Tc; Tc = Tn; Tv[ks] = Tn;
                    }
                    if (JAC) {
                        __syncwarp();                                // the previous tile's B fragments have been read
#pragma unroll
                        for (int ks = 0; ks < BT_KS; ++ks) sT[pt_l * BT_TS + 4 * ks + jq] = Tv[ks];
                    }
                    // ---- step A: ln Z(z), ln G(z) of (point pt_l, systems jq and 4 + jq) ----
                    double lz0 = 0.0, lg0 = 0.0, lz1 = 0.0, lg1 = 0.0;
                    {
                        // four independent accumulator chains (even / odd k-steps) hide the DMMA latency
                        double mz0 = 0.0, mg0 = 0.0, mz1 = 0.0, mg1 = 0.0;
#pragma unroll
                        for (int ks = 0; ks < BT_KS; ks += 2) {
                            dmma(lz0, lg0, Tv[ks], sC[(2 * ks) * 32 + lane]);
                            dmma(lz1, lg1, Tv[ks], sC[(2 * ks + 1) * 32 + lane]);
                            dmma(mz0, mg0, Tv[ks + 1], sC[(2 * ks + 2) * 32 + lane]);
                            dmma(mz1, mg1, Tv[ks + 1], sC[(2 * ks + 3) * 32 + lane]);
                        }
                        lz0 += mz0; lg0 += mg0; lz1 += mz1; lg1 += mg1;
                    }
                    // ---- step B: weights of the two (point, system) pairs ----
                    double U0[3], U1[3];
                    {
                        const double lnZz = lz0 + EZ, lnGz = lg0 + EG, lnPz = fma(P.e1, lnGz, P.e2 * lnZz);
                        const double lnZy = lz1 + EZ, lnGy = lg1 + EG, lnPy = fma(P.e1, lnGy, P.e2 * lnZy);
                        double Zz = fast_exp_tab(lnZz, s_exp), Gz = fast_exp_tab(lnGz, s_exp), Pz = fast_exp_tab(lnPz, s_exp);
                        double Zy = fast_exp_tab(lnZy, s_exp), Gw = fast_exp_tab(lnGy, s_exp), Pw = fast_exp_tab(lnPy, s_exp);
                        const int h0 = max(max(__double2hiint(lnZz) & 0x7fffffff, __double2hiint(lnGz) & 0x7fffffff),
                                           __double2hiint(lnPz) & 0x7fffffff);
                        const int h1 = max(max(__double2hiint(lnZy) & 0x7fffffff, __double2hiint(lnGy) & 0x7fffffff),
                                           __double2hiint(lnPy) & 0x7fffffff);
                        if (max(h0, h1) >= 0x4085e000) {           // |x| > 700 or NaN: library exp
                            Zz = exp(lnZz); Gz = exp(lnGz); Pz = exp(lnPz);
                            Zy = exp(lnZy); Gw = exp(lnGy); Pw = exp(lnPy);
                        }
                        const double v0 = gv * (Gy0 * Zz), wQ0 = gq * (Py0 * Pz), wM0 = gm * (Gy0 * Gz);
                        const double v1 = gv * (Gy1 * Zy), wQ1 = gq * (Py1 * Pw), wM1 = gm * (Gy1 * Gw);
                        U0[0] = P.e2 * wQ0; U0[1] = fma(P.e1, wQ0, wM0); U0[2] = v0;
                        U1[0] = P.e2 * wQ1; U1[1] = fma(P.e1, wQ1, wM1); U1[2] = v1;
                        sum0[0] += U0[0]; sum0[1] += U0[1]; sum0[2] += v0; sum0[3] += wQ0 + wM0;
                        sum1[0] += U1[0]; sum1[1] += U1[1]; sum1[2] += v1; sum1[3] += wQ1 + wM1;
                    }
                    if (JAC) __syncwarp();                           // the T tile is complete
                    // ---- step C: S[sys, j](stream) += sum_pt U[sys, pt] T[pt, j] ----
#pragma unroll
                    for (int h = 0; h < (JAC ? 2 : 0); ++h) {
                        // A fragment: row = system lane/4, col = point 4h + lane%4; its weight lives in lane
                        // 4 * point + system % 4, pair system / 4
                        const int src = 16 * h + 4 * jq + (pt_l & 3);
                        double bfr[BT_NT];
#pragma unroll
                        for (int nt = 0; nt < BT_NT; ++nt) bfr[nt] = sT[(4 * h + jq) * BT_TS + 8 * nt + pt_l];
#pragma unroll
                        for (int st = 0; st < 3; ++st) {
                            const double a0 = __shfl_sync(FULL, U0[st], src), a1 = __shfl_sync(FULL, U1[st], src);
                            const double afr = (pt_l >> 2) ? a1 : a0;
#pragma unroll
                            for (int nt = 0; nt < BT_NT; ++nt) dmma(acc[st][nt][0], acc[st][nt][1], afr, bfr[nt]);
                        }
                    }
                }
                if (GEOM) gphase ^= 1;
            }
            // row sums over the points handled by this warp: reduce over the point index (lane bits 2..4)
#pragma unroll
            for (int cpt = 0; cpt < 4; ++cpt) {
#pragma unroll
                for (int o = 4; o < 32; o <<= 1) {
                    sum0[cpt] += __shfl_xor_sync(FULL, sum0[cpt], o);
                    sum1[cpt] += __shfl_xor_sync(FULL, sum1[cpt], o);
                }
            }
            {
                const bool has_first = kb_begin == 0, has_last = kb_end == BPR;
                if (lane < 4) {                                      // lane = jq: systems jq and 4 + jq
                    double *base = has_last ? P.Apart : P.AHead;
                    const size_t r0i = ((size_t)(8 * sg + jq) * P.Next + e) * Nr + q, r1i = r0i + (size_t)4 * P.Next * Nr;
                    reinterpret_cast<double4 *>(base)[r0i] = make_double4(sum0[0], sum0[1], sum0[2], sum0[3]);
                    reinterpret_cast<double4 *>(base)[r1i] = make_double4(sum1[0], sum1[1], sum1[2], sum1[3]);
                    if (has_first && has_last) {
                        reinterpret_cast<double4 *>(P.AHead)[r0i] = make_double4(0.0, 0.0, 0.0, 0.0);
                        reinterpret_cast<double4 *>(P.AHead)[r1i] = make_double4(0.0, 0.0, 0.0, 0.0);
                    }
                }
                if (has_last) { kb = 0; ++q; if (q == Nr) seg_done = true; }
                if (rem <= 0) seg_done = true;
            }
        }
        // partial of this (warp, system group, external point): accumulator fragments go straight to the slot
        if (JAC) {
            const size_t slot = (size_t)(w + big);
            const int sys = pt_l;                                    // C fragment: row = lane/4, cols 2 (lane%4), +1
#pragma unroll
            for (int st = 0; st < 3; ++st)
#pragma unroll
                for (int nt = 0; nt < BT_NT; ++nt) {
                    double *dst = P.Spart + ((slot * 8 + sys) * 3 + st) * P.Npad + 8 * nt + 2 * jq;
                    if (8 * nt < P.Npad) *reinterpret_cast<double2 *>(dst) = make_double2(acc[st][nt][0], acc[st][nt][1]);
                }
        }
        if (q >= Nr) {
            q = 0; ++big; ++e;
            if (e == P.Next) {
                e = 0; ++sg;
                if (rem > 0) load_coef(sg);
            }
        }
    }
    if (GEOM) asm volatile("cp.async.wait_group 0;\n" ::: "memory");
}

int fail(cudaError_t e, const char *what) { return cuda_fail((int)e, what); }

}  // namespace

// 8 systems per warp: at least 8 systems, at most a quarter of the padded batch wasted, N <= 64, full-warp angular batches
bool batched_eligible(const KParams &k)
{
    const int Bpad = (k.B + 7) / 8 * 8;
    return k.B >= 8 && 4 * (Bpad - k.B) <= Bpad && k.Npad <= 64 && k.g == 32;
}

namespace {
using BatchedFn = void (*)(const KParams);
template <int NPADB> BatchedFn pick_batched(bool geom, bool jac)
{
    if (jac) return geom ? point_kernel_batched<true, NPADB, true> : point_kernel_batched<false, NPADB, true>;
    return geom ? point_kernel_batched<true, NPADB, false> : point_kernel_batched<false, NPADB, false>;
}
struct BatchedVariant { BatchedFn fn; int threads, smem; };
BatchedVariant batched_variant(const KParams &k, bool jac)
{
    const bool g = k.geom != nullptr;
    const int base = (int)sizeof(double) * (k.Ntpad * 6 + EXPTAB_DOUBLES);
#define DSE_BT_CASE(NPADB) \
    return BatchedVariant{pick_batched<NPADB>(g, jac), BT<NPADB>::THREADS, \
                          base + (int)sizeof(double) * (BT<NPADB>::THREADS / 32) * BT<NPADB>::WARP_DOUBLES}
    if (k.Npad <= 16) DSE_BT_CASE(16);
    if (k.Npad <= 32) DSE_BT_CASE(32);
    if (k.Npad <= 48) DSE_BT_CASE(48);
    DSE_BT_CASE(64);
#undef DSE_BT_CASE
}
}  // namespace

int query_point_batched(const KParams &k, PointKernelConfig &cfg)
{
    const BatchedVariant v = batched_variant(k, true);
    const void *fn = (const void *)v.fn;
    const int smem = v.smem;
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e == cudaSuccess)      // the residual-only variant runs in the same launch configuration
        e = cudaFuncSetAttribute((const void *)batched_variant(k, false).fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return fail(e, "cudaFuncSetAttribute(point_kernel_batched)");
    cudaFuncAttributes fa;
    e = cudaFuncGetAttributes(&fa, fn);
    if (e != cudaSuccess) return fail(e, "cudaFuncGetAttributes");
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, v.threads, smem);
    if (e != cudaSuccess) return fail(e, "occupancy(point_kernel_batched)");
    if (per_sm < 1) { set_error_text("point_kernel_batched does not fit on an SM"); return DSE_ECUDA; }
    const long long wpb = v.threads / 32, bpr = k.Ntpad / 32;
    const long long groups = (k.B + 7) / 8;
    const long long units = groups * k.Next * k.Nr * bpr, min_units = bpr;      // at least one row per warp
    long long grid = (long long)cfg.sms * per_sm;
    long long want = (units / min_units + wpb - 1) / wpb;
    if (want < 1) want = 1;
    if (want < grid) grid = want;
    while (grid > 1 && units / (grid * wpb) < min_units) --grid;
    cfg.grid = (int)grid; cfg.block = v.threads; cfg.smem = smem; cfg.regs = fa.numRegs; cfg.ctas_per_sm = per_sm;
    cfg.pipelined = 0; cfg.batched = 1;
    return 0;
}

int launch_point_batched(const KParams &k, const PointKernelConfig &cfg, void *stream)
{
    cudaError_t e = launch_pdl(batched_variant(k, k.want_jac != 0).fn, dim3(cfg.grid), dim3(cfg.block), (size_t)cfg.smem,
                               (cudaStream_t)stream, k);
    if (e != cudaSuccess) return fail(e, "point_kernel_batched launch");
    return 1;
}

}  // namespace dse

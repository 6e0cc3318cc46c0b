// dse_tail.cuh -- steps H7 and H8 fused into the point kernel (single-system kernels: dse_point.cu).
//
// A build used to be prep -> point -> contraction -> assemble: three dependent launches whose only job after the point
// kernel is to add up what it produced.  Here the point kernel finishes the build itself, without any CTA ever waiting
// for another one:
//   * every CTA, after its warps have written their partials (per-(warp, external point) slots of the three z-dependent
//     streams, per-row angular sums), fences, and bumps ONE arrival counter per external point it worked on;
//   * the CTA whose increment completes the count of an external point e ("last arriver") owns e: it sums e's slots in
//     ascending warp order, stages e's row sums A[q] in shared memory, takes Pi_G, Pi_Z (H5) and the z-independent
//     contraction A[q] . phi_j(t_q) (H7) from there, forms the four derivative rows of e and 1/G(x_e), 1/Z(x_e), and
//     bumps the system's counter of finished external points;
//   * the CTA that finishes the last external point of a system writes that system's J and F (MOM subtraction rows
//     eq.(14),(15), local terms, the paper's layout eq.(29),(30),(35)) and clears the counters for the next build.
// The counters only decide WHO does a sum, never the order IN a sum: every reduction runs over slot / row / part
// indices in a fixed order, so J and F are bitwise reproducible.  Data written by other CTAs of the same launch is read
// with ld.global.cg after the fence/counter handshake (L1 is not coherent).
#pragma once
#include "dse_device.cuh"

namespace dse {

__device__ __forceinline__ double4 ldcg4(const double *p)
{
    const double2 a = __ldcg(reinterpret_cast<const double2 *>(p)), b = __ldcg(reinterpret_cast<const double2 *>(p) + 1);
    return make_double4(a.x, a.y, b.x, b.y);
}

__device__ __forceinline__ int dynamic_smem_doubles()
{
    unsigned bytes;
    asm("mov.u32 %0, %%dynamic_smem_size;" : "=r"(bytes));
    return (int)(bytes >> 3);
}

// doubles of shared memory the tail needs besides the staged rows
__host__ __device__ inline int tail_fixed_doubles(int Npad, int threads) { return 3 * Npad + 3 * threads + 64; }

// The derivative rows of external point bi = b * Next + e from its partial slots [wf, wl] and row sums.
__device__ __noinline__ void tail_point(const KParams &P, double *sm, int sm_doubles, long long bi, long long wf, long long wl)
{
    const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, warp = tid >> 5, NW = T >> 5;
    const int Npad = P.Npad, N = P.N, PJ3 = 3 * Npad, Nr = P.Nr;
    const int b = (int)(bi / P.Next), e = (int)(bi - (long long)b * P.Next);
    double *sS = sm;                               // [3][Npad]   slot sums
    double *sX = sm + PJ3;                         // [3 T]       parts of the slot sums, then k-parts of the contraction
    double *sRed = sX + 3 * T;                     // [2][32]     per-warp Pi partials
    double *sA = sRed + 64;                        // [QC][3]     staged row sums
    const int QC = (sm_doubles - tail_fixed_doubles(Npad, T)) / 3;

    // (1) H6 partials: threads = (part, stream, j); every part sums a contiguous range of slots in ascending warp order
    {
        const int parts = T / PJ3 > 1 ? T / PJ3 : 1;
        const long long nw = wl - wf + 1, per = (nw + parts - 1) / parts;
        for (int item = tid; item < parts * PJ3; item += T) {
            const int part = item / PJ3, idx = item - part * PJ3;
            const long long w0 = wf + part * per, w1 = (wl + 1 < w0 + per) ? wl + 1 : w0 + per;
            const double *sp = P.Spart + (size_t)(w0 + bi) * PJ3 + idx;
            double s = 0.0;
#pragma unroll 8
            for (long long w = w0; w < w1; ++w, sp += PJ3) s += __ldcg(sp);
            sX[item] = s;
        }
        __syncthreads();
        for (int idx = tid; idx < PJ3; idx += T) {
            double s = 0.0;
            for (int p = 0; p < parts; ++p) s += sX[p * PJ3 + idx];
            sS[idx] = s;
        }
        __syncthreads();
    }

    // (2) H5 + H7: row sums -> shared memory (chunks of QC rows), Pi partials on the way, then threads = (k-part, j)
    const int KP = T / Npad, j = tid % Npad, kp = tid / Npad;       // T >= 128 >= Npad
    const double *Phi = P.phi_y + (size_t)(P.rstride ? e * P.rstride : 0) * Npad;
    const double *Arow = P.Apart + (size_t)bi * Nr * 4, *Hrow = P.AHead + (size_t)bi * Nr * 4;
    double pg = 0.0, pz = 0.0, ra = 0.0, rb = 0.0, rv = 0.0;
    for (int q0 = 0; q0 < Nr; q0 += QC) {
        const int nq = Nr - q0 < QC ? Nr - q0 : QC;
        for (int q = tid; q < nq; q += T) {
            const double4 a = ldcg4(Arow + (size_t)(q0 + q) * 4), h = ldcg4(Hrow + (size_t)(q0 + q) * 4);
            sA[3 * q] = a.x + h.x; sA[3 * q + 1] = a.y + h.y; sA[3 * q + 2] = a.z + h.z;
            pg += a.z + h.z; pz += a.w + h.w;
        }
        __syncthreads();
        if (kp < KP) {
            const int per = (nq + KP - 1) / KP, qa = kp * per, qb = nq < qa + per ? nq : qa + per;
            const double *ph = Phi + (size_t)(q0 + qa) * Npad + j;
#pragma unroll 8
            for (int q = qa; q < qb; ++q, ph += Npad) {
                const double f = __ldg(ph);
                ra = fma(sA[3 * q], f, ra); rb = fma(sA[3 * q + 1], f, rb); rv = fma(sA[3 * q + 2], f, rv);
            }
        }
        __syncthreads();
    }
    if (kp < KP) { sX[(kp * 3 + 0) * Npad + j] = ra; sX[(kp * 3 + 1) * Npad + j] = rb; sX[(kp * 3 + 2) * Npad + j] = rv; }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { pg += __shfl_xor_sync(FULL, pg, o); pz += __shfl_xor_sync(FULL, pz, o); }
    if (lane == 0) { sRed[warp] = pg; sRed[32 + warp] = pz; }
    __syncthreads();

    // (3) the four derivative rows of this external point: dPi_Z/da = Sa + Ra, dPi_Z/db = Sb + Rb, dPi_G/da = Sv,
    // dPi_G/db = Rv (the kernel accumulates the streams with T_0 = 1; phi_0 = 1/2, eq.(23),(24))
    double *D = P.Dg + (size_t)bi * 4 * Npad;
    for (int jj = tid; jj < Npad; jj += T) {
        double R0 = 0.0, R1 = 0.0, R2 = 0.0;
        for (int p = 0; p < KP; ++p) { R0 += sX[(p * 3 + 0) * Npad + jj]; R1 += sX[(p * 3 + 1) * Npad + jj]; R2 += sX[(p * 3 + 2) * Npad + jj]; }
        const double h = jj == 0 ? 0.5 : 1.0;
        D[jj] = h * sS[jj] + R0;
        D[Npad + jj] = h * sS[Npad + jj] + R1;
        D[2 * Npad + jj] = h * sS[2 * Npad + jj];
        D[3 * Npad + jj] = R2;
    }
    // Pi_G, Pi_Z (warp order) and the local terms 1/G(x_e), 1/Z(x_e) of the collocation points (series eq.(23),(24))
    if (warp == 0) {
        double lnZ = 0.0, lnG = 0.0;
        if (e < N) {
            const double *cb = P.c + (size_t)b * 2 * N, *px = P.phi_x + (size_t)e * Npad;
            for (int jj = lane; jj < N; jj += 32) {
                const double f = __ldg(px + jj);
                lnZ = fma(__ldg(cb + jj), f, lnZ);
                lnG = fma(__ldg(cb + N + jj), f, lnG);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) { lnZ += __shfl_xor_sync(FULL, lnZ, o); lnG += __shfl_xor_sync(FULL, lnG, o); }
        }
        if (lane == 0) {
            double g = 0.0, z = 0.0;
            for (int w2 = 0; w2 < NW; ++w2) { g += sRed[w2]; z += sRed[32 + w2]; }
            double *o = P.PiInv + (size_t)bi * 4;
            o[0] = g; o[1] = z;
            o[2] = e < N ? exp(-lnG) : 0.0;
            o[3] = e < N ? exp(-lnZ) : 0.0;
        }
    }
}

// J and F of system b from the rows of all its external points (eq.(29),(30),(35),(36); MOM subtraction eq.(14),(15)).
__device__ __noinline__ void tail_system(const KParams &P, double *sm, int b)
{
    const int tid = threadIdx.x, T = blockDim.x;
    const int Npad = P.Npad, N = P.N;
    const size_t bi0 = (size_t)b * P.Next, biZ = bi0 + P.iZ, biG = bi0 + P.iG;
    double *sZ = sm, *sG = sm + 2 * Npad;          // dPi_Z/da, dPi_Z/db at x_Z;  dPi_G/da, dPi_G/db at x_G
    for (int t = tid; t < 2 * Npad; t += T) {
        sZ[t] = __ldcg(P.Dg + biZ * 4 * Npad + t);
        sG[t] = __ldcg(P.Dg + biG * 4 * Npad + 2 * Npad + t);
    }
    __syncthreads();
    double *Jb = P.J + (size_t)b * 4 * N * N, *Fb = P.F + (size_t)b * 2 * N;
    for (int item = tid; item < N * Npad; item += T) {
        const int i = item / Npad, j = item - i * Npad;
        if (j >= N) continue;
        const double *Di = P.Dg + (bi0 + i) * 4 * Npad;
        const double phi = __ldg(P.phi_x + (size_t)i * Npad + j);
        const double invG = __ldcg(P.PiInv + (bi0 + i) * 4 + 2), invZ = __ldcg(P.PiInv + (bi0 + i) * 4 + 3);
        Jb[(size_t)i * 2 * N + j] = -phi * invZ - __ldcg(Di + j) + sZ[j];
        Jb[(size_t)i * 2 * N + N + j] = -__ldcg(Di + Npad + j) + sZ[Npad + j];
        Jb[(size_t)(N + i) * 2 * N + j] = -__ldcg(Di + 2 * Npad + j) + sG[j];
        Jb[(size_t)(N + i) * 2 * N + N + j] = -phi * invG - __ldcg(Di + 3 * Npad + j) + sG[Npad + j];
    }
    const double PiG_s = __ldcg(P.PiInv + biG * 4), PiZ_s = __ldcg(P.PiInv + biZ * 4 + 1);
    const double gG = P.bc[2 * b + 0], gZ = P.bc[2 * b + 1];
    for (int i = tid; i < N; i += T) {
        const double4 pi = ldcg4(P.PiInv + (bi0 + i) * 4);
        Fb[i] = pi.w - gZ - pi.y + PiZ_s;          // z(x_i) = 1/Z(x_i) - 1/Z(x_Z) - Pi_Z(x_i) + Pi_Z(x_Z)
        Fb[N + i] = pi.z - gG - pi.x + PiG_s;      // g(x_i) likewise
    }
    for (int e = tid; e < P.Next; e += T) P.cnt[bi0 + e] = 0u;       // ready for the next build on this handle
    if (tid == 0) P.done[b] = 0u;
}

// Called by ALL threads of the CTA after its last partial has been written.  [T0, T1) = the CTA's partition units;
// sm = the CTA's dynamic shared memory (free by now), sm_doubles its size.
__device__ __forceinline__ void build_tail(const KParams &P, double *sm, int sm_doubles, long long T0, long long T1)
{
    __shared__ int s_flag;
    const int tid = threadIdx.x, WPB = blockDim.x >> 5;
    __threadfence();                               // this thread's partials and row sums are visible device-wide ...
    __syncthreads();                               // ... and so are those of the whole CTA before thread 0 counts
    if (T0 >= T1) return;
    const long long upb = (long long)P.Nr * P.upr;                   // partition units per external point
    const long long bi_lo = T0 / upb, bi_hi = (T1 - 1) / upb;
    for (long long bi = bi_lo; bi <= bi_hi; ++bi) {
        // warps (hence CTAs) that own a unit of bi: unit t belongs to warp ((t + 1) W - 1) / U
        const long long rf = bi * upb, rl = rf + upb - 1;
        const long long wf = ((rf + 1) * P.W - 1) / P.U, wl = ((rl + 1) * P.W - 1) / P.U;
        const unsigned n_cta = (unsigned)(wl / WPB - wf / WPB + 1);
        if (tid == 0) s_flag = atomicAdd(P.cnt + bi, 1u) == n_cta - 1;
        __syncthreads();
        const bool last = s_flag != 0;
        __syncthreads();
        if (!last) continue;
        __threadfence();                           // acquire side of the handshake
        tail_point(P, sm, sm_doubles, bi, wf, wl);
        __threadfence();
        __syncthreads();
        const int b = (int)(bi / P.Next);
        if (tid == 0) s_flag = atomicAdd(P.done + b, 1u) == (unsigned)P.Next - 1;
        __syncthreads();
        const bool fin = s_flag != 0;
        __syncthreads();
        if (fin) {
            __threadfence();
            tail_system(P, sm, b);
            __syncthreads();
        }
    }
}

}  // namespace dse

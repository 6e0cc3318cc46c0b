// dse_tail.cuh -- steps H7 and H8 fused into the point kernel (single-system kernels: dse_point.cu).
//
// A build used to be prep -> point -> contraction -> assemble: three dependent launches whose only job after the point
// kernel is to add up what it produced.  Here the point kernel finishes the build itself, without any CTA ever waiting
// for another one:
//   * every warp keeps ONE record ("slot") per external point it works on: the three z-dependent streams (flushed from
//     registers at the end of the segment), the z-independent contraction H7 over ITS rows, R[j] = sum_q A[q] phi_j(t_q)
//     for the angular sums A[q], and its part of the self-energy sums Pi_G, Pi_Z (H5) -- the slot is private to the warp
//     until the handshake;
//   * every CTA, after its warps have written their slots, bumps ONE arrival counter per external point it worked on
//     (barrier, then fence + atomic by the counting threads);
//   * the CTA whose increment completes the count of an external point e ("last arriver") owns e: it sums e's slots in
//     ascending warp order and forms the four derivative rows of e and 1/G(x_e), 1/Z(x_e);
//   * the owners of the subtraction points x_Z, x_G publish that (counter `rdy`); the owner of a collocation point x_i
//     looks for it -- a BOUNDED number of polls: these owners are running, nobody waits for a CTA that has not been
//     scheduled -- and then writes the rows i and N + i of J and the entries i, N + i of F itself (MOM subtraction rows
//     eq.(14),(15), local terms, the paper's layout eq.(29),(30),(35)): the assembly is spread over as many CTAs as
//     there are external points.  An owner whose polls run out marks its point as pending instead;
//   * every owner bumps the system's counter of finished external points as soon as its polls are over (before it writes
//     its rows: the round trip overlaps them); the CTA that completes it writes the pending rows (normally none) and
//     clears the counters for the next build.
// The counters only decide WHO does a sum, never the order IN a sum: every reduction runs over row / slot indices in a
// fixed order, so J and F are bitwise reproducible.  Data written by other CTAs of the same launch is read with
// ld.global.cg after the counter handshake (L1 is not coherent).
#pragma once
#include "dse_device.cuh"

namespace dse {

// Phase stamps of the single-system build (profiles/r02c_phase_timeline.md): compiled in only with
// -DDSE_PHASE_TIMING (DSE_NVCC_EXTRA=-DDSE_PHASE_TIMING python -m paper_1206_1779_b200.build --force), read back through
// dse_diag_phase_stamps (include/dse_diag.h), printed by `bench.py --phase-timeline`.  One record of PHASE_SLOTS
// %globaltimer values (ns) per warp: 0 kernel entry, 1 table requests issued, 2 H1 done and first barrier passed, 3 point
// phase done, 4 tail entered (CTA barrier), 5 arrival counters done, 6 slot sums + derivative rows written (owners),
// 7 kernel exit, 8 counters cleared (finishing CTA), 9 time inside flush + H7 (sum), 10 segments, 11 subtraction rows
// seen (owners), 13 rows of J, F written (owners).
constexpr int PHASE_SLOTS = 16, PHASE_WARPS = 16, PHASE_CTAS = 148;
#ifdef DSE_PHASE_TIMING
__device__ long long g_phase[PHASE_CTAS * PHASE_WARPS * PHASE_SLOTS];
__device__ __forceinline__ long long phase_now() { long long t; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t)); return t; }
__device__ __forceinline__ long long *phase_rec() { return g_phase + ((size_t)(blockIdx.x % PHASE_CTAS) * PHASE_WARPS + ((threadIdx.x >> 5) % PHASE_WARPS)) * PHASE_SLOTS; }
#define PHASE_STAMP(slot) do { if ((threadIdx.x & 31) == 0) phase_rec()[(slot)] = phase_now(); } while (0)
#define PHASE_ADD(slot, v) do { if ((threadIdx.x & 31) == 0) phase_rec()[(slot)] += (v); } while (0)
#define PHASE_NOW() phase_now()
#else
#define PHASE_STAMP(slot) do { } while (0)
#define PHASE_ADD(slot, v) do { } while (0)
#define PHASE_NOW() 0ll
#endif


// slot of one (warp, external point): [0, 3 Npad) Sa, Sb, Sv accumulated with T_0 = 1; [3 Npad, 6 Npad) Ra, Rb, Rv with the
// table phi (phi_0 = 1/2); then Pi_G, Pi_Z
__host__ __device__ inline int slot_doubles(int Npad) { return 6 * Npad + 2; }

__device__ __forceinline__ double4 ldcg4(const double *p)
{
    const double2 a = __ldcg(reinterpret_cast<const double2 *>(p)), b = __ldcg(reinterpret_cast<const double2 *>(p) + 1);
    return make_double4(a.x, a.y, b.x, b.y);
}

// H5 + H7 of one radial row, called by the whole warp at the end of the row (generic kernel; the pipelined kernel contracts
// all rows of a segment at its end):
// rA, rB, rV = sum_k (u_a, u_b, v), rZ = sum_k (wQ + wM) over the row's angular nodes; phi = phi_j(t_q) of the row.
// The slot belongs to this warp alone, every lane updates its own addresses: plain loads and stores.
__device__ __forceinline__ void slot_row_update(double *slot, int Npad, const double *__restrict__ phi, double rA, double rB,
                                                double rV, double rZ, bool first, int lane)
{
    double *R = slot + 3 * Npad;
    for (int j = lane; j < Npad; j += 32) {
        const double f = __ldg(phi + j);
        double a = 0.0, b = 0.0, v = 0.0;
        if (!first) { a = R[j]; b = R[Npad + j]; v = R[2 * Npad + j]; }
        R[j] = fma(rA, f, a); R[Npad + j] = fma(rB, f, b); R[2 * Npad + j] = fma(rV, f, v);
    }
    if (lane == 0) {
        double g = 0.0, z = 0.0;
        if (!first) { g = slot[6 * Npad]; z = slot[6 * Npad + 1]; }
        slot[6 * Npad] = g + rV; slot[6 * Npad + 1] = z + rZ;
    }
}

// counter bump with release (everything this thread has observed, cumulatively: the slots its CTA wrote before the
// barrier) and acquire (what the CTAs counted before it wrote) semantics at device scope
__device__ __forceinline__ unsigned arrive_acq_rel(unsigned *ctr, unsigned inc = 1u)
{
    unsigned old;
    asm volatile("atom.acq_rel.gpu.global.add.u32 %0, [%1], %2;" : "=r"(old) : "l"(ctr), "r"(inc) : "memory");
    return old;
}

constexpr int TAIL_OWN = 4;            // external points a CTA finishes in one pass
constexpr int TAIL_MLP = 20;           // 16-byte slot loads in flight per thread

// parts a slot sum is split into (a function of the launch configuration only): threads per pair of slot entries
__host__ __device__ inline int tail_parts(int Npad, int threads)
{
    const int p = threads / (slot_doubles(Npad) / 2);
    return p > 1 ? p : 1;
}
// doubles of shared memory the tail needs: the slot sums of TAIL_OWN points and their parts
__host__ __device__ inline int tail_smem_doubles(int Npad, int threads)
{
    const int S = slot_doubles(Npad);
    return TAIL_OWN * S * (1 + tail_parts(Npad, threads));
}

// The derivative rows of the nown <= TAIL_OWN external points own[0..nown) (bi = b * Next + e) from their slots, in one pass.
// own[3 k + 0 .. 2] = (bi, first warp, last warp)
__device__ __noinline__ void tail_points(const KParams &P, double *sm, const int *own, int nown)
{
    const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, warp = tid >> 5, NW = T >> 5;
    const int Npad = P.Npad, N = P.N, SLOT = slot_doubles(Npad);
    double *sS = sm;                               // [nown][SLOT]          slot sums
    double *sX = sm + TAIL_OWN * SLOT;             // [parts][nown][SLOT]   parts of the slot sums
    // 1/G(x_e), 1/Z(x_e) of the collocation points (series eq.(23),(24)): the last warps, one per point
    double invG = 0.0, invZ = 0.0;
    const int myk = NW - 1 - warp;                 // owned point this warp takes the local terms of (if < nown)
    if (myk < nown) {
        const int bi = own[3 * myk], b = bi / P.Next, e = bi - b * P.Next;
        if (e < N) {
            const double *cb = P.c + (size_t)b * 2 * N, *px = P.phi_x + (size_t)e * Npad;
            double lnZ = 0.0, lnG = 0.0;
            for (int jj = lane; jj < N; jj += 32) {
                const double f = __ldg(px + jj);
                lnZ = fma(__ldg(cb + jj), f, lnZ);
                lnG = fma(__ldg(cb + N + jj), f, lnG);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) { lnZ += __shfl_xor_sync(FULL, lnZ, o); lnG += __shfl_xor_sync(FULL, lnG, o); }
            invG = exp(-lnG); invZ = exp(-lnZ);
        }
    }
    // threads = (part, owned point, PAIR of slot entries); every part sums a contiguous range of slots in ascending warp
    // order with all its loads (16 B each) in flight at once: one memory round trip.  The number of parts depends on the
    // launch configuration only -- never on how many points this CTA happens to own (that is decided by arrival order;
    // the grouping of a sum must not be)
    const int HS = SLOT / 2;                       // SLOT is even
    const int work = nown * HS, parts = tail_parts(Npad, T);
    for (int item = tid; item < parts * work; item += T) {
        const int part = item / work, rest = item - part * work, k = rest / HS, idx = rest - k * HS;
        const int bi = own[3 * k], wf = own[3 * k + 1], wl = own[3 * k + 2];
        const int per = (wl - wf + parts) / parts;
        const int w0 = wf + part * per, n = (wl + 1 < w0 + per ? wl + 1 : w0 + per) - w0;
        const double2 *sp = reinterpret_cast<const double2 *>(P.Spart + ((size_t)w0 + (size_t)bi) * SLOT) + idx;
        double2 s = make_double2(0.0, 0.0);
        for (int k0 = 0; k0 < n; k0 += TAIL_MLP) {
            double2 v[TAIL_MLP];
#pragma unroll
            for (int u = 0; u < TAIL_MLP; ++u) v[u] = k0 + u < n ? __ldcg(sp + (size_t)(k0 + u) * HS) : make_double2(0.0, 0.0);
#pragma unroll
            for (int u = 0; u < TAIL_MLP; ++u) { s.x += v[u].x; s.y += v[u].y; }
        }
        reinterpret_cast<double2 *>(sX)[item] = s;
    }
    __syncthreads();
    for (int it = tid; it < work; it += T) {
        double2 s = make_double2(0.0, 0.0);
        for (int p = 0; p < parts; ++p) { const double2 v = reinterpret_cast<const double2 *>(sX)[p * work + it]; s.x += v.x; s.y += v.y; }
        const int k = it / HS, idx = it - k * HS;
        reinterpret_cast<double2 *>(sS + k * SLOT)[idx] = s;
    }
    __syncthreads();
    // dPi_Z/da = Sa + Ra, dPi_Z/db = Sb + Rb, dPi_G/da = Sv, dPi_G/db = Rv (the S streams were accumulated with T_0 = 1;
    // phi_0 = 1/2, eq.(23),(24))
    for (int it = tid; it < nown * Npad; it += T) {
        const int k = it / Npad, jj = it - k * Npad;
        const double *S = sS + k * SLOT;
        double *D = P.Dg + (size_t)own[3 * k] * 4 * Npad;
        const double h = jj == 0 ? 0.5 : 1.0;
        D[jj] = h * S[jj] + S[3 * Npad + jj];
        D[Npad + jj] = h * S[Npad + jj] + S[4 * Npad + jj];
        D[2 * Npad + jj] = h * S[2 * Npad + jj];
        D[3 * Npad + jj] = S[5 * Npad + jj];
    }
    if (myk < nown && lane == 0) {
        double *o = P.PiInv + (size_t)own[3 * myk] * 4;
        const double *S = sS + myk * SLOT;
        o[0] = S[6 * Npad]; o[1] = S[6 * Npad + 1]; o[2] = invG; o[3] = invZ;
    }
}

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned *p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// Rows i = e and N + e of J and entries e, N + e of F for the collocation point bi = b Next + e, e < N (eq.(29),(30),(35),
// (36); MOM subtraction eq.(14),(15)), by the threads j0, j0 + jstride, ... over the columns; every operand is loaded before
// the first store.  Needs the derivative rows and Pi of e and of the subtraction points x_Z, x_G.
__device__ __forceinline__ void tail_point_rows(const KParams &P, int bi, int j0, int jstride)
{
    const int Npad = P.Npad, N = P.N;
    const int b = bi / P.Next, e = bi - b * P.Next;
    if (e >= N) return;
    const size_t bi0 = (size_t)b * P.Next, biZ = bi0 + P.iZ, biG = bi0 + P.iG;
    const double *De = P.Dg + (size_t)bi * 4 * Npad;
    const double *DZ = P.Dg + biZ * 4 * Npad, *DG = P.Dg + biG * 4 * Npad + 2 * Npad;     // rows of x_Z (a, b) and of x_G (a, b)
    double *Jb = P.J + (size_t)b * 4 * N * N, *Fb = P.F + (size_t)b * 2 * N;
    const double4 pi = ldcg4(P.PiInv + (size_t)bi * 4);                                  // Pi_G, Pi_Z, 1/G, 1/Z at x_e
    for (int j = j0; j < N; j += jstride) {
        const double d0 = __ldcg(De + j), d1 = __ldcg(De + Npad + j), d2 = __ldcg(De + 2 * Npad + j), d3 = __ldcg(De + 3 * Npad + j);
        const double sZa = __ldcg(DZ + j), sZb = __ldcg(DZ + Npad + j), sGa = __ldcg(DG + j), sGb = __ldcg(DG + Npad + j);
        const double phi = __ldg(P.phi_x + (size_t)e * Npad + j);
        Jb[(size_t)e * 2 * N + j] = -phi * pi.w - d0 + sZa;
        Jb[(size_t)e * 2 * N + N + j] = -d1 + sZb;
        Jb[(size_t)(N + e) * 2 * N + j] = -d2 + sGa;
        Jb[(size_t)(N + e) * 2 * N + N + j] = -phi * pi.z - d3 + sGb;
    }
    if (j0 == 0) {
        const double PiG_s = __ldcg(P.PiInv + biG * 4), PiZ_s = __ldcg(P.PiInv + biZ * 4 + 1);
        const double gG = __ldg(P.bc + 2 * b + 0), gZ = __ldg(P.bc + 2 * b + 1);
        Fb[e] = pi.w - gZ - pi.y + PiZ_s;          // z(x_i) = 1/Z(x_i) - 1/Z(x_Z) - Pi_Z(x_i) + Pi_Z(x_Z)
        Fb[N + e] = pi.z - gG - pi.x + PiG_s;      // g(x_i) likewise
    }
}

// The CTA that finished the last external point of system b: rows left pending by owners that did not see the
// subtraction points in time (n_pending of them, normally none), then the counters are cleared for the next build on this
// handle.
constexpr unsigned TAIL_PENDING = 1u << 16;        // a pending point counts 1 + TAIL_PENDING on the system's counter
__device__ __noinline__ void tail_finish(const KParams &P, int b, unsigned n_pending)
{
    const int tid = threadIdx.x, T = blockDim.x, PW = (P.Next + 31) / 32;
    const size_t bi0 = (size_t)b * P.Next;
    if (n_pending) {
        for (int wd = 0; wd < PW; ++wd) {
            unsigned m = __ldcg(P.pend + (size_t)b * PW + wd);
            while (m) {
                const int e = 32 * wd + __ffs(m) - 1;
                m &= m - 1;
                tail_point_rows(P, (int)bi0 + e, tid, T);
            }
        }
        __syncthreads();
        for (int wd = tid; wd < PW; wd += T) P.pend[(size_t)b * PW + wd] = 0u;
    }
    for (int e = tid; e < P.Next; e += T) P.cnt[bi0 + e] = 0u;
    if (tid == 0) { P.done[b] = 0u; P.rdy[b] = 0u; }
}

// Called by ALL threads of the CTA after its warps' last slot updates.  P.tail_cta[2 c], [2 c + 1] = first and last external
// point index CTA c works on (last < first: none); P.tail_bi[2 bi], [2 bi + 1] = first and last warp that works on bi (both
// tables are built by dse_create from the same partition formula the kernels use).  sm = the CTA's dynamic shared memory.
__device__ __forceinline__ void build_tail(const KParams &P, double *sm)
{
    __shared__ unsigned s_mask, s_fin;
    __shared__ int s_own[3 * TAIL_OWN], s_w[64];
    __shared__ unsigned s_pend[TAIL_OWN];
    const int tid = threadIdx.x, lane = tid & 31, WPB = blockDim.x >> 5, T = blockDim.x;
    const int bi_lo = P.tail_cta[2 * blockIdx.x], bi_hi = P.tail_cta[2 * blockIdx.x + 1];
    __syncthreads();                               // the slots of every warp of this CTA are written (CTA scope) ...
    PHASE_STAMP(4);
    for (int seg0 = bi_lo; seg0 <= bi_hi; seg0 += 32) {
        if (tid < 32) {
            const int bi = seg0 + lane;
            bool last = false;
            if (bi <= bi_hi) {
                const int wf = P.tail_bi[2 * bi], wl = P.tail_bi[2 * bi + 1];
                s_w[2 * lane] = wf; s_w[2 * lane + 1] = wl;
                const unsigned n_cta = (unsigned)(wl / WPB - wf / WPB + 1);
                last = arrive_acq_rel(P.cnt + bi) == n_cta - 1;      // ... and, by the release, device-wide; acquire: the
                                                                     // other CTAs' slots are visible after the count
            }
            const unsigned m = __ballot_sync(FULL, last);
            if (lane == 0) s_mask = m;
        }
        __syncthreads();
        PHASE_STAMP(5);
        unsigned mask = s_mask;                    // external points this CTA arrived last at (usually none or one)
        while (mask) {
            __syncthreads();                       // (s_own, s_mask and the shared memory of the pass before are free)
            int nown = 0;
            for (unsigned m2 = mask; m2 && nown < TAIL_OWN; m2 &= m2 - 1, ++nown)
                if (tid == 0) {
                    const int l = __ffs(m2) - 1;
                    s_own[3 * nown] = seg0 + l; s_own[3 * nown + 1] = s_w[2 * l]; s_own[3 * nown + 2] = s_w[2 * l + 1];
                }
            for (int k = 0; k < nown; ++k) mask &= mask - 1;
            __syncthreads();
            tail_points(P, sm, s_own, nown);
            __syncthreads();                       // D rows, Pi, 1/G, 1/Z of the owned points are written
            PHASE_STAMP(6);
            if (tid < 32) {
                // owners of x_Z, x_G publish; owners of collocation points look for both -- at most P.tail_polls times
                bool ok = false;
                int b = 0, e = P.N;
                if (lane < nown) {
                    b = s_own[3 * lane] / P.Next; e = s_own[3 * lane] - b * P.Next;
                    if (e == P.iZ || e == P.iG) arrive_acq_rel(P.rdy + b);
                }
                if (e < P.N) {
                    const unsigned nsub = P.iZ == P.iG ? 1u : 2u;
                    for (int it = 0; it < P.tail_polls && !ok; ++it) {
                        ok = ld_acquire_u32(P.rdy + b) >= nsub;
                        if (!ok) __nanosleep(64);
                    }
                    if (!ok) atomicOr(P.pend + (size_t)b * ((P.Next + 31) / 32) + (e >> 5), 1u << (e & 31));
                }
                const unsigned m = __ballot_sync(FULL, ok);
                if (lane == 0) s_mask = m;
            }
            __syncthreads();
            PHASE_STAMP(11);
            const unsigned okm = s_mask;           // owned collocation points whose rows this CTA writes now
            if (tid >= T - 32) {
                // the LAST warp: one count per owned point on its system's counter -- now, not after the rows: the counter
                // only has to follow the polls (it triggers the clearing of the counters the polls read) and the derivative
                // rows that a pending point leaves to the finishing CTA; its round trip overlaps the other warps' rows
                bool fin = false;
                if (lane < nown) {
                    const int b = s_own[3 * lane] / P.Next, e = s_own[3 * lane] - b * P.Next;
                    const bool pending = e < P.N && !((okm >> lane) & 1u);
                    const unsigned total = arrive_acq_rel(P.done + b, pending ? 1u + TAIL_PENDING : 1u) + 1u + (pending ? TAIL_PENDING : 0u);
                    fin = (total & (TAIL_PENDING - 1u)) == (unsigned)P.Next;
                    s_pend[lane] = total / TAIL_PENDING;
                }
                const unsigned mf = __ballot_sync(FULL, fin);
                if (lane == 0) s_fin = mf;
            }
            {
                const int G = T / P.Npad > 0 ? T / P.Npad : 1, g = tid / P.Npad, j = tid - g * P.Npad;
                for (int k = g; k < nown; k += G)
                    if (g < G && ((okm >> k) & 1u)) tail_point_rows(P, s_own[3 * k], j, P.Npad);
            }
            PHASE_STAMP(13);
            __syncthreads();
            unsigned fmask = s_fin;
            while (fmask) {                        // systems whose last external point this CTA finished
                const int l = __ffs(fmask) - 1;
                fmask &= fmask - 1;
                tail_finish(P, s_own[3 * l] / P.Next, s_pend[l]);
                PHASE_STAMP(8);
            }
        }
        __syncthreads();
    }
    PHASE_STAMP(7);
}

}  // namespace dse

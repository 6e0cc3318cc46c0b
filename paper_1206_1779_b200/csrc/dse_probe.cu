// dse_probe.cu -- fp64 throughput probes (include/dse_diag.h): the roofline denominators of an ALU-bound path and the
// micro-measurements DESIGN.md section 6 refers to.  Not part of the method.
#include <cuda_runtime.h>

#include "dse_internal.h"

namespace dse {

namespace {

constexpr int PROBE_THREADS = 256;

// 8 dependent chains, multiplier and addend are constants: every DFMA has two register operands at most
__global__ void __launch_bounds__(PROBE_THREADS) probe_dfma(int iters, double *sink)
{
    double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6,
           a7 = a0 + 7;
    const double m = 0.999999999, c = 1e-9;
    for (int i = 0; i < iters; ++i) {
        a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
        a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
    sink[blockIdx.x * (size_t)blockDim.x + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}

__device__ __forceinline__ void dmma(double &c0, double &c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(PROBE_THREADS) probe_dmma(int iters, double *sink)
{
    double c[4][2];
    for (int m = 0; m < 4; ++m) { c[m][0] = threadIdx.x * 1e-9; c[m][1] = m; }
    const double a = 1e-3 * (threadIdx.x & 7), b = 1e-3 * (threadIdx.x & 3);
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int m = 0; m < 4; ++m) dmma(c[m][0], c[m][1], a, b);
    }
    double s = 0;
    for (int m = 0; m < 4; ++m) s += c[m][0] + c[m][1];
    sink[blockIdx.x * (size_t)blockDim.x + threadIdx.x] = s;
}

// acc_i = fma(w_i, t_i, acc_i), i = 0..7 per iteration.  REUSE = false: w_i and t_i are 16 different registers, so no
// operand of an FMA equals the operand in the same slot of the one before (nothing for the operand reuse cache);
// REUSE = true: one w for all eight (the same register in the same slot of consecutive FMAs).  Inline asm keeps ptxas
// from re-associating; the registers are made opaque so that nothing is constant-folded.
template <bool REUSE>
__global__ void __launch_bounds__(PROBE_THREADS) probe_dfma_3reg(int iters, double *sink)
{
    double acc[8], w[8], t[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        acc[i] = threadIdx.x * 1e-9 + i; w[i] = 1e-9 * (i + 1) + threadIdx.x * 1e-12; t[i] = 0.5 + 1e-3 * i;
        asm volatile("" : "+d"(w[i]), "+d"(t[i]));
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(acc[i]) : "d"(REUSE ? w[0] : w[i]), "d"(t[i]));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += acc[i];
    sink[blockIdx.x * (size_t)blockDim.x + threadIdx.x] = s;
}

// 8 DFMA chains + 4 DMMA chains per warp, interleaved 2 : 1 in the instruction stream
__global__ void __launch_bounds__(PROBE_THREADS) probe_dfma_dmma(int iters, double *sink)
{
    double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    double c[4][2];
    for (int m = 0; m < 4; ++m) { c[m][0] = threadIdx.x * 1e-9; c[m][1] = m; }
    const double fa = 1e-3 * (threadIdx.x & 7), fb = 1e-3 * (threadIdx.x & 3);
    const double m = 0.999999999, cc = 1e-9;
    for (int i = 0; i < iters; ++i) {
        a0 = fma(a0, m, cc); a1 = fma(a1, m, cc); dmma(c[0][0], c[0][1], fa, fb);
        a2 = fma(a2, m, cc); a3 = fma(a3, m, cc); dmma(c[1][0], c[1][1], fa, fb);
        a4 = fma(a4, m, cc); a5 = fma(a5, m, cc); dmma(c[2][0], c[2][1], fa, fb);
        a6 = fma(a6, m, cc); a7 = fma(a7, m, cc); dmma(c[3][0], c[3][1], fa, fb);
    }
    double s = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    for (int mm = 0; mm < 4; ++mm) s += c[mm][0] + c[mm][1];
    sink[blockIdx.x * (size_t)blockDim.x + threadIdx.x] = s;
}

// acc_j += w * T_j, j = 0..7, with every T_j read from shared memory (conflict-free: one 64-bit word per lane and j)
__global__ void __launch_bounds__(PROBE_THREADS) probe_dfma_lds(int iters, double *sink)
{
    __shared__ double sT[8][PROBE_THREADS];
    for (int j = 0; j < 8; ++j) sT[j][threadIdx.x] = 0.5 + 1e-3 * j + 1e-9 * threadIdx.x;
    __syncthreads();
    double acc[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) acc[j] = j;
    double w = 1e-9 * threadIdx.x;
    asm volatile("" : "+d"(w));
    const volatile double *vt = &sT[0][threadIdx.x];
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[j] = fma(w, vt[j * PROBE_THREADS], acc[j]);
    }
    double s = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) s += acc[j];
    sink[blockIdx.x * (size_t)blockDim.x + threadIdx.x] = s;
}

// Dependent-chain latencies of the warp collectives the LU's pivot search chooses between (one warp; sink[0] receives the
// cycles per iteration, including the one integer add that closes the chain): the winner of a search hands its value to the
// other lanes either through ballot -> lane index -> shuffle or through a REDUX over masked words.
template <int OP>
__global__ void __launch_bounds__(32) probe_latency(int iters, double *sink)
{
    const int lane = threadIdx.x;
    unsigned x = 12345u + 7u * lane;
    double d = 1.25 + 1e-3 * lane;
    const long long t0 = clock64();
#pragma unroll 8
    for (int i = 0; i < iters; ++i) {
        if (OP == 0) x = __reduce_max_sync(0xffffffffu, x) + lane;
        if (OP == 1) x = __reduce_or_sync(0xffffffffu, x & (lane + i)) + 1u;
        if (OP == 2) x = __shfl_sync(0xffffffffu, x, __ffs(__ballot_sync(0xffffffffu, (x & 1u) != 0u) | 0x80000000u) - 1) + lane;
        if (OP == 3) x = __shfl_sync(0xffffffffu, x, (x + 1u) & 31u) + 1u;
        if (OP == 4) d = fma(d, 1.0000001, 0.5);
    }
    const long long t1 = clock64();
    if (lane == 0) sink[0] = (double)(t1 - t0) / iters;
    if (x == 0xdeadbeefu || d == 1.5) sink[1] = 1.0;      // (keeps both chains alive)
}

}  // namespace

int launch_probe(int kind, int blocks, int iters, double *sink, void *stream)
{
    cudaStream_t s = (cudaStream_t)stream;
    switch (kind) {
        case DSE_PROBE_DFMA: probe_dfma<<<blocks, PROBE_THREADS, 0, s>>>(iters, sink); break;
        case DSE_PROBE_DMMA: probe_dmma<<<blocks, PROBE_THREADS, 0, s>>>(iters, sink); break;
        case DSE_PROBE_DFMA_3REG: probe_dfma_3reg<false><<<blocks, PROBE_THREADS, 0, s>>>(iters, sink); break;
        case DSE_PROBE_DFMA_REUSE: probe_dfma_3reg<true><<<blocks, PROBE_THREADS, 0, s>>>(iters, sink); break;
        case DSE_PROBE_DFMA_DMMA: probe_dfma_dmma<<<blocks, PROBE_THREADS, 0, s>>>(iters, sink); break;
        case DSE_PROBE_DFMA_LDS: probe_dfma_lds<<<blocks, PROBE_THREADS, 0, s>>>(iters, sink); break;
        case DSE_PROBE_LAT_REDUX_MAX: probe_latency<0><<<1, 32, 0, s>>>(iters, sink); break;
        case DSE_PROBE_LAT_REDUX_OR: probe_latency<1><<<1, 32, 0, s>>>(iters, sink); break;
        case DSE_PROBE_LAT_BALLOT_FFS_SHFL: probe_latency<2><<<1, 32, 0, s>>>(iters, sink); break;
        case DSE_PROBE_LAT_SHFL: probe_latency<3><<<1, 32, 0, s>>>(iters, sink); break;
        case DSE_PROBE_LAT_DFMA: probe_latency<4><<<1, 32, 0, s>>>(iters, sink); break;
        default: return DSE_EINVAL;
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "probe launch");
    return 1;
}

}  // namespace dse

extern "C" {

int dse_probe(int32_t kind, int32_t blocks, int32_t iters, double *sink_dev, void *stream)
{
    if (blocks < 1 || iters < 1 || !sink_dev) return DSE_EINVAL;
    const int rc = dse::launch_probe(kind, blocks, iters, sink_dev, stream);
    return rc < 0 ? rc : DSE_OK;
}

double dse_probe_flops(int32_t kind, int32_t blocks, int32_t iters)
{
    const double thr = (double)blocks * dse::PROBE_THREADS, warps = thr / 32.0, it = (double)iters;
    switch (kind) {
        case DSE_PROBE_DFMA: case DSE_PROBE_DFMA_3REG: case DSE_PROBE_DFMA_REUSE: case DSE_PROBE_DFMA_LDS:
            return thr * 8.0 * it * 2.0;
        case DSE_PROBE_DMMA: return warps * 4.0 * it * 512.0;
        case DSE_PROBE_DFMA_DMMA: return thr * 8.0 * it * 2.0 + warps * 4.0 * it * 512.0;
        default: return 0.0;
    }
}

}  // extern "C"

/*
 * dse_diag.h -- diagnostics of libdse_b200.so that are NOT part of the method's boundary (include/dse.h):
 * fp64 throughput probes.  They supply the roofline denominators bench.py reports against
 * (MEASURED_PEAKS.json has no fp64 entry) and reproduce the three micro-measurements DESIGN.md section 6 leans on.
 * `stream` is a cudaStream_t passed as void*; sink_dev is a DEVICE pointer owned by the caller.
 */
#ifndef DSE_DIAG_H_
#define DSE_DIAG_H_

#include "dse.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Probe kinds.  Every probe launches `blocks` CTAs of 256 threads; each thread runs `iters` iterations of an unrolled body
 * of independent dependent-chains, so the issue rate of the named instruction mix is what is measured.
 * dse_probe_flops(kind, blocks, iters) returns the floating-point operations of one launch (FMA = 2, an m8n8k4 MMA = 512
 * per warp). */
#define DSE_PROBE_DFMA 0        /* 8 chains of DFMA whose multiplier and addend are immediates/constants (2 register operands) */
#define DSE_PROBE_DMMA 1        /* 4 chains of mma.sync.m8n8k4.f64 per warp (fp64 tensor path)                               */
#define DSE_PROBE_DFMA_3REG 2   /* 8 chains of DFMA with three DISTINCT register operands, none reusable from the previous
                                   instruction (acc_i = fma(w_i, t_i, acc_i), w and t rotate): the operand mix of the phase-2
                                   accumulations of the point kernel                                                        */
#define DSE_PROBE_DFMA_REUSE 3  /* as 2, but consecutive FMAs share one register operand in the same slot (operand reuse cache) */
#define DSE_PROBE_DFMA_DMMA 4   /* independent DFMA chains and DMMA chains interleaved in one warp: do the two share a unit? */
#define DSE_PROBE_DFMA_LDS 5    /* acc_j += w * T_j with EVERY T_j read from shared memory (the "stash all T_j" alternative to
                                   re-running the recurrence in phase 2): 1 LDS.64 per DFMA                                  */

/* Latency probes: ONE warp runs `iters` iterations of a dependent chain and writes the clock cycles per iteration to
 * sink_dev[0] (`blocks` is ignored; dse_probe_flops returns 0).  They are the measurements behind the LU's pivot search
 * (csrc/dse_lu.cu): how a winner lane's value reaches the other lanes. */
#define DSE_PROBE_LAT_REDUX_MAX 6        /* x = redux.max(x) + lane                                   */
#define DSE_PROBE_LAT_REDUX_OR 7         /* x = redux.or(x & m) + 1                                   */
#define DSE_PROBE_LAT_BALLOT_FFS_SHFL 8  /* x = shfl(x, ffs(ballot(p)) - 1) + lane: the textbook broadcast */
#define DSE_PROBE_LAT_SHFL 9             /* x = shfl(x, f(x)) + 1                                     */
#define DSE_PROBE_LAT_DFMA 10            /* d = fma(d, a, b)                                          */

/* sink_dev receives one double per thread (>= blocks * 256).  Asynchronous on `stream`. */
DSE_API int dse_probe(int32_t kind, int32_t blocks, int32_t iters, double *sink_dev, void *stream);
DSE_API double dse_probe_flops(int32_t kind, int32_t blocks, int32_t iters);

/* The fused tail of a single-system Jacobian build (csrc/dse_tail.cuh): the CTA that owns a collocation point looks at most
 * `polls` times for the rows of the subtraction points x_Z, x_G before it leaves its rows of J and F to the CTA that
 * finishes the system.  Default 4096; 0 sends every point down that fallback path (tests use it to cover the path).
 * Applies to the builds launched after the call. */
DSE_API int dse_diag_set_tail_polls(dse_handle *h, int32_t polls);

/* Phase stamps of the last single-system Jacobian build (which = 0: %globaltimer ns, [148 CTAs][16 warps][16 slots], slot
 * meanings in csrc/dse_tail.cuh) or of the last one-CTA LU (which = 1: clock64 of system 0, layout in csrc/dse_lu.cu), copied
 * to a HOST array.  The stamps exist only in a library built with -DDSE_PHASE_TIMING
 * (DSE_NVCC_EXTRA=-DDSE_PHASE_TIMING python -m paper_1206_1779_b200.build --force); otherwise DSE_EINVAL.  Returns the number
 * of words copied.  Synchronises the device.  `python bench.py --phase-timeline` prints the tables of DESIGN.md section 6
 * from them (profiles/r02c_phase_timeline.md). */
DSE_API int dse_diag_phase_stamps(int32_t which, int64_t *out_host, int32_t max_words);

#ifdef __cplusplus
}
#endif
#endif /* DSE_DIAG_H_ */

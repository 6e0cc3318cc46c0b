// dse_solve.cu -- dse_newton_solve: the whole Newton-Raphson iteration (eq.(31)-(35), L226) as ONE CUDA graph.
//
// The graph is a single WHILE conditional node.  Its body is captured from the same launchers that dse_newton_step
// uses (prep -> point kernel -> contraction -> assemble -> LU writing Delta) followed by solve_control_kernel, which
// applies the under-relaxed update per system, records the per-system state and decides on the device
// (cudaGraphSetConditional) whether the body runs again.  The host enqueues: solve_init_kernel (scalars of this call
// -> control block), the graph, and two device-to-device copies; it never waits for a step.
#include <cuda_runtime.h>

#include <cstdio>
#include <new>

#include "dse_internal.h"

namespace dse {

namespace {

constexpr int CTL_RHO = 0, CTL_CAP = 1, CTL_TOL = 2, CTL_MAXIT = 3, CTL_ITER = 4;
constexpr int INFO = 6;       // doubles per system in info

int fail(cudaError_t e, const char *what)
{
    char buf[256];
    snprintf(buf, sizeof(buf), "%s: %s", what, cudaGetErrorString(e));
    set_error_text(buf);
    return DSE_ECUDA;
}

__global__ void solve_init_kernel(double *ctl, double *info, int B, double rho, double cap, double tol, int max_iter)
{
    if (threadIdx.x == 0) {
        ctl[CTL_RHO] = rho; ctl[CTL_CAP] = cap; ctl[CTL_TOL] = tol; ctl[CTL_MAXIT] = (double)max_iter; ctl[CTL_ITER] = 0.0;
    }
    for (int b = threadIdx.x; b < B; b += blockDim.x) {
        double *o = info + (size_t)b * INFO;
        o[0] = 0.0; o[1] = 0.0; o[2] = 0.0; o[3] = __longlong_as_double(0x7ff0000000000000ll); o[4] = 0.0; o[5] = 0.0;
    }
}

// One CTA; warp per system.  stats[b] = { |Delta|inf, |F|inf row-scaled, min|pivot|, growth } from the LU kernel.
__global__ void __launch_bounds__(256) solve_control_kernel(cudaGraphConditionalHandle hc, double *ctl, int n2, int B,
                                                            const double *__restrict__ delta, const double *__restrict__ stats,
                                                            double *__restrict__ c, double *__restrict__ info)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, NW = blockDim.x >> 5;
    const double rho = ctl[CTL_RHO], cap = ctl[CTL_CAP], tol = ctl[CTL_TOL];
    const int it = (int)ctl[CTL_ITER] + 1, max_iter = (int)ctl[CTL_MAXIT];
    int open = 0;                                         // systems of this warp that want another step
    for (int b = warp; b < B; b += NW) {
        double *o = info + (size_t)b * INFO;
        if (o[5] != 0.0) continue;                        // frozen: converged or failed earlier
        const double *st = stats + (size_t)b * 4;
        const double dmax = st[0];
        const double INF = __longlong_as_double(0x7ff0000000000000ll);
        bool bad = false;                                 // fmax() skips NaN: look at every entry of Delta as well
        for (int j = lane; j < n2; j += 32) { const double dj = delta[(size_t)b * n2 + j]; bad = bad || !(fabs(dj) < INF); }
        const bool finite = dmax == dmax && dmax < INF && !__any_sync(0xffffffffu, bad);
        double r = rho;
        if (finite && cap > 0.0 && rho * dmax > cap) r = cap / dmax;      // rho_n = min(rho, cap/|Delta|)
        if (finite)
            for (int j = lane; j < n2; j += 32) c[(size_t)b * n2 + j] -= r * delta[(size_t)b * n2 + j];   // eq.(31),(32)
        const double status = !finite ? -1.0 : (dmax < tol ? 1.0 : 0.0);
        __syncwarp();
        if (lane == 0) {
            o[0] = (double)it; o[1] = dmax; o[2] = st[1]; o[3] = fmin(o[3], st[2]); o[4] = finite ? r : 0.0; o[5] = status;
        }
        if (status == 0.0) open = 1;
    }
    const int any = __syncthreads_or(open);
    if (threadIdx.x == 0) {
        ctl[CTL_ITER] = (double)it;
        cudaGraphSetConditional(hc, (any && it < max_iter) ? 1u : 0u);
    }
}

}  // namespace

struct SolveGraph {
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    double *ctl = nullptr, *info = nullptr;
    int B = 0, body_kernels = 0;
};

void solve_graph_destroy(SolveGraph *g)
{
    if (!g) return;
    if (g->exec) cudaGraphExecDestroy(g->exec);
    if (g->graph) cudaGraphDestroy(g->graph);
    delete g;
}

int solve_graph_create(const KParams &k, const PointKernelConfig &cfg, double *c, const double *bc, double *J, double *F,
                       double *delta, double *stats, double *lu_scratch, double *ctl, double *info, SolveGraph **out)
{
    SolveGraph *g = new (std::nothrow) SolveGraph();
    if (!g) return DSE_ENOMEM;
    g->ctl = ctl; g->info = info; g->B = k.B;
    cudaStream_t cap = nullptr;
    cudaError_t e = cudaGraphCreate(&g->graph, 0);
    if (e != cudaSuccess) { solve_graph_destroy(g); return fail(e, "cudaGraphCreate"); }
    cudaGraphConditionalHandle hc;
    e = cudaGraphConditionalHandleCreate(&hc, g->graph, 1, cudaGraphCondAssignDefault);      // first pass always runs
    if (e != cudaSuccess) { solve_graph_destroy(g); return fail(e, "cudaGraphConditionalHandleCreate"); }
    cudaGraphNodeParams np = {};
    np.type = cudaGraphNodeTypeConditional;
    np.conditional.handle = hc;
    np.conditional.type = cudaGraphCondTypeWhile;
    np.conditional.size = 1;
    cudaGraphNode_t node;
    e = cudaGraphAddNode(&node, g->graph, nullptr, 0, &np);
    if (e != cudaSuccess) { solve_graph_destroy(g); return fail(e, "cudaGraphAddNode(while)"); }
    cudaGraph_t body = np.conditional.phGraph_out[0];
    e = cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking);
    if (e != cudaSuccess) { solve_graph_destroy(g); return fail(e, "cudaStreamCreate(capture)"); }
    e = cudaStreamBeginCaptureToGraph(cap, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) { cudaStreamDestroy(cap); solve_graph_destroy(g); return fail(e, "cudaStreamBeginCaptureToGraph"); }
    int rc = launch_build(k, cfg, c, bc, J, F, cap);
    int n = rc;
    if (rc >= 0) {
        rc = launch_lu(2 * k.N, k.B, J, F, delta, nullptr, 0.0, stats, lu_scratch, cap);
        n += rc;
    }
    if (rc >= 0) {
        solve_control_kernel<<<1, 256, 0, cap>>>(hc, ctl, 2 * k.N, k.B, delta, stats, c, info);
        ++n;
    }
    cudaGraph_t captured = nullptr;
    e = cudaStreamEndCapture(cap, &captured);
    cudaStreamDestroy(cap);
    if (rc < 0) { solve_graph_destroy(g); return rc; }
    if (e != cudaSuccess) { solve_graph_destroy(g); return fail(e, "cudaStreamEndCapture"); }
    g->body_kernels = n;
    e = cudaGraphInstantiate(&g->exec, g->graph, 0);
    if (e != cudaSuccess) { solve_graph_destroy(g); return fail(e, "cudaGraphInstantiate"); }
    *out = g;
    return DSE_OK;
}

// returns the number of kernels launched at least (init + one pass of the body) or < 0
int launch_solve(SolveGraph *g, double rho, double cap, double tol, int max_iter, void *stream)
{
    cudaStream_t s = (cudaStream_t)stream;
    solve_init_kernel<<<1, 256, 0, s>>>(g->ctl, g->info, g->B, rho, cap, tol, max_iter);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(e, "solve_init launch");
    e = cudaGraphLaunch(g->exec, s);
    if (e != cudaSuccess) return fail(e, "cudaGraphLaunch(newton solve)");
    return 1 + g->body_kernels;
}

}  // namespace dse

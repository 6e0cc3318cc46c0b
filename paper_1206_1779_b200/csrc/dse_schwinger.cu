// dse_schwinger.cu -- NEXT f4: the paper's second GPU workload (Table 2):
// the Schwinger function of the gluon propagator, eq.(20),
//     Delta(t) = (1/pi) int_0^inf d|p| cos(t|p|) Z(p^2)/p^2 ,
// as a batched cosine-weighted dot product over a mapped Gauss-Legendre rule with 2^17 nodes whose nodes and
// weights are generated on the device ("the main improvements can be obtained from a parallelized generation
// of the nodes and weights", L382).  Reading A22: nodes in u = ln|p| on [ln sqrt(p2_min), ln sqrt(p2_max)].
//
//   gl_prepare_kernel   recurrence coefficients (2m-1)/m, (m-1)/m
//   gl_nodes_kernel     one thread per pair of nodes of the non-negative half: Newton iteration on the Legendre
//                       three-term recurrence (O(n) per evaluation, O(n^2) in total: the compute-bound part)
//   schwinger_prepare   p_i, f_i = w_i (du/2) p_i Z(p_i^2)/p_i^2 per node and system (series + continuation O2)
//   schwinger_kernel    one CTA per (t_m, system): fixed-order strided sum of f_i cos(t_m p_i)
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <mutex>

#include "dse_internal.h"

namespace dse {

namespace {

constexpr double PI_D = 3.14159265358979323846;

__global__ void gl_prepare_kernel(int n, double2 *__restrict__ ab)
{
    for (int m = blockIdx.x * blockDim.x + threadIdx.x; m <= n; m += gridDim.x * blockDim.x) {
        const double im = m > 0 ? 1.0 / (double)m : 0.0;
        ab[m] = make_double2((2.0 * m - 1.0) * im, (m - 1.0) * im);      // A_m = (2m-1)/m, B_m = (m-1)/m
    }
}

// P_n(x) and P_{n-1}(x) for two abscissae at once (two independent chains per thread).  One warp per CTA: the
// recurrence coefficients (2 MB at n = 2^17: L2-resident, ~300 cycles away) are staged through shared memory in chunks
// of GL_CHUNK entries with a cp.async double buffer, so the loop only sees shared-memory latency.
constexpr int GL_CHUNK = 512;
__device__ __forceinline__ void legendre2(int n, const double2 *__restrict__ ab, double2 *s_ab /*[2][GL_CHUNK]*/,
                                          double xa, double xb, double &pa, double &pam, double &pb, double &pbm)
{
    const int lane = threadIdx.x;
    auto stage = [&](int chunk, int buf) {                       // entries m = 2 + chunk * GL_CHUNK + i
        const int m0 = 2 + chunk * GL_CHUNK;
        for (int i = lane; i < GL_CHUNK; i += 32) {
            const int m = min(m0 + i, n);                        // (clamped: entries past n are never used)
            const unsigned dst = (unsigned)__cvta_generic_to_shared(s_ab + buf * GL_CHUNK + i);
            asm volatile("cp.async.ca.shared.global [%0], [%1], 16;\n" ::"r"(dst), "l"(ab + m));
        }
        asm volatile("cp.async.commit_group;\n" ::);
    };
    double a0 = 1.0, a1 = xa, b0 = 1.0, b1 = xb;
    const int nchunks = (n - 1 + GL_CHUNK - 1) / GL_CHUNK;       // steps m = 2 .. n
    if (nchunks > 0) stage(0, 0);
    for (int ch = 0; ch < nchunks; ++ch) {
        if (ch + 1 < nchunks) stage(ch + 1, (ch + 1) & 1);
        else asm volatile("cp.async.commit_group;\n" ::);
        asm volatile("cp.async.wait_group 1;\n" ::: "memory");
        __syncwarp();
        const double2 *cur = s_ab + (ch & 1) * GL_CHUNK;
        const int cnt = min(GL_CHUNK, n - 1 - ch * GL_CHUNK);
#pragma unroll 8
        for (int i = 0; i < cnt; ++i) {
            const double2 c = cur[i];
            const double a2 = fma(c.x * xa, a1, -c.y * a0);
            const double b2 = fma(c.x * xb, b1, -c.y * b0);
            a0 = a1; a1 = a2; b0 = b1; b1 = b2;
        }
        __syncwarp();                                            // the buffer is restaged two chunks later
    }
    asm volatile("cp.async.wait_group 0;\n" ::: "memory");
    pa = a1; pam = a0; pb = b1; pbm = b0;
}

// nodes ascending in (-1, 1); thread t handles the nodes i = t and i = t + q (q = quarter) of the upper half and
// mirrors them.  Newton on P_n with P_n' = n (x P_n - P_{n-1}) / (x^2 - 1); weight 2 / ((1 - x^2) P_n'^2).
__global__ void __launch_bounds__(32) gl_nodes_kernel(int n, const double2 *__restrict__ ab, double *__restrict__ x,
                                                       double *__restrict__ w)
{
    __shared__ __align__(16) double2 s_ab[2 * GL_CHUNK];
    const int half = (n + 1) / 2;                 // number of non-negative nodes
    const int q = (half + 1) / 2;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = t < q;                     // (all lanes stay: the coefficient staging is warp-wide)
    // k-th largest root (k = 0 is the largest): Tricomi-type starting value
    const int ka = min(t, half - 1), kb = min(t + q, half - 1);
    double xa = (1.0 - (n - 1.0) / (8.0 * n * (double)n * n)) * cospi((4.0 * ka + 3.0) / (4.0 * n + 2.0));
    double xb = (1.0 - (n - 1.0) / (8.0 * n * (double)n * n)) * cospi((4.0 * kb + 3.0) / (4.0 * n + 2.0));
    double pa, pam, pb, pbm, da = 1.0, db = 1.0;
    // Newton converges quadratically: once a step is below 1e-14 the node is exact to rounding after it (the error
    // left is ~step^2).  Demanding |step| <= 1e-16 never triggered at n = 2^17 -- the O(n eps) noise of the recurrence
    // keeps the steps at ~1e-15 -- and ran all 12 iterations.
    bool live_a = true, live_b = true;
    for (int it = 0; it < 12 && __any_sync(0xffffffffu, live_a || live_b); ++it) {      // warp-uniform trip count
        legendre2(n, ab, s_ab, xa, xb, pa, pam, pb, pbm);
        da = n * (xa * pa - pam) / (xa * xa - 1.0);
        db = n * (xb * pb - pbm) / (xb * xb - 1.0);
        const double sa = pa / da, sb = pb / db;
        if (live_a) { xa -= sa; live_a = fabs(sa) > 1e-14; }
        if (live_b) { xb -= sb; live_b = fabs(sb) > 1e-14; }
    }
    legendre2(n, ab, s_ab, xa, xb, pa, pam, pb, pbm);
    da = n * (xa * pa - pam) / (xa * xa - 1.0);
    db = n * (xb * pb - pbm) / (xb * xb - 1.0);
    const double wa = 2.0 / ((1.0 - xa * xa) * da * da), wb = 2.0 / ((1.0 - xb * xb) * db * db);
    if ((n & 1) && ka == half - 1) xa = 0.0;      // the middle node of an odd rule
    if ((n & 1) && kb == half - 1) xb = 0.0;
    if (!valid) return;
    x[n - 1 - ka] = xa; w[n - 1 - ka] = wa; x[ka] = -xa; w[ka] = wa;
    x[n - 1 - kb] = xb; w[n - 1 - kb] = wb; x[kb] = -xb; w[kb] = wb;
}

// per node i and system b:  p_i = exp(u_i),  f_i = w_i (u1-u0)/2 * p_i * Z(p_i^2)/p_i^2   (d|p| = |p| du)
__global__ void schwinger_prepare(const KParams P, const double *__restrict__ c, int n, double u0, double u1,
                                  const double *__restrict__ x, const double *__restrict__ w, double *__restrict__ p,
                                  double *__restrict__ f)
{
    const int b = blockIdx.y;
    const double *a = c + (size_t)b * 2 * P.N;             // a_j <-> ln Z
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const double u = u0 + 0.5 * (x[i] + 1.0) * (u1 - u0);
        const double pp = exp(u);
        const double z = pp * pp;
        // O2: series on the clamped argument + continuation (eq.(16),(19))
        const double ell = log(z * P.inv_eps2);
        double s = fma(ell, P.two_over_Lg, -1.0), EZ = 0.0;
        if (z < P.eps2) { EZ = P.pZ * ell; s = -1.0; }
        else if (z > P.L2) { EZ = P.gamma * log(fma(P.omega, ell - P.Lg, 1.0)); s = 1.0; }
        s = fmin(1.0, fmax(-1.0, s));
        double tm = 1.0, t = s, lnZ = 0.5 * a[0] + (P.N > 1 ? a[1] * s : 0.0);
        for (int j = 2; j < P.N; ++j) {
            const double tn = fma(2.0 * s, t, -tm);
            tm = t; t = tn;
            lnZ = fma(a[j], tn, lnZ);
        }
        if (b == 0) p[i] = pp;
        f[(size_t)b * n + i] = w[i] * (0.5 * (u1 - u0)) * exp(lnZ + EZ) / pp;
    }
}

__global__ void __launch_bounds__(256) schwinger_kernel(int n, int n_t, const double *__restrict__ t,
                                                        const double *__restrict__ p, const double *__restrict__ f,
                                                        double *__restrict__ out)
{
    __shared__ double s_part[8];
    const int m = blockIdx.x, b = blockIdx.y;
    const double tm = t[m];
    const double *fb = f + (size_t)b * n;
    double acc0 = 0.0, acc1 = 0.0;
    int i = threadIdx.x;
    for (; i + 256 < n; i += 512) {                          // two independent accumulators per thread
        acc0 = fma(fb[i], cos(tm * p[i]), acc0);
        acc1 = fma(fb[i + 256], cos(tm * p[i + 256]), acc1);
    }
    if (i < n) acc0 = fma(fb[i], cos(tm * p[i]), acc0);
    double acc = acc0 + acc1;
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int k = 0; k < 8; ++k) s += s_part[k];
        out[(size_t)b * n_t + m] = s / PI_D;
    }
}

int fail(cudaError_t e, const char *what)
{
    char buf[256];
    snprintf(buf, sizeof(buf), "%s: %s", what, cudaGetErrorString(e));
    set_error_text(buf);
    return DSE_ECUDA;
}

}  // namespace

// work: 2(n+1) doubles
int launch_gauss_legendre(int n, double *x, double *w, double *work, void *stream)
{
    cudaStream_t s = (cudaStream_t)stream;
    double2 *ab = reinterpret_cast<double2 *>(work);
    gl_prepare_kernel<<<(n + 256) / 256, 256, 0, s>>>(n, ab);
    const int q = (((n + 1) / 2) + 1) / 2;
    gl_nodes_kernel<<<(q + 31) / 32, 32, 0, s>>>(n, ab, x, w);      // one warp per CTA: balanced over the SMs
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(e, "gauss_legendre launch");
    return 2;
}

// ---------------------------------------------------------------------------------------------------------------
// dse_gauss_legendre_noalloc: the same two kernels with their scratch (the recurrence coefficients A_m, B_m of
// gl_prepare_kernel, 2 (n + 2) doubles) in a file-scope device array instead of a caller buffer -- for callers that
// cannot allocate (stream capture, serving loops).  DSE_GL_NOALLOC_MAX_N = 2^17 nodes (the paper's rule, fn.13) -> 2 MiB
// that every GPU that loads the library holds until exit.  In HOST code the array's name is only a stand-in: its device
// address comes from cudaGetSymbolAddress, once per device, with that device current.
static __device__ __align__(256) double g_gl_scratch[2 * (DSE_GL_NOALLOC_MAX_N + 2)];

namespace {
constexpr int GL_MAX_DEVICES = 64;
std::mutex g_gl_mu;
double *g_gl_scratch_addr[GL_MAX_DEVICES] = {};      // device address of g_gl_scratch on device d (nullptr: not asked yet)
}  // namespace

int launch_gauss_legendre_noalloc(int n, double *x, double *w, void *stream)
{
    if (n < 2 || n > DSE_GL_NOALLOC_MAX_N) {
        char buf[160];
        snprintf(buf, sizeof(buf), "dse_gauss_legendre_noalloc: n = %d is outside [2, %d] (the size of the static scratch)", n,
                 DSE_GL_NOALLOC_MAX_N);
        set_error_text(buf);
        return DSE_EINVAL;
    }
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(e, "cudaGetDevice");
    if (dev < 0 || dev >= GL_MAX_DEVICES) { set_error_text("dse_gauss_legendre_noalloc: device ordinal out of range"); return DSE_EINVAL; }
    double *scratch = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_gl_mu);
        if (!g_gl_scratch_addr[dev]) {
            void *p = nullptr;
            e = cudaGetSymbolAddress(&p, g_gl_scratch);          // `dev` is current: the address is this device's copy
            if (e != cudaSuccess || !p) return fail(e, "cudaGetSymbolAddress(g_gl_scratch)");
            g_gl_scratch_addr[dev] = static_cast<double *>(p);
        }
        scratch = g_gl_scratch_addr[dev];
    }
    // nothing in the scratch has to start at zero: gl_prepare_kernel rewrites the entries 0..n that gl_nodes_kernel reads
    return launch_gauss_legendre(n, x, w, scratch, stream);
}

// ln G(x_m), ln Z(x_m) for every system at arbitrary momenta x_m > 0: the series eq.(23),(24) on the clamped argument
// plus the continuations eq.(16)-(19) outside [eps2, L2] (the same definition the point kernel uses at z), and the
// running coupling alpha(x) = alpha(mu^2) G^2 Z.  One thread per (system, momentum).
__global__ void dressing_kernel(const KParams P, const double *__restrict__ c, int n_x, const double *__restrict__ x,
                                double alpha_mu, double *__restrict__ lnG_out, double *__restrict__ lnZ_out,
                                double *__restrict__ alpha_out)
{
    const int b = blockIdx.y;
    const double *a = c + (size_t)b * 2 * P.N, *bb = a + P.N;      // a_j <-> ln Z, b_j <-> ln G
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_x; i += gridDim.x * blockDim.x) {
        const double u = x[i];
        const double ell = log(u * P.inv_eps2);
        double s = fma(ell, P.two_over_Lg, -1.0), EG = 0.0, EZ = 0.0;
        if (u < P.eps2) { EG = P.pG * ell; EZ = P.pZ * ell; s = -1.0; }
        else if (u > P.L2) { const double t = log(fma(P.omega, ell - P.Lg, 1.0)); EG = P.delta * t; EZ = P.gamma * t; s = 1.0; }
        s = fmin(1.0, fmax(-1.0, s));
        double tm = 1.0, t = s;
        double lnZ = 0.5 * a[0] + (P.N > 1 ? a[1] * s : 0.0), lnG = 0.5 * bb[0] + (P.N > 1 ? bb[1] * s : 0.0);
        for (int j = 2; j < P.N; ++j) {
            const double tn = fma(2.0 * s, t, -tm);
            tm = t; t = tn;
            lnZ = fma(a[j], tn, lnZ);
            lnG = fma(bb[j], tn, lnG);
        }
        lnZ += EZ; lnG += EG;
        const size_t o = (size_t)b * n_x + i;
        if (lnG_out) lnG_out[o] = lnG;
        if (lnZ_out) lnZ_out[o] = lnZ;
        if (alpha_out) alpha_out[o] = alpha_mu * exp(2.0 * lnG + lnZ);
    }
}

int launch_dressing(const KParams &k, const double *c, int n_x, const double *x, double alpha_mu, double *lnG, double *lnZ,
                    double *alpha, void *stream)
{
    dressing_kernel<<<dim3((n_x + 127) / 128, k.B), 128, 0, (cudaStream_t)stream>>>(k, c, n_x, x, alpha_mu, lnG, lnZ, alpha);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(e, "dressing launch");
    return 1;
}

// work: (5 + B) n + 4 doubles:  ab[2(n+1)] | x[n] | w[n] | p[n] | f[B][n]
int launch_schwinger(const KParams &k, const double *c, int n, double p2_min, double p2_max, const double *t, int n_t,
                     double *out, double *work, void *stream)
{
    cudaStream_t s = (cudaStream_t)stream;
    double *x = work + 2 * (size_t)(n + 2), *w = x + n, *p = w + n, *f = p + n;
    int rc = launch_gauss_legendre(n, x, w, work, stream);
    if (rc < 0) return rc;
    const double u0 = 0.5 * log(p2_min), u1 = 0.5 * log(p2_max);
    schwinger_prepare<<<dim3((n + 255) / 256, k.B), 256, 0, s>>>(k, c, n, u0, u1, x, w, p, f);
    schwinger_kernel<<<dim3(n_t, k.B), 256, 0, s>>>(n, n_t, t, p, f, out);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(e, "schwinger launch");
    return rc + 2;
}

}  // namespace dse

extern "C" int dse_gauss_legendre_noalloc(int32_t n, double *x_dev, double *w_dev, void *stream)
{
    if (!x_dev || !w_dev) return DSE_EINVAL;
    const int rc = dse::launch_gauss_legendre_noalloc(n, x_dev, w_dev, stream);
    return rc < 0 ? rc : DSE_OK;
}

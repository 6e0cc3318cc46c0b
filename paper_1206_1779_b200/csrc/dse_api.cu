// dse_api.cu -- the C ABI declared in include/dse.h: parameter validation, handle and workspace
// lifetime, launch sequencing.  No arithmetic of the method happens on the host after dse_create.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "dse_internal.h"
#include "../../include/dse_diag.h"

struct dse_handle {
    dse_params params;
    dse::HostTables tab;
    dse::KParams k;
    dse::PointKernelConfig cfg;
    int device = 0;
    double *d_tables = nullptr;     // one allocation for all tables
    double *d_work = nullptr;       // one allocation for the per-build workspace
    double *d_geom = nullptr;       // geometry cache (optional)
    int *d_tail = nullptr;          // partition tables of the fused tail
    double *d_J = nullptr, *d_F = nullptr, *d_lu = nullptr;   // internal J, F for dse_newton_step (+ LU scratch)
    double *d_fd = nullptr;
    double *d_delta = nullptr, *d_stats = nullptr, *d_ctl = nullptr, *d_info = nullptr;   // dse_newton_solve
    dse::SolveGraph *solve = nullptr;                                                     // built at the first solve
    double *d_c = nullptr, *d_bc = nullptr, *d_Jh = nullptr, *d_Fh = nullptr;   // staging for *_host calls
    // dse_jacobian_host: pinned host staging.  h_in [c | bc] goes to the device in ONE copy (d_c, d_bc are adjacent);
    // small results are written by the assemble kernel straight into the mapped buffer h_out [J | F] (no copy node)
    double *h_in = nullptr, *h_out = nullptr, *m_out = nullptr;   // m_out = device alias of h_out
    static constexpr size_t ZERO_COPY_MAX_BYTES = 1u << 20;
    int64_t launches = 0;
    bool owns_const = false;
    // optional timing of the point kernel (dse_set_timing)
    static constexpr int EV_RING = 64;
    bool timing = false;
    cudaEvent_t ev[EV_RING][2] = {};
    int ev_head = 0, ev_pending = 0;
    double t_ms = 0.0;
    int64_t t_n = 0;
};

namespace {

int cuda_err(cudaError_t e, const char *what) { return dse::cuda_fail((int)e, what); }

#define CK(call)                                             \
    do {                                                     \
        cudaError_t e_ = (call);                             \
        if (e_ != cudaSuccess) return cuda_err(e_, #call);   \
    } while (0)

bool finite_pos(double v) { return std::isfinite(v) && v > 0.0; }

int validate(const dse_params *p)
{
    if (!p) return DSE_EINVAL;
    if (p->n_cheb < 2 || p->n_cheb > DSE_MAX_NCHEB) return DSE_EINVAL;
    if (p->n_r < 2 || p->n_theta < 2 || p->n_batch < 1) return DSE_EINVAL;
    // the host table builder is O(n^2) per Gauss-Legendre rule (Newton on the Legendre recurrence in long double) and the
    // angular table lives in shared memory: 2^15 radial and 2^11 angular nodes are far beyond any use of the method
    if (p->n_r > (1 << 15) || p->n_theta > (1 << 11) || p->n_batch > (1 << 20)) return DSE_EINVAL;
    if (!finite_pos(p->eps2) || !finite_pos(p->L2) || !(p->eps2 < p->L2)) return DSE_EINVAL;
    if (!finite_pos(p->alpha_mu) || !finite_pos(p->n_colors)) return DSE_EINVAL;
    if (!finite_pos(p->x_Z) || !std::isfinite(p->x_G) || p->x_G < 0.0 || (p->x_G == 0.0 && p->x_Z == 0.0)) return DSE_EINVAL;
    if (!std::isfinite(p->delta) || !std::isfinite(p->ir_exp_G) || !std::isfinite(p->ir_exp_Z)) return DSE_EINVAL;
    if (!std::isfinite(p->uv_omega) || p->uv_omega < 0.0) return DSE_EINVAL;
    const int known = DSE_FLAG_GEOMETRY_CACHE | DSE_FLAG_ANGULAR_TANH_SINH | DSE_FLAG_RADIAL_SPLIT | DSE_FLAG_USER_TABLES |
                      DSE_FLAG_CONST_COEF | DSE_FLAG_PER_SYSTEM_KERNELS;
    if (p->n_r_ir < 0 || p->n_r_ir > (1 << 15) || (p->flags & ~known)) return DSE_EINVAL;
    return DSE_OK;
}

// drains the oldest `n` pending event pairs into the accumulators
int drain_events(dse_handle *h, int n)
{
    while (n-- > 0 && h->ev_pending > 0) {
        const int idx = (h->ev_head - h->ev_pending + 2 * dse_handle::EV_RING) % dse_handle::EV_RING;
        float ms = 0.f;
        cudaError_t e = cudaEventSynchronize(h->ev[idx][1]);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, h->ev[idx][0], h->ev[idx][1]);
        if (e != cudaSuccess) return cuda_err(e, "timing events");
        h->t_ms += ms;
        h->t_n += 1;
        --h->ev_pending;
    }
    return DSE_OK;
}

// build with optional event pair around the point kernel
int do_build(dse_handle *h, const double *c, const double *bc, double *J, double *F, void *stream)
{
    void *e0 = nullptr, *e1 = nullptr;
    if (h->timing) {
        if (h->ev_pending == dse_handle::EV_RING) {
            int rc = drain_events(h, 1);
            if (rc < 0) return rc;
        }
        e0 = h->ev[h->ev_head][0];
        e1 = h->ev[h->ev_head][1];
        h->ev_head = (h->ev_head + 1) % dse_handle::EV_RING;
        ++h->ev_pending;
    }
    int rc = dse::launch_build(h->k, h->cfg, c, bc, J, F, stream, e0, e1);
    if (rc < 0) return rc;
    h->launches += rc;
    return DSE_OK;
}

template <class T>
size_t carve(size_t &off, size_t n)
{
    size_t o = off;
    off += (n + 1) & ~(size_t)1;      // keep 16-byte alignment in units of doubles
    return o;
}

}  // namespace

extern "C" {

static int create_impl(const dse_params *params, const dse_tables *user, dse_handle **out);

int dse_create(const dse_params *params, dse_handle **out)
{
    if (params && (params->flags & DSE_FLAG_USER_TABLES)) return DSE_EINVAL;      // needs dse_create_with_tables
    return create_impl(params, nullptr, out);
}

int dse_create_with_tables(const dse_params *params, const dse_tables *tables, dse_handle **out)
{
    if (!params || !(params->flags & DSE_FLAG_USER_TABLES) || !tables) return DSE_EINVAL;
    if (!tables->x_ext || !tables->y || !tables->Wy || !tables->theta || !tables->Omega) return DSE_EINVAL;
    return create_impl(params, tables, out);
}

static int create_impl(const dse_params *params, const dse_tables *user, dse_handle **out)
{
    if (!out) return DSE_EINVAL;
    int rc = validate(params);
    if (rc != DSE_OK) return rc;
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        dse::set_error_text(e != cudaSuccess ? cudaGetErrorString(e) : "no CUDA device (this library has no CPU fallback)");
        return DSE_ECUDA;
    }
    dse_handle *h = new (std::nothrow) dse_handle();
    if (!h) return DSE_ENOMEM;
    h->params = *params;
    e = cudaGetDevice(&h->device);
    if (e != cudaSuccess) { delete h; return cuda_err(e, "cudaGetDevice"); }
    try {
        dse::build_tables(*params, user, h->tab);
    } catch (const std::bad_alloc &) {
        delete h;
        return DSE_ENOMEM;
    }
    const dse::HostTables &T = h->tab;
    dse::KParams &k = h->k;
    memset(&k, 0, sizeof(k));
    k.N = T.N; k.Npad = T.Npad; k.NCH = T.Npad / dse::CJ;
    k.SUB = 32 / k.NCH; k.rounds = (32 + k.SUB - 1) / k.SUB;
    k.Nr = T.Nr; k.Nt = T.Nt; k.Ntpad = T.Ntpad;
    k.g = T.Ntpad < 32 ? T.Ntpad : 32;
    k.rpb = 32 / k.g;
    k.Next = T.Next; k.B = params->n_batch; k.iZ = T.iZ; k.iG = T.iG;
    k.rstride = T.rstride; k.Gext = T.rstride ? T.Next : 1;
    k.R = (long long)k.B * k.Next * k.Nr;
    if ((long long)k.Next * k.Nr * k.Ntpad >= (1ll << 31) || (long long)k.B * k.Next >= (1ll << 30)) {
        dse::set_error_text("grid too large: N_ext*N_r*N_theta must stay below 2^31 points per system");
        delete h;
        return DSE_EINVAL;
    }
    k.eps2 = params->eps2; k.L2 = params->L2; k.inv_eps2 = 1.0 / params->eps2;
    k.Lg = T.Lg; k.two_over_Lg = 2.0 / T.Lg;
    k.pG = params->ir_exp_G; k.pZ = params->ir_exp_Z; k.omega = params->uv_omega;
    k.delta = params->delta; k.gamma = -1.0 - 2.0 * params->delta;
    k.e1 = -2.0 - 6.0 * params->delta; k.e2 = -3.0 * params->delta;      // P = G^{e1} Z^{e2}, eq.(3),(9)
    k.C = T.C;

    // ---- tables -> device (one allocation) ----
    size_t off = 0;
    const size_t o_x = carve<double>(off, T.Next), o_sx = carve<double>(off, T.Next), o_c3 = carve<double>(off, T.Next);
    const size_t o_y = carve<double>(off, T.y.size()), o_sy = carve<double>(off, T.y.size()), o_W = carve<double>(off, T.y.size());
    const size_t o_EG = carve<double>(off, T.y.size()), o_EZ = carve<double>(off, T.y.size()), o_tr = carve<double>(off, T.y.size());
    const size_t o_ang = carve<double>(off, T.ang.size());
    const size_t o_py = carve<double>(off, T.phi_y.size()), o_px = carve<double>(off, T.phi_x.size());
    std::vector<double> host(off, 0.0);
    memcpy(&host[o_x], T.x_ext.data(), 8 * T.x_ext.size());
    memcpy(&host[o_sx], T.sx_ext.data(), 8 * T.sx_ext.size());
    memcpy(&host[o_c3], T.c3x_ext.data(), 8 * T.c3x_ext.size());
    memcpy(&host[o_y], T.y.data(), 8 * T.y.size());
    memcpy(&host[o_sy], T.sy.data(), 8 * T.sy.size());
    memcpy(&host[o_W], T.Wy.data(), 8 * T.Wy.size());
    memcpy(&host[o_EG], T.EGy.data(), 8 * T.EGy.size());
    memcpy(&host[o_tr], T.t_r.data(), 8 * T.t_r.size());
    memcpy(&host[o_EZ], T.EZy.data(), 8 * T.EZy.size());
    memcpy(&host[o_ang], T.ang.data(), 8 * T.ang.size());
    memcpy(&host[o_py], T.phi_y.data(), 8 * T.phi_y.size());
    memcpy(&host[o_px], T.phi_x.data(), 8 * T.phi_x.size());
    if (cudaMalloc(&h->d_tables, 8 * off) != cudaSuccess) { dse_destroy(h); return DSE_ENOMEM; }
    e = cudaMemcpy(h->d_tables, host.data(), 8 * off, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { dse_destroy(h); return cuda_err(e, "cudaMemcpy(tables)"); }
    double *t = h->d_tables;
    k.x_ext = t + o_x; k.sx_ext = t + o_sx; k.c3x_ext = t + o_c3;
    k.y = t + o_y; k.sy = t + o_sy; k.Wy = t + o_W; k.EGy = t + o_EG; k.EZy = t + o_EZ; k.t_r = t + o_tr; k.ang = t + o_ang; k.phi_y = t + o_py; k.phi_x = t + o_px;

    // ---- geometry cache (optional) ----
    if (params->flags & DSE_FLAG_GEOMETRY_CACHE) {
        const size_t n = (size_t)k.Next * k.Nr * k.Ntpad * 4;
        if (cudaMalloc(&h->d_geom, 8 * n) != cudaSuccess) { dse_destroy(h); return DSE_ENOMEM; }
        k.geom = h->d_geom;
    }

    // ---- launch configuration of the point kernel ----
    if (params->flags & DSE_FLAG_CONST_COEF) {            // explicit request for the library's constant-bank slot
        if (!dse::constc_shape_ok(k)) {
            dse::set_error_text("DSE_FLAG_CONST_COEF needs n_batch = 1, n_theta >= 32 and n_cheb in {8, 16, 32, 64, 128}");
            dse_destroy(h);
            return DSE_EINVAL;
        }
        if (!dse::const_slot_acquire()) {
            dse::set_error_text("DSE_FLAG_CONST_COEF: the constant-bank slot is held by another handle");
            dse_destroy(h);
            return DSE_EBUSY;
        }
        h->owns_const = true;
        k.use_constc = 1;
    }
    rc = dse::query_point_kernel(k, h->cfg);
    if (rc < 0) { dse_destroy(h); return rc; }
    if (k.use_constc && !h->cfg.pipelined) {              // (cannot happen for the shapes constc_shape_ok admits)
        dse::set_error_text("DSE_FLAG_CONST_COEF: shape does not run the pipelined kernel");
        dse_destroy(h);
        return DSE_EINVAL;
    }
    if (!(params->flags & DSE_FLAG_PER_SYSTEM_KERNELS) && dse::batched_eligible(k)) {      // 8 systems per warp on the fp64 tensor path
        rc = dse::query_point_batched(k, h->cfg);
        if (rc < 0) { dse_destroy(h); return rc; }
    }
    k.W = h->cfg.grid * (h->cfg.block / 32);
    // small builds on the generic kernel (n_theta < 32, ...): the kernel computes H1 itself, a build is one launch
    k.self_h1 = (!h->cfg.pipelined && !h->cfg.batched && (long long)k.B * k.Gext * k.Nr <= dse::SELF_H1_MAX_ROWS) ? 1 : 0;
    k.upr = (h->cfg.pipelined || h->cfg.batched) ? (k.Ntpad / 32) : 1;      // these kernels partition 32-point batches
    k.bgroup = h->cfg.batched ? 8 : 1;
    // the batched kernel works on groups of 8 systems: the batch is padded with idle systems (zero coefficients, zero
    // weights) whose rows exist in the workspace but are never read by the later kernels
    const size_t Bpad = h->cfg.batched ? ((size_t)k.B + 7) / 8 * 8 : (size_t)k.B;
    const size_t Rpad = Bpad * k.Next * k.Nr;
    k.U = (long long)(Rpad / k.bgroup) * k.upr;

    // ---- workspace (one allocation, zero-initialised: unwritten partial slots must read 0) ----
    const size_t n2 = 2 * (size_t)k.N;
    off = 0;
    const size_t o_coef = carve<double>(off, Bpad * k.Npad * 2);
    const size_t o_Gy = carve<double>(off, Bpad * k.Gext * k.Nr), o_Py = carve<double>(off, Bpad * k.Gext * k.Nr);
    const size_t o_iG = carve<double>(off, (size_t)k.B * k.N), o_iZ = carve<double>(off, (size_t)k.B * k.N);
    const size_t o_A = carve<double>(off, Rpad * 4), o_AH = carve<double>(off, Rpad * 4);
    const size_t slot = h->cfg.batched ? (size_t)3 * k.Npad : (size_t)(6 * k.Npad + 2);      // dse_tail.cuh: slot_doubles
    const size_t o_S = carve<double>(off, ((size_t)k.W * k.bgroup + Bpad * k.Next) * slot);
    const size_t o_R = carve<double>(off, (size_t)k.B * k.Next * 3 * k.Npad);
    const size_t o_Dg = carve<double>(off, (size_t)k.B * k.Next * 4 * k.Npad), o_Pi = carve<double>(off, (size_t)k.B * k.Next * 4);
    const size_t n_pend = (size_t)k.B * ((k.Next + 31) / 32);
    const size_t o_cnt = carve<double>(off, ((size_t)k.B * k.Next + 2 * (size_t)k.B + n_pend + 1) / 2 + 1);   // unsigned counters of the fused tail
    const size_t o_J = carve<double>(off, (size_t)k.B * n2 * n2), o_F = carve<double>(off, (size_t)k.B * n2);
    const size_t o_lu = carve<double>(off, (size_t)k.B * dse::lu_scratch_doubles((int)n2));
    const size_t o_c = carve<double>(off, (size_t)k.B * n2), o_bc = carve<double>(off, (size_t)k.B * 2);
    const size_t o_fd = carve<double>(off, (size_t)k.B * n2 * 3);          // finite-difference self-check: c_tmp, F+, F-
    const size_t o_dl = carve<double>(off, (size_t)k.B * n2), o_st = carve<double>(off, (size_t)k.B * 4);
    const size_t o_ctl = carve<double>(off, 8), o_info = carve<double>(off, (size_t)k.B * 6);
    if (cudaMalloc(&h->d_work, 8 * off) != cudaSuccess) { dse_destroy(h); return DSE_ENOMEM; }
    e = cudaMemset(h->d_work, 0, 8 * off);
    if (e != cudaSuccess) { dse_destroy(h); return cuda_err(e, "cudaMemset(workspace)"); }
    double *wk = h->d_work;
    k.coefP = wk + o_coef; k.Gy = wk + o_Gy; k.Py = wk + o_Py; k.invG = wk + o_iG; k.invZ = wk + o_iZ;
    k.Apart = wk + o_A; k.AHead = wk + o_AH; k.Spart = wk + o_S; k.Rz = wk + o_R; h->d_fd = wk + o_fd;
    k.Dg = wk + o_Dg; k.PiInv = wk + o_Pi;
    k.cnt = reinterpret_cast<unsigned *>(wk + o_cnt); k.done = k.cnt + (size_t)k.B * k.Next;
    k.rdy = k.done + k.B; k.pend = k.rdy + k.B;
    h->d_J = wk + o_J; h->d_F = wk + o_F; h->d_lu = wk + o_lu; h->d_c = wk + o_c; h->d_bc = wk + o_bc;
    h->d_Jh = h->d_J; h->d_Fh = h->d_F;
    h->d_delta = wk + o_dl; h->d_stats = wk + o_st; h->d_ctl = wk + o_ctl; h->d_info = wk + o_info;

    if (!h->cfg.batched) {
        // who works on what, from the same partition the kernels use: warp w owns the units [w U / W, (w + 1) U / W)
        const long long upb = (long long)k.Nr * k.upr, nbi = (long long)k.B * k.Next;
        const int wpb = h->cfg.block / 32, grid = h->cfg.grid;
        std::vector<int> tab((size_t)2 * grid + (size_t)2 * nbi);
        int *tb = tab.data() + (size_t)2 * grid;
        for (long long bi = 0; bi < nbi; ++bi) { tb[2 * bi] = 0x7fffffff; tb[2 * bi + 1] = -1; }
        for (int c = 0; c < grid; ++c) {
            tab[2 * c] = 0; tab[2 * c + 1] = -1;
            for (int wi = 0; wi < wpb; ++wi) {
                const long long w = (long long)c * wpb + wi;
                const long long t0 = (w * k.U) / k.W, t1 = ((w + 1) * k.U) / k.W;
                if (t0 >= t1) continue;
                const int b0 = (int)(t0 / upb), b1 = (int)((t1 - 1) / upb);
                if (tab[2 * c + 1] < 0) tab[2 * c] = b0;
                tab[2 * c + 1] = b1;
                for (int bi = b0; bi <= b1; ++bi) {
                    if (tb[2 * bi] > (int)w) tb[2 * bi] = (int)w;
                    if (tb[2 * bi + 1] < (int)w) tb[2 * bi + 1] = (int)w;
                }
            }
        }
        if (cudaMalloc(&h->d_tail, sizeof(int) * tab.size()) != cudaSuccess) { dse_destroy(h); return DSE_ENOMEM; }
        e = cudaMemcpy(h->d_tail, tab.data(), sizeof(int) * tab.size(), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) { dse_destroy(h); return cuda_err(e, "cudaMemcpy(tail tables)"); }
        k.tail_cta = h->d_tail; k.tail_bi = h->d_tail + (size_t)2 * h->cfg.grid;
    }
    k.tail_polls = dse::TAIL_POLLS;
    rc = dse::lu_configure((int)n2);
    if (rc < 0) { dse_destroy(h); return rc; }
    if (k.geom) {
        rc = dse::launch_geometry(k, h->d_geom, nullptr);
        if (rc < 0) { dse_destroy(h); return rc; }
        h->launches += rc;
    }
    e = cudaDeviceSynchronize();
    if (e != cudaSuccess) { dse_destroy(h); return cuda_err(e, "cudaDeviceSynchronize(create)"); }
    *out = h;
    return DSE_OK;
}

int dse_destroy(dse_handle *h)
{
    if (!h) return DSE_OK;
    cudaDeviceSynchronize();
    if (h->owns_const) dse::const_slot_release();
    dse::solve_graph_destroy(h->solve);
    if (h->d_tables) cudaFree(h->d_tables);
    if (h->d_work) cudaFree(h->d_work);
    if (h->d_geom) cudaFree(h->d_geom);
    if (h->d_tail) cudaFree(h->d_tail);
    if (h->h_in) cudaFreeHost(h->h_in);
    if (h->h_out) cudaFreeHost(h->h_out);
    for (auto &p : h->ev)
        for (auto &e : p)
            if (e) cudaEventDestroy(e);
    delete h;
    return DSE_OK;
}

int dse_jacobian(dse_handle *h, const double *c_dev, const double *bc_dev, double *J_dev, double *F_dev, void *stream)
{
    if (!h || !c_dev || !bc_dev || !J_dev || !F_dev) return DSE_EINVAL;
    return do_build(h, c_dev, bc_dev, J_dev, F_dev, stream);
}

int dse_residual(dse_handle *h, const double *c_dev, const double *bc_dev, double *F_dev, void *stream)
{
    if (!h || !c_dev || !bc_dev || !F_dev) return DSE_EINVAL;
    return do_build(h, c_dev, bc_dev, nullptr, F_dev, stream);
}

int dse_newton_step(dse_handle *h, double *c_dev, const double *bc_dev, double rho, double *stats_dev, void *stream)
{
    if (!h || !c_dev || !bc_dev || !std::isfinite(rho)) return DSE_EINVAL;
    int rc = do_build(h, c_dev, bc_dev, h->d_J, h->d_F, stream);
    if (rc < 0) return rc;
    rc = dse::launch_lu(2 * h->k.N, h->k.B, h->d_J, h->d_F, nullptr, c_dev, rho, stats_dev, h->d_lu, stream);
    if (rc < 0) return rc;
    h->launches += rc;
    return DSE_OK;
}

int dse_newton_solve(dse_handle *h, double *c_dev, const double *bc_dev, double rho, double step_cap, double tol,
                     int32_t max_iter, double *info_dev, void *stream)
{
    if (!h || !c_dev || !bc_dev || !(rho > 0.0) || !(rho <= 1.0) || !std::isfinite(step_cap) || !(tol >= 0.0) ||
        !std::isfinite(tol) || max_iter < 1)
        return DSE_EINVAL;
    const size_t n2 = 2 * (size_t)h->k.N, B = (size_t)h->k.B;
    if (!h->solve) {
        int rc = dse::solve_graph_create(h->k, h->cfg, h->d_c, h->d_bc, h->d_J, h->d_F, h->d_delta, h->d_stats, h->d_lu,
                                         h->d_ctl, h->d_info, &h->solve);
        if (rc < 0) return rc;
    }
    cudaStream_t s = (cudaStream_t)stream;
    CK(cudaMemcpyAsync(h->d_c, c_dev, 8 * B * n2, cudaMemcpyDeviceToDevice, s));
    CK(cudaMemcpyAsync(h->d_bc, bc_dev, 8 * B * 2, cudaMemcpyDeviceToDevice, s));
    int rc = dse::launch_solve(h->solve, rho, step_cap, tol, max_iter, stream);
    if (rc < 0) return rc;
    h->launches += rc;
    CK(cudaMemcpyAsync(c_dev, h->d_c, 8 * B * n2, cudaMemcpyDeviceToDevice, s));
    if (info_dev) CK(cudaMemcpyAsync(info_dev, h->d_info, 8 * B * 6, cudaMemcpyDeviceToDevice, s));
    return DSE_OK;
}

int dse_lu_solve(dse_handle *h, int32_t n, int32_t n_sys, const double *A_dev, const double *b_dev, double *x_dev,
                 double *stats_dev, void *stream)
{
    if (!h || !A_dev || !b_dev || !x_dev || n < 1 || n > 256 || n_sys < 1) return DSE_EINVAL;
    double *scratch = nullptr;
    const size_t need = dse::lu_scratch_doubles(n) * (size_t)n_sys;
    if (need) {
        // large systems eliminate in global memory: only the handle's own scratch (sized for 2N, n_batch) is available
        if (n != 2 * h->k.N || n_sys > h->k.B) return DSE_EINVAL;
        scratch = h->d_lu;
    }
    int rc = n == 2 * h->k.N ? 0 : dse::lu_configure(n);
    if (rc < 0) return rc;
    rc = dse::launch_lu(n, n_sys, A_dev, b_dev, x_dev, nullptr, 0.0, stats_dev, scratch, stream);
    if (rc < 0) return rc;
    h->launches += rc;
    return DSE_OK;
}

int dse_jacobian_host(dse_handle *h, const double *c_host, const double *bc_host, double *J_host, double *F_host)
{
    if (!h || !c_host || !bc_host || !F_host) return DSE_EINVAL;
    const size_t n2 = 2 * (size_t)h->k.N, B = (size_t)h->k.B;
    const size_t n_in = B * n2 + B * 2, n_J = B * n2 * n2, n_F = B * n2;
    if (!h->h_in) {                                      // first call: pinned staging (inputs) and mapped staging (results)
        CK(cudaHostAlloc((void **)&h->h_in, 8 * n_in, cudaHostAllocDefault));
        if (8 * (n_J + n_F) <= dse_handle::ZERO_COPY_MAX_BYTES) {
            CK(cudaHostAlloc((void **)&h->h_out, 8 * (n_J + n_F), cudaHostAllocMapped));
            CK(cudaHostGetDevicePointer((void **)&h->m_out, h->h_out, 0));
        }
    }
    memcpy(h->h_in, c_host, 8 * B * n2);
    memcpy(h->h_in + B * n2, bc_host, 8 * B * 2);
    CK(cudaMemcpyAsync(h->d_c, h->h_in, 8 * n_in, cudaMemcpyHostToDevice, nullptr));      // d_bc = d_c + B*2N
    if (h->m_out) {
        int rc = do_build(h, h->d_c, h->d_bc, J_host ? h->m_out : nullptr, h->m_out + n_J, nullptr);
        if (rc < 0) return rc;
        CK(cudaStreamSynchronize(nullptr));
        if (J_host) memcpy(J_host, h->h_out, 8 * n_J);
        memcpy(F_host, h->h_out + n_J, 8 * n_F);
        return DSE_OK;
    }
    int rc = do_build(h, h->d_c, h->d_bc, J_host ? h->d_Jh : nullptr, h->d_Fh, nullptr);
    if (rc < 0) return rc;
    if (J_host) CK(cudaMemcpyAsync(J_host, h->d_Jh, 8 * n_J, cudaMemcpyDeviceToHost, nullptr));
    CK(cudaMemcpyAsync(F_host, h->d_Fh, 8 * n_F, cudaMemcpyDeviceToHost, nullptr));
    CK(cudaStreamSynchronize(nullptr));
    return DSE_OK;
}

int dse_set_timing(dse_handle *h, int32_t enable)
{
    if (!h) return DSE_EINVAL;
    int rc = drain_events(h, h->ev_pending);
    if (rc < 0) return rc;
    if (enable)
        for (auto &p : h->ev)
            for (auto &e : p)
                if (!e) CK(cudaEventCreate(&e));
    h->timing = enable != 0;
    h->t_ms = 0.0;
    h->t_n = 0;
    return DSE_OK;
}

int dse_get_timing(dse_handle *h, double *total_ms, int64_t *launches)
{
    if (!h || !total_ms || !launches) return DSE_EINVAL;
    int rc = drain_events(h, h->ev_pending);
    if (rc < 0) return rc;
    *total_ms = h->t_ms;
    *launches = h->t_n;
    return DSE_OK;
}

int dse_jacobian_fd(dse_handle *h, const double *c_dev, const double *bc_dev, double eps_rel, double *J_dev, void *stream)
{
    if (!h || !c_dev || !bc_dev || !J_dev || !(eps_rel > 0.0) || !std::isfinite(eps_rel)) return DSE_EINVAL;
    const int n2 = 2 * h->k.N, B = h->k.B;
    double *c_tmp = h->d_fd, *Fp = c_tmp + (size_t)B * n2, *Fm = Fp + (size_t)B * n2;
    for (int j = 0; j < n2; ++j) {
        for (int sgn = 0; sgn < 2; ++sgn) {
            int rc = dse::launch_fd_perturb(n2, B, c_dev, c_tmp, j, sgn ? -1.0 : 1.0, eps_rel, stream);
            if (rc < 0) return rc;
            h->launches += rc;
            rc = do_build(h, c_tmp, bc_dev, nullptr, sgn ? Fm : Fp, stream);
            if (rc < 0) return rc;
        }
        int rc = dse::launch_fd_column(n2, B, c_dev, Fp, Fm, J_dev, j, eps_rel, stream);
        if (rc < 0) return rc;
        h->launches += rc;
    }
    return DSE_OK;
}

int dse_gauss_legendre(int32_t n, double *x_dev, double *w_dev, double *work_dev, void *stream)
{
    if (n < 2 || n > (1 << 24) || !x_dev || !w_dev || !work_dev) return DSE_EINVAL;
    int rc = dse::launch_gauss_legendre(n, x_dev, w_dev, work_dev, stream);
    return rc < 0 ? rc : DSE_OK;
}

int dse_schwinger(dse_handle *h, const double *c_dev, int32_t n_nodes, double p2_min, double p2_max, const double *t_dev,
                  int32_t n_t, double *delta_dev, double *work_dev, void *stream)
{
    if (!h || !c_dev || !t_dev || !delta_dev || !work_dev || n_nodes < 2 || n_nodes > (1 << 24) || n_t < 1) return DSE_EINVAL;
    if (!finite_pos(p2_min) || !finite_pos(p2_max) || !(p2_min < p2_max)) return DSE_EINVAL;
    int rc = dse::launch_schwinger(h->k, c_dev, n_nodes, p2_min, p2_max, t_dev, n_t, delta_dev, work_dev, stream);
    if (rc < 0) return rc;
    h->launches += rc;
    return DSE_OK;
}

int dse_dressing(dse_handle *h, const double *c_dev, const double *x_dev, int32_t n_x, double *lnG_dev, double *lnZ_dev,
                 double *alpha_dev, void *stream)
{
    if (!h || !c_dev || !x_dev || n_x < 1 || (!lnG_dev && !lnZ_dev && !alpha_dev)) return DSE_EINVAL;
    int rc = dse::launch_dressing(h->k, c_dev, n_x, x_dev, h->params.alpha_mu, lnG_dev, lnZ_dev, alpha_dev, stream);
    if (rc < 0) return rc;
    h->launches += rc;
    return DSE_OK;
}

int dse_n_ext(const dse_handle *h) { return h ? h->k.Next : DSE_EINVAL; }

int dse_get_tables(const dse_handle *h, double *x_ext_host, double *y_host, double *Wy_host, double *theta_host,
                   double *Omega_host)
{
    if (!h) return DSE_EINVAL;
    const dse::HostTables &T = h->tab;
    if (x_ext_host) memcpy(x_ext_host, T.x_ext.data(), 8 * T.x_ext.size());
    if (y_host) memcpy(y_host, T.y.data(), 8 * T.y.size());            // [n_rules][n_rad]: every rule under the split flag
    if (Wy_host) memcpy(Wy_host, T.Wy.data(), 8 * T.Wy.size());
    if (theta_host) memcpy(theta_host, T.theta.data(), 8 * T.theta.size());
    if (Omega_host) memcpy(Omega_host, T.Omega.data(), 8 * T.Omega.size());
    return DSE_OK;
}

int64_t dse_launch_count(const dse_handle *h) { return h ? h->launches : 0; }

int dse_diag_phase_stamps(int32_t which, int64_t *out_host, int32_t max_words)
{
    if (!out_host || max_words < 1 || (which != 0 && which != 1)) return DSE_EINVAL;
    static_assert(sizeof(long long) == sizeof(int64_t), "stamp words");
    const int n = which == 0 ? dse::phase_stamps_point(reinterpret_cast<long long *>(out_host), max_words)
                             : dse::phase_stamps_lu(reinterpret_cast<long long *>(out_host), max_words);
    if (n == 0) { dse::set_error_text("dse_diag_phase_stamps: the library was built without -DDSE_PHASE_TIMING"); return DSE_EINVAL; }
    return n;
}

int dse_diag_set_tail_polls(dse_handle *h, int32_t polls)
{
    if (!h || polls < 0) return DSE_EINVAL;
    h->k.tail_polls = polls;
    return DSE_OK;
}

int dse_kernel_info(const dse_handle *h, int32_t out[8])
{
    if (!h || !out) return DSE_EINVAL;
    out[0] = h->cfg.grid; out[1] = h->cfg.block; out[2] = h->cfg.smem; out[3] = h->cfg.regs;
    out[4] = h->cfg.ctas_per_sm; out[5] = h->cfg.sms;
    out[6] = h->cfg.batched ? 2 : (h->cfg.pipelined ? 1 : 0);
    out[7] = h->cfg.batched ? 4 : ((h->cfg.pipelined || h->k.self_h1) ? 1 : 2);
    return DSE_OK;
}

const char *dse_strerror(int code)
{
    switch (code) {
        case DSE_OK: return "ok";
        case DSE_EINVAL: return "invalid argument";
        case DSE_ENOMEM: return "out of memory";
        case DSE_ECUDA: return "CUDA error (see dse_last_error)";
        case DSE_EBUSY: return "constant-bank coefficient slot is held by another handle";
        default: return "unknown error";
    }
}

const char *dse_last_error(void) { return dse::last_error_text(); }

}  // extern "C"

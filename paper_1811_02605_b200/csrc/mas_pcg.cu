// mas_pcg.cu -- C ABI (include/mas_pcg.h) of the B200-native MAS PCG path: handle, coefficient
// planes, workspaces, the CUDA-graph WHILE loop and its host-chunk fallback.  Every step of the
// numerical path runs in the kernels of kernels_base.cuh / kernels_march.cuh; this file only
// marshals.  There is no CPU fallback.
#include "../../include/mas_pcg.h"

#include <cuda_runtime.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <vector>

#include "common.cuh"
#include "kernels_base.cuh"
#include "kernels_march.cuh"
#include "kernels_stencil.cuh"
#include "kernels_stencil_tma.cuh"
#include "kernels_k1_tma.cuh"
#include "kernels_persistent.cuh"

using namespace mas;

namespace {

constexpr int NT_BASE = 256;
constexpr int HOST_CHUNK = 16;       // iterations per poll in host-chunk mode

struct KLaunch {                     // one kernel launch, usable directly or as a graph node
    const void *func = nullptr;
    dim3 grid{1, 1, 1}, block{1, 1, 1};
    size_t smem = 0;
    void *args[12] = {};
    int nargs = 0;
};

template <typename T>
struct DevBuf {
    T *p = nullptr;
    size_t n = 0;
    cudaError_t alloc(size_t count)
    {
        release();
        n = count;
        return cudaMalloc((void **)&p, (count ? count : 1) * sizeof(T));
    }
    void release()
    {
        if (p) cudaFree(p);
        p = nullptr;
        n = 0;
    }
};

}  // namespace

struct mas_pcg {
    int nr = 0, nt = 0, np = 0;
    size_t n = 0;
    int device = 0, num_sms = 0;
    double dt = 0.0;
    int uniform_phi = 0;
    // device planes
    DevBuf<double> V2, SD, CP, CRoff, CT, E, F, AR, AT, Dinv, vp, wp, ip, Vinv;
    double lambda_max = 0.0;         // Gershgorin bound on the spectral radius of M = -V^-1 L_sym
    double vp0 = 0, wp0 = 0, ip0 = 0;
    // workspaces
    DevBuf<double> r, p0, p1, q, partials, hist, bdev, xdev;
    DevBuf<State> st;
    DevBuf<SolveArgs> args;
    // pinned staging
    SolveArgs *h_args = nullptr;
    State *h_st = nullptr;
    double *h_hist = nullptr;
    size_t hist_cap = 0;
    // loop
    int loop_mode = 1;               // requested: 1 graph-while, 0 host chunks
    int loop_mode_used = 1;
    int variant = 3;                 // K1 variant: 0 baseline, 1 marching tiles (64 wide), 2 wide marching tiles (cp.async),
                                     // 3 wide marching tiles with TMA bulk copies + mbarriers (default)
    int tile = 0;                    // tile configuration id of the variant
    int ci_force = 0;                // >0: override the r-chunk length (tuning)
    int apply_variant = 1;           // 1: k_stencil marching kernel for A x (apply / initial residual); 0: k_apply
    int stencil_tile = 7;            // 0..5 cp.async k_stencil, 6..11 TMA k_stencil_tma (7 = TJ 8, 2 blocks/SM: fastest)
    int k2r_tile = 0;
    int serpentine = 1;              // 1: K2 sweeps the rows backward (L2 reuse across K1 -> K2 -> K1)
    int persistent = 2;              // one cooperative kernel for the whole solve: 0 off, 1 whenever it fits, 2 auto
    int coop_ok = 0;
    int pdl = 0;                     // programmatic dependent launch edges inside the loop body: measured 5 % SLOWER
                                     // (early K1 blocks park their shared memory while K2 drains), so off
    int unroll = 4;                  // PCG iterations per WHILE trip of the graph loop (measured: +1 % c4, +3 % c3)
    int qrecompute = 0;              // 1 (needs xfuse, wide): q is not stored, K2 recomputes it: 64 B/cell/iteration
    int xfuse = 1;                   // 1: x-update fused into K1 (72 B/cell/iteration), wide variant only
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    bool graph_dirty = true;
    long long stats[8] = {};
    OpDev op{};
    Work work{};
};

namespace {

int fail(mas_pcg *h, int code)
{
    mas_pcg_destroy(h);
    return code;
}

#define CK(call)                                   \
    do {                                           \
        if ((call) != cudaSuccess) {               \
            cudaGetLastError();                    \
            return MAS_ECUDA;                      \
        }                                          \
    } while (0)

double nu_at(const mas_nu_t *nu, int nt, int i, int j) { return nu->kind == 0 ? nu->v[0] : nu->v[(size_t)i * nt + j]; }

bool positive(const double *a, int lo, int hi)
{
    for (int i = lo; i < hi; i++)
        if (!(a[i] > 0.0) || !isfinite(a[i])) return false;
    return true;
}

int upload(DevBuf<double> &d, const std::vector<double> &h)
{
    if (d.alloc(h.size()) != cudaSuccess) return MAS_ENOMEM;
    CK(cudaMemcpy(d.p, h.data(), h.size() * sizeof(double), cudaMemcpyHostToDevice));
    return MAS_OK;
}

void fill_op(mas_pcg *h)
{
    OpDev &o = h->op;
    o.nr = h->nr; o.nt = h->nt; o.np = h->np; o.nv = h->np / 2;
    o.nrows = h->nr * h->nt;
    o.uniform_phi = h->uniform_phi;
    o.n = (long long)h->n;
    o.E = h->E.p; o.F = h->F.p; o.AR = h->AR.p; o.AT = h->AT.p; o.Dinv = h->Dinv.p;
    o.V2 = h->V2.p; o.vp = h->vp.p; o.wp = h->wp.p; o.ip = h->ip.p;
    Work &w = h->work;
    w.r = h->r.p; w.p0 = h->p0.p; w.p1 = h->p1.p; w.q = h->q.p;
    w.partials = h->partials.p; w.hist = h->hist.p; w.st = h->st.p; w.args = h->args.p;
}

int scale_planes(mas_pcg *h, double dt, cudaStream_t s)
{
    PlaneSet ps;
    ps.V2 = h->V2.p; ps.SD = h->SD.p; ps.CP = h->CP.p; ps.CRoff = h->CRoff.p; ps.CT = h->CT.p;
    ps.E = h->E.p; ps.F = h->F.p; ps.AR = h->AR.p; ps.AT = h->AT.p; ps.Dinv = h->Dinv.p;
    ps.nr = h->nr; ps.nt = h->nt; ps.vp0 = h->vp0; ps.wp0 = h->wp0;
    const int total = (h->nr + 1) * (h->nt + 1);
    k_scale_planes<<<(total + 255) / 256, 256, 0, s>>>(ps, dt);
    CK(cudaGetLastError());
    h->dt = dt;
    return MAS_OK;
}

}  // namespace

extern "C" const char *mas_pcg_strerror(int status)
{
    switch (status) {
        case MAS_OK: return "converged";
        case MAS_MAXIT: return "iteration cap reached before rtol";
        case MAS_EINVAL: return "invalid argument";
        case MAS_ENOMEM: return "out of memory";
        case MAS_ECUDA: return "CUDA runtime error (no device, or a launch failed)";
        case MAS_EBREAKDOWN: return "PCG breakdown: p.Ap <= 0 or non-finite";
        default: return "unknown status";
    }
}

extern "C" void mas_pcg_destroy(mas_pcg_t *h)
{
    if (!h) return;
    if (h->exec) cudaGraphExecDestroy(h->exec);
    if (h->graph) cudaGraphDestroy(h->graph);
    DevBuf<double> *bufs[] = {&h->V2, &h->SD, &h->CP, &h->CRoff, &h->CT, &h->E, &h->F, &h->AR, &h->AT, &h->Dinv,
                              &h->vp, &h->wp, &h->ip, &h->Vinv, &h->r, &h->p0, &h->p1, &h->q, &h->partials, &h->hist,
                              &h->bdev, &h->xdev};
    for (DevBuf<double> *b : bufs) b->release();
    h->st.release();
    h->args.release();
    if (h->h_args) cudaFreeHost(h->h_args);
    if (h->h_st) cudaFreeHost(h->h_st);
    if (h->h_hist) cudaFreeHost(h->h_hist);
    cudaGetLastError();
    delete h;
}

extern "C" int mas_pcg_create(const mas_grid_t *g, const mas_metric_t *m, double dt, const mas_nu_t *nu,
                              const mas_bc_t *bc, mas_pcg_t **out)
{
    if (out) *out = nullptr;
    if (!g || !m || !nu || !bc || !out) return MAS_EINVAL;
    const int nr = g->nr, nt = g->nt, np = g->np;
    if (nr < 1 || nt < 1 || np < 2 || (np & 1)) return MAS_EINVAL;
    if ((long long)nr * nt * np >= (1LL << 31)) return MAS_EINVAL;          // 32-bit cell indices per row map
    if (!(dt >= 0.0) || !isfinite(dt)) return MAS_EINVAL;
    if (!m->r_c || !m->dr_c || !m->r_f || !m->dr_f || !m->sin_c || !m->dth_c || !m->sin_f || !m->dth_f ||
        !m->dph_c || !m->dph_f || !nu->v)
        return MAS_EINVAL;
    if ((bc->r_inner != MAS_BC_DIRICHLET && bc->r_inner != MAS_BC_NEUMANN) ||
        (bc->r_outer != MAS_BC_DIRICHLET && bc->r_outer != MAS_BC_NEUMANN))
        return MAS_EINVAL;
    if (nu->kind != 0 && nu->kind != 1) return MAS_EINVAL;
    if (!positive(m->r_c, 0, nr) || !positive(m->dr_c, 0, nr) || !positive(m->r_f, 0, nr + 1) ||
        !positive(m->dr_f, 0, nr + 1) || !positive(m->sin_c, 0, nt) || !positive(m->dth_c, 0, nt) ||
        !positive(m->dth_f, 1, nt) || !positive(m->sin_f, 1, nt) || !positive(m->dph_c, 0, np) ||
        !positive(m->dph_f, 0, np))
        return MAS_EINVAL;
    for (int i = 0; i < nr; i++)
        if (!(m->r_f[i] < m->r_f[i + 1])) return MAS_EINVAL;               // monotone mesh
    if (!positive(nu->v, 0, nu->kind == 0 ? 1 : nr * nt)) return MAS_EINVAL;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return MAS_ECUDA;                                                  // no CPU fallback
    }
    mas_pcg *h = new (std::nothrow) mas_pcg();
    if (!h) return MAS_ENOMEM;
    h->nr = nr; h->nt = nt; h->np = np;
    h->n = (size_t)nr * nt * np;
    if (cudaGetDevice(&h->device) != cudaSuccess ||
        cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, h->device) != cudaSuccess)
        return fail(h, MAS_ECUDA);

    // ---- coefficient planes (R1; the paper prints no discrete operator) ----
    const int nrows = nr * nt;
    std::vector<double> V2(nrows), CP(nrows), SD(nrows), CRf((size_t)(nr + 1) * nt), CRoff((size_t)(nr + 1) * nt),
        CT((size_t)nr * (nt + 1)), vp(np), ip(np), wp(np);
    for (int i = 0; i < nr; i++)
        for (int j = 0; j < nt; j++) {
            const double area_rt = m->sin_c[j] * m->dth_c[j];
            V2[i * nt + j] = m->r_c[i] * m->r_c[i] * m->dr_c[i] * area_rt;
            CP[i * nt + j] = nu_at(nu, nt, i, j) * m->dr_c[i] * m->dth_c[j] / m->sin_c[j];
        }
    for (int i = 0; i <= nr; i++)
        for (int j = 0; j < nt; j++) {
            const int il = i > 0 ? i - 1 : 0, ih = i < nr ? i : nr - 1;
            const double nuf = 0.5 * (nu_at(nu, nt, il, j) + nu_at(nu, nt, ih, j));
            double c = nuf * (m->r_f[i] * m->r_f[i]) * (m->sin_c[j] * m->dth_c[j]) / m->dr_f[i];
            const bool boundary = (i == 0 || i == nr);
            if (i == 0 && bc->r_inner == MAS_BC_NEUMANN) c = 0.0;
            if (i == nr && bc->r_outer == MAS_BC_NEUMANN) c = 0.0;
            CRf[(size_t)i * nt + j] = c;                        // enters the diagonal (Dirichlet face)
            CRoff[(size_t)i * nt + j] = boundary ? 0.0 : c;     // no off-diagonal partner on a boundary
        }
    for (int i = 0; i < nr; i++)
        for (int j = 0; j <= nt; j++) {
            double c = 0.0;                                     // polar faces: zero area
            if (j > 0 && j < nt)
                c = 0.5 * (nu_at(nu, nt, i, j - 1) + nu_at(nu, nt, i, j)) * m->dr_c[i] * m->sin_f[j] / m->dth_f[j];
            CT[(size_t)i * (nt + 1) + j] = c;
        }
    for (int i = 0; i < nr; i++)
        for (int j = 0; j < nt; j++)
            SD[i * nt + j] = CRf[(size_t)i * nt + j] + CRf[(size_t)(i + 1) * nt + j] + CT[(size_t)i * (nt + 1) + j] +
                             CT[(size_t)i * (nt + 1) + j + 1];
    h->uniform_phi = 1;
    for (int k = 0; k < np; k++) {
        vp[k] = m->dph_c[k];
        ip[k] = 1.0 / m->dph_f[k];
        if (m->dph_c[k] != m->dph_c[0] || m->dph_f[k] != m->dph_f[0]) h->uniform_phi = 0;
    }
    for (int k = 0; k < np; k++) wp[k] = ip[k] + ip[(k + np - 1) % np];
    std::vector<double> Vinv(nrows);
    double gmax = 0.0;                                      // max_k wp[k]/vp[k]
    for (int k = 0; k < np; k++) gmax = fmax(gmax, wp[k] / vp[k]);
    for (int t = 0; t < nrows; t++) {
        Vinv[t] = 1.0 / V2[t];
        h->lambda_max = fmax(h->lambda_max, 2.0 * (SD[t] + CP[t] * gmax) / V2[t]);
    }
    h->vp0 = vp[0];
    h->wp0 = wp[0];
    h->ip0 = ip[0];

    int rc;
    if ((rc = upload(h->V2, V2)) || (rc = upload(h->CP, CP)) || (rc = upload(h->SD, SD)) ||
        (rc = upload(h->CRoff, CRoff)) || (rc = upload(h->CT, CT)) || (rc = upload(h->vp, vp)) ||
        (rc = upload(h->wp, wp)) || (rc = upload(h->ip, ip)) || (rc = upload(h->Vinv, Vinv)))
        return fail(h, rc);
    if (h->E.alloc(nrows) || h->F.alloc(nrows) || h->Dinv.alloc(nrows) || h->AR.alloc((size_t)(nr + 1) * nt) ||
        h->AT.alloc((size_t)nr * (nt + 1)) || h->r.alloc(h->n) || h->p0.alloc(h->n) || h->p1.alloc(h->n) ||
        h->q.alloc(h->n) || h->partials.alloc(8 * (size_t)MAX_PARTIALS) || h->st.alloc(1) || h->args.alloc(1)) {
        cudaGetLastError();
        return fail(h, MAS_ENOMEM);
    }
    h->hist_cap = 1 << 13;
    if (h->hist.alloc(h->hist_cap) != cudaSuccess) return fail(h, MAS_ENOMEM);
    if (cudaMallocHost((void **)&h->h_args, sizeof(SolveArgs)) != cudaSuccess ||
        cudaMallocHost((void **)&h->h_st, sizeof(State)) != cudaSuccess ||
        cudaMallocHost((void **)&h->h_hist, h->hist_cap * sizeof(double)) != cudaSuccess)
        return fail(h, MAS_ENOMEM);
    if (cudaMemset(h->st.p, 0, sizeof(State)) != cudaSuccess) return fail(h, MAS_ECUDA);
    if (cudaMemset(h->p0.p, 0, h->n * sizeof(double)) != cudaSuccess ||
        cudaMemset(h->p1.p, 0, h->n * sizeof(double)) != cudaSuccess)
        return fail(h, MAS_ECUDA);
    fill_op(h);
    if (cudaDeviceGetAttribute(&h->coop_ok, cudaDevAttrCooperativeLaunch, h->device) != cudaSuccess) h->coop_ok = 0;
    if ((rc = scale_planes(h, dt, nullptr)) != MAS_OK) return fail(h, rc);
    if (cudaDeviceSynchronize() != cudaSuccess) return fail(h, MAS_ECUDA);
    *out = h;
    return MAS_OK;
}

// =============================================================================================
// launch descriptions
// =============================================================================================
namespace {

struct LoopCtx {                     // storage that kernel argument pointers refer to
    OpDev op;
    Work work;
    cudaGraphConditionalHandle cond;
    int use_cond;
    int reverse;
    const double *xin;
    const SolveArgs *args;
    double *y;
    MarchParams mp;
    WideParams wp;
    StencilParams sp, sp2;
};

int base_grid(const mas_pcg *h, const void *func, int nt_block)
{
    const int nv = h->np / 2;
    const int nvc = nv < nt_block ? nv : nt_block;
    const int rb = nt_block / nvc;
    const long long groups = ((long long)h->nr * h->nt + rb - 1) / rb;
    int occ = 1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, func, nt_block, 0) != cudaSuccess || occ < 1) {
        cudaGetLastError();
        occ = 1;
    }
    long long gsz = (long long)h->num_sms * occ;
    if (gsz > groups) gsz = groups;
    if (gsz > MAX_PARTIALS) gsz = MAX_PARTIALS;
    if (gsz < 1) gsz = 1;
    return (int)gsz;
}

bool use_xfuse(const mas_pcg *h) { return (h->xfuse && h->variant == 2) || h->variant == 3; }   // k1_tma is always xfuse
bool use_qrec(const mas_pcg *h) { return h->qrecompute && h->xfuse && h->variant == 2; }

void stencil_common(const mas_pcg *h, StencilParams &sp)
{
    memset(&sp, 0, sizeof(sp));
    sp.vp = h->vp0; sp.wp = h->wp0; sp.ip = h->ip0;
    sp.args = h->args.p;
}

KLaunch make_apply(const mas_pcg *h, LoopCtx &c)
{
    KLaunch k;
    if (h->apply_variant == 1) {                 // marching stencil kernel: S = A_sym (dt-scaled planes)
        stencil_common(h, c.sp);
        c.sp.E = h->E.p; c.sp.F = h->F.p; c.sp.AR = h->AR.p; c.sp.AT = h->AT.p;
        c.sp.u = c.xin; c.sp.out = c.y;
        stencil_configure_any(h->nr, h->nt, h->np, h->uniform_phi, EPI_APPLY, h->stencil_tile, h->num_sms, &c.sp,
                              &k.func, &k.grid, &k.block, &k.smem);
        k.args[0] = &c.op; k.args[1] = &c.sp;
        k.nargs = 2;
        return k;
    }
    k.func = (const void *)k_apply<NT_BASE>;
    k.block = dim3(NT_BASE);
    k.grid = dim3(base_grid(h, k.func, NT_BASE));
    k.args[0] = &c.op; k.args[1] = &c.xin; k.args[2] = &c.args; k.args[3] = &c.y;
    k.nargs = 4;
    return k;
}

KLaunch make_init(const mas_pcg *h, LoopCtx &c)
{
    KLaunch k;
    k.func = h->uniform_phi ? (const void *)k_init<NT_BASE, true> : (const void *)k_init<NT_BASE, false>;
    k.block = dim3(NT_BASE);
    k.grid = dim3(base_grid(h, k.func, NT_BASE));
    k.args[0] = &c.op; k.args[1] = &c.work; k.args[2] = &c.cond; k.args[3] = &c.use_cond;
    k.nargs = 4;
    return k;
}

KLaunch make_k2(const mas_pcg *h, LoopCtx &c)
{
    KLaunch k;
    if (use_qrec(h)) {                           // marching stencil kernel: q = A p recomputed, r updated in place
        stencil_common(h, c.sp2);
        c.sp2.E = h->E.p; c.sp2.F = h->F.p; c.sp2.AR = h->AR.p; c.sp2.AT = h->AT.p; c.sp2.Dinv = h->Dinv.p;
        c.sp2.w = c.work; c.sp2.cond = c.cond; c.sp2.use_cond = c.use_cond;
        stencil_configure(h->nr, h->nt, h->np, h->uniform_phi, EPI_K2R, h->k2r_tile, h->num_sms, &c.sp2, &k.func,
                          &k.grid, &k.block, &k.smem);
        k.args[0] = &c.op; k.args[1] = &c.sp2;
        k.nargs = 2;
        return k;
    }
    const bool xf = use_xfuse(h);
    if (xf)
        k.func = h->uniform_phi ? (const void *)k2_vec<NT_BASE, true, true> : (const void *)k2_vec<NT_BASE, false, true>;
    else
        k.func = h->uniform_phi ? (const void *)k2_vec<NT_BASE, true, false> : (const void *)k2_vec<NT_BASE, false, false>;
    k.block = dim3(NT_BASE);
    k.grid = dim3(base_grid(h, k.func, NT_BASE));
    c.reverse = h->serpentine;
    k.args[0] = &c.op; k.args[1] = &c.work; k.args[2] = &c.cond; k.args[3] = &c.use_cond; k.args[4] = &c.reverse;
    k.nargs = 5;
    return k;
}

KLaunch make_xtail(const mas_pcg *h, LoopCtx &c)
{
    KLaunch k;
    k.func = (const void *)k_xtail<NT_BASE>;
    k.block = dim3(NT_BASE);
    k.grid = dim3(base_grid(h, k.func, NT_BASE));
    k.args[0] = &c.op; k.args[1] = &c.work;
    k.nargs = 2;
    return k;
}



KLaunch make_k1(const mas_pcg *h, LoopCtx &c)
{
    KLaunch k;
    if (h->variant == 0) {
        k.func = h->uniform_phi ? (const void *)k1_v0<NT_BASE, true> : (const void *)k1_v0<NT_BASE, false>;
        k.block = dim3(NT_BASE);
        k.grid = dim3(base_grid(h, k.func, NT_BASE));
        k.args[0] = &c.op; k.args[1] = &c.work; k.args[2] = &c.cond; k.args[3] = &c.use_cond;
        k.nargs = 4;
        return k;
    }
    if (h->variant == 3) {
        k1_tma_configure(h->nr, h->nt, h->np, h->uniform_phi, h->tile, h->num_sms, h->ci_force, &c.wp, &k.func, &k.grid,
                         &k.block, &k.smem);
        c.wp.vp = h->vp0; c.wp.wp = h->wp0; c.wp.ip = h->ip0;
        k.args[0] = &c.op; k.args[1] = &c.work; k.args[2] = &c.wp; k.args[3] = &c.cond; k.args[4] = &c.use_cond;
        k.nargs = 5;
        return k;
    }
    if (h->variant == 1) {
        march_configure(h->nr, h->nt, h->np, h->uniform_phi, h->tile, h->num_sms, &c.mp, &k.func, &k.grid, &k.block,
                        &k.smem);
        k.args[2] = &c.mp;
    } else {
        wide_configure(h->nr, h->nt, h->np, h->uniform_phi, use_qrec(h) ? 2 : (use_xfuse(h) ? 1 : 0), h->tile, h->num_sms, h->ci_force, &c.wp,
                       &k.func, &k.grid, &k.block, &k.smem);
        c.wp.vp = h->vp0; c.wp.wp = h->wp0; c.wp.ip = h->ip0;
        k.args[2] = &c.wp;
    }
    k.args[0] = &c.op; k.args[1] = &c.work; k.args[3] = &c.cond; k.args[4] = &c.use_cond;
    k.nargs = 5;
    return k;
}

cudaError_t launch(const KLaunch &k, cudaStream_t s)
{
    return cudaLaunchKernel(k.func, k.grid, k.block, const_cast<void **>(k.args), k.smem, s);
}

cudaError_t add_node(cudaGraphNode_t *node, cudaGraph_t g, const cudaGraphNode_t *dep, const KLaunch &k)
{
    cudaKernelNodeParams p;
    memset(&p, 0, sizeof(p));
    p.func = const_cast<void *>(k.func);
    p.gridDim = k.grid;
    p.blockDim = k.block;
    p.sharedMemBytes = (unsigned)k.smem;
    p.kernelParams = const_cast<void **>(k.args);
    p.extra = nullptr;
    return cudaGraphAddKernelNode(node, g, dep, dep ? 1 : 0, &p);
}

void drop_graph(mas_pcg *h)
{
    if (h->exec) cudaGraphExecDestroy(h->exec);
    if (h->graph) cudaGraphDestroy(h->graph);
    h->exec = nullptr;
    h->graph = nullptr;
    h->graph_dirty = true;
}

// graph = [A x0 -> q] -> [init] -> WHILE(cond){ K1 -> K2 }   (call stack 2)
int build_graph(mas_pcg *h)
{
    drop_graph(h);
    LoopCtx c;
    c.op = h->op; c.work = h->work; c.use_cond = 1; c.xin = nullptr; c.args = h->args.p; c.y = h->q.p;
    cudaGraph_t g = nullptr;
    if (cudaGraphCreate(&g, 0) != cudaSuccess) { cudaGetLastError(); return MAS_ECUDA; }
    h->graph = g;
    if (cudaGraphConditionalHandleCreate(&c.cond, g, 1, cudaGraphCondAssignDefault) != cudaSuccess) {
        cudaGetLastError();
        return MAS_ECUDA;
    }
    cudaGraphNode_t n_apply, n_init, n_while, n_k1, n_k2;
    const KLaunch ka = make_apply(h, c), ki = make_init(h, c);
    if (add_node(&n_apply, g, nullptr, ka) != cudaSuccess || add_node(&n_init, g, &n_apply, ki) != cudaSuccess) {
        cudaGetLastError();
        return MAS_ECUDA;
    }
    cudaGraphNodeParams wp = {cudaGraphNodeTypeConditional};
    wp.conditional.handle = c.cond;
    wp.conditional.type = cudaGraphCondTypeWhile;
    wp.conditional.size = 1;
    if (cudaGraphAddNode(&n_while, g, &n_init, 1, &wp) != cudaSuccess) { cudaGetLastError(); return MAS_ECUDA; }
    cudaGraph_t body = wp.conditional.phGraph_out[0];
    const KLaunch k1 = make_k1(h, c), k2 = make_k2(h, c);
    // `unroll` iterations per WHILE trip: the conditional node is evaluated once per trip, and K1 / K2 return
    // at once when the loop has ended (device flag), so extra pairs after convergence cost two empty launches.
    // Edges inside the body are programmatic (PDL) when both kernels wait with cudaGridDependencySynchronize
    // (k1_wide and k2_vec): the successor's blocks launch while the predecessor drains and run the part of
    // their prologue that does not depend on it.
    const bool pdl = h->pdl && h->variant >= 2 && !use_qrec(h);
    cudaGraphNode_t prev = nullptr;
    for (int u = 0; u < 2 * h->unroll; u++) {
        cudaGraphNode_t node;
        if (add_node(&node, body, nullptr, (u & 1) ? k2 : k1) != cudaSuccess) { cudaGetLastError(); return MAS_ECUDA; }
        if (prev) {
            cudaGraphEdgeData ed;
            memset(&ed, 0, sizeof(ed));
            if (pdl) {
                ed.type = cudaGraphDependencyTypeProgrammatic;
                ed.from_port = cudaGraphKernelNodePortProgrammatic;
            }
            if (cudaGraphAddDependencies_v2(body, &prev, &node, &ed, 1) != cudaSuccess) {
                cudaGetLastError();
                return MAS_ECUDA;
            }
        }
        prev = node;
    }
    (void)n_k1; (void)n_k2;
    if (use_xfuse(h)) {
        cudaGraphNode_t n_tail;
        const KLaunch kt = make_xtail(h, c);
        if (add_node(&n_tail, g, &n_while, kt) != cudaSuccess) { cudaGetLastError(); return MAS_ECUDA; }
    }
    if (cudaGraphInstantiate(&h->exec, g, 0) != cudaSuccess) {
        cudaGetLastError();
        h->exec = nullptr;
        return MAS_ECUDA;
    }
    h->graph_dirty = false;
    return MAS_OK;
}

int ensure_hist(mas_pcg *h, int maxit)
{
    const size_t need = (size_t)maxit + 1;
    if (need <= h->hist_cap) return MAS_OK;
    size_t cap = h->hist_cap;
    while (cap < need) cap *= 2;
    if (h->hist.alloc(cap) != cudaSuccess) { cudaGetLastError(); return MAS_ENOMEM; }
    if (h->h_hist) cudaFreeHost(h->h_hist);
    h->h_hist = nullptr;
    if (cudaMallocHost((void **)&h->h_hist, cap * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return MAS_ENOMEM; }
    h->hist_cap = cap;
    fill_op(h);
    drop_graph(h);              // kernel nodes hold the old hist pointer
    return MAS_OK;
}

bool aligned16(const void *p) { return ((uintptr_t)p & 15u) == 0; }

constexpr long long PERSIST_AUTO_CELLS = 1LL << 40;   // auto mode: measured faster wherever the state fits on chip
                                                      // (config 1: 2.0x, config 2 = 786 k cells: 1.46x)

// Plan the one-kernel solve; returns false when it does not apply (too large, no cooperative launch, off).
bool plan_persistent(const mas_pcg *h, PersistParams *pp, int *grid, size_t *smem, const void **func)
{
    if (!h->persistent || !h->coop_ok) return false;
    if (h->persistent == 2 && (long long)h->n > PERSIST_AUTO_CELLS) return false;
    const long long nvec = (long long)h->n / 2;
    long long g = (nvec + PNT - 1) / PNT;
    if (g > h->num_sms) g = h->num_sms;
    const long long M = (nvec + g * PNT - 1) / (g * PNT);
    if (M > 64 || persist_smem((int)M) > (size_t)PMAX_SMEM) return false;
    *func = h->uniform_phi ? (const void *)k_pcg_persistent<true> : (const void *)k_pcg_persistent<false>;
    *smem = persist_smem((int)M);
    if (cudaFuncSetAttribute(*func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)*smem) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, *func, PNT, *smem) != cudaSuccess || occ < 1) {
        cudaGetLastError();
        return false;
    }
    pp->Z = h->r.p; pp->P0 = h->p0.p; pp->P1 = h->p1.p;
    pp->partials = h->partials.p; pp->hist = h->hist.p; pp->st = h->st.p; pp->args = h->args.p;
    pp->nvec = (int)nvec; pp->M = (int)M;
    *grid = (int)g;
    return true;
}

}  // namespace

extern "C" int mas_pcg_set_dt(mas_pcg_t *h, double dt, void *stream)
{
    if (!h || !(dt >= 0.0) || !isfinite(dt)) return MAS_EINVAL;
    return scale_planes(h, dt, (cudaStream_t)stream);
}

extern "C" int mas_pcg_apply(mas_pcg_t *h, const double *x_dev, double *y_dev, void *stream)
{
    if (!h || !x_dev || !y_dev || x_dev == y_dev || !aligned16(x_dev) || !aligned16(y_dev)) return MAS_EINVAL;
    LoopCtx c;
    c.op = h->op; c.xin = x_dev; c.args = h->args.p; c.y = y_dev;
    CK(launch(make_apply(h, c), (cudaStream_t)stream));
    return MAS_OK;
}

extern "C" int mas_pcg_set_option(mas_pcg_t *h, const char *name, int value)
{
    if (!h || !name) return MAS_EINVAL;
    if (!strcmp(name, "loop_mode")) {
        if (value != 0 && value != 1) return MAS_EINVAL;
        h->loop_mode = value;
    } else if (!strcmp(name, "variant")) {
        if (value < 0 || value > 3) return MAS_EINVAL;
        h->variant = value;
        h->tile = 0;
    } else if (!strcmp(name, "tile")) {
        const int nt_ = h->variant == 1 ? march_num_tiles() : (h->variant == 2 ? wide_num_tiles() : (h->variant == 3 ? k1_tma_num_tiles() : 1));
        if (value < 0 || value >= nt_) return MAS_EINVAL;
        h->tile = value;
    } else if (!strcmp(name, "apply_variant")) {
        if (value != 0 && value != 1) return MAS_EINVAL;
        h->apply_variant = value;
    } else if (!strcmp(name, "stencil_tile")) {
        if (value < 0 || value >= stencil_num_tiles_any()) return MAS_EINVAL;
        h->stencil_tile = value;
    } else if (!strcmp(name, "serpentine")) {
        if (value != 0 && value != 1) return MAS_EINVAL;
        h->serpentine = value;
    } else if (!strcmp(name, "pdl")) {
        if (value != 0 && value != 1) return MAS_EINVAL;
        h->pdl = value;
    } else if (!strcmp(name, "unroll")) {
        if (value < 1 || value > 16) return MAS_EINVAL;
        h->unroll = value;
    } else if (!strcmp(name, "persistent")) {
        if (value < 0 || value > 2) return MAS_EINVAL;
        h->persistent = value;
    } else if (!strcmp(name, "qrecompute")) {
        if (value != 0 && value != 1) return MAS_EINVAL;
        h->qrecompute = value;
    } else if (!strcmp(name, "k2r_tile")) {
        if (value < 0 || value >= stencil_num_tiles()) return MAS_EINVAL;
        h->k2r_tile = value;
    } else if (!strcmp(name, "xfuse")) {
        if (value != 0 && value != 1) return MAS_EINVAL;
        h->xfuse = value;
    } else if (!strcmp(name, "ci")) {
        if (value < 0 || value > MARCH_CI_MAX) return MAS_EINVAL;
        h->ci_force = value;
    } else {
        return MAS_EINVAL;
    }
    h->graph_dirty = true;
    return MAS_OK;
}

extern "C" int mas_pcg_stats(const mas_pcg_t *h, long long *out)
{
    if (!h || !out) return MAS_EINVAL;
    memcpy(out, h->stats, sizeof(h->stats));
    return MAS_OK;
}

extern "C" int mas_pcg_solve(mas_pcg_t *h, const double *b_dev, double *x_dev, double rtol, int maxit, void *stream,
                             int *iters_out, double *reshist_host)
{
    if (!h || !b_dev || !x_dev || b_dev == x_dev || !(rtol >= 0.0) || maxit < 0 || !aligned16(b_dev) ||
        !aligned16(x_dev))
        return MAS_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    int rc = ensure_hist(h, maxit);
    if (rc != MAS_OK) return rc;

    h->h_args->b = b_dev; h->h_args->x = x_dev; h->h_args->rtol = rtol; h->h_args->maxit = maxit; h->h_args->pad = 0;
    CK(cudaMemcpyAsync(h->args.p, h->h_args, sizeof(SolveArgs), cudaMemcpyHostToDevice, s));

    int mode = h->loop_mode;
    PersistParams ppar;
    int pgrid = 0;
    size_t psmem = 0;
    const void *pfunc = nullptr;
    const bool persistent = plan_persistent(h, &ppar, &pgrid, &psmem, &pfunc);
    long long launched_outside = 2, launched_loop = 0;
    if (persistent) {                      // init + loop + finish in one cooperative kernel
        OpDev op = h->op;
        void *kargs[2] = {&op, &ppar};
        if (cudaLaunchCooperativeKernel(pfunc, dim3(pgrid), dim3(PNT), kargs, psmem, s) == cudaSuccess) {
            mode = 2;
            launched_outside = 0;
            launched_loop = 1;
        } else {
            cudaGetLastError();            // refused (e.g. co-residency limits): use the streaming loop instead
            h->coop_ok = 0;
        }
    }
    if (mode == 1 && (h->graph_dirty || !h->exec)) {
        if (build_graph(h) != MAS_OK && h->pdl) {   // programmatic edges refused: plain edges
            h->pdl = 0;
            drop_graph(h);
        }
        if ((h->graph_dirty || !h->exec) && build_graph(h) != MAS_OK) {
            drop_graph(h);                    // driver without conditional nodes: fall back, and say so in stats
            mode = 0;
        }
    }
    if (mode == 2) {
        // launched above
    } else if (mode == 1) {
        CK(cudaGraphLaunch(h->exec, s));
    } else {
        LoopCtx c;
        c.op = h->op; c.work = h->work; c.use_cond = 0; c.xin = nullptr; c.args = h->args.p; c.y = h->q.p;
        memset(&c.cond, 0, sizeof(c.cond));
        CK(launch(make_apply(h, c), s));
        CK(launch(make_init(h, c), s));
        const KLaunch k1 = make_k1(h, c), k2 = make_k2(h, c);
        for (int done = 0; done < maxit;) {
            CK(cudaMemcpyAsync(h->h_st, h->st.p, sizeof(State), cudaMemcpyDeviceToHost, s));
            CK(cudaStreamSynchronize(s));
            if (!h->h_st->active) break;
            const int chunk = maxit - done < HOST_CHUNK ? maxit - done : HOST_CHUNK;
            for (int it = 0; it < chunk; it++) {
                CK(launch(k1, s));
                CK(launch(k2, s));
            }
            launched_loop += 2LL * chunk;
            done += chunk;
        }
        if (use_xfuse(h)) CK(launch(make_xtail(h, c), s));
    }
    if (use_xfuse(h) && mode != 2) launched_outside += 1;
    CK(cudaMemcpyAsync(h->h_st, h->st.p, sizeof(State), cudaMemcpyDeviceToHost, s));
    CK(cudaMemcpyAsync(h->h_hist, h->hist.p, ((size_t)maxit + 1) * sizeof(double), cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));          // the one host sync of a graph-mode solve
    const State &st = *h->h_st;
    if (st.bb == 0.0) {                    // zero right-hand side: x = 0
        CK(cudaMemsetAsync(x_dev, 0, h->n * sizeof(double), s));
        CK(cudaStreamSynchronize(s));
    }
    if (iters_out) *iters_out = st.k;
    if (reshist_host) memcpy(reshist_host, h->h_hist, ((size_t)st.k + 1) * sizeof(double));
    h->loop_mode_used = mode;
    h->stats[0] = mode == 1 ? (long long)st.launches : launched_loop;
    h->stats[6] = mode == 2 ? pgrid : 0;
    h->stats[7] = (mode == 1 && h->pdl && h->variant >= 2 && !use_qrec(h)) ? 1 : 0;
    h->stats[1] = launched_outside;
    h->stats[2] = mode;
    // unfused: K1 r,p -> p,q (4N); K2 x,p,r,q -> x,r (6N).  xfuse: K1 r,p,x -> p,q,x (6N); K2 r,q -> r (3N)
    h->stats[4] = use_qrec(h) ? 5 : (use_xfuse(h) ? 6 : 4);
    h->stats[5] = use_xfuse(h) ? 3 : 6;
    h->stats[3] = 8 * (h->stats[4] + h->stats[5]);
    return st.status;
}

extern "C" int mas_pcg_solve_host(mas_pcg_t *h, const double *b_host, double *x_host, double rtol, int maxit,
                                  void *stream, int *iters_out, double *reshist_host)
{
    if (!h || !b_host || !x_host) return MAS_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    if (!h->bdev.p && h->bdev.alloc(h->n) != cudaSuccess) { cudaGetLastError(); return MAS_ENOMEM; }
    if (!h->xdev.p && h->xdev.alloc(h->n) != cudaSuccess) { cudaGetLastError(); return MAS_ENOMEM; }
    const size_t bytes = h->n * sizeof(double);
    CK(cudaMemcpyAsync(h->bdev.p, b_host, bytes, cudaMemcpyHostToDevice, s));
    CK(cudaMemcpyAsync(h->xdev.p, x_host, bytes, cudaMemcpyHostToDevice, s));
    const int rc = mas_pcg_solve(h, h->bdev.p, h->xdev.p, rtol, maxit, stream, iters_out, reshist_host);
    if (rc < 0) return rc;
    CK(cudaMemcpyAsync(x_host, h->xdev.p, bytes, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    return rc;
}

extern "C" int mas_pcg_profile(mas_pcg_t *h, const double *b_dev, double *x_dev, int nit, void *stream, double *ms_out)
{
    if (!h || !b_dev || !x_dev || b_dev == x_dev || !ms_out || nit < 1 || nit > 256 || !aligned16(b_dev) ||
        !aligned16(x_dev))
        return MAS_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    h->h_args->b = b_dev; h->h_args->x = x_dev; h->h_args->rtol = 0.0; h->h_args->maxit = nit; h->h_args->pad = 0;
    int rc = ensure_hist(h, nit);
    if (rc != MAS_OK) return rc;
    CK(cudaMemcpyAsync(h->args.p, h->h_args, sizeof(SolveArgs), cudaMemcpyHostToDevice, s));
    LoopCtx c;
    c.op = h->op; c.work = h->work; c.use_cond = 0; c.xin = nullptr; c.args = h->args.p; c.y = h->q.p;
    memset(&c.cond, 0, sizeof(c.cond));
    std::vector<cudaEvent_t> ev(2 * (size_t)nit + 1);
    for (cudaEvent_t &e : ev) CK(cudaEventCreate(&e));
    CK(launch(make_apply(h, c), s));
    CK(launch(make_init(h, c), s));
    const KLaunch k1 = make_k1(h, c), k2 = make_k2(h, c);
    CK(cudaEventRecord(ev[0], s));
    for (int it = 0; it < nit; it++) {
        CK(launch(k1, s));
        CK(cudaEventRecord(ev[2 * it + 1], s));
        CK(launch(k2, s));
        CK(cudaEventRecord(ev[2 * it + 2], s));
    }
    CK(cudaStreamSynchronize(s));
    double sum1 = 0, sum2 = 0, min1 = 1e30, min2 = 1e30;
    for (int it = 0; it < nit; it++) {
        float a = 0, b = 0;
        CK(cudaEventElapsedTime(&a, ev[2 * it], ev[2 * it + 1]));
        CK(cudaEventElapsedTime(&b, ev[2 * it + 1], ev[2 * it + 2]));
        sum1 += a; sum2 += b;
        if (a < min1) min1 = a;
        if (b < min2) min2 = b;
    }
    for (cudaEvent_t &e : ev) cudaEventDestroy(e);
    ms_out[0] = sum1 / nit; ms_out[1] = sum2 / nit; ms_out[2] = min1; ms_out[3] = min2;
    h->stats[4] = use_qrec(h) ? 5 : (use_xfuse(h) ? 6 : 4);
    h->stats[5] = use_xfuse(h) ? 3 : 6;
    h->stats[3] = 8 * (h->stats[4] + h->stats[5]);
    return MAS_OK;
}

// =============================================================================================
// NEXT-1: explicit viscosity advance by RKL2 super time stepping (R7)
// =============================================================================================
namespace {

double rkl2_b(int j) { return j < 3 ? 1.0 / 3.0 : ((double)j * j + j - 2.0) / (2.0 * j * (j + 1.0)); }

void sts_planes(const mas_pcg *h, StencilParams &sp)
{
    stencil_common(h, sp);                       // S = L_sym: the dt-independent planes
    sp.E = h->SD.p; sp.F = h->CP.p; sp.AR = h->CRoff.p; sp.AT = h->CT.p; sp.Vinv = h->Vinv.p;
}

int launch_stencil(const mas_pcg *h, StencilParams &sp, int epi, cudaStream_t s)
{
    KLaunch k;
    OpDev op = h->op;
    stencil_configure_any(h->nr, h->nt, h->np, h->uniform_phi, epi, h->stencil_tile, h->num_sms, &sp, &k.func, &k.grid,
                          &k.block, &k.smem);
    k.args[0] = &op; k.args[1] = &sp;
    CK(launch(k, s));
    return MAS_OK;
}

}  // namespace

extern "C" int mas_pcg_lambda_max(const mas_pcg_t *h, double *out)
{
    if (!h || !out) return MAS_EINVAL;
    *out = h->lambda_max;
    return MAS_OK;
}

extern "C" int mas_sts_stages(const mas_pcg_t *h, double tau, int *s_out)
{
    if (!h || !s_out || !(tau >= 0.0) || !isfinite(tau)) return MAS_EINVAL;
    // stable iff tau <= (s^2 + s - 2)/4 * 2/lambda_max
    const double need = 2.0 * tau * h->lambda_max;          // s^2 + s - 2 >= need
    long long s = (long long)ceil(0.5 * (-1.0 + sqrt(9.0 + 4.0 * need)));
    if (s < 2) s = 2;
    while ((double)s * s + s - 2.0 < need) ++s;
    if (s > (1LL << 30)) return MAS_EINVAL;
    *s_out = (int)s;
    return MAS_OK;
}

extern "C" int mas_pcg_lop(mas_pcg_t *h, const double *u_dev, double *y_dev, void *stream)
{
    if (!h || !u_dev || !y_dev || u_dev == y_dev || !aligned16(u_dev) || !aligned16(y_dev)) return MAS_EINVAL;
    StencilParams sp;
    sts_planes(h, sp);
    sp.u = u_dev; sp.out = y_dev; sp.c_u = 0.0; sp.c_L = 1.0;     // out = M u
    return launch_stencil(h, sp, EPI_STS, (cudaStream_t)stream);
}

extern "C" int mas_sts_advance(mas_pcg_t *h, double *u_dev, double tau, int s, void *stream)
{
    if (!h || !u_dev || !aligned16(u_dev) || s < 2 || !(tau >= 0.0) || !isfinite(tau)) return MAS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    double *my0 = h->q.p, *ya = h->p0.p, *yb = h->p1.p;           // the PCG workspaces double as stage buffers
    const double w1 = 4.0 / ((double)s * s + s - 2.0);
    StencilParams sp;
    // stage 1: Y_1 = Y_0 + mu~_1 tau M Y_0 ; keep M Y_0
    sts_planes(h, sp);
    sp.u = u_dev; sp.out = ya; sp.out2 = my0; sp.c_u = 1.0; sp.c_L = rkl2_b(1) * w1 * tau;
    int rc = launch_stencil(h, sp, EPI_STS, st);
    if (rc != MAS_OK) return rc;
    const double *yjm1 = ya, *yjm2 = u_dev;
    for (int j = 2; j <= s; j++) {
        const double bj = rkl2_b(j), bjm1 = rkl2_b(j - 1), bjm2 = rkl2_b(j - 2);
        const double mu = (2.0 * j - 1.0) / j * bj / bjm1;
        const double nu = -(j - 1.0) / j * bj / bjm2;
        const double mut = mu * w1, gat = -(1.0 - bjm1) * mut;
        // Y_j overwrites Y_{j-2}'s buffer (each cell is read by the thread that writes it), except that
        // Y_0 = u_dev must survive until the last stage, which writes the result into it.
        double *out = (j == s) ? u_dev : (yjm2 == u_dev ? yb : const_cast<double *>(yjm2));
        sts_planes(h, sp);
        sp.u = yjm1; sp.a1 = yjm2; sp.a2 = u_dev; sp.a3 = my0; sp.out = out;
        sp.c_u = mu; sp.c_a1 = nu; sp.c_a2 = 1.0 - mu - nu; sp.c_L = mut * tau; sp.c_a3 = gat * tau;
        rc = launch_stencil(h, sp, EPI_STS, st);
        if (rc != MAS_OK) return rc;
        yjm2 = yjm1;
        yjm1 = out;
    }
    h->graph_dirty = h->graph_dirty;             // PCG workspaces were clobbered; solves re-initialise them
    return MAS_OK;
}

// Measurement aid: sustained time of a trivial linear kernel with K1's (which = 6) or K2's (which = 3) DRAM mix
// over the handle's own N-vectors (their contents are destroyed; the next solve re-initialises them).
extern "C" int mas_pcg_mix_probe(mas_pcg_t *h, int which, int reps, void *stream, double *ms_out)
{
    if (!h || !ms_out || (which != 6 && which != 3) || reps < 1 || reps > 100000) return MAS_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    if (!h->bdev.p && h->bdev.alloc(h->n) != cudaSuccess) { cudaGetLastError(); return MAS_ENOMEM; }
    CK(cudaMemsetAsync(h->bdev.p, 0, h->n * sizeof(double), s));
    CK(cudaMemsetAsync(h->r.p, 0, h->n * sizeof(double), s));
    CK(cudaMemsetAsync(h->q.p, 0, h->n * sizeof(double), s));
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    const size_t n2 = h->n / 2;
    double best = 1e30;
    for (int mult = 4; mult <= 32; mult *= 2) {                 // the grid size matters by a few percent: take the best
        const int blocks = h->num_sms * mult;
        for (int pass = 0; pass < 2; pass++) {                  // pass 0 = warm-up
            const int n = pass ? reps : 3;
            CK(cudaEventRecord(e0, s));
            for (int r = 0; r < n; r++) {
                if (which == 6)
                    k_mix6<<<blocks, 256, 0, s>>>((const double2 *)h->r.p, (const double2 *)h->p0.p, (double2 *)h->bdev.p,
                                                  (double2 *)h->p1.p, (double2 *)h->q.p, n2);
                else
                    k_mix3<<<blocks, 256, 0, s>>>((double2 *)h->r.p, (const double2 *)h->q.p, n2);
            }
            CK(cudaEventRecord(e1, s));
            CK(cudaEventSynchronize(e1));
            float ms = 0;
            CK(cudaEventElapsedTime(&ms, e0, e1));
            if (pass && ms / n < best) best = ms / n;
        }
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    CK(cudaGetLastError());
    *ms_out = best;
    return MAS_OK;
}

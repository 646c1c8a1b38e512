// mas_pcg.cu -- C ABI (include/mas_pcg.h) of the B200-native MAS PCG path: handle, coefficient planes, workspaces,
// launch plans, the CUDA-graph WHILE loop and its host-chunk fallback, batched right-hand sides, r-slab groups.
// Every step of the numerical path runs in the kernels of kernels_*.cuh; this file only marshals.
// There is no CPU fallback.
#include "../../include/mas_pcg.h"

#include <cuda_runtime.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <memory>
#include <new>
#include <vector>

#include "common.cuh"
#include "kernels_base.cuh"
#include "tile.cuh"
#include "kernels_stencil_tma.cuh"
#include "kernels_k1_tma.cuh"
#include "kernels_persistent.cuh"
#include "kernels_pc2.cuh"

using namespace mas;

namespace {

constexpr int NT_BASE = 256;
constexpr int HOST_CHUNK = 16;       // iterations per poll in host-chunk mode
constexpr int CI_FORCE_MIN = 2;      // smallest r-chunk an option may force (bounds the largest grid, see pstride)

struct KLaunch {                     // one kernel launch, usable directly or as a graph node
    const void *func = nullptr;
    dim3 grid{1, 1, 1}, block{1, 1, 1};
    size_t smem = 0;
    void *args[8] = {};
};

template <typename T>
struct DevBuf {
    T *p = nullptr;
    size_t n = 0;
    cudaError_t alloc(size_t count)
    {
        release();
        const cudaError_t e = cudaMalloc((void **)&p, (count ? count : 1) * sizeof(T));
        if (e != cudaSuccess) p = nullptr;       // a failed buffer is an empty buffer
        else n = count;
        return e;
    }
    void release()
    {
        if (p) cudaFree(p);
        p = nullptr;
        n = 0;
    }
};

struct DeviceGuard {                 // entry points run on the handle's device, whatever the caller's current device is
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; cudaGetLastError(); return; }
        if (prev != dev && cudaSetDevice(dev) != cudaSuccess) { ok = false; cudaGetLastError(); }
        if (prev == dev) prev = -1;
    }
    ~DeviceGuard()
    {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

}  // namespace

struct mas_pcg {
    int nr = 0, nt = 0, np = 0;
    size_t n = 0;
    int device = 0, num_sms = 0;
    double dt = 0.0;
    int uniform_phi = 0;
    // device planes (global mesh)
    DevBuf<double> V2, SD, CP, CRoff, CT, E, F, AR, AT, Dinv, vp, wp, ip, Vinv;
    double lambda_max = 0.0;         // Gershgorin bound on the spectral radius of M = -V^-1 L_sym
    double vp0 = 0, wp0 = 0, ip0 = 0;
    // workspaces for `nrhs_cap` right-hand sides (vectors back to back, stride n)
    int nrhs_cap = 0;
    DevBuf<double> r, p0, p1, q, partials, hist, bdev, xdev;
    // PC2 (block-Jacobi ILU(0) on phi-line boxes; kernels_pc2.cuh): z vectors, 1/pivot in chunk order, ip in chunk order
    int precond = MAS_PC1;
    int pc2_M = 0;
    DevBuf<double> z, dinvT, ipT;
    int pstride = 0;
    DevBuf<State> st;
    DevBuf<SolveArgs> args;
    DevBuf<Ctl> ctl;
    DevBuf<unsigned> tickets;
    // pinned staging
    SolveArgs *h_args = nullptr;
    State *h_st = nullptr;           // [MAX_RHS]
    Ctl *h_ctl = nullptr;
    double *h_hist = nullptr;        // [MAX_RHS][hist_cap]
    size_t hist_cap = 0;
    // options
    int loop_mode = 1;               // requested: 1 graph-while, 0 host chunks
    int tile = -1;                   // K1 tile configuration id; -1 = automatic (k1_auto_tile)
    int ci_force = 0;                // >0: override the r-chunk length (tuning)
    int stencil_tile = 1;            // k_stencil_tma tile for apply / STS
    int k2r_tile = 1;                // k_stencil_tma tile for K2R
    int serpentine = 1;              // 1: K2 sweeps backward (L2 reuse across K1 -> K2 -> K1)
    int persistent = 1;              // 1: one cooperative kernel for the whole solve whenever the state fits on chip
    int coop_ok = 0, coop_refused = 0;
    int unroll = 4;                  // PCG iterations per WHILE trip of the graph loop (measured: +1 % c4, +3 % c3)
    int qrecompute = 0;              // 1: q is not stored, K2R recomputes it: 64 B/cell/iteration; 0: 72 B (default: faster)
    L2Plan l2{0};
    cudaGraph_t graph[MAX_RHS] = {};
    cudaGraphExec_t exec[MAX_RHS] = {};
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

void drop_graphs(mas_pcg *h)
{
    for (int j = 0; j < MAX_RHS; j++) {
        if (h->exec[j]) cudaGraphExecDestroy(h->exec[j]);
        if (h->graph[j]) cudaGraphDestroy(h->graph[j]);
        h->exec[j] = nullptr;
        h->graph[j] = nullptr;
    }
}

void fill_op(mas_pcg *h)
{
    OpDev &o = h->op;
    o.nr = h->nr; o.nt = h->nt; o.np = h->np; o.nv = h->np / 2;
    o.nrows = h->nr * h->nt;
    o.uniform_phi = h->uniform_phi;
    o.i_lo = 0; o.nr_glob = h->nr;
    o.n = (long long)h->n;
    o.E = h->E.p; o.F = h->F.p; o.AR = h->AR.p; o.AT = h->AT.p; o.Dinv = h->Dinv.p;
    o.V2 = h->V2.p; o.vp = h->vp.p; o.wp = h->wp.p; o.ip = h->ip.p;
    Work &w = h->work;
    memset(&w, 0, sizeof(w));
    w.r = h->r.p; w.p0 = h->p0.p; w.p1 = h->p1.p; w.q = h->q.p;
    w.z = h->z.p;
    w.vstride = (long long)h->n;
    w.partials = h->partials.p; w.pstride = h->pstride;
    w.hist = h->hist.p; w.hstride = (int)h->hist_cap;
    w.st = h->st.p; w.tickets = h->tickets.p; w.ctl = h->ctl.p; w.args = h->args.p;
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
    if (h->precond == MAS_PC2) {                 // the ILU(0) pivots depend on dt: factor again (stream order)
        const int lines = h->nr * h->nt;
        k_pc2_factor<<<(lines + 127) / 128, 128, 0, s>>>(h->op, h->dinvT.p, h->pc2_M);
        CK(cudaGetLastError());
    }
    return MAS_OK;
}

// Upper bound on gridDim.x of every reducing kernel any option can select: the marching kernels' smallest tile is
// 6 theta-rows x 128 phi-cells x CI_FORCE_MIN planes; the row kernels launch at most 32 blocks per SM.
int partials_stride(const mas_pcg *h)
{
    const long long nkt = (h->np + TILE_TK - 1) / TILE_TK, njt = (h->nt + 5) / 6, nit = (h->nr + CI_FORCE_MIN - 1) / CI_FORCE_MIN;
    long long g = nkt * njt * nit;
    if (g < 32LL * h->num_sms) g = 32LL * h->num_sms;
    return (int)g;
}

// vectors for `nrhs` right-hand sides (grown on the first batched solve)
int ensure_rhs_capacity(mas_pcg *h, int nrhs)
{
    if (nrhs <= h->nrhs_cap) return MAS_OK;
    drop_graphs(h);
    const size_t tot = h->n * (size_t)nrhs;
    auto give_up = [&](int code) {             // leave a handle that knows it has no vectors: every user of r / p0 / p1 / q
        cudaGetLastError();                    // (solves, mas_sts_advance) comes through here again and retries
        h->r.release(); h->p0.release(); h->p1.release(); h->q.release(); h->z.release();
        h->nrhs_cap = 0;
        fill_op(h);
        return code;
    };
    if (h->r.alloc(tot) || h->p0.alloc(tot) || h->p1.alloc(tot) || h->q.alloc(tot) ||
        (h->precond == MAS_PC2 && h->z.alloc(tot)))
        return give_up(MAS_ENOMEM);
    if (cudaMemset(h->p0.p, 0, tot * sizeof(double)) != cudaSuccess ||
        cudaMemset(h->p1.p, 0, tot * sizeof(double)) != cudaSuccess)
        return give_up(MAS_ECUDA);
    h->nrhs_cap = nrhs;
    fill_op(h);
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
        case MAS_ECUDA: return "CUDA runtime error (no device, a launch failed, or a kernel reported a protocol fault)";
        case MAS_EBREAKDOWN: return "PCG breakdown: p.Ap <= 0 or a non-finite scalar";
        case MAS_ETOOBIG: return "mesh has more cells than the fixed scratch array of the allocation-free entry point can serve (MAS_PCG_STATIC_MAX_CELLS)";
        default: return "unknown status";
    }
}

extern "C" void mas_pcg_destroy(mas_pcg_t *h)
{
    if (!h) return;
    DeviceGuard dg(h->device);
    drop_graphs(h);
    DevBuf<double> *bufs[] = {&h->V2, &h->SD, &h->CP, &h->CRoff, &h->CT, &h->E, &h->F, &h->AR, &h->AT, &h->Dinv,
                              &h->vp, &h->wp, &h->ip, &h->Vinv, &h->r, &h->p0, &h->p1, &h->q, &h->partials, &h->hist,
                              &h->bdev, &h->xdev, &h->z, &h->dinvT, &h->ipT};
    for (DevBuf<double> *b : bufs) b->release();
    h->st.release();
    h->args.release();
    h->ctl.release();
    h->tickets.release();
    if (h->h_args) cudaFreeHost(h->h_args);
    if (h->h_st) cudaFreeHost(h->h_st);
    if (h->h_ctl) cudaFreeHost(h->h_ctl);
    if (h->h_hist) cudaFreeHost(h->h_hist);
    cudaGetLastError();
    delete h;
}

namespace {

// Everything of create except the per-cell workspaces: validation, planes, state, pinned staging.
int create_operator(const mas_grid_t *g, const mas_metric_t *m, double dt, const mas_nu_t *nu, const mas_bc_t *bc,
                    mas_pcg **out)
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

    // ---- coefficient planes (R1; the paper prints no discrete operator).  Face by face: the conductance
    // of a face is formed once from (area / distance) and the face's nu, and enters both adjacent cells. ----
    const int nrows = nr * nt;
    std::vector<double> V2(nrows), CP(nrows), SD(nrows, 0.0), CRoff((size_t)(nr + 1) * nt, 0.0),
        CT((size_t)nr * (nt + 1), 0.0), vp(np), ip(np), wp(np), Vinv(nrows);
    for (int t = 0; t < nrows; t++) {
        const int i = t / nt, j = t - i * nt;
        const double solid = m->sin_c[j] * m->dth_c[j];                    // sin(theta) dtheta of the row
        V2[t] = (m->r_c[i] * m->r_c[i]) * m->dr_c[i] * solid;
        Vinv[t] = 1.0 / V2[t];
        CP[t] = nu_at(nu, nt, i, j) * (m->dr_c[i] * m->dth_c[j]) / m->sin_c[j];
    }
    for (int f = 0; f <= nr; f++) {                                        // radial faces f = 0 .. nr
        const bool inner = f == 0, outer = f == nr;
        if ((inner && bc->r_inner == MAS_BC_NEUMANN) || (outer && bc->r_outer == MAS_BC_NEUMANN)) continue;
        const double geom = (m->r_f[f] * m->r_f[f]) / m->dr_f[f];
        for (int j = 0; j < nt; j++) {
            const double nu_lo = nu_at(nu, nt, inner ? 0 : f - 1, j), nu_hi = nu_at(nu, nt, outer ? nr - 1 : f, j);
            const double c = 0.5 * (nu_lo + nu_hi) * geom * (m->sin_c[j] * m->dth_c[j]);
            if (!inner) SD[(size_t)(f - 1) * nt + j] += c;                 // the cell below the face
            if (!outer) SD[(size_t)f * nt + j] += c;                       // the cell above it
            if (!inner && !outer) CRoff[(size_t)f * nt + j] = c;           // a Dirichlet face has no off-diagonal partner
        }
    }
    for (int i = 0; i < nr; i++)
        for (int f = 1; f < nt; f++) {                                     // theta faces; the polar faces have zero area
            const double c = 0.5 * (nu_at(nu, nt, i, f - 1) + nu_at(nu, nt, i, f)) * m->dr_c[i] * (m->sin_f[f] / m->dth_f[f]);
            CT[(size_t)i * (nt + 1) + f] = c;
            SD[(size_t)i * nt + f - 1] += c;
            SD[(size_t)i * nt + f] += c;
        }
    h->uniform_phi = 1;
    for (int k = 0; k < np; k++) {
        vp[k] = m->dph_c[k];
        ip[k] = 1.0 / m->dph_f[k];
        if (m->dph_c[k] != m->dph_c[0] || m->dph_f[k] != m->dph_f[0]) h->uniform_phi = 0;
    }
    for (int k = 0; k < np; k++) wp[k] = ip[k] + ip[(k + np - 1) % np];
    double gmax = 0.0;                                      // max_k wp[k]/vp[k]
    for (int k = 0; k < np; k++) gmax = fmax(gmax, wp[k] / vp[k]);
    for (int t = 0; t < nrows; t++) h->lambda_max = fmax(h->lambda_max, 2.0 * (SD[t] + CP[t] * gmax) / V2[t]);
    h->vp0 = vp[0];
    h->wp0 = wp[0];
    h->ip0 = ip[0];

    int rc;
    if ((rc = upload(h->V2, V2)) || (rc = upload(h->CP, CP)) || (rc = upload(h->SD, SD)) ||
        (rc = upload(h->CRoff, CRoff)) || (rc = upload(h->CT, CT)) || (rc = upload(h->vp, vp)) ||
        (rc = upload(h->wp, wp)) || (rc = upload(h->ip, ip)) || (rc = upload(h->Vinv, Vinv)))
        return fail(h, rc);
    h->pstride = partials_stride(h);
    if (h->E.alloc(nrows) || h->F.alloc(nrows) || h->Dinv.alloc(nrows) || h->AR.alloc((size_t)(nr + 1) * nt) ||
        h->AT.alloc((size_t)nr * (nt + 1)) || h->partials.alloc((size_t)MAX_RHS * PART_REGIONS * h->pstride) ||
        h->st.alloc(MAX_RHS) || h->args.alloc(1) || h->ctl.alloc(1) || h->tickets.alloc(MAX_RHS * 4)) {
        cudaGetLastError();
        return fail(h, MAS_ENOMEM);
    }
    h->hist_cap = 1 << 13;
    if (h->hist.alloc(MAX_RHS * h->hist_cap) != cudaSuccess) return fail(h, MAS_ENOMEM);
    if (cudaMallocHost((void **)&h->h_args, sizeof(SolveArgs)) != cudaSuccess ||
        cudaMallocHost((void **)&h->h_st, MAX_RHS * sizeof(State)) != cudaSuccess ||
        cudaMallocHost((void **)&h->h_ctl, sizeof(Ctl)) != cudaSuccess ||
        cudaMallocHost((void **)&h->h_hist, MAX_RHS * h->hist_cap * sizeof(double)) != cudaSuccess)
        return fail(h, MAS_ENOMEM);
    if (cudaMemset(h->st.p, 0, MAX_RHS * sizeof(State)) != cudaSuccess || cudaMemset(h->ctl.p, 0, sizeof(Ctl)) != cudaSuccess ||
        cudaMemset(h->tickets.p, 0, MAX_RHS * 4 * sizeof(unsigned)) != cudaSuccess)
        return fail(h, MAS_ECUDA);
    fill_op(h);
    if (cudaDeviceGetAttribute(&h->coop_ok, cudaDevAttrCooperativeLaunch, h->device) != cudaSuccess) h->coop_ok = 0;
    if ((rc = scale_planes(h, dt, nullptr)) != MAS_OK) return fail(h, rc);
    if (cudaDeviceSynchronize() != cudaSuccess) return fail(h, MAS_ECUDA);
    *out = h;
    return MAS_OK;
}

}  // namespace

extern "C" int mas_pcg_create(const mas_grid_t *g, const mas_metric_t *m, double dt, const mas_nu_t *nu,
                              const mas_bc_t *bc, mas_pcg_t **out)
{
    mas_pcg *h = nullptr;
    int rc = create_operator(g, m, dt, nu, bc, &h);
    if (rc != MAS_OK) return rc;
    if ((rc = ensure_rhs_capacity(h, 1)) != MAS_OK) return fail(h, rc);
    if (cudaDeviceSynchronize() != cudaSuccess) return fail(h, MAS_ECUDA);
    *out = h;
    return MAS_OK;
}

// =============================================================================================
// launch plans
// =============================================================================================
namespace {

// One "part" = what a set of launches works on: the whole mesh, or one r-slab of a slab group.
struct Plan {                        // storage that kernel argument pointers refer to + the launches
    OpDev op;
    Work work;
    cudaGraphConditionalHandle cond;
    int use_cond;
    int reverse;
    TileParams k1p;
    StencilParams sp_apply, sp_k2;
    KLaunch apply, init, k1, k2, xtail;
    Pc2Dev pc2;
    int zero = 0;
    int max_grid = 0;
};

int base_grid(const mas_pcg *h, const OpDev &op, const void *func, int nt_block)
{
    const long long groups = ((long long)op.nrows * op.nv + nt_block - 1) / nt_block;   // blocks of 16-byte vectors
    int occ = 1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, func, nt_block, 0) != cudaSuccess || occ < 1) {
        cudaGetLastError();
        occ = 1;
    }
    long long gsz = (long long)h->num_sms * occ;
    if (gsz > groups) gsz = groups;
    if (gsz < 1) gsz = 1;
    return (int)gsz;
}

void stencil_common(const mas_pcg *h, StencilParams &sp)
{
    memset(&sp, 0, sizeof(sp));
    sp.t.vp = h->vp0; sp.t.wp = h->wp0; sp.t.ip = h->ip0;
    sp.args = h->args.p;
    sp.fault = &h->ctl.p->fault;
}

// Fill a plan for (operator part, work set, right-hand sides).  use_cond: the kernels set the graph conditional.
int make_plan(const mas_pcg *h, const OpDev &op, const Work &work, int nrhs, int use_cond,
              cudaGraphConditionalHandle cond, Plan &c)
{
    c.op = op; c.work = work; c.cond = cond; c.use_cond = use_cond; c.reverse = h->serpentine;
    const bool uni = h->uniform_phi;
    // A x0 -> q (initial residual)
    stencil_common(h, c.sp_apply);
    c.sp_apply.ps = PlaneSetDev{h->E.p, h->F.p, h->AR.p, h->AT.p, nullptr};
    c.sp_apply.u = nullptr; c.sp_apply.out = work.q; c.sp_apply.ustride = work.vstride;
    c.sp_apply.args = work.args;
    stencil_configure(op.nr, op.nt, op.np, uni, EPI_APPLY, h->stencil_tile, h->num_sms, h->ci_force, nrhs, &c.sp_apply,
                      &c.apply.func, &c.apply.grid, &c.apply.block, &c.apply.smem);
    c.apply.args[0] = &c.op; c.apply.args[1] = &c.sp_apply;
    // init
    c.init.func = uni ? (const void *)k_init<NT_BASE, true> : (const void *)k_init<NT_BASE, false>;
    c.init.block = dim3(NT_BASE);
    c.init.grid = dim3(base_grid(h, op, c.init.func, NT_BASE), nrhs);
    c.init.args[0] = &c.op; c.init.args[1] = &c.work; c.init.args[2] = &c.cond; c.init.args[3] = &c.use_cond;
    const bool pc2 = h->precond == MAS_PC2;
    auto pc2_launch = [&](KLaunch &k, bool init, int *reverse) {       // the line kernel: init or K2P
        k.func = pc2_line_pick(h->pc2_M, uni, init);
        k.block = dim3(PC2_NT);
        k.smem = pc2_smem(h->pc2_M);
        cudaFuncSetAttribute(k.func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)k.smem);
        int occ = 1;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k.func, PC2_NT, k.smem) != cudaSuccess || occ < 1) {
            cudaGetLastError();
            occ = 1;
        }
        long long g = (long long)h->num_sms * occ, need = ((long long)op.nrows + PC2_NWARP - 1) / PC2_NWARP;
        k.grid = dim3((unsigned)(g < need ? g : need), nrhs);
        k.args[0] = &c.op; k.args[1] = &c.work; k.args[2] = &c.pc2; k.args[3] = &c.cond; k.args[4] = &c.use_cond;
        k.args[5] = reverse;
    };
    if (pc2) {
        c.pc2 = Pc2Dev{h->dinvT.p, h->ipT.p, h->ip0, h->pc2_M};
        pc2_launch(c.init, true, &c.zero);
    }
    // K1
    memset(&c.k1p, 0, sizeof(c.k1p));
    const int k1_tile = h->tile >= 0 ? h->tile : k1_auto_tile(op.nr, op.nt, op.np, h->num_sms, h->uniform_phi != 0);
    k1_tma_configure(op.nr, op.nt, op.np, uni, h->qrecompute != 0 && !pc2, k1_tile, h->num_sms, h->ci_force, nrhs, &c.k1p,
                     &c.k1.func, &c.k1.grid, &c.k1.block, &c.k1.smem);
    c.k1p.vp = h->vp0; c.k1p.wp = h->wp0; c.k1p.ip = h->ip0;
    c.k1p.l2 = h->l2;
    c.k1p.zin = pc2 ? 1 : 0;
    c.k1.args[0] = &c.op; c.k1.args[1] = &c.work; c.k1.args[2] = &c.k1p; c.k1.args[3] = &c.cond; c.k1.args[4] = &c.use_cond;
    // K2 (q stored), K2R (q recomputed), or K2P (PC2: r-update + line solves)
    if (pc2) {
        pc2_launch(c.k2, false, &c.reverse);
    } else if (h->qrecompute) {
        stencil_common(h, c.sp_k2);
        c.sp_k2.ps = PlaneSetDev{h->E.p, h->F.p, h->AR.p, h->AT.p, h->Dinv.p};
        c.sp_k2.w = work; c.sp_k2.cond = cond; c.sp_k2.use_cond = use_cond;
        c.sp_k2.args = work.args;
        stencil_configure(op.nr, op.nt, op.np, uni, EPI_K2R, h->k2r_tile, h->num_sms, h->ci_force, nrhs, &c.sp_k2,
                          &c.k2.func, &c.k2.grid, &c.k2.block, &c.k2.smem);
        c.sp_k2.t.reverse = h->serpentine;
        c.sp_k2.t.l2 = h->l2;
        c.k2.args[0] = &c.op; c.k2.args[1] = &c.sp_k2;
    } else {
        c.k2.func = uni ? (const void *)k2_vec<NT_BASE, true> : (const void *)k2_vec<NT_BASE, false>;
        c.k2.block = dim3(NT_BASE);
        c.k2.grid = dim3(base_grid(h, op, c.k2.func, NT_BASE), nrhs);
        c.k2.smem = 0;
        c.k2.args[0] = &c.op; c.k2.args[1] = &c.work; c.k2.args[2] = &c.cond; c.k2.args[3] = &c.use_cond;
        c.k2.args[4] = &c.reverse;
    }
    // x tail
    c.xtail.func = (const void *)k_xtail<NT_BASE>;
    c.xtail.block = dim3(NT_BASE);
    c.xtail.grid = dim3(base_grid(h, op, c.xtail.func, NT_BASE), nrhs);
    c.xtail.args[0] = &c.op; c.xtail.args[1] = &c.work;
    c.max_grid = (int)c.init.grid.x;
    if ((int)c.k1.grid.x > c.max_grid) c.max_grid = (int)c.k1.grid.x;
    if ((int)c.k2.grid.x > c.max_grid) c.max_grid = (int)c.k2.grid.x;
    return c.max_grid <= work.pstride ? MAS_OK : MAS_EINVAL;     // the invariant grid_sum relies on
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

// A solve as three kernel sequences: before the loop, the loop body (one PCG iteration), after the loop.
struct Seq {
    std::vector<KLaunch> pre, body, post;
};

// graph = pre... -> WHILE(cond){ body x unroll } -> post...   (call stack 2)
// `unroll` iterations per WHILE trip: the conditional node is evaluated once per trip, and the kernels return
// at once when the loop has ended (device flags), so extra copies after convergence cost empty launches.
int build_graph(const Seq &seq, cudaGraph_t g, cudaGraphConditionalHandle cond, int unroll, cudaGraphExec_t *exec)
{
    cudaGraphNode_t prev = nullptr, node;
    for (const KLaunch &k : seq.pre) {
        if (add_node(&node, g, prev ? &prev : nullptr, k) != cudaSuccess) { cudaGetLastError(); return MAS_ECUDA; }
        prev = node;
    }
    cudaGraphNodeParams wp = {cudaGraphNodeTypeConditional};
    wp.conditional.handle = cond;
    wp.conditional.type = cudaGraphCondTypeWhile;
    wp.conditional.size = 1;
    cudaGraphNode_t n_while;
    if (cudaGraphAddNode(&n_while, g, prev ? &prev : nullptr, prev ? 1 : 0, &wp) != cudaSuccess) { cudaGetLastError(); return MAS_ECUDA; }
    cudaGraph_t body = wp.conditional.phGraph_out[0];
    cudaGraphNode_t bprev = nullptr;
    for (int u = 0; u < unroll; u++)
        for (const KLaunch &k : seq.body) {
            if (add_node(&node, body, bprev ? &bprev : nullptr, k) != cudaSuccess) { cudaGetLastError(); return MAS_ECUDA; }
            bprev = node;
        }
    prev = n_while;
    for (const KLaunch &k : seq.post) {
        if (add_node(&node, g, &prev, k) != cudaSuccess) { cudaGetLastError(); return MAS_ECUDA; }
        prev = node;
    }
    if (cudaGraphInstantiate(exec, g, 0) != cudaSuccess) {
        cudaGetLastError();
        *exec = nullptr;
        return MAS_ECUDA;
    }
    return MAS_OK;
}

// host-driven loop over the same sequences: chunks of HOST_CHUNK iterations, then a poll of the loop flag
int run_host_loop(const Seq &seq, const Ctl *d_ctl, Ctl *h_ctl, int maxit, cudaStream_t s, long long *launched_loop)
{
    for (const KLaunch &k : seq.pre) CK(launch(k, s));
    for (int done = 0; done < maxit;) {
        CK(cudaMemcpyAsync(h_ctl, d_ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, s));
        CK(cudaStreamSynchronize(s));
        if (!h_ctl->loop) break;
        const int chunk = maxit - done < HOST_CHUNK ? maxit - done : HOST_CHUNK;
        for (int it = 0; it < chunk; it++)
            for (const KLaunch &k : seq.body) CK(launch(k, s));
        *launched_loop += (long long)seq.body.size() * chunk;
        done += chunk;
    }
    for (const KLaunch &k : seq.post) CK(launch(k, s));
    return MAS_OK;
}

int ensure_hist(mas_pcg *h, int maxit)
{
    const size_t need = (size_t)maxit + 1;
    if (need <= h->hist_cap) return MAS_OK;
    size_t cap = h->hist_cap ? h->hist_cap : 1;
    while (cap < need) cap *= 2;
    // the new pair first, the old pair released only once both exist: a failure leaves the handle as it was
    DevBuf<double> nd;
    double *nh = nullptr;
    if (nd.alloc(MAX_RHS * cap) != cudaSuccess) { cudaGetLastError(); return MAS_ENOMEM; }
    if (cudaMallocHost((void **)&nh, MAX_RHS * cap * sizeof(double)) != cudaSuccess) {
        cudaGetLastError();
        nd.release();
        return MAS_ENOMEM;
    }
    h->hist.release();
    h->hist = nd;
    if (h->h_hist) cudaFreeHost(h->h_hist);
    h->h_hist = nh;
    h->hist_cap = cap;
    fill_op(h);
    drop_graphs(h);             // kernel nodes hold the old hist pointer
    return MAS_OK;
}

bool aligned16(const void *p) { return ((uintptr_t)p & 15u) == 0; }

// Plan the one-kernel solve; returns false when it does not apply (too large, no cooperative launch, off).
bool plan_persistent(const mas_pcg *h, PersistParams *pp, int *grid, size_t *smem, const void **func)
{
    if (!h->persistent || !h->coop_ok || h->precond != MAS_PC1) return false;
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
    pp->partials = h->partials.p; pp->pstride = h->pstride;
    pp->hist = h->hist.p; pp->st = h->st.p; pp->args = h->args.p;
    pp->nvec = (int)nvec; pp->M = (int)M;
    *grid = (int)g;
    return true;
}

void set_traffic_stats(mas_pcg *h)
{
    // qrecompute: K1 r,p,x -> p,x (5N); K2R p,r -> r (3N).  otherwise: K1 r,p,x -> p,q,x (6N); K2 r,q -> r (3N)
    // PC2: K1 z,p,x -> p,q,x (6N); K2P r,q,1/piv -> r,z (5N)
    const bool pc2 = h->precond == MAS_PC2;
    h->stats[4] = (h->qrecompute && !pc2) ? 5 : 6;
    h->stats[5] = pc2 ? 5 : 3;
    h->stats[3] = 8 * (h->stats[4] + h->stats[5]);
}

int worst_status(int a, int b)
{
    if (a < 0 || b < 0) return a < b ? a : b;
    return a > b ? a : b;
}

void seq_for_plan(const Plan &c, Seq &seq)
{
    seq.pre = {c.apply, c.init};
    seq.body = {c.k1, c.k2};
    seq.post = {c.xtail};
}

// The common solve: nrhs right-hand sides sharing the operator, each an independent PCG (own alpha, beta, count,
// status, history), run by ONE set of launches whose grid.y is the right-hand side.
int solve_core(mas_pcg *h, int nrhs, const double *const *b_dev, double *const *x_dev, double rtol, int maxit,
               cudaStream_t s, int *iters_out, int *status_out, double *reshist_host)
{
    int rc = ensure_hist(h, maxit);
    if (rc != MAS_OK) return rc;
    if ((rc = ensure_rhs_capacity(h, nrhs)) != MAS_OK) return rc;
    memset(h->h_args, 0, sizeof(SolveArgs));
    for (int j = 0; j < nrhs; j++) { h->h_args->b[j] = b_dev[j]; h->h_args->x[j] = x_dev[j]; }
    h->h_args->rtol = rtol; h->h_args->maxit = maxit; h->h_args->nrhs = nrhs;
    CK(cudaMemcpyAsync(h->args.p, h->h_args, sizeof(SolveArgs), cudaMemcpyHostToDevice, s));

    int mode = h->loop_mode;
    PersistParams ppar;
    int pgrid = 0;
    size_t psmem = 0;
    const void *pfunc = nullptr;
    long long launched_outside = 0, launched_loop = 0;
    if (nrhs == 1 && !h->coop_refused && plan_persistent(h, &ppar, &pgrid, &psmem, &pfunc)) {
        OpDev op = h->op;                      // init + loop + finish in one cooperative kernel
        void *kargs[2] = {&op, &ppar};
        if (cudaLaunchCooperativeKernel(pfunc, dim3(pgrid), dim3(PNT), kargs, psmem, s) == cudaSuccess) {
            mode = 2;
            launched_loop = 1;
        } else {
            cudaGetLastError();                // refused (e.g. co-residency limits): use the streaming loop from now on
            h->coop_refused = 1;
        }
    }
    if (mode != 2) {
        std::unique_ptr<Plan> plan(new (std::nothrow) Plan());
        if (!plan) return MAS_ENOMEM;
        Seq seq;
        if (mode == 1 && !h->exec[nrhs - 1]) {
            cudaGraph_t g = nullptr;
            cudaGraphConditionalHandle cond;
            bool ok = cudaGraphCreate(&g, 0) == cudaSuccess;
            if (ok) h->graph[nrhs - 1] = g;
            ok = ok && cudaGraphConditionalHandleCreate(&cond, g, 1, cudaGraphCondAssignDefault) == cudaSuccess;
            if (ok) {
                if ((rc = make_plan(h, h->op, h->work, nrhs, 1, cond, *plan)) != MAS_OK) {
                    drop_graphs(h);            // the graph created above has no executable yet: do not leave it behind
                    return rc;
                }
                seq_for_plan(*plan, seq);
                ok = build_graph(seq, g, cond, h->unroll, &h->exec[nrhs - 1]) == MAS_OK;
            }
            if (!ok) {                         // driver without conditional nodes: fall back, and say so in stats
                cudaGetLastError();
                drop_graphs(h);
                mode = 0;
            }
        }
        if (mode == 1) {
            CK(cudaGraphLaunch(h->exec[nrhs - 1], s));
        } else {
            cudaGraphConditionalHandle none;
            memset(&none, 0, sizeof(none));
            if ((rc = make_plan(h, h->op, h->work, nrhs, 0, none, *plan)) != MAS_OK) return rc;
            seq.pre.clear(); seq.body.clear(); seq.post.clear();
            seq_for_plan(*plan, seq);
            if ((rc = run_host_loop(seq, h->ctl.p, h->h_ctl, maxit, s, &launched_loop)) != MAS_OK) return rc;
        }
        launched_outside = 3;
    }
    CK(cudaMemcpyAsync(h->h_st, h->st.p, MAX_RHS * sizeof(State), cudaMemcpyDeviceToHost, s));
    CK(cudaMemcpyAsync(h->h_ctl, h->ctl.p, sizeof(Ctl), cudaMemcpyDeviceToHost, s));
    for (int j = 0; j < nrhs; j++)
        CK(cudaMemcpyAsync(h->h_hist + (size_t)j * h->hist_cap, h->hist.p + (size_t)j * h->hist_cap,
                           ((size_t)maxit + 1) * sizeof(double), cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));          // the one host sync of a graph-mode solve
    if (h->h_ctl->fault) {                 // a kernel gave up on an mbarrier wait: the result is not trustworthy
        cudaMemsetAsync(&h->ctl.p->fault, 0, sizeof(int), s);
        return MAS_ECUDA;
    }
    int worst = MAS_OK;
    long long graph_launches = 0;
    for (int j = 0; j < nrhs; j++) {
        const State &st = h->h_st[j];
        if (st.bb == 0.0) CK(cudaMemsetAsync(x_dev[j], 0, h->n * sizeof(double), s));   // zero right-hand side: x = 0
        if (iters_out) iters_out[j] = st.k;
        if (status_out) status_out[j] = st.status;
        if (reshist_host)
            memcpy(reshist_host + (size_t)j * ((size_t)maxit + 1), h->h_hist + (size_t)j * h->hist_cap,
                   ((size_t)st.k + 1) * sizeof(double));
        worst = worst_status(worst, st.status);
        if (st.launches > graph_launches) graph_launches = st.launches;
    }
    CK(cudaStreamSynchronize(s));
    h->stats[0] = mode == 1 ? graph_launches : launched_loop;
    h->stats[1] = launched_outside;
    h->stats[2] = mode;
    h->stats[6] = mode == 2 ? pgrid : 0;
    h->stats[7] = h->coop_refused;
    set_traffic_stats(h);
    return worst;
}

}  // namespace

extern "C" int mas_pcg_set_dt(mas_pcg_t *h, double dt, void *stream)
{
    if (!h || !(dt >= 0.0) || !isfinite(dt)) return MAS_EINVAL;
    DeviceGuard dg(h->device);
    if (!dg.ok) return MAS_ECUDA;
    return scale_planes(h, dt, (cudaStream_t)stream);
}

extern "C" int mas_pcg_apply(mas_pcg_t *h, const double *x_dev, double *y_dev, void *stream)
{
    if (!h || !x_dev || !y_dev || x_dev == y_dev || !aligned16(x_dev) || !aligned16(y_dev)) return MAS_EINVAL;
    DeviceGuard dg(h->device);
    if (!dg.ok) return MAS_ECUDA;
    StencilParams sp;
    stencil_common(h, sp);
    sp.ps = PlaneSetDev{h->E.p, h->F.p, h->AR.p, h->AT.p, nullptr};
    sp.u = x_dev; sp.out = y_dev;
    KLaunch k;
    OpDev op = h->op;
    stencil_configure(h->nr, h->nt, h->np, h->uniform_phi, EPI_APPLY, h->stencil_tile, h->num_sms, h->ci_force, 1, &sp,
                      &k.func, &k.grid, &k.block, &k.smem);
    k.args[0] = &op; k.args[1] = &sp;
    CK(launch(k, (cudaStream_t)stream));
    return MAS_OK;
}

namespace {

// Switch the operator's preconditioner.  own_z: allocate the handle's own z vectors (a slab group keeps one per slab).
int set_precond(mas_pcg *h, int kind, int bi, int bj, int bk, bool own_z)
{
    if (kind != MAS_PC1 && kind != MAS_PC2) return MAS_EINVAL;
    if (kind == MAS_PC1) {
        if (h->precond != MAS_PC1) drop_graphs(h);
        h->precond = MAS_PC1;
        fill_op(h);
        return MAS_OK;
    }
    // the GPU path builds the line domains only: 1 x 1 x (all of phi); other boxes are the oracle's (R8)
    if (bi != 1 || bj != 1 || (bk != 0 && bk < h->np)) return MAS_EINVAL;
    const int M = pc2_chunk(h->np);
    if (M == 0) return MAS_EINVAL;                           // np < 4 or np > 1024
    const size_t lines = (size_t)h->nr * h->nt;
    if (!h->dinvT.p || h->pc2_M != M) {
        if (h->dinvT.alloc(lines * 32 * M) != cudaSuccess) { cudaGetLastError(); return MAS_ENOMEM; }
        std::vector<double> ipT((size_t)32 * M, 0.0), ip(h->np);
        CK(cudaMemcpy(ip.data(), h->ip.p, (size_t)h->np * sizeof(double), cudaMemcpyDeviceToHost));
        for (int k = 0; k < h->np; k++) ipT[(size_t)pc2_slot(k, M)] = ip[(size_t)k];
        const int rc = upload(h->ipT, ipT);
        if (rc != MAS_OK) return rc;
    }
    if (own_z && (!h->z.p || h->z.n < h->n * (size_t)h->nrhs_cap)) {
        if (h->z.alloc(h->n * (size_t)(h->nrhs_cap > 0 ? h->nrhs_cap : 1)) != cudaSuccess) { cudaGetLastError(); return MAS_ENOMEM; }
    }
    h->pc2_M = M;
    h->precond = MAS_PC2;
    fill_op(h);
    drop_graphs(h);
    k_pc2_factor<<<(unsigned)((lines + 127) / 128), 128>>>(h->op, h->dinvT.p, M);
    CK(cudaGetLastError());
    CK(cudaDeviceSynchronize());
    return MAS_OK;
}

}  // namespace

extern "C" int mas_pcg_set_preconditioner(mas_pcg_t *h, int kind, int bi, int bj, int bk)
{
    if (!h) return MAS_EINVAL;
    DeviceGuard dg(h->device);
    if (!dg.ok) return MAS_ECUDA;
    return set_precond(h, kind, bi, bj, bk, true);
}

extern "C" int mas_pcg_set_option(mas_pcg_t *h, const char *name, int value)
{
    if (!h || !name) return MAS_EINVAL;
    DeviceGuard dg(h->device);
    if (!dg.ok) return MAS_ECUDA;
    if (!strcmp(name, "loop_mode")) {
        if (value != 0 && value != 1) return MAS_EINVAL;
        h->loop_mode = value;
    } else if (!strcmp(name, "tile")) {
        if (value < -1 || value >= k1_tma_num_tiles()) return MAS_EINVAL;
        h->tile = value;
    } else if (!strcmp(name, "stencil_tile")) {
        if (value < 0 || value >= stencil_num_tiles()) return MAS_EINVAL;
        h->stencil_tile = value;
    } else if (!strcmp(name, "k2r_tile")) {
        if (value < 0 || value >= stencil_num_tiles()) return MAS_EINVAL;
        h->k2r_tile = value;
    } else if (!strcmp(name, "serpentine")) {
        if (value != 0 && value != 1) return MAS_EINVAL;
        h->serpentine = value;
    } else if (!strcmp(name, "unroll")) {
        if (value < 1 || value > 16) return MAS_EINVAL;
        h->unroll = value;
    } else if (!strcmp(name, "persistent")) {
        if (value != 0 && value != 1) return MAS_EINVAL;
        h->persistent = value;
        h->coop_refused = 0;
    } else if (!strcmp(name, "qrecompute")) {
        if (value != 0 && value != 1) return MAS_EINVAL;
        h->qrecompute = value;
    } else if (!strcmp(name, "ci")) {
        if (value != 0 && (value < CI_FORCE_MIN || value > TILE_CI_MAX)) return MAS_EINVAL;
        h->ci_force = value;
    } else if (!strcmp(name, "l2_first_x")) {
        if (value != 0 && value != 1) return MAS_EINVAL;
        h->l2.first_x = value;
    } else {
        return MAS_EINVAL;
    }
    drop_graphs(h);
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
    DeviceGuard dg(h->device);
    if (!dg.ok) return MAS_ECUDA;
    return solve_core(h, 1, &b_dev, &x_dev, rtol, maxit, (cudaStream_t)stream, iters_out, nullptr, reshist_host);
}

extern "C" int mas_pcg_solve_multi(mas_pcg_t *h, int nrhs, const double *const *b_dev, double *const *x_dev,
                                   double rtol, int maxit, void *stream, int *iters_out, int *status_out,
                                   double *reshist_host)
{
    if (!h || nrhs < 1 || nrhs > MAX_RHS || !b_dev || !x_dev || !(rtol >= 0.0) || maxit < 0) return MAS_EINVAL;
    for (int j = 0; j < nrhs; j++) {
        if (!b_dev[j] || !x_dev[j] || !aligned16(b_dev[j]) || !aligned16(x_dev[j])) return MAS_EINVAL;
        for (int l = 0; l < nrhs; l++)
            if (b_dev[j] == x_dev[l] || (l != j && x_dev[j] == x_dev[l])) return MAS_EINVAL;
    }
    DeviceGuard dg(h->device);
    if (!dg.ok) return MAS_ECUDA;
    return solve_core(h, nrhs, b_dev, x_dev, rtol, maxit, (cudaStream_t)stream, iters_out, status_out, reshist_host);
}

extern "C" int mas_pcg_solve_host(mas_pcg_t *h, const double *b_host, double *x_host, double rtol, int maxit,
                                  void *stream, int *iters_out, double *reshist_host)
{
    if (!h || !b_host || !x_host) return MAS_EINVAL;
    DeviceGuard dg(h->device);
    if (!dg.ok) return MAS_ECUDA;
    cudaStream_t s = (cudaStream_t)stream;
    if (!h->bdev.p && h->bdev.alloc(h->n) != cudaSuccess) { cudaGetLastError(); return MAS_ENOMEM; }
    if (!h->xdev.p && h->xdev.alloc(h->n) != cudaSuccess) { cudaGetLastError(); return MAS_ENOMEM; }
    const size_t bytes = h->n * sizeof(double);
    CK(cudaMemcpyAsync(h->bdev.p, b_host, bytes, cudaMemcpyHostToDevice, s));
    CK(cudaMemcpyAsync(h->xdev.p, x_host, bytes, cudaMemcpyHostToDevice, s));
    const int rc = mas_pcg_solve(h, h->bdev.p, h->xdev.p, rtol, maxit, stream, iters_out, reshist_host);
    if (rc < 0 && rc != MAS_EBREAKDOWN) return rc;
    CK(cudaMemcpyAsync(x_host, h->xdev.p, bytes, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    return rc;
}

#include "host_sts.inc"
#include "host_slabs.inc"
#include "noalloc_residual.inc"
#ifdef MAS_PCG_DEBUG_PROBES
#include "host_debug.inc"
#endif

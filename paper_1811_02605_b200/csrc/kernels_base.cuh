// kernels_base.cuh -- set_dt plane scaling, init (S1), the fused vector kernel K2 (S4), the x tail, the scalar
// steps S3 / S5 run by the last-arriving block of the reducing kernels, and the slab combine step.
// Every kernel takes the right-hand side index from blockIdx.y (batched solves: the three
// components of v share one coefficient set); a single solve is gridDim.y = 1.
#pragma once
#include "common.cuh"

namespace mas {

// ---------------------------------------------------------------------------------------------
// set_dt: base planes -> dt-scaled planes.  Tiny: O(nr*nt).
// ---------------------------------------------------------------------------------------------
struct PlaneSet {
    const double *V2, *SD, *CP, *CRoff, *CT;   // base (dt-independent)
    double *E, *F, *AR, *AT, *Dinv;            // scaled
    int nr, nt;
    double vp0, wp0;                           // phi factors of cell 0 (used when phi is uniform)
};

__global__ void k_scale_planes(PlaneSet ps, double dt)
{
    const int nrows = ps.nr * ps.nt;
    const int nAR = (ps.nr + 1) * ps.nt, nAT = ps.nr * (ps.nt + 1);
    for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < nAR + nAT; t += gridDim.x * blockDim.x) {
        if (t < nrows) {
            const double e = ps.V2[t] + dt * ps.SD[t];
            const double f = dt * ps.CP[t];
            ps.E[t] = e;
            ps.F[t] = f;
            ps.Dinv[t] = 1.0 / (ps.vp0 * e + f * ps.wp0);
        }
        if (t < nAR) ps.AR[t] = dt * ps.CRoff[t];
        if (t < nAT) ps.AT[t] = dt * ps.CT[t];
    }
}

__device__ __forceinline__ double2 ld2(const double *p, size_t cell)
{
    return *reinterpret_cast<const double2 *>(p + cell);
}
__device__ __forceinline__ void st2(double *p, size_t cell, double2 v)
{
    *reinterpret_cast<double2 *>(p + cell) = v;
}

// ---------------------------------------------------------------------------------------------
// loop control: the graph's WHILE condition (and the flag the host-chunk loop polls) = "some right-hand
// side is still active".  Every right-hand side reports once per voting kernel (init, K2): through its
// last-arriving block when it did work, through block 0 when it was already inactive.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void set_cond(cudaGraphConditionalHandle cond, int use_cond, int v)
{
    if (use_cond) cudaGraphSetConditional(cond, v ? 1u : 0u);
}

__device__ __forceinline__ void loop_vote(const Work &w, int active, int nvoters, cudaGraphConditionalHandle cond,
                                          int use_cond)
{
    Ctl *c = w.ctl;
    if (nvoters == 1) {
        c->loop = active;
        set_cond(cond, use_cond, active);
        return;
    }
    if (active) atomicAdd(&c->any, 1);
    __threadfence();
    if (atomicAdd(&c->votes, 1) == nvoters - 1) {
        __threadfence();
        const int any = atomicExch(&c->any, 0);
        c->votes = 0;                          // re-arm for the next voting kernel (stream order separates them)
        c->loop = any > 0;
        set_cond(cond, use_cond, any > 0);
    }
}

// ---------------------------------------------------------------------------------------------
// scalar steps (SURVEY 8(a) S1 tail, S3, S5), run by ONE thread once a reduction is complete
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void init_finish(const Work &w, int rhs, int nvoters, double bb, double rr, double rho,
                                            cudaGraphConditionalHandle cond, int use_cond)
{
    State *st = w.st + rhs;
    double *hist = w.hist + (size_t)rhs * w.hstride;
    st->bb = bb; st->rr = rr; st->rho = rho;
    st->beta = 0.0; st->alpha = 0.0; st->sigma = 0.0;
    st->k = 0; st->launches = 0;
    int active = 0, status = ST_OK;
    if (!isfinite(bb) || !isfinite(rr) || !isfinite(rho)) {
        hist[0] = sqrt(rr / bb);                // a non-finite scalar (NaN / Inf in b or x0): breakdown, x untouched
        status = ST_BREAKDOWN;
    } else if (bb == 0.0) {
        hist[0] = 0.0;                          // zero RHS: x = 0 (host zeroes x), 0 iterations
    } else {
        const double h = sqrt(rr / bb);
        hist[0] = h;
        active = (0 < w.args->maxit) && (h > w.args->rtol) && (rho != 0.0);
        if (!active) status = (h <= w.args->rtol || rho == 0.0) ? ST_OK : ST_MAXIT;
    }
    st->active = active;
    st->status = status;
    loop_vote(w, active, nvoters, cond, use_cond);
}

// S3: sigma -> alpha, breakdown test.  (No vote: K2 of the same iteration reports for this right-hand side.)
__device__ __forceinline__ void k1_finish(const Work &w, int rhs, double sigma)
{
    State *st = w.st + rhs;
    st->sigma = sigma;
    st->launches += 1;
    if (!(sigma > 0.0) || isinf(sigma)) {
        st->status = ST_BREAKDOWN;
        st->active = 0;
        st->alpha = 0.0;                 // nothing pending for the x tail
    } else {
        st->alpha = st->rho / sigma;
    }
}

// S5: k++, hist[k], beta, convergence test, loop condition
__device__ __forceinline__ void k2_finish(const Work &w, int rhs, int nvoters, double rho1, double rr,
                                          cudaGraphConditionalHandle cond, int use_cond)
{
    State *st = w.st + rhs;
    const int k = st->k + 1;
    const double h = sqrt(rr / st->bb);
    w.hist[(size_t)rhs * w.hstride + k] = h;
    st->beta = rho1 / st->rho;
    st->rho = rho1;
    st->rr = rr;
    st->k = k;
    st->launches += 1;
    int active = (k < w.args->maxit) && (h > w.args->rtol) && (rho1 != 0.0);
    if (!isfinite(rho1) || !isfinite(rr)) {            // iterate k is kept (the pending x-update is applied by the tail)
        active = 0;
        st->status = ST_BREAKDOWN;
    } else if (!active) st->status = (h <= w.args->rtol || rho1 == 0.0) ? ST_OK : ST_MAXIT;
    st->active = active;
    loop_vote(w, active, nvoters, cond, use_cond);
}

// What the last block of a reducing kernel does with its totals: finish the scalar step, or (slab mode)
// leave them for k_slab_combine, which adds the slabs' sums in slab order.
enum { ROLE_INIT = 0, ROLE_K1 = 1, ROLE_K2 = 2 };
template <int ROLE, int NQ>
__device__ __forceinline__ void reduction_done(const Work &w, int rhs, const double (&tot)[NQ],
                                               cudaGraphConditionalHandle cond, int use_cond)
{
    if (w.slab_sums) {
#pragma unroll
        for (int q = 0; q < NQ; q++) w.slab_sums[(ROLE * 3 + q) * MAX_SLABS + w.slab] = tot[q];
        return;
    }
    if (ROLE == ROLE_INIT) init_finish(w, rhs, gridDim.y, tot[0], tot[NQ > 1 ? 1 : 0], tot[NQ > 2 ? 2 : 0], cond, use_cond);
    else if (ROLE == ROLE_K1) k1_finish(w, rhs, tot[0]);
    else k2_finish(w, rhs, gridDim.y, tot[0], tot[NQ > 1 ? 1 : 0], cond, use_cond);
}

// Slab combine ("the two scalar reductions combine per-slab partials in fixed slab order").
// One thread; on a multi-GPU node every rank would run this on its own copy of the state after the slabs' sums
// have been exchanged, and all ranks would obtain identical scalars.
__global__ void k_slab_combine(Work w, int role, int nslab, cudaGraphConditionalHandle cond, int use_cond)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    if (role != ROLE_INIT && !w.st->active) {
        if (role == ROLE_K2) loop_vote(w, 0, 1, cond, use_cond);
        return;
    }
    double t[3] = {0.0, 0.0, 0.0};
    for (int q = 0; q < 3; q++)
        for (int s = 0; s < nslab; s++) t[q] += w.slab_sums[(role * 3 + q) * MAX_SLABS + s];
    if (role == ROLE_INIT) init_finish(w, 0, 1, t[0], t[1], t[2], cond, use_cond);
    else if (role == ROLE_K1) k1_finish(w, 0, t[0]);
    else k2_finish(w, 0, 1, t[0], t[1], cond, use_cond);
}

// ---------------------------------------------------------------------------------------------
// init (S1): r = V.b - q (q = A x0), p_in = 0, bb = |V.b|^2, rr = |r|^2, rho = r.(r/d); then the
// last block sets hist[0], k = 0, beta = 0 and the loop condition.
// ---------------------------------------------------------------------------------------------
template <int NT, bool UNIFORM>
__global__ void __launch_bounds__(NT) k_init(OpDev op, Work w, cudaGraphConditionalHandle cond, int use_cond)
{
    __shared__ double sh[32];
    const int rhs = blockIdx.y;
    const double *b = w.args->b[rhs];
    double *rv = w.r + rhs * w.vstride, *p0 = w.p0 + rhs * w.vstride;
    const double *qv0 = w.q + rhs * w.vstride;
    const int crow0 = op.i_lo * op.nt;
    double acc[3] = {0.0, 0.0, 0.0};   // bb, rr, rho
    const int total = op.nrows * op.nv;                     // flat sweep over 16-byte vectors (see k2_vec)
    for (int v = blockIdx.x * NT + threadIdx.x; v < total; v += gridDim.x * NT) {
        const int row = v / op.nv, k = 2 * (v - row * op.nv);
        const int crow = row + crow0;
        const double E = __ldg(op.E + crow), F = __ldg(op.F + crow), V2 = __ldg(op.V2 + crow);
        const double dinv = __ldg(op.Dinv + crow);
        const double vp0 = __ldg(op.vp + k), vp1 = __ldg(op.vp + k + 1);
        const double d0 = fma(vp0, E, F * __ldg(op.wp + k)), d1 = fma(vp1, E, F * __ldg(op.wp + k + 1));
        const size_t cell = 2 * (size_t)v;
        const double2 bv = ld2(b, cell), qv = ld2(qv0, cell);
        const double bs0 = V2 * vp0 * bv.x, bs1 = V2 * vp1 * bv.y;
        double2 r;
        r.x = bs0 - qv.x;
        r.y = bs1 - qv.y;
        st2(rv, cell, r);
        st2(p0, cell, make_double2(0.0, 0.0));
        acc[0] += bs0 * bs0 + bs1 * bs1;
        acc[1] += r.x * r.x + r.y * r.y;
        acc[2] += UNIFORM ? r.x * (r.x * dinv) + r.y * (r.y * dinv)      // same z as K1/K2 use
                          : r.x * (r.x * rcp_nr(d0)) + r.y * (r.y * rcp_nr(d1));
    }
    if (grid_sum<NT, 3>(acc, part_base(w, rhs), w.pstride, &w.tickets[rhs * 4 + 0], sh) && threadIdx.x == 0)
        reduction_done<ROLE_INIT, 3>(w, rhs, acc, cond, use_cond);
}

// ---------------------------------------------------------------------------------------------
// K2 (S4+S5): r -= alpha q; z = r/d (not stored); rho' = r.z; rr = r.r; last block: k++, hist[k], beta,
// convergence test, loop condition.  3N doubles of traffic: the x-update lives in K1 (deferred one iteration).
// `reverse`: sweep the rows from the last to the first (serpentine: K1 marches forward in r, so the
// planes it touched last -- q, r -- are still in L2 when K2 starts there, and K2's last rows are in L2
// when the next K1 starts at i = 0).  The row -> block -> partial mapping stays fixed, so determinism holds.
// ---------------------------------------------------------------------------------------------
template <int NT, bool UNIFORM>
__global__ void __launch_bounds__(NT, 5) k2_vec(   // 5 blocks of 256 threads per SM (<= 48 registers): K2 hides latency by memory parallelism only
OpDev op, Work w, cudaGraphConditionalHandle cond, int use_cond,
                                             int reverse)
{
    __shared__ double sh[32];
    const int rhs = blockIdx.y;
    State *st = w.st + rhs;
    if (!st->active) {                                // this right-hand side is done: report, nothing else
        if (blockIdx.x == 0 && threadIdx.x == 0 && !w.slab_sums) loop_vote(w, 0, gridDim.y, cond, use_cond);
        return;
    }
    const double alpha = st->alpha;
    double *rvec = w.r + rhs * w.vstride;
    const double *qvec = w.q + rhs * w.vstride;
    const int crow0 = op.i_lo * op.nt;
    double acc[2] = {0.0, 0.0};   // rho', rr
    // Flat sweep over the 16-byte vectors of the whole array (vector v = cells 2v, 2v+1; its row is v / nv), so that
    // every thread works whatever the row length is (a row-wise mapping idles a quarter of the block at np = 384).
    // Two vectors per trip (A and B, one grid stride apart): their loads are issued together, which doubles the
    // bytes in flight per thread -- K2 has no other latency hiding than memory parallelism.
    auto body = [&](int v, double2 rv, double2 qv) {
        const int row = v / op.nv;
        rv.x = fma(-alpha, qv.x, rv.x);
        rv.y = fma(-alpha, qv.y, rv.y);
        st2(rvec, 2 * (size_t)v, rv);
        double z0, z1;
        if (UNIFORM) {
            const double dinv = __ldg(op.Dinv + crow0 + row);
            z0 = rv.x * dinv; z1 = rv.y * dinv;
        } else {
            const int k = 2 * (v - row * op.nv);
            const double E = __ldg(op.E + crow0 + row), F = __ldg(op.F + crow0 + row);
            z0 = rv.x * rcp_nr(fma(__ldg(op.vp + k), E, F * __ldg(op.wp + k)));
            z1 = rv.y * rcp_nr(fma(__ldg(op.vp + k + 1), E, F * __ldg(op.wp + k + 1)));
        }
        acc[0] += rv.x * z0 + rv.y * z1;
        acc[1] += rv.x * rv.x + rv.y * rv.y;
    };
    {
        const int total = op.nrows * op.nv, stride = gridDim.x * NT;     // N < 2^31 cells => total < 2^30
        const double2 zero = make_double2(0.0, 0.0);
        for (int v0 = blockIdx.x * NT + threadIdx.x; v0 < total; v0 += 2 * stride) {
            int vA = v0, vB = v0 + stride;
            const bool okB = vB < total;
            if (reverse) { vA = total - 1 - vA; vB = total - 1 - vB; }
            const double2 rA = ld2(rvec, 2 * (size_t)vA), qA = ld2(qvec, 2 * (size_t)vA);
            const double2 rB = okB ? ld2(rvec, 2 * (size_t)vB) : zero, qB = okB ? ld2(qvec, 2 * (size_t)vB) : zero;
            body(vA, rA, qA);
            if (okB) body(vB, rB, qB);
        }
    }
    if (grid_sum<NT, 2>(acc, part_base(w, rhs), w.pstride, &w.tickets[rhs * 4 + 2], sh) && threadIdx.x == 0)
        reduction_done<ROLE_K2, 2>(w, rhs, acc, cond, use_cond);
}

// x tail (after the loop): the one x-update still pending, x += alpha_{k-1} p_{k-1}.  alpha is 0 when
// nothing is pending (no iteration ran, or K1 broke down after applying the previous update).
template <int NT>
__global__ void __launch_bounds__(NT) k_xtail(OpDev op, Work w)
{
    const int rhs = blockIdx.y;
    const State *st = w.st + rhs;
    const double alpha = st->alpha;
    if (alpha == 0.0) return;
    const double *p = ((st->k & 1) ? w.p1 : w.p0) + rhs * w.vstride;
    double *x = w.args->x[rhs];
    const int total = op.nrows * op.nv;
    for (int v = blockIdx.x * NT + threadIdx.x; v < total; v += gridDim.x * NT) {
        const size_t cell = 2 * (size_t)v;
        double2 xv = ld2(x, cell);
        const double2 pv = ld2(p, cell);
        xv.x = fma(alpha, pv.x, xv.x);
        xv.y = fma(alpha, pv.y, xv.y);
        st2(x, cell, xv);
    }
}

}  // namespace mas

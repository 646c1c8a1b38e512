// kernels_base.cuh -- set_dt plane scaling, plain matvec (mas_pcg_apply / init), init, the fused
// vector kernel K2, and the straightforward fused matvec K1 "variant 0" (neighbours through
// L1/L2, p_new recomputed per neighbour).  Variant 0 is the in-library correctness baseline for
// the tiled kernels in kernels_march.cuh.
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

// ---------------------------------------------------------------------------------------------
// the 7-point stencil on one double2 (cells k = 2kv, k+1 of row (i,j)), coefficient form:
//   (A u)_c = d_c u_c - vp[k] (ARm u_im + ARp u_ip + ATm u_jm + ATp u_jp) - F (ip[k] u_kp + ip[k-1] u_km)
// ---------------------------------------------------------------------------------------------
struct RowCoef {
    double E, F, ARm, ARp, ATm, ATp;
};

__device__ __forceinline__ RowCoef load_coef(const OpDev &op, int i, int j)
{
    RowCoef c;
    const int row = i * op.nt + j;
    c.E = __ldg(op.E + row);
    c.F = __ldg(op.F + row);
    c.ARm = __ldg(op.AR + row);
    c.ARp = __ldg(op.AR + row + op.nt);
    c.ATm = __ldg(op.AT + i * (op.nt + 1) + j);
    c.ATp = __ldg(op.AT + i * (op.nt + 1) + j + 1);
    return c;
}

struct PhiCoef {            // phi factors of the two cells of a vector and their outer faces
    double vp0, vp1, wp0, wp1, ipm, ip0, ip1;   // ipm = ip[k-1], ip0 = ip[k], ip1 = ip[k+1]
    int km, kp;                                 // wrapped neighbour cells k-1 and k+2
};

__device__ __forceinline__ PhiCoef load_phi(const OpDev &op, int kv)
{
    PhiCoef c;
    const int k = 2 * kv;
    c.km = k == 0 ? op.np - 1 : k - 1;
    c.kp = k + 2 >= op.np ? 0 : k + 2;
    c.vp0 = __ldg(op.vp + k);
    c.vp1 = __ldg(op.vp + k + 1);
    c.wp0 = __ldg(op.wp + k);
    c.wp1 = __ldg(op.wp + k + 1);
    c.ipm = __ldg(op.ip + c.km);
    c.ip0 = __ldg(op.ip + k);
    c.ip1 = __ldg(op.ip + k + 1);
    return c;
}

__device__ __forceinline__ double2 stencil(const RowCoef &c, const PhiCoef &f, double2 u, double2 uim,
                                           double2 uip, double2 ujm, double2 ujp, double ukm, double ukp)
{
    const double d0 = fma(f.vp0, c.E, c.F * f.wp0);
    const double d1 = fma(f.vp1, c.E, c.F * f.wp1);
    const double sx = c.ARm * uim.x + c.ARp * uip.x + c.ATm * ujm.x + c.ATp * ujp.x;
    const double sy = c.ARm * uim.y + c.ARp * uip.y + c.ATm * ujm.y + c.ATp * ujp.y;
    double2 q;
    q.x = d0 * u.x - f.vp0 * sx - c.F * (f.ip0 * u.y + f.ipm * ukm);
    q.y = d1 * u.y - f.vp1 * sy - c.F * (f.ip1 * ukp + f.ip0 * u.x);
    return q;
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
// y = A_sym u   (mas_pcg_apply; also A x0 for the initial residual).  u = xin, or args->x if null.
// ---------------------------------------------------------------------------------------------
template <int NT>
__global__ void __launch_bounds__(NT) k_apply(OpDev op, const double *xin, const SolveArgs *args, double *y)
{
    const double *u = xin ? xin : args->x;
    const RowMap m = row_map<NT>(op.nv);
    if (m.idle) return;
    const double2 zero = make_double2(0.0, 0.0);
    for (int rowbase = blockIdx.x * m.rb; rowbase < op.nrows; rowbase += gridDim.x * m.rb) {
        const int row = rowbase + m.rl;
        if (row >= op.nrows) break;
        const int i = row / op.nt, j = row - i * op.nt;
        const RowCoef c = load_coef(op, i, j);
        const size_t base = (size_t)row * op.np;
        const size_t sr = (size_t)op.nt * op.np;
        for (int kv = m.kv0; kv < op.nv; kv += m.nvc) {
            const PhiCoef f = load_phi(op, kv);
            const size_t cell = base + 2 * kv;
            const double2 uc = ld2(u, cell);
            const double2 uim = i > 0 ? ld2(u, cell - sr) : zero;
            const double2 uip = i < op.nr - 1 ? ld2(u, cell + sr) : zero;
            const double2 ujm = j > 0 ? ld2(u, cell - op.np) : zero;
            const double2 ujp = j < op.nt - 1 ? ld2(u, cell + op.np) : zero;
            const double ukm = u[base + f.km], ukp = u[base + f.kp];
            st2(y, cell, stencil(c, f, uc, uim, uip, ujm, ujp, ukm, ukp));
        }
    }
}

// ---------------------------------------------------------------------------------------------
// init (S1): r = V.b - q (q = A x0), p_in = 0, bb = |V.b|^2, rr = |r|^2, rho = r.(r/d); then the
// last block sets hist[0], k = 0, beta = 0 and the loop condition.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void set_cond(cudaGraphConditionalHandle cond, int use_cond, int v)
{
    if (use_cond) cudaGraphSetConditional(cond, v ? 1u : 0u);
}

template <int NT, bool UNIFORM>
__global__ void __launch_bounds__(NT) k_init(OpDev op, Work w, cudaGraphConditionalHandle cond, int use_cond)
{
    __shared__ double sh[32];
    const double *b = w.args->b;
    const RowMap m = row_map<NT>(op.nv);
    double acc[3] = {0.0, 0.0, 0.0};   // bb, rr, rho
    if (!m.idle)
        for (int rowbase = blockIdx.x * m.rb; rowbase < op.nrows; rowbase += gridDim.x * m.rb) {
            const int row = rowbase + m.rl;
            if (row >= op.nrows) break;
            const double E = __ldg(op.E + row), F = __ldg(op.F + row), V2 = __ldg(op.V2 + row);
            const double dinv = __ldg(op.Dinv + row);
            const size_t base = (size_t)row * op.np;
            for (int kv = m.kv0; kv < op.nv; kv += m.nvc) {
                const int k = 2 * kv;
                const double vp0 = __ldg(op.vp + k), vp1 = __ldg(op.vp + k + 1);
                const double d0 = fma(vp0, E, F * __ldg(op.wp + k)), d1 = fma(vp1, E, F * __ldg(op.wp + k + 1));
                const size_t cell = base + k;
                const double2 bv = ld2(b, cell), qv = ld2(w.q, cell);
                const double bs0 = V2 * vp0 * bv.x, bs1 = V2 * vp1 * bv.y;
                double2 r;
                r.x = bs0 - qv.x;
                r.y = bs1 - qv.y;
                st2(w.r, cell, r);
                st2(w.p0, cell, make_double2(0.0, 0.0));
                acc[0] += bs0 * bs0 + bs1 * bs1;
                acc[1] += r.x * r.x + r.y * r.y;
                acc[2] += UNIFORM ? r.x * (r.x * dinv) + r.y * (r.y * dinv)      // same z as K1/K2 use
                                  : r.x * (r.x / d0) + r.y * (r.y / d1);
            }
        }
    if (grid_sum<NT, 3>(acc, w.partials, &w.st->ticket[0], sh) && threadIdx.x == 0) {
        State *st = w.st;
        const double bb = acc[0], rr = acc[1], rho = acc[2];
        st->bb = bb; st->rr = rr; st->rho = rho;
        st->beta = 0.0; st->alpha = 0.0; st->sigma = 0.0;
        st->k = 0; st->launches = 0;
        int active = 0, status = ST_OK;
        if (!isfinite(bb) || !isfinite(rr) || !isfinite(rho)) {
            w.hist[0] = sqrt(rr / bb);          // a non-finite scalar (NaN / Inf in b or x0): breakdown, x untouched
            status = ST_BREAKDOWN;
        } else if (bb == 0.0) {
            w.hist[0] = 0.0;                    // zero RHS: x = 0 (host zeroes x), 0 iterations
        } else {
            const double h = sqrt(rr / bb);
            w.hist[0] = h;
            active = (0 < w.args->maxit) && (h > w.args->rtol) && (rho != 0.0);
            if (!active) status = (h <= w.args->rtol || rho == 0.0) ? ST_OK : ST_MAXIT;
        }
        st->active = active;
        st->status = status;
        set_cond(cond, use_cond, active);
    }
}

// ---------------------------------------------------------------------------------------------
// K2 (S4+S5): x += alpha p; r -= alpha q; z = r/d; rho' = r.z; rr = r.r; last block: k++,
// hist[k], beta, convergence test, graph conditional.  6N doubles of traffic.
// ---------------------------------------------------------------------------------------------
// XF = true: the x-update lives in K1 (deferred one iteration), K2 only touches r and q: 3N doubles.
// the last block of every K2 variant ends with this (S5): k++, hist[k], beta, convergence test
__device__ __forceinline__ void k2_finish(State *st, const Work &w, double rho1, double rr,
                                          cudaGraphConditionalHandle cond, int use_cond)
{
    const int k = st->k + 1;
    const double h = sqrt(rr / st->bb);
    w.hist[k] = h;
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
    set_cond(cond, use_cond, active);
}

// `reverse`: sweep the rows from the last to the first (serpentine: K1 marches forward in r, so the
// planes it touched last -- q, r -- are still in L2 when K2 starts there, and K2's last rows are in L2
// when the next K1 starts at i = 0).  The row -> block -> partial mapping stays fixed, so determinism holds.
template <int NT, bool UNIFORM, bool XF>
__global__ void __launch_bounds__(NT) k2_vec(OpDev op, Work w, cudaGraphConditionalHandle cond, int use_cond,
                                             int reverse)
{
    __shared__ double sh[32];
    cudaGridDependencySynchronize();                  // PDL edge from K1 (no-op for a plain launch)
    State *st = w.st;
    if (!st->active) return;
    const double alpha = st->alpha;
    const double *p = (st->k & 1) ? w.p0 : w.p1;      // written by K1 of this iteration
    double *x = w.args->x;
    const RowMap m = row_map<NT>(op.nv);
    double acc[2] = {0.0, 0.0};   // rho', rr
    // Two row groups per trip (A and B, one grid stride apart): their loads are issued together, which
    // doubles the bytes in flight per thread -- K2 has no other latency hiding than memory parallelism.
    auto body = [&](int row, int kv, double2 rv, double2 qv, double2 xv, double2 pv, double E, double F, double dinv) {
        const size_t cell = (size_t)row * op.np + 2 * kv;
        if (!XF) {
            xv.x = fma(alpha, pv.x, xv.x);
            xv.y = fma(alpha, pv.y, xv.y);
            st2(x, cell, xv);
        }
        rv.x = fma(-alpha, qv.x, rv.x);
        rv.y = fma(-alpha, qv.y, rv.y);
        st2(w.r, cell, rv);
        double z0, z1;
        if (UNIFORM) { z0 = rv.x * dinv; z1 = rv.y * dinv; }
        else {
            const int k = 2 * kv;
            z0 = rv.x / fma(__ldg(op.vp + k), E, F * __ldg(op.wp + k));
            z1 = rv.y / fma(__ldg(op.vp + k + 1), E, F * __ldg(op.wp + k + 1));
        }
        acc[0] += rv.x * z0 + rv.y * z1;
        acc[1] += rv.x * rv.x + rv.y * rv.y;
    };
    if (!m.idle) {
        const int stride = gridDim.x * m.rb;
        const double2 zero = make_double2(0.0, 0.0);
        for (int rowbase = blockIdx.x * m.rb; rowbase < op.nrows; rowbase += 2 * stride) {
            int rowA = rowbase + m.rl, rowB = rowA + stride;
            const bool okA = rowA < op.nrows, okB = rowB < op.nrows;
            if (!okA) break;
            if (reverse) { rowA = op.nrows - 1 - rowA; rowB = op.nrows - 1 - rowB; }
            double EA = 0, FA = 0, dA = 0, EB = 0, FB = 0, dB = 0;
            if (UNIFORM) { dA = __ldg(op.Dinv + rowA); if (okB) dB = __ldg(op.Dinv + rowB); }
            else {
                EA = __ldg(op.E + rowA); FA = __ldg(op.F + rowA);
                if (okB) { EB = __ldg(op.E + rowB); FB = __ldg(op.F + rowB); }
            }
            const size_t baseA = (size_t)rowA * op.np, baseB = okB ? (size_t)rowB * op.np : 0;
            for (int kv = m.kv0; kv < op.nv; kv += m.nvc) {
                const size_t cA = baseA + 2 * kv, cB = baseB + 2 * kv;
                const double2 rA = ld2(w.r, cA), qA = ld2(w.q, cA);
                const double2 rB = okB ? ld2(w.r, cB) : zero, qB = okB ? ld2(w.q, cB) : zero;
                double2 xA = zero, pA = zero, xB = zero, pB = zero;
                if (!XF) {
                    xA = ld2(x, cA); pA = ld2(p, cA);
                    if (okB) { xB = ld2(x, cB); pB = ld2(p, cB); }
                }
                body(rowA, kv, rA, qA, xA, pA, EA, FA, dA);
                if (okB) body(rowB, kv, rB, qB, xB, pB, EB, FB, dB);
            }
        }
    }
    cudaTriggerProgrammaticLaunchCompletion();        // PDL: K1 of the next iteration may start its prologue
    if (grid_sum<NT, 2>(acc, w.partials, &st->ticket[2], sh) && threadIdx.x == 0)
        k2_finish(st, w, acc[0], acc[1], cond, use_cond);
}

// XF tail (after the loop): the one x-update still pending, x += alpha_{k-1} p_{k-1}.  alpha is 0 when
// nothing is pending (no iteration ran, or K1 broke down after applying the previous update).
template <int NT>
__global__ void __launch_bounds__(NT) k_xtail(OpDev op, Work w)
{
    const State *st = w.st;
    const double alpha = st->alpha;
    const double *p = (st->k & 1) ? w.p1 : w.p0;
    double *x = w.args->x;
    const RowMap m = row_map<NT>(op.nv);
    if (m.idle) return;
    for (int rowbase = blockIdx.x * m.rb; rowbase < op.nrows; rowbase += gridDim.x * m.rb) {
        const int row = rowbase + m.rl;
        if (row >= op.nrows) break;
        const size_t base = (size_t)row * op.np;
        for (int kv = m.kv0; kv < op.nv; kv += m.nvc) {
            const size_t cell = base + 2 * kv;
            double2 xv = ld2(x, cell);
            const double2 pv = ld2(p, cell);
            xv.x = fma(alpha, pv.x, xv.x);
            xv.y = fma(alpha, pv.y, xv.y);
            st2(x, cell, xv);
        }
    }
}

// the last block of every K1 variant ends with this: sigma -> alpha, breakdown test (S3)
__device__ __forceinline__ void k1_finish(State *st, double sigma, cudaGraphConditionalHandle cond, int use_cond)
{
    st->sigma = sigma;
    st->launches += 1;
    if (!(sigma > 0.0) || isinf(sigma)) {
        st->status = ST_BREAKDOWN;
        st->active = 0;
        st->alpha = 0.0;                 // nothing pending for the XF tail
        set_cond(cond, use_cond, 0);
    } else {
        st->alpha = st->rho / sigma;
    }
}

// ---------------------------------------------------------------------------------------------
// K1 variant 0 (S2): p_new = r/d + beta p_old at the cell and at each of its 6 neighbours
// (recomputed), q = A p_new, sigma = p_new.q.  Neighbour rows come through L1/L2.
// ---------------------------------------------------------------------------------------------
template <bool UNIFORM>
__device__ __forceinline__ double pn1(double r, double p, double beta, double E, double F, double dinv, double vp,
                                      double wp)
{
    return fma(beta, p, UNIFORM ? r * dinv : r / fma(vp, E, F * wp));   // same z as K2 computes
}

template <int NT, bool UNIFORM>
__global__ void __launch_bounds__(NT) k1_v0(OpDev op, Work w, cudaGraphConditionalHandle cond, int use_cond)
{
    __shared__ double sh[32];
    State *st = w.st;
    if (!st->active) return;
    const double beta = st->beta;
    const double *pin = (st->k & 1) ? w.p1 : w.p0;
    double *pout = (st->k & 1) ? w.p0 : w.p1;
    const double *r = w.r;
    const RowMap m = row_map<NT>(op.nv);
    const double2 zero = make_double2(0.0, 0.0);
    double acc[1] = {0.0};
    if (!m.idle)
        for (int rowbase = blockIdx.x * m.rb; rowbase < op.nrows; rowbase += gridDim.x * m.rb) {
            const int row = rowbase + m.rl;
            if (row >= op.nrows) break;
            const int i = row / op.nt, j = row - i * op.nt;
            const RowCoef c = load_coef(op, i, j);
            const size_t base = (size_t)row * op.np;
            const size_t sr = (size_t)op.nt * op.np;
            for (int kv = m.kv0; kv < op.nv; kv += m.nvc) {
                const PhiCoef f = load_phi(op, kv);
                const size_t cell = base + 2 * kv;
                auto pnv = [&](size_t cl, int rw) {
                    const double2 rv = ld2(r, cl), pv = ld2(pin, cl);
                    const double E = __ldg(op.E + rw), F = __ldg(op.F + rw), di = __ldg(op.Dinv + rw);
                    return make_double2(pn1<UNIFORM>(rv.x, pv.x, beta, E, F, di, f.vp0, f.wp0),
                                        pn1<UNIFORM>(rv.y, pv.y, beta, E, F, di, f.vp1, f.wp1));
                };
                const double2 u = pnv(cell, row);
                const double2 uim = i > 0 ? pnv(cell - sr, row - op.nt) : zero;
                const double2 uip = i < op.nr - 1 ? pnv(cell + sr, row + op.nt) : zero;
                const double2 ujm = j > 0 ? pnv(cell - op.np, row - 1) : zero;
                const double2 ujp = j < op.nt - 1 ? pnv(cell + op.np, row + 1) : zero;
                const double di = __ldg(op.Dinv + row);
                const double ukm = pn1<UNIFORM>(r[base + f.km], pin[base + f.km], beta, c.E, c.F, di,
                                                __ldg(op.vp + f.km), __ldg(op.wp + f.km));
                const double ukp = pn1<UNIFORM>(r[base + f.kp], pin[base + f.kp], beta, c.E, c.F, di,
                                                __ldg(op.vp + f.kp), __ldg(op.wp + f.kp));
                const double2 q = stencil(c, f, u, uim, uip, ujm, ujp, ukm, ukp);
                st2(pout, cell, u);
                st2(w.q, cell, q);
                acc[0] += u.x * q.x + u.y * q.y;
            }
        }
    if (grid_sum<NT, 1>(acc, w.partials, &st->ticket[1], sh) && threadIdx.x == 0)
        k1_finish(st, acc[0], cond, use_cond);
}

// ---------------------------------------------------------------------------------------------
// Measurement aids (mas_pcg_mix_probe): trivial LINEAR kernels with the DRAM read/write mix of K1 and K2 and
// none of their structure -- what the memory system sustains for that mix, as context for the rooflines.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_mix6(const double2 *a, const double2 *b, double2 *x, double2 *p, double2 *q,
                                              size_t n2)        // K1 (xfuse): reads a, b, x; writes p, q, x
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n2; i += (size_t)gridDim.x * blockDim.x) {
        const double2 av = a[i], bv = b[i], xv = x[i];
        p[i] = make_double2(av.x + bv.x, av.y + bv.y);
        q[i] = make_double2(av.x - bv.x, av.y - bv.y);
        x[i] = make_double2(xv.x + 0.5 * av.x, xv.y + 0.5 * av.y);
    }
}

__global__ void __launch_bounds__(256) k_mix3(double2 *r, const double2 *q, size_t n2)   // K2: reads r, q; writes r
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n2; i += (size_t)gridDim.x * blockDim.x) {
        const double2 rv = r[i], qv = q[i];
        r[i] = make_double2(rv.x - 0.5 * qv.x, rv.y - 0.5 * qv.y);
    }
}

}  // namespace mas

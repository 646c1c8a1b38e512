// kernels_persistent.cuh -- the whole PCG solve as ONE cooperative kernel, for meshes small enough that the
// per-cell state x, r, p, q fits in the SMs' shared memory ("persistent cooperative
// single-kernel loop for L2-resident grids").  On such meshes the two-kernel graph loop is bound by launch
// and dependency latency (~25 us per iteration for 32x32x64), not by bandwidth.
//
// Same arithmetic as the streaming path (R3, R6), reorganised so that an iteration needs only two
// grid-wide barriers:
//   * a thread owns M 16-byte vectors (2 cells each) for the whole solve, kept in its own shared-memory slots;
//   * it publishes z_k (array Z) before the second barrier of iteration k-1 and p_{k-1} (array P[(k-1)&1])
//     one barrier earlier, so after that barrier every thread can form its neighbours'
//     p_k = z_k + beta p_{k-1} locally once beta is known: no third barrier for the p-update;
//   * reductions are deterministic: per-block partial -> barrier -> every block sums all partials in the
//     same fixed order, so all blocks see identical alpha, beta and take identical control flow.
#pragma once
#include <cooperative_groups.h>

#include "common.cuh"
#include "kernels_base.cuh"

namespace mas {

namespace cg = cooperative_groups;

// ---------------------------------------------------------------------------------------------
// the 7-point stencil on one double2 (cells k = 2kv, k+1 of row (i,j)), coefficient form, operands from global memory:
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

constexpr int PNT = 512;         // threads per block, one block per SM
constexpr int PMAX_SMEM = 226 * 1024;   // dynamic shared memory available to the one block per SM

struct PersistParams {
    double *Z, *P0, *P1;         // handle-owned N-vectors (the streaming path's r, p0, p1 workspaces)
    double *partials;            // [6][pstride]: regions 0 (sigma), 1-2 (rho', rr), 3-5 (init)
    int pstride;                 // >= gridDim.x
    double *hist;
    State *st;
    const SolveArgs *args;
    int nvec;                    // N / 2
    int M;                       // vectors per thread
};

inline size_t persist_smem(int M) { return (size_t)M * PNT * (4 * sizeof(double2) + sizeof(int2)); }

// fixed-order sum of NP partial arrays written by all blocks; result identical in every block
template <int NP>
__device__ __forceinline__ void all_sum(double (&v)[NP], double *partials, int pstride, double *sh, cg::grid_group &grid)
{
    const int G = gridDim.x;
#pragma unroll
    for (int q = 0; q < NP; q++) {
        const double t = block_sum<PNT>(v[q], sh);
        if (threadIdx.x == 0) partials[(size_t)q * pstride + blockIdx.x] = t;
    }
    grid.sync();
#pragma unroll
    for (int q = 0; q < NP; q++) {
        double a = 0.0;
        if (threadIdx.x < 32) {
            for (int i = threadIdx.x; i < G; i += 32) a += __ldcg(&partials[(size_t)q * pstride + i]);
            a = warp_sum(a);
        }
        if (threadIdx.x == 0) sh[q] = a;
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < NP; q++) v[q] = sh[q];
    __syncthreads();
}

template <bool UNIFORM>
__global__ void __launch_bounds__(PNT, 1) k_pcg_persistent(OpDev op, PersistParams pp)
{
    __shared__ double sh[32];
    extern __shared__ __align__(16) unsigned char psm[];
    cg::grid_group grid = cg::this_grid();
    const double *__restrict__ b = pp.args->b[0];
    double *__restrict__ xg = pp.args->x[0];
    const double rtol = pp.args->rtol;
    const int maxit = pp.args->maxit;
    const int M = pp.M, tid = threadIdx.x;
    const int T = gridDim.x * PNT, gtid = blockIdx.x * PNT + tid;
    const size_t sr = (size_t)op.nt * op.np;

    // per-thread state lives in shared memory, slot [array][m][tid]: x, r, p, q and (row, kv)
    double2 *SX = reinterpret_cast<double2 *>(psm), *SR = SX + M * PNT, *SP = SR + M * PNT, *SQ = SP + M * PNT;
    int2 *SK = reinterpret_cast<int2 *>(SQ + M * PNT);
    for (int m = 0; m < M; m++) {
        const int v = gtid + m * T;
        const int rw = v < pp.nvec ? v / op.nv : -1;
        SK[m * PNT + tid] = make_int2(rw, v < pp.nvec ? v - rw * op.nv : 0);
    }

    // neighbour value from a published array A0, or A0 + beta A1 formed on the fly (p_k = z_k + beta p_{k-1})
    auto nb2 = [&](const double *A0, const double *A1, double beta, size_t cell) {
        double2 a = __ldcg(reinterpret_cast<const double2 *>(A0 + cell));
        if (A1) {
            const double2 c = __ldcg(reinterpret_cast<const double2 *>(A1 + cell));
            a.x = fma(beta, c.x, a.x);
            a.y = fma(beta, c.y, a.y);
        }
        return a;
    };
    auto nb1 = [&](const double *A0, const double *A1, double beta, size_t cell) {
        double a = __ldcg(A0 + cell);
        if (A1) a = fma(beta, __ldcg(A1 + cell), a);
        return a;
    };
    auto matvec = [&](int rw, int kvv, double2 u, const double *A0, const double *A1, double beta) {
        const int i = rw / op.nt, j = rw - i * op.nt;
        const RowCoef c = load_coef(op, i, j);
        const PhiCoef f = load_phi(op, kvv);
        const size_t base = (size_t)rw * op.np, cell = base + 2 * kvv;
        const double2 zero = make_double2(0.0, 0.0);
        const double2 uim = i > 0 ? nb2(A0, A1, beta, cell - sr) : zero;
        const double2 uip = i < op.nr - 1 ? nb2(A0, A1, beta, cell + sr) : zero;
        const double2 ujm = j > 0 ? nb2(A0, A1, beta, cell - op.np) : zero;
        const double2 ujp = j < op.nt - 1 ? nb2(A0, A1, beta, cell + op.np) : zero;
        const double ukm = nb1(A0, A1, beta, base + f.km), ukp = nb1(A0, A1, beta, base + f.kp);
        return stencil(c, f, u, uim, uip, ujm, ujp, ukm, ukp);
    };
    auto zvec = [&](int rw, int kvv, double2 rv) {      // same z as the streaming kernels (R6)
        const int k = 2 * kvv;
        if (UNIFORM) {
            const double dinv = __ldg(op.Dinv + rw);
            return make_double2(rv.x * dinv, rv.y * dinv);
        }
        const double E = __ldg(op.E + rw), F = __ldg(op.F + rw);
        return make_double2(rv.x * rcp_nr(fma(__ldg(op.vp + k), E, F * __ldg(op.wp + k))),
                            rv.y * rcp_nr(fma(__ldg(op.vp + k + 1), E, F * __ldg(op.wp + k + 1))));
    };

    // ---- init: b_s = V b, r = b_s - A x0, z_0 -> Z, P[1] = 0 (p_{-1}), sums bb, rr, rho ----
    double acc3[3] = {0.0, 0.0, 0.0};
    for (int m = 0; m < M; m++) {
        const int2 rk = SK[m * PNT + tid];
        if (rk.x < 0) continue;
        const size_t cell = (size_t)rk.x * op.np + 2 * rk.y;
        const int k = 2 * rk.y;
        const double2 xv = ld2(xg, cell), bv = ld2(b, cell);
        const double V2 = __ldg(op.V2 + rk.x);
        const double bs0 = V2 * __ldg(op.vp + k) * bv.x, bs1 = V2 * __ldg(op.vp + k + 1) * bv.y;
        const double2 q = matvec(rk.x, rk.y, xv, xg, nullptr, 0.0);
        const double2 rv = make_double2(bs0 - q.x, bs1 - q.y);
        const double2 z = zvec(rk.x, rk.y, rv);
        SX[m * PNT + tid] = xv;
        SR[m * PNT + tid] = rv;
        SP[m * PNT + tid] = make_double2(0.0, 0.0);
        st2(pp.Z, cell, z);
        st2(pp.P1, cell, make_double2(0.0, 0.0));
        acc3[0] += bs0 * bs0 + bs1 * bs1;
        acc3[1] += rv.x * rv.x + rv.y * rv.y;
        acc3[2] += rv.x * z.x + rv.y * z.y;
    }
    all_sum<3>(acc3, pp.partials + 3 * (size_t)pp.pstride, pp.pstride, sh, grid);      // barrier: Z, P1 visible
    const double bb = acc3[0];
    double rho = acc3[2], rr = acc3[1], beta = 0.0, alpha = 0.0;
    int k = 0, status = ST_OK, active = 0;
    double h = 0.0;
    if (!isfinite(bb) || !isfinite(rr) || !isfinite(rho)) {
        h = sqrt(rr / bb);
        status = ST_BREAKDOWN;
    } else if (bb != 0.0) {
        h = sqrt(rr / bb);
        active = (0 < maxit) && (h > rtol) && (rho != 0.0);
        if (!active) status = (h <= rtol || rho == 0.0) ? ST_OK : ST_MAXIT;
    }
    if (gtid == 0) pp.hist[0] = h;

    while (active) {
        // ---- K1 role: p_k = z_k + beta p_{k-1}; publish p_k; q = A p_k with neighbours formed locally ----
        double *Pw = (k & 1) ? pp.P1 : pp.P0;              // receives p_k
        const double *Pr = (k & 1) ? pp.P0 : pp.P1;        // holds p_{k-1}
        double a1[1] = {0.0};
        for (int m = 0; m < M; m++) {
            const int2 rk = SK[m * PNT + tid];
            if (rk.x < 0) continue;
            const size_t cell = (size_t)rk.x * op.np + 2 * rk.y;
            const double2 z = zvec(rk.x, rk.y, SR[m * PNT + tid]);
            double2 pv = SP[m * PNT + tid];
            pv.x = fma(beta, pv.x, z.x);
            pv.y = fma(beta, pv.y, z.y);
            SP[m * PNT + tid] = pv;
            st2(Pw, cell, pv);
            const double2 q = matvec(rk.x, rk.y, pv, pp.Z, Pr, beta);
            SQ[m * PNT + tid] = q;
            a1[0] += pv.x * q.x + pv.y * q.y;
        }
        all_sum<1>(a1, pp.partials, pp.pstride, sh, grid);            // barrier A: all reads of Z (= z_k) are done
        const double sigma = a1[0];
        if (!(sigma > 0.0) || isinf(sigma)) { status = ST_BREAKDOWN; break; }
        alpha = rho / sigma;
        // ---- K2 role: x, r, z_{k+1} -> Z, rho', rr ----
        double a2[2] = {0.0, 0.0};
        for (int m = 0; m < M; m++) {
            const int2 rk = SK[m * PNT + tid];
            if (rk.x < 0) continue;
            const size_t cell = (size_t)rk.x * op.np + 2 * rk.y;
            const double2 pv = SP[m * PNT + tid], q = SQ[m * PNT + tid];
            double2 xv = SX[m * PNT + tid], rv = SR[m * PNT + tid];
            xv.x = fma(alpha, pv.x, xv.x);
            xv.y = fma(alpha, pv.y, xv.y);
            rv.x = fma(-alpha, q.x, rv.x);
            rv.y = fma(-alpha, q.y, rv.y);
            SX[m * PNT + tid] = xv;
            SR[m * PNT + tid] = rv;
            const double2 z = zvec(rk.x, rk.y, rv);
            st2(pp.Z, cell, z);
            a2[0] += rv.x * z.x + rv.y * z.y;
            a2[1] += rv.x * rv.x + rv.y * rv.y;
        }
        all_sum<2>(a2, pp.partials + (size_t)pp.pstride, pp.pstride, sh, grid);   // barrier B: Z (= z_{k+1}) and P[k&1] visible
        const double rho1 = a2[0];
        rr = a2[1];
        k += 1;
        h = sqrt(rr / bb);
        if (gtid == 0) pp.hist[k] = h;
        beta = rho1 / rho;
        rho = rho1;
        active = (k < maxit) && (h > rtol) && (rho1 != 0.0);
        if (!isfinite(rho1) || !isfinite(rr)) { active = 0; status = ST_BREAKDOWN; }
        else if (!active) status = (h <= rtol || rho1 == 0.0) ? ST_OK : ST_MAXIT;
    }
    // ---- finish ----
    for (int m = 0; m < M; m++) {
        const int2 rk = SK[m * PNT + tid];
        if (rk.x >= 0) st2(xg, (size_t)rk.x * op.np + 2 * rk.y, SX[m * PNT + tid]);
    }
    if (gtid == 0) {
        State *st = pp.st;
        st->bb = bb; st->rr = rr; st->rho = rho; st->alpha = alpha; st->beta = beta;
        st->k = k; st->active = 0; st->status = status; st->launches = 1;
    }
}

}  // namespace mas

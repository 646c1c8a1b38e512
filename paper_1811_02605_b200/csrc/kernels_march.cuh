// kernels_march.cuh -- K1, the fused matrix-free matvec of the PCG iteration (
// PAPER.md:98 "sparse matrix-vector products (essentially stencil operations)"), as a 2.5-D
// marching-tile kernel for sm_100a:
//
//     p_new = r/d + beta p_old      (the p-update of the previous iteration, fused as a prologue)
//     q     = A_sym p_new           (7-point, matrix-free, coefficients from 2-D planes)
//     sigma = p_new . q             (deterministic two-stage reduction)
//
// A block owns a (TJ rows) x (64 phi cells) column of the mesh and marches along r over CI planes.
// Warp w handles tile row w-1 (warps 0 and TJ+1 are the theta-halo rows); a lane handles two
// adjacent phi cells (one 16-byte vector).  Data movement per step (= one r plane):
//   * r and p_old of the plane DEPTH steps ahead stream global -> shared with cp.async (LDGSTS),
//     each thread into its own FIFO slot, so DEPTH x 32 B per thread are in flight with no
//     registers held;
//   * p_new of the current plane goes to a 3-plane shared ring for the theta neighbours; phi
//     neighbours come by warp shuffle, r neighbours stay in registers across steps;
//   * the phi-halo cells (k0-1, k0+64; periodic wrap) ride in the same FIFO as 8-byte cp.async copies
//     issued by the edge lanes; the block's coefficient columns are staged in shared memory once.
// Each cell's r and p_old are read from DRAM once; halo rows/planes are L2 hits.
// k1_march (64-cell rows, "variant 1") is kept as the validated predecessor of k1_wide ("variant 2",
// further down), which is the default.
// p is double-buffered in global memory (p[k&1] -> p[(k+1)&1]) because neighbouring blocks read
// p_old halos while this block writes p_new.
#pragma once
#include "common.cuh"
#include "kernels_base.cuh"

namespace mas {

struct MarchParams {
    int nkt, njt, nit;     // tiles in phi, theta, r
    int ci;                // interior planes per block
};

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait()
{
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory");
}

constexpr int MARCH_TK = 64;                  // phi cells per tile row (32 lanes x double2)
constexpr int MARCH_CI_MAX = 32;              // max interior planes per block (coefficient staging)

__device__ __forceinline__ void cp_async8(void *smem, const void *gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(s), "l"(gmem) : "memory");
}

template <int TJ, int DEPTH>
struct MarchSmem {
    static constexpr int NW = TJ + 2;
    static constexpr int NT = NW * 32;
    static constexpr int NPL = MARCH_CI_MAX + 2;
    double2 fifo[DEPTH][2][NT];               // [stage][r|p][thread]       main cells, 16 B per thread
    double hfifo[DEPTH][2][2][NW];            // [stage][r|p][left|right][warp]  phi-halo cells
    double2 ring[3][NW][32];                  // p_new planes, [buffer][tile row + 1][lane]
    double cE[NPL][NW], cF[NPL][NW], cD[NPL][NW];   // diag planes of (plane, row); cD = Dinv
    double cAR[NPL][NW], cAT[NPL][NW];        // AR[ii][j] (face ii-1/2), AT[ii][j] (face j-1/2)
    double red[32];
};

template <int TJ, int DEPTH, bool UNIFORM, int MINB>
__global__ void __launch_bounds__((TJ + 2) * 32, MINB)
k1_march(OpDev op, Work w, MarchParams mp, cudaGraphConditionalHandle cond, int use_cond)
{
    using Smem = MarchSmem<TJ, DEPTH>;
    constexpr int NT = Smem::NT, NW = Smem::NW;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Smem &sm = *reinterpret_cast<Smem *>(smem_raw);

    State *st = w.st;
    if (!st->active) return;
    const double beta = st->beta;
    const double *__restrict__ pin = (st->k & 1) ? w.p1 : w.p0;
    double *__restrict__ pout = (st->k & 1) ? w.p0 : w.p1;
    const double *__restrict__ rvec = w.r;

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, tid = threadIdx.x;
    // tile coordinates: phi fastest, then theta, then r  => neighbouring tiles run together
    int b = blockIdx.x;
    const int kt = b % mp.nkt; b /= mp.nkt;
    const int jt = b % mp.njt;
    const int it = b / mp.njt;
    const int i0 = it * mp.ci, i1 = min(i0 + mp.ci, op.nr);      // interior planes [i0, i1)
    const int first = i0 - 1, last = i1;                         // planes whose p_new this block needs
    const int j = jt * TJ + warp - 1;                            // this warp's theta row
    const int k0 = kt * MARCH_TK;
    const int k = k0 + 2 * lane;                                 // first of this lane's two cells
    const int tkeff = min(MARCH_TK, op.np - k0);                 // valid cells of this tile row
    const bool row_ok = (j >= 0) && (j < op.nt);
    const bool lane_ok = 2 * lane < tkeff;
    const bool load_ok = row_ok && lane_ok;
    const bool do_q = (warp >= 1) && (warp <= TJ) && load_ok;
    const bool left_edge = do_q && (lane == 0), right_edge = do_q && (2 * lane + 2 == tkeff);
    // periodic phi-halo cells of this tile row
    const int kl = k0 == 0 ? op.np - 1 : k0 - 1;
    const int kr = k0 + tkeff >= op.np ? 0 : k0 + tkeff;

    // ---- stage this block's coefficient columns (one global latency, then LDS broadcasts) ----
    for (int e = tid; e < (last - first + 1) * NW; e += NT) {
        const int pl = e / NW, wr = e - pl * NW;
        const int ii = first + pl, jj = jt * TJ + wr - 1;
        const bool in = ii >= 0 && ii < op.nr && jj >= 0 && jj < op.nt;
        const int row = ii * op.nt + jj;
        sm.cE[pl][wr] = in ? __ldg(op.E + row) : 0.0;
        sm.cF[pl][wr] = in ? __ldg(op.F + row) : 0.0;
        sm.cD[pl][wr] = in ? __ldg(op.Dinv + row) : 0.0;
        sm.cAR[pl][wr] = (ii >= 0 && ii <= op.nr && jj >= 0 && jj < op.nt) ? __ldg(op.AR + row) : 0.0;
        sm.cAT[pl][wr] = (ii >= 0 && ii < op.nr && jj >= 0 && jj <= op.nt) ? __ldg(op.AT + ii * (op.nt + 1) + jj) : 0.0;
    }

    // phi factors of the lane's cells (general mesh); uniform meshes use cell 0's
    double vp0, vp1, wp0, wp1, ipm, ip0, ip1;
    {
        const int kk = (UNIFORM || !lane_ok) ? 0 : k;
        const int km = (UNIFORM || !lane_ok) ? 0 : (kk == 0 ? op.np - 1 : kk - 1);
        vp0 = __ldg(op.vp + kk); vp1 = __ldg(op.vp + kk + 1);
        wp0 = __ldg(op.wp + kk); wp1 = __ldg(op.wp + kk + 1);
        ipm = __ldg(op.ip + km); ip0 = __ldg(op.ip + kk); ip1 = __ldg(op.ip + kk + 1);
    }
    double vpl = 0, wpl = 0, vpr = 0, wpr = 0;
    if (!UNIFORM) {
        vpl = __ldg(op.vp + kl); wpl = __ldg(op.wp + kl);
        vpr = __ldg(op.vp + kr); wpr = __ldg(op.wp + kr);
    }

    const size_t plane = (size_t)op.nt * op.np;
    const size_t rowoff = row_ok ? (size_t)j * op.np : 0;

    auto issue = [&](int ii, int stage) {       // stream plane ii of r and p_old into the FIFOs
        if (load_ok && ii >= 0 && ii < op.nr) {
            const size_t rowbase = (size_t)ii * plane + rowoff;
            cp_async16(&sm.fifo[stage][0][tid], rvec + rowbase + k);
            cp_async16(&sm.fifo[stage][1][tid], pin + rowbase + k);
            if (left_edge) {
                cp_async8(&sm.hfifo[stage][0][0][warp], rvec + rowbase + kl);
                cp_async8(&sm.hfifo[stage][1][0][warp], pin + rowbase + kl);
            }
            if (right_edge) {
                cp_async8(&sm.hfifo[stage][0][1][warp], rvec + rowbase + kr);
                cp_async8(&sm.hfifo[stage][1][1][warp], pin + rowbase + kr);
            }
        }
        cp_async_commit();
    };
    auto zval = [&](double r, double E, double F, double dinv, double vp, double wp) {
        return UNIFORM ? r * dinv : r / fma(vp, E, F * wp);
    };

#pragma unroll
    for (int s = 0; s < DEPTH; s++) issue(first + s <= last ? first + s : -1, s);
    __syncthreads();                            // coefficient columns visible

    double2 pn_m = make_double2(0.0, 0.0), pn_c = make_double2(0.0, 0.0);   // planes i-1, i
    double hl_c = 0.0, hr_c = 0.0;                                          // phi-halo p_new of plane i
    double acc = 0.0;

    for (int ii = first, t = 0; ii <= last; ++ii, ++t) {
        const int stage = t % DEPTH;
        const bool plane_ok = (ii >= 0) && (ii < op.nr);
        const double En = sm.cE[t][warp], Fn = sm.cF[t][warp], dinv = sm.cD[t][warp];
        cp_async_wait<DEPTH - 1>();              // this thread's own slots of plane ii have landed
        double2 pn_n = make_double2(0.0, 0.0);
        double hl_n = 0.0, hr_n = 0.0;
        if (load_ok && plane_ok) {
            const double2 rv = sm.fifo[stage][0][tid], pv = sm.fifo[stage][1][tid];
            pn_n.x = fma(beta, pv.x, zval(rv.x, En, Fn, dinv, vp0, wp0));
            pn_n.y = fma(beta, pv.y, zval(rv.y, En, Fn, dinv, vp1, wp1));
            if (left_edge)
                hl_n = fma(beta, sm.hfifo[stage][1][0][warp], zval(sm.hfifo[stage][0][0][warp], En, Fn, dinv, vpl, wpl));
            if (right_edge)
                hr_n = fma(beta, sm.hfifo[stage][1][1][warp], zval(sm.hfifo[stage][0][1][warp], En, Fn, dinv, vpr, wpr));
            if (do_q && ii >= i0 && ii < i1) st2(pout, (size_t)ii * plane + rowoff + k, pn_n);
        }
        issue(ii + DEPTH <= last ? ii + DEPTH : -1, stage);     // refill the slots just consumed
        sm.ring[t % 3][warp][lane] = pn_n;
        __syncthreads();
        // ---- q for plane i = ii-1 (needs p_new of planes i-1, i, i+1) ----
        const int i = ii - 1;
        double ukm = __shfl_up_sync(0xffffffffu, pn_c.y, 1);
        double ukp = __shfl_down_sync(0xffffffffu, pn_c.x, 1);
        if (do_q && i >= i0) {
            if (left_edge) ukm = hl_c;
            if (right_edge) ukp = hr_c;
            const int rb = (t + 2) % 3;                          // ring buffer holding plane i
            const double2 ujm = sm.ring[rb][warp - 1][lane], ujp = sm.ring[rb][warp + 1][lane];
            const double Ec = sm.cE[t - 1][warp], Fc = sm.cF[t - 1][warp];
            const double ARm = sm.cAR[t - 1][warp], ARp = sm.cAR[t][warp];
            const double ATm = sm.cAT[t - 1][warp], ATp = sm.cAT[t - 1][warp + 1];
            const double d0 = fma(vp0, Ec, Fc * wp0), d1 = fma(vp1, Ec, Fc * wp1);
            const double sx = ARm * pn_m.x + ARp * pn_n.x + ATm * ujm.x + ATp * ujp.x;
            const double sy = ARm * pn_m.y + ARp * pn_n.y + ATm * ujm.y + ATp * ujp.y;
            double2 q;
            q.x = d0 * pn_c.x - vp0 * sx - Fc * (ip0 * pn_c.y + ipm * ukm);
            q.y = d1 * pn_c.y - vp1 * sy - Fc * (ip1 * ukp + ip0 * pn_c.x);
            st2(w.q, (size_t)i * plane + rowoff + k, q);
            acc += pn_c.x * q.x + pn_c.y * q.y;
        }
        pn_m = pn_c; pn_c = pn_n;
        hl_c = hl_n; hr_c = hr_n;
    }
    cp_async_wait<0>();
    double a1[1] = {acc};
    if (grid_sum<NT, 1>(a1, w.partials, &st->ticket[1], sm.red) && threadIdx.x == 0)
        k1_finish(st, a1[0], cond, use_cond);
}

// =============================================================================================
// K1 "wide": same algorithm, leaner instruction stream.  A warp covers a 128-cell row segment as
// two coalesced 64-cell halves (A: cells k0+2l.., B: cells k0+64+2l..), i.e. 4 cells per lane, so
// the per-plane overhead (barrier, loop control, coefficient loads, halo handling) is spread over
// twice the cells; global addresses are bumped pointers; the step loop is unrolled by
// lcm(3, DEPTH) so FIFO stage and ring buffer are compile-time; on uniform phi meshes the phi
// factors are kernel constants.
// =============================================================================================
constexpr int WIDE_TK = 128;

struct WideParams {
    int nkt, njt, nit, ci;
    double vp, wp, ip;                        // uniform-phi factors (dph_c, 2/dph_f, 1/dph_f)
};

template <int TJ, int DEPTH, bool XF>
struct WideSmem {
    static constexpr int NW = TJ + 2;
    static constexpr int NT = NW * 32;
    static constexpr int NPL = MARCH_CI_MAX + 2;
    double2 fifo[DEPTH][XF ? 6 : 4][NT];      // [stage][rA rB pA pB (xA xB)][thread]
    double hfifo[DEPTH][4][NW];               // [stage][r_left r_right p_left p_right][warp]
    double2 ring[3][NW][64];                  // p_new planes: [buffer][row][A lanes 0..31 | B lanes 32..63]
    double cE[NPL][NW], cF[NPL][NW], cD[NPL][NW], cAR[NPL][NW], cAT[NPL][NW];
    double phv[WIDE_TK + 2], phw[WIDE_TK + 2], phi[WIDE_TK + 2];   // general phi: vp, wp, ip of cells k0-1..k0+128
    double red[32];
};

// NOQ: q is not stored (K2R recomputes it from p_new): K1 then moves 5 doubles per cell.
template <int TJ, int DEPTH, bool UNIFORM, int MINB, bool XF, bool NOQ>
__global__ void __launch_bounds__((TJ + 2) * 32, MINB)
k1_wide(OpDev op, Work w, WideParams mp, cudaGraphConditionalHandle cond, int use_cond)
{
    using Smem = WideSmem<TJ, DEPTH, XF>;
    constexpr int NT = Smem::NT, NW = Smem::NW;
    constexpr int U = (DEPTH % 3 == 0) ? DEPTH : 3 * DEPTH;     // unroll: stage and ring index static
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Smem &sm = *reinterpret_cast<Smem *>(smem_raw);

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, tid = threadIdx.x;
    int b = blockIdx.x;
    const int kt = b % mp.nkt; b /= mp.nkt;
    const int jt = b % mp.njt;
    const int it = b / mp.njt;
    const int i0 = it * mp.ci, i1 = min(i0 + mp.ci, op.nr);
    const int first = i0 - 1, nsteps = i1 - i0 + 2;
    const int j = jt * TJ + warp - 1;
    const int k0 = kt * WIDE_TK;
    const int tkeff = min(WIDE_TK, op.np - k0);
    const bool row_ok = (j >= 0) && (j < op.nt);
    const bool vA = row_ok && (2 * lane < tkeff), vB = row_ok && (64 + 2 * lane < tkeff);
    const bool interior = (warp >= 1) && (warp <= TJ);
    const bool qA = interior && vA, qB = interior && vB;
    const bool left_edge = qA && (lane == 0);
    const bool right_A = qA && (2 * lane + 2 == tkeff), right_B = qB && (64 + 2 * lane + 2 == tkeff);
    const bool right_edge = right_A || right_B;
    const int kl = k0 == 0 ? op.np - 1 : k0 - 1;
    const int kr = k0 + tkeff >= op.np ? 0 : k0 + tkeff;

    // ---- stage coefficient columns, phi factors; zero the FIFOs (invalid lanes then read zeros) ----
    for (int e = tid; e < nsteps * NW; e += NT) {
        const int pl = e / NW, wr = e - pl * NW;
        const int ii = first + pl, jj = jt * TJ + wr - 1;
        const bool in = ii >= 0 && ii < op.nr && jj >= 0 && jj < op.nt;
        const int row = ii * op.nt + jj;
        sm.cE[pl][wr] = in ? __ldg(op.E + row) : 0.0;
        sm.cF[pl][wr] = in ? __ldg(op.F + row) : 0.0;
        sm.cD[pl][wr] = in ? __ldg(op.Dinv + row) : 0.0;
        sm.cAR[pl][wr] = (ii >= 0 && ii <= op.nr && jj >= 0 && jj < op.nt) ? __ldg(op.AR + row) : 0.0;
        sm.cAT[pl][wr] = (ii >= 0 && ii < op.nr && jj >= 0 && jj <= op.nt) ? __ldg(op.AT + ii * (op.nt + 1) + jj) : 0.0;
    }
    if (!UNIFORM)
        for (int e = tid; e < WIDE_TK + 2; e += NT) {
            int kk = k0 - 1 + e;                                  // wrap once in either direction
            kk = kk < 0 ? kk + op.np : (kk >= op.np ? kk - op.np : kk);
            kk = kk >= op.np ? kk % op.np : kk;                   // tiny meshes (np < 130)
            sm.phv[e] = __ldg(op.vp + kk); sm.phw[e] = __ldg(op.wp + kk); sm.phi[e] = __ldg(op.ip + kk);
        }
#pragma unroll
    for (int s = 0; s < DEPTH; s++) {
#pragma unroll
        for (int a = 0; a < (XF ? 6 : 4); a++) sm.fifo[s][a][tid] = make_double2(0.0, 0.0);
        if (lane < 4) sm.hfifo[s][lane][warp] = 0.0;
    }
    __syncthreads();

    // Everything above depends only on the operator, not on the previous kernel: with a programmatic
    // (PDL) edge this block may have been launched while K2 of the previous iteration was still draining.
    // From here on the iteration state and the vectors are read, so wait for the predecessor to complete
    // (a no-op when the kernel was launched without the programmatic attribute).
    cudaGridDependencySynchronize();
    State *st = w.st;
    if (!st->active) return;
    const double beta = st->beta;
    const int par = st->k & 1;
    const double *__restrict__ pin = par ? w.p1 : w.p0;
    double *__restrict__ pout = par ? w.p0 : w.p1;
    const double *__restrict__ rvec = w.r;
    // XF: the x-update of the PREVIOUS iteration, x += alpha_{k-1} p_{k-1}, is applied here (p_old is
    // p_{k-1}); K2 then only updates r.  Same operations on the same operands as the unfused path.
    const double alpha_prev = XF ? st->alpha : 0.0;
    double *__restrict__ xvec = XF ? w.args->x : nullptr;

    // phi factors: cells A0,A1 (k, k+1) and B0,B1 (k+64, k+65); index into the staged arrays is cell-k0+1
    const int ea = 2 * lane + 1, eb = 2 * lane + 65;
    auto VP = [&](int e) { return UNIFORM ? mp.vp : sm.phv[e]; };
    auto WP = [&](int e) { return UNIFORM ? mp.wp : sm.phw[e]; };
    auto IP = [&](int e) { return UNIFORM ? mp.ip : sm.phi[e]; };   // ip of face e+1/2
    auto zval = [&](double r, double E, double F, double dinv, int e) {
        return UNIFORM ? r * dinv : r / fma(VP(e), E, F * WP(e));
    };

    // ---- bumped pointers ----
    const long long plane = (long long)op.nt * op.np;
    const long long rowbase0 = (long long)first * plane + (row_ok ? (long long)j * op.np : 0);
    const double *ldr = rvec + rowbase0;            // row base of the next plane to prefetch
    const double *ldp = pin + rowbase0;
    const int ka = k0 + 2 * lane, kb = ka + 64;
    double *stp = pout + rowbase0 + plane;          // row base of plane i0 (first store of p)
    double *stq = w.q + rowbase0 + plane;           // row base of plane i0 (first store of q)
    double *xrow = XF ? xvec + rowbase0 + plane : nullptr;   // row base of plane i0 (x is updated in place)
    const double *ldx = XF ? xvec + rowbase0 : nullptr;       // x rides in the FIFO with r and p_old of its plane
    int ii_ld = first;                              // plane index of the next prefetch

    auto issue = [&](int stage) {
        if ((unsigned)ii_ld < (unsigned)op.nr && ii_ld <= i1) {
            if (vA) { cp_async16(&sm.fifo[stage][0][tid], ldr + ka); cp_async16(&sm.fifo[stage][2][tid], ldp + ka); }
            if (vB) { cp_async16(&sm.fifo[stage][1][tid], ldr + kb); cp_async16(&sm.fifo[stage][3][tid], ldp + kb); }
            if (left_edge) { cp_async8(&sm.hfifo[stage][0][warp], ldr + kl); cp_async8(&sm.hfifo[stage][2][warp], ldp + kl); }
            if (right_edge) { cp_async8(&sm.hfifo[stage][1][warp], ldr + kr); cp_async8(&sm.hfifo[stage][3][warp], ldp + kr); }
            if (XF && ii_ld >= i0 && ii_ld < i1) {              // interior plane: its x
                if (qA) cp_async16(&sm.fifo[stage][XF ? 4 : 0][tid], ldx + ka);
                if (qB) cp_async16(&sm.fifo[stage][XF ? 5 : 0][tid], ldx + kb);
            }
        }
        cp_async_commit();
        ldr += plane; ldp += plane; ++ii_ld;
        if (XF) ldx += plane;
    };

#pragma unroll
    for (int s = 0; s < DEPTH; s++) issue(s);

    double2 am = make_double2(0.0, 0.0), ac = am, bm = am, bc = am;   // p_new of planes i-1 (m), i (c); halves A, B
    double hl_c = 0.0, hr_c = 0.0;
    double acc = 0.0;
    const int lm = (lane + 31) & 31, lp = (lane + 1) & 31;

    for (int tb = 0; tb < nsteps; tb += U) {
#pragma unroll
        for (int u = 0; u < U; u++) {
            const int t = tb + u;
            if (t >= nsteps) break;
            const int stage = u % DEPTH, rbw = u % 3, rbr = (u + 2) % 3;
            const int ii = first + t;
            const bool plane_ok = (unsigned)ii < (unsigned)op.nr;
            const double En = sm.cE[t][warp], Fn = sm.cF[t][warp], dinv = sm.cD[t][warp];
            cp_async_wait<DEPTH - 1>();
            double2 an = make_double2(0.0, 0.0), bn = an;
            double hl_n = 0.0, hr_n = 0.0;
            if (plane_ok) {                         // block-uniform
                const double2 ra = sm.fifo[stage][0][tid], rb = sm.fifo[stage][1][tid];
                const double2 pa = sm.fifo[stage][2][tid], pb = sm.fifo[stage][3][tid];
                if (UNIFORM || vA) {
                    an.x = fma(beta, pa.x, zval(ra.x, En, Fn, dinv, ea));
                    an.y = fma(beta, pa.y, zval(ra.y, En, Fn, dinv, ea + 1));
                }
                if (UNIFORM || vB) {
                    bn.x = fma(beta, pb.x, zval(rb.x, En, Fn, dinv, eb));
                    bn.y = fma(beta, pb.y, zval(rb.y, En, Fn, dinv, eb + 1));
                }
                if (left_edge) hl_n = fma(beta, sm.hfifo[stage][2][warp], zval(sm.hfifo[stage][0][warp], En, Fn, dinv, 0));
                if (right_edge) hr_n = fma(beta, sm.hfifo[stage][3][warp], zval(sm.hfifo[stage][1][warp], En, Fn, dinv, tkeff + 1));
                if (t >= 1 && t <= nsteps - 2) {    // interior plane: store p_new (and the deferred x-update)
                    if (qA) st2(stp, ka, an);
                    if (qB) st2(stp, kb, bn);
                    stp += plane;
                    if (XF) {
                        if (qA) {
                            double2 xa = sm.fifo[stage][XF ? 4 : 0][tid];
                            xa.x = fma(alpha_prev, pa.x, xa.x); xa.y = fma(alpha_prev, pa.y, xa.y);
                            st2(xrow, ka, xa);
                        }
                        if (qB) {
                            double2 xb = sm.fifo[stage][XF ? 5 : 0][tid];
                            xb.x = fma(alpha_prev, pb.x, xb.x); xb.y = fma(alpha_prev, pb.y, xb.y);
                            st2(xrow, kb, xb);
                        }
                        xrow += plane;
                    }
                }
            }
            issue(stage);
            sm.ring[rbw][warp][lane] = an;
            sm.ring[rbw][warp][lane + 32] = bn;
            __syncthreads();
            // ---- q for plane i = ii-1 ----
            const double mA = __shfl_sync(0xffffffffu, ac.y, lm), mB = __shfl_sync(0xffffffffu, bc.y, lm);
            const double pA = __shfl_sync(0xffffffffu, ac.x, lp), pB = __shfl_sync(0xffffffffu, bc.x, lp);
            if (t >= 2 && interior && row_ok) {
                const double Ec = sm.cE[t - 1][warp], Fc = sm.cF[t - 1][warp];
                const double ARm = sm.cAR[t - 1][warp], ARp = sm.cAR[t][warp];
                const double ATm = sm.cAT[t - 1][warp], ATp = sm.cAT[t - 1][warp + 1];
                if (qA) {
                    const double ukm = left_edge ? hl_c : mA;
                    const double ukp = right_A ? hr_c : (lane == 31 ? pB : pA);
                    const double2 ujm = sm.ring[rbr][warp - 1][lane], ujp = sm.ring[rbr][warp + 1][lane];
                    const double d0 = fma(VP(ea), Ec, Fc * WP(ea)), d1 = fma(VP(ea + 1), Ec, Fc * WP(ea + 1));
                    const double sx = ARm * am.x + ARp * an.x + ATm * ujm.x + ATp * ujp.x;
                    const double sy = ARm * am.y + ARp * an.y + ATm * ujm.y + ATp * ujp.y;
                    double2 q;
                    q.x = d0 * ac.x - VP(ea) * sx - Fc * (IP(ea) * ac.y + IP(ea - 1) * ukm);
                    q.y = d1 * ac.y - VP(ea + 1) * sy - Fc * (IP(ea + 1) * ukp + IP(ea) * ac.x);
                    if (!NOQ) st2(stq, ka, q);
                    acc += ac.x * q.x + ac.y * q.y;
                }
                if (qB) {
                    const double ukm = lane == 0 ? mA : mB;
                    const double ukp = right_B ? hr_c : pB;
                    const double2 ujm = sm.ring[rbr][warp - 1][lane + 32], ujp = sm.ring[rbr][warp + 1][lane + 32];
                    const double d0 = fma(VP(eb), Ec, Fc * WP(eb)), d1 = fma(VP(eb + 1), Ec, Fc * WP(eb + 1));
                    const double sx = ARm * bm.x + ARp * bn.x + ATm * ujm.x + ATp * ujp.x;
                    const double sy = ARm * bm.y + ARp * bn.y + ATm * ujm.y + ATp * ujp.y;
                    double2 q;
                    q.x = d0 * bc.x - VP(eb) * sx - Fc * (IP(eb) * bc.y + IP(eb - 1) * ukm);
                    q.y = d1 * bc.y - VP(eb + 1) * sy - Fc * (IP(eb + 1) * ukp + IP(eb) * bc.x);
                    if (!NOQ) st2(stq, kb, q);
                    acc += bc.x * q.x + bc.y * q.y;
                }
            }
            if (t >= 2) stq += plane;
            am = ac; ac = an; bm = bc; bc = bn;
            hl_c = hl_n; hr_c = hr_n;
        }
    }
    cudaTriggerProgrammaticLaunchCompletion();      // PDL: the successor's blocks may start their prologue
    cp_async_wait<0>();
    double a1[1] = {acc};
    if (grid_sum<NT, 1>(a1, w.partials, &st->ticket[1], sm.red) && threadIdx.x == 0)
        k1_finish(st, a1[0], cond, use_cond);
}

// ---------------------------------------------------------------------------------------------
// host-side configuration table
// ---------------------------------------------------------------------------------------------
struct MarchTile {
    int tj, depth, minb;
};
static const MarchTile kMarchTiles[] = {{8, 4, 3}, {8, 6, 2}, {14, 4, 1}, {6, 6, 3}, {14, 3, 2}, {8, 3, 4}, {6, 4, 4}};
inline int march_num_tiles() { return (int)(sizeof(kMarchTiles) / sizeof(kMarchTiles[0])); }

template <int TJ, int DEPTH, int MINB>
inline void march_pick(bool uniform, const void **func, dim3 *block, size_t *smem)
{
    *func = uniform ? (const void *)k1_march<TJ, DEPTH, true, MINB> : (const void *)k1_march<TJ, DEPTH, false, MINB>;
    *block = dim3((TJ + 2) * 32);
    *smem = sizeof(MarchSmem<TJ, DEPTH>);
    cudaFuncSetAttribute(*func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)*smem);
}

inline void march_configure(int nr, int nt, int np, int uniform, int tile, int num_sms, MarchParams *mp,
                            const void **func, dim3 *grid, dim3 *block, size_t *smem)
{
    const MarchTile T = kMarchTiles[tile];
    switch (tile) {
        case 0: march_pick<8, 4, 3>(uniform, func, block, smem); break;
        case 1: march_pick<8, 6, 2>(uniform, func, block, smem); break;
        case 2: march_pick<14, 4, 1>(uniform, func, block, smem); break;
        case 3: march_pick<6, 6, 3>(uniform, func, block, smem); break;
        case 4: march_pick<14, 3, 2>(uniform, func, block, smem); break;
        case 5: march_pick<8, 3, 4>(uniform, func, block, smem); break;
        default: march_pick<6, 4, 4>(uniform, func, block, smem); break;
    }
    mp->nkt = (np + MARCH_TK - 1) / MARCH_TK;
    mp->njt = (nt + T.tj - 1) / T.tj;
    // r-chunk length: long chunks amortise the 2 halo planes; short ones give more blocks.
    int ci = MARCH_CI_MAX;
    while (ci > 8 && (long long)mp->nkt * mp->njt * ((nr + ci - 1) / ci) < 8LL * num_sms) ci /= 2;
    mp->ci = ci;
    mp->nit = (nr + ci - 1) / ci;
    *grid = dim3((unsigned)(mp->nkt * mp->njt * mp->nit));
}

// ---- wide variant ----
struct WideTile {
    int tj, depth, minb;
};
static const WideTile kWideTiles[] = {{8, 2, 2}, {6, 3, 2}, {6, 2, 3}, {14, 3, 1}, {8, 3, 2}, {4, 3, 3}, {10, 3, 1}};
inline int wide_num_tiles() { return (int)(sizeof(kWideTiles) / sizeof(kWideTiles[0])); }

template <int TJ, int DEPTH, int MINB>
inline void wide_pick(bool uniform, int xf, const void **func, dim3 *block, size_t *smem)
{
    if (xf == 2)        // xfuse + q not stored
        *func = uniform ? (const void *)k1_wide<TJ, DEPTH, true, MINB, true, true> : (const void *)k1_wide<TJ, DEPTH, false, MINB, true, true>;
    else if (xf)
        *func = uniform ? (const void *)k1_wide<TJ, DEPTH, true, MINB, true, false> : (const void *)k1_wide<TJ, DEPTH, false, MINB, true, false>;
    else
        *func = uniform ? (const void *)k1_wide<TJ, DEPTH, true, MINB, false, false> : (const void *)k1_wide<TJ, DEPTH, false, MINB, false, false>;
    *block = dim3((TJ + 2) * 32);
    *smem = xf ? sizeof(WideSmem<TJ, DEPTH, true>) : sizeof(WideSmem<TJ, DEPTH, false>);
    cudaFuncSetAttribute(*func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)*smem);
}

inline void wide_configure(int nr, int nt, int np, int uniform, int xf, int tile, int num_sms, int ci_force, WideParams *mp,
                           const void **func, dim3 *grid, dim3 *block, size_t *smem)
{
    const WideTile T = kWideTiles[tile];
    switch (tile) {
        case 0: wide_pick<8, 2, 2>(uniform, xf, func, block, smem); break;
        case 1: wide_pick<6, 3, 2>(uniform, xf, func, block, smem); break;
        case 2: wide_pick<6, 2, 3>(uniform, xf, func, block, smem); break;
        case 3: wide_pick<14, 3, 1>(uniform, xf, func, block, smem); break;
        case 4: wide_pick<8, 3, 2>(uniform, xf, func, block, smem); break;
        case 5: wide_pick<4, 3, 3>(uniform, xf, func, block, smem); break;
        default: wide_pick<10, 3, 1>(uniform, xf, func, block, smem); break;
    }
    mp->nkt = (np + WIDE_TK - 1) / WIDE_TK;
    mp->njt = (nt + T.tj - 1) / T.tj;
    int occ = 1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, *func, (int)block->x, *smem) != cudaSuccess || occ < 1) {
        cudaGetLastError();
        occ = 1;
    }
    const long long slots = (long long)num_sms * occ, cols = (long long)mp->nkt * mp->njt;
    // r-chunk length: minimise rounds x (planes per block + halo planes + start-up), ties -> longer chunks
    int best = MARCH_CI_MAX;
    double best_cost = 1e300;
    for (int ci = MARCH_CI_MAX; ci >= 4; ci -= 2) {
        const long long tiles = cols * ((nr + ci - 1) / ci);
        if (tiles > MAX_PARTIALS) continue;
        const double rounds = (double)((tiles + slots - 1) / slots);
        const double cost = rounds * (ci + 2 + 3);
        if (cost < best_cost * 0.999) { best_cost = cost; best = ci; }
    }
    if (nr < best) best = nr;
    if (ci_force > 0 && ci_force <= MARCH_CI_MAX) best = ci_force;
    mp->ci = best;
    mp->nit = (nr + best - 1) / best;
    *grid = dim3((unsigned)(mp->nkt * mp->njt * mp->nit));
}

}  // namespace mas

// kernels_k1_tma.cuh -- K1 (fused p-update + matvec + p.Ap + deferred x-update, 6 doubles per cell; see
// kernels_march.cuh for the algorithm and the tiling) with the TMA engine as the loader and mbarriers instead of
// the block barrier:
//   * every warp owns one tile row; lane 0 bulk-copies (cp.async.bulk, SASS UBLKCP) that row's r, p_old, x segments
//     and the two 16-byte phi-halo pairs of r and p_old for the plane DEPTH steps ahead into the warp's own FIFO
//     stage, signalling the warp's own mbarrier ldfull[stage][warp] (count 1 + transaction bytes).  A warp waits only
//     for ITS row -- there is no block-wide coupling on the load path;
//   * p_new planes go to a shared ring of FOUR planes; every thread arrives on ringfull[plane % 4] after storing its
//     part, and a warp waits for plane t-1 to be complete before reading its theta-neighbours' rows.  With four
//     buffers that wait also proves the slot written at step t (plane t-4) is no longer being read, so K1 has no
//     __syncthreads in its loop: warps drift by up to a plane instead of meeting at a barrier every plane.
#pragma once
#include "kernels_march.cuh"
#include "kernels_stencil_tma.cuh"

namespace mas {

template <int TJ, int DEPTH, bool UNIFORM>
struct K1TmaSmem {
    static constexpr int NW = TJ + 2;
    static constexpr int NT = NW * 32;
    static constexpr int NPL = MARCH_CI_MAX + 2;
    alignas(16) double2 fr[DEPTH][NW][64];                // r rows (tile + theta-halo rows), 128 cells each
    alignas(16) double2 fp[DEPTH][NW][64];                // p_old rows
    alignas(16) double2 fx[DEPTH][TJ][64];                // x rows (interior rows only)
    alignas(16) double2 fh[DEPTH][NW][4];                 // phi-halo pairs: r left, r right, p left, p right
    alignas(16) double2 ring[4][NW][64];                  // p_new planes
    double cE[NPL][NW], cF[NPL][NW], cD[NPL][NW], cAR[NPL][NW], cAT[NPL][NW];
    double phv[UNIFORM ? 1 : WIDE_TK + 2], phw[UNIFORM ? 1 : WIDE_TK + 2], phi[UNIFORM ? 1 : WIDE_TK + 2];
    double red[32];
    alignas(8) uint64_t ldfull[DEPTH][NW];
    alignas(8) uint64_t ringfull[4];
};

template <int TJ, int DEPTH, bool UNIFORM, int MINB>
__global__ void __launch_bounds__((TJ + 2) * 32, MINB)
k1_tma(OpDev op, Work w, WideParams mp, cudaGraphConditionalHandle cond, int use_cond)
{
    using Smem = K1TmaSmem<TJ, DEPTH, UNIFORM>;
    constexpr int NT = Smem::NT, NW = Smem::NW;
    extern __shared__ __align__(128) unsigned char smem_raw[];
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
    const int kl = k0 == 0 ? op.np - 1 : k0 - 1;           // odd
    const int kr = k0 + tkeff >= op.np ? 0 : k0 + tkeff;   // even

    // ---- zero-fill and barrier init first, so that the first bulk copies can be issued as early as possible ----
    const double2 zero2 = make_double2(0.0, 0.0);
#pragma unroll
    for (int s = 0; s < DEPTH; s++) {
        sm.fr[s][warp][lane] = zero2; sm.fr[s][warp][lane + 32] = zero2;
        sm.fp[s][warp][lane] = zero2; sm.fp[s][warp][lane + 32] = zero2;
        if (interior) { sm.fx[s][warp - 1][lane] = zero2; sm.fx[s][warp - 1][lane + 32] = zero2; }
        if (lane < 4) sm.fh[s][warp][lane] = zero2;
    }
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < DEPTH; s++)
            for (int r = 0; r < NW; r++) mbar_init(&sm.ldfull[s][r], 1);
#pragma unroll
        for (int s = 0; s < 4; s++) mbar_init(&sm.ringfull[s], NT);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
    __syncthreads();

    cudaGridDependencySynchronize();            // (PDL-capable; a no-op for a plain launch)
    State *st = w.st;
    if (!st->active) return;
    const double beta = st->beta;
    const int par = st->k & 1;
    const double *__restrict__ pin = par ? w.p1 : w.p0;
    double *__restrict__ pout = par ? w.p0 : w.p1;
    const double *__restrict__ rvec = w.r;
    const double alpha_prev = st->alpha;        // x += alpha_{k-1} p_{k-1}: the deferred x-update (xfuse)
    double *__restrict__ xvec = w.args->x;

    const int ea = 2 * lane + 1, eb = 2 * lane + 65;
    auto VP = [&](int e) { return UNIFORM ? mp.vp : sm.phv[e]; };
    auto WP = [&](int e) { return UNIFORM ? mp.wp : sm.phw[e]; };
    auto IP = [&](int e) { return UNIFORM ? mp.ip : sm.phi[e]; };
    auto zval = [&](double r, double E, double F, double dinv, int e) {
        return UNIFORM ? r * dinv : r / fma(VP(e), E, F * WP(e));
    };

    const long long plane = (long long)op.nt * op.np;
    const long long rowbase0 = (long long)first * plane + (row_ok ? (long long)j * op.np : 0);
    const int ka = k0 + 2 * lane, kb = ka + 64;
    long long prow = rowbase0 + plane;           // row base of plane i0: p_new / x stores
    long long qrow = rowbase0 + plane;           // row base of plane i0: q stores
    const unsigned rowbytes = (unsigned)tkeff * 8u;

    // lane 0: this warp's row of plane index pl -> FIFO stage pl % DEPTH
    auto produce = [&](int pl) {
        const int stage = pl % DEPTH, ii = first + pl;
        uint64_t *bar = &sm.ldfull[stage][warp];
        const bool in = row_ok && (unsigned)ii < (unsigned)op.nr;
        const bool xin = in && interior && ii >= i0 && ii < i1;
        const unsigned bytes = in ? (2u * rowbytes + (interior ? 64u : 0u) + (xin ? rowbytes : 0u)) : 0u;
        if (bytes == 0) { mbar_arrive(bar); return; }
        mbar_arrive_expect_tx(bar, bytes);
        const long long rb = rowbase0 + (long long)pl * plane;
        bulk_g2s(&sm.fr[stage][warp][0], rvec + rb + k0, rowbytes, bar);
        bulk_g2s(&sm.fp[stage][warp][0], pin + rb + k0, rowbytes, bar);
        if (interior) {
            bulk_g2s(&sm.fh[stage][warp][0], rvec + rb + (kl - 1), 16u, bar);
            bulk_g2s(&sm.fh[stage][warp][1], rvec + rb + kr, 16u, bar);
            bulk_g2s(&sm.fh[stage][warp][2], pin + rb + (kl - 1), 16u, bar);
            bulk_g2s(&sm.fh[stage][warp][3], pin + rb + kr, 16u, bar);
        }
        if (xin) bulk_g2s(&sm.fx[stage][warp - 1][0], xvec + rb + k0, rowbytes, bar);
    };
    if (lane == 0)
        for (int pl = 0; pl < DEPTH && pl < nsteps; pl++) produce(pl);

    // ---- coefficient columns and phi factors, staged while the first planes are already in flight ----
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
            int kk = k0 - 1 + e;
            kk = kk < 0 ? kk + op.np : (kk >= op.np ? kk - op.np : kk);
            kk = kk >= op.np ? kk % op.np : kk;
            sm.phv[e] = __ldg(op.vp + kk); sm.phw[e] = __ldg(op.wp + kk); sm.phi[e] = __ldg(op.ip + kk);
        }
    __syncthreads();                            // coefficient columns visible

    double2 am = zero2, ac = zero2, bm = zero2, bc = zero2;
    double hl_c = 0.0, hr_c = 0.0;
    double acc = 0.0;
    const int lm = (lane + 31) & 31, lp = (lane + 1) & 31;

    for (int t = 0; t < nsteps; t++) {
        const int stage = t % DEPTH, rs = t & 3, rsp = (t + 3) & 3;
        const int ii = first + t;
        const bool plane_ok = (unsigned)ii < (unsigned)op.nr;
        const double En = sm.cE[t][warp], Fn = sm.cF[t][warp], dinv = sm.cD[t][warp];
        mbar_wait(&sm.ldfull[stage][warp], (unsigned)(t / DEPTH) & 1u);      // this warp's row of plane ii
        double2 an = zero2, bn = zero2;
        double hl_n = 0.0, hr_n = 0.0;
        if (plane_ok) {
            const double2 ra = sm.fr[stage][warp][lane], rb = sm.fr[stage][warp][lane + 32];
            const double2 pa = sm.fp[stage][warp][lane], pb = sm.fp[stage][warp][lane + 32];
            if (UNIFORM || vA) {
                an.x = fma(beta, pa.x, zval(ra.x, En, Fn, dinv, ea));
                an.y = fma(beta, pa.y, zval(ra.y, En, Fn, dinv, ea + 1));
            }
            if (UNIFORM || vB) {
                bn.x = fma(beta, pb.x, zval(rb.x, En, Fn, dinv, eb));
                bn.y = fma(beta, pb.y, zval(rb.y, En, Fn, dinv, eb + 1));
            }
            if (left_edge) hl_n = fma(beta, sm.fh[stage][warp][2].y, zval(sm.fh[stage][warp][0].y, En, Fn, dinv, 0));
            if (right_edge) hr_n = fma(beta, sm.fh[stage][warp][3].x, zval(sm.fh[stage][warp][1].x, En, Fn, dinv, tkeff + 1));
            if (t >= 1 && t <= nsteps - 2) {    // interior plane: store p_new and the deferred x-update
                if (qA) {
                    st2(pout, prow + ka, an);
                    double2 xa = sm.fx[stage][warp - 1][lane];
                    xa.x = fma(alpha_prev, pa.x, xa.x); xa.y = fma(alpha_prev, pa.y, xa.y);
                    st2(xvec, prow + ka, xa);
                }
                if (qB) {
                    st2(pout, prow + kb, bn);
                    double2 xb = sm.fx[stage][warp - 1][lane + 32];
                    xb.x = fma(alpha_prev, pb.x, xb.x); xb.y = fma(alpha_prev, pb.y, xb.y);
                    st2(xvec, prow + kb, xb);
                }
            }
        }
        if (t >= 1 && t <= nsteps - 2) prow += plane;
        __syncwarp();                                        // the warp is done with its FIFO stage
        if (lane == 0 && t + DEPTH < nsteps) produce(t + DEPTH);
        // ---- publish p_new of plane ii; wait for plane ii-1 of the whole tile ----
        sm.ring[rs][warp][lane] = an;
        sm.ring[rs][warp][lane + 32] = bn;
        mbar_arrive(&sm.ringfull[rs]);                       // every thread: its own stores are released
        const double mA = __shfl_sync(0xffffffffu, ac.y, lm), mB = __shfl_sync(0xffffffffu, bc.y, lm);
        const double pA = __shfl_sync(0xffffffffu, ac.x, lp), pB = __shfl_sync(0xffffffffu, bc.x, lp);
        if (t >= 1) mbar_wait(&sm.ringfull[rsp], (unsigned)((t - 1) >> 2) & 1u);
        // ---- q for plane i = ii-1 ----
        if (t >= 2 && interior && row_ok) {
            const double Ec = sm.cE[t - 1][warp], Fc = sm.cF[t - 1][warp];
            const double ARm = sm.cAR[t - 1][warp], ARp = sm.cAR[t][warp];
            const double ATm = sm.cAT[t - 1][warp], ATp = sm.cAT[t - 1][warp + 1];
            if (qA) {
                const double ukm = left_edge ? hl_c : mA;
                const double ukp = right_A ? hr_c : (lane == 31 ? pB : pA);
                const double2 ujm = sm.ring[rsp][warp - 1][lane], ujp = sm.ring[rsp][warp + 1][lane];
                const double d0 = fma(VP(ea), Ec, Fc * WP(ea)), d1 = fma(VP(ea + 1), Ec, Fc * WP(ea + 1));
                const double sx = ARm * am.x + ARp * an.x + ATm * ujm.x + ATp * ujp.x;
                const double sy = ARm * am.y + ARp * an.y + ATm * ujm.y + ATp * ujp.y;
                double2 q;
                q.x = d0 * ac.x - VP(ea) * sx - Fc * (IP(ea) * ac.y + IP(ea - 1) * ukm);
                q.y = d1 * ac.y - VP(ea + 1) * sy - Fc * (IP(ea + 1) * ukp + IP(ea) * ac.x);
                st2(w.q, qrow + ka, q);
                acc += ac.x * q.x + ac.y * q.y;
            }
            if (qB) {
                const double ukm = lane == 0 ? mA : mB;
                const double ukp = right_B ? hr_c : pB;
                const double2 ujm = sm.ring[rsp][warp - 1][lane + 32], ujp = sm.ring[rsp][warp + 1][lane + 32];
                const double d0 = fma(VP(eb), Ec, Fc * WP(eb)), d1 = fma(VP(eb + 1), Ec, Fc * WP(eb + 1));
                const double sx = ARm * bm.x + ARp * bn.x + ATm * ujm.x + ATp * ujp.x;
                const double sy = ARm * bm.y + ARp * bn.y + ATm * ujm.y + ATp * ujp.y;
                double2 q;
                q.x = d0 * bc.x - VP(eb) * sx - Fc * (IP(eb) * bc.y + IP(eb - 1) * ukm);
                q.y = d1 * bc.y - VP(eb + 1) * sy - Fc * (IP(eb + 1) * ukp + IP(eb) * bc.x);
                st2(w.q, qrow + kb, q);
                acc += bc.x * q.x + bc.y * q.y;
            }
        }
        if (t >= 2) qrow += plane;
        am = ac; ac = an; bm = bc; bc = bn;
        hl_c = hl_n; hr_c = hr_n;
    }
    cudaTriggerProgrammaticLaunchCompletion();
    double a1[1] = {acc};
    if (grid_sum<NT, 1>(a1, w.partials, &st->ticket[1], sm.red) && threadIdx.x == 0)
        k1_finish(st, a1[0], cond, use_cond);
}

// ---- host-side configuration: variant 3 ----
struct K1TmaTile {
    int tj, depth, minb;
};
static const K1TmaTile kK1TmaTiles[] = {{14, 2, 1}, {8, 2, 2}, {6, 2, 2}, {8, 3, 1}, {10, 2, 1}, {16, 2, 1}, {12, 2, 1}};
inline int k1_tma_num_tiles() { return (int)(sizeof(kK1TmaTiles) / sizeof(kK1TmaTiles[0])); }

template <int TJ, int DEPTH, int MINB>
inline void k1_tma_pick(bool uniform, const void **func, dim3 *block, size_t *smem)
{
    *func = uniform ? (const void *)k1_tma<TJ, DEPTH, true, MINB> : (const void *)k1_tma<TJ, DEPTH, false, MINB>;
    *smem = uniform ? sizeof(K1TmaSmem<TJ, DEPTH, true>) : sizeof(K1TmaSmem<TJ, DEPTH, false>);
    *block = dim3((TJ + 2) * 32);
    cudaFuncSetAttribute(*func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)*smem);
}

inline void k1_tma_configure(int nr, int nt, int np, int uniform, int tile, int num_sms, int ci_force, WideParams *mp,
                             const void **func, dim3 *grid, dim3 *block, size_t *smem)
{
    const K1TmaTile T = kK1TmaTiles[tile];
    switch (tile) {
        case 0: k1_tma_pick<14, 2, 1>(uniform, func, block, smem); break;
        case 1: k1_tma_pick<8, 2, 2>(uniform, func, block, smem); break;
        case 2: k1_tma_pick<6, 2, 2>(uniform, func, block, smem); break;
        case 3: k1_tma_pick<8, 3, 1>(uniform, func, block, smem); break;
        case 4: k1_tma_pick<10, 2, 1>(uniform, func, block, smem); break;
        case 5: k1_tma_pick<16, 2, 1>(uniform, func, block, smem); break;
        default: k1_tma_pick<12, 2, 1>(uniform, func, block, smem); break;
    }
    mp->nkt = (np + WIDE_TK - 1) / WIDE_TK;
    mp->njt = (nt + T.tj - 1) / T.tj;
    int occ = 1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, *func, (int)block->x, *smem) != cudaSuccess || occ < 1) {
        cudaGetLastError();
        occ = 1;
    }
    const long long slots = (long long)num_sms * occ, cols = (long long)mp->nkt * mp->njt;
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

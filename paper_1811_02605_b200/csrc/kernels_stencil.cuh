// kernels_stencil.cuh -- the matrix-free 7-point stencil applied to a STORED vector, as a 2.5-D marching
// kernel (same tiling as k1_wide: TJ theta rows x 128 phi cells per block, marching along r), with a fused
// epilogue.  Used by
//   * mas_pcg_apply and the initial residual (EPI_APPLY:  out = S u,  S = A_sym with the dt-scaled planes),
//   * the RKL2 super-time-stepping stages of NEXT-1 (EPI_STS: S = L_sym from the dt-independent planes,
//     M u = -S u / V,  out = c_u u + c_a1 a1 + c_a2 a2 + c_L M u + c_a3 a3,  optionally out2 = M u)
//     -- PAPER.md:65 "Runge-Kutta Legendre super time-stepping (STS) scheme [21]", "explicit
//     finite difference algorithms (such as ... the STS algorithm)".
// Because the input needs no prologue arithmetic, cp.async writes each plane (tile rows + theta-halo rows,
// plus the two periodic phi-halo cells per row) directly into a shared ring of DEPTH+2 planes: a thread reads
// its own cells after its own wait_group, neighbours' rows after the one barrier per plane.
#pragma once
#include "common.cuh"
#include "kernels_base.cuh"
#include "kernels_march.cuh"

namespace mas {

enum { EPI_APPLY = 0, EPI_STS = 1, EPI_K2R = 2 };   // K2R: PCG's K2 with q = A p recomputed (64 B/cell/it)

struct StencilParams {
    int nkt, njt, nit, ci;
    double vp, wp, ip;                    // uniform-phi factors
    const double *E, *F, *AR, *AT;        // plane set: diagonal per unit vp, phi coupling, radial / theta off-diagonals
    const double *Vinv;                   // [nrows] 1 / V2 (EPI_STS)
    const double *u;                      // the vector the stencil is applied to (null: args->x)
    const SolveArgs *args;
    double *out, *out2;
    const double *a1, *a2, *a3;           // EPI_STS: Y_{j-2}, Y_0, M Y_0 (null = absent)
    double c_u, c_a1, c_a2, c_L, c_a3;
    // EPI_K2R
    Work w;
    const double *Dinv;
    cudaGraphConditionalHandle cond;
    int use_cond;
};

template <int TJ, int DEPTH, int NX>      // NX = 6: extra streams through a cp.async FIFO; 0: none / via registers
struct StencilSmem {
    static constexpr int NW = TJ + 2;
    static constexpr int NT = NW * 32;
    static constexpr int R = DEPTH + 2;
    static constexpr int NPL = MARCH_CI_MAX + 2;
    double2 xf[NX ? DEPTH : 1][NX ? NX : 1][NX ? NT : 1];   // [stage][a1A a1B a2A a2B a3A a3B][thread]
    double2 ring[R][NW][64];              // planes of u: [slot][row][A lanes 0..31 | B lanes 32..63]
    double halo[R][NW][2];                // phi-halo cells of each row: [slot][row][left|right]
    double cE[NPL][NW], cF[NPL][NW], cAR[NPL][NW], cAT[NPL][NW], cV[NPL][NW];
    double phv[WIDE_TK + 2], phw[WIDE_TK + 2], phi[WIDE_TK + 2];
    double red[32];
};

template <int TJ, int DEPTH, bool UNIFORM, int MINB, int EPI, bool XFIFO>
__global__ void __launch_bounds__((TJ + 2) * 32, MINB)
k_stencil(OpDev op, StencilParams mp)
{
    static_assert(!XFIFO || (EPI != EPI_APPLY && DEPTH == 2), "extras FIFO: STS / K2R epilogue, DEPTH 2 (unroll = R = 4)");
    static_assert(EPI != EPI_K2R || XFIFO, "K2R takes r through the FIFO");
    using Smem = StencilSmem<TJ, DEPTH, XFIFO ? (EPI == EPI_K2R ? 2 : 6) : 0>;
    constexpr int NT = Smem::NT, NW = Smem::NW, R = Smem::R;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Smem &sm = *reinterpret_cast<Smem *>(smem_raw);

    double alpha = 0.0;
    const double *uk2 = nullptr;
    if (EPI == EPI_K2R) {                            // u = p written by K1 of this iteration; r updated in place
        if (!mp.w.st->active) return;
        alpha = mp.w.st->alpha;
        uk2 = (mp.w.st->k & 1) ? mp.w.p0 : mp.w.p1;
    }
    const double *__restrict__ uvec = EPI == EPI_K2R ? uk2 : (mp.u ? mp.u : mp.args->x);
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

    // ---- stage coefficient columns and phi factors; zero the ring (rows / lanes never loaded read 0) ----
    for (int e = tid; e < nsteps * NW; e += NT) {
        const int pl = e / NW, wr = e - pl * NW;
        const int ii = first + pl, jj = jt * TJ + wr - 1;
        const bool in = ii >= 0 && ii < op.nr && jj >= 0 && jj < op.nt;
        const int row = ii * op.nt + jj;
        sm.cE[pl][wr] = in ? __ldg(mp.E + row) : 0.0;
        sm.cF[pl][wr] = in ? __ldg(mp.F + row) : 0.0;
        sm.cV[pl][wr] = (in && EPI == EPI_STS) ? __ldg(mp.Vinv + row) : ((in && EPI == EPI_K2R) ? __ldg(mp.Dinv + row) : 0.0);
        sm.cAR[pl][wr] = (ii >= 0 && ii <= op.nr && jj >= 0 && jj < op.nt) ? __ldg(mp.AR + row) : 0.0;
        sm.cAT[pl][wr] = (ii >= 0 && ii < op.nr && jj >= 0 && jj <= op.nt) ? __ldg(mp.AT + ii * (op.nt + 1) + jj) : 0.0;
    }
    if (!UNIFORM)
        for (int e = tid; e < WIDE_TK + 2; e += NT) {
            int kk = k0 - 1 + e;
            kk = kk < 0 ? kk + op.np : (kk >= op.np ? kk - op.np : kk);
            kk = kk >= op.np ? kk % op.np : kk;
            sm.phv[e] = __ldg(op.vp + kk); sm.phw[e] = __ldg(op.wp + kk); sm.phi[e] = __ldg(op.ip + kk);
        }
#pragma unroll
    for (int s = 0; s < R; s++) {
        sm.ring[s][warp][lane] = make_double2(0.0, 0.0);
        sm.ring[s][warp][lane + 32] = make_double2(0.0, 0.0);
        if (lane < 2) sm.halo[s][warp][lane] = 0.0;
    }
    __syncthreads();

    const int ea = 2 * lane + 1, eb = 2 * lane + 65;
    auto VP = [&](int e) { return UNIFORM ? mp.vp : sm.phv[e]; };
    auto WP = [&](int e) { return UNIFORM ? mp.wp : sm.phw[e]; };
    auto IP = [&](int e) { return UNIFORM ? mp.ip : sm.phi[e]; };

    const long long plane = (long long)op.nt * op.np;
    const long long rowbase0 = (long long)first * plane + (row_ok ? (long long)j * op.np : 0);
    const double *ldu = uvec + rowbase0;            // row base of the next plane to prefetch
    const int ka = k0 + 2 * lane, kb = ka + 64;
    long long orow = rowbase0 + plane;              // row base (element offset) of plane i0: outputs / extras
    int ii_ld = first;

    const double *a1p = EPI == EPI_K2R ? mp.w.r : mp.a1;          // K2R: the one extra stream is r
    const bool has1 = (EPI == EPI_STS && mp.a1 != nullptr) || EPI == EPI_K2R,
               has2 = EPI == EPI_STS && mp.a2 != nullptr, has3 = EPI == EPI_STS && mp.a3 != nullptr;
    double acc[2] = {0.0, 0.0};                                  // K2R: rho', rr
    long long xoff = rowbase0 - plane;              // row base of plane ii_ld - 1: the plane whose outputs are
                                                    // formed when ring plane ii_ld is consumed
    auto issue = [&](int slot, int xstage) {
        if ((unsigned)ii_ld < (unsigned)op.nr && ii_ld <= i1) {
            if (vA) cp_async16(&sm.ring[slot][warp][lane], ldu + ka);
            if (vB) cp_async16(&sm.ring[slot][warp][lane + 32], ldu + kb);
            if (left_edge) cp_async8(&sm.halo[slot][warp][0], ldu + kl);
            if (right_edge) cp_async8(&sm.halo[slot][warp][1], ldu + kr);
        }
        if (XFIFO && ii_ld - 1 >= i0 && ii_ld - 1 < i1) {
            if (qA) {
                if (has1) cp_async16(&sm.xf[xstage][0][tid], a1p + xoff + ka);
                if (has2) cp_async16(&sm.xf[xstage][2][tid], mp.a2 + xoff + ka);
                if (has3) cp_async16(&sm.xf[xstage][4][tid], mp.a3 + xoff + ka);
            }
            if (qB) {
                if (has1) cp_async16(&sm.xf[xstage][1][tid], a1p + xoff + kb);
                if (has2) cp_async16(&sm.xf[xstage][3][tid], mp.a2 + xoff + kb);
                if (has3) cp_async16(&sm.xf[xstage][5][tid], mp.a3 + xoff + kb);
            }
        }
        cp_async_commit();
        ldu += plane; xoff += plane; ++ii_ld;
    };
#pragma unroll
    for (int s = 0; s < DEPTH; s++) issue(s, s % DEPTH);

    const double2 zero2 = make_double2(0.0, 0.0);
    double2 am = zero2, ac = zero2, bm = zero2, bc = zero2;
    double hl_c = 0.0, hr_c = 0.0;
    double2 x1a = zero2, x1b = zero2, x2a = zero2, x2b = zero2, x3a = zero2, x3b = zero2;   // extras of the next plane
    const int lm = (lane + 31) & 31, lp = (lane + 1) & 31;

    for (int tb = 0; tb < nsteps; tb += R) {
#pragma unroll
        for (int u = 0; u < R; u++) {
            const int t = tb + u;
            if (t >= nsteps) break;
            const int slot = u, slot_prev = (u + R - 1) % R, slot_ld = (u + DEPTH) % R;
            const int ii = first + t;
            const bool plane_ok = (unsigned)ii < (unsigned)op.nr;
            cp_async_wait<DEPTH - 1>();              // own cells of plane ii have landed
            double2 an = zero2, bn = zero2;
            double hl_n = 0.0, hr_n = 0.0;
            if (plane_ok) {                          // block-uniform; a stale slot must read as 0
                an = sm.ring[slot][warp][lane];
                bn = sm.ring[slot][warp][lane + 32];
                if (left_edge) hl_n = sm.halo[slot][warp][0];
                if (right_edge) hr_n = sm.halo[slot][warp][1];
            }
            // ---- S u for plane i = ii-1 ----
            const double mA = __shfl_sync(0xffffffffu, ac.y, lm), mB = __shfl_sync(0xffffffffu, bc.y, lm);
            const double pA = __shfl_sync(0xffffffffu, ac.x, lp), pB = __shfl_sync(0xffffffffu, bc.x, lp);
            if (t >= 2 && interior && row_ok) {
                const double Ec = sm.cE[t - 1][warp], Fc = sm.cF[t - 1][warp];
                const double ARm = sm.cAR[t - 1][warp], ARp = sm.cAR[t][warp];
                const double ATm = sm.cAT[t - 1][warp], ATp = sm.cAT[t - 1][warp + 1];
                const double vinv = EPI != EPI_APPLY ? sm.cV[t - 1][warp] : 0.0;
                auto finish = [&](double2 s, double2 uc, double2 x1, double2 x2, double2 x3, int e, int kcell) {
                    double2 o;
                    if (EPI == EPI_APPLY) {
                        o = s;
                    } else if (EPI == EPI_K2R) {                     // s = q = A p;  x1 = r
                        o.x = fma(-alpha, s.x, x1.x);
                        o.y = fma(-alpha, s.y, x1.y);
                        double z0, z1;
                        if (UNIFORM) { z0 = o.x * vinv; z1 = o.y * vinv; }     // vinv holds Dinv here
                        else { z0 = o.x / fma(VP(e), Ec, Fc * WP(e)); z1 = o.y / fma(VP(e + 1), Ec, Fc * WP(e + 1)); }
                        acc[0] += o.x * z0 + o.y * z1;
                        acc[1] += o.x * o.x + o.y * o.y;
                    } else {
                        double2 mu;                                  // M u = -S u / (V2 vp)
                        mu.x = UNIFORM ? -(s.x * vinv) * (1.0 / mp.vp) : -(s.x * vinv) / VP(e);
                        mu.y = UNIFORM ? -(s.y * vinv) * (1.0 / mp.vp) : -(s.y * vinv) / VP(e + 1);
                        if (mp.out2) st2(mp.out2, orow + kcell, mu);
                        o.x = mp.c_u * uc.x + mp.c_L * mu.x;
                        o.y = mp.c_u * uc.y + mp.c_L * mu.y;
                        if (has1) { o.x = fma(mp.c_a1, x1.x, o.x); o.y = fma(mp.c_a1, x1.y, o.y); }
                        if (has2) { o.x = fma(mp.c_a2, x2.x, o.x); o.y = fma(mp.c_a2, x2.y, o.y); }
                        if (has3) { o.x = fma(mp.c_a3, x3.x, o.x); o.y = fma(mp.c_a3, x3.y, o.y); }
                    }
                    st2(EPI == EPI_K2R ? mp.w.r : mp.out, orow + kcell, o);
                };
                // extras of this plane: the thread's own FIFO slots (landed with plane ii), or the registers
                // loaded one step ahead.  Fresh locals, so nothing is carried across steps in FIFO mode.
                const int xs = u % DEPTH;
                const double2 e1a = XFIFO ? ((has1 && qA) ? sm.xf[xs][0][tid] : zero2) : x1a;
                const double2 e1b = XFIFO ? ((has1 && qB) ? sm.xf[xs][1][tid] : zero2) : x1b;
                const double2 e2a = XFIFO ? ((has2 && qA) ? sm.xf[xs][2][tid] : zero2) : x2a;
                const double2 e2b = XFIFO ? ((has2 && qB) ? sm.xf[xs][3][tid] : zero2) : x2b;
                const double2 e3a = XFIFO ? ((has3 && qA) ? sm.xf[xs][4][tid] : zero2) : x3a;
                const double2 e3b = XFIFO ? ((has3 && qB) ? sm.xf[xs][5][tid] : zero2) : x3b;
                if (qA) {
                    const double ukm = left_edge ? hl_c : mA;
                    const double ukp = right_A ? hr_c : (lane == 31 ? pB : pA);
                    const double2 ujm = sm.ring[slot_prev][warp - 1][lane], ujp = sm.ring[slot_prev][warp + 1][lane];
                    const double d0 = fma(VP(ea), Ec, Fc * WP(ea)), d1 = fma(VP(ea + 1), Ec, Fc * WP(ea + 1));
                    const double sx = ARm * am.x + ARp * an.x + ATm * ujm.x + ATp * ujp.x;
                    const double sy = ARm * am.y + ARp * an.y + ATm * ujm.y + ATp * ujp.y;
                    double2 s;
                    s.x = d0 * ac.x - VP(ea) * sx - Fc * (IP(ea) * ac.y + IP(ea - 1) * ukm);
                    s.y = d1 * ac.y - VP(ea + 1) * sy - Fc * (IP(ea + 1) * ukp + IP(ea) * ac.x);
                    finish(s, ac, e1a, e2a, e3a, ea, ka);
                }
                if (qB) {
                    const double ukm = lane == 0 ? mA : mB;
                    const double ukp = right_B ? hr_c : pB;
                    const double2 ujm = sm.ring[slot_prev][warp - 1][lane + 32], ujp = sm.ring[slot_prev][warp + 1][lane + 32];
                    const double d0 = fma(VP(eb), Ec, Fc * WP(eb)), d1 = fma(VP(eb + 1), Ec, Fc * WP(eb + 1));
                    const double sx = ARm * bm.x + ARp * bn.x + ATm * ujm.x + ATp * ujp.x;
                    const double sy = ARm * bm.y + ARp * bn.y + ATm * ujm.y + ATp * ujp.y;
                    double2 s;
                    s.x = d0 * bc.x - VP(eb) * sx - Fc * (IP(eb) * bc.y + IP(eb - 1) * ukm);
                    s.y = d1 * bc.y - VP(eb + 1) * sy - Fc * (IP(eb + 1) * ukp + IP(eb) * bc.x);
                    finish(s, bc, e1b, e2b, e3b, eb, kb);
                }
            }
            if (t >= 2) orow += plane;
            // extras of plane ii (consumed at the next step): orow now points at plane ii when t >= 1
            if (EPI == EPI_STS && !XFIFO && t >= 1 && t <= nsteps - 2) {
                if (qA) {
                    if (has1) x1a = ld2(mp.a1, orow + ka);
                    if (has2) x2a = ld2(mp.a2, orow + ka);
                    if (has3) x3a = ld2(mp.a3, orow + ka);
                }
                if (qB) {
                    if (has1) x1b = ld2(mp.a1, orow + kb);
                    if (has2) x2b = ld2(mp.a2, orow + kb);
                    if (has3) x3b = ld2(mp.a3, orow + kb);
                }
            }
            issue(slot_ld, u % DEPTH);
            __syncthreads();                          // plane ii complete for everyone; slot (t-2) free
            am = ac; ac = an; bm = bc; bc = bn;
            hl_c = hl_n; hr_c = hr_n;
        }
    }
    cp_async_wait<0>();
    if (EPI == EPI_K2R) {
        if (grid_sum<NT, 2>(acc, mp.w.partials, &mp.w.st->ticket[2], sm.red) && threadIdx.x == 0)
            k2_finish(mp.w.st, mp.w, acc[0], acc[1], mp.cond, mp.use_cond);
    }
}

// ---------------------------------------------------------------------------------------------
// host-side configuration
// ---------------------------------------------------------------------------------------------
template <int TJ, int DEPTH, int MINB, bool XFIFO>
inline void stencil_pick(bool uniform, int epi, const void **func, dim3 *block, size_t *smem)
{
    if (epi == EPI_APPLY) {
        *func = uniform ? (const void *)k_stencil<TJ, DEPTH, true, MINB, EPI_APPLY, false>
                        : (const void *)k_stencil<TJ, DEPTH, false, MINB, EPI_APPLY, false>;
        *smem = sizeof(StencilSmem<TJ, DEPTH, 0>);
    } else if (epi == EPI_K2R) {
        *func = uniform ? (const void *)k_stencil<TJ, 2, true, MINB, EPI_K2R, true>
                        : (const void *)k_stencil<TJ, 2, false, MINB, EPI_K2R, true>;
        *smem = sizeof(StencilSmem<TJ, 2, 2>);
    } else {
        *func = uniform ? (const void *)k_stencil<TJ, DEPTH, true, MINB, EPI_STS, XFIFO>
                        : (const void *)k_stencil<TJ, DEPTH, false, MINB, EPI_STS, XFIFO>;
        *smem = sizeof(StencilSmem<TJ, DEPTH, XFIFO ? 6 : 0>);
    }
    *block = dim3((TJ + 2) * 32);
    cudaFuncSetAttribute(*func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)*smem);
}

// tiles and r-chunk length for a picked kernel (shared by the cp.async and the TMA variants)
inline void stencil_grid(int nr, int nt, int np, int epi, int tj, int num_sms, const void *func, dim3 block, size_t smem,
                         StencilParams *mp, dim3 *grid)
{
    mp->nkt = (np + WIDE_TK - 1) / WIDE_TK;
    mp->njt = (nt + tj - 1) / tj;
    int occ = 1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, func, (int)block.x, smem) != cudaSuccess || occ < 1) {
        cudaGetLastError();
        occ = 1;
    }
    const long long slots = (long long)num_sms * occ, cols = (long long)mp->nkt * mp->njt;
    int best = MARCH_CI_MAX;
    double best_cost = 1e300;
    for (int ci = MARCH_CI_MAX; ci >= 4; ci -= 2) {
        const long long tiles = cols * ((nr + ci - 1) / ci);
        if (epi == EPI_K2R && tiles > MAX_PARTIALS) continue;
        const double rounds = (double)((tiles + slots - 1) / slots);
        const double cost = rounds * (ci + 2 + 3);
        if (cost < best_cost * 0.999) { best_cost = cost; best = ci; }
    }
    if (nr < best) best = nr;
    mp->ci = best;
    mp->nit = (nr + best - 1) / best;
    *grid = dim3((unsigned)(mp->nkt * mp->njt * mp->nit));
}

inline int stencil_num_tiles() { return 6; }

inline void stencil_configure(int nr, int nt, int np, int uniform, int epi, int tile, int num_sms, StencilParams *mp,
                              const void **func, dim3 *grid, dim3 *block, size_t *smem)
{
    int tj;
    switch (tile) {
        case 0: tj = 6; stencil_pick<6, 2, 2, true>(uniform, epi, func, block, smem); break;
        case 1: tj = 8; stencil_pick<8, 2, 2, false>(uniform, epi, func, block, smem); break;
        case 2: tj = 14; stencil_pick<14, 2, 1, false>(uniform, epi, func, block, smem); break;
        case 3: tj = 4; stencil_pick<4, 2, 3, true>(uniform, epi, func, block, smem); break;
        case 4: tj = 8; stencil_pick<8, 2, 1, true>(uniform, epi, func, block, smem); break;
        default: tj = 8; stencil_pick<8, 3, 2, false>(uniform, epi, func, block, smem); break;
    }
    stencil_grid(nr, nt, np, epi, tj, num_sms, *func, *block, *smem, mp, grid);
}

}  // namespace mas

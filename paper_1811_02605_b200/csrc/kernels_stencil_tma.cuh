// kernels_stencil_tma.cuh -- k_stencil with the TMA engine as the loader: every tile row of a plane is ONE
// bulk copy (cp.async.bulk.shared::cluster.global, SASS UBLKCP) that signals an mbarrier with complete_tx, and
// the per-plane __syncthreads of k_stencil is replaced by a full/empty mbarrier pair per ring slot:
//   full[s]  : count NW; lane 0 of every warp arrives with expect_tx(bytes of its row: the 1 KB row segment, the two
//              16-byte phi-halo pairs, and for interior rows the epilogue's extra streams); it completes when all rows
//              of the plane have landed, which also makes them visible to every waiting thread;
//   empty[s] : count NW; a warp arrives once it no longer needs the plane in slot s (its theta-neighbours' rows were
//              read); lane 0 of a warp waits on it before refilling ITS row of slot s (planes are DEPTH+2 apart).
// Warps therefore drift by up to one plane instead of meeting at a block barrier every plane.
// Same tiling, arithmetic and epilogues (EPI_APPLY, EPI_STS) as k_stencil; selected by stencil tiles 6 and 7.
#pragma once
#include "kernels_stencil.cuh"

namespace mas {

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, unsigned parity)
{
    unsigned ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
                 : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
// bounded wait: a protocol mistake must abort the kernel, not hang the GPU
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity)
{
    for (unsigned spin = 0; !mbar_try_wait(bar, parity); ++spin)
        if (spin > (1u << 24)) __trap();
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

template <int TJ, int DEPTH, int NX>      // NX = 3 extra streams (EPI_STS) or 0
struct StencilTmaSmem {
    static constexpr int NW = TJ + 2;
    static constexpr int NT = NW * 32;
    static constexpr int R = DEPTH + 2;
    static constexpr int NPL = MARCH_CI_MAX + 2;
    alignas(16) double2 ring[R][NW][64];                 // [slot][row][128 cells]
    alignas(16) double2 halo[R][NW][2];                  // [slot][row][left pair (kl-1, kl) | right pair (kr, kr+1)]
    alignas(16) double2 xf[NX ? DEPTH : 1][NX ? NX : 1][NX ? TJ : 1][NX ? 64 : 1];   // [stage][a1 a2 a3][interior row][128 cells]
    double cE[NPL][NW], cF[NPL][NW], cAR[NPL][NW], cAT[NPL][NW], cV[NPL][NW];
    double phv[WIDE_TK + 2], phw[WIDE_TK + 2], phi[WIDE_TK + 2];
    alignas(8) uint64_t full[R], empty[R];
};

template <int TJ, int DEPTH, bool UNIFORM, int MINB, int EPI>
__global__ void __launch_bounds__((TJ + 2) * 32, MINB)
k_stencil_tma(OpDev op, StencilParams mp)
{
    static_assert(EPI == EPI_APPLY || EPI == EPI_STS, "TMA variant: apply and STS epilogues");
    using Smem = StencilTmaSmem<TJ, DEPTH, EPI == EPI_STS ? 3 : 0>;
    constexpr int NT = Smem::NT, NW = Smem::NW, R = Smem::R;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    Smem &sm = *reinterpret_cast<Smem *>(smem_raw);

    const double *__restrict__ uvec = mp.u ? mp.u : mp.args->x;
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
    const int kl = k0 == 0 ? op.np - 1 : k0 - 1;           // odd (k0 and np are even)
    const int kr = k0 + tkeff >= op.np ? 0 : k0 + tkeff;   // even

    // ---- stage coefficient columns and phi factors; zero the ring; init the barriers ----
    for (int e = tid; e < nsteps * NW; e += NT) {
        const int pl = e / NW, wr = e - pl * NW;
        const int ii = first + pl, jj = jt * TJ + wr - 1;
        const bool in = ii >= 0 && ii < op.nr && jj >= 0 && jj < op.nt;
        const int row = ii * op.nt + jj;
        sm.cE[pl][wr] = in ? __ldg(mp.E + row) : 0.0;
        sm.cF[pl][wr] = in ? __ldg(mp.F + row) : 0.0;
        sm.cV[pl][wr] = (in && EPI == EPI_STS) ? __ldg(mp.Vinv + row) : 0.0;
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
        if (lane < 2) sm.halo[s][warp][lane] = make_double2(0.0, 0.0);
    }
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < R; s++) { mbar_init(&sm.full[s], NW); mbar_init(&sm.empty[s], NW); }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");   // inits visible to the async proxy
    }
    // the zero-fill above was written through the generic proxy; the bulk copies write through the async proxy
    asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
    __syncthreads();

    const int ea = 2 * lane + 1, eb = 2 * lane + 65;
    auto VP = [&](int e) { return UNIFORM ? mp.vp : sm.phv[e]; };
    auto WP = [&](int e) { return UNIFORM ? mp.wp : sm.phw[e]; };
    auto IP = [&](int e) { return UNIFORM ? mp.ip : sm.phi[e]; };

    const long long plane = (long long)op.nt * op.np;
    const long long rowbase0 = (long long)first * plane + (row_ok ? (long long)j * op.np : 0);
    const int ka = k0 + 2 * lane, kb = ka + 64;
    long long orow = rowbase0 + plane;                      // row base of plane i0: outputs
    const bool has1 = EPI == EPI_STS && mp.a1 != nullptr, has2 = EPI == EPI_STS && mp.a2 != nullptr,
               has3 = EPI == EPI_STS && mp.a3 != nullptr;
    const unsigned rowbytes = (unsigned)tkeff * 8u;

    // lane 0 of each warp: load THIS warp's row of plane index pl (ring plane first+pl) and, for interior rows,
    // the extras of the plane whose outputs are formed when that ring plane is consumed (first+pl-1).
    auto produce = [&](int pl) {
        const int slot = pl % R, ii = first + pl;
        uint64_t *bar = &sm.full[slot];
        unsigned bytes = 0;
        const long long rb = rowbase0 + (long long)pl * plane;
        const bool plane_in = (unsigned)ii < (unsigned)op.nr;
        if (row_ok && plane_in) bytes += rowbytes + (interior ? 32u : 0u);
        const bool xin = EPI == EPI_STS && interior && row_ok && (ii - 1 >= i0) && (ii - 1 < i1);
        if (xin) bytes += rowbytes * ((has1 ? 1u : 0u) + (has2 ? 1u : 0u) + (has3 ? 1u : 0u));
        if (bytes == 0) { mbar_arrive(bar); return; }
        mbar_arrive_expect_tx(bar, bytes);
        if (row_ok && plane_in) {
            bulk_g2s(&sm.ring[slot][warp][0], uvec + rb + k0, rowbytes, bar);
            if (interior) {
                bulk_g2s(&sm.halo[slot][warp][0], uvec + rb + (kl - 1), 16u, bar);
                bulk_g2s(&sm.halo[slot][warp][1], uvec + rb + kr, 16u, bar);
            }
        }
        if (xin) {
            const int xs = pl % DEPTH;
            const long long xb = rb - plane + k0;
            if (has1) bulk_g2s(&sm.xf[xs][0][warp - 1][0], mp.a1 + xb, rowbytes, bar);
            if (has2) bulk_g2s(&sm.xf[xs][1][warp - 1][0], mp.a2 + xb, rowbytes, bar);
            if (has3) bulk_g2s(&sm.xf[xs][2][warp - 1][0], mp.a3 + xb, rowbytes, bar);
        }
    };
    if (lane == 0)
        for (int pl = 0; pl < DEPTH && pl < nsteps; pl++) produce(pl);

    const double2 zero2 = make_double2(0.0, 0.0);
    double2 am = zero2, ac = zero2, bm = zero2, bc = zero2;
    double hl_c = 0.0, hr_c = 0.0;
    const int lm = (lane + 31) & 31, lp = (lane + 1) & 31;

    for (int t = 0; t < nsteps; t++) {
        const int slot = t % R, slot_prev = (t + R - 1) % R;
        const int ii = first + t;
        const bool plane_ok = (unsigned)ii < (unsigned)op.nr;
        mbar_wait(&sm.full[slot], (unsigned)(t / R) & 1u);          // plane ii: every row has landed
        double2 an = zero2, bn = zero2;
        double hl_n = 0.0, hr_n = 0.0;
        if (plane_ok) {
            an = sm.ring[slot][warp][lane];
            bn = sm.ring[slot][warp][lane + 32];
            if (left_edge) hl_n = sm.halo[slot][warp][0].y;
            if (right_edge) hr_n = sm.halo[slot][warp][1].x;
        }
        const double mA = __shfl_sync(0xffffffffu, ac.y, lm), mB = __shfl_sync(0xffffffffu, bc.y, lm);
        const double pA = __shfl_sync(0xffffffffu, ac.x, lp), pB = __shfl_sync(0xffffffffu, bc.x, lp);
        if (t >= 2 && interior && row_ok) {
            const double Ec = sm.cE[t - 1][warp], Fc = sm.cF[t - 1][warp];
            const double ARm = sm.cAR[t - 1][warp], ARp = sm.cAR[t][warp];
            const double ATm = sm.cAT[t - 1][warp], ATp = sm.cAT[t - 1][warp + 1];
            const double vinv = EPI == EPI_STS ? sm.cV[t - 1][warp] : 0.0;
            const int xs = t % DEPTH;
            auto finish = [&](double2 s, double2 uc, int half, int e, int kcell) {
                double2 o;
                if (EPI == EPI_APPLY) {
                    o = s;
                } else {
                    double2 mu;
                    mu.x = UNIFORM ? -(s.x * vinv) * (1.0 / mp.vp) : -(s.x * vinv) / VP(e);
                    mu.y = UNIFORM ? -(s.y * vinv) * (1.0 / mp.vp) : -(s.y * vinv) / VP(e + 1);
                    if (mp.out2) st2(mp.out2, orow + kcell, mu);
                    o.x = mp.c_u * uc.x + mp.c_L * mu.x;
                    o.y = mp.c_u * uc.y + mp.c_L * mu.y;
                    const int xi = lane + 32 * half;
                    if (has1) { const double2 x1 = sm.xf[xs][0][warp - 1][xi]; o.x = fma(mp.c_a1, x1.x, o.x); o.y = fma(mp.c_a1, x1.y, o.y); }
                    if (has2) { const double2 x2 = sm.xf[xs][1][warp - 1][xi]; o.x = fma(mp.c_a2, x2.x, o.x); o.y = fma(mp.c_a2, x2.y, o.y); }
                    if (has3) { const double2 x3 = sm.xf[xs][2][warp - 1][xi]; o.x = fma(mp.c_a3, x3.x, o.x); o.y = fma(mp.c_a3, x3.y, o.y); }
                }
                st2(mp.out, orow + kcell, o);
            };
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
                finish(s, ac, 0, ea, ka);
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
                finish(s, bc, 1, eb, kb);
            }
        }
        if (t >= 2) orow += plane;
        __syncwarp();                                       // the warp's reads of slot_prev and of its extras are done
        if (lane == 0) {
            if (t >= 1) mbar_arrive(&sm.empty[slot_prev]);  // plane t-1 released by this warp
            const int pl = t + DEPTH;                       // refill: plane pl goes to the slot plane pl-R used
            if (pl < nsteps) {
                const int use = pl / R;                     // n-th use of that slot
                if (use >= 1) mbar_wait(&sm.empty[pl % R], (unsigned)(use - 1) & 1u);
                produce(pl);
            }
        }
        am = ac; ac = an; bm = bc; bc = bn;
        hl_c = hl_n; hr_c = hr_n;
    }
}

template <int TJ, int DEPTH, int MINB>
inline void stencil_tma_pick(bool uniform, int epi, const void **func, dim3 *block, size_t *smem)
{
    if (epi == EPI_APPLY) {
        *func = uniform ? (const void *)k_stencil_tma<TJ, DEPTH, true, MINB, EPI_APPLY>
                        : (const void *)k_stencil_tma<TJ, DEPTH, false, MINB, EPI_APPLY>;
        *smem = sizeof(StencilTmaSmem<TJ, DEPTH, 0>);
    } else {
        *func = uniform ? (const void *)k_stencil_tma<TJ, DEPTH, true, MINB, EPI_STS>
                        : (const void *)k_stencil_tma<TJ, DEPTH, false, MINB, EPI_STS>;
        *smem = sizeof(StencilTmaSmem<TJ, DEPTH, 3>);
    }
    *block = dim3((TJ + 2) * 32);
    cudaFuncSetAttribute(*func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)*smem);
}

// every stencil tile id: 0..5 = k_stencil (cp.async), 6..11 = k_stencil_tma (bulk copies + mbarriers)
inline int stencil_num_tiles_any() { return stencil_num_tiles() + 6; }

inline void stencil_configure_any(int nr, int nt, int np, int uniform, int epi, int tile, int num_sms, StencilParams *mp,
                                  const void **func, dim3 *grid, dim3 *block, size_t *smem)
{
    if (tile < stencil_num_tiles() || epi == EPI_K2R) {
        stencil_configure(nr, nt, np, uniform, epi, tile < stencil_num_tiles() ? tile : 1, num_sms, mp, func, grid, block,
                          smem);
        return;
    }
    int tj;
    switch (tile - stencil_num_tiles()) {
        case 0: tj = 6; stencil_tma_pick<6, 2, 2>(uniform, epi, func, block, smem); break;
        case 1: tj = 8; stencil_tma_pick<8, 2, 2>(uniform, epi, func, block, smem); break;
        case 2: tj = 14; stencil_tma_pick<14, 2, 1>(uniform, epi, func, block, smem); break;
        case 3: tj = 10; stencil_tma_pick<10, 2, 1>(uniform, epi, func, block, smem); break;
        case 4: tj = 8; stencil_tma_pick<8, 3, 1>(uniform, epi, func, block, smem); break;
        default: tj = 12; stencil_tma_pick<12, 3, 1>(uniform, epi, func, block, smem); break;
    }
    stencil_grid(nr, nt, np, epi, tj, num_sms, *func, *block, *smem, mp, grid);
}

}  // namespace mas

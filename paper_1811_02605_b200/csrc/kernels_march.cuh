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
//   * the phi-halo cells (k0-1, k0+64; periodic wrap) are two scalar loads by the edge lanes.
// Each cell's r and p_old are read from DRAM once; halo rows/planes are L2 hits.
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

}  // namespace mas

// kernels_k1_tma.cuh -- K1, the fused matrix-free matvec of the PCG iteration (SURVEY.md 8(a) S2 + S3;
// PAPER.md:98 "sparse matrix-vector products (essentially stencil operations)"), as a 2.5-D marching-tile
// kernel for sm_100a with the TMA engine as the loader and mbarriers instead of block barriers:
//
//     x    += alpha_{k-1} p_old       (the x-update of the PREVIOUS iteration, deferred into this pass: "xfuse")
//     p_new = r/d + beta p_old        (the p-update of the previous iteration, fused as a prologue; with PC2 the
//                                      preconditioned residual z is read from memory in place of r/d)
//     q     = A_sym p_new             (7-point, matrix-free, coefficients from 2-D planes)   [not stored when NOQ]
//     sigma = p_new . q               (deterministic two-stage reduction; last block: alpha = rho / sigma)
//
// Tiling: tile.cuh.  Data movement per step (= one r plane):
//   * every warp owns one tile row; lane 0 bulk-copies (cp.async.bulk, SASS UBLKCP) that row's r, p_old, x segments
//     for the plane DEPTH steps ahead into the warp's own FIFO stage -- r and p_old with their two phi-halo pairs,
//     ONE copy per vector when the halo cells are adjacent in memory (tile.cuh row_copy) -- signalling the warp's
//     own mbarrier ldfull[stage][warp] (count 1 + transaction bytes).  A warp waits only for ITS row -- there is no
//     block-wide coupling on the load path; source addresses are running offsets bumped by one plane per step;
//   * p_new planes go to a shared ring of FOUR planes; every thread arrives on ringfull[plane % 4] after storing its
//     part, and a warp waits for plane t-1 to be complete before reading its theta-neighbours' rows.  With four
//     buffers that wait also proves the slot written at step t (plane t-4) is no longer being read, so K1 has no
//     __syncthreads in its loop: warps drift by up to a plane instead of meeting at a barrier every plane;
//   * phi neighbours come by warp shuffle, r neighbours stay in registers across steps.
// Each cell's r, p_old, x are read from DRAM once; halo rows / planes are L2 hits.
// p is double-buffered in global memory (p[k&1] -> p[(k+1)&1]) because neighbouring blocks read p_old halos while
// this block writes p_new.
// NOQ = the 64 B/cell/iteration form of the iteration: q is not stored; K2R (k_stencil_tma<EPI_K2R>) recomputes it
// from p_new.  K1 then moves 5 doubles per cell instead of 6.
#pragma once
#include "kernels_base.cuh"
#include "tile.cuh"

namespace mas {

template <int TJ, int DEPTH, bool UNIFORM>
struct K1TmaSmem {
    static constexpr int NW = TJ + 2;
    static constexpr int NT = NW * 32;
    alignas(16) double2 fr[DEPTH][NW][ROW_V2];            // r rows (tile + theta-halo rows): [halo pair | 128 cells | halo pair]
    alignas(16) double2 fp[DEPTH][NW][ROW_V2];            // p_old rows, same layout
    alignas(16) double2 fx[DEPTH][TJ][64];                // x rows (interior rows only)
    alignas(16) double2 ring[4][NW][64];                  // p_new planes
    TileCoefs<NW, UNIFORM> c;
    double red[32];
    alignas(8) uint64_t ldfull[DEPTH][NW];
    alignas(8) uint64_t ringfull[4];
};

template <int TJ, int DEPTH, bool UNIFORM, int MINB, bool NOQ>
__global__ void __launch_bounds__((TJ + 2) * 32, MINB)
k1_tma(OpDev op, Work w, TileParams mp, cudaGraphConditionalHandle cond, int use_cond)
{
    using Smem = K1TmaSmem<TJ, DEPTH, UNIFORM>;
    constexpr int NT = Smem::NT, NW = Smem::NW;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    Smem &sm = *reinterpret_cast<Smem *>(smem_raw);

    const int rhs = blockIdx.y;
    const TileGeom g = tile_geom<TJ>(op, mp);
    const int lane = g.lane, warp = g.warp, tid = g.tid;

    // 32-bit shared addresses of this warp's barriers and staging rows (stage 0), computed once
    const unsigned s_ldfull = smem_u32(&sm.ldfull[0][warp]), s_ring = smem_u32(&sm.ringfull[0]);
    const unsigned s_fr = smem_u32(&sm.fr[0][warp][0]), s_fp = smem_u32(&sm.fp[0][warp][0]);
    const unsigned s_fx = smem_u32(&sm.fx[0][g.interior ? warp - 1 : 0][0]);
    constexpr unsigned BAR_STAGE = NW * 8u, ROWS_STAGE = NW * ROW_BYTES, X_STAGE = TJ * 1024u;

    // ---- zero-fill and barrier init first, so that the first bulk copies can be issued as early as possible ----
    const double2 zero2 = make_double2(0.0, 0.0);
#pragma unroll
    for (int s = 0; s < DEPTH; s++) {
        for (int e = lane; e < ROW_V2; e += 32) { sm.fr[s][warp][e] = zero2; sm.fp[s][warp][e] = zero2; }
        if (g.interior) { sm.fx[s][warp - 1][lane] = zero2; sm.fx[s][warp - 1][lane + 32] = zero2; }
    }
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < DEPTH; s++)
            for (int r = 0; r < NW; r++) mbar_init(smem_u32(&sm.ldfull[s][r]), 1);
#pragma unroll
        for (int s = 0; s < 4; s++) mbar_init(s_ring + 8u * s, NT);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
    __syncthreads();

    State *st = w.st + rhs;
    if (!st->active) return;
    const double beta = st->beta;
    const int par = st->k & 1;
    const long long voff = rhs * w.vstride;
    const VecHalo pV = {(par ? w.p1 : w.p0) + voff, par ? w.lo_p1 : w.lo_p0, par ? w.hi_p1 : w.hi_p0};
    const bool zin = mp.zin != 0;               // PC2: "r" below is z = M^-1 r, already preconditioned
    const VecHalo rV = zin ? VecHalo{w.z + voff, w.lo_z, w.hi_z} : VecHalo{w.r + voff, w.lo_r, w.hi_r};
    double *__restrict__ pout = (par ? w.p0 : w.p1) + voff;
    double *__restrict__ qout = w.q + voff;
    const double alpha_prev = st->alpha;        // x += alpha_{k-1} p_{k-1}: the deferred x-update (xfuse)
    double *__restrict__ xvec = w.args->x[rhs];
    int *fault = &w.ctl->fault;

    const PhiFac<UNIFORM, TileCoefs<NW, UNIFORM>> ph = {sm.c, mp.vp, mp.wp, mp.ip};
    const int ea = 2 * lane + 1, eb = 2 * lane + 65;
    auto zval = [&](double r, double E, double F, double dinv, int e) {
        return zin ? r : (UNIFORM ? r * dinv : r * rcp_nr(fma(ph.VP(e), E, F * ph.WP(e))));
    };

    auto zval2 = [&](double2 r, double E, double F, double dinv, int e) {       // the two cells (e, e + 1) of a vector
        if (zin) return r;
        if (UNIFORM) return make_double2(r.x * dinv, r.y * dinv);
        const double2 v = ph.VP2(e), wv = ph.WP2(e);
        return make_double2(r.x * rcp_nr(fma(v.x, E, F * wv.x)), r.y * rcp_nr(fma(v.y, E, F * wv.y)));
    };

    const long long plane = (long long)op.nt * op.np;
    const long long rowoff = g.row_ok ? (long long)g.j * op.np : 0;
    const long long rowbase0 = (long long)g.first * plane + rowoff;
    long long prow = rowbase0 + plane;           // row base of plane i0: p_new / x stores
    long long qrow = rowbase0 + plane;           // row base of plane i0: q stores
    const unsigned rowbytes = (unsigned)g.tkeff * 8u;
    const bool fx = mp.l2.first_x != 0;
    const uint64_t pol_first = fx ? l2_policy_evict_first() : 0;

    // lane 0: this warp's row of plane index pl -> FIFO stage `stage`.  `src` is the running offset (cell k0 of this
    // warp's row in plane first + pl of the own vectors), bumped by one plane per call: no multiplications here.
    long long src = rowbase0 + g.k0;
    const unsigned tx_rows = 2u * (rowbytes + 32u);
    auto produce = [&](int pl, int stage) {
        const unsigned bar = s_ldfull + BAR_STAGE * stage;
        const int ii = g.first + pl;
        const double *rrow, *prw;
        if (ii >= 0 && ii < op.nr) { rrow = rV.own + src; prw = pV.own + src; }
        else {                                                  // the adjacent plane of a neighbour slab, or nothing
            const double *rh = ii < 0 ? rV.lo : rV.hi, *phh = ii < 0 ? pV.lo : pV.hi;
            rrow = rh ? rh + rowoff + g.k0 : nullptr;
            prw = phh ? phh + rowoff + g.k0 : nullptr;
        }
        const bool xin = g.interior && pl >= 1 && pl <= g.nsteps - 2;
        const long long xoff = src;
        src += plane;
        if (!g.row_ok || !rrow) { mbar_arrive(bar); return; }
        mbar_arrive_expect_tx(bar, xin ? tx_rows + rowbytes : tx_rows);
        row_copy(s_fr + ROWS_STAGE * stage, rrow, g, op.np, rowbytes, bar);
        row_copy(s_fp + ROWS_STAGE * stage, prw, g, op.np, rowbytes, bar);
        if (xin) {
            if (fx) bulk_g2s_hint(s_fx + X_STAGE * stage, xvec + xoff, rowbytes, bar, pol_first);
            else bulk_g2s(s_fx + X_STAGE * stage, xvec + xoff, rowbytes, bar);
        }
    };
    if (lane == 0)
        for (int pl = 0; pl < DEPTH && pl < g.nsteps; pl++) produce(pl, pl);

    // ---- coefficient columns and phi factors, staged while the first planes are already in flight ----
    const PlaneSetDev ps = {op.E, op.F, op.AR, op.AT, op.Dinv};
    stage_coefs<TJ, UNIFORM>(sm.c, g, op, ps, mp.vp, mp.wp, mp.ip);
    __syncthreads();                            // coefficient columns visible

    double2 am = zero2, ac = zero2, bm = zero2, bc = zero2;
    double hl_c = 0.0, hr_c = 0.0;
    double acc = 0.0;

    // One step = one plane.  `uc` is the ring slot t % 4: a compile-time constant in the unrolled trips (run_trip), a
    // run-time value in the tail; with it (when DEPTH divides 4) the FIFO stage is compile-time too.
    auto step = [&](const int t, const int, auto uc) {
        const int u = uc;
        const int rs = u, rsp = (u + 3) & 3;
        const int stage = (4 % DEPTH == 0) ? u % DEPTH : t % DEPTH;
        const int ii = g.first + t;
        const bool plane_ok = (unsigned)(op.i_lo + ii) < (unsigned)op.nr_glob;
        const bool own = t >= 1 && t <= g.nsteps - 2;       // a plane of this block: p_new and x are stored
        const double En = sm.c.cE[t][warp], Fn = sm.c.cF[t][warp], dinv = sm.c.cD[t][warp];
        mbar_wait(s_ldfull + BAR_STAGE * stage, (unsigned)(t / DEPTH) & 1u, fault);   // this warp's row of plane ii
        double2 an = zero2, bn = zero2;
        double hl_n = 0.0, hr_n = 0.0;
        if (plane_ok) {
            const double2 *fr = sm.fr[stage][warp], *fp = sm.fp[stage][warp];
            const double2 ra = fr[1 + lane], rb = fr[33 + lane];
            const double2 pa = fp[1 + lane], pb = fp[33 + lane];
            if (UNIFORM || g.vA) {
                const double2 z = zval2(ra, En, Fn, dinv, ea);
                an.x = fma(beta, pa.x, z.x);
                an.y = fma(beta, pa.y, z.y);
            }
            if (UNIFORM || g.vB) {
                const double2 z = zval2(rb, En, Fn, dinv, eb);
                bn.x = fma(beta, pb.x, z.x);
                bn.y = fma(beta, pb.y, z.y);
            }
            if (g.left_edge) hl_n = fma(beta, fp[0].y, zval(fr[0].y, En, Fn, dinv, 0));
            if (g.right_edge) hr_n = fma(beta, fp[g.hr].x, zval(fr[g.hr].x, En, Fn, dinv, g.tkeff + 1));
            if (own) {                          // store p_new and the deferred x-update
                if (g.qA) {
                    st2g(pout, prow + g.ka, an);
                    double2 xa = sm.fx[stage][warp - 1][lane];
                    xa.x = fma(alpha_prev, pa.x, xa.x); xa.y = fma(alpha_prev, pa.y, xa.y);
                    if (fx) st2_hint(xvec, prow + g.ka, xa, pol_first); else st2g(xvec, prow + g.ka, xa);
                }
                if (g.qB) {
                    st2g(pout, prow + g.kb, bn);
                    double2 xb = sm.fx[stage][warp - 1][lane + 32];
                    xb.x = fma(alpha_prev, pb.x, xb.x); xb.y = fma(alpha_prev, pb.y, xb.y);
                    if (fx) st2_hint(xvec, prow + g.kb, xb, pol_first); else st2g(xvec, prow + g.kb, xb);
                }
            }
        }
        if (own) prow += plane;
        __syncwarp();                                        // the warp is done with its FIFO stage
        if (lane == 0 && t + DEPTH < g.nsteps) produce(t + DEPTH, stage);
        // ---- publish p_new of plane ii; wait for plane ii-1 of the whole tile ----
        sm.ring[rs][warp][lane] = an;
        sm.ring[rs][warp][lane + 32] = bn;
        mbar_arrive(s_ring + 8u * rs);                       // every thread: its own stores are released
        const PhiNb nb = phi_neighbours(ac, bc, lane);
        if (t >= 1) mbar_wait(s_ring + 8u * rsp, (unsigned)((t - 1) >> 2) & 1u, fault);
        // ---- q for plane i = ii-1 ----
        if (t >= 2 && g.interior && g.row_ok) {
            const RowCoefs rc = row_coefs(sm.c, t, warp);
            if (g.qA) {
                const double ukm = g.left_edge ? hl_c : nb.mA;
                const double ukp = g.right_A ? hr_c : (lane == 31 ? nb.pB : nb.pA);
                const double2 q = stencil_half(ph, ea, rc, am, ac, an, sm.ring[rsp][warp - 1][lane],
                                               sm.ring[rsp][warp + 1][lane], ukm, ukp);
                if (!NOQ) st2g(qout, qrow + g.ka, q);
                acc += ac.x * q.x + ac.y * q.y;
            }
            if (g.qB) {
                const double ukm = lane == 0 ? nb.mA : nb.mB;
                const double ukp = g.right_B ? hr_c : nb.pB;
                const double2 q = stencil_half(ph, eb, rc, bm, bc, bn, sm.ring[rsp][warp - 1][lane + 32],
                                               sm.ring[rsp][warp + 1][lane + 32], ukm, ukp);
                if (!NOQ) st2g(qout, qrow + g.kb, q);
                acc += bc.x * q.x + bc.y * q.y;
            }
        }
        if (t >= 2) qrow += plane;
        am = ac; ac = an; bm = bc; bc = bn;
        hl_c = hl_n; hr_c = hr_n;
    };
    int t0 = 0;
    for (; t0 + 4 <= g.nsteps; t0 += 4) run_trip(step, t0, 0, std::make_integer_sequence<int, 4>{});
    for (int t = t0; t < g.nsteps; t++) step(t, 0, t - t0);
    double a1[1] = {acc};
    if (grid_sum<NT, 1>(a1, part_base(w, rhs), w.pstride, &w.tickets[rhs * 4 + 1], sm.red) && threadIdx.x == 0)
        reduction_done<ROLE_K1, 1>(w, rhs, a1, cond, use_cond);
}

// ---- host-side configuration ----
struct K1TmaTile {
    int tj, depth, minb;
};
static const K1TmaTile kK1TmaTiles[] = {{14, 2, 1}, {8, 2, 2}, {6, 2, 2}, {8, 3, 1}, {10, 2, 1}, {16, 2, 1}, {12, 2, 1}};
inline int k1_tma_num_tiles() { return (int)(sizeof(kK1TmaTiles) / sizeof(kK1TmaTiles[0])); }

// Automatic tile: the 14-row tile with one 512-thread block per SM is the fastest when the mesh gives every SM several
// blocks in turn (configs 4, 5); when all of its tiles fit in ONE round (mid-size meshes such as config 3: 140 blocks on
// 148 SMs) nothing overlaps a block's start-up and reduction tail, and the 6-row tile with two blocks per SM is faster
// (measured on config 3: 0.0591 vs 0.0619 ms).
// Non-uniform phi (round 3): the general kernel issues ~30 % more instructions per cell and is latency- rather than
// DRAM-bound, so the 16-row tile (18 warps per block at 96 registers instead of 16 at 120) wins on multi-round meshes:
// 256x256x512 with +-30 % widths, K1 per tile id 0..6 = 0.2992, 0.4209, 0.3397, 0.3635, 0.3207, 0.2863, 0.3040 ms
// (profiles/r3_k1_tile_sweep_nonuniform.md).
inline int k1_auto_tile(int nr, int nt, int np, int num_sms, bool uniform_phi)
{
    const long long cols = (long long)((np + TILE_TK - 1) / TILE_TK) * ((nt + 13) / 14);
    const int ci = tile_pick_ci(nr, cols, num_sms, 0);
    if (cols * ((nr + ci - 1) / ci) <= num_sms) return 2;
    return uniform_phi ? 0 : 5;
}

template <int TJ, int DEPTH, int MINB>
inline void k1_tma_pick(bool uniform, bool noq, const void **func, dim3 *block, size_t *smem)
{
    if (noq)
        *func = uniform ? (const void *)k1_tma<TJ, DEPTH, true, MINB, true> : (const void *)k1_tma<TJ, DEPTH, false, MINB, true>;
    else
        *func = uniform ? (const void *)k1_tma<TJ, DEPTH, true, MINB, false> : (const void *)k1_tma<TJ, DEPTH, false, MINB, false>;
    *smem = uniform ? sizeof(K1TmaSmem<TJ, DEPTH, true>) : sizeof(K1TmaSmem<TJ, DEPTH, false>);
    *block = dim3((TJ + 2) * 32);
    cudaFuncSetAttribute(*func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)*smem);
}

inline void k1_tma_configure(int nr, int nt, int np, int uniform, bool noq, int tile, int num_sms, int ci_force, int ny,
                             TileParams *mp, const void **func, dim3 *grid, dim3 *block, size_t *smem)
{
    const K1TmaTile T = kK1TmaTiles[tile];
    switch (tile) {
        case 0: k1_tma_pick<14, 2, 1>(uniform, noq, func, block, smem); break;
        case 1: k1_tma_pick<8, 2, 2>(uniform, noq, func, block, smem); break;
        case 2: k1_tma_pick<6, 2, 2>(uniform, noq, func, block, smem); break;
        case 3: k1_tma_pick<8, 3, 1>(uniform, noq, func, block, smem); break;
        case 4: k1_tma_pick<10, 2, 1>(uniform, noq, func, block, smem); break;
        case 5: k1_tma_pick<16, 2, 1>(uniform, noq, func, block, smem); break;
        default: k1_tma_pick<12, 2, 1>(uniform, noq, func, block, smem); break;
    }
    mp->nkt = (np + TILE_TK - 1) / TILE_TK;
    mp->njt = (nt + T.tj - 1) / T.tj;
    int occ = 1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, *func, (int)block->x, *smem) != cudaSuccess || occ < 1) {
        cudaGetLastError();
        occ = 1;
    }
    mp->ci = tile_pick_ci(nr, (long long)mp->nkt * mp->njt, (long long)num_sms * occ, ci_force);
    mp->nit = (nr + mp->ci - 1) / mp->ci;
    *grid = dim3((unsigned)(mp->nkt * mp->njt * mp->nit), (unsigned)ny);
}

}  // namespace mas

// kernels_stencil_tma.cuh -- the matrix-free 7-point stencil applied to a STORED vector, as a 2.5-D marching kernel
// (tiling: tile.cuh) with a fused epilogue.  Used by
//   * mas_pcg_apply and the initial residual (EPI_APPLY:  out = S u,  S = A_sym with the dt-scaled planes),
//   * the RKL2 super-time-stepping stages of NEXT-1 (EPI_STS: S = L_sym from the dt-independent planes,
//     M u = -S u / V,  out = c_u u + c_a1 a1 + c_a2 a2 + c_L M u + c_a3 a3,  optionally out2 = M u)
//     -- PAPER.md:65 "Runge-Kutta Legendre super time-stepping (STS) scheme [21]", "explicit
//     finite difference algorithms (such as ... the STS algorithm)",
//   * K2R, the fused vector kernel of the 64 B/cell/iteration PCG (EPI_K2R: u = p written by K1 of this iteration,
//     q = A_sym p recomputed instead of read, r -= alpha q in place, rho' = r.z, rr = r.r, then the scalar step S5).
// The TMA engine is the loader: every tile row of a plane is ONE bulk copy (cp.async.bulk.shared::cluster.global,
// SASS UBLKCP) that signals an mbarrier with complete_tx; a full/empty mbarrier pair per ring slot replaces the
// per-plane block barrier:
//   full[s]  : count NW; lane 0 of every warp arrives with expect_tx(bytes of its row: the 1 KB row segment, the two
//              16-byte phi-halo pairs, and for interior rows the epilogue's extra streams); it completes when all rows
//              of the plane have landed, which also makes them visible to every waiting thread;
//   empty[s] : count NW; a warp arrives once it no longer needs the plane in slot s (its theta-neighbours' rows were
//              read); lane 0 of a warp waits on it before refilling ITS row of slot s (planes are DEPTH+2 apart).
// Warps therefore drift by up to one plane instead of meeting at a block barrier every plane.
#pragma once
#include "kernels_base.cuh"
#include "tile.cuh"

namespace mas {

enum { EPI_APPLY = 0, EPI_STS = 1, EPI_K2R = 2 };

struct StencilParams {
    TileParams t;
    PlaneSetDev ps;                       // plane set: A_sym (dt-scaled) or L_sym (base); ps.D = Vinv (STS) / Dinv (K2R)
    const double *u, *u_lo, *u_hi;        // the vector the stencil is applied to (null: args->x[rhs]) and its slab halos
    long long ustride;                    // right-hand side j of u / out at + j * ustride
    const SolveArgs *args;
    double *out, *out2;
    const double *a1, *a2, *a3;           // EPI_STS: Y_{j-2}, Y_0, M Y_0 (null = absent)
    double c_u, c_a1, c_a2, c_L, c_a3;
    int *fault;
    // EPI_K2R
    Work w;
    cudaGraphConditionalHandle cond;
    int use_cond;
};

template <int TJ, int DEPTH, int NX, bool UNIFORM>      // NX extra streams: 3 (EPI_STS), 1 (EPI_K2R: r), 0
struct StencilTmaSmem {
    static constexpr int NW = TJ + 2;
    static constexpr int NT = NW * 32;
    static constexpr int R = DEPTH + 2;
    alignas(16) double2 ring[R][NW][ROW_V2];             // [slot][row][left halo pair | 128 cells | right halo pair]
    alignas(16) double2 xf[NX ? DEPTH : 1][NX ? NX : 1][NX ? TJ : 1][NX ? 64 : 1];   // [stage][stream][interior row][128 cells]
    TileCoefs<NW, UNIFORM> c;
    double red[32];
    alignas(8) uint64_t full[R], empty[R];
};

template <int TJ, int DEPTH, bool UNIFORM, int MINB, int EPI>
__global__ void __launch_bounds__((TJ + 2) * 32, MINB)
k_stencil_tma(OpDev op, StencilParams mp)
{
    constexpr int NX = EPI == EPI_STS ? 3 : (EPI == EPI_K2R ? 1 : 0);
    using Smem = StencilTmaSmem<TJ, DEPTH, NX, UNIFORM>;
    constexpr int NT = Smem::NT, NW = Smem::NW, R = Smem::R;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    Smem &sm = *reinterpret_cast<Smem *>(smem_raw);

    const int rhs = blockIdx.y;
    const TileGeom g = tile_geom<TJ>(op, mp.t);
    const int lane = g.lane, warp = g.warp, tid = g.tid;

    // ---- which vectors ----
    double alpha = 0.0;
    VecHalo uV;
    double *rvec = nullptr;
    if (EPI == EPI_K2R) {                            // u = p written by K1 of this iteration; r updated in place
        const State *st = mp.w.st + rhs;
        if (!st->active) {                           // this right-hand side is done: report, nothing else
            if (blockIdx.x == 0 && tid == 0 && !mp.w.slab_sums) loop_vote(mp.w, 0, gridDim.y, mp.cond, mp.use_cond);
            return;
        }
        alpha = st->alpha;
        const int par = st->k & 1;                   // K1 wrote p[(k+1)&1]
        const long long voff = rhs * mp.w.vstride;
        uV.own = (par ? mp.w.p0 : mp.w.p1) + voff;
        uV.lo = par ? mp.w.lo_p0 : mp.w.lo_p1;
        uV.hi = par ? mp.w.hi_p0 : mp.w.hi_p1;
        rvec = mp.w.r + voff;
    } else {
        if (mp.u) { uV.own = mp.u + rhs * mp.ustride; uV.lo = mp.u_lo; uV.hi = mp.u_hi; }
        else { uV.own = mp.args->x[rhs]; uV.lo = mp.args->x_lo; uV.hi = mp.args->x_hi; }
    }
    double *out = EPI == EPI_K2R ? rvec : mp.out + rhs * mp.ustride;
    const double *x1p = EPI == EPI_K2R ? rvec : mp.a1;           // K2R: the one extra stream is r
    int *fault = mp.fault;

    // 32-bit shared addresses of the barriers and of this warp's rows (slot / stage 0), computed once
    const unsigned s_full = smem_u32(&sm.full[0]), s_empty = smem_u32(&sm.empty[0]);
    const unsigned s_ring = smem_u32(&sm.ring[0][warp][0]);
    const unsigned s_xf = smem_u32(&sm.xf[0][0][NX && g.interior ? warp - 1 : 0][0]);
    constexpr unsigned SLOT_BYTES = NW * ROW_BYTES, XSTREAM = (NX ? TJ : 1) * 1024u, XSTAGE = (NX ? NX : 1) * XSTREAM;

    // ---- zero the ring, init the barriers, start the first planes, then stage the coefficient columns ----
#pragma unroll
    for (int s = 0; s < R; s++)
        for (int e = lane; e < ROW_V2; e += 32) sm.ring[s][warp][e] = make_double2(0.0, 0.0);
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < R; s++) { mbar_init(s_full + 8u * s, NW); mbar_init(s_empty + 8u * s, NW); }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");   // inits visible to the async proxy
    }
    // the zero-fill above was written through the generic proxy; the bulk copies write through the async proxy
    asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
    __syncthreads();

    const PhiFac<UNIFORM, TileCoefs<NW, UNIFORM>> ph = {sm.c, mp.t.vp, mp.t.wp, mp.t.ip};
    const int ea = 2 * lane + 1, eb = 2 * lane + 65;
    const long long plane = (long long)op.nt * op.np;
    const long long rowoff = g.row_ok ? (long long)g.j * op.np : 0;
    const long long rowbase0 = (long long)g.first * plane + rowoff;
    long long orow = rowbase0 + plane;                      // row base of plane i0: outputs
    const bool has1 = (EPI == EPI_STS && mp.a1 != nullptr) || EPI == EPI_K2R,
               has2 = EPI == EPI_STS && mp.a2 != nullptr, has3 = EPI == EPI_STS && mp.a3 != nullptr;
    const unsigned rowbytes = (unsigned)g.tkeff * 8u;
    const unsigned tx_u = rowbytes + 32u;
    const unsigned tx_x = rowbytes * ((has1 ? 1u : 0u) + (has2 ? 1u : 0u) + (has3 ? 1u : 0u));

    // lane 0 of each warp: load THIS warp's row of plane index pl (ring plane first+pl) into `slot` and, for interior
    // rows, the extras of the plane whose outputs are formed when that ring plane is consumed (first+pl-1) into
    // `xs`.  `src` = running offset of cell k0 of this warp's row in plane first + pl (bumped by a plane per call).
    long long src = rowbase0 + g.k0;
    auto produce = [&](int pl, int slot, int xs) {
        const unsigned bar = s_full + 8u * slot;
        const int ii = g.first + pl;
        const double *urow;
        if (ii >= 0 && ii < op.nr) urow = uV.own + src;
        else { const double *h = ii < 0 ? uV.lo : uV.hi; urow = h ? h + rowoff + g.k0 : nullptr; }
        const long long xoff = src - plane;
        src += plane;
        if (!g.row_ok) urow = nullptr;
        const bool xin = NX > 0 && g.interior && g.row_ok && pl >= 2 && pl <= g.nsteps - 1 && tx_x != 0;
        const unsigned bytes = (urow ? tx_u : 0u) + (xin ? tx_x : 0u);
        if (bytes == 0) { mbar_arrive(bar); return; }
        mbar_arrive_expect_tx(bar, bytes);
        if (urow) row_copy(s_ring + SLOT_BYTES * slot, urow, g, op.np, rowbytes, bar);
        if (xin) {
            const unsigned dst = s_xf + XSTAGE * xs;
            if (has1) bulk_g2s(dst, x1p + xoff, rowbytes, bar);
            if (has2) bulk_g2s(dst + (NX > 1 ? XSTREAM : 0u), mp.a2 + xoff, rowbytes, bar);
            if (has3) bulk_g2s(dst + (NX > 2 ? 2u * XSTREAM : 0u), mp.a3 + xoff, rowbytes, bar);
        }
    };
    if (lane == 0)
        for (int pl = 0; pl < DEPTH && pl < g.nsteps; pl++) produce(pl, pl, pl);

    stage_coefs<TJ, UNIFORM>(sm.c, g, op, mp.ps, mp.t.vp, mp.t.wp, mp.t.ip);
    __syncthreads();                                        // coefficient columns visible

    const double2 zero2 = make_double2(0.0, 0.0);
    double2 am = zero2, ac = zero2, bm = zero2, bc = zero2;
    double hl_c = 0.0, hr_c = 0.0;
    double acc[2] = {0.0, 0.0};                             // K2R: rho', rr
    // One step = one plane.  `uc` is the ring slot t % R: a compile-time constant in the unrolled trips (run_trip),
    // a run-time value in the tail.
    auto step = [&](const int t, const int use0, auto uc) {
        const int u = uc;
        const unsigned full_par = (unsigned)use0 & 1u;      // use0 = t / R: how often the ring was filled before
        const int slot = u, slot_prev = (u + R - 1) % R;    // t % R, (t - 1) % R
        const int pslot = (u + DEPTH) % R;                  // slot of the plane produced at step t
        const int puse = use0 + (u + DEPTH >= R ? 1 : 0);   // which use of that slot it is: (t + DEPTH) / R
        const int xs = (R % DEPTH == 0) ? u % DEPTH : t % DEPTH;   // t % DEPTH: stage of the extras consumed at step t
        const int ii = g.first + t;
        const bool plane_ok = (unsigned)(op.i_lo + ii) < (unsigned)op.nr_glob;
        mbar_wait(s_full + 8u * slot, full_par, fault);     // plane ii: every row has landed
        double2 an = zero2, bn = zero2;
        double hl_n = 0.0, hr_n = 0.0;
        if (plane_ok) {
            const double2 *row = sm.ring[slot][warp];
            an = row[1 + lane];
            bn = row[33 + lane];
            if (g.left_edge) hl_n = row[0].y;
            if (g.right_edge) hr_n = row[g.hr].x;
        }
        const PhiNb nb = phi_neighbours(ac, bc, lane);
        if (t >= 2 && g.interior && g.row_ok) {
            const RowCoefs rc = row_coefs(sm.c, t, warp);
            const double dsc = EPI != EPI_APPLY ? sm.c.cD[t - 1][warp] : 0.0;      // 1/V2 (STS) or Dinv (K2R)
            auto finish = [&](double2 s, double2 uc, int half, int e, int kcell) {
                double2 o;
                const int xi = lane + 32 * half;
                if (EPI == EPI_APPLY) {
                    o = s;
                } else if (EPI == EPI_K2R) {                     // s = q = A p;  stream 0 = r
                    const double2 rv = sm.xf[xs][0][warp - 1][xi];
                    o.x = fma(-alpha, s.x, rv.x);
                    o.y = fma(-alpha, s.y, rv.y);
                    double z0, z1;
                    if (UNIFORM) { z0 = o.x * dsc; z1 = o.y * dsc; }
                    else {
                        const double2 v = ph.VP2(e), wv = ph.WP2(e);
                        z0 = o.x * rcp_nr(fma(v.x, rc.Ec, rc.Fc * wv.x)); z1 = o.y * rcp_nr(fma(v.y, rc.Ec, rc.Fc * wv.y));
                    }
                    acc[0] += o.x * z0 + o.y * z1;
                    acc[1] += o.x * o.x + o.y * o.y;
                } else {
                    double2 mu;                                  // M u = -S u / (V2 vp)
                    const double2 rvp = ph.RVP2(e);
                    mu.x = -(s.x * dsc) * rvp.x;
                    mu.y = -(s.y * dsc) * rvp.y;
                    if (mp.out2) st2g(mp.out2, orow + kcell, mu);
                    o.x = mp.c_u * uc.x + mp.c_L * mu.x;
                    o.y = mp.c_u * uc.y + mp.c_L * mu.y;
                    if (has1) { const double2 x1 = sm.xf[xs][0][warp - 1][xi]; o.x = fma(mp.c_a1, x1.x, o.x); o.y = fma(mp.c_a1, x1.y, o.y); }
                    if (has2) { const double2 x2 = sm.xf[xs][NX > 1 ? 1 : 0][warp - 1][xi]; o.x = fma(mp.c_a2, x2.x, o.x); o.y = fma(mp.c_a2, x2.y, o.y); }
                    if (has3) { const double2 x3 = sm.xf[xs][NX > 2 ? 2 : 0][warp - 1][xi]; o.x = fma(mp.c_a3, x3.x, o.x); o.y = fma(mp.c_a3, x3.y, o.y); }
                }
                st2g(out, orow + kcell, o);
            };
            if (g.qA) {
                const double ukm = g.left_edge ? hl_c : nb.mA;
                const double ukp = g.right_A ? hr_c : (lane == 31 ? nb.pB : nb.pA);
                const double2 s = stencil_half(ph, ea, rc, am, ac, an, sm.ring[slot_prev][warp - 1][1 + lane],
                                               sm.ring[slot_prev][warp + 1][1 + lane], ukm, ukp);
                finish(s, ac, 0, ea, g.ka);
            }
            if (g.qB) {
                const double ukm = lane == 0 ? nb.mA : nb.mB;
                const double ukp = g.right_B ? hr_c : nb.pB;
                const double2 s = stencil_half(ph, eb, rc, bm, bc, bn, sm.ring[slot_prev][warp - 1][33 + lane],
                                               sm.ring[slot_prev][warp + 1][33 + lane], ukm, ukp);
                finish(s, bc, 1, eb, g.kb);
            }
        }
        if (t >= 2) orow += plane;
        __syncwarp();                                       // the warp's reads of slot_prev and of its extras are done
        if (lane == 0) {
            if (t >= 1) mbar_arrive(s_empty + 8u * slot_prev);   // plane t-1 released by this warp
            if (t + DEPTH < g.nsteps) {                     // refill: plane t+DEPTH goes to the slot plane t+DEPTH-R used
                if (puse >= 1) mbar_wait(s_empty + 8u * pslot, (unsigned)(puse - 1) & 1u, fault);
                produce(t + DEPTH, pslot, xs);
            }
        }
        am = ac; ac = an; bm = bc; bc = bn;
        hl_c = hl_n; hr_c = hr_n;
    };
    int t0 = 0;
    for (; t0 + R <= g.nsteps; t0 += R) run_trip(step, t0, t0 / R, std::make_integer_sequence<int, R>{});
    for (int t = t0; t < g.nsteps; t++) step(t, t0 / R, t - t0);
    if (EPI == EPI_K2R) {
        if (grid_sum<NT, 2>(acc, part_base(mp.w, rhs), mp.w.pstride, &mp.w.tickets[rhs * 4 + 2], sm.red) && threadIdx.x == 0)
            reduction_done<ROLE_K2, 2>(mp.w, rhs, acc, mp.cond, mp.use_cond);
    }
}

// ---------------------------------------------------------------------------------------------
// host-side configuration
// ---------------------------------------------------------------------------------------------
template <int TJ, int DEPTH, int MINB>
inline void stencil_tma_pick(bool uniform, int epi, const void **func, dim3 *block, size_t *smem)
{
    if (epi == EPI_APPLY) {
        *func = uniform ? (const void *)k_stencil_tma<TJ, DEPTH, true, MINB, EPI_APPLY>
                        : (const void *)k_stencil_tma<TJ, DEPTH, false, MINB, EPI_APPLY>;
        *smem = uniform ? sizeof(StencilTmaSmem<TJ, DEPTH, 0, true>) : sizeof(StencilTmaSmem<TJ, DEPTH, 0, false>);
    } else if (epi == EPI_K2R) {
        *func = uniform ? (const void *)k_stencil_tma<TJ, DEPTH, true, MINB, EPI_K2R>
                        : (const void *)k_stencil_tma<TJ, DEPTH, false, MINB, EPI_K2R>;
        *smem = uniform ? sizeof(StencilTmaSmem<TJ, DEPTH, 1, true>) : sizeof(StencilTmaSmem<TJ, DEPTH, 1, false>);
    } else {
        *func = uniform ? (const void *)k_stencil_tma<TJ, DEPTH, true, MINB, EPI_STS>
                        : (const void *)k_stencil_tma<TJ, DEPTH, false, MINB, EPI_STS>;
        *smem = uniform ? sizeof(StencilTmaSmem<TJ, DEPTH, 3, true>) : sizeof(StencilTmaSmem<TJ, DEPTH, 3, false>);
    }
    *block = dim3((TJ + 2) * 32);
    cudaFuncSetAttribute(*func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)*smem);
}

inline int stencil_num_tiles() { return 6; }

// tile ids -> (TJ, DEPTH, min blocks/SM): 0 (6,2,2), 1 (8,2,2), 2 (14,2,1), 3 (10,2,1), 4 (8,3,1), 5 (12,3,1)
inline void stencil_configure(int nr, int nt, int np, int uniform, int epi, int tile, int num_sms, int ci_force, int ny,
                              StencilParams *mp, const void **func, dim3 *grid, dim3 *block, size_t *smem)
{
    int tj;
    switch (tile) {
        case 0: tj = 6; stencil_tma_pick<6, 2, 2>(uniform, epi, func, block, smem); break;
        case 1: tj = 8; stencil_tma_pick<8, 2, 2>(uniform, epi, func, block, smem); break;
        case 2: tj = 14; stencil_tma_pick<14, 2, 1>(uniform, epi, func, block, smem); break;
        case 3: tj = 10; stencil_tma_pick<10, 2, 1>(uniform, epi, func, block, smem); break;
        case 4: tj = 8; stencil_tma_pick<8, 3, 1>(uniform, epi, func, block, smem); break;
        default: tj = 12; stencil_tma_pick<12, 3, 1>(uniform, epi, func, block, smem); break;
    }
    mp->t.nkt = (np + TILE_TK - 1) / TILE_TK;
    mp->t.njt = (nt + tj - 1) / tj;
    int occ = 1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, *func, (int)block->x, *smem) != cudaSuccess || occ < 1) {
        cudaGetLastError();
        occ = 1;
    }
    mp->t.ci = tile_pick_ci(nr, (long long)mp->t.nkt * mp->t.njt, (long long)num_sms * occ, ci_force);
    mp->t.nit = (nr + mp->t.ci - 1) / mp->t.ci;
    *grid = dim3((unsigned)(mp->t.nkt * mp->t.njt * mp->t.nit), (unsigned)ny);
}

}  // namespace mas

// tile.cuh -- what the two marching-tile kernels (k1_tma: fused PCG matvec; k_stencil_tma: stencil of a stored vector
// with a fused epilogue) have in common, written once:
//   * the PTX wrappers for mbarriers, TMA bulk copies (cp.async.bulk, SASS UBLKCP) and L2 eviction-priority hints;
//   * the tile geometry: a block owns TJ theta-rows x 128 phi-cells and marches along r over `ci` planes (2.5-D blocking);
//     warp w <-> tile row w-1 (warps 0 and TJ+1 are the theta-halo rows); a lane owns 4 cells as two 16-byte vectors in
//     the two coalesced 64-cell halves A (cells k0+2l, +1) and B (cells k0+64+2l, +1);
//   * the coefficient columns of the tile staged in shared memory, and the phi factors;
//   * the 7-point stencil of one half-row vector from register / shared-memory operands.
// Slabs: vectors are indexed by LOCAL plane (0 .. op.nr-1); the planes -1 and op.nr belong to the
// neighbour slabs and are read through `VecHalo` pointers (peer mappings on a real node); coefficient planes are GLOBAL
// and indexed by op.i_lo + local plane.
#pragma once
#include "common.cuh"

namespace mas {

constexpr int TILE_TK = 128;                 // phi cells per tile row: 32 lanes x 2 halves x double2
constexpr int TILE_CI_MAX = 32;              // max interior planes per block (coefficient staging)
constexpr int TILE_NPL = TILE_CI_MAX + 2;

// ---------------------------------------------------------------------------------------------
// PTX: mbarrier, bulk copy, L2 policies
// ---------------------------------------------------------------------------------------------
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
// try_wait suspends the warp in hardware for a bounded time (it is not a busy poll), then reports the phase
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, unsigned parity)
{
    unsigned ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
                 : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
// Wait for a phase.  A wait that is still unsatisfied after MBAR_TIMEOUT_NS of wall time (%globaltimer, so that
// time-slicing, a debugger or a profiler replay cannot trip it the way an iteration count can) is a protocol error:
// it is reported through *fault (the host turns it into MAS_ECUDA) and the wait is abandoned -- no __trap(), which
// would poison the CUDA context for every handle in the process.
constexpr unsigned long long MBAR_TIMEOUT_NS = 20ull * 1000 * 1000 * 1000;
__device__ __forceinline__ unsigned long long globaltimer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;\n" : "=l"(t));
    return t;
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity, int *fault)
{
    if (mbar_try_wait(bar, parity)) return;
    const unsigned long long t0 = globaltimer_ns();
    while (!mbar_try_wait(bar, parity))
        if (globaltimer_ns() - t0 > MBAR_TIMEOUT_NS) {
            *fault = 1;
            return;
        }
}
__device__ __forceinline__ uint64_t l2_policy_evict_last()
{
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;\n" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t l2_policy_evict_first()
{
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;\n" : "=l"(p));
    return p;
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_g2s_hint(void *dst, const void *src, unsigned bytes, uint64_t *bar, uint64_t pol)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;\n"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol) : "memory");
}
__device__ __forceinline__ void st2_hint(double *p, long long cell, double2 v, uint64_t pol)
{
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;\n" ::"l"(p + cell), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}
__device__ __forceinline__ double2 ld2g(const double *p, long long cell)
{
    return *reinterpret_cast<const double2 *>(p + cell);
}
__device__ __forceinline__ void st2g(double *p, long long cell, double2 v)
{
    *reinterpret_cast<double2 *>(p + cell) = v;
}

// L2 residency plan of a launch: accesses to the first `keep` planes of the vector named in the
// kernel are issued with evict_last priority, so that this part of the vector stays in the 126 MB L2 from one kernel to
// the next; every other access of the kernels that take a plan is plain.  keep = 0: no hints at all.
struct L2Plan {
    int keep_r;                              // planes [0, keep_r) of r
    int keep_p;                              // planes [0, keep_p) of p (both ping-pong buffers)
    int first_x;                             // 1: x is streamed with evict_first
};

// ---------------------------------------------------------------------------------------------
// tile geometry
// ---------------------------------------------------------------------------------------------
struct TileParams {
    int nkt, njt, nit, ci;                   // tiles in phi, theta, r; interior planes per block
    double vp, wp, ip;                       // uniform-phi factors (dph_c, 2/dph_f, 1/dph_f)
    int reverse;                             // 1: blocks take the tiles in reverse order (serpentine sweeps)
    L2Plan l2;
};

struct TileGeom {
    int lane, warp, tid;
    int jt, i0, i1, first, nsteps;           // planes [i0, i1) are the block's own; first = i0-1; nsteps = i1-i0+2
    int j, k0, tkeff, kl, kr;                // this warp's theta row; first phi cell; valid cells; periodic halo cells
    int ka, kb;                              // first cell of this lane's A and B vectors
    bool row_ok, vA, vB, interior, qA, qB, left_edge, right_A, right_B, right_edge;
};

template <int TJ>
__device__ __forceinline__ TileGeom tile_geom(const OpDev &op, const TileParams &mp)
{
    TileGeom g;
    g.tid = threadIdx.x; g.lane = threadIdx.x & 31; g.warp = threadIdx.x >> 5;
    int b = mp.reverse ? (int)gridDim.x - 1 - (int)blockIdx.x : (int)blockIdx.x;
    const int kt = b % mp.nkt; b /= mp.nkt;  // phi fastest, then theta, then r => neighbouring tiles run together
    g.jt = b % mp.njt;
    const int it = b / mp.njt;
    g.i0 = it * mp.ci; g.i1 = min(g.i0 + mp.ci, op.nr);
    g.first = g.i0 - 1; g.nsteps = g.i1 - g.i0 + 2;
    g.j = g.jt * TJ + g.warp - 1;
    g.k0 = kt * TILE_TK;
    g.tkeff = min(TILE_TK, op.np - g.k0);
    g.row_ok = (g.j >= 0) && (g.j < op.nt);
    g.vA = g.row_ok && (2 * g.lane < g.tkeff); g.vB = g.row_ok && (64 + 2 * g.lane < g.tkeff);
    g.interior = (g.warp >= 1) && (g.warp <= TJ);
    g.qA = g.interior && g.vA; g.qB = g.interior && g.vB;
    g.left_edge = g.qA && (g.lane == 0);
    g.right_A = g.qA && (2 * g.lane + 2 == g.tkeff); g.right_B = g.qB && (64 + 2 * g.lane + 2 == g.tkeff);
    g.right_edge = g.right_A || g.right_B;
    g.kl = g.k0 == 0 ? op.np - 1 : g.k0 - 1;                    // odd (k0 and np are even)
    g.kr = g.k0 + g.tkeff >= op.np ? 0 : g.k0 + g.tkeff;        // even
    g.ka = g.k0 + 2 * g.lane; g.kb = g.ka + 64;
    return g;
}

// A vector as the tile kernels address it: own planes 0..nr-1 at `own`, plane -1 at `lo`, plane nr at `hi` (the
// adjacent planes of the neighbour slabs; null = the mesh ends there, the plane reads as zero).
struct VecHalo {
    const double *own, *lo, *hi;
};
// Row base pointer of local plane ii (first cell of theta row j), or null when the plane does not exist.
__device__ __forceinline__ const double *plane_row(const VecHalo &v, const OpDev &op, int ii, int j)
{
    const long long rowoff = (long long)j * op.np;
    if (ii >= 0 && ii < op.nr) return v.own + (long long)ii * op.nt * op.np + rowoff;
    if (ii == -1) return v.lo ? v.lo + rowoff : nullptr;
    if (ii == op.nr) return v.hi ? v.hi + rowoff : nullptr;
    return nullptr;
}

// ---------------------------------------------------------------------------------------------
// coefficient columns of a tile: [plane of the march][row incl. theta halo], and the phi factors
// ---------------------------------------------------------------------------------------------
template <int NW, bool UNIFORM>
struct TileCoefs {
    double cE[TILE_NPL][NW], cF[TILE_NPL][NW], cD[TILE_NPL][NW], cAR[TILE_NPL][NW], cAT[TILE_NPL][NW];
    double phv[UNIFORM ? 1 : TILE_TK + 2], phw[UNIFORM ? 1 : TILE_TK + 2], phi[UNIFORM ? 1 : TILE_TK + 2];
};

struct PlaneSetDev {                         // which planes the stencil uses (dt-scaled: A_sym; base: L_sym)
    const double *E, *F, *AR, *AT;           // diagonal per unit vp, phi coupling, radial / theta off-diagonals
    const double *D;                         // per-row scalar of the epilogue (Dinv, or 1/V2), may be null
};

// One global latency, then LDS broadcasts.  Coefficient planes are global: plane index op.i_lo + local.
template <int TJ, bool UNIFORM, class C>
__device__ __forceinline__ void stage_coefs(C &sm, const TileGeom &g, const OpDev &op, const PlaneSetDev &ps)
{
    constexpr int NW = TJ + 2, NT = NW * 32;
    for (int e = g.tid; e < g.nsteps * NW; e += NT) {
        const int pl = e / NW, wr = e - pl * NW;
        const int ii = op.i_lo + g.first + pl, jj = g.jt * TJ + wr - 1;
        const bool in = ii >= 0 && ii < op.nr_glob && jj >= 0 && jj < op.nt;
        const int row = ii * op.nt + jj;
        sm.cE[pl][wr] = in ? __ldg(ps.E + row) : 0.0;
        sm.cF[pl][wr] = in ? __ldg(ps.F + row) : 0.0;
        sm.cD[pl][wr] = (in && ps.D) ? __ldg(ps.D + row) : 0.0;
        sm.cAR[pl][wr] = (ii >= 0 && ii <= op.nr_glob && jj >= 0 && jj < op.nt) ? __ldg(ps.AR + row) : 0.0;
        sm.cAT[pl][wr] = (ii >= 0 && ii < op.nr_glob && jj >= 0 && jj <= op.nt) ? __ldg(ps.AT + ii * (op.nt + 1) + jj) : 0.0;
    }
    if (!UNIFORM)
        for (int e = g.tid; e < TILE_TK + 2; e += NT) {
            int kk = g.k0 - 1 + e;                                // wrap once in either direction
            kk = kk < 0 ? kk + op.np : (kk >= op.np ? kk - op.np : kk);
            kk = kk >= op.np ? kk % op.np : kk;                   // tiny meshes (np < 130)
            sm.phv[e] = __ldg(op.vp + kk); sm.phw[e] = __ldg(op.wp + kk); sm.phi[e] = __ldg(op.ip + kk);
        }
}

// phi factors of cell e (index into the staged arrays = cell - k0 + 1); uniform meshes use the kernel constants
template <bool UNIFORM, class C>
struct PhiFac {
    const C &sm;
    double vp, wp, ip;
    __device__ __forceinline__ double VP(int e) const { return UNIFORM ? vp : sm.phv[e]; }
    __device__ __forceinline__ double WP(int e) const { return UNIFORM ? wp : sm.phw[e]; }
    __device__ __forceinline__ double IP(int e) const { return UNIFORM ? ip : sm.phi[e]; }   // face e+1/2
};

struct RowCoefs {                            // coefficients of the row whose stencil is being formed (plane t-1)
    double Ec, Fc, ARm, ARp, ATm, ATp;
};
template <class C>
__device__ __forceinline__ RowCoefs row_coefs(const C &sm, int t, int warp)
{
    RowCoefs c;
    c.Ec = sm.cE[t - 1][warp]; c.Fc = sm.cF[t - 1][warp];
    c.ARm = sm.cAR[t - 1][warp]; c.ARp = sm.cAR[t][warp];
    c.ATm = sm.cAT[t - 1][warp]; c.ATp = sm.cAT[t - 1][warp + 1];
    return c;
}

// (S u) of the two cells e, e+1 of one half-row vector:
//   d u_c - vp (ARm u_im + ARp u_ip + ATm u_jm + ATp u_jp) - F (ip[k] u_kp + ip[k-1] u_km),  d = vp E + F wp
template <class PF>
__device__ __forceinline__ double2 stencil_half(const PF &ph, int e, const RowCoefs &c, double2 um, double2 uc, double2 un,
                                                double2 ujm, double2 ujp, double ukm, double ukp)
{
    const double d0 = fma(ph.VP(e), c.Ec, c.Fc * ph.WP(e)), d1 = fma(ph.VP(e + 1), c.Ec, c.Fc * ph.WP(e + 1));
    const double sx = c.ARm * um.x + c.ARp * un.x + c.ATm * ujm.x + c.ATp * ujp.x;
    const double sy = c.ARm * um.y + c.ARp * un.y + c.ATm * ujm.y + c.ATp * ujp.y;
    double2 s;
    s.x = d0 * uc.x - ph.VP(e) * sx - c.Fc * (ph.IP(e) * uc.y + ph.IP(e - 1) * ukm);
    s.y = d1 * uc.y - ph.VP(e + 1) * sy - c.Fc * (ph.IP(e + 1) * ukp + ph.IP(e) * uc.x);
    return s;
}

// phi neighbours of a lane's two vectors by warp shuffle (must be executed by all 32 lanes):
// returns {u[k-1] for A, u[k+2] for A, u[k-1] for B, u[k+2] for B} before the periodic-edge substitution.
struct PhiNb {
    double mA, pA, mB, pB;
};
__device__ __forceinline__ PhiNb phi_neighbours(double2 ac, double2 bc, int lane)
{
    const int lm = (lane + 31) & 31, lp = (lane + 1) & 31;
    PhiNb n;
    n.mA = __shfl_sync(0xffffffffu, ac.y, lm); n.mB = __shfl_sync(0xffffffffu, bc.y, lm);
    n.pA = __shfl_sync(0xffffffffu, ac.x, lp); n.pB = __shfl_sync(0xffffffffu, bc.x, lp);
    return n;
}

// r-chunk length of a marching kernel: minimise rounds x (planes per block + halo planes + start-up), ties ->
// longer chunks.  `nslots` = blocks resident at once; `ny` = gridDim.y (right-hand sides) sharing the SMs.
inline int tile_pick_ci(int nr, long long cols, long long nslots, int ny, int ci_force)
{
    int best = TILE_CI_MAX;
    double best_cost = 1e300;
    for (int ci = TILE_CI_MAX; ci >= 4; ci -= 2) {
        const long long tiles = cols * ((nr + ci - 1) / ci) * ny;
        const double rounds = (double)((tiles + nslots - 1) / nslots);
        const double cost = rounds * (ci + 2 + 3);
        if (cost < best_cost * 0.999) { best_cost = cost; best = ci; }
    }
    if (nr < best) best = nr;
    if (ci_force > 0 && ci_force <= TILE_CI_MAX) best = ci_force < nr ? ci_force : nr;
    return best;
}

}  // namespace mas

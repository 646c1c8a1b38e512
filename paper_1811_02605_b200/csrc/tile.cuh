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
#include <utility>
#include "common.cuh"

namespace mas {

constexpr int TILE_TK = 128;                 // phi cells per tile row: 32 lanes x 2 halves x double2
constexpr int TILE_CI_MAX = 32;              // max interior planes per block (coefficient staging)
constexpr int TILE_NPL = TILE_CI_MAX + 2;

// ---------------------------------------------------------------------------------------------
// PTX: mbarrier, bulk copy, L2 policies
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
// Barriers and bulk-copy destinations are addressed by their 32-bit shared-memory address, computed once per kernel:
// the generic -> shared conversion per call was 6 % of the stencil kernel's instructions (ncu, round 2).
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
// try_wait suspends the warp in hardware for a bounded time (it is not a busy poll), then reports the phase
__device__ __forceinline__ bool mbar_try_wait(unsigned bar, unsigned parity)
{
    unsigned ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
// Wait for a phase.  A wait that is still unsatisfied after MBAR_TIMEOUT_NS of wall time (%globaltimer, so that
// time-slicing, a debugger or a profiler replay cannot trip it the way an iteration count can) is a protocol error:
// it is reported through *fault (the host turns it into MAS_ECUDA) and the wait is abandoned -- no __trap(), which
// would poison the CUDA context for every handle in the process.  The clock is read once per 1024 failed polls only:
// reading it on every poll cost 4 % of K1's and 8 % of K2R's instructions (ncu, round 2).
constexpr unsigned long long MBAR_TIMEOUT_NS = 20ull * 1000 * 1000 * 1000;
__device__ __forceinline__ unsigned long long globaltimer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;\n" : "=l"(t));
    return t;
}
// the same with a suspend-time hint (ns): the warp may sleep that long in hardware unless the phase completes first
__device__ __forceinline__ bool mbar_try_wait_hint(unsigned bar, unsigned parity, unsigned ns)
{
    unsigned ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
                 : "=r"(ok) : "r"(bar), "r"(parity), "r"(ns) : "memory");
    return ok != 0;
}
__device__ __noinline__ void mbar_wait_slow(unsigned bar, unsigned parity, int *fault)
{
    unsigned long long t0 = 0;
    for (unsigned polls = 1;; polls++) {
        if (mbar_try_wait_hint(bar, parity, 20000u)) return;   // polling warps took 12 % of the stencil kernel's issue slots
        if ((polls & 1023u) == 0) {
            const unsigned long long t = globaltimer_ns();
            if (t0 == 0) t0 = t;
            else if (t - t0 > MBAR_TIMEOUT_NS) { *fault = 1; return; }
        }
    }
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity, int *fault)
{
    if (mbar_try_wait(bar, parity)) return;
    if (mbar_try_wait(bar, parity)) return;
    mbar_wait_slow(bar, parity, fault);
}
// x is read once and written once per iteration and never reused inside it: its accesses may carry the L2
// evict_first priority so that they do not displace r and p.  evict_last hints are NOT used: on
// this pool's B200s every access carrying an evict_last policy (created by createpolicy or given as the constant
// CUTLASS uses) ended the kernel with "unspecified launch failure" (gpurun, round 2); evict_first works.
__device__ __forceinline__ uint64_t l2_policy_evict_first()
{
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;\n" : "=l"(p));
    return p;
}
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void *src, unsigned bytes, unsigned bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void bulk_g2s_hint(unsigned dst, const void *src, unsigned bytes, unsigned bar, uint64_t pol)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;\n"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(pol) : "memory");
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

// L2 plan of a launch: first_x = 1: x is streamed with evict_first (see above); 0: no hints at all.
struct L2Plan {
    int first_x;
};

// ---------------------------------------------------------------------------------------------
// tile geometry
// ---------------------------------------------------------------------------------------------
struct TileParams {
    int nkt, njt, nit, ci;                   // tiles in phi, theta, r; interior planes per block
    double vp, wp, ip;                       // uniform-phi factors (dph_c, 2/dph_f, 1/dph_f)
    int reverse;                             // 1: blocks take the tiles in reverse order (serpentine sweeps)
    int zin;                                 // K1 with PC2: the preconditioned residual z is read from Work::z instead of formed as r/d
    L2Plan l2;
};

struct TileGeom {
    int lane, warp, tid;
    int jt, i0, i1, first, nsteps;           // planes [i0, i1) are the block's own; first = i0-1; nsteps = i1-i0+2
    int j, k0, tkeff, kl, kr;                // this warp's theta row; first phi cell; valid cells; periodic halo cells
    int ka, kb;                              // first cell of this lane's A and B vectors
    bool row_ok, vA, vB, interior, qA, qB, left_edge, right_A, right_B, right_edge;
    bool wrapless;                           // the two phi-halo pairs are adjacent in memory to the row segment
    int hr;                                  // index of the right halo pair in a staged row (1 + tkeff/2)
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
    g.wrapless = g.k0 > 0 && g.k0 + g.tkeff < op.np;
    g.hr = 1 + g.tkeff / 2;
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

// A tile row as it is staged in shared memory: ROW_V2 double2 = [left phi-halo pair | 128 cells | right pair]; the
// pairs are (kl-1, kl) and (kr, kr+1), so the halo cells are .y of element 0 and .x of element g.hr.  A lane's A / B
// vectors are elements 1 + lane and 33 + lane.  When the halo pairs are adjacent in memory to the segment (no periodic
// wrap inside this tile) the whole row is ONE bulk copy, otherwise three -- issued by one lane, `row_k0` = address of
// cell k0 of the row.  (Round 2: five separate copies per vector and row were 21 % of K1's instructions.)
constexpr int ROW_V2 = 66;
constexpr unsigned ROW_BYTES = ROW_V2 * 16;
__device__ __forceinline__ void row_copy(unsigned dst, const double *row_k0, const TileGeom &g, int op_np, unsigned rowbytes, unsigned bar)
{
    if (g.wrapless) {
        bulk_g2s(dst, row_k0 - 2, rowbytes + 32u, bar);
    } else if (g.k0 > 0) {                               // last tile of the row: only the right pair wraps
        bulk_g2s(dst, row_k0 - 2, rowbytes + 16u, bar);
        bulk_g2s(dst + 16u + rowbytes, row_k0 + (g.kr - g.k0), 16u, bar);
    } else if (g.tkeff < op_np) {                        // first tile: only the left pair wraps
        bulk_g2s(dst + 16u, row_k0, rowbytes + 16u, bar);
        bulk_g2s(dst, row_k0 + (g.kl - 1 - g.k0), 16u, bar);
    } else {                                             // the tile is the whole row
        bulk_g2s(dst + 16u, row_k0, rowbytes, bar);
        bulk_g2s(dst, row_k0 + (g.kl - 1 - g.k0), 16u, bar);
        bulk_g2s(dst + 16u + rowbytes, row_k0 + (g.kr - g.k0), 16u, bar);
    }
}

// ---------------------------------------------------------------------------------------------
// coefficient columns of a tile: [plane of the march][row incl. theta halo], and the phi factors
// ---------------------------------------------------------------------------------------------
template <int NW, bool UNIFORM>
struct TileCoefs {
    double cE[TILE_NPL][NW], cF[TILE_NPL][NW], cD[TILE_NPL][NW], cAR[TILE_NPL][NW], cAT[TILE_NPL][NW];
    double phv[UNIFORM ? 1 : TILE_TK + 2], phw[UNIFORM ? 1 : TILE_TK + 2], phi[UNIFORM ? 1 : TILE_TK + 2];
    double phr[UNIFORM ? 1 : TILE_TK + 2];   // 1/vp: the M u = -S u / V epilogue multiplies instead of dividing per cell
    // The same factors once more as PAIRS, for the two cells (2l+1, 2l+2) of half-row vector l (l = lane, lane + 32): a
    // lane then fetches what its vector needs with one 16-byte load per array, lanes 16 bytes apart -- conflict-free --
    // instead of two 8-byte loads 16 bytes apart (2-way bank conflicts: ncu counted 16.7 M conflicts per K1 launch on
    // the non-uniform 256x256x512 mesh against 2.1 M on the uniform one).  ipm[l] = ip of cell 2l (face 2l + 1/2).
    alignas(16) double2 pv2[UNIFORM ? 1 : TILE_TK / 2], pw2[UNIFORM ? 1 : TILE_TK / 2], pi2[UNIFORM ? 1 : TILE_TK / 2],
        pr2[UNIFORM ? 1 : TILE_TK / 2];
    double ipm[UNIFORM ? 1 : TILE_TK / 2];
};

struct PlaneSetDev {                         // which planes the stencil uses (dt-scaled: A_sym; base: L_sym)
    const double *E, *F, *AR, *AT;           // diagonal per unit vp, phi coupling, radial / theta off-diagonals
    const double *D;                         // per-row scalar of the epilogue (Dinv, or 1/V2), may be null
};

// One global latency, then LDS broadcasts.  Coefficient planes are global: plane index op.i_lo + local.
// Uniform phi: vp, wp, ip are constants, so the per-row products the stencil needs are formed HERE, once per block:
//   cE <- vp E + F wp (the diagonal d),  cF <- F ip,  cAR <- vp AR,  cAT <- vp AT
// and the stencil of a cell is 1 mul + 4 fma + 1 add + 1 fma instead of 11 operations.
template <int TJ, bool UNIFORM, class C>
__device__ __forceinline__ void stage_coefs(C &sm, const TileGeom &g, const OpDev &op, const PlaneSetDev &ps, double vp,
                                            double wp, double ip)
{
    constexpr int NW = TJ + 2, NT = NW * 32;
    for (int e = g.tid; e < g.nsteps * NW; e += NT) {
        const int pl = e / NW, wr = e - pl * NW;
        const int ii = op.i_lo + g.first + pl, jj = g.jt * TJ + wr - 1;
        const bool in = ii >= 0 && ii < op.nr_glob && jj >= 0 && jj < op.nt;
        const int row = ii * op.nt + jj;
        const double E = in ? __ldg(ps.E + row) : 0.0, F = in ? __ldg(ps.F + row) : 0.0;
        const double AR = (ii >= 0 && ii <= op.nr_glob && jj >= 0 && jj < op.nt) ? __ldg(ps.AR + row) : 0.0;
        const double AT = (ii >= 0 && ii < op.nr_glob && jj >= 0 && jj <= op.nt) ? __ldg(ps.AT + ii * (op.nt + 1) + jj) : 0.0;
        sm.cE[pl][wr] = UNIFORM ? fma(vp, E, F * wp) : E;
        sm.cF[pl][wr] = UNIFORM ? F * ip : F;
        sm.cD[pl][wr] = (in && ps.D) ? __ldg(ps.D + row) : 0.0;
        sm.cAR[pl][wr] = UNIFORM ? vp * AR : AR;
        sm.cAT[pl][wr] = UNIFORM ? vp * AT : AT;
    }
    if (!UNIFORM)
        for (int e = g.tid; e < TILE_TK + 2; e += NT) {
            int kk = g.k0 - 1 + e;                                // wrap once in either direction
            kk = kk < 0 ? kk + op.np : (kk >= op.np ? kk - op.np : kk);
            kk = kk >= op.np ? kk % op.np : kk;                   // tiny meshes (np < 130)
            const double v = __ldg(op.vp + kk), wv = __ldg(op.wp + kk), iv = __ldg(op.ip + kk), rv = 1.0 / v;
            sm.phv[e] = v; sm.phw[e] = wv; sm.phi[e] = iv; sm.phr[e] = rv;
            if (e >= 1 && e <= TILE_TK) {                         // cell e of the tile = component (e-1)&1 of pair (e-1)>>1
                const int l = (e - 1) >> 1;
                double *pv = reinterpret_cast<double *>(&sm.pv2[l]), *pw = reinterpret_cast<double *>(&sm.pw2[l]);
                double *pi = reinterpret_cast<double *>(&sm.pi2[l]), *pr = reinterpret_cast<double *>(&sm.pr2[l]);
                pv[(e - 1) & 1] = v; pw[(e - 1) & 1] = wv; pi[(e - 1) & 1] = iv; pr[(e - 1) & 1] = rv;
            }
            if (!(e & 1) && e < TILE_TK) sm.ipm[e >> 1] = iv;   // ip of cell e = 2l
        }
}

// phi factors of cell e (index into the staged arrays = cell - k0 + 1); uniform meshes use the kernel constants
template <bool UNIFORM, class C>
struct PhiFac {
    static constexpr bool uniform = UNIFORM;
    const C &sm;
    double vp, wp, ip;
    __device__ __forceinline__ double VP(int e) const { return UNIFORM ? vp : sm.phv[e]; }
    __device__ __forceinline__ double WP(int e) const { return UNIFORM ? wp : sm.phw[e]; }
    __device__ __forceinline__ double IP(int e) const { return UNIFORM ? ip : sm.phi[e]; }   // face e+1/2
    __device__ __forceinline__ double RVP(int e) const { return UNIFORM ? 1.0 / vp : sm.phr[e]; }
    // pairs for the vector whose first cell is e (odd): (X(e), X(e+1)); IPM = IP(e-1)
    __device__ __forceinline__ double2 VP2(int e) const { return UNIFORM ? make_double2(vp, vp) : sm.pv2[(e - 1) >> 1]; }
    __device__ __forceinline__ double2 WP2(int e) const { return UNIFORM ? make_double2(wp, wp) : sm.pw2[(e - 1) >> 1]; }
    __device__ __forceinline__ double2 IP2(int e) const { return UNIFORM ? make_double2(ip, ip) : sm.pi2[(e - 1) >> 1]; }
    __device__ __forceinline__ double2 RVP2(int e) const { return UNIFORM ? make_double2(1.0 / vp, 1.0 / vp) : sm.pr2[(e - 1) >> 1]; }
    __device__ __forceinline__ double IPM(int e) const { return UNIFORM ? ip : sm.ipm[(e - 1) >> 1]; }
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
    const double sx = c.ARm * um.x + c.ARp * un.x + c.ATm * ujm.x + c.ATp * ujp.x;
    const double sy = c.ARm * um.y + c.ARp * un.y + c.ATm * ujm.y + c.ATp * ujp.y;
    double2 s;
    if (PF::uniform) {                       // the staged coefficients already hold d, vp AR, vp AT, F ip (stage_coefs)
        s.x = fma(-c.Fc, uc.y + ukm, c.Ec * uc.x - sx);
        s.y = fma(-c.Fc, ukp + uc.x, c.Ec * uc.y - sy);
        return s;
    }
    const double2 v = ph.VP2(e), wv = ph.WP2(e), iv = ph.IP2(e);     // same arithmetic as with the scalar factors, in
    const double im = ph.IPM(e);                                     // the same order: results are bit-identical
    const double d0 = fma(v.x, c.Ec, c.Fc * wv.x), d1 = fma(v.y, c.Ec, c.Fc * wv.y);
    s.x = d0 * uc.x - v.x * sx - c.Fc * (iv.x * uc.y + im * ukm);
    s.y = d1 * uc.y - v.y * sy - c.Fc * (iv.y * ukp + iv.x * uc.x);
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

// One trip of a plane loop unrolled by N: calls step(t0 + I, trip, SlotC<I>) for I = 0..N-1 with NO branch
// between the steps, so that inside a trip ring slots are compile-time and the compiler renames the plane registers
// (u_{i-1}, u_i, u_{i+1}) instead of moving them; the remaining (< N) steps of a block run the same step body with a
// run-time slot.
template <int V>
struct SlotC {                               // a compile-time slot index that converts to int in device code
    __host__ __device__ constexpr operator int() const { return V; }
};
template <class F, int... I>
__device__ __forceinline__ void run_trip(F &step, int t0, int trip, std::integer_sequence<int, I...>)
{
    (step(t0 + I, trip, SlotC<I>{}), ...);
}

// r-chunk length of a marching kernel: minimise rounds x (planes per block + halo planes + start-up), ties ->
// longer chunks.  `nslots` = blocks resident at once.  The choice must NOT depend on the number of right-hand sides
// of a batched solve: the chunk length fixes the grid and with it the order of the partial sums, and a batched
// solve is promised to be bit-identical to single solves.
inline int tile_pick_ci(int nr, long long cols, long long nslots, int ci_force)
{
    int best = TILE_CI_MAX;
    double best_cost = 1e300;
    for (int ci = TILE_CI_MAX; ci >= 4; ci -= 2) {
        const long long tiles = cols * ((nr + ci - 1) / ci);
        const double rounds = (double)((tiles + nslots - 1) / nslots);
        const double cost = rounds * (ci + 2 + 3);
        if (cost < best_cost * 0.999) { best_cost = cost; best = ci; }
    }
    if (nr < best) best = nr;
    if (ci_force > 0 && ci_force <= TILE_CI_MAX) best = ci_force < nr ? ci_force : nr;
    return best;
}

}  // namespace mas

// kernels_pc2.cuh -- PC2 on the GPU (Sec. 2.2: "the second (PC2) is a
// block-Jacobi using a zero-fill incomplete LU factorization [22]"; blocks = non-overlapping boxes: DESIGN.md R8; its triangular
// solves are what the authors call not vectorizable and leave on the CPU).
//
// B200 design (R8, section 5 "PC2"): the domains of the block-Jacobi decomposition are free to choose, so
// they are chosen for the machine: every phi LINE (one (i, j) row of np cells, with its periodic wrap coupling) is
// one domain.  The oracle shows that on these meshes the line domains lose 2 iterations against the undivided ILU(0)
// (38 vs 36 on config 3, against 437 with PC1), because the stiffest couplings are the phi ones near the poles.
// A line's A_blk is cyclic tridiagonal; its ILU(0) keeps the wrap entries and drops their fill:
//     piv_0 = a_0;  piv_k = a_k - c_{k-1}^2 / piv_{k-1};  piv_{np-1} additionally - w^2 / piv_0
//     a_k = vp[k] E + F wp[k] (diagonal of A_sym),  c_k = -F ip[k] (coupling k <-> k+1),  w = c_{np-1} (np-1 <-> 0)
//     L y = r :  y_k = r_k - e_{k-1} y_{k-1},  e_k = c_k / piv_k;   y_{np-1} additionally - (w / piv_0) y_0
//     U z = y :  z_{np-1} = y_{np-1} / piv_{np-1};  z_k = y_k / piv_k - e_k z_{k+1};  z_0 additionally - (w / piv_0) z_{np-1}
// Both substitutions are first-order linear recurrences along the line.  ONE WARP solves a line: a lane owns a chunk
// of M consecutive cells, reduces its chunk to an affine map (y_out = Y + P y_in), the 32 maps are combined by a
// 5-step warp scan, and the lane then runs its chunk again from the now known y_in -- the same recurrence as the
// sequential algorithm, only the chunk's incoming value comes from the scan.  No inter-warp dependency exists, so
// the "sequential" preconditioner streams like a vector kernel:
//     K2P (k_pc2_line<.., false>):  r -= alpha q;  z = M^-1 r;  rho' = r.z;  rr = r.r;  then the scalar step S5
//                                   reads r, q, 1/piv;  writes r, z            = 5 doubles per cell
//     init (k_pc2_line<.., true>):  r = V.b - A x0;  z = M^-1 r;  bb, rr, rho
// and K1 runs with z read from memory instead of r/d (TileParams::zin).  1/piv is the one stored factor (N doubles,
// written by k_pc2_factor at set_dt), kept in the chunk order of the solve so that its loads are coalesced.
// Vectors are loaded / stored in their natural order (coalesced 16-byte accesses) and change to the chunk order
// through a padded per-warp shared-memory buffer.
#pragma once
#include "kernels_base.cuh"

namespace mas {

struct Pc2Dev {
    const double *dinvT;        // [rows][32 * M]  1 / piv, chunk order (pc2_slot)
    const double *ipT;          // [32 * M]        ip[k] in chunk order, 0 beyond np (non-uniform phi only)
    double ip0;                 // uniform phi: 1 / dph_f
    int M;                      // cells per lane: the smallest of 4, 8, 12, 16, 24, 32 with 32 M >= np
};

// where cell k of a line lives in the chunk-ordered arrays: lane l = k / M, slot u = k % M; pairs (u, u + 1) adjacent
__host__ __device__ __forceinline__ int pc2_slot(int k, int M)
{
    const int l = k / M, u = k - l * M;
    return ((u >> 1) * 32 + l) * 2 + (u & 1);
}

// ---------------------------------------------------------------------------------------------
// factorisation: one thread per line, sequential along phi (O(N) divisions, once per set_dt)
// ---------------------------------------------------------------------------------------------
__global__ void k_pc2_factor(OpDev op, double *dinvT, int M)
{
    const int line = blockIdx.x * blockDim.x + threadIdx.x;
    if (line >= op.nr_glob * op.nt) return;
    const double E = op.E[line], F = op.F[line];
    double *out = dinvT + (size_t)line * 32 * M;
    const int np = op.np;
    auto diag = [&](int k) { return fma(__ldg(op.vp + k), E, F * __ldg(op.wp + k)); };
    double inv = 1.0 / diag(0);                             // 1 / piv_{k-1}; ONE division per cell: l_k = c / piv is formed as c * (1 / piv),
    const double inv0 = inv;                                // the product the line kernel uses as well
    double even = inv;                                      // 1/piv of the last even cell: cells (k, k + 1), k even, are
    for (int k = 1; k < np; k++) {                          // adjacent in the chunk order and stored as one 16-byte pair
        double a = diag(k);
        if (k == np - 1) {                                  // lower entries in ascending column order: the wrap (column 0) first
            const double w = -F * __ldg(op.ip + np - 1);
            a -= (w * inv0) * w;
        }
        const double c = -F * __ldg(op.ip + k - 1);
        inv = 1.0 / (a - (c * inv) * c);
        if (k & 1) *reinterpret_cast<double2 *>(out + pc2_slot(k - 1, M)) = make_double2(even, inv);
        else even = inv;
    }
    for (int k = np; k < 32 * M; k += 2) *reinterpret_cast<double2 *>(out + pc2_slot(k, M)) = make_double2(0.0, 0.0);
}

// ---------------------------------------------------------------------------------------------
// the line kernel
// ---------------------------------------------------------------------------------------------
constexpr int PC2_NT = 256, PC2_NWARP = PC2_NT / 32;
__device__ __forceinline__ unsigned smem_addr(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
inline size_t pc2_smem(int M) { return (size_t)PC2_NWARP * (32 * (M + 2) + 2 * 32 * M) * sizeof(double); }   // chunk-order buffer + q, r stage

template <int M, bool UNIFORM, bool INIT>
__global__ void __launch_bounds__(PC2_NT, M >= 24 ? 1 : 2)
k_pc2_line(OpDev op, Work w, Pc2Dev pc, cudaGraphConditionalHandle cond, int use_cond, int reverse)
{
    constexpr int S = M + 2;                            // chunk stride in the staging buffer (doubles): S/2 is odd for every
    constexpr int H = M / 2;                            // supported M (multiples of 4) => conflict-free 16-byte accesses both ways
    extern __shared__ __align__(16) double pc2_buf[];
    __shared__ double sh[32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double2 *buf = reinterpret_cast<double2 *>(pc2_buf + (size_t)warp * (32 * S + 64 * M));   // [lane][S/2] double2
    // stage of the NEXT line's q and r (or b): [h][lane] double2 each, filled by cp.async (LDGSTS); a thread reads back
    // only the slots it copied itself, so cp.async.wait_group is the only synchronisation the stage needs
    double2 *stq = buf + 16 * S, *str = stq + 32 * H;
    const int rhs = blockIdx.y;
    State *st = w.st + rhs;
    double alpha = 0.0;
    if (!INIT) {
        if (!st->active) {                              // this right-hand side is done: report, nothing else
            if (blockIdx.x == 0 && threadIdx.x == 0 && !w.slab_sums) loop_vote(w, 0, gridDim.y, cond, use_cond);
            return;
        }
        alpha = st->alpha;
    }
    const long long voff = rhs * w.vstride;
    double *rvec = w.r + voff, *zvec = w.z + voff;
    const double *qvec = w.q + voff;
    const double *bvec = INIT ? w.args->b[rhs] : nullptr;
    double *p0 = w.p0 + voff;

    const int np = op.np, nv = op.nv;
    const int kbase = lane * M;
    const int lw = (np - 1) / M, uw = (np - 1) - lw * M;       // lane and slot of the last cell of the line
    double ipc[UNIFORM ? 1 : M];                                // ip[k] of this lane's cells (non-uniform phi)
    if (!UNIFORM) {
#pragma unroll
        for (int u = 0; u < M; u++) ipc[u] = __ldg(pc.ipT + pc2_slot(kbase + u, M));
    }
    const double ipw = UNIFORM ? pc.ip0 : __ldg(op.ip + np - 1);
    double acc[3] = {0.0, 0.0, 0.0};                            // rho', rr, (init) bb

    const double *rsrc = INIT ? bvec : rvec;
    auto prefetch = [&](int ln) {                               // this lane's q and r vectors of line ln -> the stage
        if (ln < op.nrows) {
            const size_t b2 = (size_t)(reverse ? op.nrows - 1 - ln : ln) * np;
#pragma unroll
            for (int h = 0; h < H; h++) {
                const int v = lane + 32 * h;
                if (v < nv) {
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_addr(stq + h * 32 + lane)), "l"(qvec + b2 + 2 * v) : "memory");
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_addr(str + h * 32 + lane)), "l"(rsrc + b2 + 2 * v) : "memory");
                }
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    const int ln0 = blockIdx.x * PC2_NWARP + warp, lstep = gridDim.x * PC2_NWARP;
    prefetch(ln0);
    for (int ln = ln0; ln < op.nrows; ln += lstep) {
        const int row = reverse ? op.nrows - 1 - ln : ln;
        const size_t base = (size_t)row * np;
        const int crow = op.i_lo * op.nt + row;             // the coefficient planes are the global ones (slabs)
        const double F = __ldg(op.F + crow);
        // ---- the line's q and r (or b) were copied into the stage while the previous line was being solved; they
        // are read into registers and the NEXT line's copies are issued at once, so that its memory latency hides
        // behind this line's recurrences (a warp has one line in flight, 16 warps share an SM) ----
        double2 qn[H], rn[H];
        double dv[M], e[M], yd[M];
        asm volatile("cp.async.wait_group 0;" ::: "memory");
#pragma unroll
        for (int h = 0; h < H; h++) {
            const int v = lane + 32 * h;
            qn[h] = rn[h] = make_double2(0.0, 0.0);
            if (v < nv) { qn[h] = stq[h * 32 + lane]; rn[h] = str[h * 32 + lane]; }
        }
        prefetch(ln + lstep);
        const double2 *dT = reinterpret_cast<const double2 *>(pc.dinvT + (size_t)crow * 32 * M);
#pragma unroll
        for (int h = 0; h < H; h++) {
            const double2 t = __ldg(dT + h * 32 + lane);
            dv[2 * h] = t.x; dv[2 * h + 1] = t.y;
        }
        // ---- natural order: r' = r - alpha q (init: V.b - A x0), stored; staged for the chunk order ----
        double V2 = 0.0;
        if (INIT) V2 = __ldg(op.V2 + crow);
#pragma unroll
        for (int h = 0; h < H; h++) {
            const int v = lane + 32 * h;
            double2 rv = make_double2(0.0, 0.0);
            if (v < nv) {
                const size_t cell = base + 2 * v;
                if (INIT) {
                    const double bs0 = V2 * __ldg(op.vp + 2 * v) * rn[h].x, bs1 = V2 * __ldg(op.vp + 2 * v + 1) * rn[h].y;
                    rv.x = bs0 - qn[h].x;
                    rv.y = bs1 - qn[h].y;
                    acc[2] += bs0 * bs0 + bs1 * bs1;
                    st2(p0, cell, make_double2(0.0, 0.0));
                } else {
                    rv.x = fma(-alpha, qn[h].x, rn[h].x);
                    rv.y = fma(-alpha, qn[h].y, rn[h].y);
                }
                st2(rvec, cell, rv);
                acc[1] += rv.x * rv.x + rv.y * rv.y;
            }
            const int l = (2 * v) / M, u2 = v - l * H;      // chunk and pair index inside it
            buf[l * (S / 2) + u2] = rv;
        }
        // ---- e_k = c_k / piv_k ----
#pragma unroll
        for (int u = 0; u < M; u++) {
            const double c = -F * (UNIFORM ? pc.ip0 : ipc[u]);
            e[u] = (kbase + u < np - 1) ? c * dv[u] : 0.0;  // the last cell couples through the wrap entry only
        }
        const double wq = -F * ipw;                         // wrap entry w (np-1 <-> 0)
        const double dinv0 = __shfl_sync(0xffffffffu, dv[0], 0);
        __syncwarp();
        const double2 *my = buf + lane * (S / 2);
        const double wl = (wq * dinv0) * buf[0].x;          // (w / piv_0) y_0,  y_0 = r'_0
        const bool wlane = lane == lw;
        // ---- forward substitution: chunk map, warp scan, chunk again from the scanned incoming value ----
        double e_in = __shfl_up_sync(0xffffffffu, e[M - 1], 1);
        if (lane == 0) e_in = 0.0;
        {
            double Y = 0.0, P = 1.0, ep = e_in;
#pragma unroll
            for (int h = 0; h < H; h++) {
                const double2 rv = my[h];
                const double r0 = (wlane && 2 * h == uw) ? rv.x - wl : rv.x;
                const double r1 = (wlane && 2 * h + 1 == uw) ? rv.y - wl : rv.y;
                Y = fma(-ep, Y, r0); P = -ep * P; ep = e[2 * h];
                Y = fma(-ep, Y, r1); P = -ep * P; ep = e[2 * h + 1];
            }
#pragma unroll
            for (int off = 1; off < 32; off <<= 1) {        // inclusive scan of the affine maps, left to right
                const double Yo = __shfl_up_sync(0xffffffffu, Y, off), Po = __shfl_up_sync(0xffffffffu, P, off);
                if (lane >= off) { Y = fma(P, Yo, Y); P *= Po; }
            }
            double y = __shfl_up_sync(0xffffffffu, Y, 1);   // y of the cell before this chunk
            if (lane == 0) y = 0.0;
            ep = e_in;
#pragma unroll
            for (int h = 0; h < H; h++) {
                const double2 rv = my[h];
                const double r0 = (wlane && 2 * h == uw) ? rv.x - wl : rv.x;
                const double r1 = (wlane && 2 * h + 1 == uw) ? rv.y - wl : rv.y;
                y = fma(-ep, y, r0); yd[2 * h] = y * dv[2 * h]; ep = e[2 * h];
                y = fma(-ep, y, r1); yd[2 * h + 1] = y * dv[2 * h + 1]; ep = e[2 * h + 1];
            }
        }
        // ---- backward substitution, right to left: z_k = y_k / piv_k - e_k z_{k+1} ----
        {
            double zl = 0.0;                                // z_{np-1} = y_{np-1} / piv_{np-1}
#pragma unroll
            for (int u = 0; u < M; u++) if (u == uw) zl = yd[u];
            zl = __shfl_sync(0xffffffffu, zl, lw);
            if (lane == 0) yd[0] = fma(-(wq * dv[0]), zl, yd[0]);   // z_0 additionally - (w / piv_0) z_{np-1}
            double Y = 0.0, P = 1.0;
#pragma unroll
            for (int u = M - 1; u >= 0; u--) { Y = fma(-e[u], Y, yd[u]); P = -e[u] * P; }
#pragma unroll
            for (int off = 1; off < 32; off <<= 1) {        // inclusive scan, right to left
                const double Yo = __shfl_down_sync(0xffffffffu, Y, off), Po = __shfl_down_sync(0xffffffffu, P, off);
                if (lane + off < 32) { Y = fma(P, Yo, Y); P *= Po; }
            }
            double z = __shfl_down_sync(0xffffffffu, Y, 1); // z of the cell after this chunk
            if (lane == 31) z = 0.0;
#pragma unroll
            for (int u = M - 1; u >= 0; u--) { z = fma(-e[u], z, yd[u]); yd[u] = z; }
        }
        // ---- rho' += r'.z (chunk order), then z back to the natural order ----
        double2 *mine = buf + lane * (S / 2);
#pragma unroll
        for (int h = 0; h < H; h++) {
            const double2 rv = mine[h];
            acc[0] += rv.x * yd[2 * h] + rv.y * yd[2 * h + 1];
            mine[h] = make_double2(yd[2 * h], yd[2 * h + 1]);
        }
        __syncwarp();
        for (int v = lane; v < nv; v += 32) {
            const int l = (2 * v) / M, u2 = v - l * H;
            st2(zvec, base + 2 * v, buf[l * (S / 2) + u2]);
        }
        __syncwarp();                                       // the buffer is free for the next line
    }
    if (INIT) {
        double a3[3] = {acc[2], acc[1], acc[0]};            // bb, rr, rho
        if (grid_sum<PC2_NT, 3>(a3, part_base(w, rhs), w.pstride, &w.tickets[rhs * 4 + 0], sh) && threadIdx.x == 0)
            reduction_done<ROLE_INIT, 3>(w, rhs, a3, cond, use_cond);
    } else {
        double a2[2] = {acc[0], acc[1]};                    // rho', rr
        if (grid_sum<PC2_NT, 2>(a2, part_base(w, rhs), w.pstride, &w.tickets[rhs * 4 + 2], sh) && threadIdx.x == 0)
            reduction_done<ROLE_K2, 2>(w, rhs, a2, cond, use_cond);
    }
}

template <int M>
inline const void *pc2_line_func(bool uniform, bool init)
{
    if (init) return uniform ? (const void *)k_pc2_line<M, true, true> : (const void *)k_pc2_line<M, false, true>;
    return uniform ? (const void *)k_pc2_line<M, true, false> : (const void *)k_pc2_line<M, false, false>;
}
inline const void *pc2_line_pick(int M, bool uniform, bool init)
{
    switch (M) {
        case 4: return pc2_line_func<4>(uniform, init);
        case 8: return pc2_line_func<8>(uniform, init);
        case 12: return pc2_line_func<12>(uniform, init);
        case 16: return pc2_line_func<16>(uniform, init);
        case 24: return pc2_line_func<24>(uniform, init);
        default: return pc2_line_func<32>(uniform, init);
    }
}
inline int pc2_chunk(int np)            // 0: unsupported
{
    if (np < 4 || np > 1024) return 0;
    for (int M : {4, 8, 12, 16, 24, 32})     // the smallest chunk that covers the line: idle lanes cost bandwidth (np = 384 -> 12)
        if (32 * M >= np) return M;
    return 0;
}

}  // namespace mas

// common.cuh -- device-side types and the deterministic two-stage reduction shared by every kernel
// of the MAS PCG path (sm_100a).  Product code; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mas {

constexpr int MAX_RHS = 3;           // right-hand sides per batched solve: v_r, v_theta, v_phi
constexpr int MAX_SLABS = 16;        // r-slabs per slab group

// Operator as the kernels see it: 2-D (r,theta) coefficient planes + 1-D phi factors, built once
// from the 1-D metric arrays (PAPER.md:65 non-uniform logically
// rectangular mesh).  "row" = i*nt + j indexes a phi-row of np cells and every [nr][nt] plane.
// A slab sees `nr` LOCAL planes of its vectors; the coefficient planes are always the GLOBAL ones
// (O(nr*nt) doubles, replicated), indexed with the plane offset i_lo.
struct OpDev {
    int nr, nt, np, nv;          // local planes; nv = np/2 (double2 vectors per row)
    int nrows;                   // nr*nt local rows
    int uniform_phi;             // 1: dph_c, dph_f constant  => Dinv plane is valid
    int i_lo, nr_glob;           // global index of local plane 0; global plane count
    long long n;                 // local cells
    // dt-scaled planes, rewritten by set_dt
    const double *E;             // [nrows]      V2 + dt*(CRf[i]+CRf[i+1]+CT[j]+CT[j+1])   (diag, per unit vp)
    const double *F;             // [nrows]      dt*CP                                      (phi coupling)
    const double *AR;            // [(nr+1)*nt]  dt*CR, zero on both radial boundary faces  (off-diagonal)
    const double *AT;            // [nr*(nt+1)]  dt*CT, zero on both polar faces
    const double *Dinv;          // [nrows]      1/(vp*E + F*wp) when uniform_phi
    // dt-independent
    const double *V2;            // [nrows]      r_c^2 dr_c sin_c dth_c
    const double *vp;            // [np] dph_c
    const double *wp;            // [np] ip[k] + ip[k-1]
    const double *ip;            // [np] 1/dph_f[k]   (face k+1/2)
};

// Per-solve arguments, written by the host before the graph launch; kernels read them through a
// device pointer so that one instantiated CUDA graph serves every solve.
struct SolveArgs {
    const double *b[MAX_RHS];
    double *x[MAX_RHS];
    const double *x_lo, *x_hi;   // slab mode: the adjacent planes of x0 owned by the neighbour slabs (null otherwise)
    double rtol;
    int maxit;
    int nrhs;
};

// Iteration scalars of ONE right-hand side; live on the device for the whole loop (the host never sees
// them per iteration -- contrast PAPER.md:134-143 where each OpenACC reduction returns to the host).
struct State {
    double rho, sigma, alpha, beta, bb, rr;
    int k;                       // iterations done
    int active;                  // 1 while this right-hand side should continue
    int status;                  // MAS_OK / MAS_MAXIT / MAS_EBREAKDOWN
    int launches;                // loop kernels that actually did work (for mas_pcg_stats)
};

// Loop control shared by all right-hand sides of a solve
struct Ctl {
    int votes, any;              // per kernel: right-hand sides that have reported / that stay active
    int loop;                    // 1 while any right-hand side is active (what the host-chunk loop polls)
    int fault;                   // set by a kernel whose mbarrier wait timed out (protocol error -> MAS_ECUDA)
};

struct Work {                    // handle-owned vectors; right-hand side j at + j * vstride
    double *r, *p0, *p1, *q;     // p ping-pongs: iteration k reads p[k&1], writes p[(k+1)&1]
    double *z;                   // PC2 only: z = M^-1 r, written by the line kernel, read by K1 (null with PC1)
    long long vstride;
    double *partials;            // [MAX_RHS][PART_REGIONS][pstride]
    int pstride;                 // >= gridDim.x of every reducing kernel of the plan
    int hstride;                 // history entries per right-hand side
    double *hist;                // [MAX_RHS][hstride]
    State *st;                   // [MAX_RHS]
    unsigned *tickets;           // [MAX_RHS][4] last-block-done counters, one per kernel role (per slab in slab mode)
    Ctl *ctl;
    const SolveArgs *args;
    // slab mode (null / 0 otherwise): the adjacent planes of the neighbour slabs, and where a slab's kernel
    // leaves its partial sums for the combine step instead of finishing the scalar step itself
    const double *lo_r, *lo_p0, *lo_p1, *hi_r, *hi_p0, *hi_p1;
    const double *lo_z, *hi_z;   // PC2: the neighbours' adjacent planes of z
    double *slab_sums;           // [3][MAX_SLABS]
    int slab;
};

constexpr int PART_REGIONS = 3;      // partial-sum regions per right-hand side (the widest reduction: init's three sums)
constexpr int ST_OK = 0, ST_MAXIT = 1, ST_BREAKDOWN = -4;

__device__ __forceinline__ double *part_base(const Work &w, int rhs) { return w.partials + (size_t)rhs * PART_REGIONS * w.pstride; }

// 1/d for the point-Jacobi step z = r/d on meshes that are non-uniform in phi, where d = vp[k] E + F wp[k] differs from
// cell to cell and no reciprocal plane exists (uniform phi: the Dinv plane).  rcp.approx.ftz.f64 gives 20 good bits;
// two Newton steps x <- x + x (1 - d x) square the error twice: < 1 ulp of 1/d, so r * rcp_nr(d) is within ~1.5 ulp of
// the IEEE quotient -- the same class of difference as r * Dinv on uniform meshes (R6) -- at 5 DFMA-class
// instructions instead of the ~20 plus a slow-path branch of the IEEE division.  d is a diagonal entry of an SPD
// operator: positive, normal range.  Every kernel that forms z uses this one function, so K1's prologue, K2's sums
// and the init step see the same z bit for bit.
__device__ __forceinline__ double rcp_nr(double d)
{
    double x;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(d));
    x = fma(x, fma(-d, x, 1.0), x);
    x = fma(x, fma(-d, x, 1.0), x);
    return x;
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;   // xor butterfly: every lane performs the same commutative pair sums => same bits
}

// Fixed-shape block sum (warp butterflies, then warp 0 over the per-warp values).  Result valid
// in thread 0.  `sh` = >= 32 doubles of shared memory.  Deterministic: no atomics on data.
template <int NT>
__device__ __forceinline__ double block_sum(double v, double *sh)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    v = warp_sum(v);
    if (lane == 0) sh[w] = v;
    __syncthreads();
    double t = 0.0;
    if (w == 0) {
        t = lane < (NT + 31) / 32 ? sh[lane] : 0.0;
        t = warp_sum(t);
    }
    __syncthreads();
    return t;
}

// Stage 2: every block stores its NP partial sums at a FIXED slot
// (its blockIdx), then the block that arrives last sums all slots in a FIXED order.  Which
// block is last varies from run to run; the summation order does not => bit-reproducible.
// Returns true in ALL threads of the last block; totals valid in thread 0 only.
// `partials` holds NP regions of `pstride` doubles; the host sizes pstride >= gridDim.x.
template <int NT, int NP>
__device__ __forceinline__ bool grid_sum(double (&v)[NP], double *partials, int pstride, unsigned *ticket, double *sh)
{
    static_assert(NP <= PART_REGIONS, "widen PART_REGIONS");
    __shared__ int s_last;
    const int G = gridDim.x;
#pragma unroll
    for (int q = 0; q < NP; q++) {
        double t = block_sum<NT>(v[q], sh);
        if (threadIdx.x == 0) partials[(size_t)q * pstride + blockIdx.x] = t;
    }
    if (threadIdx.x == 0) {
        __threadfence();
        unsigned t = atomicAdd(ticket, 1u);
        s_last = (t == (unsigned)(G - 1));
    }
    __syncthreads();
    if (!s_last) return false;
    __threadfence();
#pragma unroll
    for (int q = 0; q < NP; q++) {
        double a = 0.0;
        for (int i = threadIdx.x; i < G; i += NT) a += __ldcg(&partials[(size_t)q * pstride + i]);
        v[q] = block_sum<NT>(a, sh);
    }
    if (threadIdx.x == 0) *ticket = 0u;     // re-arm for the next launch
    return true;
}

}  // namespace mas

/*
 * mas_pcg.h -- C ABI of the B200-native MAS PCG hot path.
 *
 * What it is: the point-Jacobi (PC1) preconditioned conjugate-gradient solve of the implicit,
 * symmetric positive definite 7-point finite-difference operator of the MAS zero-beta time step
 * on MAS's non-uniform, logically rectangular spherical (r, theta, phi) mesh, in fp64
 * (Sec. 2.2: "non-uniform logically-rectangular staggered grid using finite
 * difference", "preconditioned conjugate gradient (PCG) solves", "PC1 uses the inverse diagonal
 * of the matrix (point-Jacobi)"; eq. (1): the implicit terms (1/rho) div(nu rho grad v)
 * and (1/rho) div(S rho grad dv/dt); Sec. 4.1: "sparse matrix-vector products
 * (essentially stencil operations), basic array operations, and dot products"; FP64).
 *
 * The discrete operator (the paper does not print it; reading R1):
 *   A_phys = I - dt * (1/V) * [finite-volume flux divergence of nu grad],
 *   A_sym  = diag(V) A_phys  (symmetric, "our symmetric matrices"),
 *   V_ijk  = r_c[i]^2 dr_c[i] sin_c[j] dth_c[j] dph_c[k].
 * mas_pcg_solve solves A_phys x = b for the caller (internally A_sym x = V.b).
 *
 * All vectors are fp64, C-contiguous [nr][nt][np] with phi fastest, 16-byte aligned.
 * Every entry point returns an int status (below); no exceptions, no aborts, no output.
 * There is no CPU fallback: without a CUDA device every call that needs one returns MAS_ECUDA.
 */
#ifndef MAS_PCG_H
#define MAS_PCG_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mas_pcg mas_pcg_t;              /* opaque; owns every device workspace            */

typedef struct { int nr, nt, np; } mas_grid_t; /* cell counts; nr,nt >= 1, np >= 2 and even      */

/* 1-D metric arrays, HOST pointers, copied at create (caller may free them afterwards). */
typedef struct {
    const double *r_c,  *dr_c;   /* [nr]   cell-centre radius, cell width                                   */
    const double *r_f,  *dr_f;   /* [nr+1] face radius; centre-to-centre distance across face i, and the
                                           centre-to-boundary-face distance for i = 0 and i = nr            */
    const double *sin_c, *dth_c; /* [nt]   sin(theta_c), cell width in theta                                */
    const double *sin_f, *dth_f; /* [nt+1] sin(theta_f) (polar faces are forced to zero area regardless of
                                           the value passed), centre distance; dth_f[0], dth_f[nt] unused   */
    const double *dph_c;         /* [np]   cell width in phi                                                */
    const double *dph_f;         /* [np]   distance centre k -> centre (k+1) mod np (periodic)              */
} mas_metric_t;

enum { MAS_BC_DIRICHLET = 0, MAS_BC_NEUMANN = 1 };  /* radial faces only                           */
typedef struct { int r_inner, r_outer; } mas_bc_t;  /* theta: polar axis (zero-area face); phi: periodic */

/* viscosity-like coefficient nu: kind 0 = scalar v[0]; kind 1 = HOST plane
 * [nr][nt] of cell-centre values.  Face value = arithmetic mean of the two cells (R1). */
typedef struct { int kind; const double *v; } mas_nu_t;

enum {
    MAS_OK = 0,          /* converged: ||r_k||_2 / ||V.b||_2 <= rtol (or exact zero residual)          */
    MAS_MAXIT = 1,       /* ran maxit iterations without meeting rtol; x is the last iterate.  The
                            normal return of fixed-iteration runs (rtol = 0)                            */
    MAS_EINVAL = -1,     /* bad dimension / null pointer / non-positive width / dt < 0 / nu <= 0 /
                            rtol < 0 / maxit < 0 / misaligned vector                                    */
    MAS_ENOMEM = -2,     /* host or device allocation failed                                            */
    MAS_ECUDA = -3,      /* a CUDA runtime call failed (no device, launch error, ...)                   */
    MAS_EBREAKDOWN = -4  /* p.Ap <= 0 or a non-finite scalar: the operator is not SPD for these inputs  */
};

/* Build the operator for (grid, metric, dt, nu, boundary kinds) and allocate all workspaces
 * (r, p, q, reduction partials, residual history, coefficient planes) on the CURRENT device.
 * Host arrays are read during the call only.  *out is set to NULL on failure. */
int mas_pcg_create(const mas_grid_t *grid, const mas_metric_t *metric, double dt,
                   const mas_nu_t *nu, const mas_bc_t *bc, mas_pcg_t **out);

/* Change dt (BASELINE.json config 5 varies it per step).  Asynchronous on `stream`
 * (a cudaStream_t passed as void*; NULL = default stream). */
int mas_pcg_set_dt(mas_pcg_t *h, double dt, void *stream);

/* Solve A_phys x = b by Jacobi-PCG (R3 = textbook PCG, ref. [22]).
 *   b_dev   : DEVICE, N doubles, never written.
 *   x_dev   : DEVICE, N doubles; in = initial guess x0, out = last iterate.
 *   rtol    : stop when ||r_k||_2 / ||V.b||_2 <= rtol (recurrence residual of the symmetric system).
 *   maxit   : iteration cap; with rtol = 0 exactly maxit iterations run.
 *   stream  : all work is enqueued on it; the call synchronises it ONCE, at the end, to return
 *             the count and history.  The iteration loop itself never returns to the host.
 *   iters_out    : HOST, number of iterations k performed (may be NULL).
 *   reshist_host : HOST, NULL or >= maxit+1 doubles; receives hist[0..k], hist[j] = ||r_j||/||V.b||.
 * One solve in flight per handle. */
int mas_pcg_solve(mas_pcg_t *h, const double *b_dev, double *x_dev, double rtol, int maxit,
                  void *stream, int *iters_out, double *reshist_host);

/* Same solve with HOST vectors: copies b and x0 to device buffers owned by the handle, solves,
 * copies x back.  b_host/x_host: N doubles each (pinned memory makes the copies faster). */
int mas_pcg_solve_host(mas_pcg_t *h, const double *b_host, double *x_host, double rtol, int maxit,
                       void *stream, int *iters_out, double *reshist_host);

/* y = A_sym x (the matrix-free stencil alone; asynchronous on `stream`).  x_dev != y_dev. */
int mas_pcg_apply(mas_pcg_t *h, const double *x_dev, double *y_dev, void *stream);

/* Measurement aid (bench.py roofline): runs `nit` PCG iterations (rtol = 0) from x0 = x_dev with the
 * kernels launched one by one and CUDA events recorded around each on `stream`; synchronises.
 * ms_out (HOST, 4 doubles) = { mean K1, mean K2, min K1, min K2 } kernel durations in milliseconds
 * (K1 = fused matvec, K2 = fused vector kernel).  1 <= nit <= 256.  x_dev is overwritten. */
int mas_pcg_profile(mas_pcg_t *h, const double *b_dev, double *x_dev, int nit, void *stream, double *ms_out);

/* Measurement aid (bench.py): *ms_out (HOST) = best sustained time per launch, over `reps` back-to-back
 * launches, of a trivial LINEAR kernel with the DRAM read/write mix of K1 (which = 6: three N-vectors read,
 * three written, one of them in place) or K2 (which = 3: two read, one written in place) and none of their
 * structure: what the memory system sustains for that mix.  Clobbers the handle's workspaces. */
int mas_pcg_mix_probe(mas_pcg_t *h, int which, int reps, void *stream, double *ms_out);

/* Fills HOST array out[8] with counters of the last solve:
 *   [0] kernels launched inside the iteration loop, [1] kernels launched outside it,
 *   [2] loop mode used (1 = CUDA-graph WHILE node, 0 = host-driven chunks, 2 = one persistent cooperative kernel),
 *   [3] algorithmic bytes per cell per iteration of the kernels in use,
 *   [4] doubles per cell K1 moves, [5] doubles per cell K2 moves,
 *   [6] grid size of the persistent kernel (0 if not used), [7] 1 if the loop body used programmatic (PDL) edges. */
int mas_pcg_stats(const mas_pcg_t *h, long long *out);

/* Tuning / debugging knob, takes effect at the next solve.  name in
 *   "loop_mode" (0 host chunks, 1 graph while), "variant" (K1: 0 baseline, 1 marching, 2 wide marching with cp.async,
 *   3 wide marching with TMA bulk copies + mbarriers = default),
 *   "tile" (tile configuration of the variant), "ci" (r-chunk length, 0 = automatic),
 *   "xfuse" (variant 2 only; 1: x-update fused into K1, 72 B/cell/iteration; 0: in K2, 80 B; variant 3 is always
 *   fused), "serpentine" (K2 sweeps
 *   backward), "apply_variant" (1 marching stencil kernel, 0 baseline), "stencil_tile" (0..5 cp.async, 6..11 TMA),
 *   "qrecompute" (variant 2 only: 64 B), "k2r_tile",
 *   "unroll" (PCG iterations per WHILE trip of the graph loop, 1..16), "pdl" (programmatic dependent launch
 *   edges inside the loop body; default 0: measured slower),
 *   "persistent" (small meshes: whole solve in one cooperative kernel; 0 off, 1 whenever it fits, 2 auto).
 * Unknown name or value: MAS_EINVAL. */
int mas_pcg_set_option(mas_pcg_t *h, const char *name, int value);

/* ---- NEXT-1: the explicit alternative for the viscosity term, "a Runge-Kutta Legendre super
 * time-stepping (STS) scheme [21]" (~200 sub-steps per step; the fastest GPU
 * choice).  M u = -(1/V) sum_faces G_f (u - u_nb) is the FD form of div(nu grad u), so that
 * A_phys = I - dt M.  Scheme: RKL2 of the paper's ref. [21], restated in DESIGN.md R7. ---- */

/* y = M u (asynchronous on `stream`); u_dev != y_dev, DEVICE vectors of N doubles. */
int mas_pcg_lop(mas_pcg_t *h, const double *u_dev, double *y_dev, void *stream);

/* *out = Gershgorin bound on the spectral radius of M (HOST double), computed at create. */
int mas_pcg_lambda_max(const mas_pcg_t *h, double *out);

/* Smallest stage count s >= 2 for which one RKL2 super-step of size tau is stable:
 * tau <= (s^2 + s - 2)/4 * 2/lambda_max. */
int mas_sts_stages(const mas_pcg_t *h, double tau, int *s_out);

/* Advance du/dt = M u by ONE RKL2 super-step of size tau with s >= 2 stages, in place in u_dev (DEVICE).
 * s kernel launches on `stream`, asynchronous.  Uses the handle's PCG workspaces as stage buffers, so it
 * must not overlap a solve on the same handle. */
int mas_sts_advance(mas_pcg_t *h, double *u_dev, double tau, int s, void *stream);

void mas_pcg_destroy(mas_pcg_t *h);            /* NULL is allowed                                 */

const char *mas_pcg_strerror(int status);      /* static string, never NULL                       */

#ifdef __cplusplus
}
#endif
#endif /* MAS_PCG_H */

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
 * A handle remembers the device it was created on; every call switches to that device for its own
 * duration, whatever the caller's current device is.
 *
 * Measurement probes used by bench.py are NOT here: see mas_pcg_debug.h (a separate library).
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
                            rtol < 0 / maxit < 0 / misaligned or aliased vector                         */
    MAS_ENOMEM = -2,     /* host or device allocation failed                                            */
    MAS_ECUDA = -3,      /* a CUDA runtime call failed (no device, launch error, ...), or a kernel
                            reported a protocol fault (an mbarrier wait that timed out)                 */
    MAS_EBREAKDOWN = -4, /* p.Ap <= 0, or a non-finite scalar (||V.b||^2, ||r||^2, r.z, p.Ap): the
                            operator is not SPD for these inputs, or b / x0 hold NaN / Inf.  x is the
                            last iterate (x0 if no iteration completed); iters_out and the history
                            are valid                                                                   */
    MAS_ETOOBIG = -5     /* mas_pcg_residual_static only: the mesh has more than MAS_PCG_STATIC_MAX_CELLS cells  */
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
 *   stream  : all work is enqueued on it; the call synchronises it at the end, to return the count
 *             and history (once; a second time only when ||V.b|| = 0 and x has to be zeroed, and
 *             mas_pcg_solve_host once more after copying x back).  The iteration loop itself never
 *             returns to the host.
 *   iters_out    : HOST, number of iterations k performed (may be NULL).
 *   reshist_host : HOST, NULL or >= maxit+1 doubles; receives hist[0..k], hist[j] = ||r_j||/||V.b||.
 * One solve in flight per handle. */
int mas_pcg_solve(mas_pcg_t *h, const double *b_dev, double *x_dev, double rtol, int maxit,
                  void *stream, int *iters_out, double *reshist_host);

/* Same solve with HOST vectors: copies b and x0 to device buffers owned by the handle, solves,
 * copies x back.  b_host/x_host: N doubles each (pinned memory makes the copies faster). */
int mas_pcg_solve_host(mas_pcg_t *h, const double *b_host, double *x_host, double rtol, int maxit,
                       void *stream, int *iters_out, double *reshist_host);

/* Batched solve: nrhs <= 3 right-hand sides that share the operator -- PAPER.md:50 eq. (1):
 * the implicit terms act on the vector v, whose three components share one coefficient set.  By definition these
 * are nrhs INDEPENDENT textbook solves (own alpha, beta, iteration count, status and history each), run by ONE set
 * of kernel launches per iteration: the right-hand side is the second grid dimension, a right-hand side that has
 * converged drops out, the loop ends when all have.  A batched solve always runs the streaming K1 / K2 kernels, and
 * its results are bit-identical to nrhs calls of mas_pcg_solve THAT RUN THE SAME KERNELS: option "persistent" = 0, or
 * a mesh too large for the one-kernel solve, or PC2.  With the default "persistent" = 1 a single solve of a small
 * mesh runs in the cooperative kernel, whose reductions add in another order: the two then agree to rounding (the
 * history within 1e-10 relative, x within 1e-9, as against the oracle), not bit for bit.
 *   b_dev, x_dev  : HOST arrays of nrhs DEVICE pointers (N doubles each; all distinct).
 *   iters_out     : HOST, nrhs ints (may be NULL);  status_out: HOST, nrhs ints (MAS_OK / MAS_MAXIT /
 *                   MAS_EBREAKDOWN per right-hand side; may be NULL).
 *   reshist_host  : HOST, NULL or nrhs * (maxit + 1) doubles; right-hand side j's history starts at
 *                   reshist_host + j * (maxit + 1).
 * Returns the most severe per-right-hand-side status (negative before MAS_MAXIT before MAS_OK), or an error. */
int mas_pcg_solve_multi(mas_pcg_t *h, int nrhs, const double *const *b_dev, double *const *x_dev, double rtol,
                        int maxit, void *stream, int *iters_out, int *status_out, double *reshist_host);

/* y = A_sym x (the matrix-free stencil alone; asynchronous on `stream`).  x_dev != y_dev. */
int mas_pcg_apply(mas_pcg_t *h, const double *x_dev, double *y_dev, void *stream);

/* Fills HOST array out[8] with counters of the last solve:
 *   [0] kernels launched inside the iteration loop, [1] kernels launched outside it,
 *   [2] loop mode used (1 = CUDA-graph WHILE node, 0 = host-driven chunks, 2 = one persistent cooperative kernel),
 *   [3] algorithmic bytes per cell per iteration of the kernels in use (72 default, 64 with "qrecompute", 88 with PC2),
 *   [4] doubles per cell K1 moves, [5] doubles per cell K2 moves,
 *   [6] grid size of the persistent kernel (0 if not used; slab groups: the number of slabs),
 *   [7] 1 if a cooperative launch was refused and the handle fell back to the streaming loop. */
int mas_pcg_stats(const mas_pcg_t *h, long long *out);

/* The paper's two "communication-free preconditioning options" (Sec. 2.2):
 *   MAS_PC1  point-Jacobi, "the inverse diagonal of the matrix" (the default);
 *   MAS_PC2  "a block-Jacobi using a zero-fill incomplete LU factorization [22]".  Reading
 *            (R8, not the paper's words): block Jacobi over non-overlapping boxes of bi x bj x bk cells,
 *            ILU(0) of A_sym restricted to each box, natural ordering.  PAPER.md:80: 100-200 iterations against ~550 with PC1; the
 *            authors kept it on the CPU because its triangular solves do not vectorise.
 * On the GPU the boxes are the phi lines: bi = bj = 1 and bk = 0 (or >= np) = the whole periodic line, wrap coupling
 * included; any other box shape returns MAS_EINVAL (the oracle covers general boxes and shows the line boxes within
 * 2 iterations of the undivided factorisation on the synthetic meshes).  4 <= np <= 1024.  The factors follow dt:
 * mas_pcg_set_dt refactors.  mas_pcg_solve_multi and slab groups (mas_pcg_slabs_set_preconditioner) work.
 * Synchronous: the factorisation runs on the default stream and the call returns after cudaDeviceSynchronize, so it is
 * ordered against work on every stream, blocking or not (a set-up call, not one for the step loop; mas_pcg_set_dt is
 * the in-loop way to refactor, on the caller's stream). */
enum { MAS_PC1 = 1, MAS_PC2 = 2 };
int mas_pcg_set_preconditioner(mas_pcg_t *h, int kind, int bi, int bj, int bk);

/* Tuning knob, takes effect at the next solve.  name in
 *   "loop_mode"   0 host-driven chunks of 16 iterations, 1 CUDA-graph WHILE loop (default);
 *   "persistent"  1 (default): meshes whose per-cell state fits in the SMs' shared memory are solved by ONE
 *                 cooperative kernel, whatever loop_mode says; 0: always the streaming loop;
 *   "qrecompute"  0 (default): 72 B/cell/iteration, q stored by K1 and streamed by K2; 1: 64 B -- K1 does not store q,
 *                 K2 recomputes it with the stencil kernel (fewer bytes, more instructions: measured slower);
 *   "tile"        K1 tile configuration (0..6; -1 = automatic, the default), "k2r_tile" / "stencil_tile" (0..5) the stencil kernel's tile for
 *                 K2R / for apply and RKL2 stages, "ci" r-chunk length of the marching kernels (0 = automatic, else 2..32);
 *   "serpentine"  1 (default): K2 sweeps the mesh backward (L2 reuse across K1 -> K2 -> K1);
 *   "unroll"      PCG iterations per WHILE trip of the graph loop (1..16, default 4);
 *   "l2_first_x"  1: x (read once and written once per iteration, never reused inside it) is streamed with the L2
 *                 evict_first priority so that it does not displace r and p on meshes whose vectors fit in L2; 0 (default).
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

/* ---- Residual check for callers that must not allocate device memory. ----
 *
 * Some users of this library cannot call cudaMalloc once their set-up is over: a time-stepping code that keeps every
 * field resident on the GPU (as the paper's does) and has sized its arrays or its own pool to fill
 * the card, so a later request simply fails; a process held to a fixed device-memory limit; or the inside of a step
 * loop where cudaMalloc / cudaFree are unaffordable because they stall the whole device and with it every other
 * stream.  mas_pcg_solve does not suit them: it may allocate on the way (a longer history, more right-hand sides, a
 * graph for a shape it has not seen).  This call never allocates -- no cudaMalloc, no cudaFree, no library routine
 * that allocates -- and it needs no workspace from the handle.  The handle itself must of course have been created
 * earlier, while allocating was still possible.
 *
 * What it computes (one kernel, the init step S1 of the solve applied to the caller's vectors):
 *     r = V.b - ax                 with ax = A_sym x from mas_pcg_apply (which needs no scratch memory either),
 *     sums[0] = ||V.b||^2,  sums[1] = ||r||^2,  sums[2] = r.D^-1 r     (D = diag(A_sym), whatever preconditioner is set),
 * so sqrt(sums[1] / sums[0]) is the TRUE relative residual of x, the quantity hist[] of mas_pcg_solve tracks through
 * the recurrence.  The sums are the deterministic two-stage reduction of the solve: the same
 * inputs give the same bits on every run.
 *   b_dev, ax_dev : DEVICE, N doubles each, 16-byte aligned, not written.
 *   r_dev         : DEVICE, N doubles, 16-byte aligned; may be the same buffer as ax_dev (in place), not b_dev.
 *   sums_dev      : DEVICE, 3 doubles, written by the kernel; read them after synchronising `stream`.
 *   stream        : everything is enqueued on it (one 256-byte memset node and one kernel); nothing synchronises.
 *
 * The scratch the reduction needs (per-block partial sums, an arrival counter) lives in a fixed 98 560-byte array
 * inside the library image.  Consequences:
 *   - Limit: N <= MAS_PCG_STATIC_MAX_CELLS (2^25 = 256 x 256 x 512, BASELINE.json config 4).  A larger mesh returns
 *     MAS_ETOOBIG and nothing is launched.
 *   - Every GPU that loads this library holds those 98 560 bytes until the process exits.
 *   - All calls on one device -- from any handle, any thread, any stream -- share the one array.  Two calls whose
 *     kernels may overlap on the GPU race on it and return garbage: keep calls on one stream, or order them with
 *     events.  The array keeps the previous call's contents; the call clears the part that has to start at zero.
 *   - The first call on each device looks up the array's device address (and may make the driver load the module
 *     there).  Make that first call during set-up, before any stream capture is begun; later calls on that device
 *     only enqueue the memset and the kernel.
 * Returns MAS_OK once enqueued; MAS_EINVAL (null / misaligned / overlapping pointers), MAS_ETOOBIG, MAS_ECUDA. */
#define MAS_PCG_STATIC_MAX_CELLS 33554432LL
int mas_pcg_residual_static(mas_pcg_t *h, const double *b_dev, const double *ax_dev, double *r_dev,
                            double *sums_dev, void *stream);

void mas_pcg_destroy(mas_pcg_t *h);            /* NULL is allowed                                 */

const char *mas_pcg_strerror(int status);      /* static string, never NULL                       */

/* ---- NEXT-3: r-slab decomposition (Sec. 4.3: domain split, one rank per GPU; PAPER.md:177, 183:
 * the scaling loss past one node came from host-staged halo exchange).  The mesh is split along r into nslab slabs,
 * slab s owning the planes [i_split[s], i_split[s+1]); each slab has its own vectors, as one rank per GPU would.
 * The kernels read the neighbour slab's boundary plane of r, p and x0 straight through a pointer (a peer mapping
 * over NVLink on a real node): per matvec one plane of nt*np doubles per neighbour, no halo kernel or staging
 * buffer; the two scalar reductions per iteration add the slabs' partial sums in slab order.  The undivided solve
 * is the definition: iterates agree with mas_pcg_solve up to the rounding order of the sums.
 * This library drives all slabs from ONE process on ONE device; that is the form that can be tested with one GPU,
 * and it is unmeasured on multi-GPU hardware. ---- */
typedef struct mas_pcg_slabs mas_pcg_slabs_t;

/* grid, metric, nu, bc describe the WHOLE mesh.  i_split: HOST, nslab + 1 increasing plane indices, i_split[0] = 0,
 * i_split[nslab] = nr; 1 <= nslab <= 16. */
int mas_pcg_slabs_create(const mas_grid_t *grid, const mas_metric_t *metric, double dt, const mas_nu_t *nu,
                         const mas_bc_t *bc, int nslab, const int *i_split, mas_pcg_slabs_t **out);
int mas_pcg_slabs_set_dt(mas_pcg_slabs_t *g, double dt, void *stream);
/* as mas_pcg_set_preconditioner: with PC2 every slab preconditions its own phi lines (they have no radial coupling) and
 * K1 reads the neighbours' adjacent planes of z = M^-1 r through pointers, as it reads their planes of r with PC1 */
int mas_pcg_slabs_set_preconditioner(mas_pcg_slabs_t *g, int kind, int bi, int bj, int bk);
/* same names as mas_pcg_set_option (except "persistent") */
int mas_pcg_slabs_set_option(mas_pcg_slabs_t *g, const char *name, int value);
/* b_dev, x_dev: HOST arrays of nslab DEVICE pointers; slab s's vectors hold its own planes only,
 * (i_split[s+1] - i_split[s]) * nt * np doubles.  Other arguments as mas_pcg_solve. */
int mas_pcg_slabs_solve(mas_pcg_slabs_t *g, const double *const *b_dev, double *const *x_dev, double rtol, int maxit,
                        void *stream, int *iters_out, double *reshist_host);
int mas_pcg_slabs_stats(const mas_pcg_slabs_t *g, long long *out);
void mas_pcg_slabs_destroy(mas_pcg_slabs_t *g);

#ifdef __cplusplus
}
#endif
#endif /* MAS_PCG_H */

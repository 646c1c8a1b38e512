/*
 * mas_pcg_ref.c -- ORACLE.  Test infrastructure, not product code.
 *
 * A plain, slow, single-threaded C99 statement of what the MAS PCG hot path computes: the
 * point-Jacobi (PC1) preconditioned conjugate-gradient solve of the implicit SPD 7-point
 * finite-difference operator on MAS's non-uniform, logically rectangular spherical mesh
 * (Sec. 2.2 "non-uniform logically-rectangular ... finite difference", "PCG ...
 * PC1 uses the inverse diagonal of the matrix (point-Jacobi)"; Sec. 4.1 "sparse
 * matrix-vector products (essentially stencil operations), basic array operations, and dot
 * products"; eq. (1) for the operator's form  (1/rho) div(nu rho grad v)).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load this library.  It shares no source, header, table or helper with the CUDA path
 * (paper_1811_02605_b200/csrc) and includes none of its files.
 *
 * The paper never writes the discrete operator.  The reading used here is
 * DESIGN.md R1: finite-volume flux form on cell centres, which is what makes the matrix
 * symmetric on a non-uniform mesh ("our symmetric matrices").
 *
 *   cell (i,j,k) has volume            V   = r_c[i]^2 dr_c[i] sin_c[j] dth_c[j] dph_c[k]
 *   radial face i (between i-1 and i)  G_r = nu_f r_f[i]^2 sin_c[j] dth_c[j] dph_c[k] / dr_f[i]
 *   theta  face j (between j-1 and j)  G_t = nu_f dr_c[i] sin_f[j] dph_c[k] / dth_f[j]
 *   phi    face k (between k and k+1)  G_p = nu   dr_c[i] dth_c[j] / (sin_c[j] dph_f[k])
 *
 *   (A_sym u)_c = V_c u_c + dt * sum over the 6 faces f of c of  G_f (u_c - u_neighbour(f))
 *
 * which is V times the finite-difference form of  u - dt div(nu grad u)  in spherical
 * coordinates (area/distance per face; the r's cancel on theta faces).  Boundaries:
 *   radial Dirichlet: homogeneous value ON the boundary face, neighbour value 0, distance
 *                     dr_f[0] = r_c[0]-r_f[0]  (Q4);  radial Neumann: G = 0 on that face;
 *   polar axis: sin_f = 0 exactly, so G_t = 0 (Q5);  phi: periodic index wrap.
 *   nu on a face = arithmetic mean of the two cell values; a boundary face takes its cell's (Q3).
 *
 * The system solved (R2): the caller's A_phys x = b with A_phys = diag(V)^-1 A_sym;
 * internally A_sym x = b_s, b_s = V.b; residuals, norms and the stopping test live in the
 * symmetric system.  Further down: the RKL2 super time stepping of the viscosity term (NEXT-1) and
 * the paper's second preconditioner PC2, block-Jacobi ILU(0) (NEXT-4), each with its own header.
 * Parity status: pinned by tests/test_oracle_*.py (dense LU, manufactured
 * solution, symmetry/SPD, Krylov optimality, closed forms, continuum consistency, Legendre stability
 * polynomial, the ILU(0) defining property, exactness on tridiagonal operators, randomised meshes;
 * 22 committed source mutations).  "Parity unpinned": the face-nu mean (Q3: a declared reading; the
 * harmonic mean survives every mathematical pin) and what is tied to the paper's own run (its mesh,
 * nu, RHS, its 70/550 and 100-200 iteration counts, its PC2 domains): the data are not available.
 *
 * Sums are plain index-order loops with a long double accumulator (Q22).  No blocking, no
 * fusion, no reordering.  Layout: [nr][nt][np], phi fastest.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

enum { REF_BC_DIRICHLET = 0, REF_BC_NEUMANN = 1 };
enum { REF_OK = 0, REF_MAXIT = 1, REF_EINVAL = -1, REF_ENOMEM = -2, REF_EBREAKDOWN = -4 };

typedef struct ref_op {
    int nr, nt, np;
    double dt;
    /* face conductances without their phi factor, tabulated once from the 1-D metric arrays */
    double *gr;   /* [(nr+1)][nt]  nu_f r_f^2 sin_c dth_c / dr_f ; 0 on Neumann boundary faces */
    double *gt;   /* [nr][(nt+1)]  nu_f dr_c sin_f / dth_f      ; 0 on the polar faces          */
    double *gp;   /* [nr][nt]      nu   dr_c dth_c / sin_c                                    */
    double *v2;   /* [nr][nt]      r_c^2 dr_c sin_c dth_c                                      */
    double *dph_c, *dph_f; /* [np] */
} ref_op;

static double nu_at(int kind, const double *nu, int nt, int i, int j)
{
    return kind == 0 ? nu[0] : nu[(size_t)i * nt + j];
}

void mas_ref_destroy(ref_op *op)
{
    if (!op) return;
    free(op->gr); free(op->gt); free(op->gp); free(op->v2); free(op->dph_c); free(op->dph_f);
    free(op);
}

/* Build the operator of DESIGN.md R1 from the 1-D metric arrays (all HOST pointers). */
ref_op *mas_ref_create(int nr, int nt, int np,
                       const double *r_c, const double *dr_c, const double *r_f, const double *dr_f,
                       const double *sin_c, const double *dth_c, const double *sin_f, const double *dth_f,
                       const double *dph_c, const double *dph_f,
                       double dt, int nu_kind, const double *nu, int bc_inner, int bc_outer)
{
    if (nr < 1 || nt < 1 || np < 1 || dt < 0.0) return NULL;
    ref_op *op = (ref_op *)calloc(1, sizeof(ref_op));
    if (!op) return NULL;
    op->nr = nr; op->nt = nt; op->np = np; op->dt = dt;
    op->gr = (double *)calloc((size_t)(nr + 1) * nt, sizeof(double));
    op->gt = (double *)calloc((size_t)nr * (nt + 1), sizeof(double));
    op->gp = (double *)calloc((size_t)nr * nt, sizeof(double));
    op->v2 = (double *)calloc((size_t)nr * nt, sizeof(double));
    op->dph_c = (double *)malloc(sizeof(double) * np);
    op->dph_f = (double *)malloc(sizeof(double) * np);
    if (!op->gr || !op->gt || !op->gp || !op->v2 || !op->dph_c || !op->dph_f) { mas_ref_destroy(op); return NULL; }
    memcpy(op->dph_c, dph_c, sizeof(double) * np);
    memcpy(op->dph_f, dph_f, sizeof(double) * np);

    for (int i = 0; i < nr; i++)
        for (int j = 0; j < nt; j++) {
            op->v2[(size_t)i * nt + j] = r_c[i] * r_c[i] * dr_c[i] * sin_c[j] * dth_c[j];
            op->gp[(size_t)i * nt + j] = nu_at(nu_kind, nu, nt, i, j) * dr_c[i] * dth_c[j] / sin_c[j];
        }
    /* radial faces i = 0..nr */
    for (int i = 0; i <= nr; i++)
        for (int j = 0; j < nt; j++) {
            double nuf;
            if (i == 0)        nuf = nu_at(nu_kind, nu, nt, 0, j);
            else if (i == nr)  nuf = nu_at(nu_kind, nu, nt, nr - 1, j);
            else               nuf = 0.5 * (nu_at(nu_kind, nu, nt, i - 1, j) + nu_at(nu_kind, nu, nt, i, j));
            double g = nuf * r_f[i] * r_f[i] * sin_c[j] * dth_c[j] / dr_f[i];
            if (i == 0 && bc_inner == REF_BC_NEUMANN) g = 0.0;
            if (i == nr && bc_outer == REF_BC_NEUMANN) g = 0.0;
            op->gr[(size_t)i * nt + j] = g;
        }
    /* theta faces j = 0..nt ; the polar faces j = 0 and j = nt have zero area */
    for (int i = 0; i < nr; i++)
        for (int j = 0; j <= nt; j++) {
            double g = 0.0;
            if (j > 0 && j < nt) {
                double nuf = 0.5 * (nu_at(nu_kind, nu, nt, i, j - 1) + nu_at(nu_kind, nu, nt, i, j));
                g = nuf * dr_c[i] * sin_f[j] / dth_f[j];
            }
            op->gt[(size_t)i * (nt + 1) + j] = g;
        }
    return op;
}

void mas_ref_set_dt(ref_op *op, double dt) { op->dt = dt; }

/* the six face conductances of cell (i,j,k), phi factors included */
static void faces(const ref_op *op, int i, int j, int k, double g[6])
{
    const int nt = op->nt, np = op->np;
    const int km = (k + np - 1) % np;
    g[0] = op->gr[(size_t)i * nt + j] * op->dph_c[k];             /* face to i-1 (or inner boundary) */
    g[1] = op->gr[(size_t)(i + 1) * nt + j] * op->dph_c[k];       /* face to i+1 (or outer boundary) */
    g[2] = op->gt[(size_t)i * (nt + 1) + j] * op->dph_c[k];       /* face to j-1 (or pole: 0)        */
    g[3] = op->gt[(size_t)i * (nt + 1) + j + 1] * op->dph_c[k];   /* face to j+1 (or pole: 0)        */
    g[4] = op->gp[(size_t)i * nt + j] / op->dph_f[km];            /* face to k-1 (periodic)          */
    g[5] = op->gp[(size_t)i * nt + j] / op->dph_f[k];             /* face to k+1 (periodic)          */
}

static double volume(const ref_op *op, int i, int j, int k)
{
    return op->v2[(size_t)i * op->nt + j] * op->dph_c[k];
}

void mas_ref_volume(const ref_op *op, double *V)
{
    for (int i = 0; i < op->nr; i++)
        for (int j = 0; j < op->nt; j++)
            for (int k = 0; k < op->np; k++)
                V[((size_t)i * op->nt + j) * op->np + k] = volume(op, i, j, k);
}

/* d = diag(A_sym) = V + dt * (sum of the six face conductances) */
void mas_ref_diag(const ref_op *op, double *d)
{
    double g[6];
    for (int i = 0; i < op->nr; i++)
        for (int j = 0; j < op->nt; j++)
            for (int k = 0; k < op->np; k++) {
                faces(op, i, j, k, g);
                d[((size_t)i * op->nt + j) * op->np + k] =
                    volume(op, i, j, k) + op->dt * (g[0] + g[1] + g[2] + g[3] + g[4] + g[5]);
            }
}

/* y = A_sym u, flux-difference form; a missing neighbour across a Dirichlet face has value 0 */
void mas_ref_apply(const ref_op *op, const double *u, double *y)
{
    const int nr = op->nr, nt = op->nt, np = op->np;
    double g[6];
    for (int i = 0; i < nr; i++)
        for (int j = 0; j < nt; j++)
            for (int k = 0; k < np; k++) {
                const size_t c = ((size_t)i * nt + j) * np + k;
                const int kp = (k + 1) % np, km = (k + np - 1) % np;
                faces(op, i, j, k, g);
                const double uc = u[c];
                const double u_im = i > 0      ? u[c - (size_t)nt * np] : 0.0;
                const double u_ip = i < nr - 1 ? u[c + (size_t)nt * np] : 0.0;
                const double u_jm = j > 0      ? u[c - np] : 0.0;   /* g[2] = 0 at the pole */
                const double u_jp = j < nt - 1 ? u[c + np] : 0.0;   /* g[3] = 0 at the pole */
                const double u_km = u[c - k + km];
                const double u_kp = u[c - k + kp];
                double flux = g[0] * (uc - u_im) + g[1] * (uc - u_ip)
                            + g[2] * (uc - u_jm) + g[3] * (uc - u_jp)
                            + g[4] * (uc - u_km) + g[5] * (uc - u_kp);
                y[c] = volume(op, i, j, k) * uc + op->dt * flux;
            }
}

/* s1-style stiffness: max over cells of (d - V)/V at the operator's current dt (Q12, Q13) */
double mas_ref_stiffness_max(const ref_op *op)
{
    double g[6], m = 0.0;
    for (int i = 0; i < op->nr; i++)
        for (int j = 0; j < op->nt; j++)
            for (int k = 0; k < op->np; k++) {
                faces(op, i, j, k, g);
                double s = op->dt * (g[0] + g[1] + g[2] + g[3] + g[4] + g[5]) / volume(op, i, j, k);
                if (s > m) m = s;
            }
    return m;
}

static double dot(size_t n, const double *a, const double *b)
{
    long double s = 0.0L;
    for (size_t c = 0; c < n; c++) s += (long double)a[c] * (long double)b[c];
    return (double)s;
}

/* PC2 (block-Jacobi ILU(0), defined at the end of this file): z = M^-1 r */
typedef struct ref_pc2 ref_pc2;
void mas_ref_pc2_apply(const ref_pc2 *pc, const double *r, double *z);
static size_t pc2_size(const ref_pc2 *pc);

/* z = M^-1 r:  PC1, M = diag(A_sym) (pc == NULL), or PC2, M = the block-Jacobi ILU(0) factors */
static void precondition(const ref_pc2 *pc, size_t n, const double *d, const double *r, double *z)
{
    if (pc) mas_ref_pc2_apply(pc, r, z);
    else for (size_t c = 0; c < n; c++) z[c] = r[c] / d[c];
}

/*
 * Textbook PCG ("PCG ...", Saad [22]) in the order and notation of DESIGN.md R3 / SURVEY.md 8(c) C3,
 * with the paper's two preconditioners: PC1, M = diag(A_sym) ("the inverse diagonal of the matrix
 * (point-Jacobi)"), when pc == NULL; PC2, M = block-Jacobi ILU(0), otherwise.
 *   b_phys : physical right-hand side (b_s = V.b is formed here)
 *   x      : in = x0, out = last iterate
 *   hist   : NULL or >= maxit+1 doubles; hist[k] = ||r_k||_2 / ||b_s||_2
 * returns REF_OK / REF_MAXIT / negative error; *iters = k.
 */
static int pcg_core(const ref_op *op, const ref_pc2 *pc, const double *b_phys, double *x, double rtol, int maxit,
                    int *iters, double *hist)
{
    if (!op || !b_phys || !x || !iters || rtol < 0.0 || maxit < 0) return REF_EINVAL;
    const size_t n = (size_t)op->nr * op->nt * op->np;
    if (pc && pc2_size(pc) != n) return REF_EINVAL;
    double *d = (double *)malloc(n * sizeof(double)), *r = (double *)malloc(n * sizeof(double));
    double *z = (double *)malloc(n * sizeof(double)), *p = (double *)malloc(n * sizeof(double));
    double *q = (double *)malloc(n * sizeof(double));
    int status = REF_ENOMEM, k = 0;
    if (!d || !r || !z || !p || !q) goto done;

    mas_ref_diag(op, d);
    mas_ref_volume(op, z);                       /* z used as scratch for V */
    for (size_t c = 0; c < n; c++) r[c] = z[c] * b_phys[c];     /* b_s = V.b */
    const double bb = dot(n, r, r);
    if (!isfinite(bb)) {                         /* a non-finite scalar is a breakdown; x untouched */
        if (hist) hist[0] = bb;
        *iters = 0; status = REF_EBREAKDOWN; goto done;
    }
    if (bb == 0.0) {                             /* zero right-hand side: x = 0 */
        memset(x, 0, n * sizeof(double));
        if (hist) hist[0] = 0.0;
        *iters = 0; status = REF_OK; goto done;
    }
    mas_ref_apply(op, x, q);
    for (size_t c = 0; c < n; c++) r[c] -= q[c];                /* r = b_s - A x0 */
    precondition(pc, n, d, r, z);
    memcpy(p, z, n * sizeof(double));
    double rho = dot(n, r, z), rr = dot(n, r, r);
    double h = sqrt(rr / bb);
    if (hist) hist[0] = h;
    status = REF_OK;
    if (!isfinite(rho) || !isfinite(rr)) { *iters = 0; status = REF_EBREAKDOWN; goto done; }
    while (k < maxit && h > rtol && rho != 0.0) {
        mas_ref_apply(op, p, q);
        const double sigma = dot(n, p, q);
        if (!(sigma > 0.0) || !isfinite(sigma)) { status = REF_EBREAKDOWN; break; }
        const double alpha = rho / sigma;
        for (size_t c = 0; c < n; c++) x[c] += alpha * p[c];
        for (size_t c = 0; c < n; c++) r[c] -= alpha * q[c];
        precondition(pc, n, d, r, z);
        const double rho1 = dot(n, r, z);
        rr = dot(n, r, r);
        k += 1;
        h = sqrt(rr / bb);
        if (hist) hist[k] = h;
        if (!isfinite(rho1) || !isfinite(rr)) { status = REF_EBREAKDOWN; break; }   /* iterate k is kept */
        const double beta = rho1 / rho;
        rho = rho1;
        for (size_t c = 0; c < n; c++) p[c] = z[c] + beta * p[c];
    }
    if (status == REF_OK) status = (h <= rtol || rho == 0.0) ? REF_OK : REF_MAXIT;
    *iters = k;
done:
    free(d); free(r); free(z); free(p); free(q);
    return status;
}

/* PCG with PC1 (point-Jacobi) */
int mas_ref_pcg(const ref_op *op, const double *b_phys, double *x, double rtol, int maxit,
                int *iters, double *hist)
{
    return pcg_core(op, NULL, b_phys, x, rtol, maxit, iters, hist);
}

/*
 * NEXT-2: several right-hand sides that share one operator -- the three components of v in
 * PAPER.md:50 eq. (1), which share one coefficient set (SURVEY 8(f)'s observation, not a quotation).  By definition this is nrhs INDEPENDENT textbook solves,
 * each with its own alpha, beta, iteration count, status and history: nothing is coupled across right-hand
 * sides.  b, x: nrhs vectors stored back to back (nrhs * N doubles); hist: NULL or nrhs * (maxit + 1) doubles,
 * right-hand side j's history starting at hist + j * (maxit + 1); iters, status: nrhs ints.
 * Returns the most severe status (negative before MAXIT before OK).
 */
int mas_ref_pcg_multi(const ref_op *op, int nrhs, const double *b_phys, double *x, double rtol, int maxit,
                      int *iters, int *status, double *hist)
{
    if (!op || nrhs < 1 || !b_phys || !x || !iters || !status) return REF_EINVAL;
    const size_t n = (size_t)op->nr * op->nt * op->np;
    int worst = REF_OK;
    for (int j = 0; j < nrhs; j++) {
        status[j] = mas_ref_pcg(op, b_phys + (size_t)j * n, x + (size_t)j * n, rtol, maxit, &iters[j],
                                hist ? hist + (size_t)j * ((size_t)maxit + 1) : NULL);
        if (status[j] < 0 ? (worst >= 0 || status[j] < worst) : (worst >= 0 && status[j] > worst)) worst = status[j];
    }
    return worst;
}

/* ==============================================================================================
 * NEXT-1: the explicit alternative to the viscosity PCG solve -- "a Runge-Kutta
 * Legendre super time-stepping (STS) scheme [21]" (~200 sub-steps per step, PAPER.md:80;
 * the fastest GPU choice).  The paper gives no formulas; R7 restates the
 * second-order scheme RKL2 of its reference [21] (Meyer, Balsara & Aslam, J. Comput. Phys. 257, 2014):
 *
 *   du/dt = M u,   M u = -(1/V) sum_f G_f (u_c - u_nb)      [FD form of div(nu grad u); A_phys = I - dt M]
 *   b_0 = b_1 = b_2 = 1/3,  b_j = (j^2 + j - 2) / (2 j (j + 1)),  a_j = 1 - b_j,  w_1 = 4 / (s^2 + s - 2)
 *   Y_0 = u,   Y_1 = Y_0 + mu~_1 tau M Y_0,                      mu~_1 = b_1 w_1
 *   Y_j = mu_j Y_{j-1} + nu_j Y_{j-2} + (1 - mu_j - nu_j) Y_0 + mu~_j tau M Y_{j-1} + gamma~_j tau M Y_0
 *   mu_j = (2j-1)/j * b_j/b_{j-1},  nu_j = -(j-1)/j * b_j/b_{j-2},  mu~_j = mu_j w_1,  gamma~_j = -a_{j-1} mu~_j
 *   u <- Y_s.      Stable for tau <= (s^2 + s - 2)/4 * 2/lambda_max.
 * Pinned by tests/test_oracle_sts_pins.py: the closed-form stability polynomial
 * R_s(z) = a_s + b_s P_s(1 + w_1 z) (Legendre P_s) on eigenvectors, third-order local error against
 * the matrix exponential, conservation, stability at the limit.
 * ============================================================================================== */

/* y = M u */
void mas_ref_lop(const ref_op *op, const double *u, double *y)
{
    const int nr = op->nr, nt = op->nt, np = op->np;
    double g[6];
    for (int i = 0; i < nr; i++)
        for (int j = 0; j < nt; j++)
            for (int k = 0; k < np; k++) {
                const size_t c = ((size_t)i * nt + j) * np + k;
                const int kp = (k + 1) % np, km = (k + np - 1) % np;
                faces(op, i, j, k, g);
                const double uc = u[c];
                const double u_im = i > 0      ? u[c - (size_t)nt * np] : 0.0;
                const double u_ip = i < nr - 1 ? u[c + (size_t)nt * np] : 0.0;
                const double u_jm = j > 0      ? u[c - np] : 0.0;
                const double u_jp = j < nt - 1 ? u[c + np] : 0.0;
                const double flux = g[0] * (uc - u_im) + g[1] * (uc - u_ip) + g[2] * (uc - u_jm)
                                  + g[3] * (uc - u_jp) + g[4] * (uc - u[c - k + km]) + g[5] * (uc - u[c - k + kp]);
                y[c] = -flux / volume(op, i, j, k);
            }
}

/* Gershgorin bound on the spectral radius of M: max over cells of 2 (sum of face conductances) / V */
double mas_ref_lambda_max_bound(const ref_op *op)
{
    double g[6], m = 0.0;
    for (int i = 0; i < op->nr; i++)
        for (int j = 0; j < op->nt; j++)
            for (int k = 0; k < op->np; k++) {
                faces(op, i, j, k, g);
                const double s = 2.0 * (g[0] + g[1] + g[2] + g[3] + g[4] + g[5]) / volume(op, i, j, k);
                if (s > m) m = s;
            }
    return m;
}

static double rkl2_b(int j) { return j < 3 ? 1.0 / 3.0 : ((double)j * j + j - 2.0) / (2.0 * j * (j + 1.0)); }

/* one RKL2 super-step of size tau with s >= 2 stages, in place */
int mas_ref_sts(const ref_op *op, double *u, double tau, int s)
{
    if (!op || !u || s < 2 || !(tau >= 0.0)) return REF_EINVAL;
    const size_t n = (size_t)op->nr * op->nt * op->np;
    double *y0 = (double *)malloc(n * sizeof(double)), *my0 = (double *)malloc(n * sizeof(double));
    double *yjm2 = (double *)malloc(n * sizeof(double)), *yjm1 = (double *)malloc(n * sizeof(double));
    double *yj = (double *)malloc(n * sizeof(double)), *my = (double *)malloc(n * sizeof(double));
    int status = REF_ENOMEM;
    if (!y0 || !my0 || !yjm2 || !yjm1 || !yj || !my) goto done;
    const double w1 = 4.0 / ((double)s * s + s - 2.0);
    memcpy(y0, u, n * sizeof(double));
    mas_ref_lop(op, y0, my0);
    const double mut1 = rkl2_b(1) * w1;
    for (size_t c = 0; c < n; c++) yjm1[c] = y0[c] + mut1 * tau * my0[c];      /* Y_1 */
    memcpy(yjm2, y0, n * sizeof(double));                                       /* Y_0 */
    for (int j = 2; j <= s; j++) {
        const double bj = rkl2_b(j), bjm1 = rkl2_b(j - 1), bjm2 = rkl2_b(j - 2);
        const double mu = (2.0 * j - 1.0) / j * bj / bjm1;
        const double nu = -(j - 1.0) / j * bj / bjm2;
        const double mut = mu * w1;
        const double gat = -(1.0 - bjm1) * mut;
        mas_ref_lop(op, yjm1, my);
        for (size_t c = 0; c < n; c++)
            yj[c] = mu * yjm1[c] + nu * yjm2[c] + (1.0 - mu - nu) * y0[c] + mut * tau * my[c] + gat * tau * my0[c];
        double *t = yjm2; yjm2 = yjm1; yjm1 = yj; yj = t;
    }
    memcpy(u, yjm1, n * sizeof(double));
    status = REF_OK;
done:
    free(y0); free(my0); free(yjm2); free(yjm1); free(yj); free(my);
    return status;
}

/* ==============================================================================================
 * NEXT-4: the paper's second preconditioner -- "the second (PC2) is a block-Jacobi
 * using a zero-fill incomplete LU factorization [22]" (Sec. 2.2; that the blocks are
 * non-overlapping boxes of cells is this oracle's reading, R8, not the paper's words;
 * 100-200 iterations against ~550 with PC1; its triangular solves are what the authors call
 * "not vectorizable" and leave on the CPU).
 *
 * The paper prints neither the decomposition nor the factorisation.  Reading (R8):
 *   * the domains are boxes of bi x bj x bk cells aligned at the mesh origin (the last box of a direction may be
 *     smaller); A_blk = A_sym with every coupling between cells of different boxes dropped, i.e. the
 *     block-diagonal part of A_sym in the box partition (block Jacobi; "communication-free");
 *     a box that spans all of phi keeps the periodic wrap coupling, any other box does not have it;
 *   * ILU(0) is the textbook zero-fill factorisation (Saad [22], the reference the paper cites for its solvers)
 *     of A_blk in the natural ordering (phi fastest, then theta, then r): unit lower L and upper U whose
 *     non-zeros are confined to the pattern of A_blk and with (L U)_ij = (A_blk)_ij on that pattern;
 *   * M = L U;  z = M^-1 r by a forward and a backward substitution;  the PCG loop is C3's with z = M^-1 r.
 * Written out generically on a compressed-sparse-row copy of A_blk (row-wise IKJ elimination restricted to
 * the pattern), so that nothing about the stencil's structure is assumed by the factorisation.
 * Pinned by tests/test_oracle_pc2_pins.py: (L U = A_blk on the pattern) on dense copies, exactness for
 * tridiagonal operators (1-D meshes: ILU(0) = LU, one PCG iteration), dt = 0, symmetry and positivity of
 * M^-1, box locality, dense-LU agreement of the PCG solution, fewer iterations than PC1.
 * What is tied to the paper's own run (its domains = its MPI ranks' sub-meshes, its 100-200 counts) is
 * "parity unpinned": not available.
 * ============================================================================================== */

struct ref_pc2 {
    size_t n;
    int nnz_max;
    size_t *rowptr;     /* [n+1] */
    int *col;           /* [nnz] ascending within a row */
    double *val;        /* [nnz] A_blk, overwritten by the factors: strictly lower = L (unit diagonal implied), rest = U */
    size_t *diag;       /* [n] position of the diagonal entry of each row */
};

static size_t pc2_size(const ref_pc2 *pc) { return pc->n; }

void mas_ref_pc2_destroy(ref_pc2 *pc)
{
    if (!pc) return;
    free(pc->rowptr); free(pc->col); free(pc->val); free(pc->diag);
    free(pc);
}

static int cmp_entry(const void *a, const void *b)
{
    const long long ca = *(const long long *)a, cb = *(const long long *)b;
    return ca < cb ? -1 : (ca > cb ? 1 : 0);
}

/* A_blk in CSR (values at the operator's current dt), then ILU(0) in place.  bi, bj, bk <= 0 mean "the whole extent". */
ref_pc2 *mas_ref_pc2_create(const ref_op *op, int bi, int bj, int bk)
{
    if (!op) return NULL;
    const int nr = op->nr, nt = op->nt, np = op->np;
    if (bi <= 0 || bi > nr) bi = nr;
    if (bj <= 0 || bj > nt) bj = nt;
    if (bk <= 0 || bk > np) bk = np;
    const size_t n = (size_t)nr * nt * np;
    ref_pc2 *pc = (ref_pc2 *)calloc(1, sizeof(ref_pc2));
    if (!pc) return NULL;
    pc->n = n;
    pc->rowptr = (size_t *)malloc((n + 1) * sizeof(size_t));
    pc->col = (int *)malloc(7 * n * sizeof(int));
    pc->val = (double *)malloc(7 * n * sizeof(double));
    pc->diag = (size_t *)malloc(n * sizeof(size_t));
    if (!pc->rowptr || !pc->col || !pc->val || !pc->diag) { mas_ref_pc2_destroy(pc); return NULL; }

    /* ---- rows of A_blk: diagonal of A_sym, and -dt G_f for every face whose two cells lie in the same box ---- */
    size_t nnz = 0;
    double g[6];
    for (int i = 0; i < nr; i++)
        for (int j = 0; j < nt; j++)
            for (int k = 0; k < np; k++) {
                const size_t c = ((size_t)i * nt + j) * np + k;
                faces(op, i, j, k, g);
                long long cols[7];
                double vals[7];
                int m = 0;
                cols[m] = (long long)c;
                vals[m++] = volume(op, i, j, k) + op->dt * (g[0] + g[1] + g[2] + g[3] + g[4] + g[5]);
                const int kp = (k + 1) % np, km = (k + np - 1) % np;
                const int nb_i[6] = {i - 1, i + 1, i, i, i, i};
                const int nb_j[6] = {j, j, j - 1, j + 1, j, j};
                const int nb_k[6] = {k, k, k, k, km, kp};
                for (int f = 0; f < 6; f++) {
                    const int ii = nb_i[f], jj = nb_j[f], kk = nb_k[f];
                    if (ii < 0 || ii >= nr || jj < 0 || jj >= nt) continue;          /* boundary face: no neighbour cell */
                    if (ii / bi != i / bi || jj / bj != j / bj || kk / bk != k / bk) continue;   /* another box */
                    const long long cc = (long long)(((size_t)ii * nt + jj) * np + kk);
                    int hit = -1;                                                     /* np = 2: both phi faces lead to the same cell; */
                    for (int e = 0; e < m; e++) if (cols[e] == cc) hit = e;          /* np = 1: the cell is its own phi neighbour     */
                    if (hit >= 0) vals[hit] += -op->dt * g[f];
                    else { cols[m] = cc; vals[m++] = -op->dt * g[f]; }
                }
                /* sort the row by column */
                long long key[7]; double v2[7];
                for (int e = 0; e < m; e++) key[e] = cols[e];
                qsort(key, (size_t)m, sizeof(long long), cmp_entry);
                for (int e = 0; e < m; e++)
                    for (int f2 = 0; f2 < m; f2++) if (cols[f2] == key[e]) v2[e] = vals[f2];
                pc->rowptr[c] = nnz;
                for (int e = 0; e < m; e++) {
                    if (key[e] == (long long)c) pc->diag[c] = nnz;
                    pc->col[nnz] = (int)key[e];
                    pc->val[nnz++] = v2[e];
                }
            }
    pc->rowptr[n] = nnz;

    /* ---- ILU(0), row-wise IKJ variant restricted to the pattern (Saad, "Iterative Methods for Sparse Linear
     * Systems", the zero-fill ILU algorithm):
     *   for i = 1..n-1:  for k in pattern(i), k < i (ascending):  a_ik /= a_kk
     *                        for j in pattern(i), j > k:  if (k, j) in pattern:  a_ij -= a_ik a_kj          ---- */
    for (size_t i = 0; i < n; i++)
        for (size_t e = pc->rowptr[i]; e < pc->diag[i]; e++) {
            const size_t k = (size_t)pc->col[e];
            pc->val[e] /= pc->val[pc->diag[k]];
            const double lik = pc->val[e];
            for (size_t f = e + 1; f < pc->rowptr[i + 1]; f++) {
                const int j = pc->col[f];
                for (size_t t = pc->diag[k] + 1; t < pc->rowptr[k + 1]; t++)
                    if (pc->col[t] == j) pc->val[f] -= lik * pc->val[t];
            }
        }
    return pc;
}

/* z = M^-1 r = U^-1 (L^-1 r): forward substitution with the unit lower factor, then backward with U */
void mas_ref_pc2_apply(const ref_pc2 *pc, const double *r, double *z)
{
    const size_t n = pc->n;
    for (size_t i = 0; i < n; i++) {
        double s = r[i];
        for (size_t e = pc->rowptr[i]; e < pc->diag[i]; e++) s -= pc->val[e] * z[pc->col[e]];
        z[i] = s;
    }
    for (size_t i = n; i-- > 0;) {
        double s = z[i];
        for (size_t e = pc->diag[i] + 1; e < pc->rowptr[i + 1]; e++) s -= pc->val[e] * z[pc->col[e]];
        z[i] = s / pc->val[pc->diag[i]];
    }
}

/* the factors as dense matrices, for the pins (tiny meshes): Ld = unit lower L, Ud = U, both n x n row-major */
void mas_ref_pc2_dense_factors(const ref_pc2 *pc, double *Ld, double *Ud)
{
    const size_t n = pc->n;
    memset(Ld, 0, n * n * sizeof(double));
    memset(Ud, 0, n * n * sizeof(double));
    for (size_t i = 0; i < n; i++) {
        Ld[i * n + i] = 1.0;
        for (size_t e = pc->rowptr[i]; e < pc->rowptr[i + 1]; e++) {
            if (e < pc->diag[i]) Ld[i * n + (size_t)pc->col[e]] = pc->val[e];
            else Ud[i * n + (size_t)pc->col[e]] = pc->val[e];
        }
    }
}

/* PCG of SURVEY.md 8(c) C3 with z = M^-1 r, M = the block-Jacobi ILU(0) `pc` (built from `op` at its current dt).
 * Same arguments, statuses and stopping rule as mas_ref_pcg. */
int mas_ref_pcg_pc2(const ref_op *op, const ref_pc2 *pc, const double *b_phys, double *x, double rtol, int maxit,
                    int *iters, double *hist)
{
    if (!pc) return REF_EINVAL;
    return pcg_core(op, pc, b_phys, x, rtol, maxit, iters, hist);
}

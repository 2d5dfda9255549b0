/*
 * pbref -- ORACLE (test infrastructure, not product code).
 *
 * A plain, slow, fp64 CPU implementation of what the hot path computes, written from
 * /root/reference/PAPER.md (Qi, Botello-Smith & Luo, arxiv 1704.02745):
 *   - the 7-point finite-difference operator of Eq. 3, applied row by
 *     row exactly as printed, 1/h^2 factors included (no rescaling, no blocking);
 *   - the linear system A phi = b of Eq. 4 with the free-space Dirichlet
 *     values on a ghost layer moved to the right-hand side;
 *   - the preconditioned CG iteration, steps 1-8 of PAPER.md:104-126, with the Jacobi
 *     preconditioner M = D = diag(A) of PAPER.md:138-140, phi_0 = 0.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
 * may build, load or call this file.  It shares no source, header, table or helper with
 * paper_1704_02745_b200/ (the CUDA path) and neither includes the other.
 *
 * Conventions: node (i,j,k), x fastest, idx = (k*ny + j)*nx + i.
 *   eps_x[k][j][f], f = 0..nx : face between node i=f-1 and node i=f, i.e. the paper's
 *   eps_i(i,j,k) (between (i,j,k) and (i+1,j,k)) is eps_x[k][j][i+1]; f=0 and f=nx touch
 *   the ghost layer.  eps_y[k][f][i], f = 0..ny;  eps_z[f][j][i], f = 0..nz.
 *   bc = ghost Dirichlet values packed x-,x+ ([nz][ny] each), y-,y+ ([nz][nx]), z-,z+ ([ny][nx]).
 *   The library is unit-agnostic: it solves  -div(eps grad phi) + kbar2 phi = rhs, so the
 *   paper's h^-3 q(i,j,k) is the caller's rhs (Reading 8).
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): closed-form eigenpairs of the uniform
 * 7-point Laplacian on anisotropic boxes, dense row-by-row assembly + LAPACK solve for
 * grids <= 9^3, exact termination in m iterations on m eigenvectors, the manufactured
 * solution sin(pi x)sin(pi y)sin(pi z) with its closed-form discrete error, the Born ion,
 * SPD/symmetry invariants.  Parity unpinned: anything needing the paper's protein
 * structures or energies, which are not available.
 *
 * Reductions: every dot product is a plain left-to-right fp64 sum over one k-plane;
 * the plane sums are then added in increasing k.  OpenMP (if enabled) only distributes
 * whole planes, so results are bit-identical for any thread count.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#define PAR_FOR _Pragma("omp parallel for schedule(static)")   /* elementwise loops only */
#else
#define PAR_FOR
#endif

enum { PBREF_OK = 0, PBREF_INVALID = 1, PBREF_ALLOC = 2, PBREF_NOT_SPD = 4,
       PBREF_BREAKDOWN = 5, PBREF_MAXITER = 6 };

typedef struct pbref {
    int nx, ny, nz;
    double h;
    double *eps_x, *eps_y, *eps_z;   /* private copies, layouts as above */
    double *kbar2;                   /* [nz][ny][nx], zeros if the caller passed NULL */
    double *b;                       /* right-hand side of Eq. 4 after the Dirichlet fold-in */
    double *D;                       /* diag(A) */
    double *plane;                   /* nz per-plane partial sums */
    int have_rhs;
    int periodic;                    /* 1: periodic boundary condition: indices wrap, no ghost layer */
} pbref;

/* face dielectrics touching node (i,j,k), in the paper's notation */
#define EXM(s,i,j,k) ((s)->eps_x[((size_t)(k)*(s)->ny + (j))*((s)->nx+1) + (i)])      /* eps_i(i-1,j,k) */
#define EXP(s,i,j,k) ((s)->eps_x[((size_t)(k)*(s)->ny + (j))*((s)->nx+1) + (i) + 1])  /* eps_i(i,j,k)   */
#define EYM(s,i,j,k) ((s)->eps_y[((size_t)(k)*((s)->ny+1) + (j))*(s)->nx + (i)])      /* eps_j(i,j-1,k) */
#define EYP(s,i,j,k) ((s)->eps_y[((size_t)(k)*((s)->ny+1) + (j) + 1)*(s)->nx + (i)])  /* eps_j(i,j,k)   */
#define EZM(s,i,j,k) ((s)->eps_z[((size_t)(k)*(s)->ny + (j))*(s)->nx + (i)])          /* eps_k(i,j,k-1) */
#define EZP(s,i,j,k) ((s)->eps_z[((size_t)((k)+1)*(s)->ny + (j))*(s)->nx + (i)])      /* eps_k(i,j,k)   */
#define NODE(s,i,j,k) (((size_t)(k)*(s)->ny + (j))*(s)->nx + (i))

int pbref_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* thread count for the timed CPU baseline (bench.py: all cores, and 1 thread for grids <= 129^3 like the paper's
 * single-core CPU/CG); results do not depend on it (whole planes per thread, see above) */
void pbref_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n >= 1) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

static double *dup_array(const double *src, size_t n)
{
    double *d = (double *)malloc((n ? n : 1) * sizeof(double));
    if (d && src) memcpy(d, src, n * sizeof(double));
    return d;
}

int pbref_destroy(pbref *s)
{
    if (!s) return PBREF_OK;
    free(s->eps_x); free(s->eps_y); free(s->eps_z); free(s->kbar2);
    free(s->b); free(s->D); free(s->plane);
    free(s);
    return PBREF_OK;
}

/* Ghost value seen by node (i,j,k) through each of its six faces (only read when that
 * neighbour is outside the grid). */
static double ghost_xm(const pbref *s, const double *bc, int j, int k) { return bc[(size_t)k*s->ny + j]; }
static double ghost_xp(const pbref *s, const double *bc, int j, int k) { return bc[(size_t)s->nz*s->ny + (size_t)k*s->ny + j]; }
static double ghost_ym(const pbref *s, const double *bc, int i, int k) { return bc[2*(size_t)s->nz*s->ny + (size_t)k*s->nx + i]; }
static double ghost_yp(const pbref *s, const double *bc, int i, int k) { return bc[2*(size_t)s->nz*s->ny + (size_t)s->nz*s->nx + (size_t)k*s->nx + i]; }
static double ghost_zm(const pbref *s, const double *bc, int i, int j) { return bc[2*(size_t)s->nz*s->ny + 2*(size_t)s->nz*s->nx + (size_t)j*s->nx + i]; }
static double ghost_zp(const pbref *s, const double *bc, int i, int j) { return bc[2*(size_t)s->nz*s->ny + 2*(size_t)s->nz*s->nx + (size_t)s->ny*s->nx + (size_t)j*s->nx + i]; }

/* b = rhs + h^-2 * sum over ghost neighbours of eps_face * g   (Eq. 3 with the known
 * phi(ghost) = g terms moved to the right).  rhs/bc NULL = 0. */
int pbref_set_rhs(pbref *s, const double *rhs, const double *bc)
{
    if (!s) return PBREF_INVALID;
    const int nx = s->nx, ny = s->ny, nz = s->nz;
    const double ih2 = 1.0 / (s->h * s->h);
    for (int k = 0; k < nz; k++)
        for (int j = 0; j < ny; j++)
            for (int i = 0; i < nx; i++) {
                double v = rhs ? rhs[NODE(s,i,j,k)] : 0.0;
                if (bc && !s->periodic) {
                    if (i == 0)      v += ih2 * EXM(s,i,j,k) * ghost_xm(s, bc, j, k);
                    if (i == nx - 1) v += ih2 * EXP(s,i,j,k) * ghost_xp(s, bc, j, k);
                    if (j == 0)      v += ih2 * EYM(s,i,j,k) * ghost_ym(s, bc, i, k);
                    if (j == ny - 1) v += ih2 * EYP(s,i,j,k) * ghost_yp(s, bc, i, k);
                    if (k == 0)      v += ih2 * EZM(s,i,j,k) * ghost_zm(s, bc, i, j);
                    if (k == nz - 1) v += ih2 * EZP(s,i,j,k) * ghost_zp(s, bc, i, j);
                }
                s->b[NODE(s,i,j,k)] = v;
            }
    s->have_rhs = 1;
    return PBREF_OK;
}

int pbref_create(pbref **out, int nx, int ny, int nz, double h,
                 const double *eps_x, const double *eps_y, const double *eps_z,
                 const double *kbar2, const double *rhs, const double *bc)
{
    if (!out) return PBREF_INVALID;
    *out = NULL;
    if (nx < 1 || ny < 1 || nz < 1 || !(h > 0.0) || !eps_x || !eps_y || !eps_z) return PBREF_INVALID;
    pbref *s = (pbref *)calloc(1, sizeof(pbref));
    if (!s) return PBREF_ALLOC;
    s->nx = nx; s->ny = ny; s->nz = nz; s->h = h;
    const size_t n = (size_t)nx * ny * nz;
    s->eps_x = dup_array(eps_x, (size_t)nz * ny * (nx + 1));
    s->eps_y = dup_array(eps_y, (size_t)nz * (ny + 1) * nx);
    s->eps_z = dup_array(eps_z, (size_t)(nz + 1) * ny * nx);
    s->kbar2 = (double *)calloc(n, sizeof(double));
    s->b = (double *)calloc(n, sizeof(double));
    s->D = (double *)calloc(n, sizeof(double));
    s->plane = (double *)calloc((size_t)nz, sizeof(double));
    if (!s->eps_x || !s->eps_y || !s->eps_z || !s->kbar2 || !s->b || !s->D || !s->plane) {
        pbref_destroy(s);
        return PBREF_ALLOC;
    }
    if (kbar2) memcpy(s->kbar2, kbar2, n * sizeof(double));
    /* D = diag(A): the coefficient of phi(i,j,k) in Eq. 3 */
    const double ih2 = 1.0 / (h * h);
    int bad = 0;
    for (int k = 0; k < nz; k++)
        for (int j = 0; j < ny; j++)
            for (int i = 0; i < nx; i++) {
                double d = ih2 * EXM(s,i,j,k) + ih2 * EXP(s,i,j,k)
                         + ih2 * EYM(s,i,j,k) + ih2 * EYP(s,i,j,k)
                         + ih2 * EZM(s,i,j,k) + ih2 * EZP(s,i,j,k)
                         + s->kbar2[NODE(s,i,j,k)];
                s->D[NODE(s,i,j,k)] = d;
                if (!(d > 0.0) || !isfinite(d)) bad = 1;
            }
    if (bad) { pbref_destroy(s); return PBREF_NOT_SPD; }
    if (rhs || bc) pbref_set_rhs(s, rhs, bc);
    *out = s;
    return PBREF_OK;
}

/* One k-plane of y = A x: the left-hand side of Eq. 3 term by term, as printed
 * (PAPER.md:50-62), with x = 0 on the ghost layer (the ghost values live in b). */
static void apply_plane(const pbref *s, const double *x, double *y, int k)
{
    const int nx = s->nx, ny = s->ny, nz = s->nz;
    const double ih2 = 1.0 / (s->h * s->h);
    for (int j = 0; j < ny; j++)
        for (int i = 0; i < nx; i++) {
            const double xc = x[NODE(s,i,j,k)];
            /* neighbours outside the grid: the ghost layer (value 0 here, its Dirichlet value sits in b) or, with the
             * periodic boundary condition, the node on the opposite side (phi(-1) = phi(n-1), phi(n) = phi(0)) */
            const int per = s->periodic;
            const double xim = (i > 0)      ? x[NODE(s,i-1,j,k)] : (per ? x[NODE(s,nx-1,j,k)] : 0.0);
            const double xip = (i < nx - 1) ? x[NODE(s,i+1,j,k)] : (per ? x[NODE(s,0,j,k)]    : 0.0);
            const double xjm = (j > 0)      ? x[NODE(s,i,j-1,k)] : (per ? x[NODE(s,i,ny-1,k)] : 0.0);
            const double xjp = (j < ny - 1) ? x[NODE(s,i,j+1,k)] : (per ? x[NODE(s,i,0,k)]    : 0.0);
            const double xkm = (k > 0)      ? x[NODE(s,i,j,k-1)] : (per ? x[NODE(s,i,j,nz-1)] : 0.0);
            const double xkp = (k < nz - 1) ? x[NODE(s,i,j,k+1)] : (per ? x[NODE(s,i,j,0)]    : 0.0);
            double v = 0.0;
            v += -ih2 * EXM(s,i,j,k) * (xim - xc);
            v += -ih2 * EXP(s,i,j,k) * (xip - xc);
            v += -ih2 * EYM(s,i,j,k) * (xjm - xc);
            v += -ih2 * EYP(s,i,j,k) * (xjp - xc);
            v += -ih2 * EZM(s,i,j,k) * (xkm - xc);
            v += -ih2 * EZP(s,i,j,k) * (xkp - xc);
            v += s->kbar2[NODE(s,i,j,k)] * xc;
            y[NODE(s,i,j,k)] = v;
        }
}

int pbref_apply(pbref *s, const double *x, double *y)
{
    if (!s || !x || !y) return PBREF_INVALID;
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int k = 0; k < s->nz; k++) apply_plane(s, x, y, k);
    return PBREF_OK;
}

/* u.v : left-to-right within each k-plane, planes added in increasing k */
static double dot(pbref *s, const double *u, const double *v)
{
    const size_t pl = (size_t)s->nx * s->ny;
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int k = 0; k < s->nz; k++) {
        const double *a = u + (size_t)k * pl, *c = v + (size_t)k * pl;
        double acc = 0.0;
        for (size_t t = 0; t < pl; t++) acc += a[t] * c[t];
        s->plane[k] = acc;
    }
    double tot = 0.0;
    for (int k = 0; k < s->nz; k++) tot += s->plane[k];
    return tot;
}

/* Periodic boundary condition (the paper's PBC runs): the face f = 0 and the face
 * f = n of each direction are the same physical face (the caller passes equal values), the neighbour across it is
 * the node on the opposite side, and there are no ghost values.  Call before pbref_set_rhs. */
int pbref_set_periodic(pbref *s, int flag)
{
    if (!s) return PBREF_INVALID;
    s->periodic = flag ? 1 : 0;
    return PBREF_OK;
}

int pbref_get_b(pbref *s, double *b_out)
{
    if (!s || !b_out) return PBREF_INVALID;
    memcpy(b_out, s->b, (size_t)s->nx * s->ny * s->nz * sizeof(double));
    return PBREF_OK;
}

int pbref_get_diag(pbref *s, double *d_out)
{
    if (!s || !d_out) return PBREF_INVALID;
    memcpy(d_out, s->D, (size_t)s->nx * s->ny * s->nz * sizeof(double));
    return PBREF_OK;
}

/*
 * Preconditioned CG, step numbers as in the paper.
 *   precond = 1 : M = D (Jacobi);  precond = 0 : M = I (plain CG in
 *   its PCG form; the CG listing at PAPER.md:76-94 is sign-garbled, Reading 1).
 *   Stopping rule (step 3): ||r_l||_2 / ||b||_2 < tol with the recurrence residual r_l and
 *   the folded b of Eq. 4 (Readings 3-5), strict "<" as printed.
 *   iters_out = l at exit = number of A p products (Reading 6).
 *   true_relres_out (optional) = ||b - A phi||/||b|| recomputed at exit.
 *   resid_hist (optional, length >= maxiter+1): ||r_l||/||b|| for l = 0..iters.
 * Returns PBREF_OK, PBREF_MAXITER (phi = last iterate) or PBREF_BREAKDOWN (p.Ap <= 0 or NaN).
 */
int pbref_solve(pbref *s, double tol, int maxiter, int precond, double *phi,
                int *iters_out, double *relres_out, double *true_relres_out, double *resid_hist,
                const double *phi0 /* initial guess of step 1; NULL = 0 as in the paper's runs */)
{
    if (!s || !phi || !(tol > 0.0) || maxiter < 0) return PBREF_INVALID;
    const size_t n = (size_t)s->nx * s->ny * s->nz;
    double *r = (double *)malloc(n * sizeof(double));
    double *z = (double *)malloc(n * sizeof(double));
    double *p = (double *)malloc(n * sizeof(double));
    double *Ap = (double *)malloc(n * sizeof(double));
    if (!r || !z || !p || !Ap) { free(r); free(z); free(p); free(Ap); return PBREF_ALLOC; }
    const double *b = s->b, *D = s->D;
    int status = PBREF_OK;

    /* step 1: l = 0, r_0 = b - A phi_0; phi_0 = 0 in the paper's runs gives r_0 = b */
    int l = 0;
    if (phi0) {
        PAR_FOR
    for (size_t c = 0; c < n; c++) phi[c] = phi0[c];
        pbref_apply(s, phi, Ap);
        PAR_FOR
    for (size_t c = 0; c < n; c++) r[c] = b[c] - Ap[c];
    } else {
        PAR_FOR
    for (size_t c = 0; c < n; c++) { phi[c] = 0.0; r[c] = b[c]; }
    }
    const double bb = dot(s, b, b);
    /* step 2: solve M z_0 = r_0, p_0 = z_0 */
    PAR_FOR
    for (size_t c = 0; c < n; c++) { z[c] = precond ? r[c] / D[c] : r[c]; p[c] = z[c]; }
    double rz = dot(s, r, z);
    double rr = dot(s, r, r);
    if (resid_hist) resid_hist[0] = (bb > 0.0) ? sqrt(rr / bb) : 0.0;

    for (;;) {
        /* step 3: ||r_l|| / ||b|| < delta ?  (b = 0 => phi = 0 is the answer) */
        if (bb == 0.0 || rr < tol * tol * bb) break;
        if (l == maxiter) { status = PBREF_MAXITER; break; }
        /* step 4 */
        l = l + 1;
        /* step 5: alpha_l = (r^T z)/(p^T A p); phi += alpha p; r -= alpha A p */
        pbref_apply(s, p, Ap);
        const double pAp = dot(s, p, Ap);
        if (!(pAp > 0.0) || !isfinite(pAp)) { status = PBREF_BREAKDOWN; l = l - 1; break; }
        const double alpha = rz / pAp;
        PAR_FOR
    for (size_t c = 0; c < n; c++) phi[c] += alpha * p[c];
        PAR_FOR
    for (size_t c = 0; c < n; c++) r[c] -= alpha * Ap[c];
        /* step 6: solve M z_l = r_l */
        PAR_FOR
    for (size_t c = 0; c < n; c++) z[c] = precond ? r[c] / D[c] : r[c];
        /* step 7: beta_l = (r_l^T z_l)/(r_{l-1}^T z_{l-1}); p_l = z_l + beta_l p_{l-1} */
        const double rz_new = dot(s, r, z);
        rr = dot(s, r, r);
        const double beta = rz_new / rz;
        rz = rz_new;
        PAR_FOR
    for (size_t c = 0; c < n; c++) p[c] = z[c] + beta * p[c];
        if (resid_hist) resid_hist[l] = sqrt(rr / bb);
        /* step 8: go to step 3 */
    }

    if (iters_out) *iters_out = l;
    if (relres_out) *relres_out = (bb > 0.0) ? sqrt(rr / bb) : 0.0;
    if (true_relres_out) {
        pbref_apply(s, phi, Ap);
        PAR_FOR
    for (size_t c = 0; c < n; c++) z[c] = b[c] - Ap[c];
        *true_relres_out = (bb > 0.0) ? sqrt(dot(s, z, z) / bb) : 0.0;
    }
    free(r); free(z); free(p); free(Ap);
    return status;
}

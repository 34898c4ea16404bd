/* gmg_oracle.c -- TEST INFRASTRUCTURE ONLY.  Plain, slow, FP64 CPU oracle for the
 * geometric-multigrid pressure-Poisson solve of arxiv/paper_2607_07687.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, load or call this file.  It shares no code with the CUDA path
 * (paper_2607_07687_b200/csrc) and neither includes the other.
 *
 * What the paper fixes (PAPER.md = /root/reference/PAPER.md):
 *   - variable-coefficient Poisson equation, finite volume, Cartesian grid   PAPER.md:43 (S3.1), 9
 *   - GMG = smoother + coarse-grid correction, V-cycles                       PAPER.md:39 (S3), 51 (Fig. 2)
 *   - red-black Gauss-Seidel smoother whose relaxation factor "adapts to
 *     residual growth or decay after each V-cycle"                            PAPER.md:43 (S3.1)
 *   - anisotropic coarsening "downsamples every dimension independently"      PAPER.md:47 (S3.2)
 *   - PCG as the general-purpose comparison solver                            PAPER.md:31, 39 (S3)
 * The paper gives these in words only (no equation, constant or stencil), so every
 * formula below is a READING, numbered O1..O12 as in SURVEY.md S8(c) and listed in
 * DESIGN.md "Readings of the paper".
 *
 * PARITY PINS (tests/, -m "not gpu"): operator vs a face-by-face dense assembly and
 * Fourier eigenmodes (O1,O2); symmetry / zero row sum / semi-definiteness on every level
 * (O5); half-sweep zeroes the residual of its colour and decreases the error energy (O3);
 * <Rr,e> = <r,Pe> (O6); closed-form coarse coefficients and quadratic consistency (O5);
 * level shapes (O4); dense least-squares solve on 8^3 (O7,O9,O10,O11 solutions);
 * omega rule restated against the produced history, persistence across solves (O8); the RBGS
 * cycle and its symmetric variant as compositions of the separately pinned operators with
 * (nu1,nu2,nuc) = (2,3,5|6), self-adjointness of the symmetric cycle on the active cells (O7, O11);
 * flux conservation of linear fields on random coefficients for all five coarsening patterns
 * (O5 tiling); norms / stopping test blind to inactive cells and relative to ||z|| (O9); the CG
 * smoother as the Krylov energy minimiser of the dense face-assembled system, its guards incl.
 * the step-length cap firing in FP64 on a two-region level, the CG-smoothed cycle as a composition
 * of its parts (O12).  A mutation run (each plausible slip applied to a copy of this file) turns
 * at least one pin red for every mutation listed in DESIGN.md S3.
 * PARITY UNPINNED against the paper itself: the omega rule and its constants (O8), the
 * sweep counts nu1/nu2/nuc (O7), the meaning of "GMG-PCG" (O11) and the restart, counts and
 * guards of the PCG-smoothed cycle (O12): the paper prints no worked example or constant for them.
 *
 * Layout: cell I=(i,j,k), linear index i + nx*(j + ny*k) (x fastest).  L is
 * component-major: L[d*N + idx] is the coefficient on the LOWER d-face of cell idx
 * (the face between I-e_d and I).  bc[d]: 0 periodic, 1 homogeneous Neumann.
 * On a Neumann axis the stored plane L_d(index 0) is IGNORED (the wall face carries 0)
 * and there is no upper wall face (O2).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#define GMGO_PERIODIC 0
#define GMGO_NEUMANN 1
#define GMGO_MAXLEV 32

typedef long long i64;

static i64 lin(const int n[3], int i, int j, int k) {
    return (i64)i + (i64)n[0] * ((i64)j + (i64)n[1] * (i64)k);
}

static i64 ncells(const int n[3]) { return (i64)n[0] * n[1] * n[2]; }

/* Coefficient of the face between cell I and I-e_d (lower face).  O1, O2. */
static double face_lo(const int n[3], const int bc[3], const double *L, int d, const int I[3]) {
    if (I[d] == 0 && bc[d] == GMGO_NEUMANN) return 0.0; /* wall face */
    return L[(i64)d * ncells(n) + lin(n, I[0], I[1], I[2])];
}

/* Coefficient of the face between cell I and I+e_d (upper face) = lower face of I+e_d. */
static double face_hi(const int n[3], const int bc[3], const double *L, int d, const int I[3]) {
    int J[3] = {I[0], I[1], I[2]};
    if (I[d] == n[d] - 1) {
        if (bc[d] == GMGO_NEUMANN) return 0.0; /* no upper wall face */
        J[d] = 0;                              /* periodic wrap */
    } else {
        J[d] = I[d] + 1;
    }
    return L[(i64)d * ncells(n) + lin(n, J[0], J[1], J[2])];
}

/* Value of p in the neighbour I-e_d / I+e_d.  At a Neumann wall there is no neighbour;
 * the face coefficient is 0 there, so the returned value (p_I itself) never matters. */
static double nb_lo(const int n[3], const int bc[3], const double *p, int d, const int I[3]) {
    int J[3] = {I[0], I[1], I[2]};
    if (I[d] == 0) {
        if (bc[d] == GMGO_NEUMANN) return p[lin(n, I[0], I[1], I[2])];
        J[d] = n[d] - 1;
    } else {
        J[d] = I[d] - 1;
    }
    return p[lin(n, J[0], J[1], J[2])];
}

static double nb_hi(const int n[3], const int bc[3], const double *p, int d, const int I[3]) {
    int J[3] = {I[0], I[1], I[2]};
    if (I[d] == n[d] - 1) {
        if (bc[d] == GMGO_NEUMANN) return p[lin(n, I[0], I[1], I[2])];
        J[d] = 0;
    } else {
        J[d] = I[d] + 1;
    }
    return p[lin(n, J[0], J[1], J[2])];
}

/* O1:  (A p)_I = sum_d [ L_d(I) (p_{I-e_d} - p_I) + L_d(I+e_d) (p_{I+e_d} - p_I) ]  */
static double apply_at(const int n[3], const int bc[3], const double *L, const double *p,
                       const int I[3]) {
    double pc = p[lin(n, I[0], I[1], I[2])];
    double s = 0.0;
    for (int d = 0; d < 3; ++d) {
        s += face_lo(n, bc, L, d, I) * (nb_lo(n, bc, p, d, I) - pc);
        s += face_hi(n, bc, L, d, I) * (nb_hi(n, bc, p, d, I) - pc);
    }
    return s;
}

/* O1:  D_I = - sum_d [ L_d(I) + L_d(I+e_d) ];  a cell is ACTIVE iff D_I != 0 (O9). */
static double diag_at(const int n[3], const int bc[3], const double *L, const int I[3]) {
    double s = 0.0;
    for (int d = 0; d < 3; ++d) s += face_lo(n, bc, L, d, I) + face_hi(n, bc, L, d, I);
    return -s;
}

/* out = A p on every cell */
void gmgo_apply(const int n[3], const int bc[3], const double *L, const double *p, double *out) {
#pragma omp parallel for schedule(static)
    for (int k = 0; k < n[2]; ++k)
        for (int j = 0; j < n[1]; ++j)
            for (int i = 0; i < n[0]; ++i) {
                int I[3] = {i, j, k};
                out[lin(n, i, j, k)] = apply_at(n, bc, L, p, I);
            }
}

void gmgo_diag(const int n[3], const int bc[3], const double *L, double *D) {
#pragma omp parallel for schedule(static)
    for (int k = 0; k < n[2]; ++k)
        for (int j = 0; j < n[1]; ++j)
            for (int i = 0; i < n[0]; ++i) {
                int I[3] = {i, j, k};
                D[lin(n, i, j, k)] = diag_at(n, bc, L, I);
            }
}

/* O9: r_I = b_I - (A p)_I on active cells, 0 on inactive cells. */
void gmgo_residual(const int n[3], const int bc[3], const double *L, const double *p,
                   const double *b, double *r) {
#pragma omp parallel for schedule(static)
    for (int k = 0; k < n[2]; ++k)
        for (int j = 0; j < n[1]; ++j)
            for (int i = 0; i < n[0]; ++i) {
                int I[3] = {i, j, k};
                i64 c = lin(n, i, j, k);
                r[c] = (diag_at(n, bc, L, I) != 0.0) ? b[c] - apply_at(n, bc, L, p, I) : 0.0;
            }
}

/* Plain L2 norm, sqrt(sum r^2); per-plane partial sums so the result does not depend on
 * the thread count. */
double gmgo_norm2(const int n[3], const double *r) {
    double *part = (double *)calloc((size_t)n[2], sizeof(double));
#pragma omp parallel for schedule(static)
    for (int k = 0; k < n[2]; ++k) {
        double s = 0.0;
        for (i64 c = (i64)k * n[0] * n[1]; c < (i64)(k + 1) * n[0] * n[1]; ++c) s += r[c] * r[c];
        part[k] = s;
    }
    double s = 0.0;
    for (int k = 0; k < n[2]; ++k) s += part[k];
    free(part);
    return sqrt(s);
}

double gmgo_dot(const int n[3], const double *a, const double *b) {
    double *part = (double *)calloc((size_t)n[2], sizeof(double));
#pragma omp parallel for schedule(static)
    for (int k = 0; k < n[2]; ++k) {
        double s = 0.0;
        for (i64 c = (i64)k * n[0] * n[1]; c < (i64)(k + 1) * n[0] * n[1]; ++c) s += a[c] * b[c];
        part[k] = s;
    }
    double s = 0.0;
    for (int k = 0; k < n[2]; ++k) s += part[k];
    free(part);
    return s;
}

/* O3: one colour half-sweep.  colour(I) = (i+j+k) mod 2, 0 = red.  Every active cell of
 * the colour:  p_I += omega * (b_I - (A p)_I) / D_I   (O8 update form; omega=1 is plain GS).
 * Cells of one colour never neighbour each other (periodic extents are even), so the
 * loop order inside a colour is immaterial. */
void gmgo_half_sweep(const int n[3], const int bc[3], const double *L, double *p,
                     const double *b, double omega, int colour) {
#pragma omp parallel for schedule(static)
    for (int k = 0; k < n[2]; ++k)
        for (int j = 0; j < n[1]; ++j)
            for (int i = 0; i < n[0]; ++i) {
                if (((i + j + k) & 1) != colour) continue;
                int I[3] = {i, j, k};
                double D = diag_at(n, bc, L, I);
                if (D == 0.0) continue;
                i64 c = lin(n, i, j, k);
                p[c] += omega * (b[c] - apply_at(n, bc, L, p, I)) / D;
            }
}

/* ------------------------------------------------------------------------------------
 * O4 (PAPER.md:47 S3.2 "downsamples every dimension independently"): direction d is
 * halved from one level to the next iff  n_d even  and  n_d/2 >= n_min  and
 * (axis d is Neumann or n_d/2 is even).  iso != 0 = classical isotropic coarsening:
 * coarsen all directions (of extent > 1: a 2-D grid is nx x ny x 1 with Neumann z) or stop.
 * Returns 1 if anything coarsens.
 * ---------------------------------------------------------------------------------- */
int gmgo_coarsen_rule(const int n[3], const int bc[3], int n_min, int iso, int c[3]) {
    int any = 0, all = 1;
    for (int d = 0; d < 3; ++d) {
        int h = n[d] / 2;
        int ok = (n[d] % 2 == 0) && (h >= n_min) && (bc[d] == GMGO_NEUMANN || h % 2 == 0);
        c[d] = ok ? 2 : 1;
        any |= ok;
        if (n[d] > 1) all &= ok; /* an extent-1 direction (2-D grid) has nothing to coarsen */
    }
    if (iso && !all) {
        c[0] = c[1] = c[2] = 1;
        return 0;
    }
    return any;
}

/* O5: coarse coefficient on the lower d-face of coarse cell J =
 *     (1/c_d) * sum of the fine L_d on the prod_{e!=d} c_e fine lower-d faces that tile it,
 * i.e. those of the fine children whose d-index is c_d*J_d.  (Area / distance.) */
void gmgo_coarsen_coeffs(const int nf[3], const int c[3], const double *Lf, double *Lc) {
    int nc[3] = {nf[0] / c[0], nf[1] / c[1], nf[2] / c[2]};
    i64 Nf = ncells(nf), Nc = ncells(nc);
    for (int d = 0; d < 3; ++d) {
        int e1 = (d + 1) % 3, e2 = (d + 2) % 3;
        for (int K = 0; K < nc[2]; ++K)
            for (int J = 0; J < nc[1]; ++J)
                for (int I = 0; I < nc[0]; ++I) {
                    int Jc[3] = {I, J, K};
                    double s = 0.0;
                    for (int a = 0; a < c[e1]; ++a)
                        for (int b = 0; b < c[e2]; ++b) {
                            int F[3];
                            F[d] = c[d] * Jc[d];
                            F[e1] = c[e1] * Jc[e1] + a;
                            F[e2] = c[e2] * Jc[e2] + b;
                            s += Lf[(i64)d * Nf + lin(nf, F[0], F[1], F[2])];
                        }
                    Lc[(i64)d * Nc + lin(nc, I, J, K)] = s / (double)c[d];
                }
    }
}

/* O6: restriction = SUM of the residual over the m = c_x c_y c_z children. */
void gmgo_restrict_sum(const int nf[3], const int c[3], const double *rf, double *bc_) {
    int nc[3] = {nf[0] / c[0], nf[1] / c[1], nf[2] / c[2]};
    for (int K = 0; K < nc[2]; ++K)
        for (int J = 0; J < nc[1]; ++J)
            for (int I = 0; I < nc[0]; ++I) {
                double s = 0.0;
                for (int a = 0; a < c[2]; ++a)
                    for (int b = 0; b < c[1]; ++b)
                        for (int e = 0; e < c[0]; ++e)
                            s += rf[lin(nf, c[0] * I + e, c[1] * J + b, c[2] * K + a)];
                bc_[lin(nc, I, J, K)] = s;
            }
}

/* O6: prolongation = piecewise-constant injection, added unscaled: p_I += e_{parent(I)}. */
void gmgo_prolong_add(const int nf[3], const int c[3], const double *ec, double *pf) {
    int nc[3] = {nf[0] / c[0], nf[1] / c[1], nf[2] / c[2]};
    for (int k = 0; k < nf[2]; ++k)
        for (int j = 0; j < nf[1]; ++j)
            for (int i = 0; i < nf[0]; ++i)
                pf[lin(nf, i, j, k)] += ec[lin(nc, i / c[0], j / c[1], k / c[2])];
}

/* ------------------------------------------------------------------------------------
 * Level hierarchy (D3): shapes by O4, coefficients by O5.
 * ---------------------------------------------------------------------------------- */
typedef struct {
    int nlev;
    int bc[3];
    int n[GMGO_MAXLEV][3];
    int c[GMGO_MAXLEV][3]; /* factors from level l to l+1; (1,1,1) on the last level */
    double *L[GMGO_MAXLEV];
    double *x[GMGO_MAXLEV]; /* level >= 1 unknowns */
    double *b[GMGO_MAXLEV]; /* level >= 1 right-hand sides */
    double *r;              /* level-0-sized residual scratch */
    /* parameters (O7, O8) */
    int nu1, nu2, nuc;
    double omega, omega0, omega_min, omega_down, omega_up;
    int adaptive;
} gmgo_hier;

/* L32: FP32 input coefficients (the same bits the GPU gets), shape 3*N. */
gmgo_hier *gmgo_hier_create(const int n[3], const int bc[3], const float *L32, int n_min, int iso) {
    gmgo_hier *h = (gmgo_hier *)calloc(1, sizeof(gmgo_hier));
    for (int d = 0; d < 3; ++d) {
        h->bc[d] = bc[d];
        h->n[0][d] = n[d];
    }
    i64 N = ncells(n);
    h->L[0] = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    for (i64 t = 0; t < 3 * N; ++t) h->L[0][t] = (double)L32[t];
    /* O2: the wall plane L_d(index 0) of a Neumann axis is ignored = treated as 0.  Store
     * the 0 so that coarsening (O5) sees the wall too. */
    for (int d = 0; d < 3; ++d) {
        if (bc[d] != GMGO_NEUMANN) continue;
        for (int k = 0; k < n[2]; ++k)
            for (int j = 0; j < n[1]; ++j)
                for (int i = 0; i < n[0]; ++i) {
                    int I[3] = {i, j, k};
                    if (I[d] == 0) h->L[0][(i64)d * N + lin(n, i, j, k)] = 0.0;
                }
    }
    h->r = (double *)calloc((size_t)N, sizeof(double));
    int l = 0;
    while (l + 1 < GMGO_MAXLEV && gmgo_coarsen_rule(h->n[l], bc, n_min, iso, h->c[l])) {
        for (int d = 0; d < 3; ++d) h->n[l + 1][d] = h->n[l][d] / h->c[l][d];
        i64 Nc = ncells(h->n[l + 1]);
        h->L[l + 1] = (double *)malloc(sizeof(double) * 3 * (size_t)Nc);
        gmgo_coarsen_coeffs(h->n[l], h->c[l], h->L[l], h->L[l + 1]);
        h->x[l + 1] = (double *)calloc((size_t)Nc, sizeof(double));
        h->b[l + 1] = (double *)calloc((size_t)Nc, sizeof(double));
        ++l;
    }
    h->c[l][0] = h->c[l][1] = h->c[l][2] = 1;
    h->nlev = l + 1;
    h->nu1 = 2; h->nu2 = 2; h->nuc = 32;                       /* O7 */
    h->omega0 = 1.0; h->omega = 1.0; h->omega_min = 0.5;       /* O8 */
    h->omega_down = 0.125; h->omega_up = 0.03125; h->adaptive = 1;
    return h;
}

void gmgo_hier_destroy(gmgo_hier *h) {
    if (!h) return;
    for (int l = 0; l < h->nlev; ++l) { free(h->L[l]); free(h->x[l]); free(h->b[l]); }
    free(h->r);
    free(h);
}

int gmgo_hier_nlev(const gmgo_hier *h) { return h->nlev; }
void gmgo_hier_shape(const gmgo_hier *h, int lev, int n[3], int c[3]) {
    for (int d = 0; d < 3; ++d) { n[d] = h->n[lev][d]; c[d] = h->c[lev][d]; }
}
const double *gmgo_hier_L(const gmgo_hier *h, int lev) { return h->L[lev]; }
void gmgo_hier_set_params(gmgo_hier *h, int nu1, int nu2, int nuc, double omega0, double omega_min,
                          double omega_down, double omega_up, int adaptive) {
    h->nu1 = nu1; h->nu2 = nu2; h->nuc = nuc; h->omega0 = omega0; h->omega = omega0;
    h->omega_min = omega_min; h->omega_down = omega_down; h->omega_up = omega_up;
    h->adaptive = adaptive;
}
double gmgo_hier_omega(const gmgo_hier *h) { return h->omega; }
void gmgo_hier_set_omega(gmgo_hier *h, double w) { h->omega = w; }

static void sweeps(const gmgo_hier *h, int l, double *x, const double *b, double omega, int count,
                   int first_colour) {
    for (int s = 0; s < count; ++s) {
        gmgo_half_sweep(h->n[l], h->bc, h->L[l], x, b, omega, first_colour);
        gmgo_half_sweep(h->n[l], h->bc, h->L[l], x, b, omega, 1 - first_colour);
    }
}

/* O7: V(nu1,nu2) cycle on level l for A^l x = b, x given.  sym != 0 is the symmetric
 * variant used as a CG preconditioner (O11): post-sweeps black->red, coarsest level
 * nuc/2 sweeps red->black then nuc/2 sweeps black->red. */
static void vcycle_rec(gmgo_hier *h, int l, double *x, const double *b, double omega, int sym) {
    if (l == h->nlev - 1) {
        if (!sym) {
            sweeps(h, l, x, b, omega, h->nuc, 0);
        } else {
            sweeps(h, l, x, b, omega, h->nuc / 2, 0);
            sweeps(h, l, x, b, omega, h->nuc / 2, 1);
        }
        return;
    }
    sweeps(h, l, x, b, omega, h->nu1, 0);
    i64 Nf = ncells(h->n[l]);
    double *r = (l == 0) ? h->r : (double *)malloc(sizeof(double) * (size_t)Nf);
    gmgo_residual(h->n[l], h->bc, h->L[l], x, b, r);
    gmgo_restrict_sum(h->n[l], h->c[l], r, h->b[l + 1]);
    if (l != 0) free(r);
    memset(h->x[l + 1], 0, sizeof(double) * (size_t)ncells(h->n[l + 1]));
    vcycle_rec(h, l + 1, h->x[l + 1], h->b[l + 1], omega, sym);
    gmgo_prolong_add(h->n[l], h->c[l], h->x[l + 1], x);
    sweeps(h, l, x, b, omega, h->nu2, sym ? 1 : 0);
}

void gmgo_vcycle(gmgo_hier *h, double *x, const double *b, double omega, int sym) {
    vcycle_rec(h, 0, x, b, omega, sym);
}

/* single-level entry points for per-operator parity tests */
void gmgo_level_residual(gmgo_hier *h, int l, const double *x, const double *b, double *r) {
    gmgo_residual(h->n[l], h->bc, h->L[l], x, b, r);
}
void gmgo_level_sweeps(gmgo_hier *h, int l, double *x, const double *b, double omega, int count,
                       int first_colour) {
    sweeps(h, l, x, b, omega, count, first_colour);
}

/* ------------------------------------------------------------------------------------
 * O9 + O8: GMG-RBGS solve loop.
 *   r_ref = ||z||_2 over active cells; if 0 -> 0 iterations.
 *   rho_0 = ||z - A p||_2;  while rho_k > tol*r_ref and k < maxiter:
 *       V-cycle; k++; rho_k = ||z - A p||_2; omega update:
 *           rho_k >  rho_{k-1}:  omega <- max(omega_min, omega - omega_down)   (growth)
 *           else              :  omega <- min(1,         omega + omega_up)     (decay)
 * history[k] = rho_k / r_ref (k = 0..iterations), omegas[k] = omega used in cycle k+1.
 * Returns the number of V-cycles; *status = 0 converged, 1 not converged.
 * omega persists in the hierarchy across calls (time stepping).
 * ---------------------------------------------------------------------------------- */
static double active_norm(const gmgo_hier *h, const double *z) {
    /* ||z||_2 over active cells only */
    const int *n = h->n[0];
    double s = 0.0;
    for (int k = 0; k < n[2]; ++k)
        for (int j = 0; j < n[1]; ++j)
            for (int i = 0; i < n[0]; ++i) {
                int I[3] = {i, j, k};
                if (diag_at(n, h->bc, h->L[0], I) != 0.0) {
                    double v = z[lin(n, i, j, k)];
                    s += v * v;
                }
            }
    return sqrt(s);
}

int gmgo_solve_gmg_rbgs(gmgo_hier *h, double *p, const double *z, double tol, int maxiter,
                        double *history, double *omegas, int *status, double *r_ref_out) {
    const int *n = h->n[0];
    double r_ref = active_norm(h, z);
    if (r_ref_out) *r_ref_out = r_ref;
    if (r_ref == 0.0) {
        if (history) history[0] = 0.0;
        *status = 0;
        return 0;
    }
    gmgo_residual(n, h->bc, h->L[0], p, z, h->r);
    double rho = gmgo_norm2(n, h->r);
    int k = 0;
    if (history) history[0] = rho / r_ref;
    while (rho > tol * r_ref && k < maxiter) {
        if (omegas) omegas[k] = h->omega;
        vcycle_rec(h, 0, p, z, h->omega, 0);
        ++k;
        gmgo_residual(n, h->bc, h->L[0], p, z, h->r);
        double rho_new = gmgo_norm2(n, h->r);
        if (history) history[k] = rho_new / r_ref;
        if (h->adaptive) {
            if (rho_new > rho) {
                double w = h->omega - h->omega_down;
                h->omega = (w > h->omega_min) ? w : h->omega_min;
            } else {
                double w = h->omega + h->omega_up;
                h->omega = (w < 1.0) ? w : 1.0;
            }
        }
        rho = rho_new;
    }
    *status = (rho <= tol * r_ref) ? 0 : 1;
    return k;
}

/* ------------------------------------------------------------------------------------
 * O10: preconditioned CG on A p = z.  precond 0 = Jacobi
 * (s = r / D on active cells, 0 elsewhere); precond 1 = one symmetric V(nu1,nu2) cycle from
 * a zero guess at omega = 1 (O11, "GMG-preconditioned PCG" of BASELINE.json:north_star).
 *   r = z - A p; s = M^-1 r; d = s; rho = r.s;
 *   loop { q = A d; alpha = rho/(d.q); p += alpha d; r -= alpha q;
 *          test ||r||_2 <= tol ||z||_2; s = M^-1 r; rho' = r.s; d = s + (rho'/rho) d; rho = rho' }
 * The recursive residual drives the test; history[k] = ||r_k|| / ||z||.  *true_res = true
 * relative residual recomputed at exit.  status: 0 ok, 1 not converged, -5 breakdown (d.q == 0).
 * ---------------------------------------------------------------------------------- */
static void precondition(gmgo_hier *h, int precond, const double *r, double *s) {
    const int *n = h->n[0];
    if (precond == 0) {
        for (int k = 0; k < n[2]; ++k)
            for (int j = 0; j < n[1]; ++j)
                for (int i = 0; i < n[0]; ++i) {
                    int I[3] = {i, j, k};
                    double D = diag_at(n, h->bc, h->L[0], I);
                    i64 c = lin(n, i, j, k);
                    s[c] = (D != 0.0) ? r[c] / D : 0.0;
                }
    } else {
        memset(s, 0, sizeof(double) * (size_t)ncells(n));
        vcycle_rec(h, 0, s, r, 1.0, 1);
    }
}

int gmgo_solve_pcg(gmgo_hier *h, int precond, double *p, const double *z, double tol, int maxiter,
                   double *history, int *status, double *true_res) {
    const int *n = h->n[0];
    i64 N = ncells(n);
    double r_ref = active_norm(h, z);
    *status = 0;
    if (r_ref == 0.0) {
        if (history) history[0] = 0.0;
        if (true_res) *true_res = 0.0;
        return 0;
    }
    double *r = (double *)malloc(sizeof(double) * (size_t)N);
    double *s = (double *)malloc(sizeof(double) * (size_t)N);
    double *d = (double *)malloc(sizeof(double) * (size_t)N);
    double *q = (double *)malloc(sizeof(double) * (size_t)N);
    gmgo_residual(n, h->bc, h->L[0], p, z, r);
    double rn = gmgo_norm2(n, r);
    if (history) history[0] = rn / r_ref;
    int k = 0;
    if (rn > tol * r_ref && maxiter > 0) {
        precondition(h, precond, r, s);
        memcpy(d, s, sizeof(double) * (size_t)N);
        double rho = gmgo_dot(n, r, s);
        while (k < maxiter) {
            gmgo_apply(n, h->bc, h->L[0], d, q);
            /* inactive cells have an all-zero row, so q = 0 there already */
            double dq = gmgo_dot(n, d, q);
            if (dq == 0.0) { *status = -5; break; }
            double alpha = rho / dq;
            for (i64 c = 0; c < N; ++c) { p[c] += alpha * d[c]; r[c] -= alpha * q[c]; }
            ++k;
            rn = gmgo_norm2(n, r);
            if (history) history[k] = rn / r_ref;
            if (rn <= tol * r_ref) break;
            precondition(h, precond, r, s);
            double rho_new = gmgo_dot(n, r, s);
            double beta = rho_new / rho;
            for (i64 c = 0; c < N; ++c) d[c] = s[c] + beta * d[c];
            rho = rho_new;
        }
    }
    gmgo_residual(n, h->bc, h->L[0], p, z, r);
    double tr = gmgo_norm2(n, r) / r_ref;
    if (true_res) *true_res = tr;
    if (*status == 0) *status = (rn <= tol * r_ref) ? 0 : 1;
    free(r); free(s); free(d); free(q);
    return k;
}

/* ------------------------------------------------------------------------------------
 * N1: the two steps either side of the Poisson solve in a
 * staggered projection step (Fig. 2 "predictor + corrector steps", one solve
 * each; PAPER.md:9 staggered finite volume).  u is component-major like L: u[d*N + idx] is
 * the velocity on the LOWER d-face of cell idx.
 *
 *   divergence:  z_I = sum_d [ u_d(I+e_d) - u_d(I) ]     (what configs[1..3] hand to the solver)
 *       upper face of the last cell: periodic -> u_d(index 0); Neumann -> the prescribed
 *       upper-wall value wall_hi[d].  On a Neumann axis u_d(index 0) is the lower-wall value.
 *   projection:  u_d(I) -= L_d(I) * (p_I - p_{I-e_d})     (unit spacing; reading O1's face)
 *       Neumann wall faces carry coefficient 0 (reading O2): untouched.
 * Identity that ties both to the operator:  div(project(u, p)) = div(u) - A p.
 * ---------------------------------------------------------------------------------- */
void gmgo_divergence(const int n[3], const int bc[3], const double *u, const double wall_hi[3],
                     double *z) {
    i64 N = ncells(n);
    for (int k = 0; k < n[2]; ++k)
        for (int j = 0; j < n[1]; ++j)
            for (int i = 0; i < n[0]; ++i) {
                int I[3] = {i, j, k};
                double s = 0.0;
                for (int d = 0; d < 3; ++d) {
                    double lo = u[(i64)d * N + lin(n, i, j, k)];
                    double hi;
                    if (I[d] == n[d] - 1) {
                        if (bc[d] == GMGO_NEUMANN) {
                            hi = wall_hi[d];
                        } else {
                            int J[3] = {i, j, k};
                            J[d] = 0;
                            hi = u[(i64)d * N + lin(n, J[0], J[1], J[2])];
                        }
                    } else {
                        int J[3] = {i, j, k};
                        J[d] = I[d] + 1;
                        hi = u[(i64)d * N + lin(n, J[0], J[1], J[2])];
                    }
                    s += hi - lo;
                }
                z[lin(n, i, j, k)] = s;
            }
}

void gmgo_project(const int n[3], const int bc[3], const double *L, const double *p, double *u) {
    i64 N = ncells(n);
    for (int d = 0; d < 3; ++d)
        for (int k = 0; k < n[2]; ++k)
            for (int j = 0; j < n[1]; ++j)
                for (int i = 0; i < n[0]; ++i) {
                    int I[3] = {i, j, k};
                    double w = face_lo(n, bc, L, d, I); /* 0 on a Neumann wall face */
                    double pm = nb_lo(n, bc, p, d, I);
                    i64 c = lin(n, i, j, k);
                    u[(i64)d * N + c] -= w * (p[c] - pm);
                }
}

/* ------------------------------------------------------------------------------------
 * N2 (PAPER.md:43 S3.1 "PCG can be used as a smoother", Table 1's
 * middle row "GMG-PCG" at PAPER.md:37): the SAME V(nu1,nu2) cycle as O7 with every group of
 * RBGS sweeps replaced by as many Jacobi-preconditioned CG iterations, restarted from the
 * current iterate of that level.  The paper gives no parameter for it: reading O12.
 *
 * O12a, the smoother: m CG iterations on A^l x = b from the given x (A is negative
 * semi-definite, so r.s and d.q are negative and alpha positive):
 *     r = b - A x (0 on inactive cells, O9);  s = r/D (0 on inactive);  d = s;  rho = r.s; rho0 = rho
 *     repeat m times:  q = A d;  alpha = rho/(d.q);  x += alpha d;  r -= alpha q;
 *                      s = r/D;  rho' = r.s;  d = s + (rho'/rho) d;  rho = rho'
 * Every level is singular (periodic axes and homogeneous Neumann walls only: constants span the
 * null space), and CG -- unlike Gauss-Seidel -- amplifies any component of the right-hand side
 * along the null vector without bound (d.q -> 0 there).  Restricted residuals carry such a
 * component at rounding level, so the initial residual is made compatible first:
 *     r -= mean of r over the active cells.
 * Guards: the iteration stops early when rho is not < 0 at entry, when d.q is not < 0, once
 * |rho| <= 1e-8 |rho0| (preconditioned residual reduced by 1e-4, far more than a smoother or a
 * coarsest-level solve needs; below that an FP32 run approaches its own rounding noise), or when
 * a step length alpha > 16 n_max^2 comes out (n_max = the level's largest extent).  In exact
 * arithmetic 1/alpha is bounded below by the smallest non-zero eigenvalue of D^-1 A, which is
 * about (pi/n_max)^2/6 for uniform coefficients, i.e. alpha <= 0.6 n_max^2: a step 26 times
 * longer than that is a direction that has drifted into the null space, not a solve.
 * ---------------------------------------------------------------------------------- */
#define GMGO_CGS_FREEZE 1e-8

void gmgo_level_cg_smooth(gmgo_hier *h, int l, double *x, const double *b, int m) {
    const int *n = h->n[l];
    i64 N = ncells(n);
    if (m <= 0) return;
    double *r = (double *)malloc(sizeof(double) * (size_t)N);
    double *s = (double *)malloc(sizeof(double) * (size_t)N);
    double *d = (double *)malloc(sizeof(double) * (size_t)N);
    double *q = (double *)malloc(sizeof(double) * (size_t)N);
    double *D = (double *)malloc(sizeof(double) * (size_t)N);
    gmgo_diag(n, h->bc, h->L[l], D);
    gmgo_residual(n, h->bc, h->L[l], x, b, r);
    double sum = 0.0, cnt = 0.0;
    for (i64 c = 0; c < N; ++c)
        if (D[c] != 0.0) { sum += r[c]; cnt += 1.0; }
    if (cnt > 0.0)
        for (i64 c = 0; c < N; ++c)
            if (D[c] != 0.0) r[c] -= sum / cnt;
    for (i64 c = 0; c < N; ++c) s[c] = (D[c] != 0.0) ? r[c] / D[c] : 0.0;
    memcpy(d, s, sizeof(double) * (size_t)N);
    double rho = gmgo_dot(n, r, s);
    const double rho0 = rho;
    int nmax = n[0] > n[1] ? n[0] : n[1];
    if (n[2] > nmax) nmax = n[2];
    const double alpha_cap = 16.0 * (double)nmax * (double)nmax;
    int frozen = !(rho < 0.0);
    for (int it = 0; it < m && !frozen; ++it) {
        gmgo_apply(n, h->bc, h->L[l], d, q);
        double dq = gmgo_dot(n, d, q);
        if (!(dq < 0.0)) break;
        double alpha = rho / dq;
        if (alpha > alpha_cap) break;
        for (i64 c = 0; c < N; ++c) { x[c] += alpha * d[c]; r[c] -= alpha * q[c]; }
        if (it == m - 1) break;
        for (i64 c = 0; c < N; ++c) s[c] = (D[c] != 0.0) ? r[c] / D[c] : 0.0;
        double rho_new = gmgo_dot(n, r, s);
        double beta = rho_new / rho;
        for (i64 c = 0; c < N; ++c) d[c] = s[c] + beta * d[c];
        rho = rho_new;
        if (!(fabs(rho) > GMGO_CGS_FREEZE * fabs(rho0))) frozen = 1;
    }
    free(r); free(s); free(d); free(q); free(D);
}

/* O12b: the cycle.  Coarsest level: nuc CG iterations from the zero guess. */
static void vcycle_cgs_rec(gmgo_hier *h, int l, double *x, const double *b) {
    if (l == h->nlev - 1) {
        gmgo_level_cg_smooth(h, l, x, b, h->nuc);
        return;
    }
    gmgo_level_cg_smooth(h, l, x, b, h->nu1);
    i64 Nf = ncells(h->n[l]);
    double *r = (l == 0) ? h->r : (double *)malloc(sizeof(double) * (size_t)Nf);
    gmgo_residual(h->n[l], h->bc, h->L[l], x, b, r);
    gmgo_restrict_sum(h->n[l], h->c[l], r, h->b[l + 1]);
    if (l != 0) free(r);
    memset(h->x[l + 1], 0, sizeof(double) * (size_t)ncells(h->n[l + 1]));
    vcycle_cgs_rec(h, l + 1, h->x[l + 1], h->b[l + 1]);
    gmgo_prolong_add(h->n[l], h->c[l], h->x[l + 1], x);
    gmgo_level_cg_smooth(h, l, x, b, h->nu2);
}

void gmgo_vcycle_cgs(gmgo_hier *h, double *x, const double *b) { vcycle_cgs_rec(h, 0, x, b); }

/* O12c: the solve loop is O9's, without the relaxation factor: V-cycles until
 * ||z - A p||_2 <= tol ||z||_2 over active cells or maxiter cycles. */
int gmgo_solve_gmg_cgs(gmgo_hier *h, double *p, const double *z, double tol, int maxiter,
                       double *history, int *status, double *r_ref_out) {
    const int *n = h->n[0];
    double r_ref = active_norm(h, z);
    if (r_ref_out) *r_ref_out = r_ref;
    if (r_ref == 0.0) {
        if (history) history[0] = 0.0;
        *status = 0;
        return 0;
    }
    gmgo_residual(n, h->bc, h->L[0], p, z, h->r);
    double rho = gmgo_norm2(n, h->r);
    int k = 0;
    if (history) history[0] = rho / r_ref;
    while (rho > tol * r_ref && k < maxiter) {
        vcycle_cgs_rec(h, 0, p, z);
        ++k;
        gmgo_residual(n, h->bc, h->L[0], p, z, h->r);
        rho = gmgo_norm2(n, h->r);
        if (history) history[k] = rho / r_ref;
    }
    *status = (rho <= tol * r_ref) ? 0 : 1;
    return k;
}

/* gmg.h -- C-ABI boundary of the B200-native geometric-multigrid pressure-Poisson solve
 * of arxiv/paper_2607_07687 ("Scaling WaterLily.jl with MPI and an improved geometric
 * multigrid solver").  PAPER.md = /root/reference/PAPER.md.
 *
 * What is solved (PAPER.md:43 S3.1 "variable-coefficient Poisson equations arising in
 * multiphase and immersed-boundary flows"; BASELINE.json:north_star):
 *
 *     (A p)_I = sum_d [ L_d(I) (p_{I-e_d} - p_I) + L_d(I+e_d) (p_{I+e_d} - p_I) ] = z_I
 *
 * on an nx*ny*nz Cartesian grid, L_d(I) >= 0 the coefficient on the LOWER d-face of cell
 * I (reading O1).  Solvers: GMG V-cycles with the adaptive under-relaxed
 * red-black Gauss-Seidel smoother (PAPER.md:43 S3.1) on anisotropically coarsened levels
 * (PAPER.md:47 S3.2); Jacobi-PCG and GMG-preconditioned PCG as comparison solvers
 * (PAPER.md:31, 39 S3).
 *
 * Conventions
 *  - Layout: cell I=(i,j,k) at linear index i + nx*(j + ny*k) (x fastest), FP32.
 *    L is component-major, [3][nz][ny][nx]: L[d*N + idx] = lower d-face of cell idx.
 *  - bc[d]: GMG_BC_PERIODIC (index wrap; extent must be even) or GMG_BC_NEUMANN
 *    (homogeneous: the wall faces carry coefficient 0; the caller's plane L_d(index 0)
 *    on that axis is IGNORED and there is no upper wall face).  DESIGN.md reading O2.
 *  - Pointers named *_dev are CUDA device pointers owned by the CALLER (torch
 *    allocations); *_host are host pointers.  The library never frees caller memory.
 *    The big arrays of the level hierarchy live in the caller-provided workspace; the
 *    library itself allocates only < 4 MB of device scalars / reduction partials /
 *    history and its pinned host mirror.
 *  - Alignment: every *_dev array handed to the library (p, z, L, u, the hooks' operands) must
 *    start on a 16-byte boundary (the fast paths move float4s and TMA boxes); a misaligned
 *    pointer is refused with GMG_EINVAL.  The workspace must be 256-byte aligned.
 *  - `stream` is a cudaStream_t passed as void* (0 = legacy default stream).  All work
 *    is enqueued on it; gmg_solve and the gmg_op_* hooks synchronise it before returning.
 *  - Return codes: 0 ok; >0 warning (result valid); <0 error (gmg_last_error has text).
 *    No exceptions, nothing printed.
 *  - Determinism: all reductions are two-stage, fixed order, FP64 partials; same inputs
 *    give bit-identical p and identical iteration counts run to run.
 *  - There is NO CPU fallback: every step runs in CUDA kernels (sm_100a).
 */
#ifndef GMG_H_
#define GMG_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gmg_ctx gmg_ctx;

enum { GMG_BC_PERIODIC = 0, GMG_BC_NEUMANN = 1 };
/* GMG_GMG_PCG: CG preconditioned by one symmetric V-cycle (BASELINE.json's "GMG-preconditioned PCG",
 * reading O11).  GMG_GMG_CGS: the paper's own "GMG-PCG" of Table 1 -- the V-cycle
 * whose smoother is Jacobi-PCG instead of RBGS (reading O12): every group of nu sweeps becomes nu CG
 * iterations restarted from the level's current iterate, the restart residual made mean-free over
 * the active cells (every level is singular; CG amplifies a null-space component without bound),
 * and a smoothing ends early once d.q is not < 0, |r.s| <= 1e-8 |r.s at the restart|, or a step
 * length above 16 n_max^2 comes out (a direction that drifted into the null space). */
enum { GMG_PCG = 0, GMG_GMG_PCG = 1, GMG_GMG_RBGS = 2, GMG_GMG_CGS = 3 };
enum { GMG_COARSEN_ANISO = 0, GMG_COARSEN_ISO = 1 };
enum {
    GMG_OK = 0,
    GMG_NOT_CONVERGED = 1, /* maxiter reached; p holds the last iterate */
    GMG_EINVAL = -1,       /* bad argument */
    GMG_ESTATE = -2,       /* call order: workspace / coefficients not set */
    GMG_ECUDA = -3,        /* a CUDA call failed */
    GMG_ENOMEM = -4,       /* workspace too small */
    GMG_EBREAKDOWN = -5    /* PCG: d.q == 0 */
};

/* Parameters; defaults (gmg_default_params) are DESIGN.md readings O4, O7, O8. */
typedef struct {
    int nu_pre;        /* pre-smoothing RBGS sweeps per level           (2)  O7 */
    int nu_post;       /* post-smoothing sweeps per level               (2)  O7 */
    int nu_coarse;     /* sweeps on the coarsest level, even            (32) O7 */
    float omega0;      /* initial relaxation factor                     (1)  O8 */
    float omega_min;   /* lower bound of omega                          (1/2) */
    float omega_down;  /* decrement after a V-cycle that grew the residual (1/8) */
    float omega_up;    /* increment after a V-cycle that shrank it      (1/32) */
    int adaptive;      /* 1: adapt omega after each V-cycle */
    int coarsen_mode;  /* GMG_COARSEN_ANISO or GMG_COARSEN_ISO */
    int n_min;         /* a direction coarsens only while n_d/2 >= n_min (4) O4 */
    int fast_path;     /* 1: fused/tiled kernels where shapes allow; 0: generic kernels only */
    int use_graph;     /* 1: V-cycle captured in a CUDA graph; 0: plain launches */
    int tma_min_cells; /* levels with at least this many cells (and nx % 128 == 0) use the TMA-fed
                          z-marching kernels; smaller ones the register-fed tiles (1048576);
                          0 = whenever the shape allows, -1 = never */
    int cluster_tail;  /* 1: the coarse levels that fit the shared memory of a cluster of 8 CTAs
                          (each at most 32768 cells) run as ONE thread-block-cluster kernel;
                          0: only what fits a single CTA does (1) */
    int fused_norm;    /* 1: on a finest level that runs the TMA-fed sweep, the stopping-test norm
                          ||z - A p_k|| is accumulated by the first pre-smoothing sweep of cycle k+1
                          (out of place, so p_k survives when the test ends the solve) instead of
                          by a 20 B/cell pass of its own after every cycle; the cycle expected to be
                          the last (rate-based prediction, or the maxiter-th) takes the plain pass
                          instead, so that no sweep is wasted at the exit; same iterates, same test (1) */
    int uniform_tiles; /* 1: gmg_set_coeffs marks the bricks (128 x 8 x 8 cells) of every TMA-fed level
                          whose stored coefficients all equal the level's constant per direction -- 1 on
                          the finest level (the BDIM coefficient away from bodies; north_star "L in
                          [0,1]"), (prod_{e != d} C_e) / C_d on coarser ones (reading O5 applied to ones) --
                          and a CTA whose footprint holds only such bricks and no wall skips the three
                          coefficient streams: 12 instead of 24 B/cell per sweep, 8 + 4/m instead of
                          20 + 4/m for the residual pass.  LOSSLESS: the same operations run on the
                          constants, every cell gets the same bits (SURVEY.md S8(d) "a lossless 'tile is
                          all L=1' flag ... honest only if reported as such": gmg_stats.uniform_fraction
                          and bytes_as_run report it).  0: every CTA loads its coefficients (1) */
    int small_cg;      /* 1: GMG_GMG_CGS runs a whole smoothing (restart + nu CG iterations) of a level of
                          at most 4096 cells as ONE single-CTA kernel instead of 4 launches per iteration;
                          same arithmetic and the same summation order, every cell gets the same bits (1) */
} gmg_params_t;

/* Statistics of the last gmg_solve. */
typedef struct {
    int solver;
    int status;             /* the code gmg_solve returned */
    int iterations;         /* V-cycles (GMG-RBGS, GMG-CGS) or CG iterations (PCG, GMG-PCG) */
    int levels;
    double omega_final;     /* relaxation factor after the solve (persists in the ctx) */
    double resid_ref;       /* ||z||_2 over active cells */
    double resid_init_rel;  /* ||z - A p0||_2 / resid_ref */
    double resid_final_rel; /* TRUE relative residual at exit (recomputed for PCG) */
    double gpu_ms;          /* CUDA-event time of the enqueued solve on `stream` */
    double bytes_algorithmic; /* algorithmic HBM bytes of the solve (DESIGN.md table) */
    long long kernel_launches; /* kernels launched (graph nodes count) by the solve */
    int history_len;        /* entries available through gmg_history (iterations+1) */
    double uniform_fraction; /* share of the finest level's cells swept by CTAs on the lean path
                                (uniform_tiles; 0 when off or when level 0 is not TMA-fed) */
    double bytes_as_run;    /* bytes_algorithmic minus the coefficient bytes the lean path did not move */
    double uniform_fraction_residual; /* the same share for the residual + restriction pass (its own tiling) */
} gmg_stats_t;

/* Level table and workspace size for a grid WITHOUT creating a context (host-only: no CUDA call).
 * Same rule gmg_create applies (reading O4).  params == NULL: defaults. */
#define GMG_PLAN_MAX_LEVELS 24
typedef struct {
    int levels;
    int n[GMG_PLAN_MAX_LEVELS][3];  /* extents of each level */
    int c[GMG_PLAN_MAX_LEVELS][3];  /* coarsening factors to the next level */
    int tail_start;                 /* first level run inside the single-CTA tail kernel */
    size_t workspace_bytes;         /* what gmg_workspace_bytes will report */
} gmg_plan_t;
int gmg_plan(int nx, int ny, int nz, const int bc[3], const gmg_params_t* params, gmg_plan_t* out);

/* -- life cycle ------------------------------------------------------------------------ */

/* Create a context for an nx*ny*nz grid.  A periodic axis needs an even extent (red/black
 * colouring, reading O3).  An extent of 1 is allowed on a Neumann axis: nx*ny*1 is the 2-D mode
 * (Fig. 2 left "2D flow around a circular cylinder"); that axis never coarsens and
 * its coefficients are ignored.  Builds the level-shape table by the
 * anisotropic rule (reading O4).  Uses the current CUDA device. */
int gmg_create(gmg_ctx** out, int nx, int ny, int nz, const int bc[3]);
void gmg_destroy(gmg_ctx* ctx);
const char* gmg_last_error(const gmg_ctx* ctx);

void gmg_default_params(gmg_params_t* out);
/* Changes parameters; rebuilds the level table (coefficients must be set again) and
 * resets omega to omega0.  Must precede gmg_workspace_bytes / gmg_set_workspace. */
int gmg_set_params(gmg_ctx* ctx, const gmg_params_t* params);
int gmg_get_params(const gmg_ctx* ctx, gmg_params_t* out);

/* Bytes of device workspace needed (coarse levels: L, p, b; ping-pong buffers; 4 PCG
 * vectors), and hand-over of a caller-allocated block (256-byte aligned). */
size_t gmg_workspace_bytes(const gmg_ctx* ctx);
int gmg_set_workspace(gmg_ctx* ctx, void* ws_dev, size_t bytes);

/* Set the level-0 face coefficients (kept BY POINTER: L_dev must stay valid and
 * unchanged until the next gmg_set_coeffs / gmg_destroy) and coarsen them to every level
 * (reading O5: L_d^{l+1}(J) = (1/c_d) * sum of the fine L_d on the faces tiling the coarse
 * face).  Checks on device that every value is finite and >= 0 (GMG_EINVAL otherwise).
 * Resets omega to omega0.  Calling it again with the SAME pointer after rewriting the array in
 * place (a moving body) keeps the captured solve graphs; a new pointer drops them. */
int gmg_set_coeffs(gmg_ctx* ctx, const float* L_dev, void* stream);

/* Solve A p = z.  p_dev: in = initial guess, out = solution (in place).  Stops when
 * ||z - A p||_2 <= tol * ||z||_2 (norms over active cells, reading O9) or after maxiter
 * iterations (tol = 0 runs exactly maxiter).  solver: GMG_PCG, GMG_GMG_PCG, GMG_GMG_RBGS, GMG_GMG_CGS.
 * The whole iteration runs on the device (a CUDA-graph WHILE loop); the host reads one
 * status block at the end.  Returns GMG_OK / GMG_NOT_CONVERGED or an error. */
int gmg_solve(gmg_ctx* ctx, float* p_dev, const float* z_dev, float tol, int maxiter,
              int solver, void* stream);

/* Same solve with HOST buffers (pinned or pageable): copies z (and the initial guess p)
 * host->device into library-held staging carved from the workspace, solves, copies p back.
 * This is the end-to-end entry point bench.py times as `e2e`. */
int gmg_solve_host(gmg_ctx* ctx, float* p_host, const float* z_host, float tol, int maxiter,
                   int solver, void* stream);

/* Cold-start variant: the initial guess is zero (the first pressure solve of a run; PAPER.md:51
 * "impulsive" starts), so no guess crosses the bus -- the staging buffer is zeroed on the device.
 * p_host is written only (the solution).  Otherwise as gmg_solve_host. */
int gmg_solve_host_cold(gmg_ctx* ctx, float* p_host_out, const float* z_host, float tol, int maxiter,
                        int solver, void* stream);

int gmg_stats(const gmg_ctx* ctx, gmg_stats_t* out);
/* Relative residual history of the last solve: out[k] = ||r_k|| / ||z||, k = 0..iterations.
 * Returns the number of entries written (<= cap). */
int gmg_history(const gmg_ctx* ctx, double* out, int cap);
/* Relaxation factors used by V-cycle k+1 (k = 0..iterations-1) of the last GMG-RBGS solve. */
int gmg_omega_history(const gmg_ctx* ctx, double* out, int cap);
int gmg_set_omega(gmg_ctx* ctx, float omega);

/* -- level table and per-operator hooks (parity tests; BASELINE.json tolerances for
 *    "single operator applications") --------------------------------------------------- */
int gmg_num_levels(const gmg_ctx* ctx);
/* n = extents of level lev, c = coarsening factors from lev to lev+1 ((1,1,1) on the last). */
int gmg_level_shape(const gmg_ctx* ctx, int lev, int n[3], int c[3]);
/* Copies the [3][nz][ny][nx] coefficients of level lev to L_out_dev (device). */
int gmg_level_coeffs(gmg_ctx* ctx, int lev, float* L_out_dev, void* stream);
/* r = b - A p on active cells, 0 elsewhere (reading O9). */
int gmg_op_residual(gmg_ctx* ctx, int lev, const float* p_dev, const float* b_dev, float* r_dev,
                    void* stream);
/* nsweeps RBGS sweeps in place; each sweep = colour first_colour then the other
 * (0 = red = (i+j+k) even; reading O3):  p_I += omega (b_I - (A p)_I) / D_I. */
int gmg_op_smooth(gmg_ctx* ctx, int lev, float* p_dev, const float* b_dev, float omega,
                  int nsweeps, int first_colour, void* stream);
/* b_coarse(J) = sum over the children of J of r_fine (reading O6). */
int gmg_op_restrict(gmg_ctx* ctx, int lev, const float* r_fine_dev, float* b_coarse_dev,
                    void* stream);
/* Fused form the V-cycle uses: b_coarse = R (b - A p) without storing the residual. */
int gmg_op_residual_restrict(gmg_ctx* ctx, int lev, const float* p_dev, const float* b_dev,
                             float* b_coarse_dev, void* stream);
/* p_fine(I) += e_coarse(parent(I)) (reading O6). */
int gmg_op_prolong(gmg_ctx* ctx, int lev, const float* e_coarse_dev, float* p_fine_dev,
                   void* stream);
/* One V(nu_pre,nu_post) cycle on level 0 at the given omega (reading O7); symmetric != 0
 * = the variant used as CG preconditioner (reading O11). */
int gmg_op_vcycle(gmg_ctx* ctx, float* p_dev, const float* z_dev, float omega, int symmetric,
                  void* stream);
/* ONE fused red+black sweep src -> dst (out of place) of the TMA-fed kernel that also returns
 * sum r^2, r = b - A src on active cells, and sum b^2 over active cells (the fused_norm path of
 * gmg_solve).  GMG_EINVAL when level lev cannot run that kernel (nx % 128, small levels). */
int gmg_op_sweep_with_norm(gmg_ctx* ctx, int lev, const float* src_dev, float* dst_dev, const float* b_dev,
                           float omega, int first_colour, double* rr_out_host, double* bb_out_host,
                           void* stream);
/* The smoother of GMG_GMG_CGS (reading O12, "PCG can be used as a smoother"): iters
 * Jacobi-PCG iterations on A^lev x = b restarted from x (in place), and one whole cycle of it on
 * level 0 (V(nu_pre, nu_post), nu_coarse iterations on the coarsest level). */
int gmg_op_cg_smooth(gmg_ctx* ctx, int lev, float* x_dev, const float* b_dev, int iters, void* stream);
int gmg_op_vcycle_cgs(gmg_ctx* ctx, float* p_dev, const float* z_dev, void* stream);
/* sqrt(sum r^2) of a level-lev array (deterministic two-stage reduction). */
int gmg_op_norm2(gmg_ctx* ctx, int lev, const float* r_dev, double* out_host, void* stream);

/* -- the steps either side of the solve in a staggered projection step ("predictor +
 *    corrector steps", one Poisson solve each) -----------------------
 * u_dev: [3][nz][ny][nx], u[d*N + idx] = velocity on the LOWER d-face of cell idx (like L).
 * gmg_divergence:  z_I = sum_d [ u_d(I+e_d) - u_d(I) ].  Upper face of the last cell of an axis:
 *   periodic -> u_d(index 0); Neumann -> wall_hi[d] (host array of 3 floats, NULL = zeros); on a
 *   Neumann axis u_d(index 0) is the lower-wall value.
 * gmg_project:  u_d(I) -= L_d(I) * (p_I - p_{I-e_d}) with the coefficients of gmg_set_coeffs
 *   (Neumann wall faces carry 0 and stay untouched), so that div(u_new) = div(u_old) - A p. */
int gmg_divergence(gmg_ctx* ctx, const float* u_dev, const float wall_hi[3], float* z_dev, void* stream);
int gmg_project(gmg_ctx* ctx, float* u_dev, const float* p_dev, void* stream);

/* One whole pressure step in one call (a moving body): gmg_set_coeffs(L_dev)
 * -> z = gmg_divergence(u_dev, wall_hi) into a library-held buffer -> gmg_solve(p_dev: in = guess, e.g.
 * the previous step's pressure, out = solution) -> gmg_project(u_dev, p_dev), enqueued back to back on
 * `stream` with ONE host synchronisation (the solve's status read) instead of four.  Returns the
 * solve's code (gmg_stats describes the solve), or GMG_EINVAL when L holds a negative / non-finite value
 * (u, p are then meaningless).  The projection is stream-ordered behind the return: synchronise
 * `stream` before reading u on the host. */
int gmg_pressure_step(gmg_ctx* ctx, const float* L_dev, float* u_dev, const float wall_hi[3], float* p_dev,
                      float tol, int maxiter, int solver, void* stream);

/* -- one entry point that allocates nothing ---------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops,
 * harnesses that forbid it): out_dev[0] = ||b - A p||_2 over the active cells of an nx*ny*nz grid
 * with the operator and boundary handling at the top of this file (readings O1, O2; the norm of the
 * stopping test, reading O9, PAPER.md:39 S3) -- what gmg_op_residual + gmg_op_norm2 compute on level 0,
 * without a context or a workspace.  L_dev [3][N], p_dev [N], b_dev [N] (float, 4-byte aligned) and
 * out_dev (one double, 8-byte aligned) are the caller's device memory on the CURRENT device.  The
 * reduction scratch (one FP64 partial per 2048 cells and a ticket) is a static device array of
 * 65,792 bytes that every GPU loading the library holds until exit; hence the limit
 * nx*ny*nz <= GMG_NOALLOC_MAX_CELLS (256^3), larger grids are refused with GMG_EINVAL.
 * Nothing is allocated or freed and the host is not synchronised: the result is stream-ordered on
 * `stream`.  The first call on each device looks the array's address up (make that call outside a
 * capture).  All calls share the array: calls that overlap on the GPU (two streams, two host
 * threads) race -- serialise them; calls on one stream are safe back to back.  Deterministic (two
 * stages, fixed order).  err (may be NULL) receives a NUL-terminated message of at most err_cap
 * bytes when the return code is < 0: GMG_EINVAL bad argument / too large, GMG_ECUDA enqueue failed. */
#define GMG_NOALLOC_MAX_CELLS 16777216LL
int gmg_residual_norm2_noalloc(int nx, int ny, int nz, const int bc[3], const float* L_dev,
                               const float* p_dev, const float* b_dev, double* out_dev, void* stream,
                               char* err, size_t err_cap);

/* Names of the kernels a V-cycle launches per level, for profiling notes: writes a
 * NUL-terminated description into buf. */
int gmg_describe_plan(const gmg_ctx* ctx, char* buf, size_t cap);

#ifdef __cplusplus
}
#endif
#endif /* GMG_H_ */

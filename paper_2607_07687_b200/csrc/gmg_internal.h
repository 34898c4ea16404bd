// gmg_internal.h -- host/device shared PODs and kernel-launcher prototypes of the CUDA path.
// Part of the product path; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/gmg.h"

namespace gmgf { struct UniArgs; }

#define GMG_MAX_LEVELS 24
#define GMG_TAIL_MAX_LEVELS 8

// Geometry of one multigrid level (passed to kernels by value).
struct LevelGeom {
    int n[3];     // extents (nx, ny, nz), x fastest
    int bc[3];    // 0 periodic, 1 Neumann
    int c[3];     // coarsening factors to the next level (1 or 2)
    long long N;  // nx*ny*nz
};

// Device pointers of one level.
struct LevelPtrs {
    const float* L;  // [3][N] component-major; level 0: the caller's array
    float* p;        // level >= 1 unknown (level 0: caller's p, set per call)
    float* b;        // level >= 1 right-hand side
    float* q;        // ping-pong partner of p for the fused sweep
};

// Device scalar block: everything the on-device iteration control needs.
struct DevScalars {
    double red[16];    // results of the two-stage reductions (slot per use)
    double r_ref;      // ||z||_2 over active cells
    double rho;        // current residual norm
    double rho_prev;
    double omega;      // relaxation factor (dyadic, exact in float)
    double tol;
    double alpha, beta, rho_cg, rho_cg_new;
    double omega_min, omega_down, omega_up;
    float omega_f;     // omega as the kernels read it
    float omega_one;   // constant 1.0f (GMG-PCG preconditioner runs at omega = 1)
    float omega_hook;  // omega of the gmg_op_* hooks
    int iter;
    int maxiter;
    int status;        // GMG_OK, GMG_NOT_CONVERGED, GMG_EBREAKDOWN
    int done;          // 1: loop finished
    int adaptive;
    int cgs_frozen;    // CG smoother (reading O12): 1 = the remaining iterations leave x untouched
    double cgs_rho0;   // r.s at the restart of the CG smoother
    double cgs_alpha_cap;  // longest step the CG smoother accepts on the current level
    // fused_norm path: the first sweep of cycle k+1 runs before cycle k's omega update is known
    float omega_spec_f;    // omega it ran with: the decay branch of reading O8
    int redo_first;        // 1: the update took the growth branch -- run that sweep again
    // ... and the cycle expected to be the LAST one (rate-based prediction, or maxiter reached) is
    // followed by the plain 20 B/cell norm pass instead, so that no sweep is wasted at the exit
    int predict;           // 1: prediction enabled for this solve
    int expect_last;       // 1: the cycle now running is expected to meet the stopping test
    int run_s1n;           // = !expect_last: the norm-carrying first sweep of the next cycle runs
    int need_first;        // 1: the prediction failed -- the next cycle's first sweep still has to run
};

// CG smoother: stop once |r.s| <= this * |r.s at the restart| (reading O12)
#define GMG_CGS_FREEZE 1e-8

enum {
    RED_RREF = 0,  // sum z^2 over active cells
    RED_RR = 1,    // sum r^2
    RED_DQ = 2,    // d.q
    RED_RS = 3,    // r.s
    RED_HOOK = 4,  // gmg_op_norm2
    RED_CHECK = 5, // coefficient check: count of bad values
    RED_CGS_SUM = 6,  // CG smoother: sum of the restart residual over active cells
    RED_CGS_CNT = 7,  // CG smoother: number of active cells
    RED_HOOK2 = 8     // gmg_op_sweep_with_norm: second sum
};

#ifdef __CUDACC__
// mean of the restart residual over the active cells, as the kernels subtract it
__device__ __forceinline__ float cgs_mean(const DevScalars* sc) {
    const double cnt = sc->red[RED_CGS_CNT];
    return cnt > 0.0 ? (float)(sc->red[RED_CGS_SUM] / cnt) : 0.0f;
}
#endif

// Tail: levels small enough to live in one CTA's shared memory, run as ONE kernel.
struct TailArgs {
    int nlev;                            // number of tail levels (>= 1)
    LevelGeom g[GMG_TAIL_MAX_LEVELS];
    const float* W[GMG_TAIL_MAX_LEVELS]; // [6][N] face weights of each tail level (tail_weights)
    const float* b_in;                   // right-hand side of the first tail level (global)
    const float* p_in;                   // initial guess of the first tail level; nullptr = zero
    float* p_out;                        // solution of the first tail level (global; may alias p_in)
    const float* omega;                  // device scalar
    int nu1, nu2, nuc, sym;
};

// Reduction workspace: FP64 block partials.
struct ReduceBuf {
    double* partials;       // [2][GMG_REDUCE_MAX_BLOCKS] (a kernel reduces at most two sums)
    unsigned int* counter;  // ticket of the "last block finishes the sum" stage, self-resetting
    DevScalars* sc;
    // a single-thread control step that rides on the reduction it follows (stencil.cuh,
    // finish_reduction): the thread that writes the sums runs it, instead of a <<<1, 1>>> launch
    int post;               // POST_NONE, a step of the CG smoother, or alpha / beta of the (GMG-)PCG solver
    double post_arg;        // POST_CGS_BEGIN: the step-length cap of the level
};
enum { POST_NONE = 0, POST_CGS_BEGIN = 1, POST_CGS_ALPHA = 2, POST_CGS_BETA = 3, POST_PCG_ALPHA = 4, POST_PCG_BETA = 5 };
#define GMG_REDUCE_MAX_BLOCKS 16384

// ---- launchers (kernels_generic.cu) --------------------------------------------------------
namespace gmgk {

void half_sweep(const LevelGeom& g, const float* L, float* p, const float* b, const float* omega,
                int colour, cudaStream_t s);
void residual(const LevelGeom& g, const float* L, const float* p, const float* b, float* r,
              cudaStream_t s);
void restrict_sum(const LevelGeom& gf, const float* rf, float* bc, cudaStream_t s);
// b_c = R(b - A p); also zeroes p_c (the coarse initial guess) when p_c != nullptr.
void residual_restrict(const LevelGeom& gf, const float* L, const float* p, const float* b,
                       float* b_c, float* p_c, cudaStream_t s);
void fill(float* x, long long N, float v, cudaStream_t s);
void divergence(const LevelGeom& g, const float* u, const float wall_hi[3], float* z, cudaStream_t s);
void project(const LevelGeom& g, const float* L, const float* p, float* u, cudaStream_t s);
void prolong_add(const LevelGeom& gf, const float* e_c, float* p_f, cudaStream_t s);
void coarsen_coeffs(const LevelGeom& gf, const float* Lf, float* Lc, cudaStream_t s);
void check_coeffs(const LevelGeom& g, const float* L, ReduceBuf rb, cudaStream_t s);
// float4 passes (kernels_setup.cu): bit-identical to the three kernels above
bool coarsen4_supported(const LevelGeom& gf);
void coarsen_coeffs4(const LevelGeom& gf, const float* Lf, float* Lc, bool check, ReduceBuf rb,
                     const gmgf::UniArgs& uni, cudaStream_t s);
void divergence4(const LevelGeom& g, const float* u, const float wall_hi[3], float* z, cudaStream_t s);
void project4(const LevelGeom& g, const float* L, const float* p, float* u, cudaStream_t s);
// uniform bricks (uniform.cuh): cells of a level on the lean path of a kernel with this tiling
// left_list / left_count != nullptr: the tiles that are NOT lean are appended to the list
void uniform_cells(const LevelGeom& g, const unsigned char* brick, int TXc, int TYc, int yhi, int zchunk, int rule,
                   unsigned long long* out, int* left_list, unsigned int* left_count, cudaStream_t s);
void tail_vcycle(const TailArgs& a, size_t smem_bytes, cudaStream_t s);
// W[f*N + c] = weight of face f (x-lo, x-hi, y-lo, y-hi, z-lo, z-hi) of cell c, wall faces zeroed
void tail_weights(const LevelGeom& g, const float* L, float* W, cudaStream_t s);
size_t tail_smem_bytes(const TailArgs& a);
// Cluster tail (kernels_ctail.cu): layout of a level in the shared memory of the 8 CTAs.
struct CLevelPlan {
    int dist;  // 1: cut into 8 z-slabs, one per CTA; 0: whole level in CTA 0
    int per;   // cells held per CTA
    int off;   // float offset of this level's block in every CTA: W[6][per] p[per] b[per] r[per]
};
// Returns the dynamic shared memory per CTA, or 0 when these levels cannot run on the cluster.
size_t ctail_plan(const LevelGeom* g, int nlev, CLevelPlan* lv);
int ctail_configure(size_t max_bytes);
bool ctail_launchable(size_t smem_bytes);
void ctail_vcycle(const TailArgs& t, const CLevelPlan* lv, size_t smem_bytes, cudaStream_t s);
int tail_configure(size_t max_bytes);  // sets the dynamic-smem attribute; returns cudaError

// reductions: result lands in rb.sc->red[slot]
void residual_norm2(const LevelGeom& g, const float* L, const float* p, const float* b,
                    ReduceBuf rb, int slot, cudaStream_t s);
void active_norm2(const LevelGeom& g, const float* L, const float* z, ReduceBuf rb, int slot,
                  cudaStream_t s);
void norm2(long long N, const float* r, ReduceBuf rb, int slot, cudaStream_t s);
void dot(long long N, const float* a, const float* b, ReduceBuf rb, int slot, cudaStream_t s);

// PCG pieces
// (uni: uniform bricks of the level, uniform.cuh -- the float4 kernels then skip the coefficient loads
// of the groups whose faces all carry the level's constants; nullptr = load everything)
void matvec_dot(const LevelGeom& g, const float* L, const float* d, float* q, ReduceBuf rb,
                int slot, cudaStream_t s, const gmgf::UniArgs* uni = nullptr);   // q = A d ; red[slot] = d.q
void pcg_update_pr(const LevelGeom& g, const float* L, float* p, float* r, const float* d,
                   const float* q, float* s_out, int jacobi, ReduceBuf rb, cudaStream_t st);
// p += alpha d; r -= alpha q; red[RR] = r.r; if jacobi: s = r/D, red[RS] = r.s
void pcg_update_d(long long N, float* d, const float* s_in, const DevScalars* sc, int first,
                  cudaStream_t st);                      // d = s + beta d   (first: d = s)
void jacobi_apply(const LevelGeom& g, const float* L, const float* r, float* s_out, ReduceBuf rb,
                  int slot, cudaStream_t st, const gmgf::UniArgs* uni = nullptr);   // s = r/D ; red[slot] = r.s

// on-device iteration control (single-thread kernels, kernels_ctl.cu).  `cond` is the WHILE
// node's conditional handle; use_cond = 0 outside a graph.
void ctl_init(DevScalars* sc, double tol, int maxiter, int adaptive, double omega_min,
              double omega_down, double omega_up, int predict, cudaStream_t s);
void ctl_begin(DevScalars* sc, double* hist, double* omegas, cudaGraphConditionalHandle cond,
               int use_cond, cudaStream_t s);
void ctl_rbgs_cycle_end(DevScalars* sc, double* hist, double* omegas,
                        cudaGraphConditionalHandle cond, int use_cond, cudaStream_t s);
// (alpha and beta of the PCG solvers ride on the mat-vec and on the r.s reduction: ReduceBuf::post)
void ctl_pcg_check(DevScalars* sc, double* hist, cudaGraphConditionalHandle cond, int use_cond,
                   cudaStream_t s);
void ctl_set_hook_omega(DevScalars* sc, float omega, cudaStream_t s);

// CG smoother of the paper's GMG-PCG (kernels_cgs.cu, reading O12)
// r = b - A x (0 on inactive cells); red[CGS_SUM] = sum r, red[CGS_CNT] = number of active cells
void cgs_residual_sum(const LevelGeom& g, const float* L, const float* x, const float* b, float* r,
                      ReduceBuf rb, cudaStream_t s, const gmgf::UniArgs* uni = nullptr);
// r -= mean over active cells; d = r/D; red[RS] = r.d
void cgs_start(const LevelGeom& g, const float* L, float* r, float* d, ReduceBuf rb, cudaStream_t s,
               const gmgf::UniArgs* uni = nullptr);
// (the smoother's control steps -- begin, alpha, beta -- ride on cgs_start, the mat-vec and the
// Jacobi kernel: ReduceBuf::post)
// m iterations restarted from x (in place) on a level of at most 4096 cells with nx % 4 == 0, as one
// single-CTA kernel; false = level not eligible (nothing enqueued)
bool cgs_small(const LevelGeom& g, const float* L, float* x, const float* b, int m, double alpha_cap,
               cudaStream_t s);
void ctl_set_omega(DevScalars* sc, double omega, cudaStream_t s);

}  // namespace gmgk

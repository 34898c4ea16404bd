// gmg_api.cu -- C-ABI boundary (include/gmg.h) and the host-side driver of the solve: level
// table (reading O4), workspace carving, V-cycle enqueue (reading O7), the solve
// loops (O9-O11) as CUDA graphs with a device-side WHILE node, statistics.
// Product path: no CPU fallback, nothing from oracle/.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <vector>

#include "gmg_internal.h"
#include "uniform.cuh"

namespace gmgf {  // fast-path launchers (kernels_fused.cu)
bool sweep_supported(const LevelGeom& g);
// nsweeps (even count handled by caller) fused red+black sweeps src -> dst (out of place).
// first_colour 0: red then black.  If e_c != nullptr the prolonged coarse correction is added
// to src on the fly (fused prolongation + correction).
// `uni`: the level's uniform bricks (uniform.cuh), brick == nullptr where the lean path is off
void rb_sweep(const LevelGeom& g, const float* L, const float* src, float* dst, const float* b,
              const float* omega, int first_colour, const float* e_c, int allow_tma, const UniArgs& uni,
              cudaStream_t s);
bool resrestrict_supported(const LevelGeom& g);
void residual_restrict(const LevelGeom& g, const float* L, const float* p, const float* b,
                       float* b_c, float* p_c, int allow_tma, const UniArgs& uni, cudaStream_t s);
void residual_norm2(const LevelGeom& g, const float* L, const float* p, const float* b, ReduceBuf rb,
                    int slot, int allow_tma, const UniArgs& uni, cudaStream_t s);
bool residual_and_ref_norm2_bulk(const LevelGeom& g, const float* L, const float* p, const float* b,
                                 ReduceBuf rb, int slot_rr, int slot_ref, const UniArgs& uni, cudaStream_t s);
void prolong_add4(const LevelGeom& g, const float* e_c, float* p_f, cudaStream_t s);
bool matvec_dot_bulk(const LevelGeom& g, const float* L, const float* d, float* q, ReduceBuf rb, int slot,
                     const UniArgs& uni, cudaStream_t s);
bool bulk_sweep_tiling(const LevelGeom& g, int* tile_y, int* zchunk);
bool res_bulk_tiling(const LevelGeom& g, int* tile_y, int* zchunk);
bool tma_shape_ok(const LevelGeom& g);
bool sweep_fuses_prolong(const LevelGeom& g, const UniArgs& uni);
bool bulk_sweep_edge(const LevelGeom& g, bool norm);
// one TMA-fed sweep src -> dst that also leaves sum r^2 (r = b - A src) and sum b^2 over the active
// cells in red[slot_rr] / red[slot_ref]; false = the level cannot run it (nothing launched)
bool rb_sweep_with_norm(const LevelGeom& g, const float* L, const float* src, float* dst, const float* b,
                        const float* omega, int first_colour, ReduceBuf rb, int slot_rr, int slot_ref,
                        const int* run_flag, const UniArgs& uni, cudaStream_t s);
bool residual_norm2_bulk_if(const LevelGeom& g, const float* L, const float* p, const float* b, ReduceBuf rb,
                            int slot, const int* run_flag, const UniArgs& uni, cudaStream_t s);
bool residual_norm_bulk_supported(const LevelGeom& g);
bool sweep_norm_supported(const LevelGeom& g);
// the same sweep as a no-op unless *run_flag != 0
bool rb_sweep_if(const LevelGeom& g, const float* L, const float* src, float* dst, const float* b,
                 const float* omega, int first_colour, const int* run_flag, const UniArgs& uni, cudaStream_t s);
int configure();
}  // namespace gmgf

struct GraphSlot {
    cudaGraphExec_t exec = nullptr;
    cudaGraph_t graph = nullptr;
    float* p = nullptr;
    const float* z = nullptr;
    int solver = -1;
    float tol = 0.0f;
    int maxiter = -1;
    double* hist = nullptr;
    long long n_pre = 0, n_body = 0, n_post = 0;  // kernel launches per section
    int left_n[GMG_MAX_LEVELS];   // lengths of the remaining-tile lists the launch grids were sized with
    int fold[GMG_MAX_LEVELS];     // ... and whether the prolongation rode on the first post-sweep
};

struct gmg_ctx {
    int n0[3], bc[3];
    gmg_params_t prm;
    int nlev;
    LevelGeom g[GMG_MAX_LEVELS];
    LevelPtrs lv[GMG_MAX_LEVELS];
    int tail_start;       // first level run inside the single-CTA tail kernel (nlev = none)
    size_t tail_smem;
    int ctail_start;      // first level run inside the cluster tail kernel (nlev = none); < tail_start
    size_t ctail_smem;
    gmgk::CLevelPlan ctail_lv[GMG_TAIL_MAX_LEVELS];
    bool cluster_ok;      // the device can hold a cluster of 8 CTAs with 200 KB each
    bool fast_sweep[GMG_MAX_LEVELS];
    bool fast_rr[GMG_MAX_LEVELS];
    int tma_ok[GMG_MAX_LEVELS];  // level large enough for the TMA-fed kernels
    bool fused_norm_on;   // GMG-RBGS: the stopping-test norm rides on the first pre-sweep (prm.fused_norm)
    // uniform bricks (uniform.cuh): levels that run the TMA-fed kernels
    gmgf::UniArgs uni[GMG_MAX_LEVELS];     // brick == nullptr: level not marked
    size_t ubrick_n[GMG_MAX_LEVELS];       // bricks of the level
    unsigned char* ubrick_dev;             // all levels' flags, one allocation; behind them
                                           // [2][GMG_MAX_LEVELS] counts of lean-path cells (sweep, residual)
                                           // and [GMG_MAX_LEVELS] lengths of the remaining-tile lists, then the lists
    unsigned long long* ucount_host;       // pinned mirror of the counts and lengths
    size_t ubrick_total;
    double uni_frac_sweep[GMG_MAX_LEVELS]; // cells whose sweep / residual CTA takes the lean path
    double uni_frac_res[GMG_MAX_LEVELS];
    bool uni_stats_pending;                // flags copied down, fractions not yet recomputed
    // workspace
    void* ws;
    size_t ws_bytes;
    bool ws_set, coeffs_set;
    float *pcg_r, *pcg_d, *pcg_q, *pcg_s, *stage_p, *stage_z;
    float* uni_scratch;   // level-0-sized: corrected iterate over the non-lean tiles (uniform.cuh, PRO)
    float* tail_W[GMG_MAX_LEVELS];  // [6][N] face weights of the tail levels
    // small library-owned device state
    DevScalars* sc;
    double* partials;
    unsigned int* counter;
    double *hist, *omegas;
    int hist_cap;
    double* hist_pin;     // pinned mirror: [0, cap) history, [cap, 2 cap) omegas -- read with the status block
    DevScalars* sc_host;  // pinned mirror
    std::vector<double> hist_host, omegas_host;
    gmg_stats_t stats;
    cudaEvent_t ev0, ev1;
    cudaStream_t cap_a, cap_b;  // internal streams used only for graph capture
    // forked beside the enqueuing stream (uniform.cuh: lean + general kernels side by side).  Two
    // sets: while a solve graph is built two captures are open at once (the outer graph and the WHILE
    // body), and a stream can belong to one capture only.
    cudaStream_t side[2];
    cudaEvent_t ev_fork[2], ev_join[2];
    GraphSlot slots[4];
    long long n_launch;   // launch counter of the section being enqueued
    bool enqueue_fail;    // a launcher the plan counted on refused (tensor-map encode failed)
    bool sc_fresh;        // sc_host holds the status block of the call in progress
    char err[512];
};

#define SET_ERR(ctx, ...) snprintf((ctx)->err, sizeof((ctx)->err), __VA_ARGS__)
#define CUDA_TRY(ctx, call)                                                              \
    do {                                                                                 \
        cudaError_t e_ = (call);                                                         \
        if (e_ != cudaSuccess) {                                                         \
            SET_ERR(ctx, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, \
                    __LINE__);                                                           \
            return GMG_ECUDA;                                                            \
        }                                                                                \
    } while (0)

// The TMA-fed CG mat-vec pays from 4 Mi cells on; below that the float4 kernel is faster (128^3
// Jacobi-PCG: 5.2 vs 5.7 ms per solve), whatever tma_min_cells says for the sweeps -- unless it is
// 0 ("whenever the shape allows": the tests force the TMA path on small grids that way).
static const long long kBulkMatvecMinCells = 4LL << 20;
static const long long kLeanVectorMinCells = 8LL << 20;   // (tma_min_cells = 0 forces both, for the tests)

static inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }
// behind the brick flags: [2][levels] u64 lean-cell counts, [levels] u32 remaining-tile list lengths
static const size_t kUniCountBytes = 256 * ((sizeof(unsigned long long) * 2 * GMG_MAX_LEVELS + sizeof(unsigned int) * GMG_MAX_LEVELS + 255) / 256);
static inline const gmgf::UniArgs& U(const gmg_ctx* c, int l) { return c->uni[l]; }
// The float4 / TMA paths read caller arrays 16 bytes at a time (gmg.h "Alignment").
static inline bool al16(const void* p) { return (((uintptr_t)p) & 15) == 0; }
#define MUST_LAUNCH(c, call) do { if (!(call)) (c)->enqueue_fail = true; } while (0)
static inline ReduceBuf rbuf(gmg_ctx* c) { return ReduceBuf{c->partials, c->counter, c->sc, POST_NONE, 0.0}; }

// ---- level table: reading O4 ("downsamples every dimension independently") ------
static void build_levels(gmg_ctx* c) {
    LevelGeom g0;
    for (int d = 0; d < 3; ++d) {
        g0.n[d] = c->n0[d];
        g0.bc[d] = c->bc[d];
    }
    c->nlev = 0;
    LevelGeom cur = g0;
    while (true) {
        cur.N = (long long)cur.n[0] * cur.n[1] * cur.n[2];
        int any = 0, all = 1;
        for (int d = 0; d < 3; ++d) {
            const int h = cur.n[d] / 2;
            const int ok = (cur.n[d] % 2 == 0) && (h >= c->prm.n_min) &&
                           (cur.bc[d] == GMG_BC_NEUMANN || h % 2 == 0);
            cur.c[d] = ok ? 2 : 1;
            any |= ok;
            if (cur.n[d] > 1) all &= ok;  // an extent-1 direction (2-D grid) has nothing to coarsen
        }
        if (c->prm.coarsen_mode == GMG_COARSEN_ISO && !all) any = 0;
        if (!any || c->nlev + 1 >= GMG_MAX_LEVELS) cur.c[0] = cur.c[1] = cur.c[2] = 1;
        c->g[c->nlev++] = cur;
        if (cur.c[0] * cur.c[1] * cur.c[2] == 1) break;
        for (int d = 0; d < 3; ++d) cur.n[d] /= cur.c[d];
    }
    // tail: the longest suffix of levels that fits one CTA's shared memory
    const size_t cap = 200 * 1024;
    c->tail_start = c->nlev;
    size_t cells = 0;
    for (int l = c->nlev - 1; l >= 0; --l) {
        cells += (size_t)c->g[l].N;
        // 8 floats per cell (six face weights, p, b); at most 6 cells of a level per thread
        if (cells * 8 * sizeof(float) > cap || c->g[l].N > 6144 || c->nlev - l > GMG_TAIL_MAX_LEVELS) break;
        c->tail_start = l;
        c->tail_smem = cells * 8 * sizeof(float);
    }
    // cluster tail: the longest suffix (beyond the single-CTA tail) a cluster of 8 CTAs can hold
    c->ctail_start = c->nlev;
    c->ctail_smem = 0;
    if (c->prm.fast_path && c->prm.cluster_tail && c->cluster_ok) {
        const int lo = c->nlev > GMG_TAIL_MAX_LEVELS ? c->nlev - GMG_TAIL_MAX_LEVELS : 0;
        for (int l = lo; l < c->tail_start; ++l) {
            gmgk::CLevelPlan lv[GMG_TAIL_MAX_LEVELS];
            const size_t bytes = gmgk::ctail_plan(c->g + l, c->nlev - l, lv);
            if (bytes == 0) continue;
            c->ctail_start = l;
            c->ctail_smem = bytes;
            memcpy(c->ctail_lv, lv, sizeof(lv));
            break;
        }
    }
    for (int l = 0; l < c->nlev; ++l) {
        c->fast_sweep[l] = c->prm.fast_path && gmgf::sweep_supported(c->g[l]);
        c->fast_rr[l] = c->prm.fast_path && l + 1 < c->nlev && gmgf::resrestrict_supported(c->g[l]);
        c->tma_ok[l] = c->prm.tma_min_cells >= 0 && c->g[l].N >= (long long)c->prm.tma_min_cells;
    }
    // uniform.cuh: the constant a level's coefficients take where every fine coefficient below is 1
    // (reading O5 applied to ones): (prod_{e != d} C_e) / C_d with C the cumulative coarsening factors
    {
        double C[3] = {1.0, 1.0, 1.0};
        for (int l = 0; l < c->nlev; ++l) {
            c->uni[l].ux = (float)(C[1] * C[2] / C[0]);
            c->uni[l].uy = (float)(C[0] * C[2] / C[1]);
            c->uni[l].uz = (float)(C[0] * C[1] / C[2]);
            c->uni[l].brick = nullptr;
            c->uni[l].side_stream = c->uni[l].ev_fork = c->uni[l].ev_join = nullptr;
            c->uni[l].left_list = nullptr; c->uni[l].left_count = nullptr; c->uni[l].left_n = -1;
            c->uni[l].scratch = nullptr; c->uni[l].fold = 0;
            c->ubrick_n[l] = 0;
            c->uni_frac_sweep[l] = c->uni_frac_res[l] = 0.0;
            for (int d = 0; d < 3; ++d) C[d] *= c->g[l].c[d];
        }
    }
    const int first_tail = c->ctail_start < c->tail_start ? c->ctail_start : c->tail_start;
    c->fused_norm_on = c->prm.fused_norm && c->prm.fast_path && c->nlev > 1 && first_tail > 0 &&
                       c->fast_sweep[0] && c->tma_ok[0] && c->prm.nu_pre >= 2;
}

static size_t carve(gmg_ctx* c, char* base) {
    size_t off = 0;
    auto take = [&](size_t nfloat) -> float* {
        float* ptr = base ? (float*)(base + off) : nullptr;
        off += align_up(nfloat * sizeof(float));
        return ptr;
    };
    for (int l = 0; l < c->nlev; ++l) {
        const size_t N = (size_t)c->g[l].N;
        if (l > 0) {
            float* L = take(3 * N);
            float* p = take(N);
            float* b = take(N);
            if (base) {
                c->lv[l].L = L;
                c->lv[l].p = p;
                c->lv[l].b = b;
            }
        }
        float* q = take(N);
        if (base) c->lv[l].q = q;
        if (l >= c->tail_start || l >= c->ctail_start) {
            float* w = take(6 * N);
            if (base) c->tail_W[l] = w;
        }
    }
    const size_t N0 = (size_t)c->g[0].N;
    float* v[6];
    for (int i = 0; i < 6; ++i) v[i] = take(N0);
    if (base) {
        c->pcg_r = v[0]; c->pcg_d = v[1]; c->pcg_q = v[2]; c->pcg_s = v[3];
        c->stage_p = v[4]; c->stage_z = v[5];
    }
    // the sweep that folds the prolongation in (gmgf::sweep_fuses_prolong) leaves p + P e_c of the
    // non-lean tiles here: as large as the largest level that can take that path (host-side test of
    // the shape the TMA kernels accept, so that gmg_plan gives the same size without a GPU)
    size_t nscr = 0;
    if (c->prm.uniform_tiles && c->prm.fast_path)
        for (int l = 0; l + 1 < c->nlev && l < c->tail_start && l < c->ctail_start; ++l) {
            const LevelGeom& g = c->g[l];
            const bool shape = g.n[0] >= 128 && g.n[0] % 128 == 0 && g.n[1] >= 4 && g.n[2] >= 8;
            if (shape && c->tma_ok[l] && g.c[0] == 2 && g.c[1] == 2 && g.c[2] == 2 && (size_t)g.N > nscr)
                nscr = (size_t)g.N;
        }
    float* scr = nscr ? take(nscr) : nullptr;
    if (base) c->uni_scratch = scr;
    return off;
}

// Brick flags of the levels that run the TMA-fed kernels: one small library-owned allocation.
static void free_uniform(gmg_ctx* c) {
    if (c->ubrick_dev) cudaFree(c->ubrick_dev);
    if (c->ucount_host) cudaFreeHost(c->ucount_host);
    c->ubrick_dev = nullptr;
    c->ucount_host = nullptr;
    c->ubrick_total = 0;
    for (int l = 0; l < GMG_MAX_LEVELS; ++l) {
        c->uni[l].brick = nullptr; c->ubrick_n[l] = 0;
        c->uni[l].left_list = nullptr; c->uni[l].left_count = nullptr; c->uni[l].left_n = -1;
        c->uni[l].scratch = nullptr; c->uni[l].fold = 0;
    }
}
static cudaError_t alloc_uniform(gmg_ctx* c) {
    free_uniform(c);
    if (!c->prm.uniform_tiles || !c->prm.fast_path) return cudaSuccess;
    const int first_tail = c->ctail_start < c->tail_start ? c->ctail_start : c->tail_start;
    size_t off[GMG_MAX_LEVELS], total = 0;
    for (int l = 0; l < c->nlev && l < first_tail; ++l) {
        off[l] = total;
        if (!(c->fast_sweep[l] && c->tma_ok[l] && gmgf::tma_shape_ok(c->g[l]))) continue;
        c->ubrick_n[l] = (size_t)gmgf::ub_count(c->g[l].n[0], gmgf::kUBX) * gmgf::ub_count(c->g[l].n[1], gmgf::kUBY) *
                         gmgf::ub_count(c->g[l].n[2], gmgf::kUBZ);
        total += align_up(c->ubrick_n[l], 256);
    }
    if (total == 0) return cudaSuccess;
    const size_t cbytes = kUniCountBytes;
    size_t loff[GMG_MAX_LEVELS], lbytes[GMG_MAX_LEVELS], ltotal = 0;      // remaining-tile lists of the sweep
    for (int l = 0; l < c->nlev; ++l) {
        loff[l] = ltotal;
        lbytes[l] = 0;
        int ty = 0, zc = 0;
        if (c->ubrick_n[l] && gmgf::bulk_sweep_tiling(c->g[l], &ty, &zc)) {
            const size_t tiles = (size_t)(c->g[l].n[0] / 128) * ((c->g[l].n[1] + ty - 1) / ty) * ((c->g[l].n[2] + zc - 1) / zc);
            lbytes[l] = align_up(tiles * sizeof(int), 256);
            ltotal += lbytes[l];
        }
    }
    cudaError_t e = cudaMalloc(&c->ubrick_dev, total + cbytes + ltotal);
    if (e == cudaSuccess) e = cudaMallocHost(&c->ucount_host, cbytes);
    if (e != cudaSuccess) { free_uniform(c); return e; }
    c->ubrick_total = total;
    unsigned int* lcnt = reinterpret_cast<unsigned int*>(c->ubrick_dev + total + sizeof(unsigned long long) * 2 * GMG_MAX_LEVELS);
    for (int l = 0; l < c->nlev; ++l)
        if (c->ubrick_n[l]) {
            c->uni[l].brick = c->ubrick_dev + off[l];
            c->uni[l].side_stream = c->side[0]; c->uni[l].ev_fork = c->ev_fork[0]; c->uni[l].ev_join = c->ev_join[0];
            c->uni[l].scratch = c->uni_scratch;
            if (lbytes[l]) {
                c->uni[l].left_list = reinterpret_cast<const int*>(c->ubrick_dev + total + cbytes + loff[l]);
                c->uni[l].left_count = lcnt + l;
                c->uni[l].left_n = -1;
            }
        }
    return cudaSuccess;
}

// Which fork set the launchers use from now on: 0 = plain launches and the outer graph, 1 = the
// WHILE body (captured while the outer capture is still open).
static void use_side(gmg_ctx* c, int which) {
    for (int l = 0; l < c->nlev; ++l)
        if (c->uni[l].brick) {
            c->uni[l].side_stream = c->side[which];
            c->uni[l].ev_fork = c->ev_fork[which];
            c->uni[l].ev_join = c->ev_join[which];
        }
}

static void drop_graphs(gmg_ctx* c) {
    for (auto& s : c->slots) {
        if (s.exec) cudaGraphExecDestroy(s.exec);
        if (s.graph) cudaGraphDestroy(s.graph);
        s = GraphSlot();
    }
}

extern "C" void gmg_default_params(gmg_params_t* p) {
    p->nu_pre = 2; p->nu_post = 2; p->nu_coarse = 32;
    p->omega0 = 1.0f; p->omega_min = 0.5f; p->omega_down = 0.125f; p->omega_up = 0.03125f;
    p->adaptive = 1; p->coarsen_mode = GMG_COARSEN_ANISO; p->n_min = 4;
    p->fast_path = 1; p->use_graph = 1; p->tma_min_cells = 1 << 20; p->cluster_tail = 1;
    p->fused_norm = 1;
    p->uniform_tiles = 1;
    p->small_cg = 1;
}

extern "C" int gmg_create(gmg_ctx** out, int nx, int ny, int nz, const int bc[3]) {
    if (!out || !bc) return GMG_EINVAL;
    *out = nullptr;
    const int n[3] = {nx, ny, nz};
    for (int d = 0; d < 3; ++d) {
        if (n[d] < 1) return GMG_EINVAL;
        if (bc[d] != GMG_BC_PERIODIC && bc[d] != GMG_BC_NEUMANN) return GMG_EINVAL;
        if (n[d] == 1 && bc[d] != GMG_BC_NEUMANN) return GMG_EINVAL;  // 2-D mode: walls either side
        if (bc[d] == GMG_BC_PERIODIC && (n[d] & 1)) return GMG_EINVAL;  // reading O3
    }
    if ((long long)nx * ny * nz > (1LL << 31) - 1) return GMG_EINVAL;
    gmg_ctx* c = new gmg_ctx();
    memset(c->err, 0, sizeof(c->err));
    for (int d = 0; d < 3; ++d) { c->n0[d] = n[d]; c->bc[d] = bc[d]; }
    gmg_default_params(&c->prm);
    c->ws = nullptr; c->ws_bytes = 0; c->ws_set = false; c->coeffs_set = false;
    c->uni_scratch = nullptr;
    c->hist = c->omegas = nullptr; c->hist_cap = 0; c->hist_pin = nullptr;
    memset(&c->stats, 0, sizeof(c->stats));
    memset(c->lv, 0, sizeof(c->lv));
    c->sc = nullptr; c->partials = nullptr; c->counter = nullptr; c->sc_host = nullptr;
    c->ev0 = c->ev1 = nullptr;
    c->cap_a = c->cap_b = nullptr;
    for (int i = 0; i < 2; ++i) { c->side[i] = nullptr; c->ev_fork[i] = c->ev_join[i] = nullptr; }
    c->cluster_ok = false;
    c->enqueue_fail = false; c->sc_fresh = false;
    c->ubrick_dev = nullptr; c->ucount_host = nullptr; c->ubrick_total = 0; c->uni_stats_pending = false;
    if (gmgk::ctail_configure(200 * 1024) == (int)cudaSuccess) c->cluster_ok = gmgk::ctail_launchable(200 * 1024);
    cudaGetLastError();
    build_levels(c);
    cudaError_t e = cudaMalloc(&c->sc, sizeof(DevScalars));
    if (e == cudaSuccess) e = cudaMalloc(&c->partials, 2 * GMG_REDUCE_MAX_BLOCKS * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&c->counter, sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaMemset(c->sc, 0, sizeof(DevScalars));
    if (e == cudaSuccess) e = cudaMemset(c->counter, 0, sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaMallocHost(&c->sc_host, sizeof(DevScalars));
    if (e == cudaSuccess) e = cudaEventCreate(&c->ev0);
    if (e == cudaSuccess) e = cudaEventCreate(&c->ev1);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->cap_a, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->cap_b, cudaStreamNonBlocking);
    for (int i = 0; i < 2; ++i) {
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->side[i], cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_fork[i], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_join[i], cudaEventDisableTiming);
    }
    if (e == cudaSuccess) e = (cudaError_t)gmgk::tail_configure(200 * 1024);
    if (e == cudaSuccess) e = (cudaError_t)gmgf::configure();
    if (e == cudaSuccess) {
        gmgk::ctl_set_omega(c->sc, (double)c->prm.omega0, 0);
        e = cudaDeviceSynchronize();
    }
    if (e != cudaSuccess) {
        gmg_destroy(c);
        return GMG_ECUDA;
    }
    *out = c;
    return GMG_OK;
}

extern "C" void gmg_destroy(gmg_ctx* c) {
    if (!c) return;
    drop_graphs(c);
    free_uniform(c);
    if (c->sc) cudaFree(c->sc);
    if (c->partials) cudaFree(c->partials);
    if (c->counter) cudaFree(c->counter);
    if (c->hist) cudaFree(c->hist);
    if (c->omegas) cudaFree(c->omegas);
    if (c->hist_pin) cudaFreeHost(c->hist_pin);
    if (c->sc_host) cudaFreeHost(c->sc_host);
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    if (c->cap_a) cudaStreamDestroy(c->cap_a);
    if (c->cap_b) cudaStreamDestroy(c->cap_b);
    for (int i = 0; i < 2; ++i) {
        if (c->side[i]) cudaStreamDestroy(c->side[i]);
        if (c->ev_fork[i]) cudaEventDestroy(c->ev_fork[i]);
        if (c->ev_join[i]) cudaEventDestroy(c->ev_join[i]);
    }
    delete c;
}

extern "C" const char* gmg_last_error(const gmg_ctx* c) { return c ? c->err : "null context"; }

extern "C" int gmg_set_params(gmg_ctx* c, const gmg_params_t* p) {
    if (!c || !p) return GMG_EINVAL;
    if (p->nu_pre < 0 || p->nu_post < 0 || p->nu_coarse < 0 || (p->nu_coarse & 1) || p->n_min < 1 ||
        !(p->omega0 > 0.0f) || !(p->omega_min > 0.0f) ||
        (p->coarsen_mode != GMG_COARSEN_ANISO && p->coarsen_mode != GMG_COARSEN_ISO)) {
        SET_ERR(c, "gmg_set_params: invalid parameter");
        return GMG_EINVAL;
    }
    c->prm = *p;
    drop_graphs(c);
    free_uniform(c);
    build_levels(c);
    c->ws_set = false;
    c->coeffs_set = false;
    gmgk::ctl_set_omega(c->sc, (double)p->omega0, 0);
    CUDA_TRY(c, cudaDeviceSynchronize());
    return GMG_OK;
}

extern "C" int gmg_get_params(const gmg_ctx* c, gmg_params_t* out) {
    if (!c || !out) return GMG_EINVAL;
    *out = c->prm;
    return GMG_OK;
}

extern "C" size_t gmg_workspace_bytes(const gmg_ctx* c) {
    if (!c) return 0;
    return carve(const_cast<gmg_ctx*>(c), nullptr);
}

extern "C" int gmg_set_workspace(gmg_ctx* c, void* ws, size_t bytes) {
    if (!c || !ws) return GMG_EINVAL;
    if (((uintptr_t)ws) & 255) { SET_ERR(c, "workspace must be 256-byte aligned"); return GMG_EINVAL; }
    const size_t need = carve(c, nullptr);
    if (bytes < need) { SET_ERR(c, "workspace too small: %zu < %zu", bytes, need); return GMG_ENOMEM; }
    drop_graphs(c);
    carve(c, (char*)ws);
    c->ws = ws; c->ws_bytes = bytes; c->ws_set = true; c->coeffs_set = false;
    CUDA_TRY(c, alloc_uniform(c));
    return GMG_OK;
}

// Host-only planning: no CUDA call, usable (and tested) on a machine without a GPU.
extern "C" int gmg_plan(int nx, int ny, int nz, const int bc[3], const gmg_params_t* params, gmg_plan_t* out) {
    if (!bc || !out) return GMG_EINVAL;
    const int n[3] = {nx, ny, nz};
    for (int d = 0; d < 3; ++d) {
        if (n[d] < 1) return GMG_EINVAL;
        if (bc[d] != GMG_BC_PERIODIC && bc[d] != GMG_BC_NEUMANN) return GMG_EINVAL;
        if (n[d] == 1 && bc[d] != GMG_BC_NEUMANN) return GMG_EINVAL;  // 2-D mode: walls either side
        if (bc[d] == GMG_BC_PERIODIC && (n[d] & 1)) return GMG_EINVAL;
    }
    if ((long long)nx * ny * nz > (1LL << 31) - 1) return GMG_EINVAL;
    gmg_ctx tmp;
    tmp.cluster_ok = true;   // host-side plan: assume a device that can hold the cluster
    tmp.uni_scratch = nullptr;
    for (int d = 0; d < 3; ++d) { tmp.n0[d] = n[d]; tmp.bc[d] = bc[d]; }
    if (params) tmp.prm = *params; else gmg_default_params(&tmp.prm);
    if (tmp.prm.n_min < 1) return GMG_EINVAL;
    memset(tmp.lv, 0, sizeof(tmp.lv));
    build_levels(&tmp);
    memset(out, 0, sizeof(*out));
    out->levels = tmp.nlev;
    for (int l = 0; l < tmp.nlev; ++l)
        for (int d = 0; d < 3; ++d) { out->n[l][d] = tmp.g[l].n[d]; out->c[l][d] = tmp.g[l].c[d]; }
    out->tail_start = tmp.tail_start;
    out->workspace_bytes = carve(&tmp, nullptr);
    return GMG_OK;
}

extern "C" int gmg_num_levels(const gmg_ctx* c) { return c ? c->nlev : GMG_EINVAL; }

extern "C" int gmg_level_shape(const gmg_ctx* c, int lev, int n[3], int cf[3]) {
    if (!c || lev < 0 || lev >= c->nlev) return GMG_EINVAL;
    for (int d = 0; d < 3; ++d) {
        if (n) n[d] = c->g[lev].n[d];
        if (cf) cf[d] = c->g[lev].c[d];
    }
    return GMG_OK;
}

// ---- coefficients: reading O5 ("anisotropic coarsening operators") ---------------
// Enqueues the whole coefficient pass (validation count lands in red[RED_CHECK]); no host sync.
static void set_coeffs_enqueue(gmg_ctx* c, const float* L_dev, cudaStream_t s) {
    // the captured solve graphs hold pointers only: a moving body that rewrites the SAME array
    // every step keeps them; a new array drops them
    if (c->lv[0].L != L_dev) drop_graphs(c);
    c->lv[0].L = L_dev;
    // finest level: validation rides on the coarsening pass when the float4 kernel takes it
    const bool fused_check = c->prm.fast_path && c->nlev > 1 && gmgk::coarsen4_supported(c->g[0]);
    if (!fused_check) gmgk::check_coeffs(c->g[0], L_dev, rbuf(c), s);
    for (int l = 0; l + 1 < c->nlev; ++l) {
        float* Lc = const_cast<float*>(c->lv[l + 1].L);
        if (c->prm.fast_path && gmgk::coarsen4_supported(c->g[l])) {
            // the pass that reads every coefficient of level l also marks its uniform bricks
            if (c->uni[l].brick) cudaMemsetAsync(const_cast<unsigned char*>(c->uni[l].brick), 1, c->ubrick_n[l], s);
            gmgk::coarsen_coeffs4(c->g[l], c->lv[l].L, Lc, l == 0, rbuf(c), c->uni[l], s);
        } else {
            if (c->uni[l].brick) cudaMemsetAsync(const_cast<unsigned char*>(c->uni[l].brick), 0, c->ubrick_n[l], s);
            gmgk::coarsen_coeffs(c->g[l], c->lv[l].L, Lc, s);
        }
    }
    for (int l = (c->ctail_start < c->tail_start ? c->ctail_start : c->tail_start); l < c->nlev; ++l)
        gmgk::tail_weights(c->g[l], c->lv[l].L, c->tail_W[l], s);
    // uniform bricks (uniform.cuh): how many cells of each level the lean path covers, counted on the
    // device with the kernels' own footprint test; the counts come down with the next status read
    if (c->ubrick_dev) {
        unsigned long long* cnt = reinterpret_cast<unsigned long long*>(c->ubrick_dev + c->ubrick_total);
        cudaMemsetAsync(cnt, 0, kUniCountBytes, s);
        for (int l = 0; l < c->nlev; ++l) {
            if (!c->uni[l].brick) continue;
            int ty = 0, zc = 0;
            // the sweep's pass also lists the tiles that are not lean; until the host has read the
            // list's length back the launchers size the grid for all tiles (left_n = -1)
            c->uni[l].left_n = -1;
            if (gmgf::bulk_sweep_tiling(c->g[l], &ty, &zc))
                gmgk::uniform_cells(c->g[l], c->uni[l].brick, 128, ty, ty + 2, zc, 0, cnt + l,
                                    const_cast<int*>(c->uni[l].left_list), const_cast<unsigned int*>(c->uni[l].left_count), s);
            if (gmgf::res_bulk_tiling(c->g[l], &ty, &zc))
                gmgk::uniform_cells(c->g[l], c->uni[l].brick, 128, ty, ty + 1, zc, 1, cnt + GMG_MAX_LEVELS + l, nullptr, nullptr, s);
        }
        cudaMemcpyAsync(c->ucount_host, cnt, kUniCountBytes, cudaMemcpyDeviceToHost, s);
        c->uni_stats_pending = true;
    }
    gmgk::ctl_set_omega(c->sc, (double)c->prm.omega0, s);
}

// After a synchronisation behind set_coeffs_enqueue: the share of each level's cells on the lean path.
static void refresh_uniform_stats(gmg_ctx* c) {
    if (!c->uni_stats_pending) return;
    c->uni_stats_pending = false;
    const unsigned int* lcnt = reinterpret_cast<const unsigned int*>(c->ucount_host + 2 * GMG_MAX_LEVELS);
    for (int l = 0; l < c->nlev; ++l) {
        c->uni_frac_sweep[l] = c->uni[l].brick ? (double)c->ucount_host[l] / (double)c->g[l].N : 0.0;
        c->uni_frac_res[l] = c->uni[l].brick ? (double)c->ucount_host[GMG_MAX_LEVELS + l] / (double)c->g[l].N : 0.0;
        if (c->uni[l].left_list) {
            c->uni[l].left_n = (int)lcnt[l];
            int ty = 0, zc = 0;
            if (gmgf::bulk_sweep_tiling(c->g[l], &ty, &zc)) {
                const long long tiles = (long long)(c->g[l].n[0] / 128) * ((c->g[l].n[1] + ty - 1) / ty) *
                                        ((c->g[l].n[2] + zc - 1) / zc);
                c->uni[l].fold = 2LL * c->uni[l].left_n <= tiles;
            }
        }
    }
}

extern "C" int gmg_set_coeffs(gmg_ctx* c, const float* L_dev, void* stream) {
    if (!c || !L_dev) return GMG_EINVAL;
    if (!al16(L_dev)) { SET_ERR(c, "gmg_set_coeffs: L_dev must be 16-byte aligned"); return GMG_EINVAL; }
    if (!c->ws_set) { SET_ERR(c, "gmg_set_coeffs before gmg_set_workspace"); return GMG_ESTATE; }
    cudaStream_t s = (cudaStream_t)stream;
    set_coeffs_enqueue(c, L_dev, s);
    CUDA_TRY(c, cudaGetLastError());
    CUDA_TRY(c, cudaMemcpyAsync(c->sc_host, c->sc, sizeof(DevScalars), cudaMemcpyDeviceToHost, s));
    CUDA_TRY(c, cudaStreamSynchronize(s));
    if (c->sc_host->red[RED_CHECK] != 0.0) {
        SET_ERR(c, "gmg_set_coeffs: %.0f coefficient(s) negative, NaN or infinite",
                c->sc_host->red[RED_CHECK]);
        c->coeffs_set = false;
        return GMG_EINVAL;
    }
    c->coeffs_set = true;
    refresh_uniform_stats(c);
    return GMG_OK;
}

extern "C" int gmg_level_coeffs(gmg_ctx* c, int lev, float* L_out_dev, void* stream) {
    if (!c || lev < 0 || lev >= c->nlev || !L_out_dev || !al16(L_out_dev)) return GMG_EINVAL;
    if (!c->coeffs_set) { SET_ERR(c, "coefficients not set"); return GMG_ESTATE; }
    cudaStream_t s = (cudaStream_t)stream;
    CUDA_TRY(c, cudaMemcpyAsync(L_out_dev, c->lv[lev].L, 3 * (size_t)c->g[lev].N * sizeof(float),
                                cudaMemcpyDeviceToDevice, s));
    CUDA_TRY(c, cudaStreamSynchronize(s));
    return GMG_OK;
}

// ---- smoothing: nsweeps RBGS sweeps, result in p (reading O3) --------------------
// e_c != nullptr: the coarse correction P e_c is added to p first (fused into the first sweep
// on the fast path, a separate kernel otherwise).
// skip_first: the first fused sweep p -> q of this call has already been run (fused_norm path).
// Kernels one TMA-fed sweep of level l launches beyond the first: with uniform bricks marked the lean
// tiles and the remaining tiles are two kernels (one when either set is known to be empty), and a
// sweep that folds the prolongation in copies the footprints of the remaining tiles first.
static int sweep_extra_launches(const gmg_ctx* c, int l, bool with_pro) {
    if (!(c->fast_sweep[l] && c->tma_ok[l] && gmgf::tma_shape_ok(c->g[l]))) return 0;
    const gmgf::UniArgs& u = U(c, l);
    if (!u.brick) return 0;
    int ty = 0, zc = 0;
    if (!gmgf::bulk_sweep_tiling(c->g[l], &ty, &zc)) return 0;
    const long long tiles = (long long)(c->g[l].n[0] / 128) * ((c->g[l].n[1] + ty - 1) / ty) * ((c->g[l].n[2] + zc - 1) / zc);
    if (u.left_list && u.left_n == tiles) return 0;   // no lean tile: one kernel over the whole grid
    if (u.left_n == 0) return 0;                      // every tile lean
    return with_pro ? 2 : 1;
}

static void smooth(gmg_ctx* c, int l, float* p, const float* b, const float* omega, int nsweeps,
                   int first_colour, const float* e_c, cudaStream_t s, int skip_first = 0) {
    const LevelGeom& g = c->g[l];
    int done = 0;
    if (e_c && c->fast_sweep[l] && nsweeps >= 2 && c->tma_ok[l] && gmgf::tma_shape_ok(g)) {
        if (gmgf::sweep_fuses_prolong(g, U(c, l))) {
            // uniform bricks: the first sweep takes the correction along (lean tiles on the fly, the
            // others through a corrected copy of their footprints): e_c stays
        } else {
            // in front of the general TMA-fed sweep the correction is cheaper as its own streaming pass
            gmgf::prolong_add4(g, e_c, p, s);
            c->n_launch += 1;
            e_c = nullptr;
        }
    }
    if (c->fast_sweep[l] && nsweeps >= 2) {
        float* q = c->lv[l].q;
        const int pairs = nsweeps / 2;
        for (int i = 0; i < pairs; ++i) {
            if (!(i == 0 && skip_first)) {
                gmgf::rb_sweep(g, c->lv[l].L, p, q, b, omega, first_colour, (i == 0) ? e_c : nullptr, c->tma_ok[l], U(c, l), s);
                c->n_launch += 1 + sweep_extra_launches(c, l, i == 0 && e_c != nullptr);
            }
            gmgf::rb_sweep(g, c->lv[l].L, q, p, b, omega, first_colour, nullptr, c->tma_ok[l], U(c, l), s);
            c->n_launch += 1 + sweep_extra_launches(c, l, false);
        }
        done = 2 * pairs;
        e_c = nullptr;
    }
    if (e_c) {
        gmgk::prolong_add(g, e_c, p, s);
        c->n_launch += 1;
    }
    for (int i = done; i < nsweeps; ++i) {
        gmgk::half_sweep(g, c->lv[l].L, p, b, omega, first_colour, s);
        gmgk::half_sweep(g, c->lv[l].L, p, b, omega, 1 - first_colour, s);
        c->n_launch += 2;
    }
}

// ---- V-cycle: reading O7 (PAPER.md:39 smoother + coarse-grid correction; 51 "V-cycle") -------
static void enqueue_vcycle(gmg_ctx* c, float* p0, const float* b0, const float* omega, int sym,
                           cudaStream_t s, int skip_first = 0) {
    const bool cluster = c->ctail_start < c->nlev;
    const int nlev = c->nlev, ts = cluster ? c->ctail_start : c->tail_start;
    auto P = [&](int l) { return l == 0 ? p0 : c->lv[l].p; };
    auto B = [&](int l) { return l == 0 ? b0 : (const float*)c->lv[l].b; };
    const int post_first = sym ? 1 : 0;
    int l = 0;
    for (; l < ts && l < nlev - 1; ++l) {
        smooth(c, l, P(l), B(l), omega, c->prm.nu_pre, 0, nullptr, s, l == 0 ? skip_first : 0);
        if (c->fast_rr[l])
            gmgf::residual_restrict(c->g[l], c->lv[l].L, P(l), B(l), c->lv[l + 1].b, c->lv[l + 1].p, c->tma_ok[l], U(c, l), s);
        else
            gmgk::residual_restrict(c->g[l], c->lv[l].L, P(l), B(l), c->lv[l + 1].b, c->lv[l + 1].p, s);
        c->n_launch += 1;
    }
    if (ts < nlev) {
        // l == ts: the rest of the hierarchy is one kernel (a cluster of 8 CTAs, or a single CTA)
        TailArgs a;
        memset(&a, 0, sizeof(a));
        a.nlev = nlev - ts;
        for (int t = 0; t < a.nlev; ++t) {
            a.g[t] = c->g[ts + t];
            a.W[t] = c->tail_W[ts + t];
        }
        a.b_in = B(ts);
        a.p_in = (ts == 0) ? p0 : nullptr;
        a.p_out = P(ts);
        a.omega = omega;
        a.nu1 = c->prm.nu_pre; a.nu2 = c->prm.nu_post; a.nuc = c->prm.nu_coarse; a.sym = sym;
        if (cluster) gmgk::ctail_vcycle(a, c->ctail_lv, c->ctail_smem, s);
        else gmgk::tail_vcycle(a, c->tail_smem, s);
        c->n_launch += 1;
    } else {
        // coarsest level too large for shared memory: plain half-sweep launches
        const int cl = nlev - 1;
        if (!sym) {
            smooth(c, cl, P(cl), B(cl), omega, c->prm.nu_coarse, 0, nullptr, s);
        } else {
            smooth(c, cl, P(cl), B(cl), omega, c->prm.nu_coarse / 2, 0, nullptr, s);
            smooth(c, cl, P(cl), B(cl), omega, c->prm.nu_coarse / 2, 1, nullptr, s);
        }
    }
    for (l = (ts < nlev ? ts : nlev - 1) - 1; l >= 0; --l)
        smooth(c, l, P(l), B(l), omega, c->prm.nu_post, post_first, c->lv[l + 1].p, s);
}

// ---- N2: the paper's own "GMG-PCG" (PAPER.md:43 S3.1, Table 1 at PAPER.md:37; reading O12) -------
// m Jacobi-PCG iterations on A^l x = b restarted from x.  The four CG vectors are the level-0
// sized PCG vectors of the workspace on EVERY level: the CG state does not survive the visit to
// the coarser levels (the post-smoothing restarts), so the levels can share them.
// The float4 vector kernels of the CG iterations (kernels_pcg4.cu) skip the coefficient loads of the
// groups whose faces all carry the level's constants -- where the level streams from DRAM.  On an
// L2-resident level the brick look-up in front of the loads only adds latency (256 x 96 x 96: PCG
// 22.3 -> 24.3 ms), so it stays off there.
static const gmgf::UniArgs* lean_vectors(const gmg_ctx* c, int l) {
    return (c->uni[l].brick && (c->prm.tma_min_cells == 0 || c->g[l].N >= kLeanVectorMinCells)) ? &c->uni[l] : nullptr;
}

static void cg_smooth(gmg_ctx* c, int l, float* x, const float* b, int m, cudaStream_t s) {
    if (m <= 0) return;
    const LevelGeom& g = c->g[l];
    const float* L = c->lv[l].L;
    float *r = c->pcg_r, *d = c->pcg_d, *q = c->pcg_q, *sv = c->pcg_s;
    int nmax = g.n[0] > g.n[1] ? g.n[0] : g.n[1];
    if (g.n[2] > nmax) nmax = g.n[2];
    // a step longer than 16 n_max^2 is a direction that drifted into the null space (reading O12)
    const double alpha_cap = 16.0 * (double)nmax * (double)nmax;
    // small levels: the whole smoothing in one single-CTA kernel (kernels_pcg4.cu), same bits
    if (c->prm.small_cg && gmgk::cgs_small(g, L, x, b, m, alpha_cap, s)) {
        c->n_launch += 1;
        return;
    }
    // the control steps (begin / alpha / beta, stencil.cuh) ride on the reductions they follow
    ReduceBuf rb_begin = rbuf(c), rb_alpha = rbuf(c), rb_beta = rbuf(c);
    rb_begin.post = POST_CGS_BEGIN;
    rb_begin.post_arg = alpha_cap;
    rb_alpha.post = POST_CGS_ALPHA;
    rb_beta.post = POST_CGS_BETA;
    const gmgf::UniArgs* ul = lean_vectors(c, l);   // lean path of the float4 kernels
    gmgk::cgs_residual_sum(g, L, x, b, r, rbuf(c), s, ul);
    gmgk::cgs_start(g, L, r, d, rb_begin, s, ul);  // r -= mean; d = r/D; rho = r.d; begin
    c->n_launch += 2;
    for (int it = 0; it < m; ++it) {
        if (!(c->prm.fast_path && c->tma_ok[l] && (c->prm.tma_min_cells == 0 || g.N >= kBulkMatvecMinCells) &&
              gmgf::matvec_dot_bulk(g, L, d, q, rb_alpha, RED_DQ, U(c, l), s)))
            gmgk::matvec_dot(g, L, d, q, rb_alpha, RED_DQ, s, ul);     // ... alpha
        gmgk::pcg_update_pr(g, L, x, r, d, q, nullptr, 0, rbuf(c), s);
        c->n_launch += 2;
        if (it == m - 1) break;
        gmgk::jacobi_apply(g, L, r, sv, rb_beta, RED_RS, s, ul);   // ... beta
        gmgk::pcg_update_d(g.N, d, sv, c->sc, 0, s);
        c->n_launch += 2;
    }
}

// The V(nu_pre, nu_post) cycle of reading O7 with every group of sweeps replaced by as many CG
// iterations (O12b); the coarsest level gets nu_coarse iterations from the zero guess.
static void enqueue_vcycle_cgs(gmg_ctx* c, float* p0, const float* b0, cudaStream_t s) {
    const int nlev = c->nlev;
    auto P = [&](int l) { return l == 0 ? p0 : c->lv[l].p; };
    auto B = [&](int l) { return l == 0 ? b0 : (const float*)c->lv[l].b; };
    for (int l = 0; l < nlev - 1; ++l) {
        cg_smooth(c, l, P(l), B(l), c->prm.nu_pre, s);
        if (c->fast_rr[l])
            gmgf::residual_restrict(c->g[l], c->lv[l].L, P(l), B(l), c->lv[l + 1].b, c->lv[l + 1].p, c->tma_ok[l], U(c, l), s);
        else
            gmgk::residual_restrict(c->g[l], c->lv[l].L, P(l), B(l), c->lv[l + 1].b, c->lv[l + 1].p, s);
        c->n_launch += 1;
    }
    if (nlev == 1) {
        cg_smooth(c, 0, p0, b0, c->prm.nu_coarse, s);
        return;
    }
    cg_smooth(c, nlev - 1, P(nlev - 1), B(nlev - 1), c->prm.nu_coarse, s);
    for (int l = nlev - 2; l >= 0; --l) {
        if (c->fast_sweep[l] && c->tma_ok[l] && gmgf::tma_shape_ok(c->g[l])) gmgf::prolong_add4(c->g[l], c->lv[l + 1].p, P(l), s);
        else gmgk::prolong_add(c->g[l], c->lv[l + 1].p, P(l), s);
        c->n_launch += 1;
        cg_smooth(c, l, P(l), B(l), c->prm.nu_post, s);
    }
}

// Algorithmic bytes of that cycle: a smoothing of m iterations moves 48 B/cell at the restart
// (residual + sum 24, mean-free start 24), 44 per iteration (mat-vec 20, x/r update 24) and 32
// between iterations (Jacobi 20, direction update 12).
static double vcycle_cgs_bytes(const gmg_ctx* c) {
    auto sm = [](int m) { return m > 0 ? 48.0 + 44.0 * m + 32.0 * (m - 1) : 0.0; };
    double total = 0.0;
    for (int l = 0; l < c->nlev; ++l) {
        const double N = (double)c->g[l].N;
        const double m = (double)(c->g[l].c[0] * c->g[l].c[1] * c->g[l].c[2]);
        if (l == c->nlev - 1) total += N * sm(c->prm.nu_coarse);
        else total += N * (sm(c->prm.nu_pre) + sm(c->prm.nu_post) + (20.0 + 4.0 / m) + (8.0 + 4.0 / m));
    }
    return total + 20.0 * (double)c->g[0].N;
}

// Algorithmic HBM bytes of one V-cycle + its stopping-test norm.
// as_run: minus the 12 B/cell of coefficient streams the lean path (uniform.cuh) does not move
static double vcycle_bytes(const gmg_ctx* c, bool with_norm, bool as_run = false) {
    double total = 0.0;
    for (int l = 0; l < c->nlev; ++l) {
        const double N = (double)c->g[l].N;
        const double m = (double)(c->g[l].c[0] * c->g[l].c[1] * c->g[l].c[2]);
        const double fs = as_run ? c->uni_frac_sweep[l] : 0.0, fr = as_run ? c->uni_frac_res[l] : 0.0;
        if (l == c->nlev - 1) {
            total += N * 24.0 * c->prm.nu_coarse;
        } else {
            total += N * (24.0 - 12.0 * fs) * (c->prm.nu_pre + c->prm.nu_post);  // fused red+black sweeps
            total += N * (20.0 - 12.0 * fr + 4.0 / m);                            // residual + restriction
            total += N * (4.0 / m);                                 // prolongation fused in a sweep
        }
    }
    if (with_norm) total += (20.0 - (as_run ? 12.0 * c->uni_frac_res[0] : 0.0)) * (double)c->g[0].N;
    return total;
}

// ---- solve sections (enqueue only; capturable) -------------------------------------------------
struct LoopCtl {
    cudaGraphConditionalHandle cond;
    int use_cond;
};

static void level0_residual_norm2(gmg_ctx* c, const float* p, const float* z, cudaStream_t s) {
    if (c->prm.fast_path && gmgf::resrestrict_supported(c->g[0]))
        gmgf::residual_norm2(c->g[0], c->lv[0].L, p, z, rbuf(c), RED_RR, c->tma_ok[0], U(c, 0), s);
    else
        gmgk::residual_norm2(c->g[0], c->lv[0].L, p, z, rbuf(c), RED_RR, s);
}

// GMG-RBGS (readings O8, O9): pre = reference norm + initial residual norm + loop entry test.
// fused_norm path (gmg.h): cycle k+1's first pre-sweep p -> q (out of place) also sums the squared
// residual of p = p_k and ||z||^2.  It has to run before cycle k's omega update is known, so it
// runs with the decay-branch omega (omega_spec_f); when the update takes the growth branch
// instead, k_ctl_rbgs_cycle_end raises redo_first and the sweep is run again with the right omega.
static bool fused_norm_active(const gmg_ctx* c) {
    return c->fused_norm_on && gmgf::sweep_norm_supported(c->g[0]);
}
// with_ref: also ||z||^2 over the active cells (needed once, at loop entry)
// The cycle expected to be the last (kernels_ctl.cu) gets the plain norm pass instead of the next
// cycle's norm-carrying sweep, which would be wasted when the test then ends the solve.
static bool predict_active(const gmg_ctx* c) {
    return fused_norm_active(c) && gmgf::residual_norm_bulk_supported(c->g[0]);
}
static void first_sweep_with_norm(gmg_ctx* c, float* p, const float* z, const float* omega, bool with_ref,
                                  const int* run_flag, cudaStream_t s) {
    MUST_LAUNCH(c, gmgf::rb_sweep_with_norm(c->g[0], c->lv[0].L, p, c->lv[0].q, z, omega, 0, rbuf(c), RED_RR,
                                            with_ref ? RED_RREF : -1, run_flag, U(c, 0), s));
}

static void rbgs_pre(gmg_ctx* c, float* p, const float* z, LoopCtl lc, cudaStream_t s, bool cgs = false) {
    if (!cgs && fused_norm_active(c)) {
        first_sweep_with_norm(c, p, z, &c->sc->omega_f, true, nullptr, s);
        gmgk::ctl_begin(c->sc, c->hist, c->omegas, lc.cond, lc.use_cond, s);
        c->n_launch += 2 + sweep_extra_launches(c, 0, false);
        return;
    }
    // reference norm ||z|| over active cells and initial residual norm: one fused pass on big levels
    if (c->prm.fast_path && c->tma_ok[0] &&
        gmgf::residual_and_ref_norm2_bulk(c->g[0], c->lv[0].L, p, z, rbuf(c), RED_RR, RED_RREF, U(c, 0), s)) {
        c->n_launch += 1;
    } else {
        gmgk::active_norm2(c->g[0], c->lv[0].L, z, rbuf(c), RED_RREF, s);
        level0_residual_norm2(c, p, z, s);
        c->n_launch += 2;
    }
    gmgk::ctl_begin(c->sc, c->hist, c->omegas, lc.cond, lc.use_cond, s);
    c->n_launch += 1;
}
static void rbgs_body(gmg_ctx* c, float* p, const float* z, LoopCtl lc, cudaStream_t s, bool cgs = false) {
    if (!cgs && fused_norm_active(c)) {
        const bool pred = predict_active(c);
        if (pred) {   // after a failed "last cycle" prediction the first sweep is still to run
            MUST_LAUNCH(c, gmgf::rb_sweep_if(c->g[0], c->lv[0].L, p, c->lv[0].q, z, &c->sc->omega_f, 0, &c->sc->need_first, U(c, 0), s));
            c->n_launch += 1 + sweep_extra_launches(c, 0, false);
        }
        enqueue_vcycle(c, p, z, &c->sc->omega_f, 0, s, 1);             // its first sweep already ran
        if (pred) {   // expected to be the last cycle: the plain norm pass
            MUST_LAUNCH(c, gmgf::residual_norm2_bulk_if(c->g[0], c->lv[0].L, p, z, rbuf(c), RED_RR, &c->sc->expect_last, U(c, 0), s));
            c->n_launch += 1;
        }
        // otherwise: next cycle's first sweep, + ||z - A p_k||
        first_sweep_with_norm(c, p, z, &c->sc->omega_spec_f, false, pred ? &c->sc->run_s1n : nullptr, s);
        gmgk::ctl_rbgs_cycle_end(c->sc, c->hist, c->omegas, lc.cond, lc.use_cond, s);
        MUST_LAUNCH(c, gmgf::rb_sweep_if(c->g[0], c->lv[0].L, p, c->lv[0].q, z, &c->sc->omega_f, 0, &c->sc->redo_first, U(c, 0), s));
        c->n_launch += 3 + 2 * sweep_extra_launches(c, 0, false);   // (gated launches count: they are launches)
        return;
    }
    if (cgs) enqueue_vcycle_cgs(c, p, z, s);
    else enqueue_vcycle(c, p, z, &c->sc->omega_f, 0, s);
    level0_residual_norm2(c, p, z, s);
    gmgk::ctl_rbgs_cycle_end(c->sc, c->hist, c->omegas, lc.cond, lc.use_cond, s);
    c->n_launch += 2;
}

// PCG / GMG-PCG (readings O10, O11).
static void pcg_pre(gmg_ctx* c, float* p, const float* z, LoopCtl lc, cudaStream_t s) {
    gmgk::active_norm2(c->g[0], c->lv[0].L, z, rbuf(c), RED_RREF, s);
    gmgk::residual(c->g[0], c->lv[0].L, p, z, c->pcg_r, s);
    gmgk::norm2(c->g[0].N, c->pcg_r, rbuf(c), RED_RR, s);
    gmgk::fill(c->pcg_d, c->g[0].N, 0.0f, s);
    gmgk::ctl_begin(c->sc, c->hist, nullptr, lc.cond, lc.use_cond, s);
    c->n_launch += 5;
}
static void pcg_body(gmg_ctx* c, float* p, int gmg_precond, LoopCtl lc, cudaStream_t s) {
    const long long N = c->g[0].N;
    // beta and alpha (stencil.cuh, pcg_ctl_*) ride on the reductions they follow
    ReduceBuf rb_beta = rbuf(c), rb_alpha = rbuf(c);
    rb_beta.post = POST_PCG_BETA;
    rb_alpha.post = POST_PCG_ALPHA;
    if (!gmg_precond) {
        gmgk::jacobi_apply(c->g[0], c->lv[0].L, c->pcg_r, c->pcg_s, rb_beta, RED_RS, s, lean_vectors(c, 0));
        c->n_launch += 1;
    } else {
        gmgk::fill(c->pcg_s, N, 0.0f, s);
        enqueue_vcycle(c, c->pcg_s, c->pcg_r, &c->sc->omega_one, 1, s);
        gmgk::dot(N, c->pcg_r, c->pcg_s, rb_beta, RED_RS, s);
        c->n_launch += 2;
    }
    gmgk::pcg_update_d(N, c->pcg_d, c->pcg_s, c->sc, 0, s);
    if (!(c->prm.fast_path && c->tma_ok[0] && (c->prm.tma_min_cells == 0 || c->g[0].N >= kBulkMatvecMinCells) &&
          gmgf::matvec_dot_bulk(c->g[0], c->lv[0].L, c->pcg_d, c->pcg_q, rb_alpha, RED_DQ, U(c, 0), s)))
        gmgk::matvec_dot(c->g[0], c->lv[0].L, c->pcg_d, c->pcg_q, rb_alpha, RED_DQ, s, lean_vectors(c, 0));
    gmgk::pcg_update_pr(c->g[0], c->lv[0].L, p, c->pcg_r, c->pcg_d, c->pcg_q, nullptr, 0, rbuf(c), s);
    gmgk::ctl_pcg_check(c->sc, c->hist, lc.cond, lc.use_cond, s);
    c->n_launch += 4;
}
static void pcg_post(gmg_ctx* c, float* p, const float* z, cudaStream_t s) {
    // true residual at exit (the recursive one drove the test)
    level0_residual_norm2(c, p, z, s);
    c->n_launch += 1;
}

static void enqueue_init(gmg_ctx* c, float tol, int maxiter, int solver, cudaStream_t s) {
    // the relaxation factor belongs to the RBGS smoother: the CG-smoothed cycle leaves it alone
    gmgk::ctl_init(c->sc, (double)tol, maxiter, solver == GMG_GMG_CGS ? 0 : c->prm.adaptive, (double)c->prm.omega_min,
                   (double)c->prm.omega_down, (double)c->prm.omega_up,
                   (solver == GMG_GMG_RBGS && predict_active(c)) ? 1 : 0, s);
    c->n_launch += 1;
}

static void enqueue_pre(gmg_ctx* c, int solver, float* p, const float* z, LoopCtl lc, cudaStream_t s) {
    if (solver == GMG_GMG_RBGS || solver == GMG_GMG_CGS) rbgs_pre(c, p, z, lc, s, solver == GMG_GMG_CGS);
    else pcg_pre(c, p, z, lc, s);
}
static void enqueue_body(gmg_ctx* c, int solver, float* p, const float* z, LoopCtl lc, cudaStream_t s) {
    if (solver == GMG_GMG_RBGS) rbgs_body(c, p, z, lc, s);
    else if (solver == GMG_GMG_CGS) rbgs_body(c, p, z, lc, s, true);
    else pcg_body(c, p, solver == GMG_GMG_PCG, lc, s);
}
static void enqueue_post(gmg_ctx* c, int solver, float* p, const float* z, cudaStream_t s) {
    if (solver != GMG_GMG_RBGS && solver != GMG_GMG_CGS) pcg_post(c, p, z, s);
}

// Whole solve as ONE graph: init, pre, WHILE(cond){body}, post.
static int build_graph(gmg_ctx* c, GraphSlot& slot, int solver, float* p, const float* z, float tol,
                       int maxiter) {
    if (slot.exec) { cudaGraphExecDestroy(slot.exec); slot.exec = nullptr; }
    if (slot.graph) { cudaGraphDestroy(slot.graph); slot.graph = nullptr; }
    cudaGraph_t graph = nullptr;
    CUDA_TRY(c, cudaGraphCreate(&graph, 0));
    slot.graph = graph;
    LoopCtl lc;
    lc.use_cond = 1;
    CUDA_TRY(c, cudaGraphConditionalHandleCreate(&lc.cond, graph, 0, cudaGraphCondAssignDefault));
    CUDA_TRY(c, cudaStreamBeginCaptureToGraph(c->cap_a, graph, nullptr, nullptr, 0,
                                              cudaStreamCaptureModeRelaxed));
    c->n_launch = 0;
    enqueue_init(c, tol, maxiter, solver, c->cap_a);
    enqueue_pre(c, solver, p, z, lc, c->cap_a);
    slot.n_pre = c->n_launch;
    // conditional WHILE node after everything captured so far
    cudaStreamCaptureStatus st;
    const cudaGraphNode_t* deps = nullptr;
    size_t ndeps = 0;
    cudaGraph_t gcap = nullptr;
    CUDA_TRY(c, cudaStreamGetCaptureInfo(c->cap_a, &st, nullptr, &gcap, &deps, &ndeps));
    cudaGraphNodeParams np = {cudaGraphNodeTypeConditional};
    np.type = cudaGraphNodeTypeConditional;
    np.conditional.handle = lc.cond;
    np.conditional.type = cudaGraphCondTypeWhile;
    np.conditional.size = 1;
    cudaGraphNode_t wnode = nullptr;
    CUDA_TRY(c, cudaGraphAddNode(&wnode, graph, deps, ndeps, &np));
    cudaGraph_t body = np.conditional.phGraph_out[0];
    CUDA_TRY(c, cudaStreamBeginCaptureToGraph(c->cap_b, body, nullptr, nullptr, 0,
                                              cudaStreamCaptureModeRelaxed));
    c->n_launch = 0;
    use_side(c, 1);
    enqueue_body(c, solver, p, z, lc, c->cap_b);
    use_side(c, 0);
    slot.n_body = c->n_launch;
    cudaGraph_t body_out = nullptr;
    CUDA_TRY(c, cudaStreamEndCapture(c->cap_b, &body_out));
    CUDA_TRY(c, cudaStreamUpdateCaptureDependencies(c->cap_a, &wnode, 1,
                                                    cudaStreamSetCaptureDependencies));
    c->n_launch = 0;
    enqueue_post(c, solver, p, z, c->cap_a);
    slot.n_post = c->n_launch;
    cudaGraph_t gout = nullptr;
    CUDA_TRY(c, cudaStreamEndCapture(c->cap_a, &gout));
    CUDA_TRY(c, cudaGetLastError());
    if (c->enqueue_fail) {
        SET_ERR(c, "gmg_solve: a TMA-fed kernel of the plan could not be launched (tensor-map encode failed)");
        return GMG_ECUDA;
    }
    CUDA_TRY(c, cudaGraphInstantiate(&slot.exec, graph, 0));
    slot.p = p; slot.z = z; slot.solver = solver; slot.tol = tol; slot.maxiter = maxiter;
    slot.hist = c->hist;
    for (int l = 0; l < GMG_MAX_LEVELS; ++l) {
        slot.left_n[l] = l < c->nlev ? c->uni[l].left_n : -1;
        slot.fold[l] = l < c->nlev ? c->uni[l].fold : 0;
    }
    return GMG_OK;
}

static int ensure_history(gmg_ctx* c, int maxiter) {
    const int need = maxiter + 2;
    if (need <= c->hist_cap) return GMG_OK;
    drop_graphs(c);
    if (c->hist) cudaFree(c->hist);
    if (c->omegas) cudaFree(c->omegas);
    if (c->hist_pin) cudaFreeHost(c->hist_pin);
    c->hist = c->omegas = c->hist_pin = nullptr;
    c->hist_cap = 0;
    const int cap = need < 64 ? 64 : need;
    CUDA_TRY(c, cudaMalloc(&c->hist, sizeof(double) * cap));
    CUDA_TRY(c, cudaMalloc(&c->omegas, sizeof(double) * cap));
    CUDA_TRY(c, cudaMallocHost(&c->hist_pin, sizeof(double) * 2 * cap));
    c->hist_cap = cap;
    return GMG_OK;
}

// history[0..maxiter] and omegas[0..maxiter) into the pinned mirror, behind the solve on `s`
static cudaError_t read_history_async(gmg_ctx* c, int maxiter, cudaStream_t s) {
    const size_t n = (size_t)maxiter + 1;
    cudaError_t e = cudaMemcpyAsync(c->hist_pin, c->hist, sizeof(double) * n, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(c->hist_pin + c->hist_cap, c->omegas, sizeof(double) * n, cudaMemcpyDeviceToHost, s);
    return e;
}

extern "C" int gmg_solve(gmg_ctx* c, float* p, const float* z, float tol, int maxiter, int solver,
                         void* stream) {
    if (!c) return GMG_EINVAL;
    if (!p || !z || !(tol >= 0.0f) || maxiter < 0 || solver < GMG_PCG || solver > GMG_GMG_CGS) {
        SET_ERR(c, "gmg_solve: invalid argument");
        return GMG_EINVAL;
    }
    if (!al16(p) || !al16(z)) {
        SET_ERR(c, "gmg_solve: p_dev and z_dev must be 16-byte aligned");
        return GMG_EINVAL;
    }
    if (!c->ws_set || !c->coeffs_set) {
        SET_ERR(c, "gmg_solve before gmg_set_workspace / gmg_set_coeffs");
        return GMG_ESTATE;
    }
    cudaStream_t s = (cudaStream_t)stream;
    c->sc_fresh = false;
    c->enqueue_fail = false;
    int rc = ensure_history(c, maxiter);
    if (rc != GMG_OK) return rc;
    long long launches = 0;
    CUDA_TRY(c, cudaEventRecord(c->ev0, s));
    if (c->prm.use_graph) {
        GraphSlot& slot = c->slots[solver];
        bool same_lists = true;   // the launch grids in the graph were sized with these list lengths
        for (int l = 0; l < c->nlev; ++l)
            same_lists = same_lists && slot.left_n[l] == c->uni[l].left_n && slot.fold[l] == c->uni[l].fold;
        if (!slot.exec || slot.p != p || slot.z != z || slot.tol != tol || slot.maxiter != maxiter ||
            slot.hist != c->hist || !same_lists) {
            rc = build_graph(c, slot, solver, p, z, tol, maxiter);
            if (rc != GMG_OK) {
                // leave no stream in capture mode behind
                cudaGraph_t junk = nullptr;
                cudaStreamEndCapture(c->cap_b, &junk);
                cudaStreamEndCapture(c->cap_a, &junk);
                cudaGetLastError();
                return rc;
            }
            CUDA_TRY(c, cudaEventRecord(c->ev0, s));
        }
        CUDA_TRY(c, cudaGraphLaunch(slot.exec, s));
        CUDA_TRY(c, cudaEventRecord(c->ev1, s));
        CUDA_TRY(c, cudaMemcpyAsync(c->sc_host, c->sc, sizeof(DevScalars), cudaMemcpyDeviceToHost, s));
        CUDA_TRY(c, read_history_async(c, maxiter, s));
        CUDA_TRY(c, cudaStreamSynchronize(s));
        launches = slot.n_pre + slot.n_post + slot.n_body * (long long)c->sc_host->iter;
    } else {
        LoopCtl lc;
        lc.cond = 0;
        lc.use_cond = 0;
        c->n_launch = 0;
        enqueue_init(c, tol, maxiter, solver, s);
        enqueue_pre(c, solver, p, z, lc, s);
        while (!c->enqueue_fail) {
            CUDA_TRY(c, cudaMemcpyAsync(c->sc_host, c->sc, sizeof(DevScalars), cudaMemcpyDeviceToHost, s));
            CUDA_TRY(c, cudaStreamSynchronize(s));
            if (c->sc_host->done) break;
            enqueue_body(c, solver, p, z, lc, s);
            CUDA_TRY(c, cudaGetLastError());
        }
        if (c->enqueue_fail) {
            cudaStreamSynchronize(s);
            SET_ERR(c, "gmg_solve: a TMA-fed kernel of the plan could not be launched (tensor-map encode failed)");
            return GMG_ECUDA;
        }
        enqueue_post(c, solver, p, z, s);
        CUDA_TRY(c, cudaEventRecord(c->ev1, s));
        CUDA_TRY(c, cudaMemcpyAsync(c->sc_host, c->sc, sizeof(DevScalars), cudaMemcpyDeviceToHost, s));
        CUDA_TRY(c, read_history_async(c, maxiter, s));
        CUDA_TRY(c, cudaStreamSynchronize(s));
        launches = c->n_launch;
    }
    CUDA_TRY(c, cudaGetLastError());
    c->sc_fresh = true;
    const DevScalars& h = *c->sc_host;
    const int it = h.iter;
    // history and omegas came down with the status block (one synchronisation per solve)
    c->hist_host.assign(c->hist_pin, c->hist_pin + it + 1);
    if (solver == GMG_GMG_RBGS || solver == GMG_GMG_CGS)
        c->omegas_host.assign(c->hist_pin + c->hist_cap, c->hist_pin + c->hist_cap + it);
    else
        c->omegas_host.assign((size_t)it, 0.0);
    float ms = 0.0f;
    CUDA_TRY(c, cudaEventElapsedTime(&ms, c->ev0, c->ev1));
    gmg_stats_t& st = c->stats;
    st.solver = solver;
    st.status = h.status;
    st.iterations = it;
    st.levels = c->nlev;
    st.omega_final = h.omega;
    st.resid_ref = h.r_ref;
    st.resid_init_rel = c->hist_host[0];
    if (solver == GMG_GMG_RBGS || solver == GMG_GMG_CGS) st.resid_final_rel = c->hist_host[it];
    else st.resid_final_rel = (h.r_ref == 0.0) ? 0.0 : sqrt(h.red[RED_RR]) / h.r_ref;   // NaN stays NaN
    st.gpu_ms = ms;
    st.kernel_launches = launches;
    st.history_len = it + 1;
    const double N0 = (double)c->g[0].N;
    // loop entry: one pass over p, z, L -- unless the norms ride on sweeps that run anyway (fused_norm)
    refresh_uniform_stats(c);   // gmg_pressure_step: the flags came down with this solve's status
    st.uniform_fraction = c->uni_frac_sweep[0];
    st.uniform_fraction_residual = c->uni_frac_res[0];
    if (solver == GMG_GMG_RBGS) {
        const bool fn = fused_norm_active(c);
        st.bytes_algorithmic = (fn ? 0.0 : 20.0 * N0) + it * vcycle_bytes(c, !fn);
        st.bytes_as_run = (fn ? 0.0 : (20.0 - 12.0 * c->uni_frac_res[0]) * N0) + it * vcycle_bytes(c, !fn, true);
    }
    else if (solver == GMG_GMG_CGS) st.bytes_algorithmic = 20.0 * N0 + it * vcycle_cgs_bytes(c);
    else if (solver == GMG_PCG) st.bytes_algorithmic = 60.0 * N0 + it * 64.0 * N0;
    else st.bytes_algorithmic = 60.0 * N0 + it * (vcycle_bytes(c, false) + 52.0 * N0);
    if (solver != GMG_GMG_RBGS) st.bytes_as_run = st.bytes_algorithmic;   // not modelled for the comparison solvers
    if (h.status == GMG_EBREAKDOWN) SET_ERR(c, "PCG breakdown: d.q == 0 at iteration %d", it);
    return h.status;
}

extern "C" int gmg_solve_host(gmg_ctx* c, float* p_host, const float* z_host, float tol, int maxiter,
                              int solver, void* stream) {
    if (!c || !p_host || !z_host) return GMG_EINVAL;
    if (!c->ws_set || !c->coeffs_set) { SET_ERR(c, "gmg_solve_host before setup"); return GMG_ESTATE; }
    cudaStream_t s = (cudaStream_t)stream;
    const size_t bytes = (size_t)c->g[0].N * sizeof(float);
    CUDA_TRY(c, cudaMemcpyAsync(c->stage_z, z_host, bytes, cudaMemcpyHostToDevice, s));
    CUDA_TRY(c, cudaMemcpyAsync(c->stage_p, p_host, bytes, cudaMemcpyHostToDevice, s));
    const int rc = gmg_solve(c, c->stage_p, c->stage_z, tol, maxiter, solver, stream);
    if (rc < 0) return rc;
    CUDA_TRY(c, cudaMemcpyAsync(p_host, c->stage_p, bytes, cudaMemcpyDeviceToHost, s));
    CUDA_TRY(c, cudaStreamSynchronize(s));
    return rc;
}

extern "C" int gmg_solve_host_cold(gmg_ctx* c, float* p_host_out, const float* z_host, float tol, int maxiter,
                                   int solver, void* stream) {
    if (!c || !p_host_out || !z_host) return GMG_EINVAL;
    if (!c->ws_set || !c->coeffs_set) { SET_ERR(c, "gmg_solve_host_cold before setup"); return GMG_ESTATE; }
    cudaStream_t s = (cudaStream_t)stream;
    const size_t bytes = (size_t)c->g[0].N * sizeof(float);
    CUDA_TRY(c, cudaMemcpyAsync(c->stage_z, z_host, bytes, cudaMemcpyHostToDevice, s));
    CUDA_TRY(c, cudaMemsetAsync(c->stage_p, 0, bytes, s));
    const int rc = gmg_solve(c, c->stage_p, c->stage_z, tol, maxiter, solver, stream);
    if (rc < 0) return rc;
    CUDA_TRY(c, cudaMemcpyAsync(p_host_out, c->stage_p, bytes, cudaMemcpyDeviceToHost, s));
    CUDA_TRY(c, cudaStreamSynchronize(s));
    return rc;
}

extern "C" int gmg_stats(const gmg_ctx* c, gmg_stats_t* out) {
    if (!c || !out) return GMG_EINVAL;
    *out = c->stats;
    return GMG_OK;
}

extern "C" int gmg_history(const gmg_ctx* c, double* out, int cap) {
    if (!c || !out || cap < 0) return GMG_EINVAL;
    int n = (int)c->hist_host.size();
    if (n > cap) n = cap;
    for (int i = 0; i < n; ++i) out[i] = c->hist_host[i];
    return n;
}

extern "C" int gmg_omega_history(const gmg_ctx* c, double* out, int cap) {
    if (!c || !out || cap < 0) return GMG_EINVAL;
    int n = (int)c->omegas_host.size();
    if (n > cap) n = cap;
    for (int i = 0; i < n; ++i) out[i] = c->omegas_host[i];
    return n;
}

extern "C" int gmg_set_omega(gmg_ctx* c, float omega) {
    if (!c || !(omega > 0.0f)) return GMG_EINVAL;
    gmgk::ctl_set_omega(c->sc, (double)omega, 0);
    CUDA_TRY(c, cudaDeviceSynchronize());
    return GMG_OK;
}

// ---- per-operator hooks (parity tests) -----------------------------------------------------------
#define HOOK_PROLOGUE(cond_)                                                        \
    if (!c) return GMG_EINVAL;                                                      \
    if (!(cond_)) { SET_ERR(c, "%s: invalid argument", __func__); return GMG_EINVAL; } \
    if (!c->ws_set || !c->coeffs_set) { SET_ERR(c, "%s before setup", __func__); return GMG_ESTATE; } \
    cudaStream_t s = (cudaStream_t)stream;

#define HOOK_EPILOGUE()                       \
    CUDA_TRY(c, cudaGetLastError());          \
    CUDA_TRY(c, cudaStreamSynchronize(s));    \
    return GMG_OK;

extern "C" int gmg_op_residual(gmg_ctx* c, int lev, const float* p, const float* b, float* r,
                               void* stream) {
    HOOK_PROLOGUE(lev >= 0 && lev < c->nlev && p && b && r && al16(p) && al16(b) && al16(r))
    gmgk::residual(c->g[lev], c->lv[lev].L, p, b, r, s);
    HOOK_EPILOGUE()
}

extern "C" int gmg_op_smooth(gmg_ctx* c, int lev, float* p, const float* b, float omega, int nsweeps,
                             int first_colour, void* stream) {
    HOOK_PROLOGUE(lev >= 0 && lev < c->nlev && p && b && nsweeps >= 0 && al16(p) && al16(b) &&
                  (first_colour == 0 || first_colour == 1))
    gmgk::ctl_set_hook_omega(c->sc, omega, s);
    smooth(c, lev, p, b, &c->sc->omega_hook, nsweeps, first_colour, nullptr, s);
    HOOK_EPILOGUE()
}

extern "C" int gmg_op_restrict(gmg_ctx* c, int lev, const float* r_fine, float* b_coarse, void* stream) {
    HOOK_PROLOGUE(lev >= 0 && lev < c->nlev - 1 && r_fine && b_coarse && al16(r_fine) && al16(b_coarse))
    gmgk::restrict_sum(c->g[lev], r_fine, b_coarse, s);
    HOOK_EPILOGUE()
}

extern "C" int gmg_op_residual_restrict(gmg_ctx* c, int lev, const float* p, const float* b,
                                        float* b_coarse, void* stream) {
    HOOK_PROLOGUE(lev >= 0 && lev < c->nlev - 1 && p && b && b_coarse && al16(p) && al16(b) && al16(b_coarse))
    if (c->fast_rr[lev]) gmgf::residual_restrict(c->g[lev], c->lv[lev].L, p, b, b_coarse, nullptr, c->tma_ok[lev], U(c, lev), s);
    else gmgk::residual_restrict(c->g[lev], c->lv[lev].L, p, b, b_coarse, nullptr, s);
    HOOK_EPILOGUE()
}

extern "C" int gmg_op_prolong(gmg_ctx* c, int lev, const float* e_coarse, float* p_fine, void* stream) {
    HOOK_PROLOGUE(lev >= 0 && lev < c->nlev - 1 && e_coarse && p_fine && al16(e_coarse) && al16(p_fine))
    gmgk::prolong_add(c->g[lev], e_coarse, p_fine, s);
    HOOK_EPILOGUE()
}

extern "C" int gmg_op_vcycle(gmg_ctx* c, float* p, const float* z, float omega, int symmetric,
                             void* stream) {
    HOOK_PROLOGUE(p && z && al16(p) && al16(z))
    gmgk::ctl_set_hook_omega(c->sc, omega, s);
    enqueue_vcycle(c, p, z, &c->sc->omega_hook, symmetric ? 1 : 0, s);
    HOOK_EPILOGUE()
}

extern "C" int gmg_op_sweep_with_norm(gmg_ctx* c, int lev, const float* src, float* dst, const float* b,
                                      float omega, int first_colour, double* rr_out, double* bb_out,
                                      void* stream) {
    HOOK_PROLOGUE(lev >= 0 && lev < c->nlev && src && dst && b && src != dst && rr_out && bb_out &&
                  al16(src) && al16(dst) && al16(b) &&
                  (first_colour == 0 || first_colour == 1))
    gmgk::ctl_set_hook_omega(c->sc, omega, s);
    if (!gmgf::rb_sweep_with_norm(c->g[lev], c->lv[lev].L, src, dst, b, &c->sc->omega_hook, first_colour,
                                  rbuf(c), RED_HOOK, RED_HOOK2, nullptr, U(c, lev), s)) {
        SET_ERR(c, "gmg_op_sweep_with_norm: level %d cannot run the TMA-fed sweep", lev);
        return GMG_EINVAL;
    }
    CUDA_TRY(c, cudaGetLastError());
    CUDA_TRY(c, cudaMemcpyAsync(c->sc_host, c->sc, sizeof(DevScalars), cudaMemcpyDeviceToHost, s));
    CUDA_TRY(c, cudaStreamSynchronize(s));
    *rr_out = c->sc_host->red[RED_HOOK];
    *bb_out = c->sc_host->red[RED_HOOK2];
    return GMG_OK;
}

extern "C" int gmg_op_cg_smooth(gmg_ctx* c, int lev, float* x, const float* b, int iters, void* stream) {
    HOOK_PROLOGUE(lev >= 0 && lev < c->nlev && x && b && iters >= 0 && al16(x) && al16(b))
    cg_smooth(c, lev, x, b, iters, s);
    HOOK_EPILOGUE()
}

extern "C" int gmg_op_vcycle_cgs(gmg_ctx* c, float* p, const float* z, void* stream) {
    HOOK_PROLOGUE(p && z && al16(p) && al16(z))
    enqueue_vcycle_cgs(c, p, z, s);
    HOOK_EPILOGUE()
}

extern "C" int gmg_op_norm2(gmg_ctx* c, int lev, const float* r, double* out_host, void* stream) {
    HOOK_PROLOGUE(lev >= 0 && lev < c->nlev && r && out_host && al16(r))
    gmgk::norm2(c->g[lev].N, r, rbuf(c), RED_HOOK, s);
    CUDA_TRY(c, cudaGetLastError());
    CUDA_TRY(c, cudaMemcpyAsync(c->sc_host, c->sc, sizeof(DevScalars), cudaMemcpyDeviceToHost, s));
    CUDA_TRY(c, cudaStreamSynchronize(s));
    *out_host = sqrt(c->sc_host->red[RED_HOOK]);
    return GMG_OK;
}

// ---- N1: the steps either side of the solve ------------------------------
extern "C" int gmg_divergence(gmg_ctx* c, const float* u_dev, const float wall_hi[3], float* z_dev,
                              void* stream) {
    if (!c) return GMG_EINVAL;
    if (!u_dev || !z_dev) { SET_ERR(c, "gmg_divergence: null pointer"); return GMG_EINVAL; }
    if (!al16(u_dev) || !al16(z_dev)) { SET_ERR(c, "gmg_divergence: u_dev and z_dev must be 16-byte aligned"); return GMG_EINVAL; }
    cudaStream_t s = (cudaStream_t)stream;
    const float zero[3] = {0.0f, 0.0f, 0.0f};
    if (c->prm.fast_path && c->g[0].n[0] % 4 == 0) gmgk::divergence4(c->g[0], u_dev, wall_hi ? wall_hi : zero, z_dev, s);
    else gmgk::divergence(c->g[0], u_dev, wall_hi ? wall_hi : zero, z_dev, s);
    CUDA_TRY(c, cudaGetLastError());
    CUDA_TRY(c, cudaStreamSynchronize(s));
    return GMG_OK;
}

extern "C" int gmg_project(gmg_ctx* c, float* u_dev, const float* p_dev, void* stream) {
    if (!c) return GMG_EINVAL;
    if (!u_dev || !p_dev) { SET_ERR(c, "gmg_project: null pointer"); return GMG_EINVAL; }
    if (!al16(u_dev) || !al16(p_dev)) { SET_ERR(c, "gmg_project: u_dev and p_dev must be 16-byte aligned"); return GMG_EINVAL; }
    if (!c->coeffs_set) { SET_ERR(c, "gmg_project before gmg_set_coeffs"); return GMG_ESTATE; }
    cudaStream_t s = (cudaStream_t)stream;
    if (c->prm.fast_path && c->g[0].n[0] % 4 == 0) gmgk::project4(c->g[0], c->lv[0].L, p_dev, u_dev, s);
    else gmgk::project(c->g[0], c->lv[0].L, p_dev, u_dev, s);
    CUDA_TRY(c, cudaGetLastError());
    CUDA_TRY(c, cudaStreamSynchronize(s));
    return GMG_OK;
}

// One pressure step, enqueued back to back with ONE host synchronisation (the solve's status read):
// coefficients -> z = div u* (library-held buffer) -> solve (p_dev in/out) -> u* -= L grad p.
extern "C" int gmg_pressure_step(gmg_ctx* c, const float* L_dev, float* u_dev, const float wall_hi[3],
                                 float* p_dev, float tol, int maxiter, int solver, void* stream) {
    if (!c) return GMG_EINVAL;
    if (!L_dev || !u_dev || !p_dev) { SET_ERR(c, "gmg_pressure_step: null pointer"); return GMG_EINVAL; }
    if (!al16(L_dev) || !al16(u_dev) || !al16(p_dev)) {
        SET_ERR(c, "gmg_pressure_step: L_dev, u_dev and p_dev must be 16-byte aligned");
        return GMG_EINVAL;
    }
    if (!c->ws_set) { SET_ERR(c, "gmg_pressure_step before gmg_set_workspace"); return GMG_ESTATE; }
    cudaStream_t s = (cudaStream_t)stream;
    const float zero[3] = {0.0f, 0.0f, 0.0f};
    set_coeffs_enqueue(c, L_dev, s);
    c->coeffs_set = true;   // provisionally: the validation count is read with the solve's status block
    if (c->prm.fast_path && c->g[0].n[0] % 4 == 0) gmgk::divergence4(c->g[0], u_dev, wall_hi ? wall_hi : zero, c->stage_z, s);
    else gmgk::divergence(c->g[0], u_dev, wall_hi ? wall_hi : zero, c->stage_z, s);
    CUDA_TRY(c, cudaGetLastError());
    const int rc = gmg_solve(c, p_dev, c->stage_z, tol, maxiter, solver, stream);
    if (!c->sc_fresh) {          // the solve returned before its status read: nothing is validated
        c->coeffs_set = false;
        return rc;
    }
    if (c->sc_host->red[RED_CHECK] != 0.0) {
        SET_ERR(c, "gmg_pressure_step: %.0f coefficient(s) negative, NaN or infinite", c->sc_host->red[RED_CHECK]);
        c->coeffs_set = false;
        return GMG_EINVAL;
    }
    if (rc < 0) return rc;
    if (c->prm.fast_path && c->g[0].n[0] % 4 == 0) gmgk::project4(c->g[0], c->lv[0].L, p_dev, u_dev, s);
    else gmgk::project(c->g[0], c->lv[0].L, p_dev, u_dev, s);
    CUDA_TRY(c, cudaGetLastError());
    return rc;   // the projection is stream-ordered: synchronise `stream` before reading u on the host
}

extern "C" int gmg_describe_plan(const gmg_ctx* c, char* buf, size_t cap) {
    if (!c || !buf || cap == 0) return GMG_EINVAL;
    size_t off = 0;
    buf[0] = 0;
    for (int l = 0; l < c->nlev; ++l) {
        const bool tma = c->tma_ok[l] && c->g[l].n[0] % 128 == 0 && c->g[l].n[1] >= 4 && c->g[l].n[2] >= 8;
        const bool in_cluster = c->ctail_start < c->nlev && l >= c->ctail_start;
        const bool in_tail = in_cluster || l >= c->tail_start;
        // TMA-fed sweep: which of its two instantiations the plain (not norm-carrying) sweeps run
        const char* how = in_cluster ? "tail(8-CTA cluster smem)" : in_tail ? "tail(single-CTA smem)"
                          : (c->fast_sweep[l] ? (tma ? (gmgf::bulk_sweep_edge(c->g[l], false) ? "fused-rb-sweep(TMA,EDGE)"
                                                                                               : "fused-rb-sweep(TMA,rowcopy-edges)")
                                                     : "fused-rb-sweep") : "generic-half-sweeps");
        const char* rr = (in_tail || l == c->nlev - 1) ? "-"
                         : (c->fast_rr[l] ? "tiled" : "generic");
        // prolongation + correction on the way up: its own pass, or folded into the first post-sweep
        const char* pro = (in_tail || l == c->nlev - 1) ? "-"
                          : (tma && c->fast_sweep[l] && c->prm.nu_post >= 2 && gmgf::sweep_fuses_prolong(c->g[l], c->uni[l]))
                                ? "in-sweep" : "pass";
        int w = snprintf(buf + off, cap - off, "L%d %dx%dx%d c=%d%d%d sweep=%s resrestrict=%s prolong=%s\n", l,
                         c->g[l].n[0], c->g[l].n[1], c->g[l].n[2], c->g[l].c[0], c->g[l].c[1],
                         c->g[l].c[2], how, rr, pro);
        if (w < 0 || (size_t)w >= cap - off) break;
        off += (size_t)w;
    }
    return GMG_OK;
}

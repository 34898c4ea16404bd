// kernels_reduce.cu -- deterministic reductions (residual norm, PCG inner products), the PCG
// vector kernels and the single-thread on-device iteration control (no host round trip
// inside a solve).  PAPER.md:39 S3 "global inner products require costly reductions";
// BASELINE.json:north_star "warp-shuffle plus block-level residual-norm and PCG dot-product
// reductions with no host round-trip".
//
// Reduction scheme: grid-stride with a FIXED grid (a function of N only), FP64 per-thread
// partials, warp-shuffle + shared-memory block sum, block partials to global, and the last
// block to finish (ticket counter) sums the partials in index order.  No float atomics, so
// results are bit-reproducible run to run.
#include "stencil.cuh"

namespace gmgk {
using namespace gmgd;

static constexpr int kRT = 256;  // threads per reduction block

// float4 versions (kernels_pcg4.cu); false = shape or alignment not eligible
bool matvec_dot4(const LevelGeom& g, const float* L, const float* d, float* q, ReduceBuf rb, int slot, cudaStream_t s,
                 const gmgf::UniArgs* uni);
bool jacobi_apply4(const LevelGeom& g, const float* L, const float* r, float* s_out, ReduceBuf rb, int slot, cudaStream_t st,
                   const gmgf::UniArgs* uni);
bool pcg_update_pr4(long long N, float* p, float* r, const float* d, const float* q, ReduceBuf rb, cudaStream_t st);
bool pcg_update_d4(long long N, float* d, const float* s_in, const DevScalars* sc, cudaStream_t st);
bool dot4(long long N, const float* a, const float* b, ReduceBuf rb, int slot, cudaStream_t s);

static inline unsigned int reduce_blocks(long long N) {
    long long b = (N + (long long)kRT * 8 - 1) / ((long long)kRT * 8);
    if (b < 1) b = 1;
    if (b > GMG_REDUCE_MAX_BLOCKS) b = GMG_REDUCE_MAX_BLOCKS;
    return (unsigned int)b;
}

__device__ __forceinline__ void unflat(const LevelGeom& g, long long t, int& i, int& j, int& k) {
    const int nx = g.n[0], ny = g.n[1];
    const long long row = t / nx;
    i = (int)(t - row * nx);
    k = (int)(row / ny);
    j = (int)(row - (long long)k * ny);
}

// ---- sum r^2 with r = b - A p on active cells (stopping test, reading O9) -------------------
__global__ void __launch_bounds__(kRT)
k_residual_norm2(LevelGeom g, const float* __restrict__ L, const float* __restrict__ p,
                 const float* __restrict__ b, ReduceBuf rb, int slot) {
    double acc = 0.0;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < g.N;
         t += (long long)gridDim.x * blockDim.x) {
        int i, j, k;
        unflat(g, t, i, j, k);
        const Cell c = cell_stencil(g, L, p, i, j, k);
        const float r = (c.D != 0.0f) ? b[t] - c.Ap : 0.0f;
        acc += (double)r * (double)r;
    }
    finish_reduction(acc, 0.0, false, rb, slot, 0);
}

void residual_norm2(const LevelGeom& g, const float* L, const float* p, const float* b,
                    ReduceBuf rb, int slot, cudaStream_t s) {
    k_residual_norm2<<<reduce_blocks(g.N), kRT, 0, s>>>(g, L, p, b, rb, slot);
}

// ---- sum z^2 over active cells (reference norm, reading O9) ---------------------------------
__global__ void __launch_bounds__(kRT)
k_active_norm2(LevelGeom g, const float* __restrict__ L, const float* __restrict__ z, ReduceBuf rb,
               int slot) {
    double acc = 0.0;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < g.N;
         t += (long long)gridDim.x * blockDim.x) {
        int i, j, k;
        unflat(g, t, i, j, k);
        const float D = cell_diag(g, L, i, j, k);
        const float v = (D != 0.0f) ? z[t] : 0.0f;
        acc += (double)v * (double)v;
    }
    finish_reduction(acc, 0.0, false, rb, slot, 0);
}

void active_norm2(const LevelGeom& g, const float* L, const float* z, ReduceBuf rb, int slot,
                  cudaStream_t s) {
    k_active_norm2<<<reduce_blocks(g.N), kRT, 0, s>>>(g, L, z, rb, slot);
}

__global__ void __launch_bounds__(kRT)
k_dot(long long N, const float* __restrict__ a, const float* __restrict__ b, ReduceBuf rb, int slot) {
    double acc = 0.0;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < N;
         t += (long long)gridDim.x * blockDim.x)
        acc += (double)a[t] * (double)b[t];
    finish_reduction(acc, 0.0, false, rb, slot, 0);
}

void norm2(long long N, const float* r, ReduceBuf rb, int slot, cudaStream_t s) {
    if (dot4(N, r, r, rb, slot, s)) return;
    k_dot<<<reduce_blocks(N), kRT, 0, s>>>(N, r, r, rb, slot);
}
void dot(long long N, const float* a, const float* b, ReduceBuf rb, int slot, cudaStream_t s) {
    if (dot4(N, a, b, rb, slot, s)) return;
    k_dot<<<reduce_blocks(N), kRT, 0, s>>>(N, a, b, rb, slot);
}

// ---- coefficient check: every L finite and >= 0 ----------------------------------------------
__global__ void __launch_bounds__(kRT)
k_check_coeffs(long long N3, const float* __restrict__ L, ReduceBuf rb) {
    double bad = 0.0;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < N3;
         t += (long long)gridDim.x * blockDim.x) {
        const float v = L[t];
        if (!(v >= 0.0f) || isinf(v)) bad += 1.0;
    }
    finish_reduction(bad, 0.0, false, rb, RED_CHECK, 0);
}

void check_coeffs(const LevelGeom& g, const float* L, ReduceBuf rb, cudaStream_t s) {
    k_check_coeffs<<<reduce_blocks(3 * g.N), kRT, 0, s>>>(3 * g.N, L, rb);
}

// ---- PCG (reading O10) ------------------------------------------------------
// q = A d on every cell (inactive rows are all-zero) ; red[slot] = d.q
__global__ void __launch_bounds__(kRT)
k_matvec_dot(LevelGeom g, const float* __restrict__ L, const float* __restrict__ d,
             float* __restrict__ q, ReduceBuf rb, int slot) {
    double acc = 0.0;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < g.N;
         t += (long long)gridDim.x * blockDim.x) {
        int i, j, k;
        unflat(g, t, i, j, k);
        const Cell c = cell_stencil(g, L, d, i, j, k);
        q[t] = c.Ap;
        acc += (double)c.pc * (double)c.Ap;
    }
    finish_reduction(acc, 0.0, false, rb, slot, 0);
}

void matvec_dot(const LevelGeom& g, const float* L, const float* d, float* q, ReduceBuf rb,
                int slot, cudaStream_t s, const gmgf::UniArgs* uni) {
    if (matvec_dot4(g, L, d, q, rb, slot, s, uni)) return;
    k_matvec_dot<<<reduce_blocks(g.N), kRT, 0, s>>>(g, L, d, q, rb, slot);
}

// p += alpha d ; r -= alpha q ; red[RED_RR] = r.r
__global__ void __launch_bounds__(kRT)
k_pcg_update_pr(long long N, float* __restrict__ p, float* __restrict__ r,
                const float* __restrict__ d, const float* __restrict__ q, ReduceBuf rb) {
    const float alpha = (float)rb.sc->alpha;
    double acc = 0.0;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < N;
         t += (long long)gridDim.x * blockDim.x) {
        p[t] = fmaf(alpha, d[t], p[t]);
        const float rn = fmaf(-alpha, q[t], r[t]);
        r[t] = rn;
        acc += (double)rn * (double)rn;
    }
    finish_reduction(acc, 0.0, false, rb, RED_RR, 0);
}

void pcg_update_pr(const LevelGeom& g, const float* L, float* p, float* r, const float* d,
                   const float* q, float* s_out, int jacobi, ReduceBuf rb, cudaStream_t st) {
    (void)L; (void)s_out; (void)jacobi;
    if (pcg_update_pr4(g.N, p, r, d, q, rb, st)) return;
    k_pcg_update_pr<<<reduce_blocks(g.N), kRT, 0, st>>>(g.N, p, r, d, q, rb);
}

// d = s + beta d
__global__ void __launch_bounds__(kRT)
k_pcg_update_d(long long N, float* __restrict__ d, const float* __restrict__ s_in,
               const DevScalars* __restrict__ sc) {
    const float beta = (float)sc->beta;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < N;
         t += (long long)gridDim.x * blockDim.x)
        d[t] = fmaf(beta, d[t], s_in[t]);
}

void pcg_update_d(long long N, float* d, const float* s_in, const DevScalars* sc, int first,
                  cudaStream_t st) {
    (void)first;
    if (pcg_update_d4(N, d, s_in, sc, st)) return;
    k_pcg_update_d<<<reduce_blocks(N), kRT, 0, st>>>(N, d, s_in, sc);
}

// s = r / D on active cells, 0 elsewhere (Jacobi) ; red[slot] = r.s
__global__ void __launch_bounds__(kRT)
k_jacobi_apply(LevelGeom g, const float* __restrict__ L, const float* __restrict__ r,
               float* __restrict__ s_out, ReduceBuf rb, int slot) {
    double acc = 0.0;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < g.N;
         t += (long long)gridDim.x * blockDim.x) {
        int i, j, k;
        unflat(g, t, i, j, k);
        const float D = cell_diag(g, L, i, j, k);
        const float rv = r[t];
        const float sv = (D != 0.0f) ? rv / D : 0.0f;
        s_out[t] = sv;
        acc += (double)rv * (double)sv;
    }
    finish_reduction(acc, 0.0, false, rb, slot, 0);
}

void jacobi_apply(const LevelGeom& g, const float* L, const float* r, float* s_out, ReduceBuf rb,
                  int slot, cudaStream_t st, const gmgf::UniArgs* uni) {
    if (jacobi_apply4(g, L, r, s_out, rb, slot, st, uni)) return;
    k_jacobi_apply<<<reduce_blocks(g.N), kRT, 0, st>>>(g, L, r, s_out, rb, slot);
}

}  // namespace gmgk

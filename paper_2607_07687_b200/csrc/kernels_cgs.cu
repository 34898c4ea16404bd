// kernels_cgs.cu -- the Jacobi-PCG SMOOTHER of the paper's own "GMG-PCG" (
// PAPER.md:43 S3.1 "PCG can be used as a smoother", Table 1's middle row at PAPER.md:37;
// DESIGN.md reading O12): m preconditioned CG iterations on A^l x = b restarted from the
// current iterate of a level.  The iteration itself reuses the PCG vector kernels
// (kernels_reduce.cu / kernels_pcg4.cu / the TMA-fed mat-vec); this file holds what the restart
// needs -- the residual with its sum over the active cells, the mean-free start r -= mean,
// d = r/D, rho = r.d.  The single-thread control steps with the smoother's guards (stencil.cuh,
// cgs_ctl_*) ride on the reductions they follow (ReduceBuf::post) instead of being launches.
// Per-cell arithmetic in the one-cell and the float4 kernels is identical.
#include "stencil.cuh"

namespace gmgk {
using namespace gmgd;

static constexpr int kCT = 256;

// float4 versions (kernels_pcg4.cu); false = shape or alignment not eligible
bool cgs_residual_sum4(const LevelGeom& g, const float* L, const float* x, const float* b, float* r,
                       ReduceBuf rb, cudaStream_t s, const gmgf::UniArgs* uni);
bool cgs_start4(const LevelGeom& g, const float* L, float* r, float* d, ReduceBuf rb, cudaStream_t s,
                const gmgf::UniArgs* uni);

static inline unsigned int cgs_blocks(long long N) {
    long long b = (N + (long long)kCT * 8 - 1) / ((long long)kCT * 8);
    if (b < 1) b = 1;
    if (b > GMG_REDUCE_MAX_BLOCKS) b = GMG_REDUCE_MAX_BLOCKS;
    return (unsigned int)b;
}

__device__ __forceinline__ void cgs_unflat(const LevelGeom& g, long long t, int& i, int& j, int& k) {
    const int nx = g.n[0], ny = g.n[1];
    const long long row = t / nx;
    i = (int)(t - row * nx);
    k = (int)(row / ny);
    j = (int)(row - (long long)k * ny);
}

// r = b - A x on active cells, 0 elsewhere ; red[CGS_SUM] = sum r ; red[CGS_CNT] = #active
__global__ void __launch_bounds__(kCT)
k_cgs_residual_sum(LevelGeom g, const float* __restrict__ L, const float* __restrict__ x,
                   const float* __restrict__ b, float* __restrict__ r, ReduceBuf rb) {
    double sum = 0.0, cnt = 0.0;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < g.N;
         t += (long long)gridDim.x * blockDim.x) {
        int i, j, k;
        cgs_unflat(g, t, i, j, k);
        const Cell c = cell_stencil(g, L, x, i, j, k);
        const bool act = c.D != 0.0f;
        const float rv = act ? b[t] - c.Ap : 0.0f;
        r[t] = rv;
        sum += (double)rv;
        cnt += act ? 1.0 : 0.0;
    }
    finish_reduction(sum, cnt, true, rb, RED_CGS_SUM, RED_CGS_CNT);
}

void cgs_residual_sum(const LevelGeom& g, const float* L, const float* x, const float* b, float* r,
                      ReduceBuf rb, cudaStream_t s, const gmgf::UniArgs* uni) {
    if (cgs_residual_sum4(g, L, x, b, r, rb, s, uni)) return;
    k_cgs_residual_sum<<<cgs_blocks(g.N), kCT, 0, s>>>(g, L, x, b, r, rb);
}

// active cells: r -= mean ; d = r/D ; inactive: d = 0 ; red[RS] = r.d
__global__ void __launch_bounds__(kCT)
k_cgs_start(LevelGeom g, const float* __restrict__ L, float* __restrict__ r, float* __restrict__ d,
            ReduceBuf rb) {
    const float mu = cgs_mean(rb.sc);
    double acc = 0.0;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < g.N;
         t += (long long)gridDim.x * blockDim.x) {
        int i, j, k;
        cgs_unflat(g, t, i, j, k);
        const float D = cell_diag(g, L, i, j, k);
        float rv = 0.0f, dv = 0.0f;
        if (D != 0.0f) {
            rv = r[t] - mu;
            dv = rv / D;
        }
        r[t] = rv;
        d[t] = dv;
        acc += (double)rv * (double)dv;
    }
    finish_reduction(acc, 0.0, false, rb, RED_RS, 0);
}

void cgs_start(const LevelGeom& g, const float* L, float* r, float* d, ReduceBuf rb, cudaStream_t s,
               const gmgf::UniArgs* uni) {
    if (cgs_start4(g, L, r, d, rb, s, uni)) return;
    k_cgs_start<<<cgs_blocks(g.N), kCT, 0, s>>>(g, L, r, d, rb);
}

}  // namespace gmgk

// tail_common.cuh -- per-level building blocks of the shared-memory "tail" kernels
// (kernels_tail.cu: one CTA; kernels_ctail.cu: a cluster of CTAs).  A level with N cells is worked
// on by T = min(1024, N rounded up to a warp) threads that synchronise among themselves with a
// named barrier.  Same per-cell arithmetic (stencil.cuh) as every other kernel.
#pragma once
#include "stencil.cuh"

namespace gmgk {
using namespace gmgd;

static constexpr int kTailThreads = 1024;
static constexpr int kTailMaxPerThread = 6;  // cells of one level per thread (N <= 6144)

struct TailSmem {
    float* W[GMG_TAIL_MAX_LEVELS];  // [6][N] weights: x-lo, x-hi, y-lo, y-hi, z-lo, z-hi
    float* p[GMG_TAIL_MAX_LEVELS];
    float* b[GMG_TAIL_MAX_LEVELS];
};

__device__ __forceinline__ void named_sync(int nthreads) {
    if (nthreads >= kTailThreads) __syncthreads();
    else asm volatile("bar.sync 1, %0;" ::"r"(nthreads) : "memory");
}

// Ap and D of cell c = (i,j,k) from the shared-memory weights; neighbour indices wrap (a wrapped
// neighbour across a Neumann wall is multiplied by a zero weight).
__device__ __forceinline__ Cell tail_cell(const LevelGeom& g, const float* W, const float* p, int c, int i,
                                          int j, int k) {
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2], N = (int)g.N;
    const int sy = nx, sz = nx * ny;
    const float w0 = W[c], w1 = W[N + c], w2 = W[2 * N + c], w3 = W[3 * N + c], w4 = W[4 * N + c],
                w5 = W[5 * N + c];
    const float pc = p[c];
    const float pxl = p[(i == 0) ? c + (nx - 1) : c - 1];
    const float pxh = p[(i == nx - 1) ? c - (nx - 1) : c + 1];
    const float pyl = p[(j == 0) ? c + sy * (ny - 1) : c - sy];
    const float pyh = p[(j == ny - 1) ? c - sy * (ny - 1) : c + sy];
    const float pzl = p[(k == 0) ? c + sz * (nz - 1) : c - sz];
    const float pzh = p[(k == nz - 1) ? c - sz * (nz - 1) : c + sz];
    Cell r;
    r.pc = pc;
    r.Ap = apply7(pc, w0, w1, w2, w3, w4, w5, pxl, pxh, pyl, pyh, pzl, pzh);
    r.D = diag6(w0, w1, w2, w3, w4, w5);
    return r;
}

// `count` red-black sweeps on one level by the first T threads (named barrier between colours).
__device__ __forceinline__ void tail_sweeps(const LevelGeom& g, const float* W, float* p, const float* b,
                                            float omega, int count, int first, int T) {
    if ((int)threadIdx.x >= T || count <= 0) return;
    const int N = (int)g.N, nx = g.n[0], ny = g.n[1], nz = g.n[2];
    if (N <= T) {
        // one cell per thread: weights, neighbour addresses and b stay in registers, so a colour
        // step is six shared-memory loads, the stencil arithmetic, one store and the barrier
        const int c = threadIdx.x;
        const bool act = c < N;
        const int cc = act ? c : 0;
        const int row = cc / nx, i = cc - row * nx, k = row / ny, j = row - k * ny;
        const int sy = nx, sz = nx * ny;
        const float w0 = W[cc], w1 = W[N + cc], w2 = W[2 * N + cc], w3 = W[3 * N + cc], w4 = W[4 * N + cc],
                    w5 = W[5 * N + cc];
        const float D = diag6(w0, w1, w2, w3, w4, w5);
        const float bb = b[cc];
        const float* pxl = p + ((i == 0) ? cc + (nx - 1) : cc - 1);
        const float* pxh = p + ((i == nx - 1) ? cc - (nx - 1) : cc + 1);
        const float* pyl = p + ((j == 0) ? cc + sy * (ny - 1) : cc - sy);
        const float* pyh = p + ((j == ny - 1) ? cc - sy * (ny - 1) : cc + sy);
        const float* pzl = p + ((k == 0) ? cc + sz * (nz - 1) : cc - sz);
        const float* pzh = p + ((k == nz - 1) ? cc - sz * (nz - 1) : cc + sz);
        const int mycol = (i + j + k) & 1;
        float pc = p[cc];
        for (int s = 0; s < 2 * count; ++s) {
            const int colour = (s & 1) ? 1 - first : first;
            if (act && mycol == colour) {
                const float Ap = apply7(pc, w0, w1, w2, w3, w4, w5, *pxl, *pxh, *pyl, *pyh, *pzl, *pzh);
                pc = relax(pc, bb, Ap, D, omega);
                p[cc] = pc;
            }
            named_sync(T);
        }
        return;
    }
    int cell[kTailMaxPerThread], ijk[kTailMaxPerThread];
#pragma unroll
    for (int m = 0; m < kTailMaxPerThread; ++m) {
        const int c = threadIdx.x + m * T;
        cell[m] = (c < N) ? c : -1;
        const int row = c / nx, i = c - row * nx, k = row / ny, j = row - k * ny;
        ijk[m] = i | (j << 10) | (k << 20);
    }
    for (int s = 0; s < 2 * count; ++s) {
        const int colour = (s & 1) ? 1 - first : first;
#pragma unroll
        for (int m = 0; m < kTailMaxPerThread; ++m) {
            const int c = cell[m];
            if (c < 0) continue;
            const int i = ijk[m] & 1023, j = (ijk[m] >> 10) & 1023, k = ijk[m] >> 20;
            if (((i + j + k) & 1) != colour) continue;
            const Cell r = tail_cell(g, W, p, c, i, j, k);
            p[c] = relax(r.pc, b[c], r.Ap, r.D, omega);
        }
        named_sync(T);
    }
}

}  // namespace gmgk

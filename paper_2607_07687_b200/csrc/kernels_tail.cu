// kernels_tail.cu -- the coarse "tail" of the V-cycle as ONE single-CTA kernel.
//
// Levels whose arrays fit in one CTA's shared memory are launch-bound if run kernel by kernel
// (SURVEY.md S7 hard part 3: the coarsest level alone is nu_coarse = 32 sweeps = 64
// half-sweeps).  This kernel keeps, for every tail level, the six face weights of every cell
// (wall faces already zeroed), the unknown and the right-hand side in shared memory, and runs the
// complete sub-V-cycle (pre-sweeps, residual+restriction, coarsest-level sweeps, prolongation,
// post-sweeps; reading O7) on chip.  A level with N cells is worked on
// by T = min(1024, N rounded up to a warp) threads that synchronise among themselves with a
// named barrier, so the 64-cell coarsest level costs a two-warp barrier per colour, not a
// 32-warp one.  Same per-cell arithmetic (stencil.cuh) and the same child summation order as
// the other kernels, so it is bit-identical to them.
#include "tail_common.cuh"

namespace gmgk {
using namespace gmgd;

__global__ void __launch_bounds__(kTailThreads, 1) k_tail_vcycle(TailArgs a) {
    extern __shared__ __align__(16) float smem[];
    __shared__ TailSmem S;
    __shared__ int Tl[GMG_TAIL_MAX_LEVELS];
    const int tid = threadIdx.x;
    if (tid == 0) {
        float* cur = smem;
        for (int t = 0; t < a.nlev; ++t) {
            const int N = (int)a.g[t].N;
            S.W[t] = cur; cur += 6 * N;
            S.p[t] = cur; cur += N;
            S.b[t] = cur; cur += N;
            int T = (N + 31) / 32 * 32;
            Tl[t] = T > kTailThreads ? kTailThreads : T;
        }
    }
    __syncthreads();
    const float omega = *a.omega;
    // ---- face weights of every tail level: precomputed by gmg_set_coeffs (tail_weights) ---------
    for (int t = 0; t < a.nlev; ++t) {
        const int N6 = 6 * (int)a.g[t].N;
        for (int u = tid; u < N6; u += kTailThreads) S.W[t][u] = a.W[t][u];
    }
    {
        const int N = (int)a.g[0].N;
        for (int u = tid; u < N; u += kTailThreads) {
            S.b[0][u] = a.b_in[u];
            S.p[0][u] = a.p_in ? a.p_in[u] : 0.0f;
        }
    }
    __syncthreads();
    const int last = a.nlev - 1;
    // ---- down leg -------------------------------------------------------------------------------
    for (int t = 0; t < last; ++t) {
        const LevelGeom& g = a.g[t];
        tail_sweeps(g, S.W[t], S.p[t], S.b[t], omega, a.nu1, 0, Tl[t]);
        __syncthreads();
        const int ncx = g.n[0] / g.c[0], ncy = g.n[1] / g.c[1], ncz = g.n[2] / g.c[2];
        const int Nc = ncx * ncy * ncz;
        for (int u = tid; u < Nc; u += kTailThreads) {
            const int row = u / ncx;
            const int I = u - row * ncx, K = row / ncy, J = row - K * ncy;
            S.b[t + 1][u] = restrict_tree(g.c[0], g.c[1], g.c[2], [&](int e, int bb, int aa) {
                const int i = g.c[0] * I + e, j = g.c[1] * J + bb, k = g.c[2] * K + aa;
                const int f = i + g.n[0] * (j + g.n[1] * k);
                const Cell c = tail_cell(g, S.W[t], S.p[t], f, i, j, k);
                return (c.D != 0.0f) ? S.b[t][f] - c.Ap : 0.0f;
            });
            S.p[t + 1][u] = 0.0f;
        }
        __syncthreads();
    }
    // ---- coarsest level (reading O7: nu_coarse sweeps; O11: symmetric split) ---------------------
    {
        const LevelGeom& g = a.g[last];
        if (!a.sym) {
            tail_sweeps(g, S.W[last], S.p[last], S.b[last], omega, a.nuc, 0, Tl[last]);
        } else {
            tail_sweeps(g, S.W[last], S.p[last], S.b[last], omega, a.nuc / 2, 0, Tl[last]);
            tail_sweeps(g, S.W[last], S.p[last], S.b[last], omega, a.nuc / 2, 1, Tl[last]);
        }
        __syncthreads();
    }
    // ---- up leg ---------------------------------------------------------------------------------
    for (int t = last - 1; t >= 0; --t) {
        const LevelGeom& g = a.g[t];
        const int N = (int)g.N, nx = g.n[0], ny = g.n[1];
        const int ncx = nx / g.c[0], ncy = ny / g.c[1];
        for (int u = tid; u < N; u += kTailThreads) {
            const int row = u / nx, i = u - row * nx, k = row / ny, j = row - k * ny;
            const int parent = (i / g.c[0]) + ncx * ((j / g.c[1]) + ncy * (k / g.c[2]));
            S.p[t][u] += S.p[t + 1][parent];
        }
        __syncthreads();
        tail_sweeps(g, S.W[t], S.p[t], S.b[t], omega, a.nu2, a.sym ? 1 : 0, Tl[t]);
        __syncthreads();
    }
    {
        const int N = (int)a.g[0].N;
        for (int u = tid; u < N; u += kTailThreads) a.p_out[u] = S.p[0][u];
    }
}

__global__ void __launch_bounds__(256) k_tail_weights(LevelGeom g, const float* __restrict__ L, float* __restrict__ W) {
    const int N = (int)g.N, nx = g.n[0], ny = g.n[1];
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= N) return;
    const int row = c / nx, i = c - row * nx, k = row / ny, j = row - k * ny;
    float w[6];
    face_coeffs(g, L, i, j, k, c, w);
#pragma unroll
    for (int f = 0; f < 6; ++f) W[f * N + c] = w[f];
}

void tail_weights(const LevelGeom& g, const float* L, float* W, cudaStream_t s) {
    k_tail_weights<<<(unsigned int)((g.N + 255) / 256), 256, 0, s>>>(g, L, W);
}

size_t tail_smem_bytes(const TailArgs& a) {
    size_t cells = 0;
    for (int t = 0; t < a.nlev; ++t) cells += (size_t)a.g[t].N;
    return cells * 8 * sizeof(float);
}

int tail_configure(size_t max_bytes) {
    return (int)cudaFuncSetAttribute(k_tail_vcycle, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)max_bytes);
}

void tail_vcycle(const TailArgs& a, size_t smem_bytes, cudaStream_t s) {
    k_tail_vcycle<<<1, kTailThreads, smem_bytes, s>>>(a);
}

}  // namespace gmgk

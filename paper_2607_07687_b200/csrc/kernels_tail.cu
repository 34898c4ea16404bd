// kernels_tail.cu -- the coarse "tail" of the V-cycle as ONE single-CTA kernel.
//
// Levels whose arrays (3 L + p + b, all tail levels together) fit in one CTA's shared memory
// are launch-bound if run kernel by kernel (SURVEY.md S7 hard part 3: the coarsest level alone
// is nu_coarse = 32 sweeps = 64 half-sweeps).  This kernel loads the coefficients of every tail
// level and the right-hand side of the first tail level into shared memory, runs the complete
// sub-V-cycle (pre-sweeps, residual+restriction, coarsest-level sweeps, prolongation,
// post-sweeps; reading O7) with __syncthreads() between colours, and
// writes the first tail level's solution back.  Same per-cell arithmetic (stencil.cuh) and the
// same child summation order as the generic kernels, so it is bit-identical to them.
#include "stencil.cuh"

namespace gmgk {
using namespace gmgd;

static constexpr int kTailThreads = 1024;

struct TailSmem {
    float* L[GMG_TAIL_MAX_LEVELS];
    float* p[GMG_TAIL_MAX_LEVELS];
    float* b[GMG_TAIL_MAX_LEVELS];
};

__device__ __forceinline__ void unflat_s(const LevelGeom& g, int t, int& i, int& j, int& k) {
    const int nx = g.n[0], ny = g.n[1];
    const int row = t / nx;
    i = t - row * nx;
    k = row / ny;
    j = row - k * ny;
}

__device__ __forceinline__ void tail_half_sweep(const LevelGeom& g, const float* L, float* p,
                                                const float* b, float omega, int colour) {
    const int N = (int)g.N;
    for (int t = threadIdx.x; t < N; t += blockDim.x) {
        int i, j, k;
        unflat_s(g, t, i, j, k);
        if (((i + j + k) & 1) != colour) continue;
        const Cell c = cell_stencil(g, L, p, i, j, k);
        p[t] = relax(c.pc, b[t], c.Ap, c.D, omega);
    }
    __syncthreads();
}

__device__ __forceinline__ void tail_sweeps(const LevelGeom& g, const float* L, float* p,
                                            const float* b, float omega, int count, int first) {
    for (int s = 0; s < count; ++s) {
        tail_half_sweep(g, L, p, b, omega, first);
        tail_half_sweep(g, L, p, b, omega, 1 - first);
    }
}

__global__ void __launch_bounds__(kTailThreads, 1) k_tail_vcycle(TailArgs a) {
    extern __shared__ __align__(16) float smem[];
    __shared__ TailSmem S;
    if (threadIdx.x == 0) {
        float* cur = smem;
        for (int t = 0; t < a.nlev; ++t) {
            const int N = (int)a.g[t].N;
            S.L[t] = cur; cur += 3 * N;
            S.p[t] = cur; cur += N;
            S.b[t] = cur; cur += N;
        }
    }
    __syncthreads();
    const float omega = *a.omega;
    for (int t = 0; t < a.nlev; ++t) {
        const int N = (int)a.g[t].N;
        for (int u = threadIdx.x; u < 3 * N; u += blockDim.x) S.L[t][u] = a.L[t][u];
    }
    {
        const int N = (int)a.g[0].N;
        for (int u = threadIdx.x; u < N; u += blockDim.x) {
            S.b[0][u] = a.b_in[u];
            S.p[0][u] = a.p_in ? a.p_in[u] : 0.0f;
        }
    }
    __syncthreads();
    const int last = a.nlev - 1;
    // ---- down leg
    for (int t = 0; t < last; ++t) {
        const LevelGeom& g = a.g[t];
        tail_sweeps(g, S.L[t], S.p[t], S.b[t], omega, a.nu1, 0);
        const int ncx = g.n[0] / g.c[0], ncy = g.n[1] / g.c[1], ncz = g.n[2] / g.c[2];
        const int Nc = ncx * ncy * ncz;
        for (int u = threadIdx.x; u < Nc; u += blockDim.x) {
            const int row = u / ncx;
            const int I = u - row * ncx, K = row / ncy, J = row - K * ncy;
            S.b[t + 1][u] = restrict_tree(g.c[0], g.c[1], g.c[2], [&](int e, int bb, int aa) {
                const int i = g.c[0] * I + e, j = g.c[1] * J + bb, k = g.c[2] * K + aa;
                const int f = i + g.n[0] * (j + g.n[1] * k);
                const Cell c = cell_stencil(g, S.L[t], S.p[t], i, j, k);
                return (c.D != 0.0f) ? S.b[t][f] - c.Ap : 0.0f;
            });
            S.p[t + 1][u] = 0.0f;
        }
        __syncthreads();
    }
    // ---- coarsest level (reading O7: nu_coarse sweeps; O11: symmetric split)
    {
        const LevelGeom& g = a.g[last];
        if (!a.sym) {
            tail_sweeps(g, S.L[last], S.p[last], S.b[last], omega, a.nuc, 0);
        } else {
            tail_sweeps(g, S.L[last], S.p[last], S.b[last], omega, a.nuc / 2, 0);
            tail_sweeps(g, S.L[last], S.p[last], S.b[last], omega, a.nuc / 2, 1);
        }
    }
    // ---- up leg
    for (int t = last - 1; t >= 0; --t) {
        const LevelGeom& g = a.g[t];
        const int N = (int)g.N;
        const int ncx = g.n[0] / g.c[0], ncy = g.n[1] / g.c[1];
        for (int u = threadIdx.x; u < N; u += blockDim.x) {
            int i, j, k;
            unflat_s(g, u, i, j, k);
            const int parent = (i / g.c[0]) + ncx * ((j / g.c[1]) + ncy * (k / g.c[2]));
            S.p[t][u] += S.p[t + 1][parent];
        }
        __syncthreads();
        tail_sweeps(g, S.L[t], S.p[t], S.b[t], omega, a.nu2, a.sym ? 1 : 0);
    }
    {
        const int N = (int)a.g[0].N;
        for (int u = threadIdx.x; u < N; u += blockDim.x) a.p_out[u] = S.p[0][u];
    }
}

size_t tail_smem_bytes(const TailArgs& a) {
    size_t cells = 0;
    for (int t = 0; t < a.nlev; ++t) cells += (size_t)a.g[t].N;
    return cells * 5 * sizeof(float);
}

int tail_configure(size_t max_bytes) {
    return (int)cudaFuncSetAttribute(k_tail_vcycle, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)max_bytes);
}

void tail_vcycle(const TailArgs& a, size_t smem_bytes, cudaStream_t s) {
    k_tail_vcycle<<<1, kTailThreads, smem_bytes, s>>>(a);
}

}  // namespace gmgk

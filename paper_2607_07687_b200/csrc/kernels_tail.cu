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

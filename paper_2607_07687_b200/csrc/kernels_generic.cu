// kernels_generic.cu -- shape- and BC-generic kernels of the GMG solve: one thread per cell,
// plain (L1/L2-cached) loads.  They are the correctness baseline of the CUDA path, the
// per-operator test hooks, and the fallback for levels the tiled fast path does not take
// (tiny or odd extents).  Readings O1..O9 are in DESIGN.md; citations are PAPER.md lines.
#include "stencil.cuh"

namespace gmgk {
using namespace gmgd;

static constexpr int kThreads = 256;

static inline unsigned int blocks_for(long long work, int threads = kThreads) {
    long long b = (work + threads - 1) / threads;
    if (b < 1) b = 1;
    return (unsigned int)b;
}

__device__ __forceinline__ void unflatten(const LevelGeom& g, long long t, int& i, int& j, int& k) {
    const int nx = g.n[0], ny = g.n[1];
    const long long row = t / nx;
    i = (int)(t - row * nx);
    k = (int)(row / ny);
    j = (int)(row - (long long)k * ny);
}

// ---- O3: one colour half-sweep ("Red-Black Gauss-Seidel") ----------------------
__global__ void __launch_bounds__(kThreads)
k_half_sweep(LevelGeom g, const float* __restrict__ L, float* __restrict__ p,
             const float* __restrict__ b, const float* __restrict__ omega_ptr, int colour) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= g.N) return;
    int i, j, k;
    unflatten(g, t, i, j, k);
    if (((i + j + k) & 1) != colour) return;
    const float omega = *omega_ptr;
    const Cell c = cell_stencil(g, L, p, i, j, k);
    p[t] = relax(c.pc, b[t], c.Ap, c.D, omega);
}

void half_sweep(const LevelGeom& g, const float* L, float* p, const float* b, const float* omega,
                int colour, cudaStream_t s) {
    k_half_sweep<<<blocks_for(g.N), kThreads, 0, s>>>(g, L, p, b, omega, colour);
}

// ---- O9: r = b - A p on active cells, 0 elsewhere -------------------------------------------
__global__ void __launch_bounds__(kThreads)
k_residual(LevelGeom g, const float* __restrict__ L, const float* __restrict__ p,
           const float* __restrict__ b, float* __restrict__ r) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= g.N) return;
    int i, j, k;
    unflatten(g, t, i, j, k);
    const Cell c = cell_stencil(g, L, p, i, j, k);
    r[t] = (c.D != 0.0f) ? b[t] - c.Ap : 0.0f;
}

void residual(const LevelGeom& g, const float* L, const float* p, const float* b, float* r,
              cudaStream_t s) {
    k_residual<<<blocks_for(g.N), kThreads, 0, s>>>(g, L, p, b, r);
}

// ---- O6: restriction = sum over the children (PAPER.md:39 coarse-grid correction) ----------
__global__ void __launch_bounds__(kThreads)
k_restrict_sum(LevelGeom gf, const float* __restrict__ rf, float* __restrict__ bc) {
    const int ncx = gf.n[0] / gf.c[0], ncy = gf.n[1] / gf.c[1], ncz = gf.n[2] / gf.c[2];
    const long long Nc = (long long)ncx * ncy * ncz;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= Nc) return;
    const long long row = t / ncx;
    const int I = (int)(t - row * ncx), K = (int)(row / ncy), J = (int)(row - (long long)K * ncy);
    bc[t] = restrict_tree(gf.c[0], gf.c[1], gf.c[2], [&](int e, int bb, int a) {
        const long long f = (gf.c[0] * I + e) +
                            (long long)gf.n[0] * ((gf.c[1] * J + bb) + (long long)gf.n[1] * (gf.c[2] * K + a));
        return rf[f];
    });
}

void restrict_sum(const LevelGeom& gf, const float* rf, float* bc, cudaStream_t s) {
    const long long Nc = gf.N / ((long long)gf.c[0] * gf.c[1] * gf.c[2]);
    k_restrict_sum<<<blocks_for(Nc), kThreads, 0, s>>>(gf, rf, bc);
}

// ---- residual fused with restriction (BASELINE.json:north_star) -----------------------------
// One thread per coarse cell; children summed in stencil.cuh's canonical tree order, the same
// as k_restrict_sum, so fused == unfused bit for bit.
__global__ void __launch_bounds__(kThreads)
k_residual_restrict(LevelGeom gf, const float* __restrict__ L, const float* __restrict__ p,
                    const float* __restrict__ b, float* __restrict__ b_c, float* __restrict__ p_c) {
    const int ncx = gf.n[0] / gf.c[0], ncy = gf.n[1] / gf.c[1], ncz = gf.n[2] / gf.c[2];
    const long long Nc = (long long)ncx * ncy * ncz;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= Nc) return;
    const long long row = t / ncx;
    const int I = (int)(t - row * ncx), K = (int)(row / ncy), J = (int)(row - (long long)K * ncy);
    b_c[t] = restrict_tree(gf.c[0], gf.c[1], gf.c[2], [&](int e, int bb, int a) {
        const int i = gf.c[0] * I + e, j = gf.c[1] * J + bb, k = gf.c[2] * K + a;
        const long long f = i + (long long)gf.n[0] * (j + (long long)gf.n[1] * k);
        const Cell c = cell_stencil(gf, L, p, i, j, k);
        return (c.D != 0.0f) ? b[f] - c.Ap : 0.0f;
    });
    if (p_c) p_c[t] = 0.0f;
}

void residual_restrict(const LevelGeom& gf, const float* L, const float* p, const float* b,
                       float* b_c, float* p_c, cudaStream_t s) {
    const long long Nc = gf.N / ((long long)gf.c[0] * gf.c[1] * gf.c[2]);
    k_residual_restrict<<<blocks_for(Nc), kThreads, 0, s>>>(gf, L, p, b, b_c, p_c);
}

// ---- O6: prolongation = piecewise-constant injection, added unscaled ------------------------
__global__ void __launch_bounds__(kThreads)
k_prolong_add(LevelGeom gf, const float* __restrict__ e_c, float* __restrict__ p_f) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= gf.N) return;
    int i, j, k;
    unflatten(gf, t, i, j, k);
    const int ncx = gf.n[0] / gf.c[0], ncy = gf.n[1] / gf.c[1];
    const long long parent = (i / gf.c[0]) + (long long)ncx * ((j / gf.c[1]) + (long long)ncy * (k / gf.c[2]));
    p_f[t] += e_c[parent];
}

void prolong_add(const LevelGeom& gf, const float* e_c, float* p_f, cudaStream_t s) {
    k_prolong_add<<<blocks_for(gf.N), kThreads, 0, s>>>(gf, e_c, p_f);
}

__global__ void __launch_bounds__(kThreads) k_fill(float* __restrict__ x, long long N, float v) {
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < N;
         t += (long long)gridDim.x * blockDim.x)
        x[t] = v;
}

__global__ void __launch_bounds__(kThreads) k_fill4(float4* __restrict__ x, long long groups, float v) {
    const float4 w = make_float4(v, v, v, v);
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < groups;
         t += (long long)gridDim.x * blockDim.x)
        x[t] = w;
}

void fill(float* x, long long N, float v, cudaStream_t s) {
    if (N % 4 == 0 && (reinterpret_cast<size_t>(x) & 15) == 0) {
        unsigned int nb = blocks_for(N >> 2);
        if (nb > 148u * 16u) nb = 148u * 16u;
        k_fill4<<<nb, kThreads, 0, s>>>(reinterpret_cast<float4*>(x), N >> 2, v);
        return;
    }
    unsigned int nb = blocks_for(N);
    if (nb > 148u * 16u) nb = 148u * 16u;
    k_fill<<<nb, kThreads, 0, s>>>(x, N, v);
}


// ---- N1: the two steps either side of the solve in a staggered projection step
// ("predictor + corrector steps", one Poisson solve each).  u is component-major like
// L: u[d*N + idx] = velocity on the LOWER d-face of cell idx.
// z_I = sum_d [ u_d(I+e_d) - u_d(I) ]; upper face of the last cell: periodic -> u_d(index 0),
// Neumann -> the prescribed upper-wall value wall_hi[d].
__global__ void __launch_bounds__(kThreads)
k_divergence(LevelGeom g, const float* __restrict__ u, float whx, float why, float whz,
             float* __restrict__ z) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= g.N) return;
    int i, j, k;
    unflatten(g, t, i, j, k);
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const long long N = g.N, sy = nx, sz = (long long)nx * ny;
    const float xh = (i == nx - 1) ? (g.bc[0] ? whx : u[t - (nx - 1)]) : u[t + 1];
    const float yh = (j == ny - 1) ? (g.bc[1] ? why : u[N + t - sy * (ny - 1)]) : u[N + t + sy];
    const float zh = (k == nz - 1) ? (g.bc[2] ? whz : u[2 * N + t - sz * (nz - 1)]) : u[2 * N + t + sz];
    float s = xh - u[t];
    s += yh - u[N + t];
    s += zh - u[2 * N + t];
    z[t] = s;
}

void divergence(const LevelGeom& g, const float* u, const float wall_hi[3], float* z, cudaStream_t s) {
    k_divergence<<<blocks_for(g.N), kThreads, 0, s>>>(g, u, wall_hi[0], wall_hi[1], wall_hi[2], z);
}

// u_d(I) -= L_d(I) * (p_I - p_{I-e_d}); Neumann wall faces carry coefficient 0 (reading O2).
__global__ void __launch_bounds__(kThreads)
k_project(LevelGeom g, const float* __restrict__ L, const float* __restrict__ p, float* __restrict__ u) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= g.N) return;
    int i, j, k;
    unflatten(g, t, i, j, k);
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const long long N = g.N, sy = nx, sz = (long long)nx * ny;
    const float pc = p[t];
    const float wx = (i == 0 && g.bc[0]) ? 0.0f : L[t];
    const float wy = (j == 0 && g.bc[1]) ? 0.0f : L[N + t];
    const float wz = (k == 0 && g.bc[2]) ? 0.0f : L[2 * N + t];
    const float px = p[(i == 0) ? t + (nx - 1) : t - 1];
    const float py = p[(j == 0) ? t + sy * (ny - 1) : t - sy];
    const float pz = p[(k == 0) ? t + sz * (nz - 1) : t - sz];
    u[t] = fmaf(-wx, pc - px, u[t]);
    u[N + t] = fmaf(-wy, pc - py, u[N + t]);
    u[2 * N + t] = fmaf(-wz, pc - pz, u[2 * N + t]);
}

void project(const LevelGeom& g, const float* L, const float* p, float* u, cudaStream_t s) {
    k_project<<<blocks_for(g.N), kThreads, 0, s>>>(g, L, p, u);
}

// ---- O5: coefficient coarsening ("anisotropic coarsening operators") -----------
// L_d^{l+1}(J) = (1/c_d) * sum of the fine L_d over the prod_{e != d} c_e fine lower-d faces
// tiling the coarse face.  The fine wall plane of a Neumann axis counts as 0 (reading O2).
__global__ void __launch_bounds__(kThreads)
k_coarsen_coeffs(LevelGeom gf, const float* __restrict__ Lf, float* __restrict__ Lc) {
    const int nc[3] = {gf.n[0] / gf.c[0], gf.n[1] / gf.c[1], gf.n[2] / gf.c[2]};
    const long long Nc = (long long)nc[0] * nc[1] * nc[2];
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= 3 * Nc) return;
    const int d = (int)(t / Nc);
    const long long u = t - (long long)d * Nc;
    const long long row = u / nc[0];
    int Jc[3];
    Jc[0] = (int)(u - row * nc[0]);
    Jc[2] = (int)(row / nc[1]);
    Jc[1] = (int)(row - (long long)Jc[2] * nc[1]);
    const int e1 = (d + 1) % 3, e2 = (d + 2) % 3;
    float s = 0.0f;
    if (!(Jc[d] == 0 && gf.bc[d])) {
        for (int a = 0; a < gf.c[e1]; ++a)
            for (int bb = 0; bb < gf.c[e2]; ++bb) {
                int F[3];
                F[d] = gf.c[d] * Jc[d];
                F[e1] = gf.c[e1] * Jc[e1] + a;
                F[e2] = gf.c[e2] * Jc[e2] + bb;
                s += Lf[(long long)d * gf.N + F[0] + (long long)gf.n[0] * (F[1] + (long long)gf.n[1] * F[2])];
            }
    }
    Lc[t] = (gf.c[d] == 2) ? 0.5f * s : s;
}

void coarsen_coeffs(const LevelGeom& gf, const float* Lf, float* Lc, cudaStream_t s) {
    const long long Nc = gf.N / ((long long)gf.c[0] * gf.c[1] * gf.c[2]);
    k_coarsen_coeffs<<<blocks_for(3 * Nc), kThreads, 0, s>>>(gf, Lf, Lc);
}

}  // namespace gmgk

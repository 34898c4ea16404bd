// kernels_pcg4.cu -- the vector work of the (GMG-)PCG iteration (reading
// O10), four x-adjacent cells (one float4) per thread and grid-stride loops sized
// to the machine.  Per-cell arithmetic is that of the one-cell kernels in kernels_reduce.cu
// (same apply7 / diag6 argument order); only the order in which the FP64 partial sums are
// accumulated differs.  The launchers there dispatch here when nx % 4 == 0.
#include "stencil.cuh"
#include "uniform.cuh"

namespace gmgk {
using namespace gmgd;

static constexpr int kPT = 256;

static inline unsigned int blocks4(long long groups) {
    long long b = (groups + kPT - 1) / kPT;
    if (b < 1) b = 1;
    if (b > 148LL * 32) b = 148LL * 32;
    return (unsigned int)b;
}

// Grid for the stencil kernels: one grid-stride "wave" covers about one z plane, so the z +- 1
// neighbours a wave reads are the planes the previous and the next wave stream -- a few planes of
// five arrays, which stay in L2 -- instead of a window several planes deep whose edges are
// fetched twice from DRAM (measured 1.75x the algorithmic traffic with 148 x 32 blocks at 1024^3).
static inline unsigned int blocks_plane(const LevelGeom& g) {
    const long long plane_groups = ((long long)g.n[0] * g.n[1]) >> 2;
    long long b = (plane_groups + kPT - 1) / kPT;
    if (b < 148LL * 4) b = 148LL * 4;
    if (b > 148LL * 32) b = 148LL * 32;
    const long long all = ((g.N >> 2) + kPT - 1) / kPT;
    if (b > all) b = all < 1 ? 1 : all;
    return (unsigned int)b;
}

__device__ __forceinline__ float4 ldg4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
__device__ __forceinline__ float4 splat4(float v) { return make_float4(v, v, v, v); }

// Face weights of the four cells of group (i..i+3, j, k), wall faces zeroed (face_coeffs x 4).
struct W4 {
    float4 xl, xh, yl, yh, zl, zh;
};
__device__ __forceinline__ W4 weights4(const LevelGeom& g, const float* __restrict__ L, int i, int j, int k,
                                       long long c) {
    const long long N = g.N;
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const long long sy = nx, sz = (long long)nx * ny;
    const float* Lx = L;
    const float* Ly = L + N;
    const float* Lz = L + 2 * N;
    W4 w;
    w.xl = ldg4(Lx + c);
    float x4;  // lower x face of the cell after the group
    if (i + 4 == nx) x4 = g.bc[0] ? 0.0f : __ldg(Lx + c - (nx - 4));
    else x4 = __ldg(Lx + c + 4);
    w.xh = make_float4(w.xl.y, w.xl.z, w.xl.w, x4);
    if (i == 0 && g.bc[0]) w.xl.x = 0.0f;
    w.yl = (j == 0 && g.bc[1]) ? splat4(0.0f) : ldg4(Ly + c);
    w.yh = (j == ny - 1) ? (g.bc[1] ? splat4(0.0f) : ldg4(Ly + c - sy * (ny - 1))) : ldg4(Ly + c + sy);
    w.zl = (k == 0 && g.bc[2]) ? splat4(0.0f) : ldg4(Lz + c);
    w.zh = (k == nz - 1) ? (g.bc[2] ? splat4(0.0f) : ldg4(Lz + c - sz * (nz - 1))) : ldg4(Lz + c + sz);
    return w;
}

// Uniform bricks (uniform.cuh) in the float4 kernels: where every brick that holds one of the faces of
// a group is marked and none of them is a wall face, the six weights are the level's constants and
// the three coefficient arrays are not loaded (12 of the 20-24 B/cell of these passes); the same
// diag6 / apply7 run on the constants, so every cell gets the same bits.
struct UniK {
    const unsigned char* brick;   // nullptr: disabled
    float ux, uy, uz;
};
static inline UniK unik(const gmgf::UniArgs* u) {
    UniK k;
    k.brick = u ? u->brick : nullptr;
    k.ux = u ? u->ux : 0.0f;
    k.uy = u ? u->uy : 0.0f;
    k.uz = u ? u->uz : 0.0f;
    return k;
}
__device__ __forceinline__ bool group_uniform(const LevelGeom& g, const UniK& u, int i, int j, int k) {
    if (!u.brick) return false;
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    if ((g.bc[0] && (i == 0 || i + 4 == nx)) || (g.bc[1] && (j == 0 || j == ny - 1)) ||
        (g.bc[2] && (k == 0 || k == nz - 1)))
        return false;   // wall faces carry 0, not the constant
    const int nbx = gmgf::ub_count(nx, gmgf::kUBX), nby = gmgf::ub_count(ny, gmgf::kUBY);
    const int bx = i / gmgf::kUBX, by = j / gmgf::kUBY, bz = k / gmgf::kUBZ;
    const int i4 = (i + 4 == nx) ? 0 : i + 4, j1 = (j == ny - 1) ? 0 : j + 1, k1 = (k == nz - 1) ? 0 : k + 1;
    const unsigned char* row = u.brick + ((size_t)bz * nby + by) * nbx;
    return __ldg(row + bx) && __ldg(row + i4 / gmgf::kUBX) &&
           __ldg(u.brick + ((size_t)bz * nby + j1 / gmgf::kUBY) * nbx + bx) &&
           __ldg(u.brick + ((size_t)(k1 / gmgf::kUBZ) * nby + by) * nbx + bx);
}
__device__ __forceinline__ W4 weights4_uni(const LevelGeom& g, const float* __restrict__ L, const UniK& u, int i, int j,
                                           int k, long long c) {
    if (group_uniform(g, u, i, j, k)) {
        W4 w;
        w.xl = w.xh = splat4(u.ux);
        w.yl = w.yh = splat4(u.uy);
        w.zl = w.zh = splat4(u.uz);
        return w;
    }
    return weights4(g, L, i, j, k, c);
}

// group index -> (i, j, k); 32-bit arithmetic (a level has fewer than 2^31 cells)
__device__ __forceinline__ void unflat4(const LevelGeom& g, unsigned int t, int& i, int& j, int& k) {
    const unsigned int nx4 = (unsigned int)g.n[0] >> 2, ny = (unsigned int)g.n[1];
    const unsigned int row = t / nx4;
    i = 4 * (int)(t - row * nx4);
    const unsigned int kk = row / ny;
    k = (int)kk;
    j = (int)(row - kk * ny);
}

// q = A d on every cell ; red[slot] = d.q
__global__ void __launch_bounds__(kPT)
k_matvec_dot4(LevelGeom g, const float* __restrict__ L, const float* __restrict__ d, float* __restrict__ q,
              ReduceBuf rb, int slot, UniK uni) {
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const long long sy = nx, sz = (long long)nx * ny;
    const unsigned int groups = (unsigned int)(g.N >> 2);
    double acc = 0.0;
    for (unsigned int t = blockIdx.x * kPT + threadIdx.x; t < groups; t += gridDim.x * kPT) {
        int i, j, k;
        unflat4(g, t, i, j, k);
        const long long c = 4LL * t;
        const W4 w = weights4_uni(g, L, uni, i, j, k, c);
        const float4 dc = ldg4(d + c);
        const float dxm = __ldg(d + ((i == 0) ? c + (nx - 1) : c - 1));
        const float dxp = __ldg(d + ((i + 4 == nx) ? c - (nx - 4) : c + 4));
        const float4 dyl = ldg4(d + ((j == 0) ? c + sy * (ny - 1) : c - sy));
        const float4 dyh = ldg4(d + ((j == ny - 1) ? c - sy * (ny - 1) : c + sy));
        const float4 dzl = ldg4(d + ((k == 0) ? c + sz * (nz - 1) : c - sz));
        const float4 dzh = ldg4(d + ((k == nz - 1) ? c - sz * (nz - 1) : c + sz));
        float4 o;
        o.x = apply7(dc.x, w.xl.x, w.xh.x, w.yl.x, w.yh.x, w.zl.x, w.zh.x, dxm, dc.y, dyl.x, dyh.x, dzl.x, dzh.x);
        o.y = apply7(dc.y, w.xl.y, w.xh.y, w.yl.y, w.yh.y, w.zl.y, w.zh.y, dc.x, dc.z, dyl.y, dyh.y, dzl.y, dzh.y);
        o.z = apply7(dc.z, w.xl.z, w.xh.z, w.yl.z, w.yh.z, w.zl.z, w.zh.z, dc.y, dc.w, dyl.z, dyh.z, dzl.z, dzh.z);
        o.w = apply7(dc.w, w.xl.w, w.xh.w, w.yl.w, w.yh.w, w.zl.w, w.zh.w, dc.z, dxp, dyl.w, dyh.w, dzl.w, dzh.w);
        *reinterpret_cast<float4*>(q + c) = o;
        acc += (double)dc.x * (double)o.x + (double)dc.y * (double)o.y + (double)dc.z * (double)o.z +
               (double)dc.w * (double)o.w;
    }
    finish_reduction(acc, 0.0, false, rb, slot, 0);
}

// s = r / D on active cells, 0 elsewhere (Jacobi) ; red[slot] = r.s
__global__ void __launch_bounds__(kPT)
k_jacobi_apply4(LevelGeom g, const float* __restrict__ L, const float* __restrict__ r, float* __restrict__ s_out,
                ReduceBuf rb, int slot, UniK uni) {
    const unsigned int groups = (unsigned int)(g.N >> 2);
    double acc = 0.0;
    for (unsigned int t = blockIdx.x * kPT + threadIdx.x; t < groups; t += gridDim.x * kPT) {
        int i, j, k;
        unflat4(g, t, i, j, k);
        const long long c = 4LL * t;
        const W4 w = weights4_uni(g, L, uni, i, j, k, c);
        const float4 rv = ldg4(r + c);
        const float Dx = diag6(w.xl.x, w.xh.x, w.yl.x, w.yh.x, w.zl.x, w.zh.x);
        const float Dy = diag6(w.xl.y, w.xh.y, w.yl.y, w.yh.y, w.zl.y, w.zh.y);
        const float Dz = diag6(w.xl.z, w.xh.z, w.yl.z, w.yh.z, w.zl.z, w.zh.z);
        const float Dw = diag6(w.xl.w, w.xh.w, w.yl.w, w.yh.w, w.zl.w, w.zh.w);
        float4 sv;
        sv.x = (Dx != 0.0f) ? rv.x / Dx : 0.0f;
        sv.y = (Dy != 0.0f) ? rv.y / Dy : 0.0f;
        sv.z = (Dz != 0.0f) ? rv.z / Dz : 0.0f;
        sv.w = (Dw != 0.0f) ? rv.w / Dw : 0.0f;
        *reinterpret_cast<float4*>(s_out + c) = sv;
        acc += (double)rv.x * (double)sv.x + (double)rv.y * (double)sv.y + (double)rv.z * (double)sv.z +
               (double)rv.w * (double)sv.w;
    }
    finish_reduction(acc, 0.0, false, rb, slot, 0);
}

// p += alpha d ; r -= alpha q ; red[RED_RR] = r.r
__global__ void __launch_bounds__(kPT)
k_pcg_update_pr4(long long groups, float4* __restrict__ p, float4* __restrict__ r, const float4* __restrict__ d,
                 const float4* __restrict__ q, ReduceBuf rb) {
    const float alpha = (float)rb.sc->alpha;
    double acc = 0.0;
    for (long long t = (long long)blockIdx.x * kPT + threadIdx.x; t < groups; t += (long long)gridDim.x * kPT) {
        const float4 dv = __ldg(d + t), qv = __ldg(q + t);
        float4 pv = p[t], rv = r[t];
        pv.x = fmaf(alpha, dv.x, pv.x); pv.y = fmaf(alpha, dv.y, pv.y);
        pv.z = fmaf(alpha, dv.z, pv.z); pv.w = fmaf(alpha, dv.w, pv.w);
        rv.x = fmaf(-alpha, qv.x, rv.x); rv.y = fmaf(-alpha, qv.y, rv.y);
        rv.z = fmaf(-alpha, qv.z, rv.z); rv.w = fmaf(-alpha, qv.w, rv.w);
        p[t] = pv;
        r[t] = rv;
        acc += (double)rv.x * (double)rv.x + (double)rv.y * (double)rv.y + (double)rv.z * (double)rv.z +
               (double)rv.w * (double)rv.w;
    }
    finish_reduction(acc, 0.0, false, rb, RED_RR, 0);
}

// d = s + beta d
__global__ void __launch_bounds__(kPT)
k_pcg_update_d4(long long groups, float4* __restrict__ d, const float4* __restrict__ s_in,
                const DevScalars* __restrict__ sc) {
    const float beta = (float)sc->beta;
    for (long long t = (long long)blockIdx.x * kPT + threadIdx.x; t < groups; t += (long long)gridDim.x * kPT) {
        const float4 sv = __ldg(s_in + t);
        float4 dv = d[t];
        dv.x = fmaf(beta, dv.x, sv.x); dv.y = fmaf(beta, dv.y, sv.y);
        dv.z = fmaf(beta, dv.z, sv.z); dv.w = fmaf(beta, dv.w, sv.w);
        d[t] = dv;
    }
}

// red[slot] = a.b
__global__ void __launch_bounds__(kPT)
k_dot4(long long groups, const float4* __restrict__ a, const float4* __restrict__ b, ReduceBuf rb, int slot) {
    double acc = 0.0;
    for (long long t = (long long)blockIdx.x * kPT + threadIdx.x; t < groups; t += (long long)gridDim.x * kPT) {
        const float4 x = __ldg(a + t), y = __ldg(b + t);
        acc += (double)x.x * (double)y.x + (double)x.y * (double)y.y + (double)x.z * (double)y.z +
               (double)x.w * (double)y.w;
    }
    finish_reduction(acc, 0.0, false, rb, slot, 0);
}

// ---- CG smoother restart (reading O12; one-cell versions in kernels_cgs.cu) ------------------------
// r = b - A x on active cells, 0 elsewhere ; red[CGS_SUM] = sum r ; red[CGS_CNT] = #active
__global__ void __launch_bounds__(kPT)
k_cgs_residual_sum4(LevelGeom g, const float* __restrict__ L, const float* __restrict__ x,
                    const float* __restrict__ b, float* __restrict__ r, ReduceBuf rb, UniK uni) {
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const long long sy = nx, sz = (long long)nx * ny;
    const unsigned int groups = (unsigned int)(g.N >> 2);
    double sum = 0.0, cnt = 0.0;
    for (unsigned int t = blockIdx.x * kPT + threadIdx.x; t < groups; t += gridDim.x * kPT) {
        int i, j, k;
        unflat4(g, t, i, j, k);
        const long long c = 4LL * t;
        const W4 w = weights4_uni(g, L, uni, i, j, k, c);
        const float4 xc = ldg4(x + c);
        const float xm = __ldg(x + ((i == 0) ? c + (nx - 1) : c - 1));
        const float xp = __ldg(x + ((i + 4 == nx) ? c - (nx - 4) : c + 4));
        const float4 yl = ldg4(x + ((j == 0) ? c + sy * (ny - 1) : c - sy));
        const float4 yh = ldg4(x + ((j == ny - 1) ? c - sy * (ny - 1) : c + sy));
        const float4 zl = ldg4(x + ((k == 0) ? c + sz * (nz - 1) : c - sz));
        const float4 zh = ldg4(x + ((k == nz - 1) ? c - sz * (nz - 1) : c + sz));
        const float4 bv = ldg4(b + c);
        const float Ax = apply7(xc.x, w.xl.x, w.xh.x, w.yl.x, w.yh.x, w.zl.x, w.zh.x, xm, xc.y, yl.x, yh.x, zl.x, zh.x);
        const float Ay = apply7(xc.y, w.xl.y, w.xh.y, w.yl.y, w.yh.y, w.zl.y, w.zh.y, xc.x, xc.z, yl.y, yh.y, zl.y, zh.y);
        const float Az = apply7(xc.z, w.xl.z, w.xh.z, w.yl.z, w.yh.z, w.zl.z, w.zh.z, xc.y, xc.w, yl.z, yh.z, zl.z, zh.z);
        const float Aw = apply7(xc.w, w.xl.w, w.xh.w, w.yl.w, w.yh.w, w.zl.w, w.zh.w, xc.z, xp, yl.w, yh.w, zl.w, zh.w);
        const bool ax = diag6(w.xl.x, w.xh.x, w.yl.x, w.yh.x, w.zl.x, w.zh.x) != 0.0f;
        const bool ay = diag6(w.xl.y, w.xh.y, w.yl.y, w.yh.y, w.zl.y, w.zh.y) != 0.0f;
        const bool az = diag6(w.xl.z, w.xh.z, w.yl.z, w.yh.z, w.zl.z, w.zh.z) != 0.0f;
        const bool aw = diag6(w.xl.w, w.xh.w, w.yl.w, w.yh.w, w.zl.w, w.zh.w) != 0.0f;
        float4 rv;
        rv.x = ax ? bv.x - Ax : 0.0f;
        rv.y = ay ? bv.y - Ay : 0.0f;
        rv.z = az ? bv.z - Az : 0.0f;
        rv.w = aw ? bv.w - Aw : 0.0f;
        *reinterpret_cast<float4*>(r + c) = rv;
        sum += (double)rv.x + (double)rv.y + (double)rv.z + (double)rv.w;
        cnt += (double)((int)ax + (int)ay + (int)az + (int)aw);
    }
    finish_reduction(sum, cnt, true, rb, RED_CGS_SUM, RED_CGS_CNT);
}

// active cells: r -= mean ; d = r/D ; inactive: d = 0 ; red[RS] = r.d
__global__ void __launch_bounds__(kPT)
k_cgs_start4(LevelGeom g, const float* __restrict__ L, float* __restrict__ r, float* __restrict__ d,
             ReduceBuf rb, UniK uni) {
    const unsigned int groups = (unsigned int)(g.N >> 2);
    const float mu = cgs_mean(rb.sc);
    double acc = 0.0;
    for (unsigned int t = blockIdx.x * kPT + threadIdx.x; t < groups; t += gridDim.x * kPT) {
        int i, j, k;
        unflat4(g, t, i, j, k);
        const long long c = 4LL * t;
        const W4 w = weights4_uni(g, L, uni, i, j, k, c);
        const float4 r0 = *reinterpret_cast<const float4*>(r + c);
        const float Dx = diag6(w.xl.x, w.xh.x, w.yl.x, w.yh.x, w.zl.x, w.zh.x);
        const float Dy = diag6(w.xl.y, w.xh.y, w.yl.y, w.yh.y, w.zl.y, w.zh.y);
        const float Dz = diag6(w.xl.z, w.xh.z, w.yl.z, w.yh.z, w.zl.z, w.zh.z);
        const float Dw = diag6(w.xl.w, w.xh.w, w.yl.w, w.yh.w, w.zl.w, w.zh.w);
        float4 rv = make_float4(0.0f, 0.0f, 0.0f, 0.0f), dv = rv;
        if (Dx != 0.0f) { rv.x = r0.x - mu; dv.x = rv.x / Dx; }
        if (Dy != 0.0f) { rv.y = r0.y - mu; dv.y = rv.y / Dy; }
        if (Dz != 0.0f) { rv.z = r0.z - mu; dv.z = rv.z / Dz; }
        if (Dw != 0.0f) { rv.w = r0.w - mu; dv.w = rv.w / Dw; }
        *reinterpret_cast<float4*>(r + c) = rv;
        *reinterpret_cast<float4*>(d + c) = dv;
        acc += (double)rv.x * (double)dv.x + (double)rv.y * (double)dv.y + (double)rv.z * (double)dv.z +
               (double)rv.w * (double)dv.w;
    }
    finish_reduction(acc, 0.0, false, rb, RED_RS, 0);
}

// ---- a whole smoothing of the CG smoother on a small level, one CTA ---------------------------------
// On a level of at most 4096 cells the six kernels above are one or a few blocks each and a smoothing
// of m iterations is 4 m launch-bound launches (GMG_GMG_CGS on the paper's Table-1 sizes: 185 per
// cycle at 32 x 32 x 16).  k_cgs_small runs the restart and the m iterations in ONE CTA of B x 256
// threads, B = the grid those kernels would have (1..4): thread t owns the float4 group t, keeps its
// weights, x, r, d, q, s in registers and exchanges only the vector whose neighbours a stencil needs
// (x at the restart, d in every iteration) through shared memory.  Same expressions per cell; the
// sums follow finish_reduction's order (warp tree, the 8 warp sums of each 256-thread "block", the B
// block sums in lanes 0..B-1 of one more tree), so every cell gets the bits of the multi-launch path.
// The control steps (cgs_ctl_*) run on a DevScalars block in shared memory.
static constexpr int kSmallMaxGroups = 1024;

struct SmallSmem {
    float v[4 * kSmallMaxGroups];   // the vector a stencil reads
    double warp_part[32];
    double part[4];
    double total;
    DevScalars sc;
};

// sum over the CTA in finish_reduction's order; every thread gets the result
__device__ __forceinline__ double small_sum(double v, int B, SmallSmem& S) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    __syncthreads();
    if (lane == 0) S.warp_part[wid] = v;
    __syncthreads();
    if ((wid & 7) == 0) {   // first warp of a 256-thread "block": its 8 warp sums
        double t = (lane < 8) ? S.warp_part[wid + lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
        if (lane == 0) S.part[wid >> 3] = t;
    }
    __syncthreads();
    if (wid == 0) {         // the "last block": the B partials in index order
        double t = (lane < B) ? S.part[lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
        if (lane == 0) S.total = t;
    }
    __syncthreads();
    return S.total;
}

__global__ void __launch_bounds__(1024)
k_cgs_small(LevelGeom g, const float* __restrict__ L, float* __restrict__ x, const float* __restrict__ b, int m,
            double alpha_cap) {
    __shared__ SmallSmem S;
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const int sy = nx, sz = nx * ny;
    const int groups = (int)(g.N >> 2);
    const int B = (int)(blockDim.x >> 8);
    const int t = threadIdx.x;
    const bool act = t < groups;
    const int c = 4 * t;
    int i = 0, j = 0, k = 0;
    W4 w;
    w.xl = w.xh = w.yl = w.yh = w.zl = w.zh = splat4(0.0f);
    float4 xv = splat4(0.0f), bv = xv;
    if (act) {
        unflat4(g, (unsigned int)t, i, j, k);
        w = weights4(g, L, i, j, k, c);
        xv = ldg4(x + c);
        bv = ldg4(b + c);
        *reinterpret_cast<float4*>(S.v + c) = xv;
    }
    // neighbour offsets in the shared vector (as the kernels above index global memory)
    const int o_xm = (i == 0) ? c + (nx - 1) : c - 1, o_xp = (i + 4 == nx) ? c - (nx - 4) : c + 4;
    const int o_yl = (j == 0) ? c + sy * (ny - 1) : c - sy, o_yh = (j == ny - 1) ? c - sy * (ny - 1) : c + sy;
    const int o_zl = (k == 0) ? c + sz * (nz - 1) : c - sz, o_zh = (k == nz - 1) ? c - sz * (nz - 1) : c + sz;
    auto A4 = [&](const float4 vc) {   // A v on the own group, v's neighbours from shared memory
        const float vm = S.v[o_xm], vp = S.v[o_xp];
        const float4 yl = *reinterpret_cast<const float4*>(S.v + o_yl), yh = *reinterpret_cast<const float4*>(S.v + o_yh);
        const float4 zl = *reinterpret_cast<const float4*>(S.v + o_zl), zh = *reinterpret_cast<const float4*>(S.v + o_zh);
        float4 o;
        o.x = apply7(vc.x, w.xl.x, w.xh.x, w.yl.x, w.yh.x, w.zl.x, w.zh.x, vm, vc.y, yl.x, yh.x, zl.x, zh.x);
        o.y = apply7(vc.y, w.xl.y, w.xh.y, w.yl.y, w.yh.y, w.zl.y, w.zh.y, vc.x, vc.z, yl.y, yh.y, zl.y, zh.y);
        o.z = apply7(vc.z, w.xl.z, w.xh.z, w.yl.z, w.yh.z, w.zl.z, w.zh.z, vc.y, vc.w, yl.z, yh.z, zl.z, zh.z);
        o.w = apply7(vc.w, w.xl.w, w.xh.w, w.yl.w, w.yh.w, w.zl.w, w.zh.w, vc.z, vp, yl.w, yh.w, zl.w, zh.w);
        return o;
    };
    const float Dx = diag6(w.xl.x, w.xh.x, w.yl.x, w.yh.x, w.zl.x, w.zh.x);
    const float Dy = diag6(w.xl.y, w.xh.y, w.yl.y, w.yh.y, w.zl.y, w.zh.y);
    const float Dz = diag6(w.xl.z, w.xh.z, w.yl.z, w.yh.z, w.zl.z, w.zh.z);
    const float Dw = diag6(w.xl.w, w.xh.w, w.yl.w, w.yh.w, w.zl.w, w.zh.w);
    __syncthreads();
    // ---- restart: r = b - A x on active cells (k_cgs_residual_sum4), its sum and the active count ----
    float4 rv = splat4(0.0f);
    double sum = 0.0, cnt = 0.0;
    if (act) {
        const float4 Ax = A4(xv);
        const bool ax = Dx != 0.0f, ay = Dy != 0.0f, az = Dz != 0.0f, aw = Dw != 0.0f;
        rv.x = ax ? bv.x - Ax.x : 0.0f;
        rv.y = ay ? bv.y - Ax.y : 0.0f;
        rv.z = az ? bv.z - Ax.z : 0.0f;
        rv.w = aw ? bv.w - Ax.w : 0.0f;
        sum += (double)rv.x + (double)rv.y + (double)rv.z + (double)rv.w;
        cnt += (double)((int)ax + (int)ay + (int)az + (int)aw);
    }
    const double tsum = small_sum(sum, B, S);
    const double tcnt = small_sum(cnt, B, S);
    if (t == 0) { S.sc.red[RED_CGS_SUM] = tsum; S.sc.red[RED_CGS_CNT] = tcnt; }
    __syncthreads();
    // ---- mean-free start (k_cgs_start4): r -= mean; d = r/D; rho = r.d ----
    const float mu = cgs_mean(&S.sc);
    float4 dv = splat4(0.0f);
    double acc = 0.0;
    if (act) {
        const float4 r0 = rv;
        rv = splat4(0.0f);
        if (Dx != 0.0f) { rv.x = r0.x - mu; dv.x = rv.x / Dx; }
        if (Dy != 0.0f) { rv.y = r0.y - mu; dv.y = rv.y / Dy; }
        if (Dz != 0.0f) { rv.z = r0.z - mu; dv.z = rv.z / Dz; }
        if (Dw != 0.0f) { rv.w = r0.w - mu; dv.w = rv.w / Dw; }
        acc += (double)rv.x * (double)dv.x + (double)rv.y * (double)dv.y + (double)rv.z * (double)dv.z +
               (double)rv.w * (double)dv.w;
    }
    {
        const double rho = small_sum(acc, B, S);
        if (t == 0) { S.sc.red[RED_RS] = rho; cgs_ctl_begin(&S.sc, alpha_cap); }
    }
    for (int it = 0; it < m; ++it) {
        // q = A d, d.q (k_matvec_dot4); alpha
        if (act) *reinterpret_cast<float4*>(S.v + c) = dv;
        __syncthreads();
        float4 qv = splat4(0.0f);
        acc = 0.0;
        if (act) {
            qv = A4(dv);
            acc += (double)dv.x * (double)qv.x + (double)dv.y * (double)qv.y + (double)dv.z * (double)qv.z +
                   (double)dv.w * (double)qv.w;
        }
        const double dq = small_sum(acc, B, S);
        if (t == 0) { S.sc.red[RED_DQ] = dq; cgs_ctl_alpha(&S.sc); }
        __syncthreads();
        // x += alpha d; r -= alpha q (k_pcg_update_pr4)
        const float alpha = (float)S.sc.alpha;
        xv.x = fmaf(alpha, dv.x, xv.x); xv.y = fmaf(alpha, dv.y, xv.y);
        xv.z = fmaf(alpha, dv.z, xv.z); xv.w = fmaf(alpha, dv.w, xv.w);
        rv.x = fmaf(-alpha, qv.x, rv.x); rv.y = fmaf(-alpha, qv.y, rv.y);
        rv.z = fmaf(-alpha, qv.z, rv.z); rv.w = fmaf(-alpha, qv.w, rv.w);
        if (it == m - 1) break;
        // s = r/D, r.s (k_jacobi_apply4); beta; d = s + beta d (k_pcg_update_d4)
        float4 sv;
        sv.x = (Dx != 0.0f) ? rv.x / Dx : 0.0f;
        sv.y = (Dy != 0.0f) ? rv.y / Dy : 0.0f;
        sv.z = (Dz != 0.0f) ? rv.z / Dz : 0.0f;
        sv.w = (Dw != 0.0f) ? rv.w / Dw : 0.0f;
        acc = act ? (double)rv.x * (double)sv.x + (double)rv.y * (double)sv.y + (double)rv.z * (double)sv.z +
                        (double)rv.w * (double)sv.w
                  : 0.0;
        const double rs = small_sum(acc, B, S);
        if (t == 0) { S.sc.red[RED_RS] = rs; cgs_ctl_beta(&S.sc); }
        __syncthreads();
        const float beta = (float)S.sc.beta;
        dv.x = fmaf(beta, dv.x, sv.x); dv.y = fmaf(beta, dv.y, sv.y);
        dv.z = fmaf(beta, dv.z, sv.z); dv.w = fmaf(beta, dv.w, sv.w);
    }
    if (act) *reinterpret_cast<float4*>(x + c) = xv;
}

static inline bool al16(const void* p) { return (reinterpret_cast<size_t>(p) & 15) == 0; }

bool cgs_small(const LevelGeom& g, const float* L, float* x, const float* b, int m, double alpha_cap,
               cudaStream_t s) {
    const long long groups = g.N >> 2;
    // (x extents of 128 and more may take the TMA-fed mat-vec, whose sums run in another order)
    if (g.n[0] % 4 != 0 || g.n[0] >= 128 || groups > kSmallMaxGroups || m <= 0 || !al16(L) || !al16(x) || !al16(b))
        return false;
    const int B = (int)((groups + kPT - 1) / kPT);
    k_cgs_small<<<1, B * kPT, 0, s>>>(g, L, x, b, m, alpha_cap);
    return true;
}

bool matvec_dot4(const LevelGeom& g, const float* L, const float* d, float* q, ReduceBuf rb, int slot,
                 cudaStream_t s, const gmgf::UniArgs* uni) {
    if (g.n[0] % 4 != 0 || !al16(L) || !al16(d) || !al16(q)) return false;
    k_matvec_dot4<<<blocks_plane(g), kPT, 0, s>>>(g, L, d, q, rb, slot, unik(uni));
    return true;
}
bool jacobi_apply4(const LevelGeom& g, const float* L, const float* r, float* s_out, ReduceBuf rb, int slot,
                   cudaStream_t st, const gmgf::UniArgs* uni) {
    if (g.n[0] % 4 != 0 || !al16(L) || !al16(r) || !al16(s_out)) return false;
    k_jacobi_apply4<<<blocks_plane(g), kPT, 0, st>>>(g, L, r, s_out, rb, slot, unik(uni));
    return true;
}
bool pcg_update_pr4(long long N, float* p, float* r, const float* d, const float* q, ReduceBuf rb,
                    cudaStream_t st) {
    if (N % 4 != 0 || !al16(p) || !al16(r) || !al16(d) || !al16(q)) return false;
    k_pcg_update_pr4<<<blocks4(N >> 2), kPT, 0, st>>>(N >> 2, reinterpret_cast<float4*>(p),
                                                    reinterpret_cast<float4*>(r),
                                                    reinterpret_cast<const float4*>(d),
                                                    reinterpret_cast<const float4*>(q), rb);
    return true;
}
bool pcg_update_d4(long long N, float* d, const float* s_in, const DevScalars* sc, cudaStream_t st) {
    if (N % 4 != 0 || !al16(d) || !al16(s_in)) return false;
    k_pcg_update_d4<<<blocks4(N >> 2), kPT, 0, st>>>(N >> 2, reinterpret_cast<float4*>(d),
                                                   reinterpret_cast<const float4*>(s_in), sc);
    return true;
}
bool cgs_residual_sum4(const LevelGeom& g, const float* L, const float* x, const float* b, float* r,
                       ReduceBuf rb, cudaStream_t s, const gmgf::UniArgs* uni) {
    if (g.n[0] % 4 != 0 || !al16(L) || !al16(x) || !al16(b) || !al16(r)) return false;
    k_cgs_residual_sum4<<<blocks_plane(g), kPT, 0, s>>>(g, L, x, b, r, rb, unik(uni));
    return true;
}
bool cgs_start4(const LevelGeom& g, const float* L, float* r, float* d, ReduceBuf rb, cudaStream_t s,
                const gmgf::UniArgs* uni) {
    if (g.n[0] % 4 != 0 || !al16(L) || !al16(r) || !al16(d)) return false;
    k_cgs_start4<<<blocks_plane(g), kPT, 0, s>>>(g, L, r, d, rb, unik(uni));
    return true;
}
bool dot4(long long N, const float* a, const float* b, ReduceBuf rb, int slot, cudaStream_t s) {
    if (N % 4 != 0 || !al16(a) || !al16(b)) return false;
    k_dot4<<<blocks4(N >> 2), kPT, 0, s>>>(N >> 2, reinterpret_cast<const float4*>(a),
                                          reinterpret_cast<const float4*>(b), rb, slot);
    return true;
}

}  // namespace gmgk

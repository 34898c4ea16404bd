// stencil.cuh -- device helpers shared by every kernel of the CUDA path, so that the generic,
// fused and single-CTA kernels produce bit-identical cell updates.
//
// Operator (reading O1; PAPER.md:43 S3.1 "variable-coefficient Poisson"):
//   (A p)_I = sum_d [ L_d(I)(p_{I-e_d} - p_I) + L_d(I+e_d)(p_{I+e_d} - p_I) ]
//   D_I     = - sum_d [ L_d(I) + L_d(I+e_d) ]          cell active  <=>  D_I != 0
// Boundary handling (reading O2): periodic = index wrap; Neumann = coefficient 0 on the wall
// faces (the stored plane L_d(index 0) is ignored; there is no upper wall face).
#pragma once
#include "gmg_internal.h"

namespace gmgd {

// The one arithmetic order used everywhere: x-lo, x-hi, y-lo, y-hi, z-lo, z-hi.
__device__ __forceinline__ float apply7(float pc, float wxl, float wxh, float wyl, float wyh,
                                        float wzl, float wzh, float pxl, float pxh, float pyl,
                                        float pyh, float pzl, float pzh) {
    float s = wxl * (pxl - pc);
    s = fmaf(wxh, pxh - pc, s);
    s = fmaf(wyl, pyl - pc, s);
    s = fmaf(wyh, pyh - pc, s);
    s = fmaf(wzl, pzl - pc, s);
    s = fmaf(wzh, pzh - pc, s);
    return s;
}

__device__ __forceinline__ float diag6(float wxl, float wxh, float wyl, float wyh, float wzl,
                                       float wzh) {
    return -(((wxl + wxh) + (wyl + wyh)) + (wzl + wzh));
}

// RBGS cell update (readings O3, O8):  p_I += omega (b_I - (A p)_I) / D_I  on active cells.
__device__ __forceinline__ float relax(float pc, float b, float Ap, float D, float omega) {
    // branch-free: an inactive cell (D == 0) adds 0/1
    const bool act = D != 0.0f;
    return pc + __fdividef(act ? omega * (b - Ap) : 0.0f, act ? D : 1.0f);
}

// Gathers the seven p values and six face coefficients of cell (i,j,k) with plain loads.
// Works on global or shared pointers.  Out-of-range neighbours on a Neumann axis read a
// wrapped (valid, finite) value that is multiplied by a zero coefficient.
struct Cell {
    float pc, Ap, D;
};

__device__ __forceinline__ void face_coeffs(const LevelGeom& g, const float* __restrict__ L, int i,
                                            int j, int k, long long c, float w[6]) {
    const long long N = g.N;
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const long long sy = nx, sz = (long long)nx * ny;
    const float* Lx = L;
    const float* Ly = L + N;
    const float* Lz = L + 2 * N;
    w[0] = (i == 0 && g.bc[0]) ? 0.0f : Lx[c];
    w[1] = (i == nx - 1) ? (g.bc[0] ? 0.0f : Lx[c - (nx - 1)]) : Lx[c + 1];
    w[2] = (j == 0 && g.bc[1]) ? 0.0f : Ly[c];
    w[3] = (j == ny - 1) ? (g.bc[1] ? 0.0f : Ly[c - sy * (ny - 1)]) : Ly[c + sy];
    w[4] = (k == 0 && g.bc[2]) ? 0.0f : Lz[c];
    w[5] = (k == nz - 1) ? (g.bc[2] ? 0.0f : Lz[c - sz * (nz - 1)]) : Lz[c + sz];
}

__device__ __forceinline__ Cell cell_stencil(const LevelGeom& g, const float* __restrict__ L,
                                             const float* __restrict__ p, int i, int j, int k) {
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const long long sy = nx, sz = (long long)nx * ny;
    const long long c = i + sy * j + sz * k;
    float w[6];
    face_coeffs(g, L, i, j, k, c, w);
    const float pc = p[c];
    const float pxl = p[(i == 0) ? c + (nx - 1) : c - 1];
    const float pxh = p[(i == nx - 1) ? c - (nx - 1) : c + 1];
    const float pyl = p[(j == 0) ? c + sy * (ny - 1) : c - sy];
    const float pyh = p[(j == ny - 1) ? c - sy * (ny - 1) : c + sy];
    const float pzl = p[(k == 0) ? c + sz * (nz - 1) : c - sz];
    const float pzh = p[(k == nz - 1) ? c - sz * (nz - 1) : c + sz];
    Cell r;
    r.pc = pc;
    r.Ap = apply7(pc, w[0], w[1], w[2], w[3], w[4], w[5], pxl, pxh, pyl, pyh, pzl, pzh);
    r.D = diag6(w[0], w[1], w[2], w[3], w[4], w[5]);
    return r;
}

__device__ __forceinline__ float cell_diag(const LevelGeom& g, const float* __restrict__ L, int i,
                                           int j, int k) {
    const long long c = i + (long long)g.n[0] * (j + (long long)g.n[1] * k);
    float w[6];
    face_coeffs(g, L, i, j, k, c, w);
    return diag6(w[0], w[1], w[2], w[3], w[4], w[5]);
}

// Canonical child order of the restriction (reading O6: sum over the children): x pairs first,
// then y pairs, then z pairs -- a tree every kernel (generic, tiled, TMA-fed, single-CTA) can
// reproduce, so all paths give identical bits.  r(e, b, a) = residual of child (x+e, y+b, z+a).
template <class F>
__device__ __forceinline__ float restrict_tree(int cx, int cy, int cz, F r) {
    float zs[2] = {0.0f, 0.0f};
    for (int a = 0; a < cz; ++a) {
        float ys[2] = {0.0f, 0.0f};
        for (int b = 0; b < cy; ++b) ys[b] = (cx == 2) ? r(0, b, a) + r(1, b, a) : r(0, b, a);
        zs[a] = (cy == 2) ? ys[0] + ys[1] : ys[0];
    }
    return (cz == 2) ? zs[0] + zs[1] : zs[0];
}

// Deterministic block reduction of one double per thread; result valid in thread 0.
// blockDim.x must be a multiple of 32 and <= 1024.
__device__ __forceinline__ double block_sum(double v) {
    __shared__ double warp_part[32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    __syncthreads();  // protects warp_part across successive calls
    if (lane == 0) warp_part[wid] = v;
    __syncthreads();
    double t = 0.0;
    if (wid == 0) {
        const int nw = (blockDim.x + 31) >> 5;
        t = (lane < nw) ? warp_part[lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
    }
    return t;
}

// ---- control steps of the CG smoother (reading O12; S9b), run by the one thread that has
// just written the sum they depend on.  A is negative semi-definite: r.s and d.q are negative. ------
// after the mean-free start: rho = rho0 = r.d; nothing to do when rho is not < 0
__device__ __forceinline__ void cgs_ctl_begin(DevScalars* sc, double alpha_cap) {
    const double rho = sc->red[RED_RS];
    sc->cgs_alpha_cap = alpha_cap;
    sc->rho_cg = rho;
    sc->cgs_rho0 = rho;
    sc->cgs_frozen = !(rho < 0.0);
    sc->alpha = 0.0;
    sc->beta = 0.0;
}
// after q = A d, red[DQ] = d.q: alpha = rho/(d.q); d.q not < 0 or alpha above the cap ends the
// smoothing (alpha = 0 leaves x and r untouched for the remaining iterations)
__device__ __forceinline__ void cgs_ctl_alpha(DevScalars* sc) {
    const double dq = sc->red[RED_DQ];
    double alpha = 0.0;
    bool stop = sc->cgs_frozen || !(dq < 0.0);
    if (!stop) {
        alpha = sc->rho_cg / dq;
        stop = alpha > sc->cgs_alpha_cap;
    }
    if (stop) {
        sc->cgs_frozen = 1;
        alpha = 0.0;
    }
    sc->alpha = alpha;
}
// after s = r/D, red[RS] = r.s: beta = rho'/rho; freeze once |rho'| <= 1e-8 |rho0|
__device__ __forceinline__ void cgs_ctl_beta(DevScalars* sc) {
    if (sc->cgs_frozen) {
        sc->beta = 0.0;
        return;
    }
    const double rho_new = sc->red[RED_RS];
    sc->beta = rho_new / sc->rho_cg;
    sc->rho_cg = rho_new;
    if (!(fabs(rho_new) > GMG_CGS_FREEZE * fabs(sc->cgs_rho0))) sc->cgs_frozen = 1;
}

// ---- (GMG-)PCG solver (reading O10): the same arrangement --------------------------------------
// after s = M^-1 r and red[RS] = r.s: beta = rho'/rho (0 on the first iteration)
__device__ __forceinline__ void pcg_ctl_beta(DevScalars* sc) {
    const double rho_new = sc->red[RED_RS];
    sc->beta = (sc->iter == 0) ? 0.0 : rho_new / sc->rho_cg;
    sc->rho_cg = rho_new;
}
// after q = A d and red[DQ] = d.q: alpha = rho/(d.q); breakdown if d.q == 0
__device__ __forceinline__ void pcg_ctl_alpha(DevScalars* sc) {
    const double dq = sc->red[RED_DQ];
    if (dq == 0.0) {
        sc->alpha = 0.0;  // the update kernels then leave p and r unchanged
        sc->status = GMG_EBREAKDOWN;
    } else {
        sc->alpha = sc->rho_cg / dq;
    }
}

// Finishes up to two sums: every block deposits its partial(s); the last block adds them in
// index order and writes red[slot0] (and red[slot1]), then runs the control step rb.post, if any.
__device__ __forceinline__ void finish_reduction(double v0, double v1, bool two, ReduceBuf rb,
                                                 int slot0, int slot1) {
    __shared__ bool is_last;
    const double t0 = block_sum(v0);
    const double t1 = two ? block_sum(v1) : 0.0;
    if (threadIdx.x == 0) {
        rb.partials[blockIdx.x] = t0;
        if (two) rb.partials[GMG_REDUCE_MAX_BLOCKS + blockIdx.x] = t1;
        __threadfence();
        const unsigned int ticket = atomicAdd(rb.counter, 1u);
        is_last = (ticket == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    double a0 = 0.0, a1 = 0.0;
    for (unsigned int i = threadIdx.x; i < gridDim.x; i += blockDim.x) {
        a0 += ((volatile double*)rb.partials)[i];
        if (two) a1 += ((volatile double*)rb.partials)[GMG_REDUCE_MAX_BLOCKS + i];
    }
    const double s0 = block_sum(a0);
    const double s1 = two ? block_sum(a1) : 0.0;
    if (threadIdx.x == 0) {
        rb.sc->red[slot0] = s0;
        if (two) rb.sc->red[slot1] = s1;
        *rb.counter = 0u;
        if (rb.post == POST_CGS_BEGIN) cgs_ctl_begin(rb.sc, rb.post_arg);
        else if (rb.post == POST_CGS_ALPHA) cgs_ctl_alpha(rb.sc);
        else if (rb.post == POST_CGS_BETA) cgs_ctl_beta(rb.sc);
        else if (rb.post == POST_PCG_ALPHA) pcg_ctl_alpha(rb.sc);
        else if (rb.post == POST_PCG_BETA) pcg_ctl_beta(rb.sc);
    }
}

}  // namespace gmgd

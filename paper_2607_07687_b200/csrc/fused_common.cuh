// fused_common.cuh -- small device helpers shared by the tiled fast-path kernels.
#pragma once
#include "stencil.cuh"

namespace gmgf {
using namespace gmgd;

__device__ __forceinline__ int wrapi(int v, int n) {
    v %= n;
    return v < 0 ? v + n : v;
}
// wrap for v in [-n, 2n)
__device__ __forceinline__ int wrap1(int v, int n) { return v < 0 ? v + n : (v >= n ? v - n : v); }

__device__ __forceinline__ float4 ldg4(const float* p) {
    return __ldg(reinterpret_cast<const float4*>(p));
}
__device__ __forceinline__ float4 lds4(const float* p) { return *reinterpret_cast<const float4*>(p); }
__device__ __forceinline__ float4 zero4() { return make_float4(0.f, 0.f, 0.f, 0.f); }
__device__ __forceinline__ void prefetch_l2(const void* p) {
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}
__device__ __forceinline__ void cta_sync() { asm volatile("bar.sync 0;" ::: "memory"); }

// Coefficients of the four own cells in one plane: lower x faces (+ the face above the 4th
// cell), lower / upper y faces, UPPER z faces (the lower z faces are the previous plane's
// upper ones), and the right-hand side.
struct CSet {
    float4 lx, ly, lyh, lzh, b;
    float lxh;
};

// Updates cells S and S+2 of the own group (S = 0 or 1, compile time).
template <int S>
__device__ __forceinline__ float4 update_pair(float xm, float4 own, float xp, float4 ym, float4 yp,
                                              float4 zm, float4 zp, const CSet& c, float4 lz,
                                              float omega) {
    float4 out = own;
    if (S == 0) {
        const float a1 = apply7(own.x, c.lx.x, c.lx.y, c.ly.x, c.lyh.x, lz.x, c.lzh.x, xm, own.y, ym.x, yp.x, zm.x, zp.x);
        const float a2 = apply7(own.z, c.lx.z, c.lx.w, c.ly.z, c.lyh.z, lz.z, c.lzh.z, own.y, own.w, ym.z, yp.z, zm.z, zp.z);
        out.x = relax(own.x, c.b.x, a1, diag6(c.lx.x, c.lx.y, c.ly.x, c.lyh.x, lz.x, c.lzh.x), omega);
        out.z = relax(own.z, c.b.z, a2, diag6(c.lx.z, c.lx.w, c.ly.z, c.lyh.z, lz.z, c.lzh.z), omega);
    } else {
        const float a1 = apply7(own.y, c.lx.y, c.lx.z, c.ly.y, c.lyh.y, lz.y, c.lzh.y, own.x, own.z, ym.y, yp.y, zm.y, zp.y);
        const float a2 = apply7(own.w, c.lx.w, c.lxh, c.ly.w, c.lyh.w, lz.w, c.lzh.w, own.z, xp, ym.w, yp.w, zm.w, zp.w);
        out.y = relax(own.y, c.b.y, a1, diag6(c.lx.y, c.lx.z, c.ly.y, c.lyh.y, lz.y, c.lzh.y), omega);
        out.w = relax(own.w, c.b.w, a2, diag6(c.lx.w, c.lxh, c.ly.w, c.lyh.w, lz.w, c.lzh.w), omega);
    }
    return out;
}

}  // namespace gmgf

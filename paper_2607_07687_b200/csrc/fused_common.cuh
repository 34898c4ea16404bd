// fused_common.cuh -- small device helpers shared by the tiled fast-path kernels.
#pragma once
#include <cuda.h>

#include "stencil.cuh"

namespace gmgf {
using namespace gmgd;

// Planes per CTA of a z-marching kernel.  Big levels: `zpref` planes (the redundant halo planes
// cost little and many CTAs smooth the tail of the grid).  Small, L2-resident levels are
// latency-bound: the kernel takes (waves of CTAs) x (planes per CTA + fixed start-up steps), so
// the chunk count is chosen to minimise that -- in particular never a few CTAs over a wave.
static constexpr int kZChunkPref = 64;  // planes per CTA on big levels
static constexpr int kZChunkMin = 4;    // never fewer planes per CTA than this
static inline int choose_zchunk(long long tiles, int nz, int zpref, int zmin, int slots, int even) {
    if (nz <= zmin) return nz;
    if (tiles * ((nz + zpref - 1) / zpref) >= 4LL * slots) return zpref;
    const int overhead = 5;  // prologue + drain, in steps
    long long best_t = -1;
    int best = nz;
    for (int nchunks = 1; nchunks <= nz / zmin; ++nchunks) {
        int zc = (nz + nchunks - 1) / nchunks;
        if (even && (zc & 1)) ++zc;
        if (zc > zpref * 4) continue;
        const long long ctas = tiles * ((nz + zc - 1) / zc);
        const long long waves = (ctas + slots - 1) / slots;
        const long long t = waves * (zc + overhead);
        if (best_t < 0 || t < best_t) { best_t = t; best = zc; }
    }
    return best;
}

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

// ---- bulk asynchronous copies (TMA) and mbarriers, raw PTX ---------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {
    }
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_g2s(float* dst_smem, const float* src_gmem, uint32_t bytes,
                                         uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
            smem_u32(dst_smem)),
        "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}
__device__ __forceinline__ void fence_async_smem() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

__device__ __forceinline__ void tma_load_3d(float* dst_smem, const CUtensorMap* tm, int c0, int c1, int c2,
                                            uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(
            smem_u32(dst_smem)),
        "l"(reinterpret_cast<uint64_t>(tm)), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}

}  // namespace gmgf

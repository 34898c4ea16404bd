// kernels_setup.cu -- the streaming passes either side of the solve, four x-adjacent cells
// (one float4) per thread:
//   * coefficient hierarchy (reading O5): one pass over a level's
//     three face-coefficient arrays validates every value (finest level only) and writes the next
//     level's coefficients -- 12 B read + 12/m B written per fine cell, m = children per parent;
//   * divergence of a staggered velocity field and the projection u -= L grad p (S8(f) N1;
//     PAPER.md:33-37, 51) -- 16 and 40 B per cell.
// Same per-value arithmetic and summation order as the one-thread-per-value kernels in
// kernels_generic.cu, so the two paths are bit-identical (tests compare them).
#include "stencil.cuh"
#include "uniform.cuh"

namespace gmgk {
using namespace gmgd;

static constexpr int kST = 256;

__device__ __forceinline__ float4 ld4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
__device__ __forceinline__ float get4(const float4& v, int m) {
    return m == 0 ? v.x : m == 1 ? v.y : m == 2 ? v.z : v.w;
}
__device__ __forceinline__ int bad4(const float4& v) {
    return (int)(!(v.x >= 0.0f) || isinf(v.x)) + (int)(!(v.y >= 0.0f) || isinf(v.y)) +
           (int)(!(v.z >= 0.0f) || isinf(v.z)) + (int)(!(v.w >= 0.0f) || isinf(v.w));
}

// One work item = four x-adjacent coarse cells (J, K fixed) = a 4CX x CY x CZ brick of fine cells.
// f[d][a][b][e]: float4 number e of fine row (y = CY*J + b, z = CZ*K + a) of array d.
// uni.brick != nullptr: the pass also CLEARS the uniform-brick flag (uniform.cuh; preset to 1) of
// the brick its fine values lie in as soon as one of them differs from the level's constant.
template <int CX, int CY, int CZ, bool CHECK>
__global__ void __launch_bounds__(kST)
k_coarsen4(LevelGeom gf, const float* __restrict__ Lf, float* __restrict__ Lc, ReduceBuf rb, gmgf::UniArgs uni) {
    const int ncx = gf.n[0] / CX, ncy = gf.n[1] / CY, ncz = gf.n[2] / CZ;
    const int gpr = ncx / 4;  // groups per coarse row
    const long long items = (long long)gpr * ncy * ncz;
    const long long Nc = (long long)ncx * ncy * ncz;
    const long long Nf = gf.N;
    const int nx = gf.n[0];
    const long long fsz = (long long)nx * gf.n[1];
    int bad = 0;
    for (long long t = (long long)blockIdx.x * kST + threadIdx.x; t < items; t += (long long)gridDim.x * kST) {
        const long long row = t / gpr;
        const int Ig = (int)(t - row * gpr);
        const int K = (int)(row / ncy);
        const int J = (int)(row - (long long)K * ncy);
        const long long fbase = (long long)(4 * CX * Ig) + (long long)nx * (CY * J) + fsz * (CZ * K);
        const long long cbase = (long long)(4 * Ig) + (long long)ncx * (J + (long long)ncy * K);
        bool differs = false;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const float ud = d == 0 ? uni.ux : d == 1 ? uni.uy : uni.uz;
            float4 f[CZ][CY][CX];
#pragma unroll
            for (int a = 0; a < CZ; ++a)
#pragma unroll
                for (int b = 0; b < CY; ++b)
#pragma unroll
                    for (int e = 0; e < CX; ++e) {
                        f[a][b][e] = ld4(Lf + d * Nf + fbase + a * fsz + (long long)b * nx + 4 * e);
                        if (CHECK) bad += bad4(f[a][b][e]);
                        differs = differs || f[a][b][e].x != ud || f[a][b][e].y != ud || f[a][b][e].z != ud ||
                                  f[a][b][e].w != ud;
                    }
            // fine value at (x = CX*(4 Ig + m) + ex, y = CY*J + b, z = CZ*K + a)
            auto at = [&](int m, int ex, int b, int a) -> float {
                const int xi = CX * m + ex;
                return get4(f[a][b][xi >> 2], xi & 3);
            };
            float o[4];
#pragma unroll
            for (int m = 0; m < 4; ++m) {
                float s = 0.0f;
                if (d == 0) {  // faces x = CX*I: sum over y (outer), z (inner)
#pragma unroll
                    for (int b = 0; b < CY; ++b)
#pragma unroll
                        for (int a = 0; a < CZ; ++a) s += at(m, 0, b, a);
                    if (gf.bc[0] && Ig == 0 && m == 0) s = 0.0f;
                    if (CX == 2) s *= 0.5f;
                } else if (d == 1) {  // faces y = CY*J: sum over z (outer), x (inner)
#pragma unroll
                    for (int a = 0; a < CZ; ++a)
#pragma unroll
                        for (int ex = 0; ex < CX; ++ex) s += at(m, ex, 0, a);
                    if (gf.bc[1] && J == 0) s = 0.0f;
                    if (CY == 2) s *= 0.5f;
                } else {  // faces z = CZ*K: sum over x (outer), y (inner)
#pragma unroll
                    for (int ex = 0; ex < CX; ++ex)
#pragma unroll
                        for (int b = 0; b < CY; ++b) s += at(m, ex, b, 0);
                    if (gf.bc[2] && K == 0) s = 0.0f;
                    if (CZ == 2) s *= 0.5f;
                }
                o[m] = s;
            }
            *reinterpret_cast<float4*>(Lc + d * Nc + cbase) = make_float4(o[0], o[1], o[2], o[3]);
        }
        if (uni.brick && differs) {
            // the 4CX x CY x CZ fine cells of this work item lie in ONE brick (4CX | kUBX, CY | kUBY, CZ | kUBZ)
            using namespace gmgf;
            const int bx = (4 * CX * Ig) / kUBX, by = (CY * J) / kUBY, bz = (CZ * K) / kUBZ;
            const_cast<unsigned char*>(uni.brick)[((size_t)bz * ub_count(gf.n[1], kUBY) + by) * ub_count(nx, kUBX) + bx] = 0;
        }
    }
    if (CHECK) finish_reduction((double)bad, 0.0, false, rb, RED_CHECK, 0);
}

bool coarsen4_supported(const LevelGeom& gf) {
    const int cx = gf.c[0], cy = gf.c[1], cz = gf.c[2];
    if (cx * cy * cz == 1) return false;
    return gf.n[0] % (4 * cx) == 0;
}

template <int CX, int CY, int CZ>
static void coarsen4_launch(const LevelGeom& gf, const float* Lf, float* Lc, bool check, ReduceBuf rb,
                            const gmgf::UniArgs& uni, cudaStream_t s) {
    const long long items = gf.N / ((long long)CX * CY * CZ) / 4;
    long long blocks = (items + kST - 1) / kST;
    if (blocks > 148 * 16) blocks = 148 * 16;
    if (blocks < 1) blocks = 1;
    if (check) k_coarsen4<CX, CY, CZ, true><<<(unsigned int)blocks, kST, 0, s>>>(gf, Lf, Lc, rb, uni);
    else k_coarsen4<CX, CY, CZ, false><<<(unsigned int)blocks, kST, 0, s>>>(gf, Lf, Lc, rb, uni);
}

// Next level's coefficients from this level's; check = also count invalid values into
// red[RED_CHECK] (replaces check_coeffs on the finest level).
void coarsen_coeffs4(const LevelGeom& gf, const float* Lf, float* Lc, bool check, ReduceBuf rb,
                     const gmgf::UniArgs& uni, cudaStream_t s) {
    const int key = (gf.c[0] - 1) | ((gf.c[1] - 1) << 1) | ((gf.c[2] - 1) << 2);
    switch (key) {
        case 1: coarsen4_launch<2, 1, 1>(gf, Lf, Lc, check, rb, uni, s); break;
        case 2: coarsen4_launch<1, 2, 1>(gf, Lf, Lc, check, rb, uni, s); break;
        case 3: coarsen4_launch<2, 2, 1>(gf, Lf, Lc, check, rb, uni, s); break;
        case 4: coarsen4_launch<1, 1, 2>(gf, Lf, Lc, check, rb, uni, s); break;
        case 5: coarsen4_launch<2, 1, 2>(gf, Lf, Lc, check, rb, uni, s); break;
        case 6: coarsen4_launch<1, 2, 2>(gf, Lf, Lc, check, rb, uni, s); break;
        default: coarsen4_launch<2, 2, 2>(gf, Lf, Lc, check, rb, uni, s); break;
    }
}

// ---- N1: z = div u on lower-face velocities (same arithmetic as k_divergence) --
__global__ void __launch_bounds__(kST)
k_divergence4(LevelGeom g, const float* __restrict__ u, float whx, float why, float whz,
              float* __restrict__ z) {
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const int gpr = nx >> 2;
    const long long items = g.N >> 2;
    const long long t = (long long)blockIdx.x * kST + threadIdx.x;
    if (t >= items) return;
    const long long row = t / gpr;
    const int i = 4 * (int)(t - row * gpr);
    const int k = (int)(row / ny);
    const int j = (int)(row - (long long)k * ny);
    const long long N = g.N, sy = nx, sz = (long long)nx * ny;
    const long long c = 4 * t;
    const float4 ux = ld4(u + c), uy = ld4(u + N + c), uz = ld4(u + 2 * N + c);
    float x4;  // the x face above the group's last cell
    if (i + 4 == nx) x4 = g.bc[0] ? whx : __ldg(u + c - (nx - 4));
    else x4 = __ldg(u + c + 4);
    float4 yh, zh;
    if (j == ny - 1) yh = g.bc[1] ? make_float4(why, why, why, why) : ld4(u + N + c - sy * (ny - 1));
    else yh = ld4(u + N + c + sy);
    if (k == nz - 1) zh = g.bc[2] ? make_float4(whz, whz, whz, whz) : ld4(u + 2 * N + c - sz * (nz - 1));
    else zh = ld4(u + 2 * N + c + sz);
    float4 o;
    o.x = ux.y - ux.x; o.x += yh.x - uy.x; o.x += zh.x - uz.x;
    o.y = ux.z - ux.y; o.y += yh.y - uy.y; o.y += zh.y - uz.y;
    o.z = ux.w - ux.z; o.z += yh.z - uy.z; o.z += zh.z - uz.z;
    o.w = x4 - ux.w;   o.w += yh.w - uy.w; o.w += zh.w - uz.w;
    *reinterpret_cast<float4*>(z + c) = o;
}

void divergence4(const LevelGeom& g, const float* u, const float wall_hi[3], float* z, cudaStream_t s) {
    const long long items = g.N >> 2;
    k_divergence4<<<(unsigned int)((items + kST - 1) / kST), kST, 0, s>>>(g, u, wall_hi[0], wall_hi[1],
                                                                       wall_hi[2], z);
}

// ---- N1: u_d(I) -= L_d(I) (p_I - p_{I-e_d}) (same arithmetic as k_project) --------
__global__ void __launch_bounds__(kST)
k_project4(LevelGeom g, const float* __restrict__ L, const float* __restrict__ p, float* __restrict__ u) {
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const int gpr = nx >> 2;
    const long long items = g.N >> 2;
    const long long t = (long long)blockIdx.x * kST + threadIdx.x;
    if (t >= items) return;
    const long long row = t / gpr;
    const int i = 4 * (int)(t - row * gpr);
    const int k = (int)(row / ny);
    const int j = (int)(row - (long long)k * ny);
    const long long N = g.N, sy = nx, sz = (long long)nx * ny;
    const long long c = 4 * t;
    const float4 pc = ld4(p + c);
    const float pxm = __ldg(p + ((i == 0) ? c + (nx - 1) : c - 1));
    const float4 py = ld4(p + ((j == 0) ? c + sy * (ny - 1) : c - sy));
    const float4 pz = ld4(p + ((k == 0) ? c + sz * (nz - 1) : c - sz));
    float4 wx = ld4(L + c), wy = ld4(L + N + c), wz = ld4(L + 2 * N + c);
    if (i == 0 && g.bc[0]) wx.x = 0.0f;
    if (j == 0 && g.bc[1]) wy = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    if (k == 0 && g.bc[2]) wz = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    float4* ux = reinterpret_cast<float4*>(u + c);
    float4* uy = reinterpret_cast<float4*>(u + N + c);
    float4* uz = reinterpret_cast<float4*>(u + 2 * N + c);
    float4 a = *ux, b = *uy, d = *uz;
    a.x = fmaf(-wx.x, pc.x - pxm, a.x);
    a.y = fmaf(-wx.y, pc.y - pc.x, a.y);
    a.z = fmaf(-wx.z, pc.z - pc.y, a.z);
    a.w = fmaf(-wx.w, pc.w - pc.z, a.w);
    b.x = fmaf(-wy.x, pc.x - py.x, b.x);
    b.y = fmaf(-wy.y, pc.y - py.y, b.y);
    b.z = fmaf(-wy.z, pc.z - py.z, b.z);
    b.w = fmaf(-wy.w, pc.w - py.w, b.w);
    d.x = fmaf(-wz.x, pc.x - pz.x, d.x);
    d.y = fmaf(-wz.y, pc.y - pz.y, d.y);
    d.z = fmaf(-wz.z, pc.z - pz.z, d.z);
    d.w = fmaf(-wz.w, pc.w - pz.w, d.w);
    *ux = a; *uy = b; *uz = d;
}

void project4(const LevelGeom& g, const float* L, const float* p, float* u, cudaStream_t s) {
    const long long items = g.N >> 2;
    k_project4<<<(unsigned int)((items + kST - 1) / kST), kST, 0, s>>>(g, L, p, u);
}

// ---- uniform bricks (uniform.cuh): how many cells of a level are worked on by CTAs that take the
// lean path, for a kernel's tiling (one thread per CTA of that kernel, the kernel's own footprint
// test).  rule 0 = the sweep (box-fed tiles: inside, walls in y, or first / final tile row of a
// periodic y axis), rule 1 = the residual pass (tiles inside the domain in y).  out += cells.
__global__ void __launch_bounds__(128)
k_uniform_cells(LevelGeom g, const unsigned char* __restrict__ brick, int TXc, int TYc, int yhi, int zchunk, int rule,
                unsigned long long* __restrict__ out, int* __restrict__ left_list, unsigned int* __restrict__ left_count) {
    using namespace gmgf;
    const int tiles_x = g.n[0] / TXc, tiles_y = (g.n[1] + TYc - 1) / TYc, nzc = (g.n[2] + zchunk - 1) / zchunk;
    const long long total = (long long)tiles_x * tiles_y * nzc;
    // one WARP per tile: the lanes share the bricks of its footprint (a few hundred byte loads that
    // one thread would issue one after the other: 38 instead of 6 us per pass at 1024^3)
    const int lane = threadIdx.x & 31;
    const long long t = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (t >= total) return;
    const int tx = (int)(t % tiles_x), ty = (int)((t / tiles_x) % tiles_y), zc = (int)(t / ((long long)tiles_x * tiles_y));
    const int x0 = tx * TXc, y0 = ty * TYc, z0 = zc * zchunk, z1 = min(g.n[2], z0 + zchunk), ny = g.n[1];
    bool boxfed;
    if (rule == 0) {
        const bool inside = (y0 >= 2) && (y0 + TYc + 2 <= ny);
        boxfed = g.bc[1] != 0 || inside || (tiles_y >= 2 && ((ty == 0 && TYc + 2 <= ny) || (ty == tiles_y - 1 && y0 >= 2)));
    } else {
        boxfed = (y0 >= 1) && (y0 + TYc + 1 <= ny);
    }
    if (!boxfed || !ub_box_uniform_warp(g, brick, x0 - 2, x0 + TXc + 1, y0 - 2, y0 + yhi, z0 - 2, z1 + 1, lane)) {
        // not lean: onto the list of remaining tiles (any order: tiles are independent)
        if (left_list && lane == 0) left_list[atomicAdd(left_count, 1u)] = (int)t;
        return;
    }
    const int rows = min(TYc, ny - y0);
    if (lane == 0) atomicAdd(out, (unsigned long long)TXc * rows * (z1 - z0));
}

void uniform_cells(const LevelGeom& g, const unsigned char* brick, int TXc, int TYc, int yhi, int zchunk, int rule,
                   unsigned long long* out, int* left_list, unsigned int* left_count, cudaStream_t s) {
    const int tiles_x = g.n[0] / TXc, tiles_y = (g.n[1] + TYc - 1) / TYc, nzc = (g.n[2] + zchunk - 1) / zchunk;
    const long long total = (long long)tiles_x * tiles_y * nzc;
    k_uniform_cells<<<(unsigned int)((total + 3) / 4), 128, 0, s>>>(g, brick, TXc, TYc, yhi, zchunk, rule, out, left_list, left_count);
}

}  // namespace gmgk

// kernels_residual.cu -- k_residual_bulk: residual fused with the restriction (MODE 0) or with the
// squared-norm reduction (MODE 1, 2), or the CG mat-vec q = A d with d.q (MODE 3), on the big levels, fed by TMA (cp.async.bulk.tensor + mbarrier)
// like the sweep.  r = b - A p on active cells, 0 elsewhere (readings O1, O9);
// restriction = sum over the children (O6; PAPER.md:39 coarse-grid correction, 47 anisotropic
// coarsening: any factor pattern c in {1,2}^3); BASELINE.json:north_star "a residual kernel fused
// with the restriction ... warp-shuffle plus block-level residual-norm ... reductions".
//
// A CTA owns a 128 x 16 tile in (x,y) and marches along a chunk of z planes; 8 warps, a thread owns
// one float4 group in each of two adjacent rows (8 cells per plane).  Every input stream arrives
// in shared memory as one TMA box per plane, PD planes ahead; the only CTA barrier per plane
// protects ring-slot reuse.  The x pair and y pair sums of the restriction happen in registers,
// the z pair across two consecutive steps, in stencil.cuh's canonical tree order, so the result is
// bit-identical to the generic kernel.  112 KB of shared memory per CTA: two CTAs per SM.
#include <type_traits>

#include "fused_common.cuh"
#include "uniform.cuh"

namespace gmgf {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);
extern EncodeTiledFn g_encode;
bool tensor_map(const float* ptr, const LevelGeom& g, int bw, int bh, CUtensorMap* out);
bool bulk_supported(const LevelGeom& g);

// LEAN_: ring layout of the lean path (uniform.cuh) -- no coefficient rings, so the same 112 KB hold a
// deeper pipeline of the two streams that are left (PD = 5 steps of 18 KB in flight instead of 2).
template <int PD_, bool LEAN_>
struct ResBulkCfgT {
    static constexpr int TX = 128, RY = 16, PD = PD_;
    static constexpr bool LEAN = LEAN_;
    static constexpr int THREADS = 32 * RY / 2;   // 256: a thread owns two rows
    static constexpr int PH = RY + 2;             // rows of a p plane (halo 1)
    static constexpr int NP = PD + 2, NZ = PD + 1, NC = PD, NB = PD + 1;
    static constexpr int HPAD = (PH * 4 + 31) / 32 * 32;
    static constexpr int P_HL = PH * TX, P_HR = P_HL + HPAD, P_PLANE = P_HR + HPAD;
    static constexpr int C_PLANE = RY * TX;
    static constexpr int Y_PLANE = (RY + 1) * TX;
    static constexpr int OFF_P = 0;
    static constexpr int OFF_LZ = OFF_P + NP * P_PLANE;
    static constexpr int OFF_LX = OFF_LZ + (LEAN ? 0 : NZ * C_PLANE);
    static constexpr int OFF_LY = OFF_LX + (LEAN ? 0 : NC * C_PLANE);
    static constexpr int OFF_B = OFF_LY + (LEAN ? 0 : NC * Y_PLANE);
    static constexpr int FLOATS = OFF_B + NC * C_PLANE;
    static constexpr size_t SMEM = (size_t)FLOATS * sizeof(float) + 16 * sizeof(uint64_t);
    static_assert(NB + 1 <= 16, "mbarriers");
    static constexpr uint32_t P_BYTES = (uint32_t)(PH * TX + 2 * PH * 4) * 4u;
    static constexpr uint32_t STEP_BYTES = P_BYTES + (uint32_t)(3 * RY * TX + (RY + 1) * TX) * 4u;
    static constexpr uint32_t PRO_BYTES = 2 * P_BYTES + (uint32_t)(RY * TX) * 4u;
    // lean path (uniform.cuh): only the p and b streams are copied
    static constexpr uint32_t STEP_BYTES_UNI = P_BYTES + (uint32_t)(RY * TX) * 4u;
    static constexpr uint32_t PRO_BYTES_UNI = 2 * P_BYTES;
};
using ResBulkCfg = ResBulkCfgT<2, false>;
using ResLeanCfg = ResBulkCfgT<5, true>;
static_assert(ResLeanCfg::SMEM <= ResBulkCfg::SMEM, "the lean rings live in the general kernel's allocation");

struct ResBulkArgs {
    LevelGeom g;
    const float* L;
    const float* p;
    const float* b;
    float* b_c;
    float* p_c;
    ReduceBuf rb;
    int slot, slot2;
    int zchunk;
    int tiles_x, tiles_y;
    const int* run_flag;   // != nullptr: the kernel does nothing unless *run_flag != 0
    UniArgs uni;           // uniform bricks of the level (uniform.cuh); brick == nullptr: disabled
};

struct alignas(64) ResBulkMaps {
    CUtensorMap p_main, p_halo, lz, lx, ly, b;
};

// UNI: the lean path of uniform.cuh (interior tiles in y only) -- the coefficient streams are
// neither copied nor read; the same apply7 / diag6 operations run on the level's constants.
// C222: the level coarsens by two in every direction (compile-time factors: no integer divisions
// in the store of the coarse right-hand side).
template <int MODE, bool UNI, bool C222 = false>
__device__ __forceinline__ void res_body(const ResBulkArgs& a, const ResBulkMaps& maps) {
    using C = typename std::conditional<UNI, ResLeanCfg, ResBulkCfg>::type;
    extern __shared__ __align__(128) float sm[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(sm + C::FLOATS);  // [0..NB) steps, [NB] prologue
    const LevelGeom& g = a.g;
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const size_t N = (size_t)g.N;
    const int plane = nx * ny;
    const int tid = threadIdx.x, warp_id = tid >> 5, lane_id = tid & 31;
    constexpr int NWARP = C::THREADS / 32;
    int bid = blockIdx.x;
    const int tx = bid % a.tiles_x;
    bid /= a.tiles_x;
    const int ty = bid % a.tiles_y;
    const int zc = bid / a.tiles_y;
    const int x0 = tx * C::TX, y0 = ty * C::RY;
    const int z0 = zc * a.zchunk;
    const int z1 = min(nz, z0 + a.zchunk);
    const int xL = wrapi(x0 - 4, nx), xR = wrapi(x0 + C::TX, nx);
    const bool y_inside = UNI || ((y0 >= 1) && (y0 + C::RY + 1 <= ny));   // lean tiles are box-fed by construction
    const float* Lx = a.L;
    const float* Ly = a.L + N;
    const float* Lz = a.L + 2 * N;

    auto slotP = [&](int v) -> float* { return sm + C::OFF_P + ((v - (z0 - 1)) % C::NP) * C::P_PLANE; };
    auto slotLz = [&](int v) -> float* { return sm + C::OFF_LZ + ((v - z0) % C::NZ) * C::C_PLANE; };
    auto slotLx = [&](int v) -> float* { return sm + C::OFF_LX + ((v - z0) % C::NC) * C::C_PLANE; };
    auto slotLy = [&](int v) -> float* { return sm + C::OFF_LY + ((v - z0) % C::NC) * C::Y_PLANE; };
    auto slotB = [&](int v) -> float* { return sm + C::OFF_B + ((v - z0) % C::NC) * C::C_PLANE; };

    // ---- copy issue (lane 0 of the warps).  Interior tiles: 7 TMA boxes.  Tiles touching the y
    // boundary: row-by-row bulk copies with wrapped row addresses. ------------------------------
    auto rows_p = [&](int v, uint64_t* bar) {
        float* d = slotP(v);
        const float* src = a.p + (size_t)wrap1(v, nz) * plane;
        for (int j = warp_id; j < C::PH; j += NWARP) {
            const float* rb = src + (size_t)wrapi(y0 - 1 + j, ny) * nx;
            bulk_g2s(d + j * C::TX, rb + x0, C::TX * 4u, bar);
            bulk_g2s(d + C::P_HL + j * 4, rb + xL, 16u, bar);
            bulk_g2s(d + C::P_HR + j * 4, rb + xR, 16u, bar);
        }
    };
    auto rows_c = [&](float* d, const float* src, int cnt, uint64_t* bar) {
        for (int j = warp_id; j < cnt; j += NWARP)
            bulk_g2s(d + j * C::TX, src + (size_t)wrapi(y0 + j, ny) * nx + x0, C::TX * 4u, bar);
    };
    auto issue_step = [&](int v) {  // p(v+1), Lz(v+1), Lx(v), Ly(v), b(v)
        if (lane_id != 0 || (y_inside && warp_id >= 7)) return;
        uint64_t* bar = bars + ((v - z0) % C::NB);
        if (tid == 0) mbar_expect_tx(bar, UNI ? C::STEP_BYTES_UNI : C::STEP_BYTES);
        const int gz0 = wrap1(v, nz), gz1 = wrap1(v + 1, nz);
        if (y_inside) {
            switch (warp_id) {
                case 0: tma_load_3d(slotP(v + 1), &maps.p_main, x0, y0 - 1, gz1, bar); break;
                case 1: tma_load_3d(slotP(v + 1) + C::P_HL, &maps.p_halo, xL, y0 - 1, gz1, bar); break;
                case 2: tma_load_3d(slotP(v + 1) + C::P_HR, &maps.p_halo, xR, y0 - 1, gz1, bar); break;
                case 3: if (!UNI) tma_load_3d(slotLz(v + 1), &maps.lz, x0, y0, gz1, bar); break;
                case 4: if (!UNI) tma_load_3d(slotLx(v), &maps.lx, x0, y0, gz0, bar); break;
                case 5: if (!UNI) tma_load_3d(slotLy(v), &maps.ly, x0, y0, gz0, bar); break;
                case 6: tma_load_3d(slotB(v), &maps.b, x0, y0, gz0, bar); break;
                default: break;
            }
        } else {
            rows_p(v + 1, bar);
            rows_c(slotLz(v + 1), Lz + (size_t)gz1 * plane, C::RY, bar);
            rows_c(slotLx(v), Lx + (size_t)gz0 * plane, C::RY, bar);
            rows_c(slotLy(v), Ly + (size_t)gz0 * plane, C::RY + 1, bar);
            rows_c(slotB(v), a.b + (size_t)gz0 * plane, C::RY, bar);
        }
    };

    // ---- prologue: p(z0-1), p(z0), Lz(z0); the first PD step groups ----------------------------
    if (tid == 0) {
        for (int i = 0; i <= C::NB; ++i) mbar_init(bars + i, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    fence_async_smem();
    __syncthreads();
    {
        uint64_t* bar = bars + C::NB;
        if (lane_id == 0) {
            if (tid == 0) mbar_expect_tx(bar, UNI ? C::PRO_BYTES_UNI : C::PRO_BYTES);
            const int ga = wrap1(z0 - 1, nz), gb = wrap1(z0, nz);
            if (y_inside) {
                switch (warp_id) {
                    case 0: tma_load_3d(slotP(z0 - 1), &maps.p_main, x0, y0 - 1, ga, bar); break;
                    case 1: tma_load_3d(slotP(z0 - 1) + C::P_HL, &maps.p_halo, xL, y0 - 1, ga, bar); break;
                    case 2: tma_load_3d(slotP(z0 - 1) + C::P_HR, &maps.p_halo, xR, y0 - 1, ga, bar); break;
                    case 3: tma_load_3d(slotP(z0), &maps.p_main, x0, y0 - 1, gb, bar); break;
                    case 4: tma_load_3d(slotP(z0) + C::P_HL, &maps.p_halo, xL, y0 - 1, gb, bar); break;
                    case 5: tma_load_3d(slotP(z0) + C::P_HR, &maps.p_halo, xR, y0 - 1, gb, bar); break;
                    case 6: if (!UNI) tma_load_3d(slotLz(z0), &maps.lz, x0, y0, gb, bar); break;
                    default: break;
                }
            } else {
                rows_p(z0 - 1, bar);
                rows_p(z0, bar);
                rows_c(slotLz(z0), Lz + (size_t)gb * plane, C::RY, bar);
            }
        }
        for (int v = z0; v < z0 + C::PD && v < z1; ++v) issue_step(v);
        mbar_wait(bar, 0);
    }

    // ---- per-thread constants --------------------------------------------------------------------
    const int lx = lane_id;
    const int rA = 2 * warp_id;                     // tile row of the lower own row
    const int xl = x0 + 4 * lx;
    const int yA = y0 + rA, yB = yA + 1;
    const bool vA = yA < ny, vB = yB < ny;
    const int gyA = wrapi(yA, ny), gyB = wrapi(yB, ny), gyC = wrapi(yB + 1, ny);
    const int gxh = wrapi(xl + 4, nx);
    const bool zx_lo = g.bc[0] && xl == 0, zx_hi = g.bc[0] && gxh == 0;
    const bool zyA = g.bc[1] && gyA == 0, zyB = g.bc[1] && gyB == 0, zyC = g.bc[1] && gyC == 0;
    const bool any_wall = !UNI && (zx_lo || zx_hi || zyA || zyB || zyC || g.bc[2]);
    const bool last_lane = (lx == 31);
    const int p_off = (rA + 1) * C::TX + 4 * lx;    // row A in a p plane (row B: +TX)
    const int h_off = (lx == 0 ? C::P_HL + 3 : C::P_HR) + (rA + 1) * 4;
    const int c_off = rA * C::TX + 4 * lx;
    const float* const lxhA_row = Lx + (size_t)gyA * nx + gxh;
    const float* const lxhB_row = Lx + (size_t)gyB * nx + gxh;
    const int cx = C222 ? 2 : g.c[0], cy = C222 ? 2 : g.c[1], cz = C222 ? 2 : g.c[2];
    const int ncx = nx / cx, ncy = ny / cy;

    // ring cursors
    float* const P_beg = sm + C::OFF_P;
    float* const Z_beg = sm + C::OFF_LZ;
    const float* Pm = P_beg;                        // plane v-1
    const float* P0 = P_beg + C::P_PLANE;           // plane v
    const float* Pp = P_beg + 2 * C::P_PLANE;       // plane v+1
    const float* Z0 = Z_beg;                        // Lz plane v
    const float* Z1 = Z_beg + C::C_PLANE;           // Lz plane v+1
    int ic = 0, kb = 0;
    uint32_t kpar = 0;
    int gz = z0;
    float lxhA_pf = 0.0f, lxhB_pf = 0.0f;
    if (!UNI && last_lane) {
        lxhA_pf = __ldg(lxhA_row + (size_t)gz * plane);
        lxhB_pf = __ldg(lxhB_row + (size_t)gz * plane);
    }
    const float4 ux4 = make_float4(a.uni.ux, a.uni.ux, a.uni.ux, a.uni.ux);
    const float4 uy4 = make_float4(a.uni.uy, a.uni.uy, a.uni.uy, a.uni.uy);
    const float4 uz4 = make_float4(a.uni.uz, a.uni.uz, a.uni.uz, a.uni.uz);
    double acc = 0.0, acc_b = 0.0;                  // MODE 1, 2: sum r^2 (and sum b^2 over active cells)
    float zacc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};  // MODE 0: even-plane partial sums

    auto store_coarse = [&](const float* v, int cyi, int czi) {  // one coarse row segment of this thread
        const size_t o = ((size_t)czi * ncy + cyi) * ncx + xl / cx;
        if (cx == 2) {
            *reinterpret_cast<float2*>(a.b_c + o) = make_float2(v[0], v[1]);
            if (a.p_c) *reinterpret_cast<float2*>(a.p_c + o) = make_float2(0.f, 0.f);
        } else {
            *reinterpret_cast<float4*>(a.b_c + o) = make_float4(v[0], v[1], v[2], v[3]);
            if (a.p_c) *reinterpret_cast<float4*>(a.p_c + o) = zero4();
        }
    };

    for (int v = z0; v < z1; ++v) {
        mbar_wait(bars + kb, kpar);
        const int gzp = (gz + 1 == nz) ? 0 : gz + 1;
        // ---- coefficients and p of both rows: shared memory -> registers -------------------------
        const float* X = sm + C::OFF_LX + ic * C::C_PLANE + c_off;
        const float* Y = sm + C::OFF_LY + ic * C::Y_PLANE + c_off;
        const float* Bq = sm + C::OFF_B + ic * C::C_PLANE + c_off;
        float4 lxA, lxB, lyA, lyB, lyC, lzA, lzB, lzhA, lzhB;
        float lxhA, lxhB;
        if (UNI) {
            lxA = lxB = ux4; lyA = lyB = lyC = uy4; lzA = lzB = lzhA = lzhB = uz4;
            lxhA = lxhB = a.uni.ux;
        } else {
            lxA = lds4(X); lxB = lds4(X + C::TX);
            lyA = lds4(Y); lyB = lds4(Y + C::TX); lyC = lds4(Y + 2 * C::TX);
            lzA = lds4(Z0 + c_off); lzB = lds4(Z0 + c_off + C::TX);
            lzhA = lds4(Z1 + c_off); lzhB = lds4(Z1 + c_off + C::TX);
            const float tA = __shfl_down_sync(0xffffffffu, lxA.x, 1);
            const float tB = __shfl_down_sync(0xffffffffu, lxB.x, 1);
            lxhA = last_lane ? lxhA_pf : tA;
            lxhB = last_lane ? lxhB_pf : tB;
            if (last_lane && v + 1 < z1) {
                lxhA_pf = __ldg(lxhA_row + (size_t)gzp * plane);
                lxhB_pf = __ldg(lxhB_row + (size_t)gzp * plane);
            }
        }
        const float4 bA = lds4(Bq), bB = lds4(Bq + C::TX);
        if (any_wall) {
            if (zx_lo) { lxA.x = 0.0f; lxB.x = 0.0f; }
            if (zx_hi) { lxhA = 0.0f; lxhB = 0.0f; }
            if (zyA) lyA = zero4();
            if (zyB) lyB = zero4();
            if (zyC) lyC = zero4();
            if (g.bc[2]) {
                if (gz == 0) { lzA = zero4(); lzB = zero4(); }
                if (gzp == 0) { lzhA = zero4(); lzhB = zero4(); }
            }
        }
        const float4 ym = lds4(P0 + p_off - C::TX);
        const float4 oA = lds4(P0 + p_off);
        const float4 oB = lds4(P0 + p_off + C::TX);
        const float4 yp = lds4(P0 + p_off + 2 * C::TX);
        const float4 zmA = lds4(Pm + p_off), zmB = lds4(Pm + p_off + C::TX);
        const float4 zpA = lds4(Pp + p_off), zpB = lds4(Pp + p_off + C::TX);
        float xmA = __shfl_up_sync(0xffffffffu, oA.w, 1);
        float xpA = __shfl_down_sync(0xffffffffu, oA.x, 1);
        float xmB = __shfl_up_sync(0xffffffffu, oB.w, 1);
        float xpB = __shfl_down_sync(0xffffffffu, oB.x, 1);
        if (lx == 0) { xmA = P0[h_off]; xmB = P0[h_off + 4]; }
        if (last_lane) { xpA = P0[h_off]; xpB = P0[h_off + 4]; }
        // ---- residuals of the 8 own cells (apply7 / diag6: the shared arithmetic) -----------------
        float rA[4], rB[4];
        {
            const float A0 = apply7(oA.x, lxA.x, lxA.y, lyA.x, lyB.x, lzA.x, lzhA.x, xmA, oA.y, ym.x, oB.x, zmA.x, zpA.x);
            const float A1 = apply7(oA.y, lxA.y, lxA.z, lyA.y, lyB.y, lzA.y, lzhA.y, oA.x, oA.z, ym.y, oB.y, zmA.y, zpA.y);
            const float A2 = apply7(oA.z, lxA.z, lxA.w, lyA.z, lyB.z, lzA.z, lzhA.z, oA.y, oA.w, ym.z, oB.z, zmA.z, zpA.z);
            const float A3 = apply7(oA.w, lxA.w, lxhA, lyA.w, lyB.w, lzA.w, lzhA.w, oA.z, xpA, ym.w, oB.w, zmA.w, zpA.w);
            if (MODE == 3) {  // mat-vec: q = A d on every cell (inactive rows are all-zero), d.q
                if (vA) {
                    *reinterpret_cast<float4*>(a.b_c + (size_t)gz * plane + (size_t)gyA * nx + xl) = make_float4(A0, A1, A2, A3);
                    acc += ((double)oA.x * A0 + (double)oA.y * A1) + ((double)oA.z * A2 + (double)oA.w * A3);
                }
            }
            rA[0] = (diag6(lxA.x, lxA.y, lyA.x, lyB.x, lzA.x, lzhA.x) != 0.0f) ? bA.x - A0 : 0.0f;
            rA[1] = (diag6(lxA.y, lxA.z, lyA.y, lyB.y, lzA.y, lzhA.y) != 0.0f) ? bA.y - A1 : 0.0f;
            rA[2] = (diag6(lxA.z, lxA.w, lyA.z, lyB.z, lzA.z, lzhA.z) != 0.0f) ? bA.z - A2 : 0.0f;
            rA[3] = (diag6(lxA.w, lxhA, lyA.w, lyB.w, lzA.w, lzhA.w) != 0.0f) ? bA.w - A3 : 0.0f;
            const float B0 = apply7(oB.x, lxB.x, lxB.y, lyB.x, lyC.x, lzB.x, lzhB.x, xmB, oB.y, oA.x, yp.x, zmB.x, zpB.x);
            const float B1 = apply7(oB.y, lxB.y, lxB.z, lyB.y, lyC.y, lzB.y, lzhB.y, oB.x, oB.z, oA.y, yp.y, zmB.y, zpB.y);
            const float B2 = apply7(oB.z, lxB.z, lxB.w, lyB.z, lyC.z, lzB.z, lzhB.z, oB.y, oB.w, oA.z, yp.z, zmB.z, zpB.z);
            const float B3 = apply7(oB.w, lxB.w, lxhB, lyB.w, lyC.w, lzB.w, lzhB.w, oB.z, xpB, oA.w, yp.w, zmB.w, zpB.w);
            if (MODE == 3) {
                if (vB) {
                    *reinterpret_cast<float4*>(a.b_c + (size_t)gz * plane + (size_t)gyB * nx + xl) = make_float4(B0, B1, B2, B3);
                    acc += ((double)oB.x * B0 + (double)oB.y * B1) + ((double)oB.z * B2 + (double)oB.w * B3);
                }
            }
            rB[0] = (diag6(lxB.x, lxB.y, lyB.x, lyC.x, lzB.x, lzhB.x) != 0.0f) ? bB.x - B0 : 0.0f;
            rB[1] = (diag6(lxB.y, lxB.z, lyB.y, lyC.y, lzB.y, lzhB.y) != 0.0f) ? bB.y - B1 : 0.0f;
            rB[2] = (diag6(lxB.z, lxB.w, lyB.z, lyC.z, lzB.z, lzhB.z) != 0.0f) ? bB.z - B2 : 0.0f;
            rB[3] = (diag6(lxB.w, lxhB, lyB.w, lyC.w, lzB.w, lzhB.w) != 0.0f) ? bB.w - B3 : 0.0f;
        }
        if (MODE == 3) {
            // stored above; rA / rB are unused (dead code)
        } else if (MODE >= 1) {
            if (vA) acc += ((double)rA[0] * rA[0] + (double)rA[1] * rA[1]) + ((double)rA[2] * rA[2] + (double)rA[3] * rA[3]);
            if (vB) acc += ((double)rB[0] * rB[0] + (double)rB[1] * rB[1]) + ((double)rB[2] * rB[2] + (double)rB[3] * rB[3]);
            if (MODE == 2) {  // reference norm of the solve loop: b^2 over ACTIVE cells (reading O9)
                const float a0 = (diag6(lxA.x, lxA.y, lyA.x, lyB.x, lzA.x, lzhA.x) != 0.0f) ? bA.x : 0.0f;
                const float a1 = (diag6(lxA.y, lxA.z, lyA.y, lyB.y, lzA.y, lzhA.y) != 0.0f) ? bA.y : 0.0f;
                const float a2 = (diag6(lxA.z, lxA.w, lyA.z, lyB.z, lzA.z, lzhA.z) != 0.0f) ? bA.z : 0.0f;
                const float a3 = (diag6(lxA.w, lxhA, lyA.w, lyB.w, lzA.w, lzhA.w) != 0.0f) ? bA.w : 0.0f;
                const float b0 = (diag6(lxB.x, lxB.y, lyB.x, lyC.x, lzB.x, lzhB.x) != 0.0f) ? bB.x : 0.0f;
                const float b1 = (diag6(lxB.y, lxB.z, lyB.y, lyC.y, lzB.y, lzhB.y) != 0.0f) ? bB.y : 0.0f;
                const float b2 = (diag6(lxB.z, lxB.w, lyB.z, lyC.z, lzB.z, lzhB.z) != 0.0f) ? bB.z : 0.0f;
                const float b3 = (diag6(lxB.w, lxhB, lyB.w, lyC.w, lzB.w, lzhB.w) != 0.0f) ? bB.w : 0.0f;
                if (vA) acc_b += ((double)a0 * a0 + (double)a1 * a1) + ((double)a2 * a2 + (double)a3 * a3);
                if (vB) acc_b += ((double)b0 * b0 + (double)b1 * b1) + ((double)b2 * b2 + (double)b3 * b3);
            }
        } else {
            // x pairs, then y pairs, then z pairs (stencil.cuh restrict_tree order)
            float cur[8];
            const int nv = (cx == 2) ? 2 : 4;
            if (cx == 2) {
                cur[0] = rA[0] + rA[1]; cur[1] = rA[2] + rA[3];
                cur[4] = rB[0] + rB[1]; cur[5] = rB[2] + rB[3];
            } else {
#pragma unroll
                for (int i = 0; i < 4; ++i) { cur[i] = rA[i]; cur[4 + i] = rB[i]; }
            }
            if (cy == 2) {
#pragma unroll
                for (int i = 0; i < 4; ++i) cur[i] = cur[i] + cur[4 + i];
            }
            bool emit = true;
            if (cz == 2) {
                if ((gz & 1) == 0) {
#pragma unroll
                    for (int i = 0; i < 8; ++i) zacc[i] = cur[i];
                    emit = false;
                } else {
#pragma unroll
                    for (int i = 0; i < 8; ++i) cur[i] = zacc[i] + cur[i];
                }
            }
            if (emit) {
                const int czi = gz / cz;
                if (cy == 2) {
                    if (vA) store_coarse(cur, gyA / 2, czi);
                } else {
                    if (vA) store_coarse(cur, gyA, czi);
                    if (vB) store_coarse(cur + 4, gyB, czi);
                }
                (void)nv;
            }
        }
        cta_sync();                                  // every thread is done with the slots of step v
        if (v + C::PD < z1) issue_step(v + C::PD);
        // advance the ring cursors
        Pm = P0; P0 = Pp;
        Pp += C::P_PLANE;
        if (Pp == P_beg + C::NP * C::P_PLANE) Pp = P_beg;
        Z0 = Z1;
        Z1 += C::C_PLANE;
        if (Z1 == Z_beg + C::NZ * C::C_PLANE) Z1 = Z_beg;
        if (++ic == C::NC) ic = 0;
        if (++kb == C::NB) { kb = 0; kpar ^= 1u; }
        if (++gz == nz) gz = 0;
    }
    if (MODE == 1 || MODE == 3) finish_reduction(acc, 0.0, false, a.rb, a.slot, 0);
    if (MODE == 2) finish_reduction(acc, acc_b, true, a.rb, a.slot, a.slot2);
}

template <int MODE>
__global__ void __launch_bounds__(ResBulkCfg::THREADS, 2)
k_residual_bulk(const ResBulkArgs a, const __grid_constant__ ResBulkMaps maps) {
    using C = ResBulkCfg;
    if (a.run_flag && *a.run_flag == 0) return;
    // lean path (uniform.cuh)?  Tile + ring 1, planes z0-1 .. z1; box-fed (interior in y) tiles only
    bool uni = false;
    if (a.uni.brick) {
        int bid = blockIdx.x;
        const int tx = bid % a.tiles_x;
        bid /= a.tiles_x;
        const int ty = bid % a.tiles_y;
        const int zc = bid / a.tiles_y;
        const int x0 = tx * C::TX, y0 = ty * C::RY, z0 = zc * a.zchunk, z1 = min(a.g.n[2], z0 + a.zchunk);
        if ((y0 >= 1) && (y0 + C::RY + 1 <= a.g.n[1]))
            uni = ub_box_uniform_warp(a.g, a.uni.brick, x0 - 2, x0 + C::TX + 1, y0 - 2, y0 + C::RY + 1, z0 - 2, z1 + 1,
                                      threadIdx.x & 31);
    }
    if (uni) {
        if (MODE == 0 && a.g.c[0] == 2 && a.g.c[1] == 2 && a.g.c[2] == 2) res_body<MODE, true, (MODE == 0)>(a, maps);
        else res_body<MODE, true, false>(a, maps);
    } else {
        res_body<MODE, false, false>(a, maps);
    }
}

// ---- launchers ------------------------------------------------------------------------------
static bool res_maps(const LevelGeom& g, const float* L, const float* p, const float* b, ResBulkMaps* m) {
    using C = ResBulkCfg;
    const size_t N = (size_t)g.N;
    return tensor_map(p, g, C::TX, C::PH, &m->p_main) && tensor_map(p, g, 4, C::PH, &m->p_halo) &&
           tensor_map(L + 2 * N, g, C::TX, C::RY, &m->lz) && tensor_map(L, g, C::TX, C::RY, &m->lx) &&
           tensor_map(L + N, g, C::TX, C::RY + 1, &m->ly) && tensor_map(b, g, C::TX, C::RY, &m->b);
}

// The tiling of the TMA-fed residual pass on this level (for gmg_stats' count of lean-path cells)
bool res_bulk_tiling(const LevelGeom& g, int* tile_y, int* zchunk) {
    using C = ResBulkCfg;
    if (!bulk_supported(g) || (g.n[2] & 1)) return false;
    const int tiles_x = g.n[0] / C::TX, tiles_y = (g.n[1] + C::RY - 1) / C::RY;
    *tile_y = C::RY;
    *zchunk = choose_zchunk((long long)tiles_x * tiles_y, g.n[2], kZChunkPref, kZChunkMin, 296, 1);
    return true;
}

template <int MODE>
static bool launch_res_bulk(ResBulkArgs& a, cudaStream_t s) {
    using C = ResBulkCfg;
    const LevelGeom& g = a.g;
    if (!bulk_supported(g) || (g.n[2] & 1)) return false;
    ResBulkMaps maps;
    if (!res_maps(g, a.L, a.p, a.b, &maps)) return false;
    a.tiles_x = g.n[0] / C::TX;
    a.tiles_y = (g.n[1] + C::RY - 1) / C::RY;
    // two CTAs per SM; chunks start on even planes (the z pair of the restriction)
    int zchunk = choose_zchunk((long long)a.tiles_x * a.tiles_y, g.n[2], kZChunkPref, kZChunkMin, 296, 1);
    // the deterministic reduction has a bounded number of block partials
    while (MODE >= 1 && (long long)a.tiles_x * a.tiles_y * ((g.n[2] + zchunk - 1) / zchunk) > GMG_REDUCE_MAX_BLOCKS)
        zchunk *= 2;
    a.zchunk = zchunk;
    const int nzc = (g.n[2] + zchunk - 1) / zchunk;
    const unsigned int grid = (unsigned int)(a.tiles_x * a.tiles_y * nzc);
    k_residual_bulk<MODE><<<grid, C::THREADS, C::SMEM, s>>>(a, maps);
    return true;
}

bool residual_restrict_bulk(const LevelGeom& g, const float* L, const float* p, const float* b, float* b_c,
                            float* p_c, const UniArgs& uni, cudaStream_t s) {
    ResBulkArgs a;
    a.uni = uni;
    a.g = g; a.L = L; a.p = p; a.b = b; a.b_c = b_c; a.p_c = p_c;
    a.rb = ReduceBuf{nullptr, nullptr, nullptr, POST_NONE, 0.0};
    a.slot = 0;
    a.slot2 = 0;
    a.run_flag = nullptr;
    return launch_res_bulk<0>(a, s);
}

bool residual_norm2_bulk(const LevelGeom& g, const float* L, const float* p, const float* b, ReduceBuf rb,
                         int slot, const UniArgs& uni, cudaStream_t s) {
    ResBulkArgs a;
    a.uni = uni;
    a.g = g; a.L = L; a.p = p; a.b = b; a.b_c = nullptr; a.p_c = nullptr;
    a.rb = rb;
    a.slot = slot;
    a.slot2 = 0;
    a.run_flag = nullptr;
    return launch_res_bulk<1>(a, s);
}

// the same pass as a no-op unless *run_flag != 0 (fused_norm: the cycle expected to be the last)
bool residual_norm2_bulk_if(const LevelGeom& g, const float* L, const float* p, const float* b, ReduceBuf rb,
                            int slot, const int* run_flag, const UniArgs& uni, cudaStream_t s) {
    ResBulkArgs a;
    a.uni = uni;
    a.g = g; a.L = L; a.p = p; a.b = b; a.b_c = nullptr; a.p_c = nullptr;
    a.rb = rb;
    a.slot = slot;
    a.slot2 = 0;
    a.run_flag = run_flag;
    return launch_res_bulk<1>(a, s);
}
bool residual_norm_bulk_supported(const LevelGeom& g) {
    return bulk_supported(g) && !(g.n[2] & 1);
}

// sum r^2 -> red[slot_rr] and sum b^2 over active cells -> red[slot_ref] in ONE pass (loop entry)
bool residual_and_ref_norm2_bulk(const LevelGeom& g, const float* L, const float* p, const float* b,
                                 ReduceBuf rb, int slot_rr, int slot_ref, const UniArgs& uni, cudaStream_t s) {
    ResBulkArgs a;
    a.uni = uni;
    a.g = g; a.L = L; a.p = p; a.b = b; a.b_c = nullptr; a.p_c = nullptr;
    a.rb = rb;
    a.slot = slot_rr;
    a.slot2 = slot_ref;
    a.run_flag = nullptr;
    return launch_res_bulk<2>(a, s);
}

// q = A d and red[slot] = d.q in one TMA-fed pass (the CG mat-vec, reading O10); the b stream of
// the kernel is pointed at d and ignored.
bool matvec_dot_bulk(const LevelGeom& g, const float* L, const float* d, float* q, ReduceBuf rb, int slot,
                     const UniArgs& uni, cudaStream_t s) {
    ResBulkArgs a;
    a.uni = uni;
    a.g = g; a.L = L; a.p = d; a.b = d; a.b_c = q; a.p_c = nullptr;
    a.rb = rb;
    a.slot = slot;
    a.slot2 = 0;
    a.run_flag = nullptr;
    return launch_res_bulk<3>(a, s);
}

int configure_residual_bulk() {
    cudaError_t e = cudaFuncSetAttribute(k_residual_bulk<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ResBulkCfg::SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_residual_bulk<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ResBulkCfg::SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_residual_bulk<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ResBulkCfg::SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_residual_bulk<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ResBulkCfg::SMEM);
    return (int)e;
}

}  // namespace gmgf

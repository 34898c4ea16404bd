// kernels_fused.cu -- the tiled fast path of the hot loop on big levels (sm_100a):
//
//  k_rb_sweep       one whole red+black Gauss-Seidel sweep (PAPER.md:43 S3.1; DESIGN.md readings
//                   O3, O8) in ONE streaming pass over p, b and the three face-coefficient arrays
//                   (24 B/cell instead of 48 for two colour passes; BASELINE.json:north_star "a
//                   fused red+black pass where the dependence allows"), optionally with the
//                   prolongation + correction of the coarse level fused into its loads (O6).
//  k_residual_tiled residual fused with the restriction (O6, O9; north_star "a residual kernel
//                   fused with the restriction"), or with the squared-norm reduction.
//
// k_rb_sweep: a CTA owns a TX x TY tile in (x,y) and marches along z over a chunk of planes.
// Shared memory holds a ring of NSLOT planes of p (tile + halo 2 in y, one float4 group in x).
// Per step u (one barrier per step):
//     A(u+2)  global -> registers -> smem: plane u+2 of the source iterate (+ P e_c if fused)
//     B(u)    first-colour update of plane u on the tile + ring 1 (redundant at the tile edge),
//             reading only second-colour (old) neighbours; written in place in smem
//     barrier
//     C(u-1)  second-colour update of plane u-1 on the tile, reading the first-colour values
//             B left in planes u-2, u-1, u; the whole plane (both colours) goes to dst
// Source and destination are DIFFERENT arrays (ping-pong), so neighbouring CTAs never race on
// halo cells.  A "main" thread owns four x-consecutive cells (one float4) of one row: own-row
// neighbours come from registers / warp shuffles, the y and z neighbours from shared memory.
// The face coefficients and b of the own cells stream global -> REGISTERS exactly once per
// thread: the set of plane u+1 is prefetched during step u, used by B one step later and by C
// two steps later (three sets rotate through registers), so DRAM latency is hidden by
// construction and no coefficient is re-read.  The two ring-1 columns next to the tile
// (x0-1 and x0+TX) are updated by one extra "edge" warp, one lane per (side,row).
// The per-cell arithmetic is stencil.cuh's apply7/diag6/relax, identical to the generic
// kernels, so fast and generic paths agree bit for bit on every cell.
#include "fused_common.cuh"
#include "uniform.cuh"

namespace gmgf {

template <int TX_, int TY_>
struct SweepCfg {
    static constexpr int TX = TX_, TY = TY_;
    static constexpr int LPR = TX / 4;          // lanes (float4 groups) per tile row
    static constexpr int ROWS = TY + 2;         // rows running phase B (tile + ring 1)
    static constexpr int MAIN = LPR * ROWS;     // main threads
    static constexpr int THREADS = MAIN + 32;   // + one edge warp
    static constexpr int SW = TX + 8;           // smem row stride in floats (one group each side)
    static constexpr int SH = TY + 4;           // smem rows (halo 2)
    static constexpr int PLANE = SW * SH;
    static constexpr int NSLOT = 6;
    static constexpr int AGROUPS = (LPR + 2) * SH;  // float4 groups per loaded plane
    static constexpr int APER = (AGROUPS + THREADS - 1) / THREADS;
    static constexpr size_t SMEM = (size_t)NSLOT * PLANE * sizeof(float);
    static_assert(MAIN % 32 == 0 && 32 % LPR == 0 && 2 * ROWS <= 32, "tile shape");
};

struct SweepArgs {
    LevelGeom g;
    const float* L;
    const float* src;
    float* dst;
    const float* b;
    const float* omega;
    const float* e_c;  // coarse correction to add to src on load, or nullptr
    int first_colour;
    int zchunk;        // planes per CTA
    int tiles_x, tiles_y;
    int pf;            // L2 prefetch distance in planes (0 = off)
};

template <class C, int MINB>
__global__ void __launch_bounds__(C::THREADS, MINB) k_rb_sweep(const SweepArgs a) {
    extern __shared__ __align__(16) float sm[];
    const LevelGeom& g = a.g;
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const size_t N = (size_t)g.N;
    const int plane = nx * ny;
    const int tid = threadIdx.x;
    int bid = blockIdx.x;
    const int tx = bid % a.tiles_x;
    bid /= a.tiles_x;
    const int ty = bid % a.tiles_y;
    const int zc = bid / a.tiles_y;
    const int x0 = tx * C::TX, y0 = ty * C::TY;
    const int z0 = zc * a.zchunk;
    const int z1 = min(nz, z0 + a.zchunk);
    const float omega = *a.omega;
    const int fc = a.first_colour;
    const float* Lx = a.L;
    const float* Ly = a.L + N;
    const float* Lz = a.L + 2 * N;

    // ---- plane loader (phase A), all threads ---------------------------------------------------
    int a_goff[C::APER], a_soff[C::APER], a_coff[C::APER];
    const int ncx = nx / g.c[0], ncy = ny / g.c[1];
#pragma unroll
    for (int i = 0; i < C::APER; ++i) {
        const int e = tid + i * C::THREADS;
        if (e < C::AGROUPS) {
            const int r = e / (C::LPR + 2), gc = e % (C::LPR + 2);
            const int x = wrapi(x0 - 4 + 4 * gc, nx), y = wrapi(y0 + r - 2, ny);
            a_goff[i] = y * nx + x;
            a_soff[i] = r * C::SW + 4 * gc;
            a_coff[i] = (y / g.c[1]) * ncx + x / g.c[0];
        } else {
            a_goff[i] = -1;
            a_soff[i] = 0;
            a_coff[i] = 0;
        }
    }
    auto load_plane = [&](int u, float4 (&v)[C::APER]) {
        const int gz = wrap1(u, nz);
        const float* base = a.src + (size_t)gz * plane;
#pragma unroll
        for (int i = 0; i < C::APER; ++i) {
            if (a_goff[i] >= 0) {
                v[i] = ldg4(base + a_goff[i]);
                if (a.e_c) {
                    const float* eb = a.e_c + (size_t)(gz / g.c[2]) * (ncx * ncy) + a_coff[i];
                    if (g.c[0] == 2) {
                        const float2 e2 = __ldg(reinterpret_cast<const float2*>(eb));
                        v[i].x += e2.x; v[i].y += e2.x; v[i].z += e2.y; v[i].w += e2.y;
                    } else {
                        const float4 e4 = ldg4(eb);
                        v[i].x += e4.x; v[i].y += e4.y; v[i].z += e4.z; v[i].w += e4.w;
                    }
                }
            }
        }
    };
    auto prefetch_plane = [&](int u) {   // L2 prefetch of a source plane a few steps ahead
        const float* base = a.src + (size_t)wrap1(u, nz) * plane;
#pragma unroll
        for (int i = 0; i < C::APER; ++i)
            if (a_goff[i] >= 0) prefetch_l2(base + a_goff[i]);
    };
    auto slot_of = [&](int u) -> float* { return sm + ((u - (z0 - 2)) % C::NSLOT) * C::PLANE; };
    auto store_plane = [&](int u, const float4 (&v)[C::APER]) {
        float* s = slot_of(u);
#pragma unroll
        for (int i = 0; i < C::APER; ++i)
            if (a_goff[i] >= 0) *reinterpret_cast<float4*>(s + a_soff[i]) = v[i];
    };

    // ---- prologue: planes z0-2, z0-1, z0 -------------------------------------------------------
    float4 va[C::APER];  // source plane in flight: loaded during one step, stored during the next
    {
        // all four loads are issued before the first store: one memory latency, not four
        float4 v0[C::APER], v1[C::APER], v2[C::APER];
        load_plane(z0 - 2, v0);
        load_plane(z0 - 1, v1);
        load_plane(z0, v2);
        if (z0 + 1 <= z1 + 1) load_plane(z0 + 1, va);
        store_plane(z0 - 2, v0);
        store_plane(z0 - 1, v1);
        store_plane(z0, v2);
    }
    cta_sync();

    if (tid < C::MAIN) {
        // ---- main threads: one float4 group of one row ---------------------------------------
        const int lx = tid % C::LPR, ry = tid / C::LPR;
        const int xl = x0 + 4 * lx;   // logical x of the first own cell (may overhang the domain)
        const int yl = y0 + ry - 1;   // logical y of the own row (-1 ..)
        const int gx = wrapi(xl, nx), gy = wrapi(yl, ny), gyp = wrapi(yl + 1, ny);
        const int gxh = wrapi(xl + 4, nx);
        const bool row_c = (ry >= 1) && (ry <= C::TY) && (yl < ny);
        const bool store_ok = row_c && (xl < nx);
        const bool zx_lo = g.bc[0] && gx == 0, zx_hi = g.bc[0] && gxh == 0;
        const bool zy_lo = g.bc[1] && gy == 0, zy_hi = g.bc[1] && gyp == 0;
        const bool last_lane = (lx == C::LPR - 1);
        const int own_off = (ry + 1) * C::SW + 4 + 4 * lx;  // own float4 in a smem plane
        const int o_row = gy * nx + gx, o_rowp = gyp * nx + gx, o_xh = gy * nx + gxh;

        auto fetch = [&](int u, CSet& s) {  // issue the global loads of plane u's coefficient set
            const int gz = wrap1(u, nz), gzp = wrap1(u + 1, nz);
            const size_t pz = (size_t)gz * plane, pzp = (size_t)gzp * plane;
            s.lx = ldg4(Lx + pz + o_row);
            s.ly = ldg4(Ly + pz + o_row);
            s.lyh = ldg4(Ly + pz + o_rowp);
            s.lzh = ldg4(Lz + pzp + o_row);
            s.b = ldg4(a.b + pz + o_row);
            if (last_lane) s.lxh = __ldg(Lx + pz + o_xh);
        };
        auto prefetch_set = [&](int u) {  // L2 prefetch of a coefficient set a few steps ahead
            const int gz = wrap1(u, nz), gzp = wrap1(u + 1, nz);
            const size_t pz = (size_t)gz * plane, pzp = (size_t)gzp * plane;
            prefetch_l2(Lx + pz + o_row);
            prefetch_l2(Ly + pz + o_row);
            prefetch_l2(Lz + pzp + o_row);
            prefetch_l2(a.b + pz + o_row);
        };
        auto finish = [&](int u, CSet& s) {  // first use of a set: neighbour face + wall faces
            const float t = __shfl_down_sync(0xffffffffu, s.lx.x, 1);
            if (!last_lane) s.lxh = t;
            if (zx_lo) s.lx.x = 0.0f;
            if (zx_hi) s.lxh = 0.0f;
            if (zy_lo) s.ly = zero4();
            if (zy_hi) s.lyh = zero4();
            if (g.bc[2] && wrap1(u + 1, nz) == 0) s.lzh = zero4();
        };
        auto phase = [&](int u, int colour, const CSet& s, const float4& lz) -> float4 {
            const float* P = slot_of(u);
            const float4 own = lds4(P + own_off);
            const float4 ym = lds4(P + own_off - C::SW);
            const float4 yp = lds4(P + own_off + C::SW);
            const float4 zm = lds4(slot_of(u - 1) + own_off);
            const float4 zp = lds4(slot_of(u + 1) + own_off);
            float xm = __shfl_up_sync(0xffffffffu, own.w, 1);
            float xp = __shfl_down_sync(0xffffffffu, own.x, 1);
            if (lx == 0) xm = P[own_off - 1];
            if (last_lane) xp = P[own_off + 4];
            return ((yl + u + colour) & 1) ? update_pair<1>(xm, own, xp, ym, yp, zm, zp, s, lz, omega)
                                           : update_pair<0>(xm, own, xp, ym, yp, zm, zp, s, lz, omega);
        };
        auto step = [&](int u, CSet& Sp, CSet& Sc, CSet& Sn, float4& lzpp) {
            if (u + 1 <= z1) fetch(u + 1, Sn);
            if (a.pf > 0 && u + 1 + a.pf <= z1) prefetch_set(u + 1 + a.pf);
            if (a.pf > 0 && u + 3 + a.pf <= z1 + 1) prefetch_plane(u + 3 + a.pf);
            finish(u, Sc);
            {   // B(u): first colour on tile + ring 1, in place in shared memory
                const float4 nw = phase(u, fc, Sc, Sp.lzh);
                *reinterpret_cast<float4*>(slot_of(u) + own_off) = nw;
            }
            // plane u+2 was requested a step ago; plane u+3 has until the next step to arrive
            if (u + 2 <= z1 + 1) store_plane(u + 2, va);
            if (u + 3 <= z1 + 1) load_plane(u + 3, va);
            cta_sync();
            if (u - 1 >= z0 && __any_sync(0xffffffffu, row_c)) {  // C(u-1): second colour, tile only
                const float4 nw = phase(u - 1, fc ^ 1, Sp, lzpp);
                if (store_ok)
                    *reinterpret_cast<float4*>(a.dst + (size_t)(u - 1) * plane + o_row) = nw;
            }
            lzpp = Sp.lzh;
        };
        CSet S0, S1, S2;
        float4 lzpp = zero4();
        {
            const int gzm = wrap1(z0 - 1, nz);
            S0.lzh = (g.bc[2] && gzm == 0) ? zero4() : ldg4(Lz + (size_t)gzm * plane + o_row);
            S0.lx = S0.ly = S0.lyh = S0.b = zero4();
            S0.lxh = 0.0f;
            fetch(z0 - 1, S1);
            S2 = S0;
        }
        int u = z0 - 1;
        while (true) {
            step(u, S0, S1, S2, lzpp);
            if (++u > z1) break;
            step(u, S1, S2, S0, lzpp);
            if (++u > z1) break;
            step(u, S2, S0, S1, lzpp);
            if (++u > z1) break;
        }
    } else {
        // ---- edge warp: ring-1 cells x0-1 and x0+TX of every row, phase B only ----------------
        const int el = tid - C::MAIN;
        const bool e_act = el < 2 * C::ROWS;
        const int side = el & 1, ery = e_act ? (el >> 1) : 0;
        const int xs = side ? x0 + C::TX : x0 - 1;
        const int eyl = y0 + ery - 1;
        const int gxs = wrapi(xs, nx), gxs1 = wrapi(xs + 1, nx);
        const int egy = wrapi(eyl, ny), egyp = wrapi(eyl + 1, ny);
        const int e_off = (ery + 1) * C::SW + (side ? 4 + C::TX : 3);
        const int o_c = egy * nx + gxs, o_x1 = egy * nx + gxs1, o_yp = egyp * nx + gxs;
        const bool ex_lo = g.bc[0] && gxs == 0, ex_hi = g.bc[0] && gxs1 == 0;
        const bool ey_lo = g.bc[1] && egy == 0, ey_hi = g.bc[1] && egyp == 0;
        struct ESet { float wxl, wxh, wyl, wyh, wzl, wzh, b; };
        auto fetch_e = [&](int u, ESet& s) {
            const int gz = wrap1(u, nz), gzp = wrap1(u + 1, nz);
            const size_t pz = (size_t)gz * plane, pzp = (size_t)gzp * plane;
            s.wxl = ex_lo ? 0.0f : __ldg(Lx + pz + o_c);
            s.wxh = ex_hi ? 0.0f : __ldg(Lx + pz + o_x1);
            s.wyl = ey_lo ? 0.0f : __ldg(Ly + pz + o_c);
            s.wyh = ey_hi ? 0.0f : __ldg(Ly + pz + o_yp);
            s.wzl = (g.bc[2] && gz == 0) ? 0.0f : __ldg(Lz + pz + o_c);
            s.wzh = (g.bc[2] && gzp == 0) ? 0.0f : __ldg(Lz + pzp + o_c);
            s.b = __ldg(a.b + pz + o_c);
        };
        ESet Ec, En;
        fetch_e(z0 - 1, Ec);
        En = Ec;
        for (int u = z0 - 1; u <= z1; ++u) {
            if (u + 1 <= z1) fetch_e(u + 1, En);
            if (a.pf > 0 && u + 3 + a.pf <= z1 + 1) prefetch_plane(u + 3 + a.pf);
            if (e_act && ((xs + eyl + u) & 1) == fc) {
                float* P = slot_of(u);
                const float pc = P[e_off];
                const float Ap = apply7(pc, Ec.wxl, Ec.wxh, Ec.wyl, Ec.wyh, Ec.wzl, Ec.wzh, P[e_off - 1],
                                        P[e_off + 1], P[e_off - C::SW], P[e_off + C::SW],
                                        slot_of(u - 1)[e_off], slot_of(u + 1)[e_off]);
                P[e_off] = relax(pc, Ec.b, Ap,
                                 diag6(Ec.wxl, Ec.wxh, Ec.wyl, Ec.wyh, Ec.wzl, Ec.wzh), omega);
            }
            if (u + 2 <= z1 + 1) store_plane(u + 2, va);
            if (u + 3 <= z1 + 1) load_plane(u + 3, va);
            cta_sync();
            Ec = En;
        }
    }
}

// ---- residual fused with restriction / with the squared norm ------------------------------------
// CTA tile TX x RY x RZ fine cells, one float4 group per thread.  The residual of every cell is
// r = b - A p on active cells, 0 elsewhere (O9).  MODE 0: r goes to shared memory and each
// coarse cell of the tile sums its children in the order z, y, x (x innermost) -- the order of
// the generic kernel, so both paths give identical bits (O6: restriction = sum).  MODE 1: sum r^2
// in FP64, finished by the deterministic two-stage reduction.
template <int TX_, int RY_, int RZ_>
struct ResCfg {
    static constexpr int TX = TX_, RY = RY_, RZ = RZ_;
    static constexpr int LPR = TX / 4;
    static constexpr int THREADS = LPR * RY * RZ;
    static_assert(THREADS % 32 == 0 && 32 % LPR == 0, "row segments must tile warps");
};

struct ResArgs {
    LevelGeom g;
    const float* L;
    const float* p;
    const float* b;
    float* b_c;
    float* p_c;
    ReduceBuf rb;
    int slot;
    int tiles_x, tiles_y, tiles_z;
};

template <class C, int MODE>
__global__ void __launch_bounds__(C::THREADS) k_residual_tiled(const ResArgs a) {
    __shared__ __align__(16) float rs[(MODE == 0) ? C::TX * C::RY * C::RZ : 4];
    const LevelGeom& g = a.g;
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const long long N = g.N;
    const long long plane = (long long)nx * ny;
    const int tid = threadIdx.x;
    const int lx = tid % C::LPR;
    const int ry = (tid / C::LPR) % C::RY;
    const int rz = tid / (C::LPR * C::RY);
    const float* Lx = a.L;
    const float* Ly = a.L + N;
    const float* Lz = a.L + 2 * N;
    const int ntiles = a.tiles_x * a.tiles_y * a.tiles_z;
    double acc = 0.0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        int t = tile;
        const int tx = t % a.tiles_x;
        t /= a.tiles_x;
        const int ty = t % a.tiles_y;
        const int tz = t / a.tiles_y;
        const int x0 = tx * C::TX, y0 = ty * C::RY, z0 = tz * C::RZ;
        const int xl = x0 + 4 * lx, yl = y0 + ry, zl = z0 + rz;
        const bool in_dom = xl < nx && yl < ny && zl < nz;
        // wrapped coordinates keep every lane's loads valid (shuffles need all lanes)
        const int gx = wrapi(xl, nx), gy = wrapi(yl, ny), gz = wrapi(zl, nz);
        const int gxm = wrapi(xl - 1, nx), gxh = wrapi(xl + 4, nx);
        const int gym = wrapi(yl - 1, ny), gyp = wrapi(yl + 1, ny);
        const int gzm = wrapi(zl - 1, nz), gzp = wrapi(zl + 1, nz);
        const long long row = gz * plane + (long long)gy * nx;
        const float4 own = ldg4(a.p + row + gx);
        const float4 ym = ldg4(a.p + gz * plane + (long long)gym * nx + gx);
        const float4 yp = ldg4(a.p + gz * plane + (long long)gyp * nx + gx);
        const float4 zm = ldg4(a.p + gzm * plane + (long long)gy * nx + gx);
        const float4 zp = ldg4(a.p + gzp * plane + (long long)gy * nx + gx);
        float xm = __shfl_up_sync(0xffffffffu, own.w, 1);
        float xp = __shfl_down_sync(0xffffffffu, own.x, 1);
        if (lx == 0) xm = __ldg(a.p + row + gxm);
        if (lx == C::LPR - 1) xp = __ldg(a.p + row + gxh);
        float4 wx = ldg4(Lx + row + gx);
        float4 wy = ldg4(Ly + row + gx);
        float4 wyh = ldg4(Ly + gz * plane + (long long)gyp * nx + gx);
        float4 wz = ldg4(Lz + row + gx);
        float4 wzh = ldg4(Lz + gzp * plane + (long long)gy * nx + gx);
        const float4 bb = ldg4(a.b + row + gx);
        float wxh = __shfl_down_sync(0xffffffffu, wx.x, 1);
        if (lx == C::LPR - 1) wxh = __ldg(Lx + row + gxh);
        if (g.bc[0] && gx == 0) wx.x = 0.0f;
        if (g.bc[0] && gxh == 0) wxh = 0.0f;
        if (g.bc[1] && gy == 0) wy = make_float4(0.f, 0.f, 0.f, 0.f);
        if (g.bc[1] && gyp == 0) wyh = make_float4(0.f, 0.f, 0.f, 0.f);
        if (g.bc[2] && gz == 0) wz = make_float4(0.f, 0.f, 0.f, 0.f);
        if (g.bc[2] && gzp == 0) wzh = make_float4(0.f, 0.f, 0.f, 0.f);
        float4 r;
        {
            const float A0 = apply7(own.x, wx.x, wx.y, wy.x, wyh.x, wz.x, wzh.x, xm, own.y, ym.x, yp.x, zm.x, zp.x);
            const float A1 = apply7(own.y, wx.y, wx.z, wy.y, wyh.y, wz.y, wzh.y, own.x, own.z, ym.y, yp.y, zm.y, zp.y);
            const float A2 = apply7(own.z, wx.z, wx.w, wy.z, wyh.z, wz.z, wzh.z, own.y, own.w, ym.z, yp.z, zm.z, zp.z);
            const float A3 = apply7(own.w, wx.w, wxh, wy.w, wyh.w, wz.w, wzh.w, own.z, xp, ym.w, yp.w, zm.w, zp.w);
            const float D0 = diag6(wx.x, wx.y, wy.x, wyh.x, wz.x, wzh.x);
            const float D1 = diag6(wx.y, wx.z, wy.y, wyh.y, wz.y, wzh.y);
            const float D2 = diag6(wx.z, wx.w, wy.z, wyh.z, wz.z, wzh.z);
            const float D3 = diag6(wx.w, wxh, wy.w, wyh.w, wz.w, wzh.w);
            r.x = (D0 != 0.0f) ? bb.x - A0 : 0.0f;
            r.y = (D1 != 0.0f) ? bb.y - A1 : 0.0f;
            r.z = (D2 != 0.0f) ? bb.z - A2 : 0.0f;
            r.w = (D3 != 0.0f) ? bb.w - A3 : 0.0f;
        }
        if (MODE == 1) {
            if (in_dom)
                acc += ((double)r.x * r.x + (double)r.y * r.y) + ((double)r.z * r.z + (double)r.w * r.w);
        } else {
            *reinterpret_cast<float4*>(rs + (rz * C::RY + ry) * C::TX + 4 * lx) = r;
            __syncthreads();
            const int cx = g.c[0], cy = g.c[1], cz = g.c[2];
            const int tcx = C::TX / cx, tcy = C::RY / cy, tcz = C::RZ / cz;
            const int ncx = nx / cx, ncy = ny / cy, ncz = nz / cz;
            for (int u = tid; u < tcx * tcy * tcz; u += C::THREADS) {
                const int I = u % tcx, J = (u / tcx) % tcy, K = u / (tcx * tcy);
                const int GI = x0 / cx + I, GJ = y0 / cy + J, GK = z0 / cz + K;
                if (GI < ncx && GJ < ncy && GK < ncz) {
                    const float s = restrict_tree(cx, cy, cz, [&](int e, int bq, int aa) {
                        return rs[((cz * K + aa) * C::RY + (cy * J + bq)) * C::TX + cx * I + e];
                    });
                    const long long o = GI + (long long)ncx * (GJ + (long long)ncy * GK);
                    a.b_c[o] = s;
                    if (a.p_c) a.p_c[o] = 0.0f;
                }
            }
            __syncthreads();
        }
    }
    if (MODE == 1) finish_reduction(acc, 0.0, false, a.rb, a.slot, 0);
}


// ---- prolongation + correction as its own pass (O6): p_f(I) += e_c(parent(I)), one float4 of
// fine cells per thread.  Used in front of the TMA-fed sweep, where fusing the correction into the
// sweep's shared-memory planes costs more than this 8.5 B/cell streaming pass.
__global__ void __launch_bounds__(256)
k_prolong_add4(LevelGeom g, const float* __restrict__ e_c, float* __restrict__ p_f) {
    // one work item = the (up to four) fine rows under one coarse row segment: the parent values
    // are fetched once and up to four float4 of p are in flight per thread
    const int nx4 = g.n[0] >> 2;
    const int cy = g.c[1], cz = g.c[2];
    const int ncx = g.n[0] / g.c[0], ncy = g.n[1] / cy, ncz = g.n[2] / cz;
    const long long items = (long long)nx4 * ncy * ncz;
    const long long srow = nx4, splane = (long long)nx4 * g.n[1];   // in float4 units
    float4* p4 = reinterpret_cast<float4*>(p_f);
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < items;
         t += (long long)gridDim.x * blockDim.x) {
        const long long row = t / nx4;
        const int i4 = (int)(t - row * nx4);
        const int K = (int)(row / ncy);
        const int J = (int)(row - (long long)K * ncy);
        const long long pc = (long long)K * ncy + J;
        float4 e;
        if (g.c[0] == 2) {
            const float2 h = __ldg(reinterpret_cast<const float2*>(e_c + pc * ncx + 2 * i4));
            e = make_float4(h.x, h.x, h.y, h.y);
        } else {
            e = ldg4(e_c + pc * ncx + 4 * i4);
        }
        const long long base = (long long)(K * cz) * splane + (long long)(J * cy) * srow + i4;
        float4 v[2][2];
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int b = 0; b < 2; ++b)
                if (a < cz && b < cy) v[a][b] = p4[base + a * splane + b * srow];
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int b = 0; b < 2; ++b)
                if (a < cz && b < cy) {
                    float4 w = v[a][b];
                    w.x += e.x; w.y += e.y; w.z += e.z; w.w += e.w;
                    p4[base + a * splane + b * srow] = w;
                }
    }
}

void prolong_add4(const LevelGeom& g, const float* e_c, float* p_f, cudaStream_t s) {
    const long long items = (g.N >> 2) / ((long long)g.c[1] * g.c[2]);
    long long nb = (items + 255) / 256;
    if (nb > 148LL * 64) nb = 148LL * 64;
    if (nb < 1) nb = 1;
    k_prolong_add4<<<(unsigned int)nb, 256, 0, s>>>(g, e_c, p_f);
}

// ---- launchers ----------------------------------------------------------------------------------
using Sweep128 = SweepCfg<128, 9>;
using Sweep64 = SweepCfg<64, 14>;
using Sweep32 = SweepCfg<32, 14>;
static constexpr int kSweepMinBlocks = 1;
using Res128 = ResCfg<128, 4, 4>;
using Res64 = ResCfg<64, 8, 4>;
using Res32 = ResCfg<32, 16, 4>;

bool sweep_v2_supported(const LevelGeom& g) {
    return g.n[0] % 4 == 0 && g.n[0] >= 16 && g.n[1] >= 2 && g.n[2] >= 4 &&
           (long long)g.n[0] * g.n[1] < (1LL << 30);
}

template <class C, int MB = kSweepMinBlocks>
static void launch_sweep(SweepArgs& a, cudaStream_t s) {
    const LevelGeom& g = a.g;
    a.tiles_x = (g.n[0] + C::TX - 1) / C::TX;
    a.tiles_y = (g.n[1] + C::TY - 1) / C::TY;
    const int zchunk = choose_zchunk((long long)a.tiles_x * a.tiles_y, g.n[2], kZChunkPref, kZChunkMin, 148, 0);
    a.zchunk = zchunk;
    a.pf = 3;   // L2 prefetch distance of the coefficient streams, in planes
    const int nzc = (g.n[2] + zchunk - 1) / zchunk;
    const unsigned int grid = (unsigned int)(a.tiles_x * a.tiles_y * nzc);
    k_rb_sweep<C, MB><<<grid, C::THREADS, C::SMEM, s>>>(a);
}

void rb_sweep_v2(const LevelGeom& g, const float* L, const float* src, float* dst, const float* b,
                 const float* omega, int first_colour, const float* e_c, cudaStream_t s) {
    SweepArgs a;
    a.g = g; a.L = L; a.src = src; a.dst = dst; a.b = b; a.omega = omega; a.e_c = e_c;
    a.first_colour = first_colour;
    if (g.n[0] >= 128) launch_sweep<Sweep128>(a, s);
    else if (g.n[0] >= 64) launch_sweep<Sweep64>(a, s);
    else launch_sweep<Sweep32>(a, s);
}

bool resrestrict_supported(const LevelGeom& g) {
    return g.n[0] % 4 == 0 && g.n[0] >= 16 && g.n[1] >= 2 && g.n[2] >= 2;
}

template <class C, int MODE>
static void launch_res(ResArgs& a, cudaStream_t s) {
    const LevelGeom& g = a.g;
    a.tiles_x = (g.n[0] + C::TX - 1) / C::TX;
    a.tiles_y = (g.n[1] + C::RY - 1) / C::RY;
    a.tiles_z = (g.n[2] + C::RZ - 1) / C::RZ;
    long long nt = (long long)a.tiles_x * a.tiles_y * a.tiles_z;
    if (MODE == 1 && nt > GMG_REDUCE_MAX_BLOCKS) nt = GMG_REDUCE_MAX_BLOCKS;
    k_residual_tiled<C, MODE><<<(unsigned int)nt, C::THREADS, 0, s>>>(a);
}

bool residual_restrict_bulk(const LevelGeom& g, const float* L, const float* p, const float* b, float* b_c,
                            float* p_c, const UniArgs& uni, cudaStream_t s);
bool residual_norm2_bulk(const LevelGeom& g, const float* L, const float* p, const float* b, ReduceBuf rb,
                         int slot, const UniArgs& uni, cudaStream_t s);
int configure_residual_bulk();

void residual_restrict(const LevelGeom& g, const float* L, const float* p, const float* b,
                       float* b_c, float* p_c, int allow_tma, const UniArgs& uni, cudaStream_t s) {
    if (allow_tma && residual_restrict_bulk(g, L, p, b, b_c, p_c, uni, s)) return;
    ResArgs a;
    a.g = g; a.L = L; a.p = p; a.b = b; a.b_c = b_c; a.p_c = p_c;
    a.rb = ReduceBuf{nullptr, nullptr, nullptr, POST_NONE, 0.0};
    a.slot = 0;
    if (g.n[0] >= 128) launch_res<Res128, 0>(a, s);
    else if (g.n[0] >= 64) launch_res<Res64, 0>(a, s);
    else launch_res<Res32, 0>(a, s);
}

void residual_norm2(const LevelGeom& g, const float* L, const float* p, const float* b, ReduceBuf rb,
                    int slot, int allow_tma, const UniArgs& uni, cudaStream_t s) {
    if (allow_tma && residual_norm2_bulk(g, L, p, b, rb, slot, uni, s)) return;
    ResArgs a;
    a.g = g; a.L = L; a.p = p; a.b = b; a.b_c = nullptr; a.p_c = nullptr;
    a.rb = rb;
    a.slot = slot;
    if (g.n[0] >= 128) launch_res<Res128, 1>(a, s);
    else if (g.n[0] >= 64) launch_res<Res64, 1>(a, s);
    else launch_res<Res32, 1>(a, s);
}

int configure_v2() {
    if (configure_residual_bulk() != 0) return 1;
    cudaError_t e = cudaFuncSetAttribute(k_rb_sweep<Sweep128, kSweepMinBlocks>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Sweep128::SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_rb_sweep<Sweep64, kSweepMinBlocks>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Sweep64::SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_rb_sweep<Sweep32, kSweepMinBlocks>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Sweep32::SMEM);
    return (int)e;
}

}  // namespace gmgf

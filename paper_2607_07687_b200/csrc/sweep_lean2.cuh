// sweep_lean2.cuh -- lean_body2: the fused red+black sweep of a tile whose coefficients are the level's
// constants (uniform.cuh), for the kernel that runs ONLY such tiles (k_rb_sweep_lean, two CTAs per SM),
// with TWO vertically adjacent rows per thread.  Same schedule as sweep_body: per z step B(u) on tile +
// ring 1 in shared memory, C(u-1) streamed to the destination, one CTA barrier, TMA boxes PD steps ahead;
// the z loop is unrolled twice so that the colour parity of a step is a compile-time constant.  The lean sweep is bound by the shared-memory pipe (every cell is read six
// times per sweep and the x-neighbour shuffles share the queue: profiles/r02_top_kernels_c4.md); a
// thread that owns rows r and r+1 has each row's vertical neighbour in its own registers -- in plane u
// (source values) for phase B, in plane u-1 (its own phase-B results of the step before) for phase C --
// and carries plane u+1 into the next step as "own": 8 instead of 18 float4 loads per 8 cells.  Eight
// main warps cover the 15 phase-B rows of a 128 x 13 tile (the last thread row has one row only), one
// edge warp the two ring-1 columns: 288 threads, two CTAs per SM, 96 registers (a CTA's 9 warps are allocated as 10), operands of
// the next step loaded in front of the barrier as in sweep_body.  Same update_pair_* calls on the same
// operands: bit-identical to sweep_body (tests).  Included by kernels_sweep.cu.
#pragma once

namespace gmgf {

// RIM = false: 8 main warps + an edge warp (288 threads; 96 registers at two CTAs per SM, a few
// spills -- the faster shape for the plain sweep: 2.98 vs 3.16 ms at 1024^3); RIM = true: the last
// main warp, which owns one row only, also updates the ring-1 cells (256 threads, up to 128
// registers: the norm-carrying variants need them -- 3.66 vs 3.93 ms).
template <bool RIM> struct Lean2Threads { static constexpr int value = RIM ? 256 : 288; };

// PRO: the sweep starts from p + P e_c (prolongation + correction, reading O6: each fine cell gets its
// parent's value) without p having been rewritten: every SOURCE value is corrected where it enters a
// register, with the same single addition k_prolong_add4 performs, so the result equals "correction
// pass, then sweep" bit for bit.  Phase B stores whole float4s of corrected values, so the operands
// other threads store to during a step are loaded in front of the barrier (main threads: as always;
// the edge warp: its one in-tile neighbour) -- and one more CTA barrier separates the loads in front
// of step 0 from step 0's stores.  The parents change every second plane: a thread keeps the float2
// parents of its four operand rows (and of the x-halo cell) for the current coarse plane in registers
// and fetches the next coarse plane's right in front of the loads that use them (fetched at the top
// of the step, a step body ahead, they are live across the step and spill: 3.20 vs 2.94 ms at
// 1024^3; the plain lean sweep takes 2.38 ms).  2x2x2 coarsening, plain sweep only.
template <class C, int YMODE, int NORM, bool RIM, bool PRO = false>
__device__ __forceinline__ void lean_body2(const BulkArgs& a, const BulkMaps& allmaps, const int tile) {
    static_assert(C::LEAN && C::PD == 4 && C::NP == 6 && C::NC == 6 && C::NB == 6, "rings of period 6");
    static_assert(YMODE == 0 || YMODE == 2, "box-fed tiles only");
    static_assert(!PRO || (NORM == 0 && !RIM), "prolongation rides on the plain sweep");
    constexpr int R = 6, PD = C::PD;
    extern __shared__ __align__(1024) float sm[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(sm + C::FLOATS);  // [0..6) step groups, [6] prologue
    const LevelGeom& g = a.g;
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const int plane = nx * ny;
    const int tid = threadIdx.x;
    const int warp_id = tid >> 5, lane_id = tid & 31;
    constexpr int NMAIN = 8;   // main warps, two rows per thread; the last one has ONE row (and, RIM, the edge cells)
    int bid = tile;
    const int tx = bid % a.tiles_x;
    bid /= a.tiles_x;
    const int ty = bid % a.tiles_y;
    const int zc = bid / a.tiles_y;
    const int x0 = tx * C::TX, y0 = ty * C::TY;
    const int z0 = zc * a.zchunk;
    const int z1 = min(nz, z0 + a.zchunk);
    const int T = z1 - z0 + 2;                       // steps t = 0 .. T-1 work on plane u = z0-1+t
    const float omega = *a.omega;
    const int fc = a.first_colour;
    const int xL = wrapi(x0 - 4, nx), xR = wrapi(x0 + C::TX, nx);  // halo column groups
    // YMODE 2 geometry: see sweep_body
    const bool y_first = (y0 == 0);
    const MapSet& maps = allmaps.m[YMODE == 2 ? (y_first ? 1 : 2) : 0];
    const int hP = ny - y0 + 2, hC = ny - y0 + 1;
    const int e_oP = y_first ? 2 : 0, e_oC = y_first ? 1 : 0;
    const int hs = (YMODE == 2 && y_first) ? 24 : 0;
    const int e_yP = y_first ? 0 : y0 - 2, e_yC = y_first ? 0 : y0 - 1;
    const int e_pj0 = y_first ? 0 : hP, e_py0 = y_first ? ny - 2 : 0;
    const int e_cj = y_first ? 0 : hC, e_cy = y_first ? ny - 1 : 0;
    const uint32_t e_pbytes = (uint32_t)((y_first ? C::SH : hP + 2) * (C::TX + 8)) * 4u;
    const uint32_t e_cbytes = (uint32_t)((y_first ? C::ROWS : hC + 1) * C::TX) * 4u;
    const uint32_t step_bytes = (YMODE == 2) ? e_pbytes + e_cbytes : C::STEP_BYTES_UNI;
    const uint32_t pro_bytes = (YMODE == 2) ? 2u * e_pbytes : C::PRO_BYTES_UNI;

    // Plane v = z0-2+s lives in p slot s mod 6; the b plane of step t and its mbarrier in slot t mod 6.
    auto slotP = [&](int s) -> float* { return sm + C::OFF_P + s * C::P_PLANE; };
    auto slotB = [&](int s) -> float* { return sm + C::OFF_B + s * C::C_PLANE; };

    // ---- copy issue: the group of step t = p plane u+1 and b plane u (u = z0-1+t); J = t mod 6 ----
    auto issue = [&](int t, int J) {
        if (lane_id != 0 || warp_id >= (YMODE == 2 ? 7 : 4)) return;
        const int sp = (J + 2 >= R) ? J + 2 - R : J + 2, sb = J;
        uint64_t* bar = bars + J;
        if (tid == 0) mbar_expect_tx(bar, step_bytes);
        const int u = z0 - 1 + t;
        const int gz0 = wrap1(u, nz), gz1 = wrap1(u + 1, nz);
        if (YMODE == 0) {
            switch (warp_id) {
                case 0: tma_load_3d(slotP(sp), &maps.p_main, x0, y0 - 2, gz1, bar); break;
                case 1: tma_load_3d(slotP(sp) + C::P_HL, &maps.p_halo, xL, y0 - 2, gz1, bar); break;
                case 2: tma_load_3d(slotP(sp) + C::P_HR, &maps.p_halo, xR, y0 - 2, gz1, bar); break;
                case 3: tma_load_3d(slotB(sb), &maps.b, x0, y0 - 1, gz0, bar); break;
                default: break;
            }
        } else {
            const size_t pz0 = (size_t)gz0 * plane, pz1 = (size_t)gz1 * plane;
            switch (warp_id) {
                case 0: tma_load_3d(slotP(sp) + e_oP * C::TX, &maps.p_main, x0, e_yP, gz1, bar); break;
                case 1: tma_load_3d(slotP(sp) + C::P_HL + hs + e_oP * 4, &maps.p_halo, xL, e_yP, gz1, bar); break;
                case 2: tma_load_3d(slotP(sp) + C::P_HR + hs + e_oP * 4, &maps.p_halo, xR, e_yP, gz1, bar); break;
                case 3: tma_load_3d(slotB(sb) + e_oC * C::TX, &maps.b, x0, e_yC, gz0, bar); break;
                case 4: case 5: {   // the two wrapped p rows
                    const int r = warp_id - 4, j = e_pj0 + r;
                    const float* rb = a.src + pz1 + (size_t)(e_py0 + r) * nx;
                    float* d = slotP(sp);
                    bulk_g2s(d + j * C::TX, rb + x0, C::TX * 4u, bar);
                    bulk_g2s(d + C::P_HL + hs + j * 4, rb + xL, 16u, bar);
                    bulk_g2s(d + C::P_HR + hs + j * 4, rb + xR, 16u, bar);
                } break;
                case 6: bulk_g2s(slotB(sb) + e_cj * C::TX, a.b + pz0 + (size_t)e_cy * nx + x0, C::TX * 4u, bar); break;
                default: break;
            }
        }
    };

    // ---- prologue: barriers; p(z0-2), p(z0-1); the first PD step groups -------------------------
    if (tid == 0) {
        for (int i = 0; i <= R; ++i) mbar_init(bars + i, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    fence_async_smem();
    __syncthreads();
    {
        uint64_t* bar = bars + R;
        if (lane_id == 0) {
            if (tid == 0) mbar_expect_tx(bar, pro_bytes);
            const int pl = warp_id / 3, k = warp_id % 3;
            if (pl < 2) {
                const int gv = wrapi(z0 - 2 + pl, nz);
                if (YMODE == 0) {
                    if (k == 0) tma_load_3d(slotP(pl), &maps.p_main, x0, y0 - 2, gv, bar);
                    else if (k == 1) tma_load_3d(slotP(pl) + C::P_HL, &maps.p_halo, xL, y0 - 2, gv, bar);
                    else tma_load_3d(slotP(pl) + C::P_HR, &maps.p_halo, xR, y0 - 2, gv, bar);
                } else {
                    if (k == 0) tma_load_3d(slotP(pl) + e_oP * C::TX, &maps.p_main, x0, e_yP, gv, bar);
                    else if (k == 1) tma_load_3d(slotP(pl) + C::P_HL + hs + e_oP * 4, &maps.p_halo, xL, e_yP, gv, bar);
                    else tma_load_3d(slotP(pl) + C::P_HR + hs + e_oP * 4, &maps.p_halo, xR, e_yP, gv, bar);
                }
            } else if (YMODE == 2 && warp_id >= 6 && warp_id <= 7) {   // wrapped p rows of the two planes
                const int pl2 = warp_id - 6;
                for (int r = 0; r < 2; ++r) {
                    const int j = e_pj0 + r;
                    const float* rb = a.src + (size_t)wrapi(z0 - 2 + pl2, nz) * plane + (size_t)(e_py0 + r) * nx;
                    float* d = slotP(pl2);
                    bulk_g2s(d + j * C::TX, rb + x0, C::TX * 4u, bar);
                    bulk_g2s(d + C::P_HL + hs + j * 4, rb + xL, 16u, bar);
                    bulk_g2s(d + C::P_HR + hs + j * 4, rb + xR, 16u, bar);
                }
            }
        }
#pragma unroll
        for (int t = 0; t < PD; ++t)
            if (t < T) issue(t, t);
        mbar_wait(bar, 0);
    }


    const float wx = a.uni.ux, wy = a.uni.uy, wz = a.uni.uz;
    float acc_rr_out = 0.0f, acc_bb_out = 0.0f, acc_rr_out2 = 0.0f, acc_bb_out2 = 0.0f;   // NORM: per row
    if (warp_id < NMAIN) {
        // ---- main threads: one float4 group of TWO rows, a = 2 warp_id and b = a + 1 (phase-B row
        // indices 0 .. ROWS-1; the last warp's row b does not exist) -----------------------------
        const int lx = lane_id, ra = 2 * warp_id;
        const bool vb = (ra + 1 < C::ROWS);
        const int xl = x0 + 4 * lx;
        const int yla = y0 + ra - 1, ylb = yla + 1;
        const int gya = wrapi(yla, ny), gyb = wrapi(ylb, ny);
        const bool ca = (ra >= 1) && (ra <= C::TY) && (yla < ny);            // rows phase C writes out
        const bool cb = vb && (ra + 1 >= 1) && (ra + 1 <= C::TY) && (ylb < ny);
        const bool first_lane = (lx == 0), last_lane = (lx == C::LPR - 1);
        float* const pp = sm + C::OFF_P + (ra + 1) * C::TX + 4 * lx;         // row a's float4 in slot 0 (row b: + TX)
        const float* const ph = sm + C::OFF_P + (lx == 0 ? C::P_HL + 3 : C::P_HR) + hs + (ra + 1) * 4;  // x-halo cell (row b: + 4)
        const float* const pb = sm + C::OFF_B + ra * C::TX + 4 * lx;         // row a's b float4 in slot 0 (row b: + TX)
        float* dsta = a.dst + ((long long)gya * nx + xl + (long long)(z0 - 2) * plane);   // plane u-1
        float* dstb = a.dst + ((long long)gyb * nx + xl + (long long)(z0 - 2) * plane);
        const int par = (yla + (z0 - 1) + fc) & 1;   // row a updates cells (sel, sel+2), sel = par ^ (t & 1); row b the other two
        CFull Sc;      // the level's constants; only Sc.b changes
        Sc.lx = make_float4(wx, wx, wx, wx);
        Sc.lxh = wx;
        Sc.ly = Sc.lyh = make_float4(wy, wy, wy, wy);
        Sc.lz = Sc.lzh = make_float4(wz, wz, wz, wz);
        CPair Ka, Kb;  // coefficients of the cells phase C updates: constants, and two b values per row
        Ka.lxa0 = Ka.lxa1 = Ka.lxb0 = Ka.lxb1 = wx;
        Ka.lya = Ka.lyb = Ka.lyha = Ka.lyhb = wy;
        Ka.lza = Ka.lzb = Ka.lzha = Ka.lzhb = wz;
        Ka.ba = Ka.bb = 0.0f;
        Kb = Ka;
        // PRO: parents of the own float4 (two coarse cells) in coarse row gy/2 of coarse plane gz/2, and of
        // the x-halo cell (first / last lane)
        const int ncx = nx >> 1, cplane = ncx * (ny >> 1);
        const int xc = xl >> 1;
        // float offsets (coarse plane 0) of the parents of rows a-1, a, b, b+1 at the own float4
        const int em_o = (wrapi(yla - 1, ny) >> 1) * ncx + xc, ea_o = (gya >> 1) * ncx + xc;
        const int eb_o = (gyb >> 1) * ncx + xc, ep_o = (wrapi(ylb + 1, ny) >> 1) * ncx + xc;
        const int eh_d = ((first_lane ? wrapi(x0 - 1, nx) : wrapi(x0 + C::TX, nx)) >> 1) - xc;   // x-halo cell's parent
        const bool has_h = first_lane || last_lane;
        auto ld2 = [&](int o) { return __ldg(reinterpret_cast<const float2*>(a.e_c + o)); };
        auto add2 = [](float4& v, const float2 e) { v.x += e.x; v.y += e.x; v.z += e.y; v.w += e.y; };
        float2 Em = make_float2(0.f, 0.f), Ea = Em, Eb = Em, Ep = Em;   // parents in coarse plane gzs/2
        float2 Aa = Em, Ab = Em;                                        // rows a, b one coarse plane on
        float Ha = 0.0f, Hb = 0.0f;
        int gzs = wrap1(z0 - 1, nz);    // PRO: wrapped plane index of the step whose operands load_step fetches
        // what load_step will need for plane gzs: all of coarse plane gzs/2 (fetched when gzs is even:
        // the plane before was the last of its pair) or, gzs odd, rows a and b of the next coarse plane
        auto fetch_parents = [&](bool all) {
            if (all || !(gzs & 1)) {
                const int o = (gzs >> 1) * cplane;
                Em = ld2(o + em_o); Ea = ld2(o + ea_o); Eb = ld2(o + eb_o); Ep = ld2(o + ep_o);
                if (has_h) { Ha = __ldg(a.e_c + o + ea_o + eh_d); Hb = __ldg(a.e_c + o + eb_o + eh_d); }
            }
            if (gzs & 1) {
                const int o = (wrap1(gzs + 1, nz) >> 1) * cplane;
                Aa = ld2(o + ea_o); Ab = ld2(o + eb_o);
            }
        };
        // plane u-1 at the own positions (t = 0: source values), plane u-2 under the cells C updates
        float4 q1a = lds4(pp), q1b = lds4(pp + C::TX);
        if (PRO) {
            const int o = (wrapi(z0 - 2, nz) >> 1) * cplane;
            add2(q1a, ld2(o + ea_o)); add2(q1b, ld2(o + eb_o));
        }
        float z2a0 = 0.0f, z2a1 = 0.0f, z2b0 = 0.0f, z2b1 = 0.0f;
        float zsa0 = 0.0f, zsa1 = 0.0f, zsb0 = 0.0f, zsb1 = 0.0f;   // NORM (see sweep_body)
        float acc_rr = 0.0f, acc_bb = 0.0f, acc_rr2 = 0.0f, acc_bb2 = 0.0f;   // one pair of sums per ROW, as sweep_body keeps them
        // ring cursors: float offsets of planes u-1, u, u+1, of the b plane, the mbarrier and its parity
        int oM = 0, o0 = C::P_PLANE, oP = 2 * C::P_PLANE, ob = 0, jb = 0;
        uint32_t kpar = 0;
        // operands of phase B of the step to come, loaded in front of the barrier (source values no
        // other thread changes before it): rows above a / below b and the x-halo cells of plane u,
        // plane u+1 at the own positions, the right-hand side; plane u itself is last step's plane u+1
        float4 owna, ownb, ym, yp, zpa, zpb, ba, bb;
        float hva, hvb;
        auto load_step = [&]() {   // cursors already point at the step to come
            mbar_wait(bars + jb, kpar);
            ym = lds4(pp + o0 - C::TX);
            yp = lds4(pp + o0 + 2 * C::TX);
            zpa = lds4(pp + oP);
            zpb = lds4(pp + oP + C::TX);
            ba = lds4(pb + ob);
            bb = vb ? lds4(pb + ob + C::TX) : zero4();
            hva = ph[o0];
            hvb = ph[o0 + 4];
            if (PRO) {
                add2(ym, Em); add2(yp, Ep);
                hva += Ha; hvb += Hb;      // (only the first and the last lane use them)
                add2(zpa, (gzs & 1) ? Aa : Ea); add2(zpb, (gzs & 1) ? Ab : Eb);
                gzs = (gzs + 1 == nz) ? 0 : gzs + 1;
            }
        };
        owna = lds4(pp + o0);
        ownb = lds4(pp + o0 + C::TX);
        if (PRO) { fetch_parents(true); add2(owna, Ea); add2(ownb, Eb); }
        load_step();
        if (PRO) cta_sync();   // step 0 stores corrected float4s into rows other warps have just read

        // The last warp owns one row only (phase-B row 14, the ring row) and also updates the ring-1
        // CELLS x0-1 and x0+TX of all 15 rows (phase B only; lane = 2 row + side), as sweep_body's edge
        // warp does: its neighbours are second-colour cells, which phase B leaves alone.
        const bool rim = RIM && (warp_id == NMAIN - 1);
        const bool e_act = rim && lane_id < 2 * C::ROWS;
        const int e_side = lane_id & 1, e_r = (e_act ? (lane_id >> 1) : 0) + 1;
        const int e_xs = e_side ? x0 + C::TX : x0 - 1, e_yl = y0 + e_r - 2;
        const int e_pc = hs + (e_side ? C::P_HR + e_r * 4 : C::P_HL + e_r * 4 + 3);   // the edge cell
        const int e_xm = e_side ? e_r * C::TX + C::TX - 1 : e_pc - 1;               // its x neighbours
        const int e_xp = e_side ? e_pc + 1 : e_r * C::TX;
        const float* const e_bptr = a.b + (size_t)wrapi(e_yl, ny) * nx + wrapi(e_xs, nx);
        int e_gz = wrap1(z0 - 1, nz);
        float e_b = rim ? __ldg(e_bptr + (size_t)e_gz * plane) : 0.0f, e_bn = e_b;
        const int e_col0 = (e_xs + e_yl + (z0 - 1)) & 1;   // colour of the edge cell in plane u at t = 0
        const float e_D = diag6(wx, wx, wy, wy, wz, wz);
        float* const Pbase = sm + C::OFF_P;

        auto step = [&](auto Sc_, const int t) {
            constexpr int SA = decltype(Sc_)::value, SB = SA ^ 1;
            const float4 cym = lds4(pp + oM - C::TX);       // plane u-1, B-updated: row above a
            const float4 cyp = lds4(pp + oM + 2 * C::TX);   //                       row below b
            const float hca = ph[oM], hcb = ph[oM + 4];
            float xma = __shfl_up_sync(0xffffffffu, owna.w, 1);
            float xpa = __shfl_down_sync(0xffffffffu, owna.x, 1);
            float xmb = __shfl_up_sync(0xffffffffu, ownb.w, 1);
            float xpb = __shfl_down_sync(0xffffffffu, ownb.x, 1);
            float cxma = __shfl_up_sync(0xffffffffu, q1a.w, 1);
            float cxpa = __shfl_down_sync(0xffffffffu, q1a.x, 1);
            float cxmb = __shfl_up_sync(0xffffffffu, q1b.w, 1);
            float cxpb = __shfl_down_sync(0xffffffffu, q1b.x, 1);
            xma = first_lane ? hva : xma;   xpa = last_lane ? hva : xpa;
            xmb = first_lane ? hvb : xmb;   xpb = last_lane ? hvb : xpb;
            cxma = first_lane ? hca : cxma; cxpa = last_lane ? hca : cxpa;
            cxmb = first_lane ? hcb : cxmb; cxpb = last_lane ? hcb : cxpb;
            if (NORM) {
                // residual of the SOURCE iterate on the eight cells of plane u (see sweep_body): plane u-1
                // under a row's second-colour cells comes from zs*, elsewhere q1* still holds source values
                const float a0 = SA ? zsa0 : q1a.x, a1 = SA ? q1a.y : zsa0, a2 = SA ? zsa1 : q1a.z, a3 = SA ? q1a.w : zsa1;
                const float b0 = SB ? zsb0 : q1b.x, b1 = SB ? q1b.y : zsb0, b2 = SB ? zsb1 : q1b.z, b3 = SB ? q1b.w : zsb1;
                const float A0 = apply7(owna.x, wx, wx, wy, wy, wz, wz, xma, owna.y, ym.x, ownb.x, a0, zpa.x);
                const float A1 = apply7(owna.y, wx, wx, wy, wy, wz, wz, owna.x, owna.z, ym.y, ownb.y, a1, zpa.y);
                const float A2 = apply7(owna.z, wx, wx, wy, wy, wz, wz, owna.y, owna.w, ym.z, ownb.z, a2, zpa.z);
                const float A3 = apply7(owna.w, wx, wx, wy, wy, wz, wz, owna.z, xpa, ym.w, ownb.w, a3, zpa.w);
                const float B0 = apply7(ownb.x, wx, wx, wy, wy, wz, wz, xmb, ownb.y, owna.x, yp.x, b0, zpb.x);
                const float B1 = apply7(ownb.y, wx, wx, wy, wy, wz, wz, ownb.x, ownb.z, owna.y, yp.y, b1, zpb.y);
                const float B2 = apply7(ownb.z, wx, wx, wy, wy, wz, wz, ownb.y, ownb.w, owna.z, yp.z, b2, zpb.z);
                const float B3 = apply7(ownb.w, wx, wx, wy, wy, wz, wz, ownb.z, xpb, owna.w, yp.w, b3, zpb.w);
                if (t >= 1 && t <= T - 2) {   // every cell of a lean tile is active
                    if (ca) {
                        const float r0 = ba.x - A0, r1 = ba.y - A1, r2 = ba.z - A2, r3 = ba.w - A3;
                        acc_rr = __fadd_rn(acc_rr, __fadd_rn(__fadd_rn(__fmul_rn(r0, r0), __fmul_rn(r1, r1)),
                                                             __fadd_rn(__fmul_rn(r2, r2), __fmul_rn(r3, r3))));
                        if (NORM == 2)
                            acc_bb = __fadd_rn(acc_bb, __fadd_rn(__fadd_rn(__fmul_rn(ba.x, ba.x), __fmul_rn(ba.y, ba.y)),
                                                                 __fadd_rn(__fmul_rn(ba.z, ba.z), __fmul_rn(ba.w, ba.w))));
                    }
                    if (cb) {
                        const float r0 = bb.x - B0, r1 = bb.y - B1, r2 = bb.z - B2, r3 = bb.w - B3;
                        acc_rr2 = __fadd_rn(acc_rr2, __fadd_rn(__fadd_rn(__fmul_rn(r0, r0), __fmul_rn(r1, r1)),
                                                               __fadd_rn(__fmul_rn(r2, r2), __fmul_rn(r3, r3))));
                        if (NORM == 2)
                            acc_bb2 = __fadd_rn(acc_bb2, __fadd_rn(__fadd_rn(__fmul_rn(bb.x, bb.x), __fmul_rn(bb.y, bb.y)),
                                                                 __fadd_rn(__fmul_rn(bb.z, bb.z), __fmul_rn(bb.w, bb.w))));
                    }
                }
                zsa0 = SA ? owna.y : owna.x; zsa1 = SA ? owna.w : owna.z;
                zsb0 = SB ? ownb.y : ownb.x; zsb1 = SB ? ownb.w : ownb.z;
            }
            // phase B on plane u: row a's lower y neighbour is row b and vice versa (source values)
            Sc.b = ba;
            const float4 nwa = update_pair_full<SA>(xma, owna, xpa, ym, ownb, q1a, zpa, Sc, omega);
            float4 nwb = ownb, ncb = q1b;
            if (vb) {   // (warp-uniform: only the last warp has no row b)
                Sc.b = bb;
                nwb = update_pair_full<SB>(xmb, ownb, xpb, owna, yp, q1b, zpb, Sc, omega);
            }
            // phase C on plane u-1: the neighbouring row of the pair is q1 of the other row (phase-B
            // results of the step before, in registers)
            const float4 nca = update_pair_carried<SA>(cxma, q1a, cxpa, cym, q1b, z2a0, z2a1, nwa, Ka, omega);
            if (vb) ncb = update_pair_carried<SB>(cxmb, q1b, cxpb, q1a, cyp, z2b0, z2b1, nwb, Kb, omega);
            // the next step's C works on the other two cells of plane u
            if (SA) { Ka.ba = ba.x; Ka.bb = ba.z; z2a0 = q1a.x; z2a1 = q1a.z; Kb.ba = bb.y; Kb.bb = bb.w; z2b0 = q1b.y; z2b1 = q1b.w; }
            else { Ka.ba = ba.y; Ka.bb = ba.w; z2a0 = q1a.y; z2a1 = q1a.w; Kb.ba = bb.x; Kb.bb = bb.z; z2b0 = q1b.x; z2b1 = q1b.z; }
            *reinterpret_cast<float4*>(pp + o0) = nwa;
            if (vb) *reinterpret_cast<float4*>(pp + o0 + C::TX) = nwb;
            if (t >= 2) {
                if (ca) *reinterpret_cast<float4*>(dsta) = nca;
                if (cb) *reinterpret_cast<float4*>(dstb) = ncb;
            }
            q1a = nwa; q1b = nwb;
            owna = zpa; ownb = zpb;
            dsta += plane; dstb += plane;
            if (rim) {   // the ring-1 cells of plane u
                if (t + 1 < T) {   // the next plane's right-hand side, one step ahead
                    e_gz = (e_gz + 1 == nz) ? 0 : e_gz + 1;
                    e_bn = __ldg(e_bptr + (size_t)e_gz * plane);
                }
                if (e_act && ((e_col0 ^ t) & 1) == fc) {
                    float* P0 = Pbase + o0;
                    const float pc = P0[e_pc];
                    const float Ap = apply7(pc, wx, wx, wy, wy, wz, wz, P0[e_xm], P0[e_xp], P0[e_pc - 4],
                                            P0[e_pc + 4], Pbase[oM + e_pc], Pbase[oP + e_pc]);
                    P0[e_pc] = relax(pc, e_b, Ap, e_D, omega);
                }
                e_b = e_bn;
            }
            // rotate the cursors to step t+1 and load its operands in front of the barrier
            const int jb_issue = jb + PD >= R ? jb + PD - R : jb + PD;
            oM = o0; o0 = oP;
            oP = (oP == (R - 1) * C::P_PLANE) ? 0 : oP + C::P_PLANE;
            ob = (ob == (R - 1) * C::C_PLANE) ? 0 : ob + C::C_PLANE;
            if (++jb == R) { jb = 0; kpar ^= 1u; }
            if (PRO && t + 1 < T) fetch_parents(false);
            if (t + 1 < T) load_step();
            fence_async_smem();  // order this thread's smem writes before later TMA overwrites
            cta_sync();
            if (t + PD < T) issue(t + PD, jb_issue);
        };
        auto run = [&](auto Pc) {
            constexpr int P = decltype(Pc)::value;
            for (int t = 0;;) {
                step(std::integral_constant<int, P>(), t); if (++t == T) break;
                step(std::integral_constant<int, P ^ 1>(), t); if (++t == T) break;
            }
        };
        if (par) run(std::integral_constant<int, 1>());
        else run(std::integral_constant<int, 0>());
        if (NORM) { acc_rr_out = acc_rr; acc_bb_out = acc_bb; acc_rr_out2 = acc_rr2; acc_bb_out2 = acc_bb2; }
    } else {   // (RIM == false only)
        // ---- edge warp: ring-1 cells x0-1 and x0+TX of every row, phase B only ----------------
        const int el = lane_id;
        const bool e_act = el < 2 * C::ROWS;
        const int side = el & 1, ery = e_act ? (el >> 1) : 0;
        const int xs = side ? x0 + C::TX : x0 - 1;
        const int eyl = y0 + ery - 1;
        const int r = ery + 1;
        const int pc_off = hs + (side ? C::P_HR + r * 4 : C::P_HL + r * 4 + 3);   // the edge cell
        const int xm_off = side ? r * C::TX + C::TX - 1 : pc_off - 1;             // its x neighbours
        const int xp_off = side ? pc_off + 1 : r * C::TX;
        float* const P = sm + C::OFF_P;
        const float* bptr = a.b + (size_t)wrapi(eyl, ny) * nx + wrapi(xs, nx);   // b of the edge cell, plane by plane
        int gz = wrap1(z0 - 1, nz);
        float bc_ = __ldg(bptr + (size_t)gz * plane), bn = bc_;
        const int ecol0 = (xs + eyl + (z0 - 1)) & 1;   // colour of the edge cell in plane u at t = 0
        const float D = diag6(wx, wx, wy, wy, wz, wz);
        int oM = 0, o0 = C::P_PLANE, oP = 2 * C::P_PLANE, jb = 0;
        uint32_t kpar = 0;
        // PRO: parents of the edge cell and its six neighbours; the neighbour INSIDE the tile is a cell a
        // main thread stores to during the step, so it is read in front of the barrier
        const int ncx = nx >> 1, cplane = ncx * (ny >> 1);
        const int in_off = side ? xm_off : xp_off;
        const int c0 = wrapi(xs, nx) >> 1;                                   // coarse columns of the cell,
        const int cin = wrapi(side ? xs - 1 : xs + 1, nx) >> 1;              // its neighbour inside the tile
        const int cout = wrapi(side ? xs + 1 : xs - 1, nx) >> 1;             // and the one outside
        const int r0 = (wrapi(eyl, ny) >> 1) * ncx, rl = (wrapi(eyl - 1, ny) >> 1) * ncx, rh = (wrapi(eyl + 1, ny) >> 1) * ncx;
        int gzu = wrap1(z0 - 1, nz);   // wrapped plane index of step t
        float xin = 0.0f;
        if (PRO) {
            mbar_wait(bars, 0);
            xin = P[o0 + in_off];
            cta_sync();   // (the main threads' barrier in front of step 0)
        }
        for (int t = 0; t < T; ++t) {
            if (t + 1 < T) {   // the next plane's right-hand side, one step ahead
                gz = (gz + 1 == nz) ? 0 : gz + 1;
                bn = __ldg(bptr + (size_t)gz * plane);
            }
            const bool upd = e_act && ((ecol0 ^ t) & 1) == fc;
            float e_c0 = 0.f, e_in = 0.f, e_out = 0.f, e_yl = 0.f, e_yh = 0.f, e_zl = 0.f, e_zh = 0.f;
            if (PRO && upd) {   // the seven parents, fetched before the wait for the plane
                const int k0 = (gzu >> 1) * cplane;
                const int kl = ((gzu == 0 ? nz - 1 : gzu - 1) >> 1) * cplane, kh = ((gzu + 1 == nz ? 0 : gzu + 1) >> 1) * cplane;
                e_c0 = __ldg(a.e_c + k0 + r0 + c0);
                e_in = __ldg(a.e_c + k0 + r0 + cin);
                e_out = __ldg(a.e_c + k0 + r0 + cout);
                e_yl = __ldg(a.e_c + k0 + rl + c0);
                e_yh = __ldg(a.e_c + k0 + rh + c0);
                e_zl = __ldg(a.e_c + kl + r0 + c0);
                e_zh = __ldg(a.e_c + kh + r0 + c0);
            }
            mbar_wait(bars + jb, kpar);
            if (upd) {
                float* P0 = P + o0;
                if (PRO) {
                    const float pc = P0[pc_off] + e_c0;
                    const float vin = xin + e_in;
                    const float vout = P0[side ? xp_off : xm_off] + e_out;
                    const float Ap = apply7(pc, wx, wx, wy, wy, wz, wz, side ? vin : vout, side ? vout : vin,
                                            P0[pc_off - 4] + e_yl, P0[pc_off + 4] + e_yh,
                                            P[oM + pc_off] + e_zl, P[oP + pc_off] + e_zh);
                    P0[pc_off] = relax(pc, bc_, Ap, D, omega);
                } else {
                    const float pc = P0[pc_off];
                    const float Ap = apply7(pc, wx, wx, wy, wy, wz, wz, P0[xm_off], P0[xp_off], P0[pc_off - 4],
                                            P0[pc_off + 4], P[oM + pc_off], P[oP + pc_off]);
                    P0[pc_off] = relax(pc, bc_, Ap, D, omega);
                }
            }
            if (PRO && t + 1 < T) {   // the in-tile neighbour of the next step (plane u+1 has landed): still a source value
                xin = P[oP + in_off];
                gzu = gzu + 1 == nz ? 0 : gzu + 1;
            }
            fence_async_smem();
            cta_sync();
            bc_ = bn;
            oM = o0; o0 = oP;
            oP = (oP == (R - 1) * C::P_PLANE) ? 0 : oP + C::P_PLANE;
            if (++jb == R) { jb = 0; kpar ^= 1u; }
        }
    }
    if (NORM) norm_finish<NORM>(a, tile, acc_rr_out, acc_bb_out, acc_rr_out2, acc_bb_out2, true, sm);
}

}  // namespace gmgf

// sweep_lean.cuh -- lean_body: the fused red+black sweep of a tile whose coefficients are the
// level's constants (uniform.cuh), written for the kernel that runs ONLY such tiles
// (k_rb_sweep_lean: 64 registers per thread, two CTAs per SM).  Same schedule as sweep_body --
// per z step B(u) on tile + ring 1 in shared memory, C(u-1) streamed to the destination, one CTA
// barrier, TMA boxes PD steps ahead -- and the same update_pair_full / update_pair_carried calls on
// the same operands, so every cell gets the bits sweep_body gives it (tests compare the two).
// What differs is the bookkeeping around the arithmetic, which is most of the instruction stream
// once the coefficient loads are gone: every ring (p planes, b planes, mbarriers) has the SAME
// period 6 and the z loop is unrolled six times, so ring slots, mbarrier indices and the colour
// parity of a step are compile-time constants -- no ring cursors, no per-step branch on the
// parity, no address arithmetic in the loop -- and a step's operands are loaded at its top (the
// second CTA of the SM covers the shared-memory latency), which keeps the live state under the
// register limit.  Included by kernels_sweep.cu.
#pragma once

namespace gmgf {

template <class C, int YMODE, int NORM>
__device__ __forceinline__ void lean_body(const BulkArgs& a, const BulkMaps& allmaps, const int tile) {
    static_assert(C::LEAN && C::PD == 4 && C::NP == 6 && C::NC == 6 && C::NB == 6, "rings of period 6");
    static_assert(YMODE == 0 || YMODE == 2, "box-fed tiles only");
    constexpr int R = 6, PD = C::PD;
    extern __shared__ __align__(1024) float sm[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(sm + C::FLOATS);  // [0..6) step groups, [6] prologue
    const LevelGeom& g = a.g;
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const int plane = nx * ny;
    const int tid = threadIdx.x;
    const int warp_id = tid >> 5, lane_id = tid & 31;
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
        if (lane_id != 0 || warp_id >= (YMODE == 2 ? 13 : 4)) return;
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
                case 7: case 8: {   // the two wrapped p rows
                    const int r = warp_id - 7, j = e_pj0 + r;
                    const float* rb = a.src + pz1 + (size_t)(e_py0 + r) * nx;
                    float* d = slotP(sp);
                    bulk_g2s(d + j * C::TX, rb + x0, C::TX * 4u, bar);
                    bulk_g2s(d + C::P_HL + hs + j * 4, rb + xL, 16u, bar);
                    bulk_g2s(d + C::P_HR + hs + j * 4, rb + xR, 16u, bar);
                } break;
                case 12: bulk_g2s(slotB(sb) + e_cj * C::TX, a.b + pz0 + (size_t)e_cy * nx + x0, C::TX * 4u, bar); break;
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
            } else if (YMODE == 2 && warp_id >= 7 && warp_id <= 10) {   // wrapped p rows of the two planes
                const int pl2 = (warp_id - 7) / 2, r = (warp_id - 7) & 1, j = e_pj0 + r;
                const float* rb = a.src + (size_t)wrapi(z0 - 2 + pl2, nz) * plane + (size_t)(e_py0 + r) * nx;
                float* d = slotP(pl2);
                bulk_g2s(d + j * C::TX, rb + x0, C::TX * 4u, bar);
                bulk_g2s(d + C::P_HL + hs + j * 4, rb + xL, 16u, bar);
                bulk_g2s(d + C::P_HR + hs + j * 4, rb + xR, 16u, bar);
            }
        }
#pragma unroll
        for (int t = 0; t < PD; ++t)
            if (t < T) issue(t, t);
        mbar_wait(bar, 0);
    }

    const float wx = a.uni.ux, wy = a.uni.uy, wz = a.uni.uz;
    float acc_rr_out = 0.0f, acc_bb_out = 0.0f;   // NORM: the thread's partial sums
    if (tid < C::MAIN) {
        // ---- main threads: one float4 group of one row ---------------------------------------
        const int lx = lane_id, ry = warp_id;
        const int xl = x0 + 4 * lx;
        const int yl = y0 + ry - 1;
        const int gy = wrapi(yl, ny);
        const bool row_c = (ry >= 1) && (ry <= C::TY) && (yl < ny);
        const bool first_lane = (lx == 0), last_lane = (lx == C::LPR - 1);
        const float* const pp = sm + C::OFF_P + (ry + 1) * C::TX + 4 * lx;         // own float4, slot 0
        const float* const ph = sm + C::OFF_P + (lx == 0 ? C::P_HL + 3 : C::P_HR) + hs + (ry + 1) * 4;  // x-halo cell
        const float* const pb = sm + C::OFF_B + ry * C::TX + 4 * lx;               // own b float4, slot 0
        float* dst_ptr = a.dst + ((long long)gy * nx + xl + (long long)(z0 - 2) * plane);  // plane u-1
        const int par = (yl + (z0 - 1) + fc) & 1;   // cells (sel, sel+2) are updated, sel = par ^ (t & 1)
        CFull Sc;      // the level's constants; only Sc.b changes from step to step
        Sc.lx = make_float4(wx, wx, wx, wx);
        Sc.lxh = wx;
        Sc.ly = Sc.lyh = make_float4(wy, wy, wy, wy);
        Sc.lz = Sc.lzh = make_float4(wz, wz, wz, wz);
        CPair K;       // coefficients of the two cells C updates: constants, and the two b values
        K.lxa0 = K.lxa1 = K.lxb0 = K.lxb1 = wx;
        K.lya = K.lyb = K.lyha = K.lyhb = wy;
        K.lza = K.lzb = K.lzha = K.lzhb = wz;
        K.ba = K.bb = 0.0f;
        float4 q1 = lds4(pp);                       // plane u-1 at the own position (t = 0: source values)
        float z2a = 0.0f, z2b = 0.0f;               // plane u-2 under the cells C updates
        float zs_a = 0.0f, zs_b = 0.0f, acc_rr = 0.0f, acc_bb = 0.0f;   // NORM (see sweep_body)

        // Ring cursors (float offsets of planes u-1, u, u+1 in the p ring, of the b plane, the
        // mbarrier index and its phase parity), rotated once per step.  The loop is unrolled TWICE so
        // that the colour parity S of a step is a compile-time constant; unrolling over the ring
        // period as well (slots as immediates) was measured slower: 20 KB of loop body miss the
        // instruction cache (stall reason no_instruction 0.1 -> 3.7 per issued instruction).
        int oM = 0, o0 = C::P_PLANE, oP = 2 * C::P_PLANE, ob = 0, jb = 0;
        uint32_t kpar = 0;
        // NORM: the residual of the SOURCE iterate also reads the FIRST-colour cells of the rows above
        // and below and of the x-halo column in plane u -- cells other warps update during step u.
        // Those three operands are therefore loaded in front of the barrier of step u-1 (as sweep_body
        // loads all of them); the plain sweep reads second-colour neighbours only and needs no such care.
        float4 ymn = zero4(), ypn = zero4();
        float hvn = 0.0f;
        if (NORM) {
            mbar_wait(bars, 0);
            ymn = lds4(pp + o0 - C::TX);
            ypn = lds4(pp + o0 + C::TX);
            hvn = ph[o0];
        }
        auto step = [&](auto Sc_, const int t) {
            constexpr int S = decltype(Sc_)::value;
            mbar_wait(bars + jb, kpar);
            Sc.b = lds4(pb + ob);
            const float4 own = lds4(pp + o0);
            const float4 ym = NORM ? ymn : lds4(pp + o0 - C::TX);
            const float4 yp = NORM ? ypn : lds4(pp + o0 + C::TX);
            const float4 zp = lds4(pp + oP);
            const float hvB = NORM ? hvn : ph[o0];
            const float4 cym = lds4(pp + oM - C::TX);   // plane u-1, B-updated rows above / below
            const float4 cyp = lds4(pp + oM + C::TX);
            const float hvC = ph[oM];
            float xm = __shfl_up_sync(0xffffffffu, own.w, 1);
            float xp = __shfl_down_sync(0xffffffffu, own.x, 1);
            float cxm = __shfl_up_sync(0xffffffffu, q1.w, 1);
            float cxp = __shfl_down_sync(0xffffffffu, q1.x, 1);
            xm = first_lane ? hvB : xm;
            xp = last_lane ? hvB : xp;
            cxm = first_lane ? hvC : cxm;
            cxp = last_lane ? hvC : cxp;
            if (NORM) {
                const float s0 = S ? zs_a : q1.x, s1 = S ? q1.y : zs_a;
                const float s2 = S ? zs_b : q1.z, s3 = S ? q1.w : zs_b;
                const float A0 = apply7(own.x, wx, wx, wy, wy, wz, wz, xm, own.y, ym.x, yp.x, s0, zp.x);
                const float A1 = apply7(own.y, wx, wx, wy, wy, wz, wz, own.x, own.z, ym.y, yp.y, s1, zp.y);
                const float A2 = apply7(own.z, wx, wx, wy, wy, wz, wz, own.y, own.w, ym.z, yp.z, s2, zp.z);
                const float A3 = apply7(own.w, wx, wx, wy, wy, wz, wz, own.z, xp, ym.w, yp.w, s3, zp.w);
                if (row_c && t >= 1 && t <= T - 2) {   // every cell of a lean tile is active
                    const float r0 = Sc.b.x - A0, r1 = Sc.b.y - A1, r2 = Sc.b.z - A2, r3 = Sc.b.w - A3;
                    acc_rr = __fadd_rn(acc_rr, __fadd_rn(__fadd_rn(__fmul_rn(r0, r0), __fmul_rn(r1, r1)),
                                                         __fadd_rn(__fmul_rn(r2, r2), __fmul_rn(r3, r3))));
                    if (NORM == 2)
                        acc_bb = __fadd_rn(acc_bb, __fadd_rn(__fadd_rn(__fmul_rn(Sc.b.x, Sc.b.x), __fmul_rn(Sc.b.y, Sc.b.y)),
                                                             __fadd_rn(__fmul_rn(Sc.b.z, Sc.b.z), __fmul_rn(Sc.b.w, Sc.b.w))));
                }
                zs_a = S ? own.y : own.x;
                zs_b = S ? own.w : own.z;
            }
            const float4 nw = update_pair_full<S>(xm, own, xp, ym, yp, q1, zp, Sc, omega);
            const float4 nc = update_pair_carried<S>(cxm, q1, cxp, cym, cyp, z2a, z2b, nw, K, omega);
            // the next step's C works on the other two cells of plane u
            if (S) { K.ba = Sc.b.x; K.bb = Sc.b.z; z2a = q1.x; z2b = q1.z; }
            else { K.ba = Sc.b.y; K.bb = Sc.b.w; z2a = q1.y; z2b = q1.w; }
            *reinterpret_cast<float4*>(const_cast<float*>(pp) + o0) = nw;
            if (t >= 2 && row_c) *reinterpret_cast<float4*>(dst_ptr) = nc;
            q1 = nw;
            dst_ptr += plane;
            if (NORM && t + 1 < T) {   // next step's rows above / below and halo cell: still source values
                const int jn = (jb + 1 == R) ? 0 : jb + 1;
                mbar_wait(bars + jn, jn == 0 ? kpar ^ 1u : kpar);
                ymn = lds4(pp + oP - C::TX);
                ypn = lds4(pp + oP + C::TX);
                hvn = ph[oP];
            }
            fence_async_smem();  // order this thread's smem writes before later TMA overwrites
            cta_sync();
            if (t + PD < T) issue(t + PD, jb + PD >= R ? jb + PD - R : jb + PD);
            oM = o0; o0 = oP;
            oP = (oP == (R - 1) * C::P_PLANE) ? 0 : oP + C::P_PLANE;
            ob = (ob == (R - 1) * C::C_PLANE) ? 0 : ob + C::C_PLANE;
            if (++jb == R) { jb = 0; kpar ^= 1u; }
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
        if (NORM) { acc_rr_out = acc_rr; acc_bb_out = acc_bb; }
    } else {
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
        for (int t = 0; t < T; ++t) {
            if (t + 1 < T) {   // the next plane's right-hand side, one step ahead
                gz = (gz + 1 == nz) ? 0 : gz + 1;
                bn = __ldg(bptr + (size_t)gz * plane);
            }
            mbar_wait(bars + jb, kpar);
            if (e_act && ((ecol0 ^ t) & 1) == fc) {
                float* P0 = P + o0;
                const float pc = P0[pc_off];
                const float Ap = apply7(pc, wx, wx, wy, wy, wz, wz, P0[xm_off], P0[xp_off], P0[pc_off - 4],
                                        P0[pc_off + 4], P[oM + pc_off], P[oP + pc_off]);
                P0[pc_off] = relax(pc, bc_, Ap, D, omega);
            }
            fence_async_smem();
            cta_sync();
            bc_ = bn;
            oM = o0; o0 = oP;
            oP = (oP == (R - 1) * C::P_PLANE) ? 0 : oP + C::P_PLANE;
            if (++jb == R) { jb = 0; kpar ^= 1u; }
        }
    }
    if (NORM) norm_finish<NORM>(a, tile, acc_rr_out, acc_bb_out, 0.0f, 0.0f, false, sm);
}

}  // namespace gmgf

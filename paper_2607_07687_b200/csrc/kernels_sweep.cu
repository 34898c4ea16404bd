// kernels_sweep.cu -- k_rb_sweep_bulk: the fused red+black Gauss-Seidel sweep of the big levels
// (PAPER.md:43 S3.1; readings O3, O8), fed by the Tensor Memory Accelerator
// (cp.async.bulk.tensor + mbarrier, SASS UTMALDG) instead of register loads.
//
// A CTA owns a 128 x TY tile and marches along z.  EVERY input stream (source iterate p,
// right-hand side b, the three face-coefficient arrays) arrives in shared memory as one TMA box
// per stream and plane (128 x rows floats, 5.6-6.6 KB; plus two 4-float-wide halo boxes for p),
// issued PD steps ahead of use: 7 TMA operations per step, no registers tied up by loads in
// flight.  Step u, per thread (one float4 of one row):
//     B(u)    first-colour update of plane u on tile + ring 1, in place in shared memory;
//     C(u-1)  second-colour update of plane u-1, streamed to the destination array;
//     loads of B(u+1)'s operands;  barrier;  issue the copies of step u+PD.
// B and C sit between the same two barriers because of what each one reads.  A first-colour
// cell has only second-colour neighbours, and those keep their SOURCE value in shared memory
// (phase C writes to the destination array only): B(u) depends on no other thread's update,
// so its operands can be loaded ahead of the barrier.  C(u-1) needs the B(u-1) results of the
// rows above and below (other warps: behind the barrier of step u-1) and, at its own position,
// the planes u-2, u-1, u this thread itself produced -- kept in registers.
// Periodic wrap in x = the halo boxes are fetched at wrapped coordinates; in z = a wrapped plane
// coordinate; tiles touching the y boundary (2 tile rows of ~80 at 1024^3) take a row-by-row
// bulk-copy path (cp.async.bulk, UBLKCP) with wrapped row addresses.  Neumann walls = zeroed
// coefficients.  Every shared-memory cell holds the periodic image of its cell, as in k_rb_sweep.
#include <cuda.h>

#include <map>
#include <mutex>
#include <tuple>
#include <type_traits>

#include "fused_common.cuh"
#include "uniform.cuh"

namespace gmgf {
// LEAN_: the layout of the kernel that runs ONLY the lean path (uniform.cuh): no coefficient rings,
// 102 KB instead of 190 KB, so that two CTAs share an SM.
template <int TY_, int PD_, bool LEAN_ = false>
struct BulkCfg {
    static constexpr int TX = 128, TY = TY_, PD = PD_;
    static constexpr bool LEAN = LEAN_;
    static constexpr int LPR = 32;
    static constexpr int ROWS = TY + 2;          // rows running phase B (tile + ring 1)
    static constexpr int MAIN = LPR * ROWS;
    static constexpr int THREADS = MAIN + 32;    // + one edge warp
    static constexpr int SH = TY + 4;            // rows of a p plane (halo 2)
    // Ring depths.  G(u+PD) is issued behind the barrier of step u and may overwrite what step u
    // was the last to read AND to use: p plane u-1 (rows above/below for C(u-1)), Lz plane u,
    // Lx/Ly/b plane u.  Still to come are planes u..u+PD (+1 for p, whose group runs one ahead).
    static constexpr int NP = PD + 2;
    static constexpr int NZ = PD + 1;
    // (the lean layout gives every ring the period of the p ring: one cursor rotation serves all, sweep_lean2.cuh)
    static constexpr int NC = LEAN ? PD + 2 : PD;
    static constexpr int NB = LEAN ? PD + 2 : PD + 1;   // mbarriers of the step groups
    static constexpr int HPAD = (SH * 4 + 31) / 32 * 32;  // one halo column group, padded to 128 B
    static constexpr int P_HL = SH * TX;                   // p slot: main | left halo | right halo
    static constexpr int P_HR = P_HL + HPAD;
    static constexpr int P_PLANE = P_HR + HPAD;
    static constexpr int C_PLANE = ROWS * TX;        // Lx, Lz, b
    static constexpr int Y_PLANE = (ROWS + 1) * TX;  // Ly (needs the row above too)
    static constexpr int OFF_P = 0;
    static constexpr int OFF_LZ = OFF_P + NP * P_PLANE;
    static constexpr int OFF_LX = OFF_LZ + (LEAN ? 0 : NZ * C_PLANE);
    static constexpr int OFF_LY = OFF_LX + (LEAN ? 0 : NC * C_PLANE);
    static constexpr int OFF_B = OFF_LY + (LEAN ? 0 : NC * Y_PLANE);
    static constexpr int FLOATS = OFF_B + NC * C_PLANE;
    static constexpr int NROWCOPY = SH + 4 * ROWS + 1;  // rows per step on the row-copy path
    static constexpr size_t SMEM = (size_t)FLOATS * sizeof(float) + 16 * sizeof(uint64_t) + (size_t)NROWCOPY * 16;
    static constexpr uint32_t STEP_BYTES =
        (uint32_t)(SH * TX + 2 * SH * 4 + 3 * ROWS * TX + (ROWS + 1) * TX) * 4u;
    static constexpr uint32_t PRO_BYTES = (uint32_t)(2 * (SH * TX + 2 * SH * 4) + ROWS * TX) * 4u;
    // lean path (uniform.cuh): only the p and b streams are copied
    static constexpr uint32_t STEP_BYTES_UNI = (uint32_t)(SH * TX + 2 * SH * 4 + ROWS * TX) * 4u;
    static constexpr uint32_t PRO_BYTES_UNI = (uint32_t)(2 * (SH * TX + 2 * SH * 4)) * 4u;
    static_assert(2 * ROWS <= 32 && NB <= 8 && THREADS / 32 >= 7, "tile shape");
    static_assert(SMEM <= 227 * 1024, "shared memory");
};

struct BulkArgs {
    LevelGeom g;
    const float* L;
    const float* src;
    float* dst;
    const float* b;
    const float* omega;
    int first_colour;
    int zchunk;
    int tiles_x, tiles_y;
    int ntiles;            // tiles of the level = tickets of a norm-carrying sweep (lean + remaining kernel)
    // NORM variant: sums over the tile cells of r^2 (r = b - A src on active cells: the residual of
    // the SOURCE iterate) and of b^2 on active cells, into rb.sc->red[slot_rr / slot_ref]
    ReduceBuf rb;
    int slot_rr, slot_ref;
    const int* run_flag;   // != nullptr: the kernel does nothing unless *run_flag != 0
    UniArgs uni;           // uniform bricks of the level (uniform.cuh); brick == nullptr: disabled
    const float* e_c;      // lean kernel, PRO: the coarse correction to be added to src on the fly
};

struct alignas(64) MapSet {
    CUtensorMap p_main, p_halo, lz, lx, ly, b;
};
// [0] full boxes (tiles inside the domain in y; with a Neumann y axis every tile: rows outside
// arrive as zeros, which is what a wall needs); [1] the FIRST tile row of a periodic y axis: boxes
// that start at y = 0; [2] its FINAL tile row: boxes that end at y = ny - 1.  The few wrapped rows
// of [1] and [2] come as row copies (YMODE 2 below).
struct alignas(64) BulkMaps {
    MapSet m[3];
};

struct CFull {  // coefficients of the four own cells in one plane (lower faces, the y/z faces above, b)
    float4 lx, ly, lyh, lz, lzh, b;
    float lxh;  // the x face above the fourth cell
};

struct CPair {  // coefficients of the two cells (a, b) = (S, S+2) phase C updates, carried one step
    float lxa0, lxa1, lxb0, lxb1, lya, lyb, lyha, lyhb, lza, lzb, lzha, lzhb, ba, bb;
};

template <int S>
__device__ __forceinline__ void pick_pair(const CFull& c, CPair& k) {
    if (S == 0) {
        k.lxa0 = c.lx.x; k.lxa1 = c.lx.y; k.lxb0 = c.lx.z; k.lxb1 = c.lx.w;
        k.lya = c.ly.x; k.lyb = c.ly.z; k.lyha = c.lyh.x; k.lyhb = c.lyh.z;
        k.lza = c.lz.x; k.lzb = c.lz.z; k.lzha = c.lzh.x; k.lzhb = c.lzh.z;
        k.ba = c.b.x; k.bb = c.b.z;
    } else {
        k.lxa0 = c.lx.y; k.lxa1 = c.lx.z; k.lxb0 = c.lx.w; k.lxb1 = c.lxh;
        k.lya = c.ly.y; k.lyb = c.ly.w; k.lyha = c.lyh.y; k.lyhb = c.lyh.w;
        k.lza = c.lz.y; k.lzb = c.lz.w; k.lzha = c.lzh.y; k.lzhb = c.lzh.w;
        k.ba = c.b.y; k.bb = c.b.w;
    }
}

// Phase C on cells S and S+2 of `own` (plane v); zm_a/zm_b = plane v-1 and zp = plane v+1 at the
// own position.  Same operations in the same order as update_pair.
template <int S>
__device__ __forceinline__ float4 update_pair_carried(float xm, float4 own, float xp, float4 ym, float4 yp,
                                                      float zm_a, float zm_b, float4 zp, const CPair& k,
                                                      float omega) {
    float4 out = own;
    if (S == 0) {
        const float a1 = apply7(own.x, k.lxa0, k.lxa1, k.lya, k.lyha, k.lza, k.lzha, xm, own.y, ym.x, yp.x, zm_a, zp.x);
        const float a2 = apply7(own.z, k.lxb0, k.lxb1, k.lyb, k.lyhb, k.lzb, k.lzhb, own.y, own.w, ym.z, yp.z, zm_b, zp.z);
        out.x = relax(own.x, k.ba, a1, diag6(k.lxa0, k.lxa1, k.lya, k.lyha, k.lza, k.lzha), omega);
        out.z = relax(own.z, k.bb, a2, diag6(k.lxb0, k.lxb1, k.lyb, k.lyhb, k.lzb, k.lzhb), omega);
    } else {
        const float a1 = apply7(own.y, k.lxa0, k.lxa1, k.lya, k.lyha, k.lza, k.lzha, own.x, own.z, ym.y, yp.y, zm_a, zp.y);
        const float a2 = apply7(own.w, k.lxb0, k.lxb1, k.lyb, k.lyhb, k.lzb, k.lzhb, own.z, xp, ym.w, yp.w, zm_b, zp.w);
        out.y = relax(own.y, k.ba, a1, diag6(k.lxa0, k.lxa1, k.lya, k.lyha, k.lza, k.lzha), omega);
        out.w = relax(own.w, k.bb, a2, diag6(k.lxb0, k.lxb1, k.lyb, k.lyhb, k.lzb, k.lzhb), omega);
    }
    return out;
}

template <int S>
__device__ __forceinline__ float4 update_pair_full(float xm, float4 own, float xp, float4 ym, float4 yp,
                                                   float4 zm, float4 zp, const CFull& c, float omega) {
    CSet s;
    s.lx = c.lx; s.ly = c.ly; s.lyh = c.lyh; s.lzh = c.lzh; s.b = c.b; s.lxh = c.lxh;
    return update_pair<S>(xm, own, xp, ym, yp, zm, zp, s, c.lz, omega);
}

// Finish of a norm-carrying sweep: deterministic two-stage reduction, FP64 from the warp on, the
// same for every kernel that contributes (sweep_body with one row per warp, lean_body2 with two rows
// per warp, whatever their CTA sizes), so that the sums do not depend on which kernel a tile ran in
// or which CTA comes last.  Per tile: one partial per phase-B ROW (16 slots; a warp fills the slot(s)
// of its row(s)), added in row order.  Across tiles: the first 256 threads of the last CTA add the
// tile partials with stride 256.  Callers have passed a CTA barrier since their last ring access.
template <int NORM>
__device__ __forceinline__ void norm_finish(const BulkArgs& a, const int tile, float rr0, float bb0, float rr1,
                                            float bb1, const bool two_rows, float* sm) {
    const int tid = threadIdx.x, warp_id = tid >> 5, lane_id = tid & 31;
    double v0 = (double)rr0, w0 = (double)bb0, v1 = (double)rr1, w1 = (double)bb1;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        v0 += __shfl_down_sync(0xffffffffu, v0, o);
        w0 += __shfl_down_sync(0xffffffffu, w0, o);
        if (two_rows) {
            v1 += __shfl_down_sync(0xffffffffu, v1, o);
            w1 += __shfl_down_sync(0xffffffffu, w1, o);
        }
    }
    double* scratch = reinterpret_cast<double*>(sm);   // [0..16) sum r^2 per row, [16..32) sum b^2 per row
    int* last = reinterpret_cast<int*>(scratch + 32);
    if (lane_id == 0) {
        if (two_rows) {
            if (2 * warp_id + 1 < 16) {
                scratch[2 * warp_id] = v0; scratch[16 + 2 * warp_id] = w0;
                scratch[2 * warp_id + 1] = v1; scratch[16 + 2 * warp_id + 1] = w1;
            }
        } else if (warp_id < 16) {
            scratch[warp_id] = v0; scratch[16 + warp_id] = w0;
        }
    }
    __syncthreads();
    if (tid == 0) {
        double t0 = 0.0, t1 = 0.0;
        for (int r = 0; r < 16; ++r) { t0 += scratch[r]; t1 += scratch[16 + r]; }
        a.rb.partials[tile] = t0;
        a.rb.partials[GMG_REDUCE_MAX_BLOCKS + tile] = t1;
        __threadfence();
        *last = (atomicAdd(a.rb.counter, 1u) == (unsigned int)a.ntiles - 1u) ? 1 : 0;   // one ticket per TILE
    }
    __syncthreads();
    if (*last) {
        __threadfence();
        double a0 = 0.0, a1 = 0.0;
        if (tid < 256)
            for (unsigned int i = tid; i < (unsigned int)a.ntiles; i += 256u) {
                a0 += ((volatile double*)a.rb.partials)[i];
                a1 += ((volatile double*)a.rb.partials)[GMG_REDUCE_MAX_BLOCKS + i];
            }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            a0 += __shfl_down_sync(0xffffffffu, a0, o);
            a1 += __shfl_down_sync(0xffffffffu, a1, o);
        }
        __syncthreads();
        if (lane_id == 0 && warp_id < 8) { scratch[warp_id] = a0; scratch[16 + warp_id] = a1; }
        __syncthreads();
        if (tid == 0) {
            double t0 = 0.0, t1 = 0.0;
            for (int w = 0; w < 8; ++w) { t0 += scratch[w]; t1 += scratch[16 + w]; }
            a.rb.sc->red[a.slot_rr] = t0;
            if (NORM == 2) a.rb.sc->red[a.slot_ref] = t1;
            *a.rb.counter = 0u;
        }
    }
}

// YMODE 0: full TMA boxes.  YMODE 1: row-by-row bulk copies with wrapped row addresses (odd cases
// of a periodic y axis).  YMODE 2: first / final tile row of a periodic y axis -- shorter boxes over
// the rows inside the domain plus row copies for the two or three wrapped rows of each stream;
// box and row copies write disjoint rows of a slot and complete on the same mbarrier.
// (was) YIN: the tile's TMA boxes stay inside the domain in y (every tile but the first and last
// tile rows); the other instantiation carries the row-copy path, so the common one stays small.
// NORM: 0 = plain sweep; 1 = also sum r^2 of the source iterate; 2 = also sum b^2 over active cells
// (Tiles whose coefficients are the level's constants take lean_body2, sweep_lean2.cuh, instead.)
template <class C, int YMODE, int NORM>
__device__ __forceinline__ void sweep_body(const BulkArgs& a, const BulkMaps& allmaps, const int tile) {
    extern __shared__ __align__(1024) float sm[];  // no static shared memory: base is 1 KB aligned
    uint64_t* bars = reinterpret_cast<uint64_t*>(sm + C::FLOATS);  // [0..NB) step groups, [NB] prologue
    const float** row_base = reinterpret_cast<const float**>(bars + 16);  // row-copy path tables
    int* row_kind = reinterpret_cast<int*>(row_base + C::NROWCOPY);
    int* row_idx = row_kind + C::NROWCOPY;
    const LevelGeom& g = a.g;
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const size_t N = (size_t)g.N;
    const int plane = nx * ny;
    const int tid = threadIdx.x;
    const int warp_id = tid >> 5, lane_id = tid & 31;
    constexpr int NWARP = C::THREADS / 32;
    int bid = tile;
    const int tx = bid % a.tiles_x;
    bid /= a.tiles_x;
    const int ty = bid % a.tiles_y;
    const int zc = bid / a.tiles_y;
    const int x0 = tx * C::TX, y0 = ty * C::TY;
    const int z0 = zc * a.zchunk;
    const int z1 = min(nz, z0 + a.zchunk);
    const float omega = *a.omega;
    const int fc = a.first_colour;
    const int xL = wrapi(x0 - 4, nx), xR = wrapi(x0 + C::TX, nx);  // halo column groups
    constexpr bool y_inside = (YMODE == 0);
    constexpr bool y_rows = (YMODE == 1);
    // YMODE 2 geometry (uniform over the CTA): which map set, where the boxes start (global row and
    // row offset in the slot), the wrapped rows (slot row j <- global row y), the bytes per group
    const bool y_first = (y0 == 0);
    const MapSet& maps = allmaps.m[YMODE == 2 ? (y_first ? 1 : 2) : 0];
    const int hP = ny - y0 + 2, hC = ny - y0 + 1;          // FINAL: rows of the p / coefficient boxes
    const int e_oP = y_first ? 2 : 0, e_oC = y_first ? 1 : 0;
    // a tensor box must land on a 128-byte boundary: in a FIRST tile the x-halo columns (16 B per
    // row) are kept 6 rows further down in their padded area, so that row 2 -- where the box
    // starts -- sits at byte 128 (HPAD leaves room: (SH + 6) * 4 <= HPAD)
    static_assert((C::SH + 6) * 4 <= C::HPAD, "halo padding");
    const int hs = (YMODE == 2 && y_first) ? 24 : 0;
    const int e_yP = y_first ? 0 : y0 - 2, e_yC = y_first ? 0 : y0 - 1;
    const int e_pj0 = y_first ? 0 : hP, e_py0 = y_first ? ny - 2 : 0;     // p: rows j0, j0+1 <- y0', y0'+1
    const int e_cj = y_first ? 0 : hC, e_cy = y_first ? ny - 1 : 0;       // Lz, Lx, b, Ly: row j <- y
    const bool e_ly2 = !y_first;                                          // Ly FINAL: also row j+1 <- 1
    const uint32_t e_pbytes = (uint32_t)((y_first ? C::SH : hP + 2) * (C::TX + 8)) * 4u;
    const uint32_t e_cbytes = (uint32_t)((y_first ? C::ROWS : hC + 1) * C::TX) * 4u;
    const uint32_t e_lybytes = (uint32_t)((y_first ? C::ROWS + 1 : hC + 2) * C::TX) * 4u;
    const uint32_t step_bytes = (YMODE == 2) ? e_pbytes + 3u * e_cbytes + e_lybytes : C::STEP_BYTES;
    const uint32_t pro_bytes = (YMODE == 2) ? 2u * e_pbytes + e_cbytes : C::PRO_BYTES;
    const float* Lx = a.L;
    const float* Ly = a.L + N;
    const float* Lz = a.L + 2 * N;

    // ring slots: plane v of each stream
    auto slotP = [&](int v) -> float* { return sm + C::OFF_P + ((v - (z0 - 2)) % C::NP) * C::P_PLANE; };
    auto slotLz = [&](int v) -> float* { return sm + C::OFF_LZ + ((v - (z0 - 1)) % C::NZ) * C::C_PLANE; };
    auto slotLx = [&](int v) -> float* { return sm + C::OFF_LX + ((v - (z0 - 1)) % C::NC) * C::C_PLANE; };
    auto slotLy = [&](int v) -> float* { return sm + C::OFF_LY + ((v - (z0 - 1)) % C::NC) * C::Y_PLANE; };
    auto slotB = [&](int v) -> float* { return sm + C::OFF_B + ((v - (z0 - 1)) % C::NC) * C::C_PLANE; };

    // ---- copy issue ------------------------------------------------------------------------------
    // Interior tiles: 7 TMA boxes per step, one per warp 0..6 (lane 0).  Tiles touching the y
    // boundary: row-by-row bulk copies with wrapped row addresses, dealt round-robin to the warps.
    // kind 0: p(v+1) rows y0-2..   1: Lz(v+1)   2: Lx(v)   3: Ly(v) (one more row)   4: b(v)
    if (y_rows && tid < C::NROWCOPY) {
        int t = tid, ck, crow;
        if (t < C::SH) { ck = 0; crow = t; }
        else if ((t -= C::SH) < C::ROWS) { ck = 1; crow = t; }
        else if ((t -= C::ROWS) < C::ROWS) { ck = 2; crow = t; }
        else if ((t -= C::ROWS) < C::ROWS + 1) { ck = 3; crow = t; }
        else { t -= C::ROWS + 1; ck = 4; crow = t; }
        const int y = wrapi(ck == 0 ? y0 - 2 + crow : y0 - 1 + crow, ny);
        const float* arr = ck == 0 ? a.src : ck == 1 ? Lz : ck == 2 ? Lx : ck == 3 ? Ly : a.b;
        row_base[tid] = arr + (size_t)y * nx;
        row_kind[tid] = ck;
        row_idx[tid] = crow;
    }
    auto copy_p_rows = [&](int v, uint64_t* bar) {  // row path: the SH rows of p plane v
        float* d = slotP(v);
        const size_t pz = (size_t)wrapi(v, nz) * plane;
        for (int j = warp_id; j < C::SH; j += NWARP) {
            const float* rb = row_base[j] + pz;
            bulk_g2s(d + j * C::TX, rb + x0, C::TX * 4u, bar);
            bulk_g2s(d + C::P_HL + j * 4, rb + xL, 16u, bar);
            bulk_g2s(d + C::P_HR + j * 4, rb + xR, 16u, bar);
        }
    };
    auto copy_c_rows = [&](int kind, float* d, size_t pz, uint64_t* bar) {  // row path: one coefficient plane
        const int first = kind == 1 ? C::SH : kind == 2 ? C::SH + C::ROWS : kind == 3 ? C::SH + 2 * C::ROWS
                                                                          : C::SH + 3 * C::ROWS + 1;
        const int cnt = kind == 3 ? C::ROWS + 1 : C::ROWS;
        for (int j = warp_id; j < cnt; j += NWARP)
            bulk_g2s(d + j * C::TX, row_base[first + j] + pz + x0, C::TX * 4u, bar);
    };
    auto issue_step = [&](int v) {  // the data B(v) newly needs: p(v+1), Lz(v+1), Lx(v), Ly(v), b(v)
        if (lane_id != 0 || (y_inside && warp_id >= 7)) return;
        uint64_t* bar = bars + ((v - (z0 - 1)) % C::NB);
        if (tid == 0) mbar_expect_tx(bar, step_bytes);
        const int gz0 = wrap1(v, nz), gz1 = wrap1(v + 1, nz);
        const int vp = v + 1, gzv = gz1;                     // the p plane of this group
        if (y_inside) {
            switch (warp_id) {
                case 0: tma_load_3d(slotP(vp), &maps.p_main, x0, y0 - 2, gzv, bar); break;
                case 1: tma_load_3d(slotP(vp) + C::P_HL, &maps.p_halo, xL, y0 - 2, gzv, bar); break;
                case 2: tma_load_3d(slotP(vp) + C::P_HR, &maps.p_halo, xR, y0 - 2, gzv, bar); break;
                case 3: tma_load_3d(slotLz(v + 1), &maps.lz, x0, y0 - 1, gz1, bar); break;
                case 4: tma_load_3d(slotLx(v), &maps.lx, x0, y0 - 1, gz0, bar); break;
                case 5: tma_load_3d(slotLy(v), &maps.ly, x0, y0 - 1, gz0, bar); break;
                case 6: tma_load_3d(slotB(v), &maps.b, x0, y0 - 1, gz0, bar); break;
                default: break;
            }
        } else if (YMODE == 2) {
            const size_t pz0 = (size_t)gz0 * plane, pz1 = (size_t)gz1 * plane;
            switch (warp_id) {
                case 0: tma_load_3d(slotP(vp) + e_oP * C::TX, &maps.p_main, x0, e_yP, gzv, bar); break;
                case 1: tma_load_3d(slotP(vp) + C::P_HL + hs + e_oP * 4, &maps.p_halo, xL, e_yP, gzv, bar); break;
                case 2: tma_load_3d(slotP(vp) + C::P_HR + hs + e_oP * 4, &maps.p_halo, xR, e_yP, gzv, bar); break;
                case 3: tma_load_3d(slotLz(v + 1) + e_oC * C::TX, &maps.lz, x0, e_yC, gz1, bar); break;
                case 4: tma_load_3d(slotLx(v) + e_oC * C::TX, &maps.lx, x0, e_yC, gz0, bar); break;
                case 5: tma_load_3d(slotLy(v) + e_oC * C::TX, &maps.ly, x0, e_yC, gz0, bar); break;
                case 6: tma_load_3d(slotB(v) + e_oC * C::TX, &maps.b, x0, e_yC, gz0, bar); break;
                case 7: case 8: {   // the two wrapped p rows
                    const int r = warp_id - 7, j = e_pj0 + r;
                    const float* rb = a.src + pz1 + (size_t)(e_py0 + r) * nx;
                    float* d = slotP(vp);
                    bulk_g2s(d + j * C::TX, rb + x0, C::TX * 4u, bar);
                    bulk_g2s(d + C::P_HL + hs + j * 4, rb + xL, 16u, bar);
                    bulk_g2s(d + C::P_HR + hs + j * 4, rb + xR, 16u, bar);
                } break;
                case 9: bulk_g2s(slotLz(v + 1) + e_cj * C::TX, Lz + pz1 + (size_t)e_cy * nx + x0, C::TX * 4u, bar); break;
                case 10: bulk_g2s(slotLx(v) + e_cj * C::TX, Lx + pz0 + (size_t)e_cy * nx + x0, C::TX * 4u, bar); break;
                case 11:
                    bulk_g2s(slotLy(v) + e_cj * C::TX, Ly + pz0 + (size_t)e_cy * nx + x0, C::TX * 4u, bar);
                    if (e_ly2) bulk_g2s(slotLy(v) + (e_cj + 1) * C::TX, Ly + pz0 + (size_t)(e_cy + 1) * nx + x0, C::TX * 4u, bar);
                    break;
                case 12: bulk_g2s(slotB(v) + e_cj * C::TX, a.b + pz0 + (size_t)e_cy * nx + x0, C::TX * 4u, bar); break;
                default: break;
            }
        } else {
            copy_p_rows(vp, bar);
            copy_c_rows(1, slotLz(v + 1), (size_t)gz1 * plane, bar);
            copy_c_rows(2, slotLx(v), (size_t)gz0 * plane, bar);
            copy_c_rows(3, slotLy(v), (size_t)gz0 * plane, bar);
            copy_c_rows(4, slotB(v), (size_t)gz0 * plane, bar);
        }
    };

    // ---- prologue: barriers; p(z0-2), p(z0-1), Lz(z0-1); the first PD step groups --------------
    if (tid == 0) {
        for (int i = 0; i <= C::NB; ++i) mbar_init(bars + i, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    fence_async_smem();
    __syncthreads();
    {
        uint64_t* bar = bars + C::NB;
        if (lane_id == 0) {
            if (tid == 0) mbar_expect_tx(bar, pro_bytes);
            const int gb = wrap1(z0 - 1, nz);
            if (y_inside) {
                // planes z0-2, z0-1: three boxes each, one per warp; then Lz(z0-1)
                const int pl = warp_id / 3, k = warp_id % 3;
                if (pl < 2) {
                    const int v = z0 - 2 + pl, gv = wrapi(v, nz);
                    if (k == 0) tma_load_3d(slotP(v), &maps.p_main, x0, y0 - 2, gv, bar);
                    else if (k == 1) tma_load_3d(slotP(v) + C::P_HL, &maps.p_halo, xL, y0 - 2, gv, bar);
                    else tma_load_3d(slotP(v) + C::P_HR, &maps.p_halo, xR, y0 - 2, gv, bar);
                } else if (warp_id == 6) {
                    tma_load_3d(slotLz(z0 - 1), &maps.lz, x0, y0 - 1, gb, bar);
                }
            } else if (YMODE == 2) {
                const int pl = warp_id / 3, k = warp_id % 3;
                if (pl < 2) {
                    const int v = z0 - 2 + pl, gv = wrapi(v, nz);
                    if (k == 0) tma_load_3d(slotP(v) + e_oP * C::TX, &maps.p_main, x0, e_yP, gv, bar);
                    else if (k == 1) tma_load_3d(slotP(v) + C::P_HL + hs + e_oP * 4, &maps.p_halo, xL, e_yP, gv, bar);
                    else tma_load_3d(slotP(v) + C::P_HR + hs + e_oP * 4, &maps.p_halo, xR, e_yP, gv, bar);
                } else if (warp_id == 6) {
                    tma_load_3d(slotLz(z0 - 1) + e_oC * C::TX, &maps.lz, x0, e_yC, gb, bar);
                } else if (warp_id >= 7 && warp_id <= 10) {      // wrapped p rows of the two planes
                    const int v = z0 - 2 + (warp_id - 7) / 2, r = (warp_id - 7) & 1, j = e_pj0 + r;
                    const float* rb = a.src + (size_t)wrapi(v, nz) * plane + (size_t)(e_py0 + r) * nx;
                    float* d = slotP(v);
                    bulk_g2s(d + j * C::TX, rb + x0, C::TX * 4u, bar);
                    bulk_g2s(d + C::P_HL + hs + j * 4, rb + xL, 16u, bar);
                    bulk_g2s(d + C::P_HR + hs + j * 4, rb + xR, 16u, bar);
                } else if (warp_id == 11) {
                    bulk_g2s(slotLz(z0 - 1) + e_cj * C::TX, Lz + (size_t)gb * plane + (size_t)e_cy * nx + x0, C::TX * 4u, bar);
                }
            } else {
                for (int pl = 0; pl < 2; ++pl) copy_p_rows(z0 - 2 + pl, bar);
                copy_c_rows(1, slotLz(z0 - 1), (size_t)gb * plane, bar);
            }
        }
        for (int v = z0 - 1; v < z0 - 1 + C::PD && v <= z1; ++v) issue_step(v);
        mbar_wait(bar, 0);
    }

    // ring cursors of step u (advanced once per step; no modulo in the loop)
    float* const P_beg = sm + C::OFF_P;
    float* const Z_beg = sm + C::OFF_LZ;
    float* Pm1 = P_beg;                             // plane u-1
    float* P0 = P_beg + C::P_PLANE;                 // plane u
    float* Pp1 = P_beg + 2 * C::P_PLANE;            // plane u+1
    const float* Z0 = Z_beg;                        // Lz plane u
    const float* Z1 = Z_beg + C::C_PLANE;           // Lz plane u+1
    int ic = 0;                                     // slot of Lx / Ly / b plane u
    int kb = 0;                                     // mbarrier of step u and its phase parity
    uint32_t kpar = 0;
    int gz = wrap1(z0 - 1, nz);                     // wrapped plane index of u
    auto advance = [&]() {
        Pm1 = P0; P0 = Pp1;
        Pp1 += C::P_PLANE;
        if (Pp1 == P_beg + C::NP * C::P_PLANE) Pp1 = P_beg;
        Z0 = Z1;
        Z1 += C::C_PLANE;
        if (Z1 == Z_beg + C::NZ * C::C_PLANE) Z1 = Z_beg;
        if (++ic == C::NC) ic = 0;
        if (++kb == C::NB) { kb = 0; kpar ^= 1u; }
        if (++gz == nz) gz = 0;
    };

    float acc_rr_out = 0.0f, acc_bb_out = 0.0f;   // NORM: the thread's partial sums
    if (tid < C::MAIN) {
        // ---- main threads: one float4 group of one row ---------------------------------------
        const int lx = lane_id, ry = warp_id;
        const int xl = x0 + 4 * lx;
        const int yl = y0 + ry - 1;
        const int gx = xl, gy = wrapi(yl, ny), gyp = wrapi(yl + 1, ny);
        const int gxh = wrapi(xl + 4, nx);
        const bool row_c = (ry >= 1) && (ry <= C::TY) && (yl < ny);
        const bool zx_lo = g.bc[0] && gx == 0, zx_hi = g.bc[0] && gxh == 0;
        const bool zy_lo = g.bc[1] && gy == 0, zy_hi = g.bc[1] && gyp == 0;
        const bool last_lane = (lx == C::LPR - 1);
        const int p_off = (ry + 1) * C::TX + 4 * lx;        // own float4 in a p plane
        const int h_off = (lx == 0 ? C::P_HL + 3 : C::P_HR) + hs + (ry + 1) * 4;  // x-halo cell (first / last lane)
        const int c_off = ry * C::TX + 4 * lx;              // own float4 in a coefficient plane
        float* dst_ptr = a.dst + ((long long)gy * nx + gx + (long long)(z0 - 2) * plane);  // plane u-1
        const float* const lxh_row = Lx + (size_t)gy * nx + gxh;  // face above the tile's last cell
        // cells (sel, sel+2) of the group are updated: same parity for B(u) and C(u-1); sel is
        // warp-uniform and alternates every step
        int sel = (yl + (z0 - 1) + fc) & 1;
        float lxh_pf = last_lane ? __ldg(lxh_row + (size_t)gz * plane) : 0.0f;
        const bool any_wall = zx_lo || zx_hi || zy_lo || zy_hi || g.bc[2];
        // K = the coefficients of the two cells C updates next step, picked out of this step's
        // set (14 floats, not a second full set); q1 / z2 = planes u-1 / u-2 at the own position
        CPair K;
        K.lxa0 = K.lxa1 = K.lxb0 = K.lxb1 = K.lya = K.lyb = K.lyha = K.lyhb = 0.0f;
        K.lza = K.lzb = K.lzha = K.lzhb = K.ba = K.bb = 0.0f;
        float4 q1 = lds4(Pm1 + p_off);   // u = z0-1: source values
        float z2a = 0.0f, z2b = 0.0f;
        // NORM: SOURCE values of plane u-1 at the lanes of plane u's second-colour cells (q1 holds
        // the B-updated ones there), and this thread's partial sums
        float zs_a = 0.0f, zs_b = 0.0f, acc_rr = 0.0f, acc_bb = 0.0f;
        CFull Sc;
        float4 own, ym, yp, zp;
        float hvB;
        // Operands of B(u) -- TMA data and source values no other thread changes.  Loaded at the
        // end of step u-1, in front of the barrier: behind it only the two rows phase C needs
        // are still to be read, so the 16 warps do not all queue on the shared-memory pipe at once.
        auto load_step = [&]() {
            mbar_wait(bars + kb, kpar);
            Sc.lx = lds4(sm + C::OFF_LX + ic * C::C_PLANE + c_off);
            const float* Y = sm + C::OFF_LY + ic * C::Y_PLANE + c_off;
            Sc.ly = lds4(Y);
            Sc.lyh = lds4(Y + C::TX);
            Sc.lz = lds4(Z0 + c_off);
            Sc.lzh = lds4(Z1 + c_off);
            Sc.b = lds4(sm + C::OFF_B + ic * C::C_PLANE + c_off);
            own = lds4(P0 + p_off);
            ym = lds4(P0 + p_off - C::TX);
            yp = lds4(P0 + p_off + C::TX);
            zp = lds4(Pp1 + p_off);
            hvB = P0[h_off];
        };
        load_step();
        for (int u = z0 - 1; u <= z1; ++u) {
            const int gzp = (gz + 1 == nz) ? 0 : gz + 1;
            const float4 cym = lds4(Pm1 + p_off - C::TX);   // plane u-1, B-updated rows above / below
            const float4 cyp = lds4(Pm1 + p_off + C::TX);
            const float hvC = Pm1[h_off];
            const float t = __shfl_down_sync(0xffffffffu, Sc.lx.x, 1);
            Sc.lxh = last_lane ? lxh_pf : t;
            if (last_lane && u + 1 <= z1) lxh_pf = __ldg(lxh_row + (size_t)gzp * plane);
            if (any_wall) {   // Neumann wall faces carry coefficient 0 (reading O2)
                if (zx_lo) Sc.lx.x = 0.0f;
                if (zx_hi) Sc.lxh = 0.0f;
                if (zy_lo) Sc.ly = zero4();
                if (zy_hi) Sc.lyh = zero4();
                if (g.bc[2]) {
                    if (gz == 0) Sc.lz = zero4();
                    if (gzp == 0) Sc.lzh = zero4();
                }
            }
            float xm = __shfl_up_sync(0xffffffffu, own.w, 1);
            float xp = __shfl_down_sync(0xffffffffu, own.x, 1);
            float cxm = __shfl_up_sync(0xffffffffu, q1.w, 1);
            float cxp = __shfl_down_sync(0xffffffffu, q1.x, 1);
            xm = (lx == 0) ? hvB : xm;
            xp = last_lane ? hvB : xp;
            cxm = (lx == 0) ? hvC : cxm;
            cxp = last_lane ? hvC : cxp;
            float4 nw, nc;   // B(u) and C(u-1) results
            if (NORM) {
                // residual of the SOURCE iterate on all four cells of plane u: every operand B(u)
                // has is a source value except plane u-1 under the second-colour cells (zs_a, zs_b)
                const float s0 = sel ? zs_a : q1.x, s1 = sel ? q1.y : zs_a;
                const float s2 = sel ? zs_b : q1.z, s3 = sel ? q1.w : zs_b;
                const float A0 = apply7(own.x, Sc.lx.x, Sc.lx.y, Sc.ly.x, Sc.lyh.x, Sc.lz.x, Sc.lzh.x, xm, own.y, ym.x, yp.x, s0, zp.x);
                const float A1 = apply7(own.y, Sc.lx.y, Sc.lx.z, Sc.ly.y, Sc.lyh.y, Sc.lz.y, Sc.lzh.y, own.x, own.z, ym.y, yp.y, s1, zp.y);
                const float A2 = apply7(own.z, Sc.lx.z, Sc.lx.w, Sc.ly.z, Sc.lyh.z, Sc.lz.z, Sc.lzh.z, own.y, own.w, ym.z, yp.z, s2, zp.z);
                const float A3 = apply7(own.w, Sc.lx.w, Sc.lxh, Sc.ly.w, Sc.lyh.w, Sc.lz.w, Sc.lzh.w, own.z, xp, ym.w, yp.w, s3, zp.w);
                const bool a0 = diag6(Sc.lx.x, Sc.lx.y, Sc.ly.x, Sc.lyh.x, Sc.lz.x, Sc.lzh.x) != 0.0f;
                const bool a1 = diag6(Sc.lx.y, Sc.lx.z, Sc.ly.y, Sc.lyh.y, Sc.lz.y, Sc.lzh.y) != 0.0f;
                const bool a2 = diag6(Sc.lx.z, Sc.lx.w, Sc.ly.z, Sc.lyh.z, Sc.lz.z, Sc.lzh.z) != 0.0f;
                const bool a3 = diag6(Sc.lx.w, Sc.lxh, Sc.ly.w, Sc.lyh.w, Sc.lz.w, Sc.lzh.w) != 0.0f;
                if (row_c && u >= z0 && u < z1) {
                    const float r0 = a0 ? Sc.b.x - A0 : 0.0f, r1 = a1 ? Sc.b.y - A1 : 0.0f;
                    const float r2 = a2 ? Sc.b.z - A2 : 0.0f, r3 = a3 ? Sc.b.w - A3 : 0.0f;
                    // explicit roundings (no FMA contraction): general and lean path add the same bits
                    acc_rr = __fadd_rn(acc_rr, __fadd_rn(__fadd_rn(__fmul_rn(r0, r0), __fmul_rn(r1, r1)),
                                                         __fadd_rn(__fmul_rn(r2, r2), __fmul_rn(r3, r3))));
                    if (NORM == 2) {
                        const float b0 = a0 ? Sc.b.x : 0.0f, b1 = a1 ? Sc.b.y : 0.0f;
                        const float b2 = a2 ? Sc.b.z : 0.0f, b3 = a3 ? Sc.b.w : 0.0f;
                        acc_bb = __fadd_rn(acc_bb, __fadd_rn(__fadd_rn(__fmul_rn(b0, b0), __fmul_rn(b1, b1)),
                                                             __fadd_rn(__fmul_rn(b2, b2), __fmul_rn(b3, b3))));
                    }
                }
                zs_a = sel ? own.y : own.x;
                zs_b = sel ? own.w : own.z;
            }
            if (sel) {
                nw = update_pair_full<1>(xm, own, xp, ym, yp, q1, zp, Sc, omega);
                nc = update_pair_carried<1>(cxm, q1, cxp, cym, cyp, z2a, z2b, nw, K, omega);
                pick_pair<0>(Sc, K);     // the next step's C works on cells 0 and 2 of plane u
                z2a = q1.x; z2b = q1.z;
            } else {
                nw = update_pair_full<0>(xm, own, xp, ym, yp, q1, zp, Sc, omega);
                nc = update_pair_carried<0>(cxm, q1, cxp, cym, cyp, z2a, z2b, nw, K, omega);
                pick_pair<1>(Sc, K);
                z2a = q1.y; z2b = q1.w;
            }
            *reinterpret_cast<float4*>(P0 + p_off) = nw;
            if (u - 1 >= z0 && row_c) *reinterpret_cast<float4*>(dst_ptr) = nc;
            q1 = nw;
            sel ^= 1;
            dst_ptr += plane;
            advance();
            if (u + 1 <= z1) load_step();
            fence_async_smem();  // order this thread's smem writes before later TMA overwrites
            cta_sync();
            if (u + C::PD <= z1) issue_step(u + C::PD);
        }
        if (NORM) { acc_rr_out = acc_rr; acc_bb_out = acc_bb; }
    } else {
        // ---- edge warp: ring-1 cells x0-1 and x0+TX of every row, phase B only ----------------
        const int el = lane_id;
        const bool e_act = el < 2 * C::ROWS;
        const int side = el & 1, ery = e_act ? (el >> 1) : 0;
        const int xs = side ? x0 + C::TX : x0 - 1;
        const int eyl = y0 + ery - 1;
        const int gxs = wrapi(xs, nx), gxs1 = wrapi(xs + 1, nx);
        const int egy = wrapi(eyl, ny), egyp = wrapi(eyl + 1, ny);
        const int r = ery + 1;
        const int pc_off = hs + (side ? C::P_HR + r * 4 : C::P_HL + r * 4 + 3);   // the edge cell
        const int xm_off = side ? r * C::TX + C::TX - 1 : pc_off - 1;      // its x neighbours
        const int xp_off = side ? pc_off + 1 : r * C::TX;
        const int o_c = egy * nx + gxs, o_x1 = egy * nx + gxs1, o_yp = egyp * nx + gxs;
        const bool ex_lo = g.bc[0] && gxs == 0, ex_hi = g.bc[0] && gxs1 == 0;
        const bool ey_lo = g.bc[1] && egy == 0, ey_hi = g.bc[1] && egyp == 0;
        struct ESet { float wxl, wxh, wyl, wyh, wzl, wzh, b; };
        auto fetch_e = [&](int gzc, ESet& s) {  // global loads, issued one step ahead
            const int gzn = (gzc + 1 == nz) ? 0 : gzc + 1;
            const size_t pz = (size_t)gzc * plane, pzp = (size_t)gzn * plane;
            s.wxl = ex_lo ? 0.0f : __ldg(Lx + pz + o_c);
            s.wxh = ex_hi ? 0.0f : __ldg(Lx + pz + o_x1);
            s.wyl = ey_lo ? 0.0f : __ldg(Ly + pz + o_c);
            s.wyh = ey_hi ? 0.0f : __ldg(Ly + pz + o_yp);
            s.wzl = (g.bc[2] && gzc == 0) ? 0.0f : __ldg(Lz + pz + o_c);
            s.wzh = (g.bc[2] && gzn == 0) ? 0.0f : __ldg(Lz + pzp + o_c);
            s.b = __ldg(a.b + pz + o_c);
        };
        ESet Ec, En;
        fetch_e(gz, Ec);
        En = Ec;
        int ecol = (xs + eyl + (z0 - 1)) & 1;  // colour of the edge cell in plane u
        for (int u = z0 - 1; u <= z1; ++u) {
            if (u + 1 <= z1) fetch_e((gz + 1 == nz) ? 0 : gz + 1, En);
            mbar_wait(bars + kb, kpar);
            if (e_act && ecol == fc) {
                const float pc = P0[pc_off];
                const float Ap = apply7(pc, Ec.wxl, Ec.wxh, Ec.wyl, Ec.wyh, Ec.wzl, Ec.wzh, P0[xm_off],
                                        P0[xp_off], P0[pc_off - 4], P0[pc_off + 4], Pm1[pc_off],
                                        Pp1[pc_off]);
                P0[pc_off] = relax(pc, Ec.b, Ap,
                                   diag6(Ec.wxl, Ec.wxh, Ec.wyl, Ec.wyh, Ec.wzl, Ec.wzh), omega);
            }
            fence_async_smem();
            cta_sync();
            if (u + C::PD <= z1) issue_step(u + C::PD);
            Ec = En;
            ecol ^= 1;
            advance();
        }
    }
    if (NORM) norm_finish<NORM>(a, tile, acc_rr_out, acc_bb_out, 0.0f, 0.0f, false, sm);
}

}  // namespace gmgf
#include "sweep_lean2.cuh"
namespace gmgf {

// How a tile's planes reach shared memory: 0 = full boxes (inside the domain in y, or walls in y:
// rows outside arrive zero-filled), 2 = first / final tile row of a periodic y axis: boundary boxes
// plus a few row copies, 1 = row copies only (odd cases: a single tile row, a final row too short).
template <class C>
__device__ __forceinline__ int tile_ymode(const BulkArgs& a, int ty) {
    const int y0 = ty * C::TY, ny = a.g.n[1];
    if (a.g.bc[1] != 0 || ((y0 >= 2) && (y0 + C::TY + 2 <= ny))) return 0;
    if (a.tiles_y >= 2 && ((ty == 0 && C::TY + 2 <= ny) || (ty == a.tiles_y - 1 && y0 >= 2))) return 2;
    return 1;
}

// Lean path (uniform.cuh)?  Every warp evaluates the same few brick flags (CTA-uniform verdict): the
// tile is box-fed and all coefficients the CTA would touch -- tile + ring 2, planes z0-2 .. z1+1 --
// are the level's constants with no Neumann wall in reach.  Such tiles belong to k_rb_sweep_lean.
template <class C>
__device__ __forceinline__ bool tile_is_lean(const BulkArgs& a, int tile, int ymode) {
    if (!a.uni.brick || ymode == 1) return false;
    int bid = tile;
    const int tx = bid % a.tiles_x;
    bid /= a.tiles_x;
    const int ty = bid % a.tiles_y;
    const int zc = bid / a.tiles_y;
    const int x0 = tx * C::TX, y0 = ty * C::TY, z0 = zc * a.zchunk, z1 = min(a.g.n[2], z0 + a.zchunk);
    return ub_box_uniform_warp(a.g, a.uni.brick, x0 - 2, x0 + C::TX + 1, y0 - 2, y0 + C::TY + 2, z0 - 2, z1 + 1,
                               threadIdx.x & 31);
}

// EDGE: the kernel also carries the YMODE 2 body and sends every tile of a Neumann y axis through
// the full boxes.  It pays on grids with few tile rows (a 1024 x 384 x 384 channel: -5 % per solve);
// on a 1024^3 cube the third body costs the interior loop its register allocation (+2.6 % per
// sweep, measured A/B on one box), so the launcher picks the kernel by the number of tile rows.
// With uniform bricks marked (a.uni.brick) the lean tiles are k_rb_sweep_lean's; this kernel then
// runs one CTA per entry of the list of remaining tiles (a.uni.left_list), or -- the list's length
// not yet known on the host -- over the whole grid, where the lean tiles return at once.
template <class C, int NORM = 0, bool EDGE = false>
__global__ void __launch_bounds__(C::THREADS, 1)
k_rb_sweep_bulk(const BulkArgs a, const __grid_constant__ BulkMaps maps) {
    if (a.run_flag && *a.run_flag == 0) return;   // a re-run that turned out not to be needed
    int tile = blockIdx.x;
    if (a.uni.left_list) {
        if (blockIdx.x >= *a.uni.left_count) return;
        tile = a.uni.left_list[blockIdx.x];
    }
    const int ty = (tile / a.tiles_x) % a.tiles_y;
    const int ymode = tile_ymode<C>(a, ty);
    if (!a.uni.left_list && tile_is_lean<C>(a, tile, ymode)) return;
    if (EDGE) {
        if (ymode == 0) sweep_body<C, 0, NORM>(a, maps, tile);
        else if (ymode == 2) sweep_body<C, 2, NORM>(a, maps, tile);
        else sweep_body<C, 1, NORM>(a, maps, tile);
    } else {
        const int y0 = ty * C::TY;
        if ((y0 >= 2) && (y0 + C::TY + 2 <= a.g.n[1])) sweep_body<C, 0, NORM>(a, maps, tile);
        else sweep_body<C, 1, NORM>(a, maps, tile);
    }
}

// The lean path as a kernel of its own: the box-fed tiles whose footprint is uniform; every other
// tile of the grid returns at once (k_rb_sweep_bulk takes those).  Without coefficient rings a CTA
// needs 102 KB of shared memory and 96-128 registers per thread, so TWO CTAs share an SM and one fills
// the other's barrier and latency gaps (issue slots 44 % -> 69 % busy).
template <class C, int NORM = 0>
__global__ void __launch_bounds__(Lean2Threads<(NORM != 0)>::value, 2)
k_rb_sweep_lean(const BulkArgs a, const __grid_constant__ BulkMaps maps) {
    if (a.run_flag && *a.run_flag == 0) return;
    const int tile = blockIdx.x;
    const int ty = (tile / a.tiles_x) % a.tiles_y;
    const int ymode = tile_ymode<C>(a, ty);
    if (!tile_is_lean<C>(a, tile, ymode)) return;
    if (ymode == 0) lean_body2<C, 0, NORM, (NORM != 0)>(a, maps, tile);
    else lean_body2<C, 2, NORM, (NORM != 0)>(a, maps, tile);
}

// ... with the prolongation + correction folded in (lean_body2<PRO>): 288 threads, two CTAs per SM
// (96 registers: warps are allocated in pairs, 2 x 10 x 32 x 96 = 61,440 of the 65,536; at 112
// registers only one CTA fits and the kernel takes 4.2 instead of 2.4 ms at 1024^3)
template <class C>
__global__ void __launch_bounds__(Lean2Threads<false>::value, 2)
k_rb_sweep_lean_pro(const BulkArgs a, const __grid_constant__ BulkMaps maps) {
    if (a.run_flag && *a.run_flag == 0) return;
    const int tile = blockIdx.x;
    const int ty = (tile / a.tiles_x) % a.tiles_y;
    const int ymode = tile_ymode<C>(a, ty);
    if (!tile_is_lean<C>(a, tile, ymode)) return;
    if (ymode == 0) lean_body2<C, 0, 0, false, true>(a, maps, tile);
    else lean_body2<C, 2, 0, false, true>(a, maps, tile);
}

// Prolongation + correction for the tiles that are NOT lean, when the first post-sweep folds it in
// (lean tiles: lean_body2<PRO>): scratch = src + P e_c over the footprint of each such tile (tile +
// the halo the TMA boxes of k_rb_sweep_bulk fetch, wrapped on periodic axes), one CTA per entry of
// the remaining-tile list.  k_rb_sweep_bulk then sweeps scratch -> dst on those tiles.  Footprints
// of neighbouring tiles overlap; they write the same values.  2x2x2 coarsening.
template <class C>
__global__ void __launch_bounds__(256)
k_prolong_tiles(const BulkArgs a, float* __restrict__ scratch) {
    int tile = blockIdx.x;
    if (a.uni.left_list) {
        if (blockIdx.x >= *a.uni.left_count) return;
        tile = a.uni.left_list[blockIdx.x];
    } else {
        const int ty_ = (tile / a.tiles_x) % a.tiles_y;
        if (tile_is_lean<C>(a, tile, tile_ymode<C>(a, ty_))) return;
    }
    const LevelGeom& g = a.g;
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const int tx = tile % a.tiles_x, ty = (tile / a.tiles_x) % a.tiles_y, zc = tile / (a.tiles_x * a.tiles_y);
    const int x0 = tx * C::TX, y0 = ty * C::TY, z0 = zc * a.zchunk, z1 = min(nz, z0 + a.zchunk);
    constexpr int GX = C::TX / 4 + 2, GY = C::TY + 4;      // float4 groups x0-4 .. x0+TX+3, rows y0-2 .. y0+TY+1
    const int GZ = z1 - z0 + 4;                            // planes z0-2 .. z1+1
    const int ncx = nx >> 1, ncy = ny >> 1;
    for (int t = threadIdx.x; t < GX * GY * GZ; t += 256) {
        const int gxi = t % GX, r = t / GX;
        const int y = y0 - 2 + r % GY, z = z0 - 2 + r / GY;
        int x = x0 - 4 + 4 * gxi;
        // out of the domain: wrapped on every axis -- behind a wall the boxes fill zeros, but the row
        // copies of a tile row at a y wall read the wrapped rows (times a zero coefficient)
        x = wrapi(x, nx);
        const int gy = wrapi(y, ny), gz = wrapi(z, nz);
        const size_t o = ((size_t)gz * ny + gy) * nx + x;
        float4 v = ldg4(a.src + o);
        const float2 e = __ldg(reinterpret_cast<const float2*>(a.e_c + ((size_t)(gz >> 1) * ncy + (gy >> 1)) * ncx + (x >> 1)));
        v.x += e.x; v.y += e.x; v.z += e.y; v.w += e.y;
        *reinterpret_cast<float4*>(scratch + o) = v;
    }
}

// ---- launchers ------------------------------------------------------------------------------
bool sweep_v2_supported(const LevelGeom& g);
void rb_sweep_v2(const LevelGeom& g, const float* L, const float* src, float* dst, const float* b,
                 const float* omega, int first_colour, const float* e_c, cudaStream_t s);
int configure_v2();

using Bulk = BulkCfg<13, 4>;
using Lean = BulkCfg<13, 4, true>;
static_assert(2 * (Lean::SMEM + 1024) <= 227 * 1024, "two lean CTAs per SM");

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);
EncodeTiledFn g_encode = nullptr;

// 3-D tiled tensor map over an [nz][ny][nx] FP32 array with a bw x bh x 1 box.  Cached per
// (pointer, extents, box): encoding costs a few microseconds on the host.
bool tensor_map(const float* ptr, const LevelGeom& g, int bw, int bh, CUtensorMap* out) {
    typedef std::tuple<const float*, int, int, int, int, int> Key;
    static std::map<Key, CUtensorMap> cache;
    static std::mutex cache_mutex;   // contexts on several host threads share the cache
    std::lock_guard<std::mutex> lock(cache_mutex);
    const Key key(ptr, g.n[0], g.n[1], g.n[2], bw, bh);
    auto it = cache.find(key);
    if (it != cache.end()) {
        *out = it->second;
        return true;
    }
    if (!g_encode) return false;
    const cuuint64_t dims[3] = {(cuuint64_t)g.n[0], (cuuint64_t)g.n[1], (cuuint64_t)g.n[2]};
    const cuuint64_t strides[2] = {(cuuint64_t)g.n[0] * 4, (cuuint64_t)g.n[0] * g.n[1] * 4};
    const cuuint32_t box[3] = {(cuuint32_t)bw, (cuuint32_t)bh, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    alignas(64) CUtensorMap tm;
    const CUresult r = g_encode(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(ptr), dims, strides,
                                box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return false;
    if (cache.size() > 4096) cache.clear();
    cache[key] = tm;
    *out = tm;
    return true;
}

bool sweep_supported(const LevelGeom& g) { return sweep_v2_supported(g); }

bool bulk_supported(const LevelGeom& g) {
    return g_encode && g.n[0] >= 128 && g.n[0] % 128 == 0 && g.n[1] >= 4 && g.n[2] >= 8;
}

bool tma_shape_ok(const LevelGeom& g) { return bulk_supported(g); }

static bool rb_sweep_bulk_launch(const LevelGeom& g, const float* L, const float* src, float* dst, const float* b,
                                 const float* omega, int first_colour, const ReduceBuf* norm, int slot_rr,
                                 int slot_ref, const int* run_flag, const UniArgs& uni, cudaStream_t s,
                                 const float* e_c = nullptr);

bool bulk_sweep_edge(const LevelGeom& g, bool norm);
static unsigned int bulk_grid(const LevelGeom& g, int* zchunk_out) {
    const int tiles_x = g.n[0] / Bulk::TX, tiles_y = (g.n[1] + Bulk::TY - 1) / Bulk::TY;
    const int zchunk = choose_zchunk((long long)tiles_x * tiles_y, g.n[2], kZChunkPref, kZChunkMin, 148, 0);
    if (zchunk_out) *zchunk_out = zchunk;
    return (unsigned int)(tiles_x * tiles_y * ((g.n[2] + zchunk - 1) / zchunk));
}

// The tiling of the TMA-fed sweep on this level (for gmg_stats' count of lean-path cells)
bool bulk_sweep_tiling(const LevelGeom& g, int* tile_y, int* zchunk) {
    if (!bulk_supported(g)) return false;
    *tile_y = Bulk::TY;
    bulk_grid(g, zchunk);
    return true;
}

// rb_sweep_with_norm will run on this level (shape fits the TMA kernel, one partial per CTA fits)
bool sweep_norm_supported(const LevelGeom& g) {
    return tma_shape_ok(g) && bulk_grid(g, nullptr) <= GMG_REDUCE_MAX_BLOCKS;
}

// The TMA-fed sweep of this level takes the prolongation + correction along (lean tiles on the fly,
// the others through the scratch copy): uniform bricks marked, 2x2x2 coarsening, scratch at hand, and
// at least half of the tiles lean when the coefficients were last counted (uni.fold): a remaining
// tile costs 11.8 B per cell for its corrected copy against 8.5 for the separate pass.
bool sweep_fuses_prolong(const LevelGeom& g, const UniArgs& uni) {
    return tma_shape_ok(g) && uni.brick && uni.left_list && uni.scratch && uni.fold && g.c[0] == 2 && g.c[1] == 2 &&
           g.c[2] == 2;
}

void rb_sweep(const LevelGeom& g, const float* L, const float* src, float* dst, const float* b,
              const float* omega, int first_colour, const float* e_c, int allow_tma, const UniArgs& uni,
              cudaStream_t s) {
    // in front of the TMA kernel the caller applies the prolongation as its own pass (e_c == nullptr)
    // unless sweep_fuses_prolong
    if (allow_tma && e_c && sweep_fuses_prolong(g, uni) &&
        rb_sweep_bulk_launch(g, L, src, dst, b, omega, first_colour, nullptr, 0, 0, nullptr, uni, s, e_c))
        return;
    if (allow_tma && !e_c && rb_sweep_bulk_launch(g, L, src, dst, b, omega, first_colour, nullptr, 0, 0, nullptr, uni, s))
        return;
    rb_sweep_v2(g, L, src, dst, b, omega, first_colour, e_c, s);
}

// The same sweep src -> dst which ALSO leaves sum r^2 (r = b - A src, active cells) in
// red[slot_rr] and (slot_ref >= 0) sum b^2 over active cells in red[slot_ref]: the stopping-test norm of the
// iterate a V-cycle starts from, for the price of two more stencils per thread and step instead
// of a 20 B/cell pass.  run_flag != nullptr: the launch is a no-op unless *run_flag != 0.
// false = this level cannot use the TMA kernel (nothing launched).
bool rb_sweep_with_norm(const LevelGeom& g, const float* L, const float* src, float* dst, const float* b,
                        const float* omega, int first_colour, ReduceBuf rb, int slot_rr, int slot_ref,
                        const int* run_flag, const UniArgs& uni, cudaStream_t s) {
    return rb_sweep_bulk_launch(g, L, src, dst, b, omega, first_colour, &rb, slot_rr, slot_ref, run_flag, uni, s);
}
bool rb_sweep_if(const LevelGeom& g, const float* L, const float* src, float* dst, const float* b,
                 const float* omega, int first_colour, const int* run_flag, const UniArgs& uni, cudaStream_t s) {
    return rb_sweep_bulk_launch(g, L, src, dst, b, omega, first_colour, nullptr, 0, 0, run_flag, uni, s);
}

// Which instantiation of k_rb_sweep_bulk a level gets: true = EDGE (the kernel that carries the
// boundary-box body), false = the two-body kernel whose y-boundary tile rows take row copies.
// Few tile rows, or walls in y: EDGE.  The norm-carrying variants come out faster with the third
// body at any size (5.91 vs 6.04 ms at 1024^3 in the same A/B).
bool bulk_sweep_edge(const LevelGeom& g, bool norm) {
    const int tiles_y = (g.n[1] + Bulk::TY - 1) / Bulk::TY;
    return g.bc[1] != 0 || (tiles_y >= 2 && (tiles_y <= 40 || norm));
}

static bool rb_sweep_bulk_launch(const LevelGeom& g, const float* L, const float* src, float* dst, const float* b,
                                 const float* omega, int first_colour, const ReduceBuf* norm, int slot_rr,
                                 int slot_ref, const int* run_flag, const UniArgs& uni_in, cudaStream_t s,
                                 const float* e_c) {
    BulkMaps maps;
    const size_t N = (size_t)g.N;
    bool ok = tma_shape_ok(g);
    int zchunk = 0;
    const unsigned int grid = bulk_grid(g, &zchunk);
    // No lean tile on this level (walls all around, bodies everywhere) and the host knows it: one
    // kernel over the whole grid, no empty k_rb_sweep_lean launch, no fork and join.
    UniArgs uni = uni_in;
    if (uni.brick && uni.left_list && uni.left_n == (int)grid) {
        uni.brick = nullptr; uni.left_list = nullptr; uni.left_count = nullptr;
    }
    if (e_c && !uni.brick) return false;
    const float* psrc = src;   // the array the p boxes are cut from
    auto set = [&](MapSet& m, int hp, int hc, int hly) {
        return tensor_map(psrc, g, Bulk::TX, hp, &m.p_main) && tensor_map(psrc, g, 4, hp, &m.p_halo) &&
               tensor_map(L + 2 * N, g, Bulk::TX, hc, &m.lz) && tensor_map(L, g, Bulk::TX, hc, &m.lx) &&
               tensor_map(L + N, g, Bulk::TX, hly, &m.ly) && tensor_map(b, g, Bulk::TX, hc, &m.b);
    };
    ok = ok && set(maps.m[0], Bulk::SH, Bulk::ROWS, Bulk::ROWS + 1);
    const int tiles_y_ = (g.n[1] + Bulk::TY - 1) / Bulk::TY;
    const int rem = g.n[1] - (tiles_y_ - 1) * Bulk::TY;      // rows of the final tile row
    const bool edge = bulk_sweep_edge(g, norm != nullptr);
    if (ok && (edge || uni.brick) && g.bc[1] == 0 && tiles_y_ >= 2) {
        ok = ok && set(maps.m[1], Bulk::SH - 2, Bulk::ROWS - 1, Bulk::ROWS);   // FIRST: from y = 0
        ok = ok && set(maps.m[2], rem + 2, rem + 1, rem + 1);                  // FINAL: up to y = ny - 1
    } else {
        maps.m[1] = maps.m[0];
        maps.m[2] = maps.m[0];
    }
    // e_c: the sweep folds the prolongation in (sweep_fuses_prolong).  The lean kernel corrects src on
    // the fly; the kernel of the remaining tiles reads the corrected copy k_prolong_tiles leaves in
    // uni.scratch, through a second set of p boxes.
    BulkMaps gmaps = maps;
    if (ok && e_c) {
        psrc = uni.scratch;
        ok = set(gmaps.m[0], Bulk::SH, Bulk::ROWS, Bulk::ROWS + 1);
        if (ok && g.bc[1] == 0 && tiles_y_ >= 2) {
            ok = ok && set(gmaps.m[1], Bulk::SH - 2, Bulk::ROWS - 1, Bulk::ROWS);
            ok = ok && set(gmaps.m[2], rem + 2, rem + 1, rem + 1);
        } else {
            gmaps.m[1] = gmaps.m[0];
            gmaps.m[2] = gmaps.m[0];
        }
        psrc = src;
    }
    if (!ok) return false;
    BulkArgs a;
    a.e_c = e_c;
    a.g = g; a.L = L; a.src = src; a.dst = dst; a.b = b; a.omega = omega;
    a.first_colour = first_colour;
    a.rb = norm ? *norm : ReduceBuf{nullptr, nullptr, nullptr, POST_NONE, 0.0};
    a.slot_rr = slot_rr; a.slot_ref = slot_ref;
    a.run_flag = run_flag;
    a.uni = uni;
    a.tiles_x = g.n[0] / Bulk::TX;
    a.tiles_y = (g.n[1] + Bulk::TY - 1) / Bulk::TY;
    a.zchunk = zchunk;
    a.ntiles = (int)grid;
    if (grid > GMG_REDUCE_MAX_BLOCKS && norm) return false;
    const int nv = (norm && slot_ref >= 0) ? 2 : (norm ? 1 : 0);
    // grid of the kernel of the remaining tiles: the list's length where the host knows it
    const unsigned int gl = (uni.brick && uni.left_list && uni.left_n >= 0) ? (unsigned int)uni.left_n : grid;
    // With uniform bricks marked, two kernels share the grid: k_rb_sweep_lean (two CTAs per SM) takes
    // the lean tiles, k_rb_sweep_bulk the rest.  They touch disjoint tiles of dst, so they run side by
    // side -- the general one first, on a forked stream, so that its few long CTAs are spread over the
    // SMs while the lean CTAs fill in -- and the caller's stream waits for both.  The partial sums of a
    // norm-carrying sweep are shared: every tile is worked on by exactly one kernel and only working
    // CTAs take a ticket, so the last of either kernel finishes the sum.
    cudaStream_t sg = s;
    const bool fork = uni.brick && uni.side_stream;
    if (fork) {
        sg = (cudaStream_t)uni.side_stream;
        cudaEventRecord((cudaEvent_t)uni.ev_fork, s);
        cudaStreamWaitEvent(sg, (cudaEvent_t)uni.ev_fork, 0);
    }
    auto launch_lean = [&]() {
        if (e_c) k_rb_sweep_lean_pro<Lean><<<grid, Lean2Threads<false>::value, Lean::SMEM, s>>>(a, maps);
        else if (nv == 2) k_rb_sweep_lean<Lean, 2><<<grid, Lean2Threads<true>::value, Lean::SMEM, s>>>(a, maps);
        else if (nv == 1) k_rb_sweep_lean<Lean, 1><<<grid, Lean2Threads<true>::value, Lean::SMEM, s>>>(a, maps);
        else k_rb_sweep_lean<Lean, 0><<<grid, Lean2Threads<false>::value, Lean::SMEM, s>>>(a, maps);
    };
    if (uni.brick && !fork) launch_lean();
    BulkArgs ga = a;   // the kernel of the remaining tiles
    if (e_c && gl != 0) {
        k_prolong_tiles<Bulk><<<gl, 256, 0, sg>>>(a, uni.scratch);
        ga.src = uni.scratch;
    }
    const BulkMaps& bm = e_c ? gmaps : maps;
    if (gl == 0) {
        // every tile is lean
    } else if (edge) {
        if (nv == 2) k_rb_sweep_bulk<Bulk, 2, true><<<gl, Bulk::THREADS, Bulk::SMEM, sg>>>(ga, bm);
        else if (nv == 1) k_rb_sweep_bulk<Bulk, 1, true><<<gl, Bulk::THREADS, Bulk::SMEM, sg>>>(ga, bm);
        else k_rb_sweep_bulk<Bulk, 0, true><<<gl, Bulk::THREADS, Bulk::SMEM, sg>>>(ga, bm);
    } else {
        if (nv == 2) k_rb_sweep_bulk<Bulk, 2, false><<<gl, Bulk::THREADS, Bulk::SMEM, sg>>>(ga, bm);
        else if (nv == 1) k_rb_sweep_bulk<Bulk, 1, false><<<gl, Bulk::THREADS, Bulk::SMEM, sg>>>(ga, bm);
        else k_rb_sweep_bulk<Bulk, 0, false><<<gl, Bulk::THREADS, Bulk::SMEM, sg>>>(ga, bm);
    }
    if (fork) {
        launch_lean();
        cudaEventRecord((cudaEvent_t)uni.ev_join, sg);
        cudaStreamWaitEvent(s, (cudaEvent_t)uni.ev_join, 0);
    }
    return true;
}

int configure() {
    cudaError_t e = (cudaError_t)configure_v2();
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_rb_sweep_bulk<Bulk, 0, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Bulk::SMEM);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_rb_sweep_bulk<Bulk, 1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Bulk::SMEM);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_rb_sweep_bulk<Bulk, 2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Bulk::SMEM);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_rb_sweep_bulk<Bulk, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Bulk::SMEM);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_rb_sweep_bulk<Bulk, 1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Bulk::SMEM);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_rb_sweep_bulk<Bulk, 2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Bulk::SMEM);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_rb_sweep_lean<Lean, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Lean::SMEM);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_rb_sweep_lean<Lean, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Lean::SMEM);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_rb_sweep_lean<Lean, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Lean::SMEM);
    // two lean CTAs per SM need the large shared-memory carve-out
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_rb_sweep_lean_pro<Lean>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Lean::SMEM);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_rb_sweep_lean_pro<Lean>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_rb_sweep_lean<Lean, 0>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_rb_sweep_lean<Lean, 1>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_rb_sweep_lean<Lean, 2>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    if (e == cudaSuccess && !g_encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            g_encode = (EncodeTiledFn)fn;
        else
            cudaGetLastError();  // the TMA path is simply not used
    }
    return (int)e;
}

}  // namespace gmgf

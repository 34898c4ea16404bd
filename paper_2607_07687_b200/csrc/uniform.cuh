// uniform.cuh -- "uniform bricks": where the face coefficients of a level are one constant per
// direction (away from immersed bodies the BDIM coefficient is exactly 1: BASELINE.json:north_star
// "per-face coefficients L in [0,1]", "immersed-boundary flows"; on coarse levels
// reading O5 turns that into (prod_{e!=d} C_e)/C_d, a power of two), the TMA-fed kernels need not
// LOAD the three coefficient streams at all: 12 of the 24 B/cell of a sweep, 12 of the 20.5 B/cell
// of the residual pass.  SURVEY.md S8(d) names this "a lossless 'tile is all L=1' flag that skips
// L loads ... an honest optimisation only if reported as such": it is lossless -- the same
// apply7/diag6/relax operations run on the constants, so every cell gets the same bits as on the
// general path (tests compare bit for bit) -- and it is reported (gmg_stats.uniform_fraction,
// bytes_as_run; bench.py keeps the 24-B accounting as the reference line).
//
// gmg_set_coeffs marks every brick of kUBX x kUBY x kUBZ cells whose stored Lx, Ly, Lz all equal
// the level's constants (the marking rides on the coefficient-coarsening pass, which reads every
// value anyway); a CTA takes the lean path iff every brick its footprint touches is marked and the
// footprint stays clear of Neumann walls (wall faces carry 0, not the constant).  Bricks are 32
// cells wide so that the two halo columns of a 128-wide tile cost a quarter of the neighbouring
// tile, not all of it (1024^3, 64 spheres: 90 % of the cells on the lean path instead of 83 %).
#pragma once
#include "gmg_internal.h"

namespace gmgf {

static constexpr int kUBX = 32, kUBY = 8, kUBZ = 8;

struct UniArgs {
    const unsigned char* brick;  // [nbz][nby][nbx] flags of the level; nullptr: lean path disabled
    float ux, uy, uz;            // the level's constants
    // the tiles of the sweep that are NOT lean, as a compact list (built by gmg_set_coeffs on the
    // device): the kernel of the remaining tiles launches one CTA per entry instead of a grid full
    // of CTAs that return at once.  left_n: the count as the host knows it, -1 = not read back yet
    // (gmg_pressure_step): the kernel then gets the full grid and bounds itself by *left_count.
    const int* left_list;
    const unsigned int* left_count;
    int left_n;
    // a level-0-sized scratch array (workspace): the corrected iterate p + P e_c over the footprints of
    // the non-lean tiles, for the sweep that folds the prolongation in (sweep_lean2.cuh, PRO)
    float* scratch;
    // host-side hint, kept across coefficient updates: at the last count at least half of the level's
    // tiles were lean, so folding the prolongation into the sweep pays
    int fold;
    // host side only: a side stream and two events with which a launcher runs the kernel of the
    // remaining (non-uniform) tiles beside the lean kernel; nullptr = one after the other
    void* side_stream;
    void* ev_fork;
    void* ev_join;
};

__host__ __device__ inline int ub_count(int n, int b) { return (n + b - 1) / b; }
__host__ __device__ inline int ub_floor_div(int v, int b) { return v >= 0 ? v / b : -((-v + b - 1) / b); }

// Brick range of the cell range [lo, hi] (inclusive, may leave [0, n)) on one axis: first brick
// (wrapped into [0, nb)) and how many consecutive (cyclic) bricks.  Returns false when the range
// leaves the domain on a Neumann axis.
__host__ __device__ inline bool ub_axis(int lo, int hi, int n, int b, int neumann, int& first, int& cnt) {
    const int nb = ub_count(n, b);
    if (neumann && (lo < 0 || hi >= n)) return false;
    if (hi - lo + 1 >= n) { first = 0; cnt = nb; return true; }
    const int lo_w = lo < 0 ? lo + n : (lo >= n ? lo - n : lo);          // range length < n: one wrap at most
    const int hi_w = hi < 0 ? hi + n : (hi >= n ? hi - n : hi);
    const int bl = lo_w / b, bh = hi_w / b;
    first = bl;
    cnt = bh >= bl && hi_w >= lo_w ? bh - bl + 1 : (nb - bl) + bh + 1;   // wrapped range: up to the end, then from 0
    if (cnt > nb) cnt = nb;
    return true;
}

// Host or single-thread version (statistics): are all bricks of the box marked?
__host__ __device__ inline bool ub_box_uniform(const LevelGeom& g, const unsigned char* brick, int x0, int x1,
                                               int y0, int y1, int z0, int z1) {
    int fx, cx, fy, cy, fz, cz;
    if (!ub_axis(x0, x1, g.n[0], kUBX, g.bc[0], fx, cx)) return false;
    if (!ub_axis(y0, y1, g.n[1], kUBY, g.bc[1], fy, cy)) return false;
    if (!ub_axis(z0, z1, g.n[2], kUBZ, g.bc[2], fz, cz)) return false;
    const int nbx = ub_count(g.n[0], kUBX), nby = ub_count(g.n[1], kUBY), nbz = ub_count(g.n[2], kUBZ);
    for (int k = 0; k < cz; ++k)
        for (int j = 0; j < cy; ++j)
            for (int i = 0; i < cx; ++i) {
                const int bx = (fx + i) % nbx, by = (fy + j) % nby, bz = (fz + k) % nbz;
                if (!brick[((size_t)bz * nby + by) * nbx + bx]) return false;
            }
    return true;
}

#ifdef __CUDACC__
// Warp-collective version: every lane returns the verdict.
__device__ __forceinline__ bool ub_box_uniform_warp(const LevelGeom& g, const unsigned char* brick, int x0, int x1,
                                                    int y0, int y1, int z0, int z1, int lane) {
    int fx, cx, fy, cy, fz, cz;
    bool ok = ub_axis(x0, x1, g.n[0], kUBX, g.bc[0], fx, cx);
    ok = ub_axis(y0, y1, g.n[1], kUBY, g.bc[1], fy, cy) && ok;
    ok = ub_axis(z0, z1, g.n[2], kUBZ, g.bc[2], fz, cz) && ok;
    if (ok) {
        const int nbx = ub_count(g.n[0], kUBX), nby = ub_count(g.n[1], kUBY), nbz = ub_count(g.n[2], kUBZ);
        const int total = cx * cy * cz;
        for (int t = lane; t < total; t += 32) {
            const int i = t % cx, r = t / cx;
            const int j = r % cy, k = r / cy;
            const int bx = (fx + i) % nbx, by = (fy + j) % nby, bz = (fz + k) % nbz;
            ok = ok && (__ldg(brick + ((size_t)bz * nby + by) * nbx + bx) != 0);
        }
    }
    return __all_sync(0xffffffffu, ok);
}
#endif

}  // namespace gmgf

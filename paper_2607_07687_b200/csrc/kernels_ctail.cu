// kernels_ctail.cu -- the coarse tail of the V-cycle on a thread-block CLUSTER.
//
// kernels_tail.cu runs the levels that fit ONE CTA's shared memory; the level above them (32^3 for
// the 128^3 configs) then still costs a dozen launch- and latency-bound kernels per cycle.  Here
// a cluster of 8 CTAs (8 SMs, 8 x 200 KB of shared memory) holds those levels too:
//   * a DISTRIBUTED level (1024 < N <= 32768 cells, nz % 8 == 0) is cut into 8 z-slabs, one per
//     CTA: six face weights, p, b and a residual scratch per cell.  x and y neighbours are local;
//     the z neighbours of a slab's first and last plane are read from the neighbouring CTA's
//     shared memory (DSMEM, ld.shared::cluster), and a colour half-sweep ends in a cluster
//     barrier instead of a kernel boundary;
//   * a SMALL level (N <= 1024) lives in CTA 0 and runs exactly as in kernels_tail.cu while the
//     other CTAs wait at the next cluster barrier.
// Same per-cell arithmetic (stencil.cuh) and child summation order (restrict_tree) as every other
// kernel, so results are bit-identical to the single-CTA tail and to the per-level kernels.
// DESIGN.md reading O7.
#include "tail_common.cuh"

namespace gmgk {
using namespace gmgd;

static constexpr int kCR = 8;       // CTAs per cluster
static constexpr int kCSlots = 4;   // cells of a distributed level per thread (per <= 4096)

struct CTailArgs {
    TailArgs t;
    CLevelPlan lv[GMG_TAIL_MAX_LEVELS];
};

__device__ __forceinline__ void cluster_sync() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ int cluster_rank() {
    int r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t saddr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
// shared::cluster address of the same shared-memory location in CTA `rank`
__device__ __forceinline__ uint32_t map_rank(uint32_t a, int rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(rank));
    return r;
}
// Generic pointer to a shared::cluster address: loads through it are ordinary loads, which the
// compiler may batch and overlap (and orders against the barriers' memory clobber).
__device__ __forceinline__ const float* cluster_ptr(uint32_t a) {
    unsigned long long g;
    asm("cvta.shared::cluster.u64 %0, %1;" : "=l"(g) : "l"((unsigned long long)a));
    return reinterpret_cast<const float*>(g);
}
__device__ __forceinline__ float ld_cluster(uint32_t a) { return *cluster_ptr(a); }

// n floats global -> shared by the whole CTA (read-only path: the loads need not be ordered
// against the shared-memory stores)
__device__ __forceinline__ void copy_g2s(float* dst, const float* __restrict__ src, int n) {
    for (int u = threadIdx.x; u < n; u += kTailThreads) dst[u] = __ldg(src + u);
}
// The six face-weight arrays of a level: W[f][0..per) <- src[f * N + 0..per), all six loads of a
// cell group in flight before the first store.
__device__ __forceinline__ void copy_weights(float* W, const float* __restrict__ src, int N, int per) {
    const bool vec = ((per & 3) == 0) && ((N & 3) == 0) && ((reinterpret_cast<size_t>(src) & 15) == 0) &&
                     ((saddr(W) & 15) == 0);
    if (vec) {
        for (int u = threadIdx.x; u < (per >> 2); u += kTailThreads) {
            float4 v[6];
#pragma unroll
            for (int f = 0; f < 6; ++f) v[f] = __ldg(reinterpret_cast<const float4*>(src + (size_t)f * N) + u);
#pragma unroll
            for (int f = 0; f < 6; ++f) reinterpret_cast<float4*>(W + f * per)[u] = v[f];
        }
    } else {
        for (int u = threadIdx.x; u < per; u += kTailThreads) {
            float v[6];
#pragma unroll
            for (int f = 0; f < 6; ++f) v[f] = __ldg(src + (size_t)f * N + u);
#pragma unroll
            for (int f = 0; f < 6; ++f) W[f * per + u] = v[f];
        }
    }
}

struct CLevel {  // one level as this CTA sees it
    LevelGeom g;
    int dist, per, c0;  // c0 = first global cell held here
    float *W, *p, *b, *r;
};

// Neighbours of the local cell l of a distributed level, two words per cell so that the four slots
// of a thread stay in registers (a cluster barrier invalidates L1, spilled slots would come back
// from L2 after every half-sweep): x/y neighbours as local indices (12 bits each), the colour, and
// one flag per z direction: the neighbouring plane lies in ANOTHER CTA's slab.  A slab is whole
// planes, so only its first and its last plane look across; the other z accesses are plain
// shared-memory loads at l -+ plane.
struct CSlot {
    uint32_t x, y;  // x = xm | xp << 12 | zm remote << 24 | zp remote << 25 | colour << 30 (3 = no cell); y = ym | yp << 12
    __device__ __forceinline__ int colour() const { return (int)(x >> 30); }
};

// What the z accesses of a level need besides the slot
struct CZ {
    int plane, wrap;      // wrap = per - plane: from the first plane of a slab to the last of the one below
    uint32_t pa;          // shared address of p
    int rm, rp;           // ranks of the slabs below and above (periodic; across a wall the weight is zero)
};

__device__ __forceinline__ CZ make_cz(const CLevel& L, int rank) {
    CZ z;
    z.plane = L.g.n[0] * L.g.n[1];
    z.wrap = L.per - z.plane;
    z.pa = saddr(L.p);
    z.rm = (rank + kCR - 1) % kCR;
    z.rp = (rank + 1) % kCR;
    return z;
}

// Visits the cells tid, tid + T, tid + 2T, ... of the slab with their global (i, j, k): one division
// pair for the first cell, then (i, j, k) advance by T cells with carries.
template <class F>
__device__ __forceinline__ void for_slab_cells(const CLevel& L, F f) {
    const int nx = L.g.n[0], ny = L.g.n[1], plane = nx * ny;
    const int di = kTailThreads % nx, dj = (kTailThreads / nx) % ny, dk = kTailThreads / plane;
    const int c = L.c0 + (int)threadIdx.x;
    int k = c / plane;
    const int rem = c - k * plane;
    int j = rem / nx, i = rem - j * nx;
#pragma unroll
    for (int m = 0; m < kCSlots; ++m) {
        const int l = (int)threadIdx.x + m * kTailThreads;
        f(m, l, l < L.per, i, j, k);
        i += di;
        if (i >= nx) { i -= nx; ++j; }
        j += dj;
        if (j >= ny) { j -= ny; ++k; }
        k += dk;
    }
}

__device__ __forceinline__ void make_slots_dist(const CLevel& L, int rank, CSlot (&s)[kCSlots]) {
    const int nx = L.g.n[0], ny = L.g.n[1], plane = nx * ny;
    const int zs = L.g.n[2] / kCR;                 // planes per slab (per = zs * plane)
    for_slab_cells(L, [&](int m, int l, bool in, int i, int j, int k) {
        CSlot q;
        q.x = 3u << 30;
        q.y = 0;
        if (in) {
            const int xm = (i == 0) ? l + (nx - 1) : l - 1;
            const int xp = (i == nx - 1) ? l - (nx - 1) : l + 1;
            const int ym = (j == 0) ? l + (plane - nx) : l - nx;
            const int yp = (j == ny - 1) ? l - (plane - nx) : l + nx;
            const int kl = k - rank * zs;          // plane index inside the slab
            q.x = (uint32_t)xm | ((uint32_t)xp << 12) | ((uint32_t)(kl == 0) << 24) | ((uint32_t)(kl == zs - 1) << 25) |
                  ((uint32_t)((i + j + k) & 1) << 30);
            q.y = (uint32_t)ym | ((uint32_t)yp << 12);
        }
        s[m] = q;
    });
}

__device__ __forceinline__ Cell slot_cell(const CLevel& L, const CZ& z, const CSlot& s, int l) {
    const int per = L.per;
    const float* W = L.W;
    const float w0 = W[l], w1 = W[per + l], w2 = W[2 * per + l], w3 = W[3 * per + l], w4 = W[4 * per + l],
                w5 = W[5 * per + l];
    const float* p = L.p;
    // below / above: the same column one plane away -- in the neighbouring slab its last / first plane
    const float pzm = (s.x & (1u << 24)) ? ld_cluster(map_rank(z.pa + 4u * (uint32_t)(l + z.wrap), z.rm)) : p[l - z.plane];
    const float pzp = (s.x & (1u << 25)) ? ld_cluster(map_rank(z.pa + 4u * (uint32_t)(l - z.wrap), z.rp)) : p[l + z.plane];
    Cell r;
    r.pc = p[l];
    r.Ap = apply7(r.pc, w0, w1, w2, w3, w4, w5, p[s.x & 0xfffu], p[(s.x >> 12) & 0xfffu], p[s.y & 0xfffu],
                  p[s.y >> 12], pzm, pzp);
    r.D = diag6(w0, w1, w2, w3, w4, w5);
    return r;
}

// `count` red-black sweeps on a distributed level; every colour half-sweep ends in a cluster barrier.
__device__ __forceinline__ void dist_sweeps(const CLevel& L, const CZ& z, const CSlot (&s)[kCSlots], float omega,
                                            int count, int first) {
    for (int h = 0; h < 2 * count; ++h) {
        const int colour = (h & 1) ? 1 - first : first;
#pragma unroll
        for (int m = 0; m < kCSlots; ++m) {
            if (s[m].colour() != colour) continue;
            const int l = threadIdx.x + m * kTailThreads;
            const Cell c = slot_cell(L, z, s[m], l);
            L.p[l] = relax(c.pc, L.b[l], c.Ap, c.D, omega);
        }
        cluster_sync();
    }
}

// Sweeps on any level; all CTAs leave through the same number of cluster barriers.
__device__ __forceinline__ void level_sweeps(const CLevel& L, const CSlot (&s)[kCSlots], int rank, float omega,
                                             int count, int first) {
    if (count <= 0) return;
    if (L.dist) {
        dist_sweeps(L, make_cz(L, rank), s, omega, count, first);
    } else {
        if (rank == 0) {
            int T = ((int)L.g.N + 31) / 32 * 32;
            T = T > kTailThreads ? kTailThreads : T;
            tail_sweeps(L.g, L.W, L.p, L.b, omega, count, first, T);
        }
        cluster_sync();
    }
}

__global__ void __cluster_dims__(kCR, 1, 1) __launch_bounds__(kTailThreads, 1) k_tail_cluster(const CTailArgs a) {
    extern __shared__ __align__(16) float smem[];
    const int tid = threadIdx.x;
    const int rank = cluster_rank();
    const int nlev = a.t.nlev, last = nlev - 1;
    const float omega = *a.t.omega;
    auto level = [&](int t) {
        CLevel L;
        L.g = a.t.g[t];
        L.dist = a.lv[t].dist;
        L.per = a.lv[t].per;
        L.c0 = L.dist ? rank * L.per : 0;
        L.W = smem + a.lv[t].off;
        L.p = L.W + 6 * L.per;
        L.b = L.p + L.per;
        L.r = L.b + L.per;
        return L;
    };
    auto holds = [&](const CLevel& L) { return L.dist || rank == 0; };

    // ---- face weights of every level (precomputed by gmg_set_coeffs), right-hand side, guess ----
    for (int t = 0; t < nlev; ++t) {
        const CLevel L = level(t);
        if (!holds(L)) continue;
        const int N = (int)L.g.N;
        copy_weights(L.W, a.t.W[t] + L.c0, N, L.per);
    }
    {
        const CLevel L = level(0);
        if (holds(L)) {
            copy_g2s(L.b, a.t.b_in + L.c0, L.per);
            if (a.t.p_in) copy_g2s(L.p, a.t.p_in + L.c0, L.per);
            else
                for (int l = tid; l < L.per; l += kTailThreads) L.p[l] = 0.0f;
        }
    }
    cluster_sync();

    CSlot s[kCSlots];
    auto make_slots = [&](const CLevel& L) {
        if (L.dist) {
            make_slots_dist(L, rank, s);
        } else {   // small level: no slots
#pragma unroll
            for (int m = 0; m < kCSlots; ++m) {
                s[m].x = 3u << 30;
                s[m].y = 0;
            }
        }
    };

    // ---- down leg ---------------------------------------------------------------------------------
    for (int t = 0; t < last; ++t) {
        const CLevel L = level(t), Lc = level(t + 1);
        make_slots(L);
        level_sweeps(L, s, rank, omega, a.t.nu1, 0);
        // residual of the cells held here (0 on inactive cells)
        if (L.dist) {
            const CZ cz_res = make_cz(L, rank);
#pragma unroll
            for (int m = 0; m < kCSlots; ++m) {
                if (s[m].colour() > 1) continue;
                const int l = tid + m * kTailThreads;
                const Cell c = slot_cell(L, cz_res, s[m], l);
                L.r[l] = (c.D != 0.0f) ? L.b[l] - c.Ap : 0.0f;
            }
        } else if (rank == 0) {
            const int N = (int)L.g.N, nx = L.g.n[0], ny = L.g.n[1];
            for (int c = tid; c < N; c += kTailThreads) {
                const int row = c / nx, i = c - row * nx, k = row / ny, j = row - k * ny;
                const Cell q = tail_cell(L.g, L.W, L.p, c, i, j, k);
                L.r[c] = (q.D != 0.0f) ? L.b[c] - q.Ap : 0.0f;
            }
        }
        cluster_sync();
        // restriction: the holder of a coarse cell sums its children (wherever they live)
        if (holds(Lc)) {
            const int cx = L.g.c[0], cy = L.g.c[1], cz = L.g.c[2];
            const int ncx = L.g.n[0] / cx, ncy = L.g.n[1] / cy;
            const uint32_t ra = saddr(L.r);
            for (int l = tid; l < Lc.per; l += kTailThreads) {
                const int u = Lc.c0 + l;
                const int row = u / ncx, I = u - row * ncx, K = row / ncy, J = row - K * ncy;
                if (Lc.dist) {
                    // both levels cut into slabs: a coarse slab's children are this CTA's fine slab
                    // (planes cz K .. cz K + cz - 1 with K in the coarse slab): plain shared-memory loads
                    Lc.b[l] = restrict_tree(cx, cy, cz, [&](int e, int bb, int aa) {
                        const int f = (cx * I + e) + L.g.n[0] * ((cy * J + bb) + L.g.n[1] * (cz * K + aa));
                        return L.r[f - L.c0];
                    });
                } else {
                    Lc.b[l] = restrict_tree(cx, cy, cz, [&](int e, int bb, int aa) {
                        const int f = (cx * I + e) + L.g.n[0] * ((cy * J + bb) + L.g.n[1] * (cz * K + aa));
                        const int fr = L.dist ? f / L.per : 0;
                        return ld_cluster(map_rank(ra + 4u * (uint32_t)(f - fr * L.per), fr));
                    });
                }
                Lc.p[l] = 0.0f;
            }
        }
        cluster_sync();
    }
    // ---- coarsest level (reading O7: nu_coarse sweeps; O11: symmetric split) -----------------------
    {
        const CLevel L = level(last);
        make_slots(L);
        if (!a.t.sym) {
            level_sweeps(L, s, rank, omega, a.t.nuc, 0);
        } else {
            level_sweeps(L, s, rank, omega, a.t.nuc / 2, 0);
            level_sweeps(L, s, rank, omega, a.t.nuc / 2, 1);
        }
    }
    // ---- up leg -----------------------------------------------------------------------------------
    for (int t = last - 1; t >= 0; --t) {
        const CLevel L = level(t), Lc = level(t + 1);
        if (L.dist) {
            // factors are 1 or 2.  With the coarse level cut into slabs too, the parents of this
            // slab are the CTA's own coarse slab.
            const int sx = L.g.c[0] >> 1, sy = L.g.c[1] >> 1, sz = L.g.c[2] >> 1;
            const int ncx = L.g.n[0] >> sx, ncy = L.g.n[1] >> sy;
            const uint32_t pa = saddr(Lc.p);
            for_slab_cells(L, [&](int, int l, bool in, int i, int j, int k) {
                if (!in) return;
                const int parent = (i >> sx) + ncx * ((j >> sy) + ncy * (k >> sz));
                L.p[l] += Lc.dist ? Lc.p[parent - Lc.c0] : ld_cluster(map_rank(pa + 4u * (uint32_t)parent, 0));
            });
        } else if (rank == 0) {
            const int nx = L.g.n[0], ny = L.g.n[1];
            const int ncx = nx / L.g.c[0], ncy = ny / L.g.c[1];
            for (int l = tid; l < L.per; l += kTailThreads) {
                const int row = l / nx, i = l - row * nx, k = row / ny, j = row - k * ny;
                const int parent = (i / L.g.c[0]) + ncx * ((j / L.g.c[1]) + ncy * (k / L.g.c[2]));
                L.p[l] += Lc.p[parent];   // both levels live here
            }
        }
        cluster_sync();
        make_slots(L);
        level_sweeps(L, s, rank, omega, a.t.nu2, a.t.sym ? 1 : 0);
    }
    {
        const CLevel L = level(0);
        if (holds(L))
            for (int l = tid; l < L.per; l += kTailThreads) a.t.p_out[L.c0 + l] = L.p[l];
    }
    cluster_sync();  // no CTA leaves while another may still read its shared memory
}

// Lays the levels out; returns the dynamic shared memory per CTA, or 0 when this suffix of the
// hierarchy cannot run on the cluster (then the single-CTA tail / per-level kernels take it).
size_t ctail_plan(const LevelGeom* g, int nlev, CLevelPlan* lv) {
    if (nlev < 1 || nlev > GMG_TAIL_MAX_LEVELS) return 0;
    size_t off = 0;
    int ndist = 0;
    for (int t = 0; t < nlev; ++t) {
        const long long N = g[t].N;
        CLevelPlan L;
        if (N <= 1024) {
            L.dist = 0;
            L.per = (int)N;
        } else {
            if (N > (long long)kCR * kCSlots * kTailThreads || g[t].n[2] % kCR != 0) return 0;
            if (t > 0 && !lv[t - 1].dist) return 0;  // levels only shrink
            L.dist = 1;
            L.per = (int)(N / kCR);
            ++ndist;
        }
        L.off = (int)off;
        off += (size_t)9 * L.per;
        off = (off + 3) / 4 * 4;
        lv[t] = L;
    }
    if (ndist == 0) return 0;  // nothing the single-CTA tail could not do
    const size_t bytes = off * sizeof(float);
    return bytes <= 200 * 1024 ? bytes : 0;
}

int ctail_configure(size_t max_bytes) {
    return (int)cudaFuncSetAttribute(k_tail_cluster, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)max_bytes);
}

// Whether a cluster of kCR CTAs with this much shared memory can be resident on this device.
bool ctail_launchable(size_t smem_bytes) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(kCR, 1, 1);
    cfg.blockDim = dim3(kTailThreads, 1, 1);
    cfg.dynamicSmemBytes = smem_bytes;
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, k_tail_cluster, &cfg) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return n >= 1;
}

void ctail_vcycle(const TailArgs& t, const CLevelPlan* lv, size_t smem_bytes, cudaStream_t s) {
    CTailArgs a;
    a.t = t;
    for (int i = 0; i < t.nlev; ++i) a.lv[i] = lv[i];
    k_tail_cluster<<<kCR, kTailThreads, smem_bytes, s>>>(a);
}

}  // namespace gmgk

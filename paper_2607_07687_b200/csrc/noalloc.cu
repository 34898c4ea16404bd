// noalloc.cu -- gmg_residual_norm2_noalloc: the stopping-test norm ||b - A p||_2 over the active
// cells (readings O1, O2, O9; PAPER.md:39 S3 "global inner products") for callers that
// may not allocate: code under CUDA-graph capture, tight serving loops, harnesses that forbid
// cudaMalloc.  It is k_residual_norm2 (kernels_reduce.cu) with the reduction scratch -- the FP64
// block partials and the ticket of the "last block finishes the sum" stage -- in a file-scope
// device array instead of a context's allocation, and the result written to the caller's device
// pointer instead of a context's scalar block.  No context, no workspace, no cudaMalloc / cudaFree /
// allocating library call anywhere on the path.
//
// The array is one per GPU that loads the library and stays until the process exits (65,792 bytes).
// Every call shares it and it keeps the last call's contents: the partials are overwritten before
// they are read and the ticket is cleared on the stream in front of every launch, so a call that was
// cut short leaves nothing behind -- but two calls that OVERLAP on the GPU (different streams, or
// two host threads) race on it.  Serialise them.
#include <mutex>
#include <stdarg.h>
#include <stdio.h>

#include "stencil.cuh"

namespace {
using namespace gmgd;

constexpr int kRT = 256;             // threads per block, as k_residual_norm2
constexpr int kCellsPerThread = 8;   // grid = ceil(N / (kRT * kCellsPerThread)), as reduce_blocks()
constexpr long long kMaxCells = GMG_NOALLOC_MAX_CELLS;
constexpr int kMaxBlocks = (int)(kMaxCells / (kRT * kCellsPerThread));  // 8192 partials = 64 KB
constexpr int kTicketSlot = kMaxBlocks;   // the ticket lives behind the partials, in a 256-byte tail
constexpr int kScratchDoubles = kMaxBlocks + 32;
static_assert(kMaxCells % (kRT * kCellsPerThread) == 0, "whole blocks");

// In host code this name is a host-side stand-in, not a device address: the address a kernel can
// use comes from cudaGetSymbolAddress (scratch_of_current_device below).
static __device__ __align__(256) double g_noalloc_scratch[kScratchDoubles];

__global__ void __launch_bounds__(kRT)
k_residual_norm2_static(LevelGeom g, const float* __restrict__ L, const float* __restrict__ p,
                        const float* __restrict__ b, double* __restrict__ scratch,
                        double* __restrict__ out) {
    const int nx = g.n[0], ny = g.n[1];
    double acc = 0.0;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < g.N;
         t += (long long)gridDim.x * blockDim.x) {
        const long long row = t / nx;
        const int i = (int)(t - row * nx);
        const int k = (int)(row / ny);
        const int j = (int)(row - (long long)k * ny);
        const Cell c = cell_stencil(g, L, p, i, j, k);
        const float r = (c.D != 0.0f) ? b[t] - c.Ap : 0.0f;
        acc += (double)r * (double)r;
    }
    // two-stage, fixed order (the scheme of finish_reduction in stencil.cuh)
    __shared__ bool is_last;
    unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch + kTicketSlot);
    const double part = block_sum(acc);
    if (threadIdx.x == 0) {
        scratch[blockIdx.x] = part;
        __threadfence();
        is_last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    double a = 0.0;
    for (unsigned int i = threadIdx.x; i < gridDim.x; i += blockDim.x)
        a += ((volatile double*)scratch)[i];
    const double total = block_sum(a);
    if (threadIdx.x == 0) {
        out[0] = sqrt(total);
        *ticket = 0u;
    }
}

constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
double* g_scratch_ptr[kMaxDevices];  // device address of g_noalloc_scratch, per device; nullptr = not looked up

// Set-up, once per device, with that device current.
cudaError_t scratch_of_current_device(double** out, int* dev_out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    *dev_out = dev;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_ptr[dev]) {
        double* ptr = nullptr;
        e = cudaGetSymbolAddress((void**)&ptr, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        if (!ptr) return cudaErrorInvalidSymbol;
        g_scratch_ptr[dev] = ptr;
    }
    *out = g_scratch_ptr[dev];
    return cudaSuccess;
}

__attribute__((format(printf, 4, 5)))
int fail(char* err, size_t cap, int code, const char* fmt, ...) {
    if (err && cap) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(err, cap, fmt, ap);
        va_end(ap);
    }
    return code;
}

}  // namespace

extern "C" int gmg_residual_norm2_noalloc(int nx, int ny, int nz, const int bc[3], const float* L_dev,
                                          const float* p_dev, const float* b_dev, double* out_dev,
                                          void* stream, char* err, size_t err_cap) {
    if (err && err_cap) err[0] = '\0';
    if (!bc || !L_dev || !p_dev || !b_dev || !out_dev)
        return fail(err, err_cap, GMG_EINVAL, "gmg_residual_norm2_noalloc: null argument");
    if (nx < 1 || ny < 1 || nz < 1)
        return fail(err, err_cap, GMG_EINVAL, "gmg_residual_norm2_noalloc: extents must be >= 1");
    for (int d = 0; d < 3; ++d)
        if (bc[d] != GMG_BC_PERIODIC && bc[d] != GMG_BC_NEUMANN)
            return fail(err, err_cap, GMG_EINVAL, "gmg_residual_norm2_noalloc: bc[%d] is not 0 or 1", d);
    const long long N = (long long)nx * ny * nz;
    if (N > kMaxCells)
        return fail(err, err_cap, GMG_EINVAL,
                    "gmg_residual_norm2_noalloc: %lld cells exceed GMG_NOALLOC_MAX_CELLS = %lld "
                    "(the static scratch holds one partial per 2048 cells); use gmg_create + gmg_solve / "
                    "gmg_op_residual + gmg_op_norm2 for larger grids", N, kMaxCells);
    if ((((uintptr_t)L_dev | (uintptr_t)p_dev | (uintptr_t)b_dev) & 3) || ((uintptr_t)out_dev & 7))
        return fail(err, err_cap, GMG_EINVAL,
                    "gmg_residual_norm2_noalloc: L, p, b must be 4-byte and out_dev 8-byte aligned");

    double* scratch = nullptr;
    int dev = -1;
    cudaError_t e = scratch_of_current_device(&scratch, &dev);
    if (e != cudaSuccess)
        return fail(err, err_cap, GMG_ECUDA, "gmg_residual_norm2_noalloc: scratch look-up on device %d failed: %s",
                    dev, cudaGetErrorString(e));

    LevelGeom g;
    g.n[0] = nx; g.n[1] = ny; g.n[2] = nz;
    for (int d = 0; d < 3; ++d) { g.bc[d] = bc[d]; g.c[d] = 1; }
    g.N = N;
    cudaStream_t s = (cudaStream_t)stream;
    const unsigned int blocks = (unsigned int)((N + kRT * kCellsPerThread - 1) / (kRT * kCellsPerThread));
    // the ticket must start at zero whatever an earlier (possibly aborted) call left in the array
    e = cudaMemsetAsync(scratch + kTicketSlot, 0, 256, s);
    if (e == cudaSuccess) {
        k_residual_norm2_static<<<blocks, kRT, 0, s>>>(g, L_dev, p_dev, b_dev, scratch, out_dev);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess)
        return fail(err, err_cap, GMG_ECUDA, "gmg_residual_norm2_noalloc: enqueue on device %d failed: %s", dev,
                    cudaGetErrorString(e));
    return GMG_OK;
}

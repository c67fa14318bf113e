// gg_noalloc.cu -- gg_diagnostics_noalloc (include/gg.h): the field diagnostics for callers that
// have no device memory to give and no way of getting any.
//
// Who that is.  Every other call of this library works on a context whose workspace the caller
// allocated (gg_workspace_bytes / gg_bind).  A monitoring hook that another code's time loop calls
// with nothing but the device pointers of its U, V, W -- an in-situ probe, a plug-in of a host
// application whose memory pool took the whole GPU at start-up, a callback that runs while the
// host's step loop is pipelined several launches ahead -- cannot do that: it owns no allocator,
// cudaMalloc may simply fail when a pool already holds the device, and where it succeeds it
// synchronises the whole device and stalls exactly the loop the hook is meant to watch.  Such a
// caller still wants the masses, the gap count and the extrema of the current fields
// (PAPER.md:100-111 reads them off every experiment).
//
// What is different from gg_diagnostics.  The reduction needs somewhere to put one partial result
// per thread block.  gg_diagnostics keeps them in the context's workspace; this file keeps them
// in ONE array that is part of the library image itself (g_noalloc_scratch below, 1.3 MiB), which
// the CUDA runtime places on every GPU that loads libgg.so and keeps there until the process
// exits.  The entry point therefore calls no cudaMalloc, no cudaFree and no library routine that
// allocates: it validates, clears a few counters with cudaMemsetAsync, launches ONE kernel (the
// last block of a simulation to finish combines that simulation's partials; gg_diagnostics uses
// two launches) and returns.  Both the inputs and the output stay the caller's device memory.
//
// Consequences of the shared array, all stated again in gg.h:
//   * at most GG_NOALLOC_MAX_BATCH simulations per call (the array is sized for that; any grid
//     size is fine, the number of partials per simulation does not grow with it);
//   * all calls on one GPU use the same array, so two calls whose kernels may run at the same
//     time (different streams, or different host threads) overwrite each other's partials: the
//     caller has to order them.  Calls on one stream are ordered by the stream;
//   * the array keeps whatever the previous call left.  Partials are always written before they
//     are read within a call, the arrival counters are the only part that must start at zero, and
//     every call clears them on its stream before its kernel;
//   * the first call on each GPU looks the array's device address up (cudaGetSymbolAddress, which
//     also makes the runtime load this library's kernels onto that GPU).  Make that first call
//     with the GPU current and outside any stream capture.
//
// Product code; shares nothing with oracle/.
#include "../../include/gg.h"

#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <mutex>
#include <string>

namespace {

constexpr int kSlots = GG_DIAG_COUNT;       // slot order GG_DIAG_* of gg.h
constexpr int kThreads = 256;
constexpr int kMaxBlocks = 296;             // partial blocks per simulation (2 per SM on a B200)
constexpr int kMaxBatch = GG_NOALLOC_MAX_BATCH;
constexpr int kMaxDevices = 64;

// carving of the static array: [kMaxBatch][kMaxBlocks][kSlots] doubles, then [kMaxBatch] counters
constexpr size_t kPartialBytes = (size_t)kMaxBatch * kMaxBlocks * kSlots * sizeof(double);
constexpr size_t kCounterBytes = (size_t)kMaxBatch * sizeof(unsigned int);
constexpr size_t kScratchBytes = kPartialBytes + kCounterBytes;
static_assert(kPartialBytes % 256 == 0, "counters start 256-byte aligned");
static_assert(kScratchBytes <= (size_t)3 << 19, "the resident scratch is meant to stay modest (1.5 MiB)");

// The scratch itself.  In HOST code this name is only a handle for the runtime (its host address
// is not device memory): the device address comes from cudaGetSymbolAddress, once per GPU, in
// scratch_of() below, and that is what the kernel is given.
static __device__ __align__(256) unsigned char g_noalloc_scratch[kScratchBytes];

struct Acc {
    double v[kSlots];
    __device__ __forceinline__ void init() {
        v[GG_DIAG_SUM_U] = v[GG_DIAG_SUM_V] = v[GG_DIAG_SUM_W] = 0.0;
        v[GG_DIAG_GAP] = v[GG_DIAG_TUMOUR] = v[GG_DIAG_NONFINITE] = 0.0;
        v[GG_DIAG_MIN_W] = INFINITY;
        v[GG_DIAG_MAX_U] = v[GG_DIAG_MAX_W] = -INFINITY;
    }
    __device__ __forceinline__ void cell(double u, double vv, double w, double eps) {
        v[GG_DIAG_SUM_U] += u; v[GG_DIAG_SUM_V] += vv; v[GG_DIAG_SUM_W] += w;
        v[GG_DIAG_GAP] += (u < eps && vv < eps) ? 1.0 : 0.0;
        v[GG_DIAG_TUMOUR] += (vv >= 0.5) ? 1.0 : 0.0;
        v[GG_DIAG_MIN_W] = fmin(v[GG_DIAG_MIN_W], w);
        v[GG_DIAG_MAX_U] = fmax(v[GG_DIAG_MAX_U], u);
        v[GG_DIAG_MAX_W] = fmax(v[GG_DIAG_MAX_W], w);
        v[GG_DIAG_NONFINITE] += (isfinite(u) && isfinite(vv) && isfinite(w)) ? 0.0 : 1.0;
    }
    __device__ __forceinline__ void merge(const double* o) {
        v[GG_DIAG_SUM_U] += o[GG_DIAG_SUM_U]; v[GG_DIAG_SUM_V] += o[GG_DIAG_SUM_V]; v[GG_DIAG_SUM_W] += o[GG_DIAG_SUM_W];
        v[GG_DIAG_GAP] += o[GG_DIAG_GAP]; v[GG_DIAG_TUMOUR] += o[GG_DIAG_TUMOUR];
        v[GG_DIAG_NONFINITE] += o[GG_DIAG_NONFINITE];
        v[GG_DIAG_MIN_W] = fmin(v[GG_DIAG_MIN_W], o[GG_DIAG_MIN_W]);
        v[GG_DIAG_MAX_U] = fmax(v[GG_DIAG_MAX_U], o[GG_DIAG_MAX_U]);
        v[GG_DIAG_MAX_W] = fmax(v[GG_DIAG_MAX_W], o[GG_DIAG_MAX_W]);
    }
};

// fixed-order tree over shared memory; the block's result ends up in thread 0's acc
__device__ __forceinline__ void block_reduce(Acc& acc, double (*sh)[kSlots]) {
    const int t = threadIdx.x;
#pragma unroll
    for (int q = 0; q < kSlots; ++q) sh[t][q] = acc.v[q];
    __syncthreads();
    for (int s = kThreads / 2; s > 0; s >>= 1) {
        if (t < s) {
            acc.merge(sh[t + s]);
#pragma unroll
            for (int q = 0; q < kSlots; ++q) sh[t][q] = acc.v[q];
        }
        __syncthreads();
    }
}

// grid = (nblk, nbatch).  Block b of simulation s reduces cells [b*seg, min((b+1)*seg, plane)) of
// that simulation into partial[s][b][.]; the block that finds itself the nblk-th to arrive at
// arrived[s] combines the nblk partials in index order (so the sums do not depend on which block
// that was) and writes out[s][.].  `partial` and `arrived` point into g_noalloc_scratch.
template <typename T>
__global__ void __launch_bounds__(kThreads)
gg_diag_noalloc(const T* __restrict__ U, const T* __restrict__ V, const T* __restrict__ W, size_t plane,
                size_t seg, double eps, int vec_ok, double* partial, unsigned int* arrived,
                double* __restrict__ out) {
    __shared__ double sh[kThreads][kSlots];
    __shared__ unsigned int ticket;
    const int s = blockIdx.y, nblk = gridDim.x;
    const size_t base = (size_t)s * plane;
    const size_t lo = (size_t)blockIdx.x * seg;
    const size_t hi = lo + seg < plane ? lo + seg : plane;
    const T* pu = U + base; const T* pv = V + base; const T* pw = W + base;
    Acc acc;
    acc.init();
    constexpr int VC = 16 / (int)sizeof(T);   // cells per 16-byte load
    constexpr int UN = 4;                     // 16-byte loads in flight per thread and field
    size_t q = lo;
    if (vec_ok) {                             // every simulation's plane starts 16-byte aligned
        const size_t stride = (size_t)kThreads * VC * UN;
        for (; q + stride <= hi; q += stride) {
            T u[UN][VC], v[UN][VC], w[UN][VC];
#pragma unroll
            for (int n = 0; n < UN; ++n) {
                const size_t e = q + ((size_t)n * kThreads + threadIdx.x) * VC;
                *reinterpret_cast<uint4*>(u[n]) = *reinterpret_cast<const uint4*>(pu + e);
                *reinterpret_cast<uint4*>(v[n]) = *reinterpret_cast<const uint4*>(pv + e);
                *reinterpret_cast<uint4*>(w[n]) = *reinterpret_cast<const uint4*>(pw + e);
            }
#pragma unroll
            for (int n = 0; n < UN; ++n)
#pragma unroll
                for (int c = 0; c < VC; ++c) acc.cell((double)u[n][c], (double)v[n][c], (double)w[n][c], eps);
        }
    }
    for (q += threadIdx.x; q < hi; q += kThreads)
        acc.cell((double)pu[q], (double)pv[q], (double)pw[q], eps);
    block_reduce(acc, sh);

    double* mine = partial + ((size_t)s * nblk + blockIdx.x) * kSlots;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < kSlots; ++k) mine[k] = acc.v[k];
        __threadfence();                                  // partial visible before the ticket is
        ticket = atomicAdd(&arrived[s], 1u);
    }
    __syncthreads();
    if (ticket != (unsigned int)(nblk - 1)) return;       // not the last block of this simulation
    __threadfence();                                      // order the reads below after the ticket

    acc.init();
    const volatile double* all = partial + (size_t)s * nblk * kSlots;
    for (int b = threadIdx.x; b < nblk; b += kThreads) {
        double o[kSlots];
#pragma unroll
        for (int k = 0; k < kSlots; ++k) o[k] = all[(size_t)b * kSlots + k];
        acc.merge(o);
    }
    __syncthreads();                                      // sh is reused
    block_reduce(acc, sh);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < kSlots; ++k) out[(size_t)s * kSlots + k] = acc.v[k];
        arrived[s] = 0;                                   // leave the counter clean as well
    }
}

thread_local std::string g_error;

int fail(int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_error = buf;
    return code;
}

// Device address of g_noalloc_scratch on the CURRENT device, looked up on the first call per
// device and remembered.  (The symbol's host-side name must never be handed to a kernel.)
std::mutex g_setup_mutex;
unsigned char* g_scratch_dev[kMaxDevices] = {};

int scratch_of(unsigned char** ptr) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(GG_ERR_CUDA, "gg_diagnostics_noalloc: cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices)
        return fail(GG_ERR_UNSUPPORTED, "gg_diagnostics_noalloc: device ordinal %d outside [0, %d)", dev, kMaxDevices);
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_dev[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p)
            return fail(GG_ERR_CUDA, "gg_diagnostics_noalloc: cudaGetSymbolAddress on device %d: %s", dev, cudaGetErrorString(e));
        g_scratch_dev[dev] = static_cast<unsigned char*>(p);
    }
    *ptr = g_scratch_dev[dev];
    return GG_OK;
}

}  // namespace

extern "C" {

int gg_diagnostics_noalloc(const void* U, const void* V, const void* W, int nbatch, int nx, int ny,
                           int dtype, double eps, double* out, void* cuda_stream) {
    if (!U || !V || !W || !out) return fail(GG_ERR_ARG, "gg_diagnostics_noalloc: U, V, W and out must not be NULL");
    if (dtype != GG_F64 && dtype != GG_F32) return fail(GG_ERR_UNSUPPORTED, "gg_diagnostics_noalloc: dtype %d is neither GG_F64 nor GG_F32", dtype);
    if (nx < 1 || ny < 1) return fail(GG_ERR_ARG, "gg_diagnostics_noalloc: nx = %d, ny = %d must be >= 1", nx, ny);
    if (nbatch < 1) return fail(GG_ERR_ARG, "gg_diagnostics_noalloc: nbatch = %d must be >= 1", nbatch);
    if (nbatch > kMaxBatch)
        return fail(GG_ERR_ARG, "gg_diagnostics_noalloc: nbatch = %d exceeds GG_NOALLOC_MAX_BATCH = %d, the size the "
                    "library's built-in scratch was compiled for; split the batch or use gg_diagnostics", nbatch, kMaxBatch);
    if (!(eps >= 0.0) || !std::isfinite(eps)) return fail(GG_ERR_ARG, "gg_diagnostics_noalloc: eps must be finite and >= 0");
    const size_t esize = dtype == GG_F64 ? 8 : 4;
    if (((uintptr_t)U | (uintptr_t)V | (uintptr_t)W) % esize != 0 || (uintptr_t)out % sizeof(double) != 0)
        return fail(GG_ERR_ARG, "gg_diagnostics_noalloc: an array is not aligned to its element size");

    unsigned char* scratch = nullptr;
    if (int rc = scratch_of(&scratch)) return rc;
    double* partial = reinterpret_cast<double*>(scratch);
    unsigned int* arrived = reinterpret_cast<unsigned int*>(scratch + kPartialBytes);

    // same segmenting as gg_diagnostics: at most kMaxBlocks segments, each a multiple of the block
    const size_t plane = (size_t)nx * ny;
    size_t seg = (plane + kMaxBlocks - 1) / kMaxBlocks;
    seg = (seg + kThreads - 1) / kThreads * kThreads;
    const int nblk = (int)((plane + seg - 1) / seg);
    const int vec_ok = (((uintptr_t)U | (uintptr_t)V | (uintptr_t)W) % 16 == 0) && (plane * esize) % 16 == 0;

    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    cudaError_t e = cudaMemsetAsync(arrived, 0, (size_t)nbatch * sizeof(unsigned int), stream);
    if (e != cudaSuccess) return fail(GG_ERR_CUDA, "gg_diagnostics_noalloc: cudaMemsetAsync: %s", cudaGetErrorString(e));
    const dim3 grid(nblk, nbatch);
    if (dtype == GG_F64)
        gg_diag_noalloc<double><<<grid, kThreads, 0, stream>>>((const double*)U, (const double*)V, (const double*)W,
                                                              plane, seg, eps, vec_ok, partial, arrived, out);
    else
        gg_diag_noalloc<float><<<grid, kThreads, 0, stream>>>((const float*)U, (const float*)V, (const float*)W,
                                                             plane, seg, eps, vec_ok, partial, arrived, out);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(GG_ERR_CUDA, "gg_diagnostics_noalloc: launch: %s", cudaGetErrorString(e));
    return GG_OK;
}

const char* gg_noalloc_last_error(void) { return g_error.c_str(); }

}  // extern "C"

// gg_diag.cuh -- device-side reductions next to the step:
//
//  * gg_diag_partial / gg_diag_final: per-simulation diagnostics of the current state without a
//    full gg_get_state -- the quantities the paper's experiments read off the fields (tumour and
//    acid mass, the interstitial gap U ~ 0 and V ~ 0 between the fronts): sums of
//    U, V, W, the gap and tumour cell counts, the extrema that show the scheme's documented
//    over/undershoots (reading A7), and the number of cells holding a NaN or Inf (the
//    step itself never repairs or hides one: eq. (3) has no such rule).
//  * gg_lambda_max_partial: max over cells of the larger eigenvalue of [[a,b],[b,c]] (eq. (2),
//    PAPER.md:40), the quantity the explicit step bound needs (DESIGN.md
//    reading A6).
//
// Both are one pass over HBM (24 B per cell), two-stage and DETERMINISTIC: every block reduces a
// fixed contiguous segment in a fixed order (per-thread strided serial sum, then a shared-memory
// tree), the partials are combined by one block per simulation in a fixed order.  Accumulation is
// always in double, whatever the storage type.
#pragma once
#include "gg_common.cuh"

namespace gg {

constexpr int kDiagCount = 9;      // == GG_DIAG_COUNT in include/gg.h
constexpr int kDiagThreads = 256;
constexpr int kDiagMaxBlocks = 296;  // partial blocks per simulation (2 per SM on B200)

// slot order == GG_DIAG_* in include/gg.h
enum { kSumU = 0, kSumV, kSumW, kGap, kTumour, kMinW, kMaxU, kMaxW, kNonFinite };

struct DiagAcc {
    double v[kDiagCount];
    __device__ __forceinline__ void init() {
        v[kSumU] = v[kSumV] = v[kSumW] = v[kGap] = v[kTumour] = v[kNonFinite] = 0.0;
        v[kMinW] = INFINITY;
        v[kMaxU] = v[kMaxW] = -INFINITY;
    }
    __device__ __forceinline__ void cell(double u, double vv, double w, double eps) {
        v[kSumU] += u; v[kSumV] += vv; v[kSumW] += w;
        v[kGap] += (u < eps && vv < eps) ? 1.0 : 0.0;
        v[kTumour] += (vv >= 0.5) ? 1.0 : 0.0;
        v[kMinW] = fmin(v[kMinW], w);
        v[kMaxU] = fmax(v[kMaxU], u);
        v[kMaxW] = fmax(v[kMaxW], w);
        v[kNonFinite] += (isfinite(u) && isfinite(vv) && isfinite(w)) ? 0.0 : 1.0;
    }
    __device__ __forceinline__ void merge(const double* o) {
        v[kSumU] += o[kSumU]; v[kSumV] += o[kSumV]; v[kSumW] += o[kSumW];
        v[kGap] += o[kGap]; v[kTumour] += o[kTumour]; v[kNonFinite] += o[kNonFinite];
        v[kMinW] = fmin(v[kMinW], o[kMinW]);
        v[kMaxU] = fmax(v[kMaxU], o[kMaxU]);
        v[kMaxW] = fmax(v[kMaxW], o[kMaxW]);
    }
};

// fixed-order block reduction of `acc` (tree over shared memory); result valid in thread 0
__device__ __forceinline__ void diag_block_reduce(DiagAcc& acc, double (*sh)[kDiagCount]) {
    const int t = threadIdx.x;
#pragma unroll
    for (int q = 0; q < kDiagCount; ++q) sh[t][q] = acc.v[q];
    __syncthreads();
    for (int s = kDiagThreads / 2; s > 0; s >>= 1) {
        if (t < s) {
            acc.merge(sh[t + s]);
#pragma unroll
            for (int q = 0; q < kDiagCount; ++q) sh[t][q] = acc.v[q];
        }
        __syncthreads();
    }
}

// grid = (nblk, nbatch).  Block b of simulation s reduces cells [b*seg, min((b+1)*seg, plane)).
template <typename T>
__global__ void __launch_bounds__(kDiagThreads)
gg_diag_partial(const T* __restrict__ U, const T* __restrict__ V, const T* __restrict__ W,
                size_t plane, size_t seg, double eps, double* __restrict__ partial) {
    __shared__ double sh[kDiagThreads][kDiagCount];
    const size_t base = (size_t)blockIdx.y * plane;
    const size_t lo = (size_t)blockIdx.x * seg;
    const size_t hi = lo + seg < plane ? lo + seg : plane;
    DiagAcc acc;
    acc.init();
    constexpr int VC = 16 / (int)sizeof(T);           // cells per 16-byte vector
    constexpr int UN = 4;                             // vectors in flight per thread and array
    const T* pu = U + base; const T* pv = V + base; const T* pw = W + base;
    size_t q = lo;
    if ((plane * sizeof(T)) % 16 == 0 && lo % VC == 0) {
        // 16-byte loads, UN x 3 of them in flight per thread (the pass is HBM-bound)
        const size_t stride = (size_t)kDiagThreads * VC * UN;
        for (; q + stride <= hi; q += stride) {
            T u[UN][VC], v[UN][VC], w[UN][VC];
#pragma unroll
            for (int n = 0; n < UN; ++n) {
                const size_t e = q + ((size_t)n * kDiagThreads + threadIdx.x) * VC;
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
    for (q += threadIdx.x; q < hi; q += kDiagThreads)   // tail (or unaligned planes): scalar
        acc.cell((double)pu[q], (double)pv[q], (double)pw[q], eps);
    diag_block_reduce(acc, sh);
    if (threadIdx.x == 0) {
        double* o = partial + ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * kDiagCount;
#pragma unroll
        for (int q = 0; q < kDiagCount; ++q) o[q] = acc.v[q];
    }
}

// grid = nbatch.  Combines the nblk partials of one simulation in a fixed order.
__global__ void __launch_bounds__(kDiagThreads)
gg_diag_final(const double* __restrict__ partial, int nblk, double* __restrict__ out) {
    __shared__ double sh[kDiagThreads][kDiagCount];
    DiagAcc acc;
    acc.init();
    for (int b = threadIdx.x; b < nblk; b += kDiagThreads)
        acc.merge(partial + ((size_t)blockIdx.x * nblk + b) * kDiagCount);
    diag_block_reduce(acc, sh);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int q = 0; q < kDiagCount; ++q) out[(size_t)blockIdx.x * kDiagCount + q] = acc.v[q];
    }
}

// max over cells of lambda_+ = (a+c)/2 + sqrt(((a-c)/2)^2 + b^2).  grid = nblk; partial[nblk].
template <typename T>
__global__ void __launch_bounds__(kDiagThreads)
gg_lambda_max_partial(const T* __restrict__ a, const T* __restrict__ b, const T* __restrict__ c,
                      size_t plane, size_t seg, double* __restrict__ partial) {
    __shared__ double sh[kDiagThreads];
    const size_t lo = (size_t)blockIdx.x * seg;
    const size_t hi = lo + seg < plane ? lo + seg : plane;
    double m = -INFINITY;
    // rounding points written out (no FMA contraction): the value is a pure function of the
    // stored entries, bit-identical to the same formula evaluated in plain fp64 anywhere
    auto lam = [](double aa, double bb, double cc) {
        const double hd = __dmul_rn(0.5, __dsub_rn(aa, cc));
        return __dadd_rn(__dmul_rn(0.5, __dadd_rn(aa, cc)),
                         __dsqrt_rn(__dadd_rn(__dmul_rn(hd, hd), __dmul_rn(bb, bb))));
    };
    constexpr int VC = 16 / (int)sizeof(T);
    constexpr int UN = 4;
    size_t q = lo;
    if ((plane * sizeof(T)) % 16 == 0 && lo % VC == 0) {
        const size_t stride = (size_t)kDiagThreads * VC * UN;
        for (; q + stride <= hi; q += stride) {
            T va[UN][VC], vb[UN][VC], vc[UN][VC];
#pragma unroll
            for (int n = 0; n < UN; ++n) {
                const size_t e = q + ((size_t)n * kDiagThreads + threadIdx.x) * VC;
                *reinterpret_cast<uint4*>(va[n]) = *reinterpret_cast<const uint4*>(a + e);
                *reinterpret_cast<uint4*>(vb[n]) = *reinterpret_cast<const uint4*>(b + e);
                *reinterpret_cast<uint4*>(vc[n]) = *reinterpret_cast<const uint4*>(c + e);
            }
#pragma unroll
            for (int n = 0; n < UN; ++n)
#pragma unroll
                for (int k = 0; k < VC; ++k) m = fmax(m, lam((double)va[n][k], (double)vb[n][k], (double)vc[n][k]));
        }
    }
    for (q += threadIdx.x; q < hi; q += kDiagThreads) m = fmax(m, lam((double)a[q], (double)b[q], (double)c[q]));
    sh[threadIdx.x] = m;
    __syncthreads();
    for (int s = kDiagThreads / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] = fmax(sh[threadIdx.x], sh[threadIdx.x + s]);
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}

// Front position along a grid line ("front position along a ray"): the first
// and the last cell index q in [0, len) with F[q*stride] >= level along one row (stride 1) or one
// column (stride nx) of field F of every simulation; (-1, -1) if no cell qualifies.  One block
// per simulation; min / max over the qualifying indices, so the result is order-independent.
template <typename T>
__global__ void __launch_bounds__(kDiagThreads)
gg_front_line(const T* __restrict__ F, size_t plane, size_t offset, size_t stride, int len,
              double level, int* __restrict__ out) {
    __shared__ int lo[kDiagThreads], hi[kDiagThreads];
    const T* p = F + (size_t)blockIdx.x * plane + offset;
    int a = len, b = -1;
    for (int q = threadIdx.x; q < len; q += kDiagThreads)
        if ((double)p[(size_t)q * stride] >= level) { a = min(a, q); b = max(b, q); }
    lo[threadIdx.x] = a; hi[threadIdx.x] = b;
    __syncthreads();
    for (int s = kDiagThreads / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) {
            lo[threadIdx.x] = min(lo[threadIdx.x], lo[threadIdx.x + s]);
            hi[threadIdx.x] = max(hi[threadIdx.x], hi[threadIdx.x + s]);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        out[2 * blockIdx.x + 0] = hi[0] < 0 ? -1 : lo[0];
        out[2 * blockIdx.x + 1] = hi[0];
    }
}

}  // namespace gg

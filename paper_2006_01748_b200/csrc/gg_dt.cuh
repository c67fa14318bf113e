// gg_dt.cuh -- the step size lives ON THE DEVICE.
//
// The paper recomputes a non-uniform step dt_k on the host after every iteration, from results it
// downloads every iteration ("nonuniform step-size dt_k ... computed after each
// iteration", PAPER.md:127-128 steps 3-4).  Here neither the download nor the host exists inside
// the step loop:
//
//  * DevClock (one per context, in the workspace) holds the current dt, the simulated time, the
//    number of steps taken and lambda_max(A).  The step kernels never see dt: they read folded
//    per-simulation StepCoef<double> records (gg_common.cuh) that the kernels below write from
//    the dt that is current on the device.  A captured CUDA graph therefore survives any dt.
//  * gg_fold_fixed: gg_step(n, dt) -- dt arrives by value in a plain launch in front of the graph
//    replay (launched only when dt differs from what the device already holds).
//  * gg_min_u_partial + gg_fold_adaptive: gg_step_adaptive -- every `every_k` steps the device
//    reduces min U per simulation (one pass over U: 1/9 of a step's traffic), forms
//        dt_k = safety * min(dx,dy)^2 / max(lambda_max(A), max_s alpha_s * max_ij (1 - U^k_s,ij))
//    (reading A6; the paper prints no formula: the RULE is "parity unpinned"), folds the
//    coefficients and advances the clock -- all inside the captured graph, no host round trip.
//  * gg_lambda_final: lambda_max(A) reduced once per gg_set_tensor and cached in the DevClock.
//  * gg_face_tensor: a, c are stored pre-scaled and summed over the faces (StepCoef comment in
//    gg_common.cuh).
//
// All reductions are max/min (order-independent, exact), so dt_k is a deterministic function of
// the stored state: the oracle's dt_k is bit-identical for fp64 storage.
#pragma once
#include "gg_diag.cuh"

namespace gg {

struct DevClock {
    double dt;            // step size of the launches that follow
    double time;          // sum of the step sizes of all steps taken since gg_set_state
    double lambda_max;    // max over cells of the larger eigenvalue of [[a,b],[b,c]]
    double rate;          // adaptive: the max(...) of the last dt_k rule evaluation
    double safety;        // adaptive: the safety factor of the rule (set in front of the replay)
    long long steps;      // steps taken since gg_set_state
    long long bad_rule;   // adaptive: evaluations of the dt_k rule that gave no usable step size since
                          // gg_set_state (sticky; the steps of such a group run with dt = 0, i.e. leave
                          // the state as it is, and gg_get_clock reports the failure)
    long long pad_[1];
};

// dt by value (gg_step): fold every simulation's coefficients, advance the clock by n steps.
// fold == 0: dt is what the device already holds (only the clock moves).
__global__ void __launch_bounds__(128)
gg_fold_fixed(DevClock* __restrict__ clk, const SimScalars* __restrict__ sims,
              StepCoef<double>* __restrict__ coefs, int nbatch, double dt, double dx, double dy,
              long long n, int fold) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (fold && s < nbatch) coefs[s] = fold_coef(sims[s], dt, dx, dy);
    if (s == 0) {
        clk->dt = dt;
        clk->time += dt * (double)n;
        clk->steps += n;
    }
}

__global__ void gg_clock_reset(DevClock* __restrict__ clk) {
    clk->time = 0.0;
    clk->steps = 0;
    clk->rate = 0.0;
    clk->bad_rule = 0;
}
__global__ void gg_clock_safety(DevClock* __restrict__ clk, double safety) { clk->safety = safety; }

// min over the cells of U per simulation.  grid = (nblk, nbatch); partial[nbatch][nblk].
// fmin skips NaNs; a state without a finite U gives +inf and the rule falls back to lambda_max.
template <typename T>
__global__ void __launch_bounds__(kDiagThreads)
gg_min_u_partial(const T* __restrict__ U, size_t plane, size_t seg, double* __restrict__ partial) {
    __shared__ double sh[kDiagThreads];
    const T* pu = U + (size_t)blockIdx.y * plane;
    const size_t lo = (size_t)blockIdx.x * seg;
    const size_t hi = lo + seg < plane ? lo + seg : plane;
    double m = INFINITY;
    constexpr int VC = 16 / (int)sizeof(T);
    constexpr int UN = 8;
    size_t q = lo;
    if ((plane * sizeof(T)) % 16 == 0 && lo % VC == 0) {
        const size_t stride = (size_t)kDiagThreads * VC * UN;
        for (; q + stride <= hi; q += stride) {
            T u[UN][VC];
#pragma unroll
            for (int n = 0; n < UN; ++n)
                *reinterpret_cast<uint4*>(u[n]) = *reinterpret_cast<const uint4*>(
                    pu + q + ((size_t)n * kDiagThreads + threadIdx.x) * VC);
#pragma unroll
            for (int n = 0; n < UN; ++n)
#pragma unroll
                for (int c = 0; c < VC; ++c) m = fmin(m, (double)u[n][c]);
        }
    }
    for (q += threadIdx.x; q < hi; q += kDiagThreads) m = fmin(m, (double)pu[q]);
    sh[threadIdx.x] = m;
    __syncthreads();
    for (int s = kDiagThreads / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] = fmin(sh[threadIdx.x], sh[threadIdx.x + s]);
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = sh[0];
}

// One block.  The dt_k rule (header comment) from the per-simulation partial minima of U, then
// the fold and the clock, for the `k` steps that follow.  max_ij fl(1 - U_ij) = fl(1 - min_ij U_ij)
// because rounding is monotone, so reducing min U is exact.
__global__ void __launch_bounds__(kDiagThreads)
gg_fold_adaptive(DevClock* __restrict__ clk, const SimScalars* __restrict__ sims,
                 StepCoef<double>* __restrict__ coefs, const double* __restrict__ partial, int nblk,
                 int nbatch, double dx, double dy, long long k) {
    __shared__ double sh[kDiagThreads];
    __shared__ double s_dt;
    double p = -INFINITY;                      // max_s alpha_s * (1 - min U_s)
    for (int s = threadIdx.x; s < nbatch; s += kDiagThreads) {
        double m = INFINITY;
        for (int b = 0; b < nblk; ++b) m = fmin(m, partial[(size_t)s * nblk + b]);
        p = fmax(p, __dmul_rn(sims[s].alpha, __dsub_rn(1.0, m)));
    }
    sh[threadIdx.x] = p;
    __syncthreads();
    for (int s = kDiagThreads / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] = fmax(sh[threadIdx.x], sh[threadIdx.x + s]);
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const double rate = fmax(clk->lambda_max, sh[0]);
        const double hmin = dx < dy ? dx : dy;
        double dt = __ddiv_rn(__dmul_rn(__dmul_rn(clk->safety, hmin), hmin), rate);
        // No usable bound (A == 0 with U >= 1 everywhere, alpha == 0 with a zero tensor, a non-finite
        // tensor entry, a state without one finite U): do not fold inf / NaN / a negative dt into
        // the coefficients.  The group's steps run with dt = 0 (the state stays what it is, the
        // clock's time does not move) and the failure is counted for gg_get_clock to report.
        if (!(rate > 0.0) || !isfinite(rate) || !(dt > 0.0) || !isfinite(dt)) {
            dt = 0.0;
            clk->bad_rule += 1;
        }
        clk->rate = rate;
        clk->dt = dt;
        clk->time += dt * (double)k;
        clk->steps += k;
        s_dt = dt;
    }
    __syncthreads();
    const double dt = s_dt;
    for (int s = threadIdx.x; s < nbatch; s += kDiagThreads) coefs[s] = fold_coef(sims[s], dt, dx, dy);
}

// One block: max of the nblk partials of gg_lambda_max_partial into the clock.
__global__ void __launch_bounds__(kDiagThreads)
gg_lambda_final(const double* __restrict__ partial, int nblk, DevClock* __restrict__ clk) {
    __shared__ double sh[kDiagThreads];
    double m = -INFINITY;
    for (int b = threadIdx.x; b < nblk; b += kDiagThreads) m = fmax(m, partial[b]);
    sh[threadIdx.x] = m;
    __syncthreads();
    for (int s = kDiagThreads / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] = fmax(sh[threadIdx.x], sh[threadIdx.x + s]);
        __syncthreads();
    }
    if (threadIdx.x == 0) clk->lambda_max = sh[0];
}

// The stored tensor (StepCoef comment in gg_common.cuh): a' = a * scale rounded once to T, then the
// face sums  aw_ij = a'_i-1,j + a'_ij  (shift = 1: west faces)  or  cs_ij = c'_i,j-1 + c'_ij
// (shift = nx: south faces), added in T -- exactly the sum the step kernels used to form per face
// and step.  Cells without a neighbour on that side (i = 0 / j = 0) get 2 a'_ij: the flux through
// a boundary face is zero whatever its coefficient.  src and dst must not overlap.
template <typename T>
__global__ void __launch_bounds__(256) gg_face_tensor(const T* __restrict__ src, T* __restrict__ dst, int nx, size_t n,
                                                      int shift, double scale) {
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (size_t)gridDim.x * blockDim.x) {
        const bool has = shift == 1 ? (q % (size_t)nx) != 0 : q >= (size_t)nx;
        const T k1 = (T)((double)src[q] * scale);
        const T k0 = has ? (T)((double)src[q - (size_t)shift] * scale) : k1;
        dst[q] = add(k0, k1);
    }
}

}  // namespace gg

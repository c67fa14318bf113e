// gg_common.cuh -- types shared by the step kernels of libgg.so (product code; nothing here is
// shared with oracle/).
//
// Scheme: eq. (3) of arXiv 2006.01748 with the stencils of Table 1
// and Table 2, evaluated in FLUX FORM:
//
//   V face flux   phiE_ij = (1 - (U_ij + U_i+1,j)/2) (V_i+1,j - V_ij)          [Table 1, E entry x h^2]
//                 phiN_ij = (1 - (U_ij + U_i,j+1)/2) (V_i,j+1 - V_ij)
//   W cross terms G_ij = b_ij (W_i,j+1 - W_i,j-1),  H_ij = b_ij (W_i+1,j - W_i-1,j)
//   W face flux   FE_ij = (a_ij + a_i+1,j)/2 (W_i+1,j - W_ij) + (G_ij + G_i+1,j)/4   [Table 2: E entry
//                 FN_ij = (c_ij + c_i,j+1)/2 (W_i,j+1 - W_ij) + (H_ij + H_i,j+1)/4    and the 4 corners]
//   update        U' = U + dt U (1-U) - d dt U W
//                 V' = V + r dt V (1-V) + (alpha dt/h^2) [phiE_ij - phiE_i-1,j + phiN_ij - phiN_i,j-1]
//                 W' = W + c_r dt (V - W) + (dt/h^2)     [FE_ij   - FE_i-1,j   + FN_ij   - FN_i,j-1]
//
// Neumann (reading A2): every face on the domain boundary carries zero flux, and the tangential
// differences in G, H at boundary cells use the mirrored (= clamped) neighbour.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gg {

// Scalars of eq. (1) for one simulation, as stored in the workspace (always double; the kernels
// fold them with dt and 1/h^2 in double and round once to the arithmetic type).
struct SimScalars {
    double r, d, alpha, c_r;
};

// Step coefficients in the arithmetic type T.
template <typename T>
struct StepCoef {
    T dt;     // dt
    T ddt;    // d * dt
    T rdt;    // r * dt
    T adt;    // alpha * dt / h^2
    T crdt;   // c_r * dt
    T s;      // dt / h^2
};

template <typename T>
__device__ __forceinline__ StepCoef<T> fold_coef(const SimScalars& p, double dt, double inv_h2) {
    StepCoef<T> k;
    k.dt = (T)dt;
    k.ddt = (T)(p.d * dt);
    k.rdt = (T)(p.r * dt);
    k.adt = (T)(p.alpha * dt * inv_h2);
    k.crdt = (T)(p.c_r * dt);
    k.s = (T)(dt * inv_h2);
    return k;
}

// Pointwise pieces used by every kernel.  fma contraction is left to the compiler (tolerances
// in DESIGN.md section 6 absorb the evaluation order).
template <typename T>
__device__ __forceinline__ T upd_U(const StepCoef<T>& k, T u, T w) {
    // eq. (3) line 1: U + dt U (1-U) - d dt U W
    return u + u * (k.dt * ((T)1 - u) - k.ddt * w);
}
template <typename T>
__device__ __forceinline__ T upd_V(const StepCoef<T>& k, T v, T div) {
    // eq. (3) line 2, div = sum of the four face-flux differences (x h^2)
    return v + k.rdt * v * ((T)1 - v) + k.adt * div;
}
template <typename T>
__device__ __forceinline__ T upd_W(const StepCoef<T>& k, T v, T w, T div) {
    // eq. (3) line 3
    return w + k.crdt * (v - w) + k.s * div;
}
template <typename T>
__device__ __forceinline__ T flux_V(T u0, T u1, T v0, T v1) {
    // Table 1 face weight x h^2 times the V difference across the face (from cell 0 to cell 1)
    return ((T)1 - (T)0.5 * (u0 + u1)) * (v1 - v0);
}
template <typename T>
__device__ __forceinline__ T flux_W(T k0, T k1, T w0, T w1, T x0, T x1) {
    // Table 2: face-mean diffusivity times normal difference + mean of the two cross terms / 2
    return (T)0.5 * (k0 + k1) * (w1 - w0) + (T)0.25 * (x0 + x1);
}

}  // namespace gg

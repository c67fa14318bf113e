// gg_common.cuh -- types shared by the step kernels of libgg.so (product code; nothing here is
// shared with oracle/).
//
// Scheme: eq. (3) of arXiv 2006.01748 with the stencils of Table 1
// and Table 2, evaluated in FLUX FORM:
//
//   (the code carries 2 phi and pre-scaled 2 F and folds the factors into the step coefficients and
//    the stored tensor entries instead, see StepCoef and flux_V; the tensor is stored as the FACE
//    sums a_i-1,j + a_ij and c_i,j-1 + c_ij, which do not change in time, and U enters the V fluxes
//    through M = 1 - U, formed once per cell)
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

// Step coefficients of one simulation.  They live in the workspace as StepCoef<double>, written
// by the device-side fold kernel (gg_dt.cuh) from the step size that is current ON THE DEVICE, so
// that neither a new dt nor an adaptive dt_k changes a kernel argument (a captured graph survives
// any dt).  The step kernels load them and round once to the arithmetic type T.
//
// The tensor fields are stored PRE-SCALED and PRE-SUMMED over the faces (gg_set_tensor,
// gg_face_tensor in gg_dt.cuh): with a' = a * 2dy/dx, c' = c * 2dx/dy the workspace holds
//     aw_ij = a'_i-1,j + a'_ij   (west face of cell ij;  aw_0j = 2 a'_0j, never used: zero flux)
//     cs_ij = c'_i,j-1 + c'_ij   (south face of cell ij; cs_i0 = 2 c'_i0, never used)
// and b as given.  With G = b (W_i,j+1 - W_i,j-1), H = b (W_i+1,j - W_i-1,j) the doubled W face
// fluxes of the header comment, divided by the cross-term weights dx/(2dy) resp. dy/(2dx), become
//     FE' = aw_i+1,j (W_i+1,j - W_ij) + (G_ij + G_i+1,j)
//     FN' = cs_i,j+1 (W_i,j+1 - W_ij) + (H_ij + H_i,j+1)
// and both carry the same step weight dt/(4 dx dy): two operations less per face than Table 2's
// literal form (the face sums are time-independent), one array element per face and cell as
// before, and bit for bit the values of summing a', c' in the kernel.
template <typename T>
struct StepCoef {
    T dt;     // dt
    T ddt;    // d * dt
    T rdt;    // r * dt
    T adx;    // alpha * dt / (2 dx^2)   (the V face fluxes carry a factor 2, see flux_V)
    T ady;    // alpha * dt / (2 dy^2)
    T crdt;   // c_r * dt
    T sw;     // dt / (4 dx dy): weight of the pre-scaled W face fluxes FE', FN'
    T pad_;
};

__host__ __device__ __forceinline__ StepCoef<double> fold_coef(const SimScalars& p, double dt, double dx, double dy) {
    StepCoef<double> k;
    k.dt = dt;
    k.ddt = p.d * dt;
    k.rdt = p.r * dt;
    k.adx = 0.5 * p.alpha * dt / (dx * dx);
    k.ady = 0.5 * p.alpha * dt / (dy * dy);
    k.crdt = p.c_r * dt;
    k.sw = 0.25 * dt / (dx * dy);
    k.pad_ = 0.0;
    return k;
}
// factors the tensor entries a and c are stored with (see above)
__host__ __device__ __forceinline__ double tensor_scale_a(double dx, double dy) { return 2.0 * dy / dx; }
__host__ __device__ __forceinline__ double tensor_scale_c(double dx, double dy) { return 2.0 * dx / dy; }

template <typename T>
__device__ __forceinline__ StepCoef<T> load_coef(const StepCoef<double>* __restrict__ p) {
    const StepCoef<double> c = *p;
    StepCoef<T> k;
    k.dt = (T)c.dt; k.ddt = (T)c.ddt; k.rdt = (T)c.rdt; k.adx = (T)c.adx; k.ady = (T)c.ady;
    k.crdt = (T)c.crdt; k.sw = (T)c.sw; k.pad_ = (T)0;
    return k;
}

// Arithmetic with the rounding points written out: _rn intrinsics are never contracted or
// re-associated by the compiler, so every kernel (generic, single-step, two-step, resident;
// whatever its instantiation) performs the SAME sequence of roundings per cell.  All kernels of
// the library are therefore bit-identical to one another, and gg_step(n) does not depend on how
// the n steps are split into launches or calls (tests/test_gpu_parity.py).
__device__ __forceinline__ double add(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double sub(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ double mul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double fma_(double a, double b, double c) { return __fma_rn(a, b, c); }
__device__ __forceinline__ float add(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float sub(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ float mul(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float fma_(float a, float b, float c) { return __fmaf_rn(a, b, c); }

// Face fluxes carry a common factor (flux_V = 2 phi, flux_W = 2 F / cross-term weight) that
// fold_coef puts into adx, ady and sw: fewer multiplications per face.
// M = 1 - U: formed once per cell and time level, used by the U reaction and by the V face weights
template <typename T>
__device__ __forceinline__ T one_minus(T u) { return sub((T)1, u); }
template <typename T>
__device__ __forceinline__ T upd_U(const StepCoef<T>& k, T u, T m, T w) {
    // eq. (3) line 1: U + dt U (1-U) - d dt U W  =  U + U (dt M - d dt W),  M = 1 - U
    return fma_(u, fma_(k.dt, m, -mul(k.ddt, w)), u);
}
template <typename T>
__device__ __forceinline__ T upd_V(const StepCoef<T>& k, T v, T fe, T fw, T fn, T fs) {
    // eq. (3) line 2; fe, fw, fn, fs: doubled fluxes through the east, west, north, south faces
    return fma_(k.adx, sub(fe, fw), fma_(k.ady, sub(fn, fs), fma_(mul(k.rdt, v), sub((T)1, v), v)));
}
template <typename T>
__device__ __forceinline__ T upd_W(const StepCoef<T>& k, T v, T w, T fe, T fw, T fn, T fs) {
    // eq. (3) line 3
    return fma_(k.sw, sub(fe, fw), fma_(k.sw, sub(fn, fs), fma_(k.crdt, sub(v, w), w)));
}
template <typename T>
__device__ __forceinline__ T flux_V(T m0, T m1, T v0, T v1) {
    // 2 x [Table 1 face weight x h^2] x (V difference across the face, from cell 0 to cell 1):
    // 2 (1 - (U0 + U1)/2) = M0 + M1 with M = 1 - U
    return mul(add(m0, m1), sub(v1, v0));
}
template <typename T>
__device__ __forceinline__ T flux_W(T kf, T w0, T w1, T x0, T x1) {
    // pre-scaled doubled face flux (Table 2): kf (w1-w0) + (x0+x1), kf = the stored face sum aw or
    // cs of the face, x = b x (tangential difference of W) of the two cells the face separates
    return fma_(kf, sub(w1, w0), add(x0, x1));
}
// cross term b (W_+ - W_-) of one cell (G: y difference, H: x difference)
template <typename T>
__device__ __forceinline__ T cross(T b, T wp, T wm) { return mul(b, sub(wp, wm)); }

}  // namespace gg

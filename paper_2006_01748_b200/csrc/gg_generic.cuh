// gg_generic.cuh -- GG_KERNEL_GENERIC: one thread per cell, global memory, clamp-indexed.
//
// The shape-agnostic path (any nx, ny >= 2, any alignment).  It is roughly the design the paper
// describes for its own port (one data-parallel evaluation of eq. (3) over global memory,
// PAPER.md:125-126) and serves (i) shapes the TMA path cannot take (row pitch not a multiple of
// 16 bytes) and (ii) as an independent in-library cross-check of the tiled kernels in the GPU
// tests.  Every thread evaluates its four faces itself (no sharing), boundary faces carry zero
// flux, tangential differences use clamped neighbours (gg_common.cuh, reading A2).
#pragma once
#include "gg_common.cuh"

namespace gg {

template <typename T>
struct GenericArgs {
    const T* __restrict__ U;   // [B][ny][nx] time k
    const T* __restrict__ V;
    const T* __restrict__ W;
    T* __restrict__ U1;        // [B][ny][nx] time k+1
    T* __restrict__ V1;
    T* __restrict__ W1;
    const T* __restrict__ a;   // [ny][nx]: aw, the west-face sums of the stored tensor (gg_common.cuh)
    const T* __restrict__ b;
    const T* __restrict__ c;   // cs, the south-face sums
    const StepCoef<double>* __restrict__ coefs;  // [B], folded on the device (gg_dt.cuh)
    int nx, ny, nbatch;
};

template <typename T>
__global__ void __launch_bounds__(256) gg_step_generic(GenericArgs<T> A) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int sim = blockIdx.z;
    if (i >= A.nx || j >= A.ny) return;
    const int nx = A.nx, ny = A.ny;
    const size_t plane = (size_t)nx * ny;
    const T* U = A.U + sim * plane;
    const T* V = A.V + sim * plane;
    const T* W = A.W + sim * plane;
    const StepCoef<T> k = load_coef<T>(A.coefs + sim);

    const bool hasW = i > 0, hasE = i < nx - 1, hasS = j > 0, hasN = j < ny - 1;
    const int iw = hasW ? i - 1 : i, ie = hasE ? i + 1 : i;
    const int js = hasS ? j - 1 : j, jn = hasN ? j + 1 : j;
    auto at = [nx](const T* P, int ii, int jj) { return P[(size_t)jj * nx + ii]; };

    const T u = at(U, i, j), v = at(V, i, j), w = at(W, i, j);
    // 3x3 neighbourhood of W with clamped (mirrored) indices
    const T wW = at(W, iw, j), wE = at(W, ie, j), wS = at(W, i, js), wN = at(W, i, jn);
    const T wSW = at(W, iw, js), wSE = at(W, ie, js), wNW = at(W, iw, jn), wNE = at(W, ie, jn);

    // ---- V: four face fluxes (zero on boundary faces because the clamped neighbour equals the cell)
    const T m = one_minus(u);
    const T pE = flux_V(m, one_minus(at(U, ie, j)), v, at(V, ie, j));
    const T pW = flux_V(one_minus(at(U, iw, j)), m, at(V, iw, j), v);
    const T pN = flux_V(m, one_minus(at(U, i, jn)), v, at(V, i, jn));
    const T pS = flux_V(one_minus(at(U, i, js)), m, at(V, i, js), v);

    // ---- W: cross terms at the cell and its four edge neighbours (clamped tangential differences)
    const T b0 = at(A.b, i, j);
    const T G0 = cross(b0, wN, wS), H0 = cross(b0, wE, wW);
    const T GE = cross(at(A.b, ie, j), wNE, wSE);
    const T GW = cross(at(A.b, iw, j), wNW, wSW);
    const T HN = cross(at(A.b, i, jn), wNE, wNW);
    const T HS = cross(at(A.b, i, js), wSE, wSW);
    // face sums: the east face of cell i is the west face of cell i+1, the north face of row j the
    // south face of row j+1 (boundary faces: any finite value, the flux is zeroed below)
    T fE = flux_W(at(A.a, ie, j), w, wE, G0, GE);
    T fW = flux_W(at(A.a, i, j), wW, w, GW, G0);
    T fN = flux_W(at(A.c, i, jn), w, wN, H0, HN);
    T fS = flux_W(at(A.c, i, j), wS, w, HS, H0);
    // zero total normal flux through boundary faces (the cross part does not vanish by clamping)
    if (!hasE) fE = (T)0;
    if (!hasW) fW = (T)0;
    if (!hasN) fN = (T)0;
    if (!hasS) fS = (T)0;

    const size_t q = sim * plane + (size_t)j * nx + i;
    A.U1[q] = upd_U(k, u, m, w);
    A.V1[q] = upd_V(k, v, pE, pW, pN, pS);
    A.W1[q] = upd_W(k, v, w, fE, fW, fN, fS);
}

}  // namespace gg

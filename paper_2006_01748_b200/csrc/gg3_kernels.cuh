// gg3_kernels.cuh -- step kernels of the three-dimensional extension (include/gg3.h; product code,
// nothing shared with oracle/).
//
// Scheme (reading A13; PAPER.md:74, :81-92 one dimension up), evaluated per cell in
// DIVERGENCE form.  Stored tensor (gg3_store_tensor): the face coefficients
//     fx_ijk = (axx_i-1 + axx_i)/(2 dx^2)   (west face),   fy: south face with ayy,   fz: bottom face with azz
// and the pre-scaled off-diagonals gxy = axy/(4 dx dy), gxz = axz/(4 dx dz), gyz = ayz/(4 dy dz).
//     D2 W = fx_E (W_E - W) - fx (W - W_W) + [same in y, z]
//          + [Pxy(E) - Pxy(W)] + [Pyx(N) - Pyx(S)] + [Pxz(E) - Pxz(W)] + [Pzx(T) - Pzx(B)]
//          + [Pyz(N) - Pyz(S)] + [Pzy(T) - Pzy(B)],
//     Ppq(cell) = g_pq(cell) (W(cell + e_q) - W(cell - e_q)),
// which is Table 2's corner entries written as nested central differences.  Neumann faces:
// neighbour indices are clamped (even mirror of U, V, W: every diagonal and V flux through a
// boundary face is exactly 0) and a cross term taken at a clamped neighbour changes sign (the
// off-diagonal entry is odd across that face), which makes the total normal flux zero.
// V: doubled face fluxes (M_c + M_nb)(V_nb - V_c), M = 1 - U, weights alpha dt/(2 d^2) (flux_V of
// gg_common.cuh).  Both kernels gather their operands and call the SAME cell function =>
// bit-identical to each other.
#pragma once
#include "gg_common.cuh"

namespace gg3 {

using gg::add; using gg::sub; using gg::mul; using gg::fma_; using gg::cross; using gg::flux_V; using gg::one_minus;

template <typename T>
struct Coef3 {
    T dt, ddt, rdt, crdt, adx, ady, adz;   // dt, d dt, r dt, c_r dt, alpha dt/(2 dx^2), /(2 dy^2), /(2 dz^2)
};

// operands of one cell: centre values, the six face neighbours (clamped) of U, V, W, the twelve
// edge neighbours of W, the face coefficients of the cell and of its E / N / T neighbour, the
// off-diagonals at the face neighbours that use them
template <typename T>
struct Cell3 {
    T u, v, w;
    T uE, uW, uN, uS, uT, uB;
    T vE, vW, vN, vS, vT, vB;
    T wE, wW, wN, wS, wT, wB;
    T wNE, wNW, wSE, wSW;      // (i+-1, j+-1, k)
    T wTE, wTW, wBE, wBW;      // (i+-1, j, k+-1)
    T wTN, wTS, wBN, wBS;      // (i, j+-1, k+-1)
    T fxC, fxE, fyC, fyN, fzC, fzT;
    T gxyE, gxyW, gxyN, gxyS;
    T gxzE, gxzW, gxzT, gxzB;
    T gyzN, gyzS, gyzT, gyzB;
};

// hasX: the cell has a neighbour on that side (else the operand is the clamped value)
template <typename T>
__device__ __forceinline__ void cell3(const Coef3<T>& k, const Cell3<T>& c, bool hasE, bool hasW, bool hasN, bool hasS,
                                      bool hasT, bool hasB, T& oU, T& oV, T& oW) {
    // ---- U, V
    const T m = one_minus(c.u);
    const T pE = flux_V(m, one_minus(c.uE), c.v, c.vE), pW = flux_V(one_minus(c.uW), m, c.vW, c.v);
    const T pN = flux_V(m, one_minus(c.uN), c.v, c.vN), pS = flux_V(one_minus(c.uS), m, c.vS, c.v);
    const T pT = flux_V(m, one_minus(c.uT), c.v, c.vT), pB = flux_V(one_minus(c.uB), m, c.vB, c.v);
    oU = fma_(c.u, fma_(k.dt, m, -mul(k.ddt, c.w)), c.u);
    oV = fma_(k.adx, sub(pE, pW), fma_(k.ady, sub(pN, pS), fma_(k.adz, sub(pT, pB), fma_(mul(k.rdt, c.v), sub((T)1, c.v), c.v))));
    // ---- W: diagonal part
    const T tX = fma_(c.fxE, sub(c.wE, c.w), -mul(c.fxC, sub(c.w, c.wW)));
    const T tY = fma_(c.fyN, sub(c.wN, c.w), -mul(c.fyC, sub(c.w, c.wS)));
    const T tZ = fma_(c.fzT, sub(c.wT, c.w), -mul(c.fzC, sub(c.w, c.wB)));
    // cross terms at the six face neighbours; at a clamped neighbour the term changes sign
    T pxyE = cross(c.gxyE, c.wNE, c.wSE), pxyW = cross(c.gxyW, c.wNW, c.wSW);
    T pyxN = cross(c.gxyN, c.wNE, c.wNW), pyxS = cross(c.gxyS, c.wSE, c.wSW);
    T pxzE = cross(c.gxzE, c.wTE, c.wBE), pxzW = cross(c.gxzW, c.wTW, c.wBW);
    T pzxT = cross(c.gxzT, c.wTE, c.wTW), pzxB = cross(c.gxzB, c.wBE, c.wBW);
    T pyzN = cross(c.gyzN, c.wTN, c.wBN), pyzS = cross(c.gyzS, c.wTS, c.wBS);
    T pzyT = cross(c.gyzT, c.wTN, c.wTS), pzyB = cross(c.gyzB, c.wBN, c.wBS);
    if (!hasE) { pxyE = -pxyE; pxzE = -pxzE; }
    if (!hasW) { pxyW = -pxyW; pxzW = -pxzW; }
    if (!hasN) { pyxN = -pyxN; pyzN = -pyzN; }
    if (!hasS) { pyxS = -pyxS; pyzS = -pyzS; }
    if (!hasT) { pzxT = -pzxT; pzyT = -pzyT; }
    if (!hasB) { pzxB = -pzxB; pzyB = -pzyB; }
    const T cXY = add(sub(pxyE, pxyW), sub(pyxN, pyxS));
    const T cXZ = add(sub(pxzE, pxzW), sub(pzxT, pzxB));
    const T cYZ = add(sub(pyzN, pyzS), sub(pzyT, pzyB));
    const T D2 = add(add(add(tX, tY), tZ), add(add(cXY, cXZ), cYZ));
    oW = fma_(k.dt, D2, fma_(k.crdt, sub(c.v, c.w), c.w));
}

template <typename T>
struct Args3 {
    const T* __restrict__ U; const T* __restrict__ V; const T* __restrict__ W;     // time k   [nz][ny][nx]
    T* __restrict__ U1; T* __restrict__ V1; T* __restrict__ W1;                    // time k+1
    const T* __restrict__ fx; const T* __restrict__ fy; const T* __restrict__ fz;  // stored tensor
    const T* __restrict__ gxy; const T* __restrict__ gxz; const T* __restrict__ gyz;
    Coef3<T> k;
    int nx, ny, nz;
};

// Stored tensor from the entries as given (src and dst must not overlap).
//   mode 0: face coefficient: dst_q = (src_{q - shift} + src_q) * scale  (2 src_q * scale on the low boundary)
//   mode 1: dst_q = src_q * scale
template <typename T>
__global__ void __launch_bounds__(256) gg3_store_tensor(const T* __restrict__ src, T* __restrict__ dst, int nx, int ny, int nz,
                                                        int axis, int mode, double scale) {
    const size_t n = (size_t)nx * ny * nz;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (size_t)gridDim.x * blockDim.x) {
        double x = (double)src[q];
        if (mode == 0) {
            const size_t i = q % (size_t)nx, j = (q / (size_t)nx) % (size_t)ny, kz = q / ((size_t)nx * ny);
            const size_t shift = axis == 0 ? 1 : axis == 1 ? (size_t)nx : (size_t)nx * ny;
            const bool has = axis == 0 ? i > 0 : axis == 1 ? j > 0 : kz > 0;
            x += has ? (double)src[q - shift] : x;
        }
        dst[q] = (T)(x * scale);
    }
}

// GG3_KERNEL_GENERIC: one thread per cell, clamp-indexed global loads (L1/L2 provide the reuse).
template <typename T>
__global__ void __launch_bounds__(256) gg3_step_generic(const Args3<T> A) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int kz = blockIdx.z * blockDim.z + threadIdx.z;
    const int nx = A.nx, ny = A.ny, nz = A.nz;
    if (i >= nx || j >= ny || kz >= nz) return;
    const bool hasW = i > 0, hasE = i < nx - 1, hasS = j > 0, hasN = j < ny - 1, hasB = kz > 0, hasT = kz < nz - 1;
    const int iw = hasW ? i - 1 : i, ie = hasE ? i + 1 : i, js = hasS ? j - 1 : j, jn = hasN ? j + 1 : j;
    const int kb = hasB ? kz - 1 : kz, kt = hasT ? kz + 1 : kz;
    auto at = [nx, ny](const T* P, int ii, int jj, int kk) { return __ldg(P + ((size_t)kk * ny + jj) * nx + ii); };
    Cell3<T> c;
    c.u = at(A.U, i, j, kz); c.v = at(A.V, i, j, kz); c.w = at(A.W, i, j, kz);
    c.uE = at(A.U, ie, j, kz); c.uW = at(A.U, iw, j, kz); c.uN = at(A.U, i, jn, kz); c.uS = at(A.U, i, js, kz);
    c.uT = at(A.U, i, j, kt); c.uB = at(A.U, i, j, kb);
    c.vE = at(A.V, ie, j, kz); c.vW = at(A.V, iw, j, kz); c.vN = at(A.V, i, jn, kz); c.vS = at(A.V, i, js, kz);
    c.vT = at(A.V, i, j, kt); c.vB = at(A.V, i, j, kb);
    c.wE = at(A.W, ie, j, kz); c.wW = at(A.W, iw, j, kz); c.wN = at(A.W, i, jn, kz); c.wS = at(A.W, i, js, kz);
    c.wT = at(A.W, i, j, kt); c.wB = at(A.W, i, j, kb);
    c.wNE = at(A.W, ie, jn, kz); c.wNW = at(A.W, iw, jn, kz); c.wSE = at(A.W, ie, js, kz); c.wSW = at(A.W, iw, js, kz);
    c.wTE = at(A.W, ie, j, kt); c.wTW = at(A.W, iw, j, kt); c.wBE = at(A.W, ie, j, kb); c.wBW = at(A.W, iw, j, kb);
    c.wTN = at(A.W, i, jn, kt); c.wTS = at(A.W, i, js, kt); c.wBN = at(A.W, i, jn, kb); c.wBS = at(A.W, i, js, kb);
    c.fxC = at(A.fx, i, j, kz); c.fxE = at(A.fx, ie, j, kz);
    c.fyC = at(A.fy, i, j, kz); c.fyN = at(A.fy, i, jn, kz);
    c.fzC = at(A.fz, i, j, kz); c.fzT = at(A.fz, i, j, kt);
    c.gxyE = at(A.gxy, ie, j, kz); c.gxyW = at(A.gxy, iw, j, kz); c.gxyN = at(A.gxy, i, jn, kz); c.gxyS = at(A.gxy, i, js, kz);
    c.gxzE = at(A.gxz, ie, j, kz); c.gxzW = at(A.gxz, iw, j, kz); c.gxzT = at(A.gxz, i, j, kt); c.gxzB = at(A.gxz, i, j, kb);
    c.gyzN = at(A.gyz, i, jn, kz); c.gyzS = at(A.gyz, i, js, kz); c.gyzT = at(A.gyz, i, j, kt); c.gyzB = at(A.gyz, i, j, kb);
    T oU, oV, oW;
    cell3(A.k, c, hasE, hasW, hasN, hasS, hasT, hasB, oU, oV, oW);
    const size_t q = ((size_t)kz * ny + j) * nx + i;
    A.U1[q] = oU; A.V1[q] = oV; A.W1[q] = oW;
}

}  // namespace gg3

// gg3_tiled.cuh -- GG3_KERNEL_TILED: the 3-D step on xy tiles marched along z.
//
// The 3-D step is HBM-bound like the 2-D one: 3 fields read, 3 written, 6 stored tensor fields
// read = 96 B (fp64) / 48 B (fp32) of compulsory traffic per cell-step against ~90 arithmetic
// instructions.  The one-thread-per-cell kernel touches 60 operands per cell through L1/L2; this
// kernel reads every operand from HBM once per tile:
//
//  * A CTA owns a kTileX x kTileY tile of the xy plane and a chunk of z; thread (li, lj) owns the
//    cell column (i, j, .) and marches up the chunk one plane at a time.
//  * What a cell needs from its own column (U, V, gxz, gyz of planes k-1, k, k+1; fz of k, k+1) rolls
//    through REGISTERS: each value is loaded once, one plane ahead.
//  * What it needs from neighbouring columns goes through SHARED MEMORY planes with a one-cell
//    halo: W of planes k-1, k, k+1 (a ring of three), U, V, gxy, gxz, gyz, fx, fy of plane k.  A
//    plane's interior is written from the owners' registers, its halo ring (84 cells) by the first
//    84 threads straight from global memory.  Coordinates are clamped to the domain, so the planes
//    hold the even-mirror extension and the Neumann faces need no special case here (cell3 flips
//    the sign of the cross terms taken at clamped neighbours).
//  * Same operands, same cell3 as the generic kernel => bit-identical results.
#pragma once
#include "gg3_kernels.cuh"

namespace gg3 {

constexpr int kTileX = 32, kTileY = 8;
constexpr int kPX = kTileX + 2, kPY = kTileY + 2, kPlane = kPX * kPY;   // haloed plane
constexpr int kHalo = 2 * kPX + 2 * kTileY;                              // cells of the halo ring

__host__ __device__ inline bool tiled_shape_ok(int nx, int ny, int nz) { return nx >= 2 && ny >= 2 && nz >= 2; }
// chunks along z: enough CTAs to fill the GPU several times over, but at least 8 planes per chunk
// (every chunk re-reads two planes of W and one of everything else)
__host__ __device__ inline int tiled_zchunks(int nx, int ny, int nz) {
    const long long tiles = (long long)((nx + kTileX - 1) / kTileX) * ((ny + kTileY - 1) / kTileY);
    long long want = (148LL * 16 + tiles - 1) / tiles;
    const long long most = nz / 8 > 0 ? nz / 8 : 1;
    if (want > most) want = most;
    if (want < 1) want = 1;
    return (int)want;
}

template <typename T>
__global__ void __launch_bounds__(kTileX * kTileY) gg3_step_tiled(const Args3<T> A) {
    __shared__ T sW[3][kPlane];
    __shared__ T sU[kPlane], sV[kPlane], sGxy[kPlane], sGxz[kPlane], sGyz[kPlane], sFx[kPlane], sFy[kPlane];
    const int nx = A.nx, ny = A.ny, nz = A.nz;
    const int li = threadIdx.x, lj = threadIdx.y, tid = lj * kTileX + li;
    const int i0 = blockIdx.x * kTileX, j0 = blockIdx.y * kTileY;
    const int i = i0 + li, j = j0 + lj;
    const bool active = i < nx && j < ny;
    const int ic = min(i, nx - 1), jc = min(j, ny - 1);                  // clamped own column (inactive threads)
    const int nch = gridDim.z, per = (nz + nch - 1) / nch;
    const int z0 = blockIdx.z * per, z1 = min(z0 + per, nz);
    if (z0 >= z1) return;
    const size_t plane = (size_t)nx * ny;
    const size_t col = (size_t)jc * nx + ic;
    // the halo cell this thread fills (threads 0..kHalo-1), as plane index and clamped global column
    int hp = -1;
    size_t hcol = 0;
    if (tid < kHalo) {
        int hi, hj;
        if (tid < kPX) { hi = tid - 1; hj = -1; }
        else if (tid < 2 * kPX) { hi = tid - kPX - 1; hj = kTileY; }
        else { const int q = tid - 2 * kPX; hi = q < kTileY ? -1 : kTileX; hj = q < kTileY ? q : q - kTileY; }
        hp = (hj + 1) * kPX + (hi + 1);
        hcol = (size_t)min(max(j0 + hj, 0), ny - 1) * nx + min(max(i0 + hi, 0), nx - 1);
    }
    const int cp = (lj + 1) * kPX + (li + 1);                            // own cell in a haloed plane
    const bool hasW = i > 0, hasE = i < nx - 1, hasS = j > 0, hasN = j < ny - 1;
    auto zc = [nz](int k) { return min(max(k, 0), nz - 1); };

    // ---- prologue: planes z0-1 and z0 of W; column registers for planes z0-1, z0
    {
        const size_t pb = (size_t)zc(z0 - 1) * plane, pc = (size_t)z0 * plane;
        sW[(z0 + 2) % 3][cp] = A.W[pb + col];
        sW[z0 % 3][cp] = A.W[pc + col];
        if (hp >= 0) { sW[(z0 + 2) % 3][hp] = A.W[pb + hcol]; sW[z0 % 3][hp] = A.W[pc + hcol]; }
    }
    T uB = A.U[(size_t)zc(z0 - 1) * plane + col], uC = A.U[(size_t)z0 * plane + col];
    T vB = A.V[(size_t)zc(z0 - 1) * plane + col], vC = A.V[(size_t)z0 * plane + col];
    T gxzB = A.gxz[(size_t)zc(z0 - 1) * plane + col], gxzC = A.gxz[(size_t)z0 * plane + col];
    T gyzB = A.gyz[(size_t)zc(z0 - 1) * plane + col], gyzC = A.gyz[(size_t)z0 * plane + col];
    T fzC = A.fz[(size_t)z0 * plane + col];

    for (int k = z0; k < z1; ++k) {
        const size_t pk = (size_t)k * plane, pt = (size_t)zc(k + 1) * plane;
        // one plane ahead: own column
        const T wT = A.W[pt + col], uT = A.U[pt + col], vT = A.V[pt + col];
        const T gxzT = A.gxz[pt + col], gyzT = A.gyz[pt + col], fzT = A.fz[pt + col];
        const T gxyC = A.gxy[pk + col], fxC = A.fx[pk + col], fyC = A.fy[pk + col];
        __syncthreads();                       // everybody is done with the planes of step k-1
        T* wt = sW[(k + 1) % 3];
        wt[cp] = wT;
        sU[cp] = uC; sV[cp] = vC; sGxy[cp] = gxyC; sGxz[cp] = gxzC; sGyz[cp] = gyzC; sFx[cp] = fxC; sFy[cp] = fyC;
        if (hp >= 0) {
            wt[hp] = A.W[pt + hcol];
            sU[hp] = A.U[pk + hcol]; sV[hp] = A.V[pk + hcol];
            sGxy[hp] = A.gxy[pk + hcol]; sGxz[hp] = A.gxz[pk + hcol]; sGyz[hp] = A.gyz[pk + hcol];
            sFx[hp] = A.fx[pk + hcol]; sFy[hp] = A.fy[pk + hcol];
        }
        __syncthreads();
        if (active) {
            const T* wb = sW[(k + 2) % 3];
            const T* wc = sW[k % 3];
            Cell3<T> c;
            c.u = uC; c.v = vC; c.w = wc[cp];
            c.uE = sU[cp + 1]; c.uW = sU[cp - 1]; c.uN = sU[cp + kPX]; c.uS = sU[cp - kPX]; c.uT = uT; c.uB = uB;
            c.vE = sV[cp + 1]; c.vW = sV[cp - 1]; c.vN = sV[cp + kPX]; c.vS = sV[cp - kPX]; c.vT = vT; c.vB = vB;
            c.wE = wc[cp + 1]; c.wW = wc[cp - 1]; c.wN = wc[cp + kPX]; c.wS = wc[cp - kPX]; c.wT = wt[cp]; c.wB = wb[cp];
            c.wNE = wc[cp + kPX + 1]; c.wNW = wc[cp + kPX - 1]; c.wSE = wc[cp - kPX + 1]; c.wSW = wc[cp - kPX - 1];
            c.wTE = wt[cp + 1]; c.wTW = wt[cp - 1]; c.wBE = wb[cp + 1]; c.wBW = wb[cp - 1];
            c.wTN = wt[cp + kPX]; c.wTS = wt[cp - kPX]; c.wBN = wb[cp + kPX]; c.wBS = wb[cp - kPX];
            c.fxC = fxC; c.fxE = sFx[cp + 1]; c.fyC = fyC; c.fyN = sFy[cp + kPX]; c.fzC = fzC; c.fzT = fzT;
            c.gxyE = sGxy[cp + 1]; c.gxyW = sGxy[cp - 1]; c.gxyN = sGxy[cp + kPX]; c.gxyS = sGxy[cp - kPX];
            c.gxzE = sGxz[cp + 1]; c.gxzW = sGxz[cp - 1]; c.gxzT = gxzT; c.gxzB = gxzB;
            c.gyzN = sGyz[cp + kPX]; c.gyzS = sGyz[cp - kPX]; c.gyzT = gyzT; c.gyzB = gyzB;
            T oU, oV, oW;
            cell3(A.k, c, hasE, hasW, hasN, hasS, k < nz - 1, k > 0, oU, oV, oW);
            A.U1[pk + col] = oU; A.V1[pk + col] = oV; A.W1[pk + col] = oW;
        }
        uB = uC; uC = uT; vB = vC; vC = vT; gxzB = gxzC; gxzC = gxzT; gyzB = gyzC; gyzC = gyzT; fzC = fzT;
    }
}

}  // namespace gg3

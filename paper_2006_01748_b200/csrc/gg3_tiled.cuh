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
//    halo: W of planes k-1, k, k+1 (a ring of four: plane k+2 is staged while k is computed), U, V,
//    gxy, gxz, gyz, fx, fy of plane k (two buffers).  A plane's interior is written from the owners'
//    registers, its halo ring (84 cells) by the first 84 threads; every global load is issued one
//    step before its value is stored to shared memory or used, and ONE barrier separates planes.  Coordinates are clamped to the domain, so the planes
//    hold the even-mirror extension and the Neumann faces need no special case here (cell3 flips
//    the sign of the cross terms taken at clamped neighbours).
//  * Same operands, same cell3 as the generic kernel => bit-identical results.
#pragma once
#include "gg3_kernels.cuh"

namespace gg3 {

#ifndef GG3_TILE_Y
#define GG3_TILE_Y 4
#endif
#ifndef GG3_TILE_X
#define GG3_TILE_X 64
#endif
constexpr int kTileX = GG3_TILE_X, kTileY = GG3_TILE_Y;
constexpr int kPX = kTileX + 2, kPY = kTileY + 2, kPlane = kPX * kPY;   // haloed plane
constexpr int kHalo = 2 * kPX + 2 * kTileY;                              // cells of the halo ring
static_assert(kHalo <= kTileX * kTileY, "one halo cell per thread at most");

__host__ __device__ inline bool tiled_shape_ok(int nx, int ny, int nz) { return nx >= 2 && ny >= 2 && nz >= 2; }
// chunks along z: enough CTAs to fill the GPU several times over, but at least 8 planes per chunk
// (every chunk re-reads two planes of W and one of everything else)
__host__ __device__ inline int tiled_zchunks(int nx, int ny, int nz, int num_sms) {
    const long long tiles = (long long)((nx + kTileX - 1) / kTileX) * ((ny + kTileY - 1) / kTileY);
    long long want = ((long long)num_sms * 16 + tiles - 1) / tiles;
    const long long most = nz / 8 > 0 ? nz / 8 : 1;
    if (want > most) want = most;
    if (want < 1) want = 1;
    return (int)want;
}

// dynamic shared memory: W ring of four haloed planes, then two buffers of seven haloed planes
// (U, V, gxy, gxz, gyz, fx, fy)
template <typename T> __host__ __device__ constexpr size_t tiled_smem_bytes() { return (size_t)(4 + 2 * 7) * kPlane * sizeof(T); }

template <typename T>
__global__ void __launch_bounds__(kTileX * kTileY) gg3_step_tiled(const Args3<T> A) {
    extern __shared__ __align__(16) unsigned char smem3[];
    T* sW = reinterpret_cast<T*>(smem3);                 // [4][kPlane]
    T* sP = sW + 4 * kPlane;                             // [2][7][kPlane]
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
    const bool halo = tid < kHalo;
    int hp = 0;
    size_t hcol = 0;
    if (halo) {
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
    const T* gP[7] = {A.U, A.V, A.gxy, A.gxz, A.gyz, A.fx, A.fy};

    // ---- prologue: W planes z0-1, z0, z0+1; the seven planes of z0; column registers
    for (int q = -1; q <= 1; ++q) {
        const size_t pq = (size_t)zc(z0 + q) * plane;
        T* w = sW + ((z0 + q + 4) & 3) * kPlane;
        w[cp] = A.W[pq + col];
        if (halo) w[hp] = A.W[pq + hcol];
    }
    {
        const size_t pc = (size_t)z0 * plane;
        T* b = sP + (z0 & 1) * 7 * kPlane;
#pragma unroll
        for (int f = 0; f < 7; ++f) {
            b[f * kPlane + cp] = gP[f][pc + col];
            if (halo) b[f * kPlane + hp] = gP[f][pc + hcol];
        }
    }
    const size_t pb0 = (size_t)zc(z0 - 1) * plane, pc0 = (size_t)z0 * plane, pt0 = (size_t)zc(z0 + 1) * plane;
    T uB = A.U[pb0 + col], uC = A.U[pc0 + col], uT = A.U[pt0 + col];
    T vB = A.V[pb0 + col], vC = A.V[pc0 + col], vT = A.V[pt0 + col];
    T gxzB = A.gxz[pb0 + col], gxzC = A.gxz[pc0 + col], gxzT = A.gxz[pt0 + col];
    T gyzB = A.gyz[pb0 + col], gyzC = A.gyz[pc0 + col], gyzT = A.gyz[pt0 + col];
    T fzC = A.fz[pc0 + col], fzT = A.fz[pt0 + col];
    T gxyC = A.gxy[pc0 + col], fxC = A.fx[pc0 + col], fyC = A.fy[pc0 + col];
    __syncthreads();

    for (int k = z0; k < z1; ++k) {
        const size_t pk = (size_t)k * plane, p1 = (size_t)zc(k + 1) * plane, p2 = (size_t)zc(k + 2) * plane;
        const bool more = k + 1 < z1;
        // in flight while plane k is computed: own column two planes ahead, what plane k+1 needs
        // from the tensor, and the halo cells of both
        T w2 = (T)0, u2 = (T)0, v2 = (T)0, gxz2 = (T)0, gyz2 = (T)0, fz2 = (T)0, gxy1 = (T)0, fx1 = (T)0, fy1 = (T)0;
        T hw2 = (T)0, h1[7] = {(T)0, (T)0, (T)0, (T)0, (T)0, (T)0, (T)0};
        if (more) {
            w2 = A.W[p2 + col]; u2 = A.U[p2 + col]; v2 = A.V[p2 + col];
            gxz2 = A.gxz[p2 + col]; gyz2 = A.gyz[p2 + col]; fz2 = A.fz[p2 + col];
            gxy1 = A.gxy[p1 + col]; fx1 = A.fx[p1 + col]; fy1 = A.fy[p1 + col];
            if (halo) {
                hw2 = A.W[p2 + hcol];
#pragma unroll
                for (int f = 0; f < 7; ++f) h1[f] = gP[f][p1 + hcol];
            }
        }
        if (active) {
            const T* wb = sW + ((k + 3) & 3) * kPlane;
            const T* wc = sW + (k & 3) * kPlane;
            const T* wt = sW + ((k + 1) & 3) * kPlane;
            const T* b = sP + (k & 1) * 7 * kPlane;
            const T *sU = b, *sV = b + kPlane, *sGxy = b + 2 * kPlane, *sGxz = b + 3 * kPlane, *sGyz = b + 4 * kPlane,
                    *sFx = b + 5 * kPlane, *sFy = b + 6 * kPlane;
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
        if (more) {
            // stage plane k+2 of W (ring slot last read as plane k-2) and the seven planes of k+1
            // (the buffer last read at step k-1); one barrier per plane
            T* w = sW + ((k + 2) & 3) * kPlane;
            T* b = sP + ((k + 1) & 1) * 7 * kPlane;
            w[cp] = w2;
            b[cp] = uT; b[kPlane + cp] = vT; b[2 * kPlane + cp] = gxy1; b[3 * kPlane + cp] = gxzT; b[4 * kPlane + cp] = gyzT;
            b[5 * kPlane + cp] = fx1; b[6 * kPlane + cp] = fy1;
            if (halo) {
                w[hp] = hw2;
#pragma unroll
                for (int f = 0; f < 7; ++f) b[f * kPlane + hp] = h1[f];
            }
            __syncthreads();
        }
        uB = uC; uC = uT; uT = u2; vB = vC; vC = vT; vT = v2;
        gxzB = gxzC; gxzC = gxzT; gxzT = gxz2; gyzB = gyzC; gyzC = gyzT; gyzT = gyz2;
        fzC = fzT; fzT = fz2; gxyC = gxy1; fxC = fx1; fyC = fy1;
    }
}

}  // namespace gg3

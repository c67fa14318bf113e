// gg_stream.cuh -- GG_KERNEL_STREAM: the fused single-step kernel for sm_100a.
//
// Design.  The step is HBM-bound (72 B and ~45 flops per cell in fp64), so
// the kernel is built around keeping many TMA loads in flight and touching every byte once:
//
//  * The grid is cut into column STRIPS 512 bytes wide (64 fp64 / 128 fp32 cells) and row CHUNKS.
//    One WARP owns one (simulation, chunk, strip) item at a time and is a self-contained
//    producer + consumer: its lane 0 issues `cp.async.bulk.tensor` (TMA) loads of RB-row boxes of
//    the six input arrays (U, V, W, a, b, c; strip plus a 16-byte halo on each side, rows j0-1..j1)
//    into a warp-private ring of NST stages in shared memory, completion signalled on one
//    mbarrier per stage.  No __syncthreads, no inter-warp dependence: warps drift apart and keep
//    the memory system evenly loaded.  Out-of-domain parts of a box are zero-filled by TMA.
//  * The warp marches up its strip one row at a time.  Every lane owns 16 bytes of each row
//    (2 fp64 / 4 fp32 cells) and keeps a rolling window of rows j-1, j, j+1 in REGISTERS, so each
//    shared-memory element is read once per lane that needs it.  The north face fluxes of row j
//    are kept and reused as the south face fluxes of row j+1; x-face fluxes inside a lane's run
//    are computed once and used by both adjacent cells.  (The run's west face is recomputed by
//    the lane instead of shuffled from its neighbour: cheaper than the exchange.)
//  * Neumann boundaries (reading A2): faces on the domain boundary carry zero flux, tangential
//    differences use the mirrored neighbour.  Handled with warp-uniform row tests and two
//    per-lane flags; TMA's zero fill keeps every discarded value finite.
//  * Results leave as one 16-byte store per lane per field per row: 512 contiguous bytes per warp.
#pragma once
#include <cuda.h>

#include "gg_common.cuh"

namespace gg {

constexpr int kStripBytes = 512;              // 32 lanes x 16 B
constexpr int kRowBytes = kStripBytes + 32;   // + 16 B halo each side (TMA box inner extent)

template <int RB>
__host__ __device__ constexpr int slab_bytes() { return (RB * kRowBytes + 127) / 128 * 128; }

struct alignas(64) StreamArgs {
    CUtensorMap mU, mV, mW, ma, mb, mc;  // rank-3 maps {nx, ny, B}, box {row, RB, 1}
    void* U1;                            // outputs [B][ny][nx]
    void* V1;
    void* W1;
    const SimScalars* sims;
    int nx, ny, nbatch;
    int nstrips, nchunks, chunk_rows;
    long long nitems;
    double dt, inv_h2;
};

// Host-side plan: tensor maps for both ping-pong copies and the launch geometry.
struct StreamPlan {
    CUtensorMap state[2][3];
    CUtensorMap coef[3];
    int nstrips = 0, nchunks = 0, chunk_rows = 0;
    long long nitems = 0;
    int grid = 0, block = 0;
    size_t smem = 0;
    int rb = 0, nst = 0, nw = 0;
};

// ------------------------------------------------------------------------------------------
// PTX wrappers (sm_100a)
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    // bounded spin: a lost TMA completion traps instead of hanging the GPU
    for (uint32_t spins = 0; !mbar_try_wait(bar, parity); ++spins)
        if (spins > (1u << 26)) __trap();
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, uint32_t bar,
                                            int x, int y, int z) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes "
        "[%0], [%1, {%3, %4, %5}], [%2];" ::"r"(dst),
        "l"(map), "r"(bar), "r"(x), "r"(y), "r"(z)
        : "memory");
}
__device__ __forceinline__ void fence_barrier_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

// 16-byte vector of T
template <typename T> struct Vec16;
template <> struct Vec16<double> { using type = double2; };
template <> struct Vec16<float> { using type = float4; };

template <typename T, int C>
__device__ __forceinline__ void lds_own(const char* p, T* x) {
    typename Vec16<T>::type v = *reinterpret_cast<const typename Vec16<T>::type*>(p);
    if constexpr (C == 2) { x[0] = v.x; x[1] = v.y; }
    else { x[0] = v.x; x[1] = v.y; x[2] = v.z; x[3] = v.w; }
}
// own C cells into x[1..C], west neighbour into x[0], east neighbour into x[C+1]
template <typename T, int C>
__device__ __forceinline__ void lds_ext(const char* p, T* x) {
    lds_own<T, C>(p, x + 1);
    x[0] = *reinterpret_cast<const T*>(p - sizeof(T));
    x[C + 1] = *reinterpret_cast<const T*>(p + 16);
}
template <typename T, int C>
__device__ __forceinline__ void stg_own(T* g, const T* x) {
    typename Vec16<T>::type v;
    if constexpr (C == 2) { v.x = x[0]; v.y = x[1]; }
    else { v.x = x[0]; v.y = x[1]; v.z = x[2]; v.w = x[3]; }
    *reinterpret_cast<typename Vec16<T>::type*>(g) = v;
}

// ------------------------------------------------------------------------------------------
// The kernel.  T: arithmetic/storage type; RB: rows per TMA box (= per ring stage); NST: ring
// stages per warp; NW: warps per CTA.  Dynamic shared memory:
//   [NW*NST mbarriers, padded to 128 B][NW warps][NST stages][6 arrays][slab_bytes<RB>()]
// ------------------------------------------------------------------------------------------
template <typename T, int RB, int NST, int NW>
__global__ void __launch_bounds__(NW * 32, 1) gg_step_stream(const __grid_constant__ StreamArgs A) {
    constexpr int C = 16 / (int)sizeof(T);  // cells per lane per row
    constexpr int SW = 32 * C;              // strip width in cells
    constexpr int E = C + 2;                // extended run: west nbr, C own cells, east nbr
    constexpr int SLAB = slab_bytes<RB>();
    constexpr int STAGE = 6 * SLAB;
    constexpr uint32_t STAGE_TX = 6u * RB * kRowBytes;
    constexpr int BAR_BYTES = (NW * NST * 8 + 127) / 128 * 128;

    extern __shared__ __align__(128) char smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t bar0 = smem_u32(smem) + (uint32_t)(warp * NST) * 8u;
    char* ring = smem + BAR_BYTES + (size_t)warp * NST * STAGE;
    const uint32_t ring_u32 = smem_u32(ring);

    if (lane == 0) {
        for (int s = 0; s < NST; ++s) mbar_init(bar0 + 8u * s, 1);
        fence_barrier_init();
        fence_proxy_async();
    }
    __syncwarp();

    const int nx = A.nx, ny = A.ny;
    const size_t plane = (size_t)nx * ny;
    const long long gwarp = (long long)blockIdx.x * NW + warp;
    const long long nwarps = (long long)gridDim.x * NW;
    uint32_t gq = 0;  // stages consumed so far by this warp (slot = gq % NST, phase = gq / NST & 1)

    for (long long item = gwarp; item < A.nitems; item += nwarps) {
        const int strip = (int)(item % A.nstrips);
        const long long t = item / A.nstrips;
        const int chunk = (int)(t % A.nchunks);
        const int sim = (int)(t / A.nchunks);
        const int i0 = strip * SW;
        const int j0 = chunk * A.chunk_rows;
        const int j1 = min(j0 + A.chunk_rows, ny);
        const int nr = j1 - j0 + 2;             // rows j0-1 .. j1 arrive
        const int nstage = (nr + RB - 1) / RB;
        const int iown = i0 + lane * C;         // first own cell
        const bool valid = iown < nx;           // nx % C == 0: a lane's run is all in or all out
        const bool atW = iown == 0, atE = iown + C == nx;
        const StepCoef<T> k = fold_coef<T>(A.sims[sim], A.dt, A.inv_h2);
        T* gU = (T*)A.U1 + sim * plane + iown;
        T* gV = (T*)A.V1 + sim * plane + iown;
        T* gW = (T*)A.W1 + sim * plane + iown;

        auto issue = [&](int q, uint32_t slot) {  // lane 0 only
            const uint32_t bar = bar0 + 8u * slot;
            const uint32_t dst = ring_u32 + slot * STAGE;
            const int x = i0 - C, y = j0 - 1 + q * RB;
            mbar_expect_tx(bar, STAGE_TX);
            tma_load_3d(dst + 0 * SLAB, &A.mU, bar, x, y, sim);
            tma_load_3d(dst + 1 * SLAB, &A.mV, bar, x, y, sim);
            tma_load_3d(dst + 2 * SLAB, &A.mW, bar, x, y, sim);
            tma_load_3d(dst + 3 * SLAB, &A.ma, bar, x, y, 0);
            tma_load_3d(dst + 4 * SLAB, &A.mb, bar, x, y, 0);
            tma_load_3d(dst + 5 * SLAB, &A.mc, bar, x, y, 0);
        };
        if (lane == 0) {
            const int pre = nstage < NST ? nstage : NST;
            for (int q = 0; q < pre; ++q) issue(q, (gq + q) % NST);
        }

        // rolling register window (rows jc-1, jc, jc+1 = P, C, N)
        T wP[E], wC[E], wN[E], uC[E], uN[E], vC[E], vN[E], aC[E], aN[E], bC[E], bN[E];
        T cC[C], cN[C], hC[C], hN[C], sV[C], sW[C];
#pragma unroll
        for (int e = 0; e < E; ++e) wP[e] = wC[e] = uC[e] = vC[e] = aC[e] = bC[e] = (T)0;
#pragma unroll
        for (int c = 0; c < C; ++c) cC[c] = hC[c] = sV[c] = sW[c] = (T)0;

        for (int q = 0; q < nstage; ++q, ++gq) {
            const uint32_t slot = gq % NST;
            mbar_wait(bar0 + 8u * slot, (gq / NST) & 1u);
            const char* st = ring + (size_t)slot * STAGE + 16 + 16 * lane;
#pragma unroll
            for (int rr = 0; rr < RB; ++rr) {
                const int n = q * RB + rr;  // arrival index; arriving row = j0-1+n
                if (n < nr) {
                    const char* row = st + rr * kRowBytes;
                    lds_ext<T, C>(row + 0 * SLAB, uN);
                    lds_ext<T, C>(row + 1 * SLAB, vN);
                    lds_ext<T, C>(row + 2 * SLAB, wN);
                    lds_ext<T, C>(row + 3 * SLAB, aN);
                    lds_ext<T, C>(row + 4 * SLAB, bN);
                    lds_own<T, C>(row + 5 * SLAB, cN);
                    // mirrored x ghosts of W (tangential difference in H at boundary cells)
                    if (atW) wN[0] = wN[1];
                    if (atE) wN[C + 1] = wN[C];
#pragma unroll
                    for (int c = 0; c < C; ++c) hN[c] = bN[c + 1] * (wN[c + 2] - wN[c]);

                    const int jc = j0 - 2 + n;  // centre row being computed (valid output if n >= 2)
                    if (n >= 1) {
                        // cross term G with mirrored y ghosts (warp-uniform tests)
                        T G[E];
                        if (jc == 0) {
#pragma unroll
                            for (int e = 0; e < E; ++e) G[e] = bC[e] * (wN[e] - wC[e]);
                        } else if (jc == ny - 1) {
#pragma unroll
                            for (int e = 0; e < E; ++e) G[e] = bC[e] * (wC[e] - wP[e]);
                        } else {
#pragma unroll
                            for (int e = 0; e < E; ++e) G[e] = bC[e] * (wN[e] - wP[e]);
                        }
                        // x faces f = 0..C (face f lies between extended cells f and f+1)
                        T pV[C + 1], pW[C + 1];
#pragma unroll
                        for (int f = 0; f <= C; ++f) {
                            pV[f] = flux_V(uC[f], uC[f + 1], vC[f], vC[f + 1]);
                            pW[f] = flux_W(aC[f], aC[f + 1], wC[f], wC[f + 1], G[f], G[f + 1]);
                        }
                        if (atW) { pV[0] = (T)0; pW[0] = (T)0; }
                        if (atE) { pV[C] = (T)0; pW[C] = (T)0; }
                        // north faces of the own cells; zero on the domain boundary
                        T nV[C], nW[C];
                        if (jc >= 0 && jc < ny - 1) {
#pragma unroll
                            for (int c = 0; c < C; ++c) {
                                nV[c] = flux_V(uC[c + 1], uN[c + 1], vC[c + 1], vN[c + 1]);
                                nW[c] = flux_W(cC[c], cN[c], wC[c + 1], wN[c + 1], hC[c], hN[c]);
                            }
                        } else {
#pragma unroll
                            for (int c = 0; c < C; ++c) nV[c] = nW[c] = (T)0;
                        }
                        if (n >= 2) {
                            T oU[C], oV[C], oW[C];
#pragma unroll
                            for (int c = 0; c < C; ++c) {
                                const T divV = (pV[c + 1] - pV[c]) + (nV[c] - sV[c]);
                                const T divW = (pW[c + 1] - pW[c]) + (nW[c] - sW[c]);
                                oU[c] = upd_U(k, uC[c + 1], wC[c + 1]);
                                oV[c] = upd_V(k, vC[c + 1], divV);
                                oW[c] = upd_W(k, vC[c + 1], wC[c + 1], divW);
                            }
                            if (valid) {
                                const size_t off = (size_t)jc * nx;
                                stg_own<T, C>(gU + off, oU);
                                stg_own<T, C>(gV + off, oV);
                                stg_own<T, C>(gW + off, oW);
                            }
                        }
#pragma unroll
                        for (int c = 0; c < C; ++c) { sV[c] = nV[c]; sW[c] = nW[c]; }
                    }
                    // roll the window
#pragma unroll
                    for (int e = 0; e < E; ++e) {
                        wP[e] = wC[e]; wC[e] = wN[e];
                        uC[e] = uN[e]; vC[e] = vN[e]; aC[e] = aN[e]; bC[e] = bN[e];
                    }
#pragma unroll
                    for (int c = 0; c < C; ++c) { cC[c] = cN[c]; hC[c] = hN[c]; }
                }
            }
            // the stage has been read into registers by every lane: refill it
            __syncwarp();
            if (lane == 0 && q + NST < nstage) issue(q + NST, slot);
        }
    }
}

}  // namespace gg

// gg_stream2.cuh -- GG_KERNEL_STREAM2: two time steps fused per launch (temporal blocking).
//
// The single-step kernel (gg_stream.cuh) already moves 1.02x the compulsory bytes at the HBM copy
// rate with the SMs ~22 % busy, so the only way up is to move fewer bytes per step: advance the
// state by TWO steps per pass over HBM.  The kernel is two copies of the row
// march chained through shared memory:
//
//   TMA producer warp --ring0 (U,V,W,a,b,c at time k)--> NW "step-1" warps + 1 halo warp
//                     --ring1 (U,V,W at time k+1 + a,b,c)--> NW "step-2" warps --> HBM (time k+2)
//
//  * A CTA owns a tile column of NW = 4 adjacent 512-byte strips.  ring0 stages are filled by TMA
//    exactly as in the single-step kernel, with a two-column halo box on each side of the tile.
//  * Step-1 warp w marches strip w through ring0 and, instead of storing to HBM, writes the
//    time-(k+1) row and the row's a, b, c into ring1 at the same offsets.  The two tile-edge
//    columns of time k+1 (x0-1 and x0+TW), which step 2 needs as halo, are marched by two lanes
//    of the halo warp (a C = 1 instance of the same march) from ring0's halo slabs.
//  * Step-2 warp w marches strip w through ring1 -- the same code, ghost rows and boundary faces
//    included -- and stores time k+2.  It trails step 1 by about one stage.
//  * Rows: a chunk [j0, j1) loads rows j0-2 .. j1+1, computes time-(k+1) rows j0-1 .. j1 and
//    stores time-(k+2) rows j0 .. j1-1 (2 redundant rows per chunk and step).
//  * mbarriers: full0 (TMA bytes), empty0 (NW+1 step-1 consumers), full1 (NW+1 ring1 writers),
//    empty1 (NW step-2 consumers).  No __syncthreads after start-up.
// Arithmetic is the single-step march's, applied twice: results are bit-identical to two
// launches of GG_KERNEL_STREAM (tests/test_gpu_parity.py checks that).
#pragma once
#include "gg_stream.cuh"

namespace gg {

constexpr int kHalo2Arrays = 6;  // U, V, W, a, b, c halo slabs per side

__host__ __device__ constexpr int stream2_stage_bytes(int rb, int nw) {
    return nw * 6 * rb * kStripBytes + 2 * kHalo2Arrays * kHaloSlab;
}
__host__ __device__ constexpr int stream2_smem_bytes(int rb, int nst0, int nst1, int nw) {
    return 256 + (nst0 + nst1) * stream2_stage_bytes(rb, nw);
}

struct Stream2Item {
    int sim, i0, j0, j1, nr, nstage;
};
template <int RB, int TILE_CELLS>
__device__ __forceinline__ Stream2Item stream2_item(const StreamArgs& A, long long item) {
    Stream2Item it;
    const int tc = (int)(item % A.ntilecols);
    const long long t = item / A.ntilecols;
    const int chunk = (int)(t % A.nchunks);
    it.sim = (int)(t / A.nchunks);
    it.i0 = tc * TILE_CELLS;
    it.j0 = chunk * A.chunk_rows;
    it.j1 = min(it.j0 + A.chunk_rows, A.ny);
    it.nr = it.j1 - it.j0 + 4;  // time-k rows j0-2 .. j1+1 arrive
    it.nstage = (it.nr + RB - 1) / RB;
    return it;
}

template <typename T, int RB, int NST0, int NST1, int NW>
__global__ void __launch_bounds__((2 * NW + 2) * 32, 1)
gg_step_stream2(const __grid_constant__ StreamArgs A) {
    constexpr int C = 16 / (int)sizeof(T);
    constexpr int SW = 32 * C;
    constexpr int GW = (256 / SW) < NW ? (256 / SW) : NW;
    constexpr int NG = NW / GW;
    constexpr int BOXB = GW * kStripBytes;
    constexpr int SLABG = RB * BOXB;
    constexpr int ARR = NG * SLABG;
    constexpr int MAIN = 6 * ARR;
    constexpr int HSIDE = kHalo2Arrays * kHaloSlab;  // halo slabs of one side
    constexpr int STAGE = stream2_stage_bytes(RB, NW);
    static_assert(NW % GW == 0, "warps per step must be a multiple of the strips per box");
    static_assert(RB * kHaloBytes <= kHaloSlab, "halo slab too small");
    static_assert((2 * NST0 + 2 * NST1) * 8 <= 256, "too many stages");

    extern __shared__ __align__(128) char smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t full0 = smem_u32(smem), empty0 = full0 + 8u * NST0;
    const uint32_t full1 = empty0 + 8u * NST0, empty1 = full1 + 8u * NST1;
    char* ring0 = smem + 256;
    char* ring1 = ring0 + (size_t)NST0 * STAGE;
    const uint32_t ring0_u32 = smem_u32(ring0);

    if (threadIdx.x == 0) {
        for (int s = 0; s < NST0; ++s) {
            mbar_init(full0 + 8u * s, 1);
            mbar_init(empty0 + 8u * s, NW + 1);
        }
        for (int s = 0; s < NST1; ++s) {
            mbar_init(full1 + 8u * s, NW + 1);
            mbar_init(empty1 + 8u * s, NW);
        }
        fence_barrier_init();
        fence_proxy_async();
    }
    __syncthreads();

    const int nx = A.nx, ny = A.ny;
    const size_t plane = (size_t)nx * ny;

    // ------------------------------------------------------------------ TMA producer warp
    if (warp == 2 * NW + 1) {
        constexpr int NBOX = NG * 6 + 2 * kHalo2Arrays;
        constexpr uint32_t STAGE_TX = (uint32_t)(MAIN + 2 * kHalo2Arrays * RB * kHaloBytes);
        uint32_t gp = 0;
        for (long long item = blockIdx.x; item < A.nitems; item += gridDim.x) {
            const Stream2Item it = stream2_item<RB, NW * SW>(A, item);
            for (int q = 0; q < it.nstage; ++q, ++gp) {
                const uint32_t slot = gp % NST0;
                if (gp >= NST0) mbar_wait(empty0 + 8u * slot, ((gp / NST0) - 1u) & 1u);
                const uint32_t bar = full0 + 8u * slot;
                const uint32_t dst = ring0_u32 + slot * STAGE;
                const int y = it.j0 - 2 + q * RB;
                if (lane == 0) mbar_expect_tx(bar, STAGE_TX);
                __syncwarp();
                for (int bx = lane; bx < NBOX; bx += 32) {
                    const CUtensorMap* map;
                    uint32_t d;
                    int x, z;
                    if (bx < NG * 6) {
                        const int f = bx / NG, g = bx - NG * f;
                        map = f == 0 ? &A.mU : f == 1 ? &A.mV : f == 2 ? &A.mW : f == 3 ? &A.ma : f == 4 ? &A.mb : &A.mc;
                        d = dst + f * ARR + g * SLABG;
                        x = it.i0 + g * GW * SW;
                        z = f < 3 ? it.sim : 0;
                    } else {
                        const int hb = bx - NG * 6, side = hb / kHalo2Arrays, f = hb - kHalo2Arrays * side;
                        map = f == 0 ? &A.hU : f == 1 ? &A.hV : f == 2 ? &A.hW : f == 3 ? &A.ha : f == 4 ? &A.hb : &A.hc;
                        d = dst + MAIN + hb * kHaloSlab;
                        x = side == 0 ? it.i0 - C : it.i0 + NW * SW;
                        z = f < 3 ? it.sim : 0;
                    }
                    tma_load_3d(d, map, bar, x, y, z);
                }
            }
        }
        return;
    }

    // ------------------------------------------------------------------ lane maps
    // Main lanes (step-1 and step-2 warps): own 16-byte run of strip w; neighbours in the
    // adjacent lane / strip / halo slab.  Identical offsets in ring0 and ring1.
    auto main_map = [&](int w) {
        LaneMap L;
        const int grp = w / GW, wig = w % GW;
        L.oOff = grp * SLABG + wig * kStripBytes + 16 * lane; L.oSF = ARR; L.oSR = BOXB;
        if (lane > 0 || wig > 0) { L.wOff = L.oOff - (int)sizeof(T); L.wSF = ARR; L.wSR = BOXB; }
        else if (grp > 0) { L.wOff = (grp - 1) * SLABG + BOXB - (int)sizeof(T); L.wSF = ARR; L.wSR = BOXB; }
        else { L.wOff = MAIN + kHaloBytes - (int)sizeof(T); L.wSF = kHaloSlab; L.wSR = kHaloBytes; }
        if (lane < 31 || wig < GW - 1) { L.eOff = L.oOff + 16; L.eSF = ARR; L.eSR = BOXB; }
        else if (grp < NG - 1) { L.eOff = (grp + 1) * SLABG; L.eSF = ARR; L.eSR = BOXB; }
        else { L.eOff = MAIN + HSIDE; L.eSF = kHaloSlab; L.eSR = kHaloBytes; }
        return L;
    };

    // ------------------------------------------------------------------ halo warp (step 1 of the
    // two tile-edge columns): lane 0 = column x0-1, lane 1 = column x0+TW, one cell per row.
    if (warp == 2 * NW) {
        const int side = lane & 1;
        LaneMap L;
        if (side == 0) {
            L.oOff = MAIN + kHaloBytes - (int)sizeof(T); L.oSF = kHaloSlab; L.oSR = kHaloBytes;
            L.wOff = L.oOff - (int)sizeof(T); L.wSF = kHaloSlab; L.wSR = kHaloBytes;
            L.eOff = 0; L.eSF = ARR; L.eSR = BOXB;
        } else {
            L.oOff = MAIN + HSIDE; L.oSF = kHaloSlab; L.oSR = kHaloBytes;
            L.eOff = L.oOff + (int)sizeof(T); L.eSF = kHaloSlab; L.eSR = kHaloBytes;
            L.wOff = (NG - 1) * SLABG + BOXB - (int)sizeof(T); L.wSF = ARR; L.wSR = BOXB;
        }
        uint32_t g = 0;
        for (long long item = blockIdx.x; item < A.nitems; item += gridDim.x) {
            const Stream2Item it = stream2_item<RB, NW * SW>(A, item);
            const StepCoef<T> k = load_coef<T>(A.coefs + it.sim);
            MarchWindow<T, 1> win;
            win.clear();
            for (int q = 0; q < it.nstage; ++q, ++g) {
                const uint32_t s0 = g % NST0, s1 = g % NST1;
                mbar_wait(full0 + 8u * s0, (g / NST0) & 1u);
                if (g >= NST1) mbar_wait(empty1 + 8u * s1, ((g / NST1) - 1u) & 1u);
                const char* src = ring0 + (size_t)s0 * STAGE;
                char* dst = ring1 + (size_t)s1 * STAGE;
                const int jfirst = it.j0 - 2 + q * RB;
                const bool ghost = !(jfirst > 0 && jfirst + RB - 1 < ny);
#pragma unroll
                for (int rr = 0; rr < RB; ++rr) {
                    const int jn = jfirst + rr;
                    win.load(src, L, rr, false, false);
                    T oU[1], oV[1], oW[1];
                    if (ghost) win.template advance<true>(jn, ny, false, false, k, oU, oV, oW);
                    else win.template advance<false>(jn, ny, false, false, k, oU, oV, oW);
                    if (lane < 2) {
                        char* o = dst + L.oOff + rr * L.oSR;
                        *reinterpret_cast<T*>(o + 0 * kHaloSlab) = oU[0];
                        *reinterpret_cast<T*>(o + 1 * kHaloSlab) = oV[0];
                        *reinterpret_cast<T*>(o + 2 * kHaloSlab) = oW[0];
                        *reinterpret_cast<T*>(o + 3 * kHaloSlab) = win.centre_a()[0];
                        *reinterpret_cast<T*>(o + 4 * kHaloSlab) = win.centre_b()[0];
                        *reinterpret_cast<T*>(o + 5 * kHaloSlab) = win.centre_c()[0];
                    }
                    win.roll();
                }
                __syncwarp();
                if (lane == 0) {
                    mbar_arrive(empty0 + 8u * s0);
                    mbar_arrive(full1 + 8u * s1);
                }
            }
        }
        return;
    }

    // ------------------------------------------------------------------ step-1 warps
    if (warp < NW) {
        const LaneMap L = main_map(warp);
        uint32_t g = 0;
        for (long long item = blockIdx.x; item < A.nitems; item += gridDim.x) {
            const Stream2Item it = stream2_item<RB, NW * SW>(A, item);
            const int iown = it.i0 + warp * SW + lane * C;
            const bool atW = iown == 0, atE = iown + C == nx;
            const StepCoef<T> k = load_coef<T>(A.coefs + it.sim);
            MarchWindow<T, C> win;
            win.clear();
            for (int q = 0; q < it.nstage; ++q, ++g) {
                const uint32_t s0 = g % NST0, s1 = g % NST1;
                mbar_wait(full0 + 8u * s0, (g / NST0) & 1u);
                if (g >= NST1) mbar_wait(empty1 + 8u * s1, ((g / NST1) - 1u) & 1u);
                const char* src = ring0 + (size_t)s0 * STAGE;
                char* dst = ring1 + (size_t)s1 * STAGE + L.oOff;
                const int jfirst = it.j0 - 2 + q * RB;  // first time-k row arriving in this stage
                auto row_body = [&](auto ghost_c, const int rr) {
                    constexpr bool GHOST = decltype(ghost_c)::value;
                    win.load(src, L, rr, atW, atE);
                    T oU[C], oV[C], oW[C];
                    win.template advance<GHOST>(jfirst + rr, ny, atW, atE, k, oU, oV, oW);
                    char* o = dst + rr * BOXB;  // time-(k+1) row jfirst+rr-1 and its coefficients
                    st_run<T, C>(o + 0 * ARR, oU);
                    st_run<T, C>(o + 1 * ARR, oV);
                    st_run<T, C>(o + 2 * ARR, oW);
                    st_run<T, C>(o + 3 * ARR, win.centre_a());
                    st_run<T, C>(o + 4 * ARR, win.centre_b());
                    st_run<T, C>(o + 5 * ARR, win.centre_c());
                    win.roll();
                };
                if (jfirst > 0 && jfirst + RB - 1 < ny) {
#pragma unroll
                    for (int rr = 0; rr < RB; ++rr) row_body(std::false_type{}, rr);
                } else {
#pragma unroll
                    for (int rr = 0; rr < RB; ++rr) row_body(std::true_type{}, rr);
                }
                __syncwarp();
                if (lane == 0) {
                    mbar_arrive(empty0 + 8u * s0);  // ring0 stage is in registers
                    mbar_arrive(full1 + 8u * s1);   // ring1 stage written (release)
                }
            }
        }
        return;
    }

    // ------------------------------------------------------------------ step-2 warps
    {
        const int w = warp - NW;
        const LaneMap L = main_map(w);
        uint32_t g = 0;
        for (long long item = blockIdx.x; item < A.nitems; item += gridDim.x) {
            const Stream2Item it = stream2_item<RB, NW * SW>(A, item);
            const int iown = it.i0 + w * SW + lane * C;
            const bool valid = iown < nx;
            const bool atW = iown == 0, atE = iown + C == nx;
            const StepCoef<T> k = load_coef<T>(A.coefs + it.sim);
            T* gU = (T*)A.U1 + it.sim * plane + iown;
            T* gV = (T*)A.V1 + it.sim * plane + iown;
            T* gW = (T*)A.W1 + it.sim * plane + iown;
            MarchWindow<T, C> win;
            win.clear();
            for (int q = 0; q < it.nstage; ++q, ++g) {
                const uint32_t s1 = g % NST1;
                mbar_wait(full1 + 8u * s1, (g / NST1) & 1u);
                const char* src = ring1 + (size_t)s1 * STAGE;
                const int jfirst = it.j0 - 3 + q * RB;  // first time-(k+1) row arriving
                auto row_body = [&](auto ghost_c, const int rr) {
                    constexpr bool GHOST = decltype(ghost_c)::value;
                    const int m = q * RB + rr;
                    win.load(src, L, rr, atW, atE);
                    T oU[C], oV[C], oW[C];
                    win.template advance<GHOST>(jfirst + rr, ny, atW, atE, k, oU, oV, oW);
                    if (valid && m >= 4 && m < it.nr) {
                        const size_t off = (size_t)(jfirst + rr - 1) * nx;
                        st_run<T, C>((char*)(gU + off), oU);
                        st_run<T, C>((char*)(gV + off), oV);
                        st_run<T, C>((char*)(gW + off), oW);
                    }
                    win.roll();
                };
                if (jfirst > 0 && jfirst + RB - 1 < ny) {
#pragma unroll
                    for (int rr = 0; rr < RB; ++rr) row_body(std::false_type{}, rr);
                } else {
#pragma unroll
                    for (int rr = 0; rr < RB; ++rr) row_body(std::true_type{}, rr);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(empty1 + 8u * s1);
            }
        }
    }
}

}  // namespace gg

// gg_stream.cuh -- GG_KERNEL_STREAM: the fused single-step kernel for sm_100a.
//
// Design.  The step is HBM-bound (72 B and ~45 flops per cell in fp64), so
// the kernel is built around keeping many TMA loads in flight and touching every DRAM byte once:
//
//  * The grid is cut into TILE COLUMNS of NW adjacent STRIPS, each strip 512 bytes wide (64 fp64 /
//    128 fp32 cells), and into row CHUNKS.  One CTA of NW warps owns one (simulation, chunk, tile
//    column) item at a time; warp w owns strip w of the tile and marches up it row by row.
//  * Input rows travel through an NST-stage ring in shared memory, RB rows per stage.  Every warp
//    is the producer of its own strip: its lane 0 issues `cp.async.bulk.tensor` (TMA) loads of
//    exactly aligned RB x 512-byte boxes of the six input arrays (U, V, W, a, b, c) -- whole
//    32-byte sectors and 128-byte lines only, so nothing is fetched from L2/DRAM twice.  The one
//    column of halo each side of the TILE comes from two 16-byte-wide boxes per array; inside the
//    tile a strip's halo column is simply its neighbour warp's edge column in shared memory.
//    (A first version gave every warp its own 544-byte box with the halo inside: ncu showed
//    1.34x the compulsory DRAM reads, because TMA fetches whole 128-byte lines at both ragged
//    ends and independent warps drift too far apart for L2 to merge them.)
//    One `full` mbarrier per stage (NW producer arrivals + the bytes) and one `empty` mbarrier
//    (NW consumer arrivals); no __syncthreads anywhere.  Out-of-domain box parts are zero-filled.
//  * Every lane owns 16 bytes of each row (2 fp64 / 4 fp32 cells) and keeps a rolling window of
//    rows j-1, j, j+1 in REGISTERS, so each shared-memory element is read once per lane that needs
//    it.  The north face fluxes of row j are kept and reused as the south face fluxes of row j+1;
//    x-face fluxes inside a lane's run are computed once and used by both adjacent cells.  (The
//    run's west face is recomputed by the lane instead of shuffled from its neighbour: same cost
//    as the exchange plus its divergent edge case, and no cross-lane dependence.)
//  * Neumann boundaries (reading A2): faces on the domain boundary carry zero flux, tangential
//    differences use the mirrored neighbour.  Handled with warp-uniform row tests and two
//    per-lane flags; TMA's zero fill keeps every discarded value finite.
//  * Results leave as one 16-byte store per lane per field per row: 512 contiguous bytes per warp,
//    NW x 512 contiguous bytes per CTA row.
#pragma once
#include <cuda.h>

#include <type_traits>

#include "gg_common.cuh"
#include "gg_march.cuh"

namespace gg {

constexpr int kStripBytes = 512;   // 32 lanes x 16 B
constexpr int kHaloBytes = 16;     // inner extent of a tile-edge halo box (minimum TMA box width)
constexpr int kHaloSlab = 128;     // shared-memory bytes reserved per halo box (TMA dst alignment)

struct alignas(64) StreamArgs {
    // rank-3 tensor maps {nx, ny, B}: main boxes {512 B, RB, 1}; halo boxes {16 B, RB, 1}
    CUtensorMap mU, mV, mW, ma, mb, mc;
    CUtensorMap hU, hV, hW, ha, hb, hc;
    void* U1;                            // outputs [B][ny][nx]
    void* V1;
    void* W1;
    const StepCoef<double>* coefs;   // [B], folded on the device (gg_dt.cuh)
    int nx, ny, nbatch;
    int ntilecols, nchunks, chunk_rows;
    long long nitems;
};

// Host-side plan: tensor maps for both ping-pong copies and the launch geometry.
struct StreamPlan {
    CUtensorMap state[2][3], state_halo[2][3];
    CUtensorMap coef[3], coef_halo[3];
    int ntilecols = 0, nchunks = 0, chunk_rows = 0;
    long long nitems = 0;
    int grid = 0, block = 0;
    size_t smem = 0;
    int rb = 0, nst = 0, nst1 = 0, nw = 0;
    int steps = 1;  // time steps per launch
    const void* fn = nullptr;
};

__host__ __device__ constexpr int stream_stage_bytes(int rb, int nw) {
    return nw * 6 * rb * kStripBytes + 2 * 5 * kHaloSlab;
}
__host__ __device__ constexpr int stream_smem_bytes(int rb, int nst, int nw) {
    return 128 + nst * stream_stage_bytes(rb, nw);
}

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

__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// One work item of a CTA: simulation `sim`, tile column starting at cell i0, rows [j0, j1).
struct StreamItem {
    int sim, i0, j0, j1, nr, nstage;
};
template <int RB, int TILE_CELLS>
__device__ __forceinline__ StreamItem stream_item(const StreamArgs& A, long long item) {
    StreamItem it;
    const int tc = (int)(item % A.ntilecols);
    const long long t = item / A.ntilecols;
    const int chunk = (int)(t % A.nchunks);
    it.sim = (int)(t / A.nchunks);
    it.i0 = tc * TILE_CELLS;
    it.j0 = chunk * A.chunk_rows;
    it.j1 = min(it.j0 + A.chunk_rows, A.ny);
    it.nr = it.j1 - it.j0 + 2;  // input rows j0-1 .. j1 arrive
    it.nstage = (it.nr + RB - 1) / RB;
    return it;
}

// ------------------------------------------------------------------------------------------
// The kernel.  T: arithmetic/storage type; RB: rows per TMA box (= per ring stage); NST: ring
// stages; NW: warps (= strips) per CTA.  Dynamic shared memory:
//   [full[NST], empty[NST] mbarriers, 128 B][NST stages]; a stage is
//   [6 arrays][NG boxes][RB rows][GW strips x 512 B] followed by [west, east][5 arrays][128 B
//   halo slab]  (GW = strips per TMA box, NG = NW / GW).
// ------------------------------------------------------------------------------------------
template <typename T, int RB, int NST, int NW>
__global__ void __launch_bounds__((NW + 1) * 32, 1) gg_step_stream(const __grid_constant__ StreamArgs A) {
    constexpr int C = 16 / (int)sizeof(T);  // cells per lane per row
    constexpr int SW = 32 * C;              // strip width in cells
    // A TMA box may be 256 elements wide, so GW adjacent strips (4 in fp64, 2 in fp32) travel in
    // one box: fewer, larger TMA instructions for the producer warp.
    constexpr int GW = (256 / SW) < NW ? (256 / SW) : NW;  // strips per box
    constexpr int NG = NW / GW;                            // boxes (strip groups) per array
    constexpr int BOXB = GW * kStripBytes;                 // box row bytes = smem row pitch
    constexpr int SLABG = RB * BOXB;                       // one box
    constexpr int ARR = NG * SLABG;                        // one array of the whole tile
    constexpr int MAIN = 6 * ARR;
    static_assert(NW % GW == 0, "warps per CTA must be a multiple of the strips per box");
    constexpr int STAGE = stream_stage_bytes(RB, NW);
    static_assert(RB * kHaloBytes <= kHaloSlab, "halo slab too small");
    static_assert(2 * NST * 8 <= 128, "too many stages");

    extern __shared__ __align__(128) char smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t full0 = smem_u32(smem), empty0 = full0 + 8u * NST;
    char* ring = smem + 128;
    const uint32_t ring_u32 = smem_u32(ring);

    if (threadIdx.x == 0) {
        for (int s = 0; s < NST; ++s) {
            mbar_init(full0 + 8u * s, 1);    // the producer's arrive.expect_tx (+ the bytes)
            mbar_init(empty0 + 8u * s, NW);  // one arrival per consumer warp
        }
        fence_barrier_init();
        fence_proxy_async();
    }
    __syncthreads();  // once, before the pipeline starts

    // ---------------------------------------------------------------------------------------
    // Producer warp (warp NW): walks the same item / stage sequence as the consumers, waits for
    // a ring slot to be released by all NW consumer warps, then issues the stage's TMA boxes
    // (6 per strip + 5 per tile-edge halo), spread over its lanes.
    // ---------------------------------------------------------------------------------------
    if (warp == NW) {
        constexpr int NBOX = NG * 6 + 10;
        constexpr uint32_t STAGE_TX = (uint32_t)(MAIN + 10 * RB * kHaloBytes);
        uint32_t gp = 0;
        for (long long item = blockIdx.x; item < A.nitems; item += gridDim.x) {
            const StreamItem it = stream_item<RB, NW * SW>(A, item);
            for (int q = 0; q < it.nstage; ++q, ++gp) {
                const uint32_t slot = gp % NST;
                if (gp >= NST) mbar_wait(empty0 + 8u * slot, ((gp / NST) - 1u) & 1u);
                const uint32_t bar = full0 + 8u * slot;
                const uint32_t dst = ring_u32 + slot * STAGE;
                const int y = it.j0 - 1 + q * RB;
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
                        const int hb = bx - NG * 6, side = hb / 5, f = hb - 5 * side;
                        map = f == 0 ? &A.hU : f == 1 ? &A.hV : f == 2 ? &A.hW : f == 3 ? &A.ha : &A.hb;
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

    // per-lane byte offsets inside a stage: own run, west and east neighbour elements
    const int grp = warp / GW, wig = warp % GW;  // strip group (box) and strip within it
    LaneMap L;
    L.oOff = grp * SLABG + wig * kStripBytes + 16 * lane; L.oSF = ARR; L.oSR = BOXB;
    if (lane > 0 || wig > 0) { L.wOff = L.oOff - (int)sizeof(T); L.wSF = ARR; L.wSR = BOXB; }
    else if (grp > 0) { L.wOff = (grp - 1) * SLABG + BOXB - (int)sizeof(T); L.wSF = ARR; L.wSR = BOXB; }
    else { L.wOff = MAIN + kHaloBytes - (int)sizeof(T); L.wSF = kHaloSlab; L.wSR = kHaloBytes; }
    if (lane < 31 || wig < GW - 1) { L.eOff = L.oOff + 16; L.eSF = ARR; L.eSR = BOXB; }
    else if (grp < NG - 1) { L.eOff = (grp + 1) * SLABG; L.eSF = ARR; L.eSR = BOXB; }
    else { L.eOff = MAIN + 5 * kHaloSlab; L.eSF = kHaloSlab; L.eSR = kHaloBytes; }

    const int nx = A.nx, ny = A.ny;
    const size_t plane = (size_t)nx * ny;

    uint32_t gc = 0;  // global stages consumed (identical sequence in every warp of the CTA)
    for (long long item = blockIdx.x; item < A.nitems; item += gridDim.x) {
        const StreamItem it = stream_item<RB, NW * SW>(A, item);
        const int j0 = it.j0, nr = it.nr;
        const int iown = it.i0 + warp * SW + lane * C;  // first own cell
        const bool valid = iown < nx;                   // nx % C == 0: a run is all in or all out
        const bool atW = iown == 0, atE = iown + C == nx;
        const StepCoef<T> k = load_coef<T>(A.coefs + it.sim);
        T* gU = (T*)A.U1 + it.sim * plane + iown;
        T* gV = (T*)A.V1 + it.sim * plane + iown;
        T* gW = (T*)A.W1 + it.sim * plane + iown;

        MarchWindow<T, C> win;  // rolling register window (rows jc-1, jc, jc+1)
        win.clear();

        for (int q = 0; q < it.nstage; ++q, ++gc) {
            const uint32_t slot = gc % NST;
            mbar_wait(full0 + 8u * slot, (gc / NST) & 1u);
            const char* st = ring + (size_t)slot * STAGE;
            // Row body instantiated twice: GHOST = false for stages strictly inside the domain
            // (the hot path: no boundary code at all), GHOST = true for the few stages that
            // contain ghost row -1 or ny.  Arrival index n: arriving row jn = j0-1+n, centre row
            // jn-1.  Rows outside [j0, j1) are computed but never stored; the ring always holds
            // finite data (real rows or TMA zero fill).
            auto row_body = [&](auto ghost_c, const int rr) {
                constexpr bool GHOST = decltype(ghost_c)::value;
                const int n = q * RB + rr;
                const int jn = j0 - 1 + n;
                win.load(st, L, rr, atW, atE);
                T oU[C], oV[C], oW[C];
                win.template advance<GHOST>(jn, ny, atW, atE, k, oU, oV, oW);
                if (valid && n >= 2 && n < nr) {
                    const size_t off = (size_t)(jn - 1) * nx;
                    st_run<T, C>((char*)(gU + off), oU);
                    st_run<T, C>((char*)(gV + off), oV);
                    st_run<T, C>((char*)(gW + off), oW);
                }
                win.roll();
            };
            const int jfirst = j0 - 1 + q * RB;  // first row arriving in this stage
            if (jfirst > 0 && jfirst + RB - 1 < ny) {
#pragma unroll
                for (int rr = 0; rr < RB; ++rr) row_body(std::false_type{}, rr);
            } else {
#pragma unroll
                for (int rr = 0; rr < RB; ++rr) row_body(std::true_type{}, rr);
            }
            // every lane of this warp has the stage in registers: release it
            __syncwarp();
            if (lane == 0) mbar_arrive(empty0 + 8u * slot);
        }
    }
}

}  // namespace gg

// gg_pair.cuh -- GG_KERNEL_PAIR: two time steps per launch, chained in REGISTERS.
//
// ncu on the shared-memory chained two-step kernel (gg_stream2.cuh) shows the shared-memory data
// pipe as its nearest ceiling (73 % of peak wavefronts: every time level is written to and read
// back from a ring, and every x-neighbour is an 8-byte load at a 16-byte lane stride).  This
// kernel keeps the intermediate time level in registers and exchanges x-neighbours by warp
// shuffle, so shared memory is touched once per input element:
//
//  * A lane owns a run of C cells (16 bytes) of a row and marches up the grid.  On every arriving
//    time-k row it advances row j-1 to time k+1 (level 1) and, from that result, row j-2 to time
//    k+2 (level 2); both levels keep their rolling window (rows j-1, j of W; row j of U, V, a, b,
//    c, H; the south face fluxes) in registers.
//  * x-neighbours: the face between the runs of lanes l-1 and l is computed ONCE, by lane l, from
//    lane l-1's edge values (M = 1-U, V, G: warp shuffles; W: the H shuffle of one row earlier; the
//    face's coefficient is the lane's own stored face sum) and handed back to lane l-1 by shuffle;
//    the W neighbours of the tangential difference H come by shuffle too.  Seven shuffled values
//    per level and row; no neighbour loads.
//  * A warp therefore loads a 32-lane strip and, after two levels, lanes 1..30 hold valid time-k+2
//    cells (the edge lanes lack a neighbour): strips overlap by two lanes, a warp stores 30 x 16 B
//    = 480 contiguous bytes per row and field.  The NW strips of a CTA tile arrive in ring stages
//    of RB rows, filled by TMA boxes of GW strips (+ the overlap) per array.  There is no
//    producer warp (a ninth warp would cap every warp at 168 registers): the warp that releases
//    a ring slot last issues its refill.  `full` mbarriers, per-slot release counters; no
//    __syncthreads after start-up.
//  * Arithmetic: the same flux_V / flux_W / cross / upd_* calls with the same operand order as
//    every other kernel => bit-identical results (gg_common.cuh).
//  * Neumann faces as in gg_march.cuh: per-lane atW/atE flags zero the boundary face flux and
//    mirror W's neighbour; the GHOST instantiation mirrors rows -1 and ny.
#pragma once
#include "gg_stream.cuh"

namespace gg {

constexpr int kPairLanes = 30;  // lanes of a warp that hold valid cells after two levels

// fp32: arithmetic on packed pairs of cells (FADD2 / FMUL2 / FFMA2), bit-identical to the scalar code
#ifndef GG_PACKED_F32
#define GG_PACKED_F32 1
#endif
constexpr bool kPackedF32 = GG_PACKED_F32 != 0;


struct alignas(64) PairArgs {
    CUtensorMap mU, mV, mW, ma, mb, mc;  // rank-3 maps {nx, ny, B}, box {GW*30*C + 2C, RB, 1}
    void* U1;
    void* V1;
    void* W1;
    const StepCoef<double>* coefs;   // [B], folded on the device (gg_dt.cuh)
    int nx, ny, nbatch;
    int nw;                               // strips (compute warps) per CTA
    int ntilecols, nchunks, chunk_rows;
    long long nitems;
};

template <typename T> __host__ __device__ constexpr int pair_gw() { return sizeof(T) == 8 ? 4 : 2; }
// bytes of one box row: GW strips of 30 lanes plus one lane of overlap on each side
template <typename T> __host__ __device__ constexpr int pair_box_bytes() {
    return pair_gw<T>() * kPairLanes * 16 + 32;
}
__host__ __device__ constexpr int pair_slab_bytes(int rb, int box_bytes) {
    return (rb * box_bytes + 127) / 128 * 128;
}
template <typename T> __host__ __device__ constexpr int pair_stage_bytes(int rb, int nw) {
    return 6 * ((nw + pair_gw<T>() - 1) / pair_gw<T>()) * pair_slab_bytes(rb, pair_box_bytes<T>());
}

template <typename T>
__device__ __forceinline__ T shfl_up1(T x) { return __shfl_up_sync(0xffffffffu, x, 1); }
template <typename T>
__device__ __forceinline__ T shfl_down1(T x) { return __shfl_down_sync(0xffffffffu, x, 1); }

// One time level of the in-register march: window of the centre row (and W one row below).
// aC holds the west-face sums aw of the centre row, cN (an argument) the south-face sums cs of the
// arriving row (gg_common.cuh); cC is carried only to hand the centre row's cs on to the next level.
template <typename T, int C>
struct PairLevel {
    T wP[C], wC[C], uC[C], mC[C], vC[C], aC[C], bC[C], cC[C], hC[C], sV[C], sW[C];
    T wWC;   // W of the centre row's west neighbour cell (the shuffled wNw of one row earlier)

    __device__ __forceinline__ void clear() {
#pragma unroll
        for (int c = 0; c < C; ++c)
            wP[c] = wC[c] = uC[c] = mC[c] = vC[c] = aC[c] = bC[c] = cC[c] = hC[c] = sV[c] = sW[c] = (T)0;
        wWC = (T)0;
    }

    // Row `jn` arrives (own cells uN..cN); the centre row jn-1 is advanced one step into
    // oU, oV, oW and its coefficients are copied to oa, ob, oc; then the window rolls.
    // atW / atE: the run touches the domain's west / east face (mirrored W neighbour in H);
    // edge0: the run's face 0 lies ON a domain face (iown == 0 or iown == nx: the first run
    // outside the east face computes, and zeroes, the east boundary face of its west neighbour).
    // All 32 lanes must call this together (warp shuffles).
    template <bool GHOST>
    __device__ __forceinline__ void advance(int jn, int ny, bool atW, bool atE, bool edge0, const StepCoef<T>& k,
                                            T* uN, T* vN, T* wN, const T* aN, const T* bN, const T* cN,
                                            T* oU, T* oV, T* oW, T* oa, T* ob, T* oc) {
        if constexpr (kPackedF32 && sizeof(T) == 4 && C == 4) {
            advance_packed<GHOST>(jn, ny, atW, atE, edge0, k, uN, vN, wN, aN, bN, cN, oU, oV, oW, oa, ob, oc);
            return;
        }
        // cross term H of the arriving row: tangential (x) difference with the lanes' neighbours
        T wNw = shfl_up1(wN[C - 1]), wNe = shfl_down1(wN[0]);
        if (atW) wNw = wN[0];
        if (atE) wNe = wN[C - 1];
        T hN[C], mN[C];
#pragma unroll
        for (int c = 0; c < C; ++c) {
            hN[c] = cross(bN[c], c == C - 1 ? wNe : wN[c + 1 < C ? c + 1 : c], c == 0 ? wNw : wN[c > 0 ? c - 1 : 0]);
            mN[c] = one_minus(uN[c]);
        }
        if constexpr (GHOST) {
            if (jn == 0) {       // centre is ghost row -1: even mirror of row 0, H odd
#pragma unroll
                for (int c = 0; c < C; ++c) { uC[c] = uN[c]; mC[c] = mN[c]; vC[c] = vN[c]; wC[c] = wN[c]; hC[c] = -hN[c]; }
                wWC = wNw;
            }
            if (jn == ny) {      // arriving row is ghost row ny: mirror of row ny-1
#pragma unroll
                for (int c = 0; c < C; ++c) { uN[c] = uC[c]; mN[c] = mC[c]; vN[c] = vC[c]; wN[c] = wC[c]; hN[c] = -hC[c]; }
                wNw = wWC;
            }
        }
        if constexpr (sizeof(T) == 8) {
            // fp64: M of the centre row is re-formed here instead of living in the window across rows:
            // one operation more per cell, 8 registers less for a kernel that sits at the register
            // cap (fewer moves and register swaps: 223 -> 228 GLUPS at 8192^2)
#pragma unroll
            for (int c = 0; c < C; ++c) mC[c] = one_minus(uC[c]);
        }
        T G[C];
#pragma unroll
        for (int c = 0; c < C; ++c) G[c] = cross(bC[c], wN[c], wP[c]);
        // x faces 0..C of the run: face 0 (shared with lane-1) is computed here from that lane's
        // edge values, face C is lane+1's face 0
        T pV[C + 1], pW[C + 1];
        {
            const T mW = shfl_up1(mC[C - 1]), vW = shfl_up1(vC[C - 1]), GW = shfl_up1(G[C - 1]);
            pV[0] = flux_V(mW, mC[0], vW, vC[0]);
            pW[0] = flux_W(aC[0], wWC, wC[0], GW, G[0]);
        }
        if (edge0) { pV[0] = (T)0; pW[0] = (T)0; }
#pragma unroll
        for (int f = 1; f < C; ++f) {
            pV[f] = flux_V(mC[f - 1], mC[f], vC[f - 1], vC[f]);
            pW[f] = flux_W(aC[f], wC[f - 1], wC[f], G[f - 1], G[f]);
        }
        pV[C] = shfl_down1(pV[0]);
        pW[C] = shfl_down1(pW[0]);
        T nV[C], nW[C];
#pragma unroll
        for (int c = 0; c < C; ++c) {
            nV[c] = flux_V(mC[c], mN[c], vC[c], vN[c]);
            nW[c] = flux_W(cN[c], wC[c], wN[c], hC[c], hN[c]);
        }
#pragma unroll
        for (int c = 0; c < C; ++c) {
            oU[c] = upd_U(k, uC[c], mC[c], wC[c]);
            oV[c] = upd_V(k, vC[c], pV[c + 1], pV[c], nV[c], sV[c]);
            oW[c] = upd_W(k, vC[c], wC[c], pW[c + 1], pW[c], nW[c], sW[c]);
            oa[c] = aC[c]; ob[c] = bC[c]; oc[c] = cC[c];
        }
#pragma unroll
        for (int c = 0; c < C; ++c) {  // roll
            wP[c] = wC[c]; wC[c] = wN[c]; uC[c] = uN[c]; mC[c] = mN[c]; vC[c] = vN[c];
            aC[c] = aN[c]; bC[c] = bN[c]; cC[c] = cN[c]; hC[c] = hN[c]; sV[c] = nV[c]; sW[c] = nW[c];
        }
        wWC = wNw;
    }

    // fp32, four cells per lane: the same operations on PACKED pairs of cells (Blackwell's FADD2 /
    // FMUL2 / FFMA2: two fp32 operations per instruction and issue slot).  Everything whose operands
    // are aligned per cell -- M, G, H's product, the y faces, the three updates, the face products --
    // runs on the pairs (cells 0,1) and (2,3); the differences and sums of x-NEIGHBOURS (shifted by
    // one cell) stay scalar and write straight into pair halves.  Each component is rounded exactly
    // as in the scalar code (a - b = fma(b, -1, a)), so the results are bit-identical to it.
    template <bool GHOST>
    __device__ __forceinline__ void advance_packed(int jn, int ny, bool atW, bool atE, bool edge0, const StepCoef<T>& k,
                                                   T* uN, T* vN, T* wN, const T* aN, const T* bN, const T* cN,
                                                   T* oU, T* oV, T* oW, T* oa, T* ob, T* oc) {
        auto P = [](const T* x, int p) { return make_float2((float)x[2 * p], (float)x[2 * p + 1]); };
        auto S = [](T* x, int p, float2 v) { x[2 * p] = (T)v.x; x[2 * p + 1] = (T)v.y; };
        auto sub2 = [](float2 a, float2 b) { return __ffma2_rn(b, make_float2(-1.f, -1.f), a); };
        auto rep = [](T x) { return make_float2((float)x, (float)x); };
        T wNw = shfl_up1(wN[3]), wNe = shfl_down1(wN[0]);
        if (atW) wNw = wN[0];
        if (atE) wNe = wN[3];
        T hN[4], mN[4], dh[4];
        dh[0] = sub(wN[1], wNw); dh[1] = sub(wN[2], wN[0]); dh[2] = sub(wN[3], wN[1]); dh[3] = sub(wNe, wN[2]);
#pragma unroll
        for (int p = 0; p < 2; ++p) {
            S(hN, p, __fmul2_rn(P(bN, p), P(dh, p)));
            S(mN, p, __ffma2_rn(P(uN, p), make_float2(-1.f, -1.f), make_float2(1.f, 1.f)));
        }
        if constexpr (GHOST) {
            if (jn == 0) {
#pragma unroll
                for (int c = 0; c < 4; ++c) { uC[c] = uN[c]; mC[c] = mN[c]; vC[c] = vN[c]; wC[c] = wN[c]; hC[c] = -hN[c]; }
                wWC = wNw;
            }
            if (jn == ny) {
#pragma unroll
                for (int c = 0; c < 4; ++c) { uN[c] = uC[c]; mN[c] = mC[c]; vN[c] = vC[c]; wN[c] = wC[c]; hN[c] = -hC[c]; }
                wNw = wWC;
            }
        }
        T G[4];
#pragma unroll
        for (int p = 0; p < 2; ++p) S(G, p, __fmul2_rn(P(bC, p), sub2(P(wN, p), P(wP, p))));
        // x faces 0..3: sums and differences of x-neighbours (scalar), then the products (packed)
        const T mW = shfl_up1(mC[3]), vW = shfl_up1(vC[3]), GW = shfl_up1(G[3]);
        T sm[4], dv[4], dw[4], sg[4], pV[5], pW[5];
        sm[0] = add(mW, mC[0]); dv[0] = sub(vC[0], vW); dw[0] = sub(wC[0], wWC); sg[0] = add(GW, G[0]);
#pragma unroll
        for (int f = 1; f < 4; ++f) {
            sm[f] = add(mC[f - 1], mC[f]); dv[f] = sub(vC[f], vC[f - 1]);
            dw[f] = sub(wC[f], wC[f - 1]); sg[f] = add(G[f - 1], G[f]);
        }
#pragma unroll
        for (int p = 0; p < 2; ++p) {
            S(pV, p, __fmul2_rn(P(sm, p), P(dv, p)));
            S(pW, p, __ffma2_rn(P(aC, p), P(dw, p), P(sg, p)));
        }
        if (edge0) { pV[0] = (T)0; pW[0] = (T)0; }
        pV[4] = shfl_down1(pV[0]);
        pW[4] = shfl_down1(pW[0]);
        T dpv[4], dpw[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) { dpv[c] = sub(pV[c + 1], pV[c]); dpw[c] = sub(pW[c + 1], pW[c]); }
        const float2 kdt = rep(k.dt), knd = rep(-k.ddt), krd = rep(k.rdt), kax = rep(k.adx), kay = rep(k.ady),
                     kcr = rep(k.crdt), ksw = rep(k.sw);
        T nV[4], nW[4];
#pragma unroll
        for (int p = 0; p < 2; ++p) {
            const float2 u = P(uC, p), m = P(mC, p), v = P(vC, p), w = P(wC, p);
            // north faces
            const float2 nv = __fmul2_rn(__fadd2_rn(m, P(mN, p)), sub2(P(vN, p), v));
            const float2 nw = __ffma2_rn(P(cN, p), sub2(P(wN, p), w), __fadd2_rn(P(hC, p), P(hN, p)));
            S(nV, p, nv);
            S(nW, p, nw);
            // eq. (3): same nesting as upd_U / upd_V / upd_W
            S(oU, p, __ffma2_rn(u, __ffma2_rn(kdt, m, __fmul2_rn(knd, w)), u));
            const float2 rv = __ffma2_rn(__fmul2_rn(krd, v), __ffma2_rn(v, make_float2(-1.f, -1.f), make_float2(1.f, 1.f)), v);
            S(oV, p, __ffma2_rn(kax, P(dpv, p), __ffma2_rn(kay, sub2(nv, P(sV, p)), rv)));
            const float2 rw = __ffma2_rn(kcr, sub2(v, w), w);
            S(oW, p, __ffma2_rn(ksw, P(dpw, p), __ffma2_rn(ksw, sub2(nw, P(sW, p)), rw)));
        }
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            oa[c] = aC[c]; ob[c] = bC[c]; oc[c] = cC[c];
            wP[c] = wC[c]; wC[c] = wN[c]; uC[c] = uN[c]; mC[c] = mN[c]; vC[c] = vN[c];
            aC[c] = aN[c]; bC[c] = bN[c]; cC[c] = cN[c]; hC[c] = hN[c]; sV[c] = nV[c]; sW[c] = nW[c];
        }
        wWC = wNw;
    }
};

struct PairItem {
    int sim, i0, j0, j1, nr, nstage;
};
template <int RB>
__device__ __forceinline__ PairItem pair_item(const PairArgs& A, long long item, int tile_cells) {
    PairItem it;
    const int tc = (int)(item % A.ntilecols);
    const long long t = item / A.ntilecols;
    const int chunk = (int)(t % A.nchunks);
    it.sim = (int)(t / A.nchunks);
    it.i0 = tc * tile_cells;
    it.j0 = chunk * A.chunk_rows;
    it.j1 = min(it.j0 + A.chunk_rows, A.ny);
    it.nr = it.j1 - it.j0 + 4;  // time-k rows j0-2 .. j1+1 arrive
    it.nstage = (it.nr + RB - 1) / RB;
    return it;
}

// Producer cursor: the (item, stage) the NEXT refill of a ring slot will load.  Every warp keeps
// its own copy and advances it once per consumed stage, so whichever warp happens to release a
// slot last can issue the refill without talking to anybody.
struct PairCursor {
    long long item;
    int q;
    PairItem it;
};

// T: arithmetic/storage type; RB: rows per ring stage; NST: ring stages.  blockDim = nw*32: every
// warp computes (eight warps leave each of them 255 registers; a ninth, producer-only warp would
// cap all of them at 168 and spill the two windows).  A ring slot is refilled by the warp that
// releases it LAST (shared-memory counter per slot): lanes of that warp issue the TMA boxes.
// Dynamic shared memory: [full[NST] mbarriers, count[NST], 128 B][NST stages]; a stage is
// [6 arrays][NG boxes][RB rows][box bytes] with every box slab padded to 128 bytes.
template <typename T, int RB, int NST>
__global__ void __launch_bounds__(256, 1) gg_step_pair(const __grid_constant__ PairArgs A) {
    constexpr int C = 16 / (int)sizeof(T);
    constexpr int GW = pair_gw<T>();
    constexpr int VW = kPairLanes * C;            // valid cells per strip
    constexpr int BOXB = pair_box_bytes<T>();
    constexpr int SLAB = pair_slab_bytes(RB, BOXB);
    static_assert(NST * 12 <= 128, "too many stages");

    extern __shared__ __align__(128) char smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nw = A.nw, ng = (nw + GW - 1) / GW;
    const int ARR = ng * SLAB, STAGE = 6 * ARR;
    const uint32_t full0 = smem_u32(smem);
    unsigned int* count = reinterpret_cast<unsigned int*>(smem + 8 * NST);
    char* ring = smem + 128;
    const uint32_t ring_u32 = smem_u32(ring);
    const int nx = A.nx, ny = A.ny;
    const int tile_cells = VW * nw;
    const int nbox = 6 * ng;
    const uint32_t stage_tx = (uint32_t)(nbox * RB * BOXB);

    // issue the TMA boxes of the cursor's stage into ring slot `slot` (whole warp)
    auto issue = [&](const PairCursor& pc, uint32_t slot) {
        const uint32_t bar = full0 + 8u * slot;
        const uint32_t dst = ring_u32 + slot * STAGE;
        const int y = pc.it.j0 - 2 + pc.q * RB;
        if (lane == 0) mbar_expect_tx(bar, stage_tx);
        __syncwarp();
        for (int bx = lane; bx < nbox; bx += 32) {
            const int f = bx / ng, g = bx - ng * f;
            const CUtensorMap* map = f == 0 ? &A.mU : f == 1 ? &A.mV : f == 2 ? &A.mW
                                   : f == 3 ? &A.ma : f == 4 ? &A.mb : &A.mc;
            tma_load_3d(dst + f * ARR + g * SLAB, map, bar, pc.it.i0 - C + g * GW * VW, y,
                        f < 3 ? pc.it.sim : 0);
        }
    };
    auto advance_cursor = [&](PairCursor& pc) {
        if (pc.item >= A.nitems) return;
        if (++pc.q == pc.it.nstage) {
            pc.q = 0;
            pc.item += gridDim.x;
            if (pc.item < A.nitems) pc.it = pair_item<RB>(A, pc.item, tile_cells);
        }
    };

    if (threadIdx.x == 0) {
        for (int s = 0; s < NST; ++s) {
            mbar_init(full0 + 8u * s, 1);
            count[s] = 0u;
        }
        fence_barrier_init();
        fence_proxy_async();
    }
    __syncthreads();

    PairCursor pc;
    pc.item = blockIdx.x;
    pc.q = 0;
    if (pc.item < A.nitems) pc.it = pair_item<RB>(A, pc.item, tile_cells);
    // prologue: warp 0 fills the ring; every warp moves its cursor past those NST stages
    for (int s = 0; s < NST; ++s) {
        if (warp == 0 && pc.item < A.nitems) issue(pc, (uint32_t)s);
        advance_cursor(pc);
    }

    const int grp = warp / GW, wig = warp % GW;
    const int own_off = grp * SLAB + wig * (VW * (int)sizeof(T)) + 16 * lane;
    const size_t plane = (size_t)nx * ny;
    const bool lane_ok = lane >= 1 && lane <= kPairLanes;

    uint32_t gc = 0;
    for (long long item = blockIdx.x; item < A.nitems; item += gridDim.x) {
        const PairItem it = pair_item<RB>(A, item, tile_cells);
        const int iown = it.i0 + warp * VW + (lane - 1) * C;  // first own cell (lane 0: halo, may be < 0)
        const bool store_ok = lane_ok && iown < nx;
        const bool atW = iown == 0, atE = iown + C == nx, edge0 = atW || iown == nx;
        const StepCoef<T> k = load_coef<T>(A.coefs + it.sim);
        T* gU = (T*)A.U1 + it.sim * plane + iown;
        T* gV = (T*)A.V1 + it.sim * plane + iown;
        T* gW = (T*)A.W1 + it.sim * plane + iown;

        PairLevel<T, C> L1, L2;
        L1.clear();
        L2.clear();

        for (int q = 0; q < it.nstage; ++q, ++gc) {
            const uint32_t slot = gc % NST;
            mbar_wait(full0 + 8u * slot, (gc / NST) & 1u);
            const char* st = ring + (size_t)slot * STAGE + own_off;
            const int jfirst = it.j0 - 2 + q * RB;  // first time-k row arriving in this stage
            auto row_body = [&](auto ghost_c, const int rr) {
                constexpr bool GHOST = decltype(ghost_c)::value;
                const int jn = jfirst + rr;
                const char* p = st + rr * BOXB;
                T uN[C], vN[C], wN[C], aN[C], bN[C], cN[C];
                ld_run<T, C>(p + 0 * ARR, uN);
                ld_run<T, C>(p + 1 * ARR, vN);
                ld_run<T, C>(p + 2 * ARR, wN);
                ld_run<T, C>(p + 3 * ARR, aN);
                ld_run<T, C>(p + 4 * ARR, bN);
                ld_run<T, C>(p + 5 * ARR, cN);
                T u1[C], v1[C], w1[C], a1[C], b1[C], c1[C];   // row jn-1 at time k+1
                L1.template advance<GHOST>(jn, ny, atW, atE, edge0, k, uN, vN, wN, aN, bN, cN, u1, v1, w1, a1, b1, c1);
                T u2[C], v2[C], w2[C], a2[C], b2[C], c2[C];   // row jn-2 at time k+2
                L2.template advance<GHOST>(jn - 1, ny, atW, atE, edge0, k, u1, v1, w1, a1, b1, c1, u2, v2, w2, a2, b2, c2);
                const int r = jn - 2;
                if (store_ok && r >= it.j0 && r < it.j1) {
                    const size_t off = (size_t)r * nx;
                    st_run<T, C>((char*)(gU + off), u2);
                    st_run<T, C>((char*)(gV + off), v2);
                    st_run<T, C>((char*)(gW + off), w2);
                }
            };
            if (jfirst >= 2 && jfirst + RB - 1 < ny) {
                // fp32's row body is twice as long per lane (4 cells): unrolling two rows keeps
                // the hot loop inside the instruction cache (+2 % at 8192^2); fp64 wants all RB
                constexpr int UNR = sizeof(T) == 4 && RB % 2 == 0 ? 2 : RB;
#pragma unroll UNR
                for (int rr = 0; rr < RB; ++rr) row_body(std::false_type{}, rr);
            } else {
#pragma unroll
                for (int rr = 0; rr < RB; ++rr) row_body(std::true_type{}, rr);
            }
            // Release the slot: every lane has the stage in registers.  The warp that releases it
            // last refills it with the stage NST ahead (the cursor), if there is one.
            __syncwarp();
            unsigned int prev = 0;
            if (lane == 0) {
                __threadfence_block();
                prev = atomicAdd(&count[slot], 1u);
            }
            prev = __shfl_sync(0xffffffffu, prev, 0);
            if (prev == (unsigned)nw - 1u) {
                if (lane == 0) { count[slot] = 0u; __threadfence_block(); }
                if (pc.item < A.nitems) issue(pc, slot);
            }
            advance_cursor(pc);
        }
    }
}

}  // namespace gg

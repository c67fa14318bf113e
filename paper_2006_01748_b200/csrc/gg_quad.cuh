// gg_quad.cuh -- GG_KERNEL_QUAD: FOUR time steps per launch.
//
// The register-chained pair kernel (gg_pair.cuh) runs at the HBM rate with the SM ~45 % busy
// (profiles/r01_ncu_full_pair_f64.txt), so the remaining headroom is again in crossing HBM less
// often.  Two pair marches are chained through one shared-memory ring:
//
//   TMA --ring0: U,V,W,a,b,c at time k--> 4 "A" warps: k -> k+1 -> k+2 in registers
//       --ring1: U,V,W at time k+2 (+ the rows' a,b,c)--> 4 "B" warps: k+2 -> k+3 -> k+4 --> HBM
//
//  * Geometry in units of lane runs (one run = C cells = 16 bytes).  A pair march loses one lane
//    on each side of a warp, and a lane's result depends on its own and its two neighbours'
//    inputs only.  A warp w lane l owns run 30w-2+l of the tile and leaves 120 valid time-k+2
//    runs [-1, 119) in ring1; B warp w lane l owns run 30w-1+l; the tile's time-k+4 output is
//    runs [0, 118): 118 x 16 B = 1888 contiguous bytes per row and field.  Work per output
//    cell-step: 8 x 32 lanes x 2 levels / (118 x 4) = 1.085 lane-rows (1.067 in the pair kernel).
//  * ring0 is the pair kernel's ring for four warps (TMA boxes of GW strips + overlap); a slot is
//    refilled by the A warp that releases it last.  ring1 rows are contiguous (123 runs).  A
//    writes lanes 1..30; B's outermost lanes read two runs nobody writes (zeroed at start-up) and
//    produce nothing that is kept.  mbarriers: full0 (TMA bytes), full1 (4 A warps), empty1 (4 B
//    warps); no __syncthreads after start-up.
//  * Rows: a chunk [j0, j1) loads rows j0-4 .. j1+3; A emits time-k+2 rows j0-2 .. j1+1; B stores
//    time-k+4 rows j0 .. j1-1.
//  * Both roles run the SAME row body (PairLevel twice); they differ in where a row comes from and
//    where the result goes.  Arithmetic and operand order are every other kernel's => bit-identical.
//  * "C" builds (NSTC > 0, the fp64 default): the coefficient rows a, b, c do not change in time,
//    so the B warps need not receive them from the A warps: their last-releasing warp fetches the
//    B rows' own coefficient boxes by TMA (L2-hot: the A warps' TMA just read them) into a third
//    ring.  ring1 then carries U, V, W only and the A warps shed three of their six shared-memory
//    stores per row.
#pragma once
#include "gg_pair.cuh"

namespace gg {

// NWR = warps per role (A and B): 4 (one 8-warp CTA per SM) or 2 (two 4-warp CTAs per SM: the same
// eight warps, registers and shared memory per SM).  The narrower tile fits grid widths that
// 236-cell tiles pad badly (1024 fp64 cells = 4.34 tiles of 4 warps but 8.83 tiles of 2) at the
// price of a little more overlap (116 output cells per 128 lanes instead of 236 per 256).
__host__ __device__ constexpr int quad_runs(int nwr) { return 30 * nwr - 2; }        // output runs per tile row
__host__ __device__ constexpr int quad_ring1_runs(int nwr) { return 30 * nwr + 3; }  // runs per ring1 row (run -2 ..)
template <typename T> __host__ __device__ constexpr int quad_gw(int nwr) { return nwr < pair_gw<T>() ? nwr : pair_gw<T>(); }
// bytes of one TMA box row: up to GW strips of 30 runs plus one run of overlap on each side
template <typename T> __host__ __device__ constexpr int quad_box_bytes(int nwr) { return quad_gw<T>(nwr) * kPairLanes * 16 + 32; }
template <typename T> __host__ __device__ constexpr int quad_ng(int nwr) { return (nwr + quad_gw<T>(nwr) - 1) / quad_gw<T>(nwr); }
template <typename T> __host__ __device__ constexpr int quad_ring0_stage(int rb, int nwr) {
    return 6 * quad_ng<T>(nwr) * pair_slab_bytes(rb, quad_box_bytes<T>(nwr));
}
__host__ __device__ constexpr int quad_ring1_stage(int rb, int nwr) { return 6 * rb * quad_ring1_runs(nwr) * 16; }
// nstc == 0: ring1 carries U, V, W and the rows' a, b, c.  nstc > 0 (the "C" builds, fp64): the
// B warps fetch their own coefficient rows by TMA into a third ring of nstc stages and ring1
// carries U, V, W only.
template <typename T> __host__ __device__ constexpr int quad_smem_bytes(int rb, int nst0, int nst1, int nstc, int nwr) {
    return 256 + nst0 * quad_ring0_stage<T>(rb, nwr) +
           (nstc > 0 ? nst1 * (quad_ring1_stage(rb, nwr) / 2) + nstc * (quad_ring0_stage<T>(rb, nwr) / 2)
                     : nst1 * quad_ring1_stage(rb, nwr));
}

template <int RB>
__device__ __forceinline__ PairItem quad_item(const PairArgs& A, long long item, int tile_cells) {
    PairItem it = pair_item<RB>(A, item, tile_cells);
    it.nr = it.j1 - it.j0 + 8;  // time-k rows j0-4 .. j1+3 arrive
    it.nstage = (it.nr + RB - 1) / RB;
    return it;
}

// blockDim = 64 NWR: warps 0..NWR-1 = A, NWR..2NWR-1 = B.  Dynamic shared memory:
// [full0[NST0], full1[NST1], empty1[NST1], fullC[NSTC] mbarriers, count0[NST0], countC[NSTC];
//  256 B][ring0: 6 arrays][ringC: a,b,c for the B warps (NSTC > 0)][ring1: U,V,W (+ a,b,c if NSTC == 0)].
template <typename T, int RB, int NST0, int NST1, int NSTC, int NWR>
__global__ void __launch_bounds__(64 * NWR, NWR == 4 ? 1 : 2) gg_step_quad(const __grid_constant__ PairArgs A) {
    constexpr int C = 16 / (int)sizeof(T);
    constexpr int GW = quad_gw<T>(NWR);
    constexpr int NG = quad_ng<T>(NWR);
    constexpr int VW = kPairLanes * C;
    constexpr int BOXB = quad_box_bytes<T>(NWR);
    constexpr int SLAB = pair_slab_bytes(RB, BOXB);
    constexpr int ARR0 = NG * SLAB, STAGE0 = 6 * ARR0;
    constexpr bool CB = NSTC > 0;                       // B warps own a coefficient ring
    constexpr int NF1 = CB ? 3 : 6;                     // arrays travelling through ring1
    constexpr int P1 = quad_ring1_runs(NWR) * 16, ARR1 = RB * P1, STAGE1 = NF1 * ARR1;
    constexpr int STAGEC = 3 * ARR0;
    constexpr int NTHR = 64 * NWR;
    static_assert(STAGE0 == quad_ring0_stage<T>(RB, NWR), "layout");
    static_assert((NST0 + 2 * NST1 + NSTC) * 8 + (NST0 + NSTC) * 4 <= 256, "too many stages");

    extern __shared__ __align__(128) char smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const bool isA = warp < NWR;
    const int w = isA ? warp : warp - NWR;
    const uint32_t full0 = smem_u32(smem), full1 = full0 + 8u * NST0, empty1 = full1 + 8u * NST1;
    const uint32_t fullC = empty1 + 8u * NST1;
    unsigned int* count0 = reinterpret_cast<unsigned int*>(smem + 8 * (NST0 + 2 * NST1 + NSTC));
    unsigned int* countC = count0 + NST0;
    char* ring0 = smem + 256;
    char* ringC = ring0 + (size_t)NST0 * STAGE0;      // TMA destinations first: 128-byte aligned
    char* ring1 = ringC + (size_t)NSTC * STAGEC;
    const uint32_t ring0_u32 = smem_u32(ring0), ringC_u32 = smem_u32(ringC);
    const int nx = A.nx, ny = A.ny;
    const int tile_cells = quad_runs(NWR) * C;
    constexpr int NBOX = 6 * NG;
    constexpr uint32_t STAGE_TX = (uint32_t)(NBOX * RB * BOXB);

    auto issue = [&](const PairCursor& pc, uint32_t slot) {
        const uint32_t bar = full0 + 8u * slot;
        const uint32_t dst = ring0_u32 + slot * STAGE0;
        const int y = pc.it.j0 - 4 + pc.q * RB;
        if (lane == 0) mbar_expect_tx(bar, STAGE_TX);
        __syncwarp();
        if (lane < NBOX) {
            const int f = lane / NG, g = lane - NG * f;
            const CUtensorMap* map = f == 0 ? &A.mU : f == 1 ? &A.mV : f == 2 ? &A.mW
                                   : f == 3 ? &A.ma : f == 4 ? &A.mb : &A.mc;
            tma_load_3d(dst + f * ARR0 + g * SLAB, map, bar, pc.it.i0 - 2 * C + g * GW * VW, y,
                        f < 3 ? pc.it.sim : 0);
        }
    };
    // C builds: the B warps' coefficient rows of the cursor's stage (a, b, c two rows below the A
    // warps' rows)
    auto issueC = [&](const PairCursor& pc, uint32_t slot) {
        const uint32_t bar = fullC + 8u * slot;
        const uint32_t dst = ringC_u32 + slot * STAGEC;
        const int y = pc.it.j0 - 6 + pc.q * RB;
        if (lane == 0) mbar_expect_tx(bar, (uint32_t)(3 * NG * RB * BOXB));
        __syncwarp();
        if (lane < 3 * NG) {
            const int f = lane / NG, g = lane - NG * f;
            const CUtensorMap* map = f == 0 ? &A.ma : f == 1 ? &A.mb : &A.mc;
            tma_load_3d(dst + f * ARR0 + g * SLAB, map, bar, pc.it.i0 - 2 * C + g * GW * VW, y, 0);
        }
    };
    auto advance_cursor = [&](PairCursor& pc) {
        if (pc.item >= A.nitems) return;
        if (++pc.q == pc.it.nstage) {
            pc.q = 0;
            pc.item += gridDim.x;
            if (pc.item < A.nitems) pc.it = quad_item<RB>(A, pc.item, tile_cells);
        }
    };

    if (threadIdx.x == 0) {
        for (int s = 0; s < NST0; ++s) { mbar_init(full0 + 8u * s, 1); count0[s] = 0u; }
        for (int s = 0; s < NSTC; ++s) { mbar_init(fullC + 8u * s, 1); countC[s] = 0u; }
        for (int s = 0; s < NST1; ++s) { mbar_init(full1 + 8u * s, NWR); mbar_init(empty1 + 8u * s, NWR); }
        fence_barrier_init();
        fence_proxy_async();
    }
    // ring1 runs that no A lane writes are read (and discarded) by B's outermost lanes
    for (int o = threadIdx.x * 16; o < NST1 * STAGE1; o += NTHR * 16)
        *reinterpret_cast<uint4*>(ring1 + o) = make_uint4(0u, 0u, 0u, 0u);
    __syncthreads();

    PairCursor pc;
    pc.item = blockIdx.x;
    pc.q = 0;
    if (pc.item < A.nitems) pc.it = quad_item<RB>(A, pc.item, tile_cells);
    if (isA) {
        for (int s = 0; s < NST0; ++s) {
            if (warp == 0 && pc.item < A.nitems) issue(pc, (uint32_t)s);
            advance_cursor(pc);
        }
    } else if constexpr (CB) {
        for (int s = 0; s < NSTC; ++s) {
            if (warp == NWR && pc.item < A.nitems) issueC(pc, (uint32_t)s);
            advance_cursor(pc);
        }
    }

    // where this lane finds its run in a stage of its source ring, and the ring's strides
    const int src_off = isA ? (w / GW) * SLAB + (w % GW) * (VW * (int)sizeof(T)) + 16 * lane
                            : (30 * w + lane + 1) * 16;
    const int src_arr = isA ? ARR0 : ARR1, src_row = isA ? BOXB : P1;
    // coefficient rows: A finds them in its ring0 stage (arrays 3..5); B in ring1 (arrays 3..5) or,
    // in the C builds, in its own boxes (same origins as ring0's boxes: run -2 + 30 GW g; a run in
    // the two-run overlap of two boxes is taken from the later one; the outermost lane of the last
    // B warp owns the run one past the last box: it reads, and discards, that box's last run)
    const int cof_t = 30 * w + lane + 1;                   // the B lane's run, counted from run -2
    const int cof_g = min(cof_t / (30 * GW), NG - 1);
    const int cof_off = isA || !CB ? src_off : cof_g * SLAB + min(cof_t - 30 * GW * cof_g, BOXB / 16 - 1) * 16;
    const int cof_arr = isA || CB ? ARR0 : ARR1, cof_row = isA || CB ? BOXB : P1;
    const int dst_off = (30 * w + lane) * 16;              // A: own run in a ring1 row
    const int run0 = isA ? 30 * w - 2 + lane : 30 * w - 1 + lane;  // tile run this lane owns
    const bool lane_ok = lane >= 1 && lane <= (isA || w < NWR - 1 ? kPairLanes : kPairLanes - 2);
    const size_t plane = (size_t)nx * ny;

    uint32_t gc = 0;
    for (long long item = blockIdx.x; item < A.nitems; item += gridDim.x) {
        const PairItem it = quad_item<RB>(A, item, tile_cells);
        const int iown = it.i0 + run0 * C;               // first own cell (may lie outside the domain)
        const bool store_ok = lane_ok && iown >= 0 && iown < nx;
        const bool atW = iown == 0, atE = iown + C == nx, edge0 = atW || iown == nx;
        const StepCoef<T> k = load_coef<T>(A.coefs + it.sim);
        T* gU = (T*)A.U1 + it.sim * plane + iown;
        T* gV = (T*)A.V1 + it.sim * plane + iown;
        T* gW = (T*)A.W1 + it.sim * plane + iown;

        PairLevel<T, C> L1, L2;
        L1.clear();
        L2.clear();

        for (int q = 0; q < it.nstage; ++q, ++gc) {
            const uint32_t s0 = gc % NST0, s1 = gc % NST1, sc = CB ? gc % (CB ? NSTC : 1) : 0u;
            if (isA) {
                mbar_wait(full0 + 8u * s0, (gc / NST0) & 1u);
                if (gc >= NST1) mbar_wait(empty1 + 8u * s1, ((gc / NST1) - 1u) & 1u);
            } else {
                if constexpr (CB) mbar_wait(fullC + 8u * sc, (gc / (CB ? NSTC : 1)) & 1u);
                mbar_wait(full1 + 8u * s1, (gc / NST1) & 1u);
            }
            const char* src = (isA ? ring0 + (size_t)s0 * STAGE0 : ring1 + (size_t)s1 * STAGE1) + src_off;
            const char* cof = (isA ? ring0 + (size_t)s0 * STAGE0 + 3 * ARR0
                               : CB ? ringC + (size_t)sc * STAGEC : ring1 + (size_t)s1 * STAGE1 + 3 * ARR1) + cof_off;
            char* dst = ring1 + (size_t)s1 * STAGE1 + dst_off;
            // first row arriving at this role in this stage: time k for A, time k+2 for B
            const int jfirst = it.j0 - 4 + q * RB - (isA ? 0 : 2);
            auto row_body = [&](auto ghost_c, const int rr) {
                constexpr bool GHOST = decltype(ghost_c)::value;
                const int jn = jfirst + rr;
                const char* p = src + rr * src_row;
                T uN[C], vN[C], wN[C], aN[C], bN[C], cN[C];
                ld_run<T, C>(p + 0 * src_arr, uN);
                ld_run<T, C>(p + 1 * src_arr, vN);
                ld_run<T, C>(p + 2 * src_arr, wN);
                const char* pcf = cof + rr * cof_row;
                ld_run<T, C>(pcf + 0 * cof_arr, aN);
                ld_run<T, C>(pcf + 1 * cof_arr, bN);
                ld_run<T, C>(pcf + 2 * cof_arr, cN);
                T u1[C], v1[C], w1[C], a1[C], b1[C], c1[C];   // row jn-1, one level up
                L1.template advance<GHOST>(jn, ny, atW, atE, edge0, k, uN, vN, wN, aN, bN, cN, u1, v1, w1, a1, b1, c1);
                T u2[C], v2[C], w2[C], a2[C], b2[C], c2[C];   // row jn-2, two levels up
                L2.template advance<GHOST>(jn - 1, ny, atW, atE, edge0, k, u1, v1, w1, a1, b1, c1, u2, v2, w2, a2, b2, c2);
                if constexpr (CB) {
                    // both roles' stores, predicated, no branch: the RB rows of a stage stay one
                    // basic block, which ptxas schedules across rows (+3 % fp64, +5 % fp32 at 8192^2
                    // over a branch per role and row)
                    const uint32_t o = smem_u32(dst) + rr * P1;
                    const bool sa = isA && lane_ok;
                    st_run_shared_if<T, C>(sa, o + 0 * ARR1, u2);
                    st_run_shared_if<T, C>(sa, o + 1 * ARR1, v2);
                    st_run_shared_if<T, C>(sa, o + 2 * ARR1, w2);
                    const int r = jn - 2;
                    const bool sb = !isA && store_ok && r >= it.j0 && r < it.j1;
                    const size_t off = (size_t)(sb ? r : 0) * nx;
                    st_run_global_if<T, C>(sb, gU + off, u2);
                    st_run_global_if<T, C>(sb, gV + off, v2);
                    st_run_global_if<T, C>(sb, gW + off, w2);
                } else
                if (isA) {
                    if (lane_ok) {                            // time-k+2 row jn-2 (and its coefficients)
                        char* o = dst + rr * P1;
                        st_run<T, C>(o + 0 * ARR1, u2);
                        st_run<T, C>(o + 1 * ARR1, v2);
                        st_run<T, C>(o + 2 * ARR1, w2);
                        if constexpr (!CB) {
                            st_run<T, C>(o + 3 * ARR1, a2);
                            st_run<T, C>(o + 4 * ARR1, b2);
                            st_run<T, C>(o + 5 * ARR1, c2);
                        }
                    }
                } else {
                    const int r = jn - 2;                     // time-k+4 row
                    if (store_ok && r >= it.j0 && r < it.j1) {
                        const size_t off = (size_t)r * nx;
                        st_run<T, C>((char*)(gU + off), u2);
                        st_run<T, C>((char*)(gV + off), v2);
                        st_run<T, C>((char*)(gW + off), w2);
                    }
                }
            };
            if (jfirst >= 2 && jfirst + RB - 1 < ny) {
#pragma unroll
                for (int rr = 0; rr < RB; ++rr) row_body(std::false_type{}, rr);
            } else {
#pragma unroll
                for (int rr = 0; rr < RB; ++rr) row_body(std::true_type{}, rr);
            }
            __syncwarp();
            // Slot hand-off.  A: ring1 stage written (release); ring0 slot read: the A warp that
            // releases it last refills it with the stage NST0 ahead.  B: ring1 stage read; in the
            // C builds the B warp that releases the coefficient slot last refills it.
            if (isA) {
                unsigned int prev = 0;
                if (lane == 0) {
                    mbar_arrive(full1 + 8u * s1);
                    __threadfence_block();
                    prev = atomicAdd(&count0[s0], 1u);
                }
                prev = __shfl_sync(0xffffffffu, prev, 0);
                if (prev == (unsigned)NWR - 1u) {
                    if (lane == 0) { count0[s0] = 0u; __threadfence_block(); }
                    if (pc.item < A.nitems) issue(pc, s0);
                }
                advance_cursor(pc);
            } else if constexpr (CB) {
                unsigned int prev = 0;
                if (lane == 0) {
                    mbar_arrive(empty1 + 8u * s1);
                    __threadfence_block();
                    prev = atomicAdd(&countC[sc], 1u);
                }
                prev = __shfl_sync(0xffffffffu, prev, 0);
                if (prev == (unsigned)NWR - 1u) {
                    if (lane == 0) { countC[sc] = 0u; __threadfence_block(); }
                    if (pc.item < A.nitems) issueC(pc, sc);
                }
                advance_cursor(pc);
            } else if (lane == 0) {
                mbar_arrive(empty1 + 8u * s1);
            }
        }
    }
}

}  // namespace gg

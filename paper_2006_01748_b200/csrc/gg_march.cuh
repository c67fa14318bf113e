// gg_march.cuh -- the register-rolling row march shared by the streaming kernels.
//
// A lane owns a run of C consecutive cells of one grid row (16 bytes: C = 2 fp64 / 4 fp32 cells;
// C = 1 for the tile-edge halo lanes of the two-step kernel) and walks up the grid one row at a
// time.  It keeps, in registers, the extended run (west neighbour, C own cells, east neighbour)
// of W for rows jc-1, jc, jc+1 and of M = 1 - U, V, aw, b for rows jc, jc+1, plus U, cs, the cross
// term H and the south face fluxes of its own cells (aw, cs: the stored face sums of the tensor,
// gg_common.cuh).  On every arriving row it evaluates the flux form of
// Tables 1-2 (gg_common.cuh) for the centre row jc:
//   * x faces 0..C of the run (interior ones shared by the two cells they separate; the run's
//     outer faces are recomputed by the neighbouring lane rather than exchanged),
//   * north faces of the own cells, kept as the next row's south faces,
//   * the three updates of eq. (3).
// Neumann faces (reading A2): `atW` / `atE` lanes zero the flux through the domain's west / east
// face and mirror W's neighbour; the GHOST instantiation mirrors U, V, W evenly and H oddly when
// the centre or the arriving row is ghost row -1 / ny, which makes that face's fluxes exactly 0.
// The body is straight-line: no join points, so the window is renamed, not moved, across the
// rows a caller unrolls.
#pragma once
#include "gg_common.cuh"

namespace gg {

// 16-byte vector of T
template <typename T> struct Vec16;
template <> struct Vec16<double> { using type = double2; };
template <> struct Vec16<float> { using type = float4; };

// C consecutive elements from a 16-byte-aligned (C > 1) shared or global address
template <typename T, int C>
__device__ __forceinline__ void ld_run(const char* p, T* x) {
    if constexpr (C == 1) {
        x[0] = *reinterpret_cast<const T*>(p);
    } else {
        typename Vec16<T>::type v = *reinterpret_cast<const typename Vec16<T>::type*>(p);
        if constexpr (C == 2) { x[0] = v.x; x[1] = v.y; }
        else { x[0] = v.x; x[1] = v.y; x[2] = v.z; x[3] = v.w; }
    }
}
template <typename T, int C>
__device__ __forceinline__ void st_run(char* p, const T* x) {
    if constexpr (C == 1) {
        *reinterpret_cast<T*>(p) = x[0];
    } else {
        typename Vec16<T>::type v;
        if constexpr (C == 2) { v.x = x[0]; v.y = x[1]; }
        else { v.x = x[0]; v.y = x[1]; v.z = x[2]; v.w = x[3]; }
        *reinterpret_cast<typename Vec16<T>::type*>(p) = v;
    }
}

// Predicated 16-byte stores without a branch (the row bodies of gg_quad.cuh stay one basic block).
// They carry a "memory" clobber: the compiler is TOLD they write memory, so it can neither hoist a
// later load of the ring above them nor sink them below the mbarrier arrive that publishes the
// row -- the A-warp -> B-warp hand-off of gg_quad.cuh no longer rests on `volatile` ordering alone.
// (-DGG_ST_NO_CLOBBER builds the round-2 form without it, for A/B timing; both forms are
// bit-identical in the fuzz.)
#ifdef GG_ST_NO_CLOBBER
#define GG_ST_CLOBBER
#else
#define GG_ST_CLOBBER : "memory"
#endif
template <typename T, int C>
__device__ __forceinline__ void st_run_shared_if(bool ok, uint32_t addr, const T* x) {
    static_assert(C * sizeof(T) == 16, "16-byte runs");
    if constexpr (sizeof(T) == 8)
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %0, 0;\n\t@p st.shared.v2.f64 [%1], {%2, %3};\n\t}"
                     ::"r"((uint32_t)ok), "r"(addr), "d"(x[0]), "d"(x[1]) GG_ST_CLOBBER);
    else
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %0, 0;\n\t@p st.shared.v4.f32 [%1], {%2, %3, %4, %5};\n\t}"
                     ::"r"((uint32_t)ok), "r"(addr), "f"(x[0]), "f"(x[1]), "f"(x[2]), "f"(x[3]) GG_ST_CLOBBER);
}
template <typename T, int C>
__device__ __forceinline__ void st_run_global_if(bool ok, void* addr, const T* x) {
    static_assert(C * sizeof(T) == 16, "16-byte runs");
    if constexpr (sizeof(T) == 8)
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %0, 0;\n\t@p st.global.v2.f64 [%1], {%2, %3};\n\t}"
                     ::"r"((uint32_t)ok), "l"(addr), "d"(x[0]), "d"(x[1]) GG_ST_CLOBBER);
    else
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %0, 0;\n\t@p st.global.v4.f32 [%1], {%2, %3, %4, %5};\n\t}"
                     ::"r"((uint32_t)ok), "l"(addr), "f"(x[0]), "f"(x[1]), "f"(x[2]), "f"(x[3]) GG_ST_CLOBBER);
}

// Where a lane finds its data inside one ring stage: byte offset of row 0 of array 0, stride per
// array, stride per row -- for the own run and for the west / east neighbour elements (which may
// live in the neighbour warp's strip or in a tile-edge halo slab with different strides).
struct LaneMap {
    int oOff, oSF, oSR;
    int wOff, wSF, wSR;
    int eOff, eSF, eSR;
};

template <typename T, int C>
struct MarchWindow {
    static constexpr int E = C + 2;
    T wP[E], wC[E], wN[E], mC[E], mN[E], vC[E], vN[E], aC[E], aN[E], bC[E], bN[E];
    T uC[C], uN[C], cC[C], cN[C], hC[C], hN[C], sV[C], sW[C];

    __device__ __forceinline__ void clear() {
#pragma unroll
        for (int e = 0; e < E; ++e) wP[e] = wC[e] = mC[e] = vC[e] = aC[e] = bC[e] = (T)0;
#pragma unroll
        for (int c = 0; c < C; ++c) uC[c] = cC[c] = hC[c] = sV[c] = sW[c] = (T)0;
    }

    // Load row `rr` of the stage at `st` (arrays in the order U, V, W, a, b, c) as the arriving
    // row N, and form its cross term H.
    __device__ __forceinline__ void load(const char* st, const LaneMap& L, int rr, bool atW, bool atE) {
        const char* own = st + L.oOff + rr * L.oSR;
        const char* west = st + L.wOff + rr * L.wSR;
        const char* east = st + L.eOff + rr * L.eSR;
        T* dst[5] = {mN, vN, wN, aN, bN};
#pragma unroll
        for (int f = 0; f < 5; ++f) {
            ld_run<T, C>(own + f * L.oSF, dst[f] + 1);
            dst[f][0] = *reinterpret_cast<const T*>(west + f * L.wSF);
            dst[f][C + 1] = *reinterpret_cast<const T*>(east + f * L.eSF);
        }
#pragma unroll
        for (int c = 0; c < C; ++c) uN[c] = mN[c + 1];
#pragma unroll
        for (int e = 0; e < E; ++e) mN[e] = one_minus(mN[e]);
        ld_run<T, C>(own + 5 * L.oSF, cN);
        // mirrored x ghosts of W (tangential difference in H at boundary cells)
        if (atW) wN[0] = wN[1];
        if (atE) wN[C + 1] = wN[C];
#pragma unroll
        for (int c = 0; c < C; ++c) hN[c] = cross(bN[c + 1], wN[c + 2], wN[c]);
    }

    // Advance the centre row (the row below the arriving row `jn`) by one time step into
    // oU, oV, oW, then roll the window.  GHOST: handle jn == 0 (centre is ghost row -1) and
    // jn == ny (arriving row is ghost row ny); callers use it only for stages that contain them.
    template <bool GHOST>
    __device__ __forceinline__ void advance(int jn, int ny, bool atW, bool atE, const StepCoef<T>& k,
                                            T* oU, T* oV, T* oW) {
        if constexpr (GHOST) {
            if (jn == 0) {
#pragma unroll
                for (int e = 0; e < E; ++e) { mC[e] = mN[e]; vC[e] = vN[e]; wC[e] = wN[e]; }
#pragma unroll
                for (int c = 0; c < C; ++c) { uC[c] = uN[c]; hC[c] = -hN[c]; }
            }
            if (jn == ny) {
#pragma unroll
                for (int e = 0; e < E; ++e) { mN[e] = mC[e]; vN[e] = vC[e]; wN[e] = wC[e]; }
#pragma unroll
                for (int c = 0; c < C; ++c) { uN[c] = uC[c]; hN[c] = -hC[c]; }
            }
        }
        T G[E];  // cross term of the x faces (rows jc-1, jc+1)
#pragma unroll
        for (int e = 0; e < E; ++e) G[e] = cross(bC[e], wN[e], wP[e]);
        T pV[C + 1], pW[C + 1];  // x faces f = 0..C (face f lies between extended cells f, f+1)
#pragma unroll
        for (int f = 0; f <= C; ++f) {
            pV[f] = flux_V(mC[f], mC[f + 1], vC[f], vC[f + 1]);
            pW[f] = flux_W(aC[f + 1], wC[f], wC[f + 1], G[f], G[f + 1]);   // aw of extended cell f+1
        }
        if (atW) { pV[0] = (T)0; pW[0] = (T)0; }
        if (atE) { pV[C] = (T)0; pW[C] = (T)0; }
        T nV[C], nW[C];  // north faces of the own cells
#pragma unroll
        for (int c = 0; c < C; ++c) {
            nV[c] = flux_V(mC[c + 1], mN[c + 1], vC[c + 1], vN[c + 1]);
            nW[c] = flux_W(cN[c], wC[c + 1], wN[c + 1], hC[c], hN[c]);     // cs of the arriving row
        }
#pragma unroll
        for (int c = 0; c < C; ++c) {
            oU[c] = upd_U(k, uC[c], mC[c + 1], wC[c + 1]);
            oV[c] = upd_V(k, vC[c + 1], pV[c + 1], pV[c], nV[c], sV[c]);
            oW[c] = upd_W(k, vC[c + 1], wC[c + 1], pW[c + 1], pW[c], nW[c], sW[c]);
        }
#pragma unroll
        for (int c = 0; c < C; ++c) { sV[c] = nV[c]; sW[c] = nW[c]; }  // next row's south faces
    }

    // Own-cell coefficients of the centre row (valid between advance() and roll()).
    __device__ __forceinline__ const T* centre_a() const { return aC + 1; }
    __device__ __forceinline__ const T* centre_b() const { return bC + 1; }
    __device__ __forceinline__ const T* centre_c() const { return cC; }

    __device__ __forceinline__ void roll() {
#pragma unroll
        for (int e = 0; e < E; ++e) {
            wP[e] = wC[e]; wC[e] = wN[e];
            mC[e] = mN[e]; vC[e] = vN[e]; aC[e] = aN[e]; bC[e] = bN[e];
        }
#pragma unroll
        for (int c = 0; c < C; ++c) { uC[c] = uN[c]; cC[c] = cN[c]; hC[c] = hN[c]; }
    }
};

}  // namespace gg

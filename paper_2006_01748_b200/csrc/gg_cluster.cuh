// gg_cluster.cuh -- the on-chip kernel for grids that fit into ONE thread-block cluster.
//
// Small grids (BASELINE config 0: 64^2) are latency-bound, not bandwidth-bound: what a step costs
// is the longest dependent chain plus whatever the CTAs need to tell each other, not bytes.  The
// row march of the streaming kernels (and of gg_resident.cuh) evaluates the rows of a slab one
// after another -- ~300 cycles per row -- and gg_resident.cuh exchanges edge rows through global
// memory (three L2 round trips per step).  Here:
//
//  * One cluster of CL CTAs per simulation (batches: one cluster each, independent, no
//    co-residency requirement).  CTA r of the cluster keeps rows [r R, r R + R) of U, V, W twice
//    (ping-pong), one halo row on each side, and the matching rows of the stored tensor (aw, b, cs)
//    in shared memory for all n steps of the call.
//  * EVERY cell of the slab is evaluated in parallel: a thread owns one run of C cells of one row
//    (C = 1 while every cell of the slab can have a thread of its own, else a 16-byte run; several
//    rows per thread if the slab has more runs than the CTA threads) and computes its cells
//    directly from shared memory: the run's C + 1 x faces once each, the 2 C y faces.  No march,
//    no register window: the depth of a step is one run, whatever the slab height.  The CTA is
//    two-dimensional (runs of a row x rows), so no index arithmetic is left in the step loop.
//  * A thread on the slab's first / last row also sends its result into the neighbour CTA's halo
//    row through distributed shared memory: `st.async ... mbarrier::complete_tx::bytes` on the
//    NEIGHBOUR's mbarrier of that state copy.  A step ends with a CTA barrier (own rows) and a wait
//    on the CTA's own mbarrier (both neighbours' edge rows have landed): point to point, no
//    cluster-wide barrier in the step loop (one per step cost 0.2 us more), no global memory, no
//    flags, no L2 round trip between the first load and the last store of a call.  A neighbour can
//    only be one step ahead (it needs this CTA's edge row to go on), and what it then writes is
//    the halo of the OTHER state copy, which this CTA's edge threads finished reading before
//    they sent: the two copies and two mbarriers (one per copy, armed one round ahead) suffice.
//  * Arithmetic: the per-cell formulas of gg_generic.cuh (clamped neighbours, boundary W fluxes
//    zeroed) through the same functions with the same operands => bit-identical to every other
//    kernel of the library.
#pragma once
#include "gg_common.cuh"
#include "gg_march.cuh"
#include "gg_stream.cuh"   // mbarrier wrappers

namespace gg {

struct ClusterArgs {
    const void* U0; const void* V0; const void* W0;   // state at time k   [B][ny][nx]
    void* U1; void* V1; void* W1;                     // state at time k+n [B][ny][nx]
    const void* a; const void* b; const void* c;      // stored tensor aw, b, cs  [ny][nx]
    const StepCoef<double>* coefs;                    // [B], folded on the device (gg_dt.cuh)
    int nx, ny, nbatch;
    int CL, R;                  // CTAs per cluster (= per simulation); rows per CTA
    int pitch;                  // shared-memory row pitch in bytes (nx * sizeof(T) + 32)
    long long nsteps;
};

__host__ __device__ constexpr int cluster_pitch(int nx, int esize) { return nx * esize + 32; }
__host__ __device__ constexpr size_t cluster_smem_bytes(int nx, int esize, int R) {
    return (size_t)9 * (R + 2) * cluster_pitch(nx, esize) + 64;   // 2 x (U,V,W) + (aw,b,cs) + two mbarriers
}

__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
// shared::cluster address of `addr` (a shared::cta address of this CTA) in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t cluster_map(uint32_t addr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
// one run (4, 8 or 16 bytes) into another CTA's shared memory, completing its byte count on that
// CTA's mbarrier when it lands
template <int BYTES>
__device__ __forceinline__ void st_async_run(uint32_t addr, const void* x, uint32_t mbar) {
    if constexpr (BYTES == 16) {
        const uint4 v = *reinterpret_cast<const uint4*>(x);
        asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.b32 [%0], {%1, %2, %3, %4}, [%5];"
                     ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w), "r"(mbar) : "memory");
    } else if constexpr (BYTES == 8) {
        const uint2 v = *reinterpret_cast<const uint2*>(x);
        asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.b32 [%0], {%1, %2}, [%3];"
                     ::"r"(addr), "r"(v.x), "r"(v.y), "r"(mbar) : "memory");
    } else {
        asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b32 [%0], %1, [%2];"
                     ::"r"(addr), "r"(*reinterpret_cast<const uint32_t*>(x)), "r"(mbar) : "memory");
    }
}
__device__ __forceinline__ void cluster_barrier() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

// gridDim.x = nbatch * CL, cluster dimension CL (launch attribute); blockDim = (runs per row, rows
// evaluated at once).  Dynamic shared memory: [set 0: U,V,W][set 1: U,V,W][aw,b,cs], every array
// (R+2) rows x pitch bytes; row m of the slab holds domain row r0-1+m; a row starts with 16 bytes
// of padding so that the west neighbour element of cell 0 is addressable (its value is never
// used: clamped / zero-flux faces).
template <typename T, int C>
__global__ void __launch_bounds__(512, 1) gg_step_cluster(const ClusterArgs A) {
    constexpr int ES = (int)sizeof(T);
    constexpr int RUNB = C * ES;
    constexpr int E = C + 2;
    extern __shared__ __align__(128) char smem[];
    const int nx = A.nx, ny = A.ny, R = A.R, pitch = A.pitch;
    const int ARRS = (R + 2) * pitch, SET = 3 * ARRS;
    char* coef = smem + 2 * SET;
    const int rank = (int)cluster_ctarank();
    const int sim = blockIdx.x / A.CL;
    const int r0 = min(rank * R, ny), r1 = min(r0 + R, ny), rows = r1 - r0;
    const int l = threadIdx.x;                                // the thread's run: cells [l C, l C + C) of a row
    const int lanes = blockDim.x;                             // = nx / C
    const size_t plane = (size_t)nx * ny;
    const StepCoef<T> k = load_coef<T>(A.coefs + sim);
    const uint32_t smem_u = (uint32_t)__cvta_generic_to_shared(smem);
    const int tid = threadIdx.y * blockDim.x + threadIdx.x, nthr = blockDim.x * blockDim.y;
    const bool atW = l == 0, atE = l == lanes - 1;
    const int o = 16 + RUNB * l;                              // byte offset of the run in a shared-memory row

    // hbar[b]: "the halo rows of state copy b are complete" -- expects, per round, the bytes of the
    // edge rows the neighbour CTAs send (3 fields x one row each), armed by thread 0 one round ahead
    const uint32_t hbar = smem_u + 3 * SET;
    const bool has_below = rows > 0 && rank > 0, has_above = rows > 0 && r1 < ny;
    const uint32_t halo_tx = (uint32_t)(((has_below ? 1 : 0) + (has_above ? 1 : 0)) * 3 * nx * ES);
    if (tid == 0) {
        mbar_init(hbar, 1);
        mbar_init(hbar + 8, 1);
        fence_barrier_init();
        if (halo_tx != 0u) {                    // (a CTA without neighbours never touches them)
            mbar_expect_tx(hbar + 8, halo_tx);  // round of step 0 (fills copy 1)
            mbar_expect_tx(hbar, halo_tx);      // round of step 1 (fills copy 0)
        }
    }
    // ---- start-up: zero everything, then load the slab and the halo rows inside the domain
    for (int q = tid * 16; q < 3 * SET; q += nthr * 16)
        *reinterpret_cast<uint4*>(smem + q) = make_uint4(0u, 0u, 0u, 0u);
    __syncthreads();
    if (rows > 0) {
        const T* gs[3] = {(const T*)A.U0 + sim * plane, (const T*)A.V0 + sim * plane, (const T*)A.W0 + sim * plane};
        const T* gc[3] = {(const T*)A.a, (const T*)A.b, (const T*)A.c};
        for (int m = threadIdx.y; m < rows + 2; m += blockDim.y) {
            const int j = r0 - 1 + m;
            if (j < 0 || j >= ny) continue;
#pragma unroll
            for (int f = 0; f < 3; ++f) {
                T x[C];
                ld_run<T, C>((const char*)(gs[f] + (size_t)j * nx + l * C), x);
                st_run<T, C>(smem + f * ARRS + m * pitch + o, x);
                ld_run<T, C>((const char*)(gc[f] + (size_t)j * nx + l * C), x);
                st_run<T, C>(coef + f * ARRS + m * pitch + o, x);
            }
        }
    }
    cluster_barrier();

    for (long long step = 0; step < A.nsteps; ++step) {
        const char* src = smem + (int)(step & 1) * SET;
        const int dset = (int)((step + 1) & 1) * SET;
        for (int r = threadIdx.y; r < rows; r += blockDim.y) {
            const int j = r0 + r, m = r + 1;
            const bool hasS = j > 0, hasN = j < ny - 1;
            const int oc = m * pitch + o, os = (hasS ? m - 1 : m) * pitch + o, on = (hasN ? m + 1 : m) * pitch + o;
            // extended runs (west neighbour, C own cells, east neighbour), clamped at the domain's
            // west / east faces: W of rows j-1, j, j+1; U, V, b of row j; own cells of rows j-1, j+1
            auto ld_ext = [&](const char* base, int off, T* x) {
                ld_run<T, C>(base + off, x + 1);
                x[0] = *reinterpret_cast<const T*>(base + off - ES);
                x[C + 1] = *reinterpret_cast<const T*>(base + off + RUNB);
                if (atW) x[0] = x[1];
                if (atE) x[C + 1] = x[C];
            };
            T wS[E], wC[E], wN[E], mC[E], vC[E], bC[E], uC[C];
            ld_ext(src + 2 * ARRS, os, wS);
            ld_ext(src + 2 * ARRS, oc, wC);
            ld_ext(src + 2 * ARRS, on, wN);
            ld_ext(src + 0 * ARRS, oc, mC);
            ld_ext(src + 1 * ARRS, oc, vC);
            ld_ext(coef + 1 * ARRS, oc, bC);
#pragma unroll
            for (int c = 0; c < C; ++c) uC[c] = mC[c + 1];
#pragma unroll
            for (int e = 0; e < E; ++e) mC[e] = one_minus(mC[e]);
            T mS[C], mN[C], vS[C], vN[C], bS[C], bN[C], awx[C + 1], csC[C], csN[C];
            ld_run<T, C>(src + 0 * ARRS + os, mS);
            ld_run<T, C>(src + 0 * ARRS + on, mN);
            ld_run<T, C>(src + 1 * ARRS + os, vS);
            ld_run<T, C>(src + 1 * ARRS + on, vN);
            ld_run<T, C>(coef + 1 * ARRS + os, bS);
            ld_run<T, C>(coef + 1 * ARRS + on, bN);
            ld_run<T, C>(coef + 0 * ARRS + oc, awx);              // west faces of the own cells ...
            awx[C] = *reinterpret_cast<const T*>(coef + 0 * ARRS + oc + RUNB);   // ... and of the east neighbour
            ld_run<T, C>(coef + 2 * ARRS + oc, csC);
            ld_run<T, C>(coef + 2 * ARRS + on, csN);
#pragma unroll
            for (int c = 0; c < C; ++c) { mS[c] = one_minus(mS[c]); mN[c] = one_minus(mN[c]); }

            // cross terms: G of the extended run (x faces), H of the own cells and of their
            // north / south neighbours (y faces)
            T G[E], H0[C], HN[C], HS[C];
#pragma unroll
            for (int e = 0; e < E; ++e) G[e] = cross(bC[e], wN[e], wS[e]);
#pragma unroll
            for (int c = 0; c < C; ++c) {
                H0[c] = cross(bC[c + 1], wC[c + 2], wC[c]);
                HN[c] = cross(bN[c], wN[c + 2], wN[c]);
                HS[c] = cross(bS[c], wS[c + 2], wS[c]);
            }
            // x faces f = 0..C (face f lies between extended cells f and f+1), once each
            T pV[C + 1], pW[C + 1];
#pragma unroll
            for (int f = 0; f <= C; ++f) {
                pV[f] = flux_V(mC[f], mC[f + 1], vC[f], vC[f + 1]);
                pW[f] = flux_W(awx[f], wC[f], wC[f + 1], G[f], G[f + 1]);
            }
            if (atW) pW[0] = (T)0;
            if (atE) pW[C] = (T)0;
            T oU[C], oV[C], oW[C];
#pragma unroll
            for (int c = 0; c < C; ++c) {
                const T pN = flux_V(mC[c + 1], mN[c], vC[c + 1], vN[c]);
                const T pS = flux_V(mS[c], mC[c + 1], vS[c], vC[c + 1]);
                T fN = flux_W(csN[c], wC[c + 1], wN[c + 1], H0[c], HN[c]);
                T fS = flux_W(csC[c], wS[c + 1], wC[c + 1], HS[c], H0[c]);
                if (!hasN) fN = (T)0;
                if (!hasS) fS = (T)0;
                oU[c] = upd_U(k, uC[c], mC[c + 1], wC[c + 1]);
                oV[c] = upd_V(k, vC[c + 1], pV[c + 1], pV[c], pN, pS);
                oW[c] = upd_W(k, vC[c + 1], wC[c + 1], pW[c + 1], pW[c], fN, fS);
            }
            char* d = smem + dset + oc;
            st_run<T, C>(d + 0 * ARRS, oU);
            st_run<T, C>(d + 1 * ARRS, oV);
            st_run<T, C>(d + 2 * ARRS, oW);
            // edge rows also go into the neighbour CTAs' halo rows (distributed shared memory)
            if (r == 0 && rank > 0) {                       // bottom row -> top halo (row R+1) of the CTA below
                const uint32_t ra = cluster_map(smem_u + dset + (R + 1) * pitch + o, (uint32_t)(rank - 1));
                const uint32_t rb = cluster_map(hbar + 8u * (uint32_t)((step + 1) & 1), (uint32_t)(rank - 1));
                st_async_run<RUNB>(ra + 0 * ARRS, oU, rb);
                st_async_run<RUNB>(ra + 1 * ARRS, oV, rb);
                st_async_run<RUNB>(ra + 2 * ARRS, oW, rb);
            }
            if (r == rows - 1 && r1 < ny) {                 // top row -> bottom halo (row 0) of the CTA above
                const uint32_t ra = cluster_map(smem_u + dset + o, (uint32_t)(rank + 1));
                const uint32_t rb = cluster_map(hbar + 8u * (uint32_t)((step + 1) & 1), (uint32_t)(rank + 1));
                st_async_run<RUNB>(ra + 0 * ARRS, oU, rb);
                st_async_run<RUNB>(ra + 1 * ARRS, oV, rb);
                st_async_run<RUNB>(ra + 2 * ARRS, oW, rb);
            }
        }
        // own rows of the new level: a CTA barrier; the neighbours' edge rows: this copy's mbarrier
        // (its phase flips every second step).  Thread 0 then arms it for its next round, two
        // steps on -- before this CTA sends anything a neighbour could answer with that round.
        __syncthreads();
        if (halo_tx != 0u) {
            const uint32_t hb = hbar + 8u * (uint32_t)((step + 1) & 1);
            mbar_wait(hb, (uint32_t)((step >> 1) & 1));
            if (tid == 0) mbar_expect_tx(hb, halo_tx);
        }
    }
    cluster_barrier();   // nobody leaves while a neighbour may still be sending to it

    // ---- the call's last time level goes back to HBM
    {
        const char* fin = smem + (int)(A.nsteps & 1) * SET;
        T* gd[3] = {(T*)A.U1 + sim * plane, (T*)A.V1 + sim * plane, (T*)A.W1 + sim * plane};
        for (int r = threadIdx.y; r < rows; r += blockDim.y) {
#pragma unroll
            for (int f = 0; f < 3; ++f) {
                T x[C];
                ld_run<T, C>(fin + f * ARRS + (r + 1) * pitch + o, x);
                st_run<T, C>((char*)(gd[f] + (size_t)(r0 + r) * nx + l * C), x);
            }
        }
    }
}

}  // namespace gg

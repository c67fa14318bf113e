// gg_resident.cuh -- GG_KERNEL_RESIDENT: the whole state stays ON CHIP for all n steps of a call.
//
// Small grids (BASELINE configs 0 and 1: 64^2 and 512^2) are launch-latency bound with one kernel
// per step or two: 4.5-6 us per step, whatever the kernel does.  Here ONE cooperative launch
// advances all n steps (stage 8):
//
//  * The grid is cut into row slabs of R rows; one CTA per (simulation, slab), all CTAs resident
//    at once (cooperative launch).  A CTA keeps its slab of U, V, W (plus one halo row above and
//    below) twice (ping-pong) and the matching rows of a, b, c in shared memory for the whole call.
//  * Per step every lane marches its 16-byte column run up the R+2 rows of the slab with the
//    stream kernel's register window (gg_march.cuh: same arithmetic, same operand order =>
//    bit-identical), reading the ping copy and writing the pong copy; x-neighbours are adjacent
//    shared-memory elements.
//  * Slabs exchange their edge rows through a small double-buffered global array (L2-resident) and
//    a per-slab step counter: after step k a CTA publishes its bottom and top rows, releases
//    counter = k, and waits until both neighbours have released k too before it copies their rows
//    into its halo rows.  Point-to-point: no grid-wide barrier.  Buffer parity k & 1 is safe
//    because a neighbour can only be one step ahead.  Spins are bounded (trap, never hang).
//  * Neumann boundaries as everywhere: atW / atE lane flags, ghost rows -1 and ny mirrored by the
//    march (the slab's out-of-domain halo rows just hold zeros).
#pragma once
#include "gg_common.cuh"
#include "gg_march.cuh"

namespace gg {

struct ResidentArgs {
    const void* U0; const void* V0; const void* W0;   // state at time k   [B][ny][nx]
    void* U1; void* V1; void* W1;                     // state at time k+n [B][ny][nx]
    const void* a; const void* b; const void* c;      // [ny][nx]
    const StepCoef<double>* coefs;   // [B], folded on the device (gg_dt.cuh)
    void* halo;                 // [2 parity][nslabs][2 sides][3 fields][nx] elements
    unsigned int* flags;        // [nslabs] last step whose edge rows the slab has published
    int nx, ny, nbatch;
    int R, slabs_per_sim;       // rows per slab; slabs per simulation
    int pitch;                  // shared-memory row pitch in bytes (nx * sizeof(T) + 32)
    long long nsteps;
    unsigned int epoch;         // flags start at epoch (set by the host before the launch)
};

__host__ __device__ constexpr int resident_pitch(int nx, int esize) { return nx * esize + 32; }
__host__ __device__ constexpr size_t resident_smem_bytes(int nx, int esize, int R) {
    return (size_t)9 * (R + 2) * resident_pitch(nx, esize);   // 2 x (U,V,W) + (a,b,c)
}

__device__ __forceinline__ unsigned int ld_acquire_gpu(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_gpu(unsigned int* p, unsigned int v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// 16 bytes from global memory, bypassing L1 (the halo buffers are rewritten every other step)
__device__ __forceinline__ uint4 ld_cg16(const void* p) {
    return __ldcg(reinterpret_cast<const uint4*>(p));
}

// blockDim.x = lanes rounded up to a warp multiple, lane t owns cells [t*C, t*C + C) of every row
// of the slab.  Dynamic shared memory: [set 0: U,V,W][set 1: U,V,W][a,b,c], every array
// (R+2) rows x pitch bytes; row m of the slab holds domain row r0-1+m; a row starts with 16 bytes
// of padding so that a lane's west neighbour element of cell 0 is addressable.
template <typename T>
__global__ void __launch_bounds__(256, 1) gg_step_resident(const ResidentArgs A) {
    constexpr int C = 16 / (int)sizeof(T);
    constexpr int ES = (int)sizeof(T);
    extern __shared__ __align__(128) char smem[];
    const int nx = A.nx, ny = A.ny, R = A.R, pitch = A.pitch;
    const int ARRS = (R + 2) * pitch, SET = 3 * ARRS;
    char* coef = smem + 2 * SET;
    const int slab = blockIdx.x, nslabs = gridDim.x;
    const int sim = slab / A.slabs_per_sim, s = slab - sim * A.slabs_per_sim;
    const int r0 = s * R, r1 = min(r0 + R, ny), rows = r1 - r0;
    const int t = threadIdx.x, iown = t * C;
    const bool valid = iown < nx;
    const bool atW = iown == 0, atE = iown + C == nx;
    const size_t plane = (size_t)nx * ny;
    const StepCoef<T> k = load_coef<T>(A.coefs + sim);
    const int own = 16 + 16 * t;   // byte offset of the lane's run inside a shared-memory row

    // ---- start-up: zero everything, then load the slab (+ halo rows inside the domain)
    for (int o = t * 16; o < 2 * SET + 3 * ARRS; o += blockDim.x * 16)
        *reinterpret_cast<uint4*>(smem + o) = make_uint4(0u, 0u, 0u, 0u);
    __syncthreads();
    if (valid) {
        const T* gs[3] = {(const T*)A.U0 + sim * plane, (const T*)A.V0 + sim * plane, (const T*)A.W0 + sim * plane};
        const T* gc[3] = {(const T*)A.a, (const T*)A.b, (const T*)A.c};
        for (int m = 0; m < rows + 2; ++m) {
            const int j = r0 - 1 + m;
            if (j < 0 || j >= ny) continue;
            for (int f = 0; f < 3; ++f) {
                *reinterpret_cast<uint4*>(smem + f * ARRS + m * pitch + own) =
                    *reinterpret_cast<const uint4*>(gs[f] + (size_t)j * nx + iown);
                *reinterpret_cast<uint4*>(coef + f * ARRS + m * pitch + own) =
                    *reinterpret_cast<const uint4*>(gc[f] + (size_t)j * nx + iown);
            }
        }
    }
    __syncthreads();

    T* halo = (T*)A.halo;
    auto halo_row = [&](int parity, int sl, int side, int f) {
        return halo + ((((size_t)parity * nslabs + sl) * 2 + side) * 3 + f) * nx;
    };

    for (long long step = 1; step <= A.nsteps; ++step) {
        const int p = (int)((step - 1) & 1);
        const char* src = smem + p * SET;
        char* dst = smem + (p ^ 1) * SET;
        const bool last = step == A.nsteps;
        const int par = (int)(step & 1);
        if (valid) {
            MarchWindow<T, C> win;
            win.clear();
            for (int m = 0; m < rows + 2; ++m) {
                // arriving row m (domain row r0-1+m): own run and the two neighbour elements
                const char* so = src + m * pitch + own;
                const char* co = coef + m * pitch + own;
                T* sd[3] = {win.mN, win.vN, win.wN};      // mN: raw U first, then M = 1 - U
#pragma unroll
                for (int f = 0; f < 3; ++f) {
                    ld_run<T, C>(so + f * ARRS, sd[f] + 1);
                    sd[f][0] = *reinterpret_cast<const T*>(so + f * ARRS - ES);
                    sd[f][C + 1] = *reinterpret_cast<const T*>(so + f * ARRS + 16);
                }
                T* cd[2] = {win.aN, win.bN};
#pragma unroll
                for (int f = 0; f < 2; ++f) {
                    ld_run<T, C>(co + f * ARRS, cd[f] + 1);
                    cd[f][0] = *reinterpret_cast<const T*>(co + f * ARRS - ES);
                    cd[f][C + 1] = *reinterpret_cast<const T*>(co + f * ARRS + 16);
                }
                ld_run<T, C>(co + 2 * ARRS, win.cN);
#pragma unroll
                for (int c = 0; c < C; ++c) win.uN[c] = win.mN[c + 1];
#pragma unroll
                for (int e = 0; e < C + 2; ++e) win.mN[e] = one_minus(win.mN[e]);
                if (atW) win.wN[0] = win.wN[1];
                if (atE) win.wN[C + 1] = win.wN[C];
#pragma unroll
                for (int c = 0; c < C; ++c) win.hN[c] = cross(win.bN[c + 1], win.wN[c + 2], win.wN[c]);
                if (m >= 1) {
                    T oU[C], oV[C], oW[C];
                    win.template advance<true>(r0 - 1 + m, ny, atW, atE, k, oU, oV, oW);
                    if (m >= 2) {                      // centre = slab row m-1 = domain row r0+m-2
                        const int j = r0 + m - 2;
                        char* o = dst + (m - 1) * pitch + own;
                        st_run<T, C>(o + 0 * ARRS, oU);
                        st_run<T, C>(o + 1 * ARRS, oV);
                        st_run<T, C>(o + 2 * ARRS, oW);
                        if (last) {
                            st_run<T, C>((char*)((T*)A.U1 + sim * plane + (size_t)j * nx + iown), oU);
                            st_run<T, C>((char*)((T*)A.V1 + sim * plane + (size_t)j * nx + iown), oV);
                            st_run<T, C>((char*)((T*)A.W1 + sim * plane + (size_t)j * nx + iown), oW);
                        } else {
                            if (j == r0) {             // bottom edge row: read by the slab below
                                st_run<T, C>((char*)(halo_row(par, slab, 0, 0) + iown), oU);
                                st_run<T, C>((char*)(halo_row(par, slab, 0, 1) + iown), oV);
                                st_run<T, C>((char*)(halo_row(par, slab, 0, 2) + iown), oW);
                            }
                            if (j == r1 - 1) {         // top edge row: read by the slab above
                                st_run<T, C>((char*)(halo_row(par, slab, 1, 0) + iown), oU);
                                st_run<T, C>((char*)(halo_row(par, slab, 1, 1) + iown), oV);
                                st_run<T, C>((char*)(halo_row(par, slab, 1, 2) + iown), oW);
                            }
                        }
                    }
                }
                win.roll();
            }
        }
        if (last) break;
        __syncthreads();   // the pong copy and this step's edge rows are written
        if (t == 0) {
            __threadfence();   // (measured: faster than leaving the whole flush to the release)
            st_release_gpu(A.flags + slab, A.epoch + (unsigned int)step);
        }
        // wait for the neighbours' edge rows of this step (same simulation only)
        const int waiter = blockDim.x > 32 ? 32 : 1;
        if ((t == 0 && s > 0) || (t == waiter && s + 1 < A.slabs_per_sim)) {
            const unsigned int* f = A.flags + (t == 0 ? slab - 1 : slab + 1);
            const unsigned int want = A.epoch + (unsigned int)step;
            for (unsigned int spins = 0; (int)(ld_acquire_gpu(f) - want) < 0; ++spins)
                if (spins > (1u << 24)) __trap();
        }
        __syncthreads();
        if (valid) {
            if (s > 0)
                for (int f = 0; f < 3; ++f)
                    *reinterpret_cast<uint4*>(dst + f * ARRS + own) = ld_cg16(halo_row(par, slab - 1, 1, f) + iown);
            if (s + 1 < A.slabs_per_sim)
                for (int f = 0; f < 3; ++f)
                    *reinterpret_cast<uint4*>(dst + f * ARRS + (rows + 1) * pitch + own) =
                        ld_cg16(halo_row(par, slab + 1, 0, f) + iown);
        }
        __syncthreads();
    }
}

}  // namespace gg

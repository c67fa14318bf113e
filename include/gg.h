/* gg.h -- C ABI of libgg.so: the explicit finite-volume step of the anisotropic, heterogeneous
 * Gatenby-Gawlinski model (Mascia, Pera, Simeoni, arXiv 2006.01748) on one B200 (sm_100a).
 *
 * What the library computes (citations are lines of /root/reference/PAPER.md):
 *   eq. (1)  PAPER.md:35     U_t = U(1-U) - d U W
 *                            V_t = r V(1-V) + alpha div((1-U) grad V)
 *                            W_t = c (V - W) + div(A grad W),   A = [[a,b],[b,c]]  (eq. (2), :40)
 *   eq. (3)  PAPER.md:74     explicit Euler in time, every right-hand side at time level k;
 *   Table 1  PAPER.md:81-85  five-point stencil D1(V;U), face diffusivity 1 - mean of adjacent U;
 *   Table 2  PAPER.md:89-92  nine-point stencil D2(W;A), face means of a (x) and c (y), corner
 *                            weights +-(b_{i+-1,j} + b_{i,j+-1})/(4 dx dy);
 *   Neumann boundaries (no formula printed): DESIGN.md reading A2 -- mirror
 *   extension across every boundary face with U,V,W,a,c even and b odd, i.e. zero total normal
 *   flux through every boundary face and clamped neighbours in tangential differences.
 * The kernels evaluate the stencils in flux form (each face flux once); the
 * result equals the tables' up to floating-point evaluation order.  No clamping, no positivity
 * fix, no NaN repair anywhere (eq. (3) has none).  No stability policing: dt is the caller's.
 *
 * The paper overloads `c`: gg_create's `c` is the reaction rate of eq. (1) (called c_r in
 * DESIGN.md), gg_set_tensor's `c` is the tensor entry c(x,y) of eq. (2) (c_T).
 *
 * Layout.  Every field is row-major [ny][nx], x (index i) fastest: element (i,j) at j*nx + i;
 * "right" is (i+1,j), "upper" is (i,j+1).  Batched states are [nbatch][ny][nx].
 * Element type is the context's dtype (GG_F64: double, GG_F32: float) for state AND tensor.
 * The nx x ny cells tile [0, nx*h] x [0, ny*h]; the domain boundary lies on cell faces.
 *
 * Memory.  The library never allocates device memory.  The caller allocates
 * gg_workspace_bytes() bytes of device memory (256-byte aligned; a torch uint8 tensor will do)
 * and hands it over with gg_bind; it must stay alive until gg_destroy.  All array arguments
 * marked DEVICE are device pointers on the current CUDA device; HOST are host pointers.  The
 * caller keeps ownership of every array it passes; the library copies in/out of its workspace.
 * (One call, gg_diagnostics_noalloc, takes no workspace: its small scratch is a fixed array inside
 * the library's own device image -- see there.)
 *
 * Streams.  Every call enqueues on the stream given to gg_bind (a cudaStream_t cast to void*,
 * NULL = the legacy default stream) and returns without synchronising, except gg_destroy,
 * gg_set_state_host/gg_get_state_host/gg_set_tensor_host (which synchronise that stream) and
 * gg_last_step_ms.  Calls on one context must not be issued concurrently from several threads.
 *
 * Errors.  Every entry point returns GG_OK or an error code; nothing throws or aborts across the
 * ABI.  gg_last_error gives a context-owned message for the last failing call (never freed by
 * the caller; valid until the next call on that context).
 */
#ifndef GG_H_
#define GG_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gg_ctx gg_ctx; /* opaque; one per simulation or per batch of simulations */

enum { GG_F64 = 0, GG_F32 = 1 }; /* storage AND arithmetic type of state and tensor arrays */

enum {
    GG_OK = 0,
    GG_ERR_ARG = 1,         /* null pointer, bad size, non-finite / non-positive h or dt, n < 0 */
    GG_ERR_STATE = 2,       /* call order: step/get before bind + set_tensor + set_state */
    GG_ERR_CUDA = 3,        /* CUDA runtime / driver failure; text in gg_last_error */
    GG_ERR_UNSUPPORTED = 4  /* unknown dtype or option */
};

/* Kernel selection for gg_set_option(GG_OPT_KERNEL, .).  AUTO picks the fastest path that the
 * shape allows; every path computes the same scheme. */
enum {
    GG_KERNEL_AUTO = 0,
    GG_KERNEL_GENERIC = 1,  /* one thread per cell, global memory, clamp-indexed (any nx, ny)   */
    GG_KERNEL_STREAM = 2,   /* TMA-staged shared-memory row ring, register-rolling y march;     */
                            /* needs nx*sizeof(elem) % 16 == 0                                  */
    GG_KERNEL_STREAM2 = 3,  /* as STREAM with two time steps fused per launch (temporal block)  */
    GG_KERNEL_RESIDENT = 4, /* all n steps of a call in ONE launch, state resident in shared     */
                            /* memory: one thread-block cluster per simulation with halo rows    */
                            /* through distributed shared memory where a simulation fits one     */
                            /* (gg_cluster.cuh), else row slabs over the whole GPU exchanging    */
                            /* edge rows point-to-point (cooperative launch; at most 148 slabs   */
                            /* with rows <= 4096 B; gg_resident.cuh).  AUTO uses it for calls of */
                            /* >= 4 (cluster) resp. >= 8 (slabs) steps, STREAM2 for shorter ones */
    GG_KERNEL_PAIR = 5,     /* two time steps per launch chained in REGISTERS, x-neighbours by  */
                            /* warp shuffle (gg_pair.cuh); needs nx*sizeof(elem) % 16 == 0      */
    GG_KERNEL_QUAD = 6      /* FOUR time steps per launch: two register-chained pair marches    */
                            /* linked by one shared-memory ring (gg_quad.cuh); same shape rule  */
};
enum {
    GG_OPT_KERNEL = 0,      /* one of GG_KERNEL_*                                               */
    GG_OPT_GRAPH = 1,       /* 1 (default): step loop replayed from a cached CUDA graph; 0: plain launches */
    GG_OPT_GRAPH_CHUNK = 2  /* steps per captured graph (default 64)                            */
    /* option numbers >= 3 are tuning knobs (which compiled build, warps per CTA, ...); they are
     * declared in the library's non-installed csrc/gg_tuning.h and are not part of this interface */
};

/* One simulation.  nx, ny >= 2 cells; h > 0 the mesh size (dx = dy = h);
 * r, d, alpha, c the scalars of eq. (1); dtype GG_F64 or GG_F32.
 * On success *out owns host-side resources only; free with gg_destroy. */
int gg_create(gg_ctx** out, int nx, int ny, double h, double r, double d, double alpha, double c,
              int dtype);

/* nbatch >= 1 independent simulations on the same grid and the same tensor field, advanced
 * together by every gg_step (the paper's "fast comparative simulations").
 * r, d, alpha, c: HOST arrays [nbatch], copied. */
int gg_create_batch(gg_ctx** out, int nbatch, int nx, int ny, double h, const double* r,
                    const double* d, const double* alpha, const double* c, int dtype);

/* The general mesh of the paper: distinct mesh sizes dx, dy > 0 ("x_i = i dx, y_j = j dy",
 * PAPER.md:58; Tables 1-2 carry 1/dx^2, 1/dy^2 and 1/(4 dx dy) separately), any
 * nbatch >= 1.  gg_create / gg_create_batch are this call with dx = dy = h.  The cells tile
 * [0, nx*dx] x [0, ny*dy].  r, d, alpha, c: HOST arrays [nbatch], copied. */
int gg_create_xy(gg_ctx** out, int nbatch, int nx, int ny, double dx, double dy, const double* r,
                 const double* d, const double* alpha, const double* c, int dtype);

/* Bytes of device memory the context needs: two copies of the state (ping-pong), one of the
 * tensor, the per-simulation scalars, reduction scratch, plus alignment padding.  0 if ctx is NULL. */
size_t gg_workspace_bytes(const gg_ctx* ctx);

/* Hand over caller-owned DEVICE memory (>= gg_workspace_bytes, 256-byte aligned) and the stream
 * all later calls enqueue on.  Must be called once, before any set/step/get. */
int gg_bind(gg_ctx* ctx, void* dev_workspace, size_t bytes, void* cuda_stream);

/* Tensor field of eq. (2): a, b, c DEVICE arrays [ny][nx] of the context's dtype, cell-indexed
 * like the unknowns; copied into the workspace.  Positive definiteness
 * is assumed, not checked. */
int gg_set_tensor(gg_ctx* ctx, const void* a, const void* b, const void* c);

/* State at the current time level: U, V, W DEVICE arrays [nbatch][ny][nx]; copied. */
int gg_set_state(gg_ctx* ctx, const void* U, const void* V, const void* W);

/* n >= 0 explicit Euler steps of eq. (3) with constant step dt > 0.  All
 * three fields advance together from time-k data only.  n == 0 is a no-op.  dt is handed to the
 * device in front of the step loop and is not part of any cached graph: a new dt on every call
 * (the paper's host loop) re-captures nothing.  If the call fails with GG_ERR_CUDA after
 * its first launch, state and clock no longer describe one time level: the context drops its state
 * (later step/get calls return GG_ERR_STATE) until gg_set_state loads one again. */
int gg_step(gg_ctx* ctx, long long n, double dt);

/* n >= 0 steps with the NON-UNIFORM step size dt_k of PAPER.md:62 ("computed after each iteration
 * ... to ensure numerical stability"), re-evaluated ON THE DEVICE every `every_k` >= 1 steps with
 * no host round trip (the paper's steps 3-4, download the results and let the
 * CPU compute dt_k).  The paper prints no formula; reading A6 is used:
 *     dt_k = safety * min(dx,dy)^2 / max( lambda_max(A),  max_s alpha_s * max_ij (1 - U^k_s,ij) ),
 * lambda_max(A) as in gg_max_stable_dt (cached by gg_set_tensor), alpha (1 - U) the largest
 * diffusivity of the V equation at time level k (eq. (1)); one dt_k for the whole
 * batch, held for the every_k steps that follow (the last group may be shorter).  safety > 0.
 * The reductions are exact (max / min), so dt_k is a deterministic function of the stored state.
 * GG_KERNEL_RESIDENT cannot change dt inside its single launch: GG_ERR_UNSUPPORTED if it was
 * selected explicitly (AUTO runs STREAM2 on such grids instead).  Enqueues and returns.
 * The rule bounds the two DIFFUSION operators only; it knows nothing of the reaction terms
 * (d W dt, r dt, c dt of eq. (1)), whose stiffness is the caller's to cover with `safety`.
 * When the rule has no positive finite bound (a zero tensor with alpha == 0 or U >= 1 everywhere, a
 * non-finite tensor entry, no finite U) the device does not fold inf or NaN into the step: the
 * steps of that group run with dt = 0 (state and simulated time stay put, the step count still
 * advances), and the next gg_get_clock returns GG_ERR_ARG with the details; from then on gg_step
 * and gg_step_adaptive refuse the context until gg_set_state.  (The call itself cannot report it:
 * it returns before the device has evaluated anything.) */
int gg_step_adaptive(gg_ctx* ctx, long long n, double safety, long long every_k);

/* The device-side clock: simulated time (the sum of the step sizes of all steps since the last
 * gg_set_state), the step size of the most recent step, and the number of steps since
 * gg_set_state.  Any of the three pointers may be NULL.  Synchronises the bound stream.  Returns
 * GG_ERR_ARG (after filling the outputs) if a gg_step_adaptive since the last gg_set_state found
 * no usable step size -- see there. */
int gg_get_clock(gg_ctx* ctx, double* time, double* dt, long long* steps);

/* Copy the current state (after every step issued so far) into DEVICE arrays [nbatch][ny][nx]. */
int gg_get_state(gg_ctx* ctx, void* U, void* V, void* W);

/* Host-buffer variants: the same calls with HOST arrays; the host<->device copies run on the
 * bound stream and the call returns after they completed.  Pinned host memory copies fastest. */
int gg_set_tensor_host(gg_ctx* ctx, const void* a, const void* b, const void* c);
int gg_set_state_host(gg_ctx* ctx, const void* U, const void* V, const void* W);
int gg_get_state_host(gg_ctx* ctx, void* U, void* V, void* W);

/* Diagnostics of the current state, reduced on the device (no gg_get_state): the quantities the
 * paper's experiments read off the fields -- tumour and acid mass, the interstitial gap between
 * the fronts where both cell densities are ~0 -- plus the extrema that expose
 * the scheme's known over/undershoots for b != 0.  out: HOST array
 * [nbatch][GG_DIAG_COUNT] of doubles, slot order GG_DIAG_*: plain sums over cells (multiply by
 * dx*dy for masses), cell counts as doubles.  eps >= 0 is the gap threshold.  Accumulation is in
 * double in a fixed order (deterministic).  Synchronises the bound stream. */
enum {
    GG_DIAG_SUM_U = 0,   /* sum_ij U                                   */
    GG_DIAG_SUM_V = 1,   /* sum_ij V                                   */
    GG_DIAG_SUM_W = 2,   /* sum_ij W                                   */
    GG_DIAG_GAP = 3,     /* #{(i,j): U < eps and V < eps}              */
    GG_DIAG_TUMOUR = 4,  /* #{(i,j): V >= 1/2}                         */
    GG_DIAG_MIN_W = 5,   /* min W (negative: undershoot, reading A7)   */
    GG_DIAG_MAX_U = 6,   /* max U (> 1: overshoot)                     */
    GG_DIAG_MAX_W = 7,   /* max W                                      */
    GG_DIAG_NONFINITE = 8, /* #{(i,j): U, V or W is NaN or +-Inf} (min/max skip NaNs) */
    GG_DIAG_COUNT = 9
};
int gg_diagnostics(gg_ctx* ctx, double eps, double* out);

/* The same nine diagnostics for a caller that has NO context, NO workspace and NO way to allocate
 * one.  gg_diagnostics needs a context bound to caller-allocated device memory; a monitoring hook
 * that some other program's time loop hands bare device pointers to (an in-situ probe, a plug-in
 * of an application whose memory pool already owns the whole GPU) has no allocator to ask, and a
 * cudaMalloc of its own may fail or, where it works, synchronises the device and stalls the loop
 * it is watching.  This call allocates nothing, on the host side of the API or the device side:
 * no cudaMalloc / cudaFree / allocating library routine.  Its per-block partial results live in a
 * fixed 1.3 MiB array that is part of libgg.so's device image, present on every GPU that loads
 * the library for the life of the process (csrc/gg_noalloc.cu).
 *   U, V, W   DEVICE arrays [nbatch][ny][nx] of `dtype` (GG_F64 / GG_F32) on the current device,
 *             element-aligned (16-byte alignment enables the wide loads); read only;
 *   nbatch    1 .. GG_NOALLOC_MAX_BATCH -- the built-in array is sized for that many simulations;
 *             more is refused with GG_ERR_ARG (split the batch, or use gg_diagnostics).  nx, ny >= 1,
 *             any size;
 *   eps       gap threshold, finite and >= 0;
 *   out       DEVICE array [nbatch][GG_DIAG_COUNT] of doubles, slot order GG_DIAG_*, written by the
 *             kernel; the caller owns it and reads it after ordering with `cuda_stream`;
 *   cuda_stream  a cudaStream_t cast to void* (NULL = legacy default stream).  The call enqueues
 *             one memset of a few counters and ONE kernel on it and returns without synchronising.
 * Values: the sums are accumulated in double in a fixed order (deterministic from call to call);
 * they agree with gg_diagnostics to summation order (~1e-15 relative), counts and extrema exactly.
 * Sharing: every call on a GPU uses the same built-in array.  Calls on one stream are safe (the
 * stream orders them; nothing is carried from one call to the next -- the counters are re-zeroed
 * by every call).  Calls that may OVERLAP on the GPU (different streams or threads) race on it and
 * give wrong results: order them yourself.
 * First call on each GPU: looks up the array's device address and makes the runtime load the
 * library's kernels there; make it once with that GPU current, outside any stream capture.
 * Errors: GG_OK or a code; the message is per host thread, from gg_noalloc_last_error(). */
enum { GG_NOALLOC_MAX_BATCH = 64 };
int gg_diagnostics_noalloc(const void* U, const void* V, const void* W, int nbatch, int nx, int ny,
                           int dtype, double eps, double* out, void* cuda_stream);
const char* gg_noalloc_last_error(void);

/* Front position along a grid line (the paper reads the tumour and acid fronts and the gap between
 * them off the fields): for every simulation the first and the last cell index
 * along row `index` (axis 0: the line runs along x) or column `index` (axis 1: along y) where
 * field `field` (0 = U, 1 = V, 2 = W) is >= level; (-1, -1) if no cell qualifies.  out: HOST array
 * [nbatch][2] of int.  The comparison is made on the stored values converted exactly to double.
 * Synchronises the bound stream. */
int gg_front(gg_ctx* ctx, int field, int axis, int index, double level, int* out);

/* Step-size bound for the explicit scheme (PAPER.md:62, :79, :128 say the host recomputes dt "to
 * ensure numerical stability" and print no formula; reading A6 is used):
 *     *dt = safety * min(dx,dy)^2 / max(max_s alpha_s, lambda_max),
 * lambda_max = max over cells of the larger eigenvalue of [[a,b],[b,c]] (eq. (2)),
 * reduced on the device by gg_set_tensor and cached there (this call reads 8 bytes back).  safety <= 1/4 keeps the linear
 * part L2-stable (max |symbol| <= 8 lambda_max / h^2); BASELINE.json's workloads use 0.2.
 * lambda_max may be NULL.  Synchronises the bound stream. */
int gg_max_stable_dt(gg_ctx* ctx, double safety, double* dt, double* lambda_max);

/* Tuning / path selection; see GG_OPT_*.  Returns GG_ERR_UNSUPPORTED for an unknown option or a
 * kernel the context's shape cannot run (the selection is never silently downgraded). */
int gg_set_option(gg_ctx* ctx, int option, long long value);

/* Introspection for benchmarks and tests.
 * gg_kernel_used: GG_KERNEL_* the next gg_step will run (resolves AUTO), or -1.
 * gg_launches:    number of step kernels this context has launched so far (graph replays count
 *                 every kernel node; a STREAM2 / PAIR launch advances two steps, a QUAD launch
 *                 four, a RESIDENT launch all n steps of its gg_step call).
 * gg_graph_captures: number of CUDA graphs this context has captured and instantiated so far (a
 *                 graph is keyed by length, ping-pong parity, kernel and every_k -- never by dt).
 * gg_last_step_ms: device time of the most recent gg_step call, measured with CUDA events
 *                 recorded on the bound stream around its launches; synchronises on the end
 *                 event.  *ms < 0 if no step has run. */
int gg_kernel_used(const gg_ctx* ctx);
/* Name of the kernel instantiation behind gg_kernel_used, as a profiler prints it, e.g.
 * "gg_step_quad<double,4,2,2,2,4>" (context-owned; "" before the first gg_step built its plan). */
const char* gg_kernel_name(const gg_ctx* ctx);
long long gg_launches(const gg_ctx* ctx);
long long gg_graph_captures(const gg_ctx* ctx);
int gg_last_step_ms(gg_ctx* ctx, float* ms);

/* Synchronises the bound stream, releases graphs and host resources.  The workspace stays the
 * caller's.  gg_destroy(NULL) is GG_OK. */
int gg_destroy(gg_ctx* ctx);

/* Message of the last failing call on ctx ("" if none); for ctx == NULL, the message of the
 * last failing gg_create* on this thread. */
const char* gg_last_error(const gg_ctx* ctx);

/* Library version string, e.g. "gg-b200 0.2 sm_100a". */
const char* gg_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GG_H_ */

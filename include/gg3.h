/* gg3.h -- C ABI of libgg.so for the THREE-DIMENSIONAL extension of the explicit finite-volume step
 * of the anisotropic, heterogeneous Gatenby-Gawlinski model (arXiv 2006.01748).
 *
 * The paper names three-dimensional modelling as the direction its CUDA work is heading
 * and prints no 3-D scheme.  This interface advances the construction of eq. (3)
 * and Tables 1-2 taken one dimension up (reading A13): on an
 * nx x ny x nz Cartesian cell grid with spacings dx, dy, dz and Neumann boundaries,
 *
 *     U' = U + dt U (1-U) - d dt U W
 *     V' = V + r dt V (1-V) + alpha dt D1(V;U)      D1: seven-point stencil, Table 1 plus the z faces
 *     W' = W + c dt (V-W)   + dt D2(W;A)            D2: nineteen-point stencil for div(A grad W),
 *
 * A = [[axx,axy,axz],[axy,ayy,ayz],[axz,ayz,azz]] symmetric, heterogeneous, cell-indexed: Table 2's
 * face entries with the diagonal entry of each direction and Table 2's four corner entries in each
 * of the three coordinate planes with that plane's off-diagonal entry.  Every right-hand side at
 * time level k.  Boundaries: zero normal flux through every boundary face (mirror extension;
 * an off-diagonal entry a_pq is odd across the faces normal to p or q).  No clamping, no
 * positivity fix, no stability policing: dt is the caller's.
 *
 * Layout.  Every field is [nz][ny][nx], x (index i) fastest: element (i,j,k) at (k*ny + j)*nx + i.
 * Element type is the context's dtype (GG_F64 = 0: double, GG_F32 = 1: float) for state AND tensor.
 *
 * Memory, streams, errors: as in gg.h.  The caller allocates gg3_workspace_bytes() bytes of device
 * memory (256-byte aligned) and hands it over with gg3_bind; the library never allocates device
 * memory.  DEVICE arguments are device pointers, HOST arguments host pointers; the caller keeps
 * every array it passes.  Every call enqueues on the stream given to gg3_bind; only the *_host
 * calls, gg3_last_step_ms and gg3_destroy synchronise.  Every function returns GG_OK (0) or a
 * GG_ERR_* code of gg.h and never throws or aborts; gg3_last_error gives the message of the last
 * failure of that context.
 */
#ifndef GG3_H_
#define GG3_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gg3_ctx gg3_ctx;

/* step kernels (GG3_OPT_KERNEL) */
enum {
    GG3_KERNEL_AUTO = 0,     /* TILED where the shape allows it, else GENERIC                        */
    GG3_KERNEL_GENERIC = 1,  /* one thread per cell, global memory, clamp-indexed: any shape         */
    GG3_KERNEL_TILED = 2     /* xy tiles marched along z, planes staged in shared memory             */
};
enum {
    GG3_OPT_KERNEL = 0,      /* one of GG3_KERNEL_*                                                   */
    GG3_OPT_GRAPH = 1,       /* 1 (default): gg3_step replays cached CUDA graphs of up to              */
                             /* GG3_OPT_GRAPH_CHUNK launches (keyed by length, ping-pong parity, kernel */
                             /* and dt); 0: one host launch per step                                   */
    GG3_OPT_GRAPH_CHUNK = 2  /* launches per captured graph (default 64, 1..4096)                      */
};

/* One simulation on an nx x ny x nz grid (each >= 2), spacings dx, dy, dz > 0; r, d, alpha, c: the
 * scalars of eq. (1) (c is the reaction rate the paper calls c).  They must be finite;
 * their signs are not policed (as in gg_create: a negative rate is the caller's business).  HOST call.
 * The message of a failed gg3_create is per host thread (gg3_last_error(NULL)).
 *
 * Step size.  This interface has no gg3_max_stable_dt (and no device-side clock, diagnostics or
 * batching: those exist for the 2-D path, gg.h).  dt is the caller's; for the linear part of the
 * scheme the explicit bound in three dimensions is
 *     dt <= safety * min(dx,dy,dz)^2 / max(alpha, lambda_max(A)),   safety <= 1/6
 * (2-D: 1/4), lambda_max the largest eigenvalue of A over all cells -- a Gershgorin row sum
 * max_p (a_pp + sum_{q != p} |a_pq|) is a safe stand-in.  The seeded recipe
 * (paper_2006_01748_b200/workloads.py: dt_rule3) uses that row sum with safety 0.12. */
int gg3_create(gg3_ctx** out, int nx, int ny, int nz, double dx, double dy, double dz, double r,
               double d, double alpha, double c, int dtype);

/* Device bytes the context needs: two copies of the state (ping-pong) and the six stored tensor
 * fields, plus alignment padding.  0 if ctx is NULL. */
size_t gg3_workspace_bytes(const gg3_ctx* ctx);

/* Hand over caller-owned DEVICE memory (>= gg3_workspace_bytes, 256-byte aligned) and the stream
 * (a cudaStream_t cast to void*, NULL = the default stream) all later calls enqueue on. */
int gg3_bind(gg3_ctx* ctx, void* dev_workspace, size_t bytes, void* cuda_stream);

/* The tensor of div(A grad W): six DEVICE (resp. HOST) arrays [nz][ny][nx] in the order axx, ayy,
 * azz, axy, axz, ayz, copied and converted to the stored form (face coefficients and pre-scaled
 * off-diagonals).  Positive definiteness is the caller's business. */
int gg3_set_tensor(gg3_ctx* ctx, const void* axx, const void* ayy, const void* azz, const void* axy,
                   const void* axz, const void* ayz);
int gg3_set_tensor_host(gg3_ctx* ctx, const void* axx, const void* ayy, const void* azz,
                        const void* axy, const void* axz, const void* ayz);

/* State at the current time level: DEVICE (resp. HOST) arrays [nz][ny][nx], copied. */
int gg3_set_state(gg3_ctx* ctx, const void* U, const void* V, const void* W);
int gg3_set_state_host(gg3_ctx* ctx, const void* U, const void* V, const void* W);

/* n >= 0 explicit Euler steps of eq. (3) in three dimensions with step size dt > 0 (finite).  If the
 * call fails with GG_ERR_CUDA after its first launch the context drops its state (gg3_set_state
 * again). */
int gg3_step(gg3_ctx* ctx, long long n, double dt);

/* Copy the current state out: DEVICE (resp. HOST, synchronising) arrays [nz][ny][nx]. */
int gg3_get_state(gg3_ctx* ctx, void* U, void* V, void* W);
int gg3_get_state_host(gg3_ctx* ctx, void* U, void* V, void* W);

int gg3_set_option(gg3_ctx* ctx, int option, long long value);
/* The kernel gg3_step runs for this context (a GG3_KERNEL_* value other than AUTO). */
int gg3_kernel_used(const gg3_ctx* ctx);
/* Kernel launches enqueued by gg3_step so far (graph replays count every kernel node). */
long long gg3_launches(const gg3_ctx* ctx);
/* CUDA graphs this context has captured so far (a loop with a fixed dt captures each chunk length
 * and parity once; a new dt captures anew: the 3-D kernels take their coefficients by value). */
long long gg3_graph_captures(const gg3_ctx* ctx);
/* Device time of the last gg3_step call in milliseconds (CUDA events on the bound stream);
 * synchronises on the second event. */
int gg3_last_step_ms(gg3_ctx* ctx, float* ms);

int gg3_destroy(gg3_ctx* ctx);
const char* gg3_last_error(const gg3_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* GG3_H_ */

// gg3_api.cu -- host side of the three-dimensional extension: the C ABI of include/gg3.h.
// Second translation unit of libgg.so (paper_2006_01748_b200/build.py).  Product code.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <algorithm>
#include <cstdio>
#include <cstring>
#include <map>
#include <new>
#include <string>
#include <tuple>

#include "../../include/gg.h"
#include "../../include/gg3.h"
#include "gg3_kernels.cuh"
#include "gg3_tiled.cuh"

// A captured run of gg3_step launches.  The 3-D kernels take their folded coefficients BY VALUE
// (Args3::k), so unlike the 2-D graphs these are keyed by dt as well (its bit pattern).
struct Graph3Key {
    long long len;
    int parity, kernel;
    unsigned long long dt_bits;
    bool operator<(const Graph3Key& o) const {
        return std::tie(len, parity, kernel, dt_bits) < std::tie(o.len, o.parity, o.kernel, o.dt_bits);
    }
};

struct gg3_ctx {
    int nx = 0, ny = 0, nz = 0, dtype = GG_F64;
    double dx = 1, dy = 1, dz = 1, r = 0, d = 0, alpha = 0, c_r = 0;
    char* ws = nullptr;
    size_t ws_bytes = 0;
    cudaStream_t stream = nullptr;
    void* state[2][3] = {};
    void* tens[6] = {};          // fx, fy, fz, gxy, gxz, gyz
    int cur = 0;
    bool bound = false, have_tensor = false, have_state = false, timed = false;
    int opt_kernel = GG3_KERNEL_AUTO;
    int opt_graph = 1;           // GG3_OPT_GRAPH
    long long opt_chunk = 64;    // GG3_OPT_GRAPH_CHUNK
    std::map<Graph3Key, cudaGraphExec_t> graphs;
    long long graph_captures = 0;
    int num_sms = 148;           // of the device current at gg3_bind (sizes the grids)
    long long launches = 0;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    mutable std::string err;
    size_t esize() const { return dtype == GG_F64 ? 8 : 4; }
    size_t cells() const { return (size_t)nx * ny * nz; }
};

namespace {

thread_local std::string g3_create_error;   // per thread, like gg_api.cu's: concurrent failing gg3_create calls do not race

int fail3(const gg3_ctx* c, int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    try { if (c) c->err = buf; else g3_create_error = buf; } catch (...) {}
    return code;
}

#define GG3_CUDA(c, call)                                                                    \
    do {                                                                                     \
        cudaError_t e_ = (call);                                                             \
        if (e_ != cudaSuccess)                                                               \
            return fail3((c), GG_ERR_CUDA, "%s: %s (%s:%d)", #call, cudaGetErrorString(e_),  \
                         __FILE__, __LINE__);                                                \
    } while (0)

size_t align256(size_t x) { return (x + 255) / 256 * 256; }
size_t array_bytes(const gg3_ctx* c) { return align256(c->cells() * c->esize()); }

int resolve3(const gg3_ctx* c) {
    if (c->opt_kernel != GG3_KERNEL_AUTO) return c->opt_kernel;
    return gg3::tiled_shape_ok(c->nx, c->ny, c->nz) ? GG3_KERNEL_TILED : GG3_KERNEL_GENERIC;
}

template <typename T>
gg3::Args3<T> make_args(const gg3_ctx* c, int src, double dt) {
    gg3::Args3<T> a;
    a.U = (const T*)c->state[src][0]; a.V = (const T*)c->state[src][1]; a.W = (const T*)c->state[src][2];
    a.U1 = (T*)c->state[src ^ 1][0]; a.V1 = (T*)c->state[src ^ 1][1]; a.W1 = (T*)c->state[src ^ 1][2];
    a.fx = (const T*)c->tens[0]; a.fy = (const T*)c->tens[1]; a.fz = (const T*)c->tens[2];
    a.gxy = (const T*)c->tens[3]; a.gxz = (const T*)c->tens[4]; a.gyz = (const T*)c->tens[5];
    // scalars folded in double and rounded once to the arithmetic type
    a.k.dt = (T)dt; a.k.ddt = (T)(c->d * dt); a.k.rdt = (T)(c->r * dt); a.k.crdt = (T)(c->c_r * dt);
    a.k.adx = (T)(0.5 * c->alpha * dt / (c->dx * c->dx));
    a.k.ady = (T)(0.5 * c->alpha * dt / (c->dy * c->dy));
    a.k.adz = (T)(0.5 * c->alpha * dt / (c->dz * c->dz));
    a.nx = c->nx; a.ny = c->ny; a.nz = c->nz;
    return a;
}

template <typename T>
int launch_step(gg3_ctx* c, int kernel, int src, double dt) {
    const gg3::Args3<T> a = make_args<T>(c, src, dt);
    if (kernel == GG3_KERNEL_TILED) {
        const dim3 block(gg3::kTileX, gg3::kTileY);
        const dim3 grid((c->nx + gg3::kTileX - 1) / gg3::kTileX, (c->ny + gg3::kTileY - 1) / gg3::kTileY,
                        gg3::tiled_zchunks(c->nx, c->ny, c->nz, c->num_sms));
        gg3::gg3_step_tiled<T><<<grid, block, gg3::tiled_smem_bytes<T>(), c->stream>>>(a);
    } else {
        const dim3 block(32, 4, 2);
        const dim3 grid((c->nx + 31) / 32, (c->ny + 3) / 4, (c->nz + 1) / 2);
        gg3::gg3_step_generic<T><<<grid, block, 0, c->stream>>>(a);
    }
    GG3_CUDA(c, cudaGetLastError());
    return GG_OK;
}

void drop_graphs3(gg3_ctx* c) {
    for (auto& kv : c->graphs) cudaGraphExecDestroy(kv.second);
    c->graphs.clear();
}

// `len` plain launches from copy `src` on c->stream (ping-pong); the caller flips c->cur.
int enqueue_steps3(gg3_ctx* c, int kernel, int src, long long len, double dt) {
    for (long long s = 0; s < len; ++s, src ^= 1) {
        const int rc = c->dtype == GG_F64 ? launch_step<double>(c, kernel, src, dt) : launch_step<float>(c, kernel, src, dt);
        if (rc) return rc;
    }
    return GG_OK;
}

// Capture `len` steps starting at copy `src` into an executable graph (on a private capture stream;
// thread-local capture mode, so other threads' CUDA calls are not disturbed).
int capture_graph3(gg3_ctx* c, int kernel, int src, long long len, double dt, cudaGraphExec_t* out) {
    cudaStream_t cap = nullptr;
    GG3_CUDA(c, cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
    cudaStream_t user = c->stream;
    c->stream = cap;
    cudaGraph_t graph = nullptr;
    int rc = GG_OK;
    cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) {
        rc = fail3(c, GG_ERR_CUDA, "cudaStreamBeginCapture: %s", cudaGetErrorString(e));
    } else {
        rc = enqueue_steps3(c, kernel, src, len, dt);
        e = cudaStreamEndCapture(cap, &graph);
        if (rc == GG_OK && e != cudaSuccess) rc = fail3(c, GG_ERR_CUDA, "cudaStreamEndCapture: %s", cudaGetErrorString(e));
    }
    c->stream = user;
    if (rc == GG_OK) {
        e = cudaGraphInstantiate(out, graph, 0);
        if (e != cudaSuccess) rc = fail3(c, GG_ERR_CUDA, "cudaGraphInstantiate: %s", cudaGetErrorString(e));
        else ++c->graph_captures;
    }
    if (graph) cudaGraphDestroy(graph);
    cudaStreamDestroy(cap);
    return rc;
}

template <typename F>
int guarded3(const gg3_ctx* c, const char* what, F&& f) {
    try {
        return f();
    } catch (const std::bad_alloc&) {
        return fail3(c, GG_ERR_ARG, "%s: out of host memory", what);
    } catch (...) {
        return fail3(c, GG_ERR_CUDA, "%s: unexpected C++ exception", what);
    }
}

}  // namespace

extern "C" {

int gg3_create(gg3_ctx** out, int nx, int ny, int nz, double dx, double dy, double dz, double r, double d,
               double alpha, double c, int dtype) {
    if (!out) return GG_ERR_ARG;
    *out = nullptr;
    return guarded3(nullptr, "gg3_create", [&]() -> int {
        if (nx < 2 || ny < 2 || nz < 2) return fail3(nullptr, GG_ERR_ARG, "gg3_create: nx, ny, nz must be >= 2");
        if ((double)nx * ny * nz > 2.0e10) return fail3(nullptr, GG_ERR_ARG, "gg3_create: grid too large");
        if (ny > 65535 * gg3::kTileY || nz > 65535) return fail3(nullptr, GG_ERR_ARG, "gg3_create: ny or nz too large");
        if (!(dx > 0) || !(dy > 0) || !(dz > 0) || !std::isfinite(dx) || !std::isfinite(dy) || !std::isfinite(dz))
            return fail3(nullptr, GG_ERR_ARG, "gg3_create: dx, dy, dz must be finite and > 0");
        if (!std::isfinite(r) || !std::isfinite(d) || !std::isfinite(alpha) || !std::isfinite(c))
            return fail3(nullptr, GG_ERR_ARG, "gg3_create: non-finite parameter");
        if (dtype != GG_F64 && dtype != GG_F32) return fail3(nullptr, GG_ERR_ARG, "gg3_create: dtype must be GG_F64 or GG_F32");
        gg3_ctx* ctx = new gg3_ctx;
        ctx->nx = nx; ctx->ny = ny; ctx->nz = nz; ctx->dtype = dtype;
        ctx->dx = dx; ctx->dy = dy; ctx->dz = dz; ctx->r = r; ctx->d = d; ctx->alpha = alpha; ctx->c_r = c;
        *out = ctx;
        return GG_OK;
    });
}

size_t gg3_workspace_bytes(const gg3_ctx* ctx) { return ctx ? 12 * array_bytes(ctx) + 256 : 0; }

int gg3_bind(gg3_ctx* ctx, void* ws, size_t bytes, void* stream) {
    if (!ctx) return GG_ERR_ARG;
    if (!ws || ((size_t)ws & 255)) return fail3(ctx, GG_ERR_ARG, "gg3_bind: workspace must be non-NULL and 256-byte aligned");
    if (bytes < gg3_workspace_bytes(ctx)) return fail3(ctx, GG_ERR_ARG, "gg3_bind: workspace too small");
    if (ctx->bound) return fail3(ctx, GG_ERR_STATE, "gg3_bind: already bound");
    int dev = 0;
    GG3_CUDA(ctx, cudaGetDevice(&dev));
    GG3_CUDA(ctx, cudaDeviceGetAttribute(&ctx->num_sms, cudaDevAttrMultiProcessorCount, dev));
    ctx->ws = (char*)ws; ctx->ws_bytes = bytes; ctx->stream = (cudaStream_t)stream;
    size_t off = 0;
    for (int p = 0; p < 2; ++p)
        for (int f = 0; f < 3; ++f) { ctx->state[p][f] = ctx->ws + off; off += array_bytes(ctx); }
    for (int f = 0; f < 6; ++f) { ctx->tens[f] = ctx->ws + off; off += array_bytes(ctx); }
    GG3_CUDA(ctx, cudaEventCreate(&ctx->ev0));
    GG3_CUDA(ctx, cudaEventCreate(&ctx->ev1));
    GG3_CUDA(ctx, cudaFuncSetAttribute(gg3::gg3_step_tiled<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gg3::tiled_smem_bytes<double>()));
    GG3_CUDA(ctx, cudaFuncSetAttribute(gg3::gg3_step_tiled<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gg3::tiled_smem_bytes<float>()));
    ctx->bound = true;
    return GG_OK;
}

static int set_tensor3(gg3_ctx* ctx, const void* const src[6], bool host) {
    if (!ctx) return GG_ERR_ARG;
    if (!ctx->bound) return fail3(ctx, GG_ERR_STATE, "gg3_set_tensor: call gg3_bind first");
    for (int f = 0; f < 6; ++f)
        if (!src[f]) return fail3(ctx, GG_ERR_ARG, "gg3_set_tensor: NULL array");
    ctx->have_tensor = false;
    const size_t bytes = ctx->cells() * ctx->esize();
    // the entries as given are staged in the ping-pong copy that holds no live time level, three at
    // a time (the stored form of an entry needs its neighbour along one axis)
    void* scratch[3] = {ctx->state[ctx->cur ^ 1][0], ctx->state[ctx->cur ^ 1][1], ctx->state[ctx->cur ^ 1][2]};
    const int blocks = (int)std::min<size_t>((ctx->cells() + 255) / 256, (size_t)ctx->num_sms * 8);
    const double sc[6] = {0.5 / (ctx->dx * ctx->dx), 0.5 / (ctx->dy * ctx->dy), 0.5 / (ctx->dz * ctx->dz),
                          0.25 / (ctx->dx * ctx->dy), 0.25 / (ctx->dx * ctx->dz), 0.25 / (ctx->dy * ctx->dz)};
    for (int f = 0; f < 6; ++f) {
        GG3_CUDA(ctx, cudaMemcpyAsync(scratch[f % 3], src[f], bytes, host ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, ctx->stream));
        if (ctx->dtype == GG_F64)
            gg3::gg3_store_tensor<double><<<blocks, 256, 0, ctx->stream>>>((const double*)scratch[f % 3], (double*)ctx->tens[f], ctx->nx,
                                                                           ctx->ny, ctx->nz, f < 3 ? f : 0, f < 3 ? 0 : 1, sc[f]);
        else
            gg3::gg3_store_tensor<float><<<blocks, 256, 0, ctx->stream>>>((const float*)scratch[f % 3], (float*)ctx->tens[f], ctx->nx,
                                                                          ctx->ny, ctx->nz, f < 3 ? f : 0, f < 3 ? 0 : 1, sc[f]);
        GG3_CUDA(ctx, cudaGetLastError());
    }
    if (host) GG3_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->have_tensor = true;
    return GG_OK;
}
int gg3_set_tensor(gg3_ctx* c, const void* axx, const void* ayy, const void* azz, const void* axy, const void* axz, const void* ayz) {
    const void* s[6] = {axx, ayy, azz, axy, axz, ayz};
    return set_tensor3(c, s, false);
}
int gg3_set_tensor_host(gg3_ctx* c, const void* axx, const void* ayy, const void* azz, const void* axy, const void* axz, const void* ayz) {
    const void* s[6] = {axx, ayy, azz, axy, axz, ayz};
    return set_tensor3(c, s, true);
}

static int copy_state3(gg3_ctx* ctx, void* const dst[3], const void* const src[3], cudaMemcpyKind kind, bool sync) {
    const size_t bytes = ctx->cells() * ctx->esize();
    for (int f = 0; f < 3; ++f) GG3_CUDA(ctx, cudaMemcpyAsync(dst[f], src[f], bytes, kind, ctx->stream));
    if (sync) GG3_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return GG_OK;
}
static int set_state3(gg3_ctx* ctx, const void* U, const void* V, const void* W, bool host) {
    if (!ctx) return GG_ERR_ARG;
    if (!ctx->bound) return fail3(ctx, GG_ERR_STATE, "gg3_set_state: call gg3_bind first");
    if (!U || !V || !W) return fail3(ctx, GG_ERR_ARG, "gg3_set_state: NULL array");
    const void* src[3] = {U, V, W};
    const int rc = copy_state3(ctx, ctx->state[ctx->cur], src, host ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, host);
    if (rc) return rc;
    ctx->have_state = true;
    return GG_OK;
}
static int get_state3(gg3_ctx* ctx, void* U, void* V, void* W, bool host) {
    if (!ctx) return GG_ERR_ARG;
    if (!ctx->bound || !ctx->have_state) return fail3(ctx, GG_ERR_STATE, "gg3_get_state: no state set");
    if (!U || !V || !W) return fail3(ctx, GG_ERR_ARG, "gg3_get_state: NULL array");
    void* dst[3] = {U, V, W};
    return copy_state3(ctx, dst, ctx->state[ctx->cur], host ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, host);
}
int gg3_set_state(gg3_ctx* c, const void* U, const void* V, const void* W) { return set_state3(c, U, V, W, false); }
int gg3_set_state_host(gg3_ctx* c, const void* U, const void* V, const void* W) { return set_state3(c, U, V, W, true); }
int gg3_get_state(gg3_ctx* c, void* U, void* V, void* W) { return get_state3(c, U, V, W, false); }
int gg3_get_state_host(gg3_ctx* c, void* U, void* V, void* W) { return get_state3(c, U, V, W, true); }

int gg3_step(gg3_ctx* ctx, long long n, double dt) {
    if (!ctx) return GG_ERR_ARG;
    if (!ctx->bound || !ctx->have_tensor || !ctx->have_state)
        return fail3(ctx, GG_ERR_STATE, "gg3_step: needs gg3_bind, gg3_set_tensor and gg3_set_state first");
    if (n < 0) return fail3(ctx, GG_ERR_ARG, "gg3_step: n = %lld < 0", n);
    if (!(dt > 0.0) || !std::isfinite(dt)) return fail3(ctx, GG_ERR_ARG, "gg3_step: dt must be finite and > 0");
    if (n == 0) return GG_OK;
    const int kernel = resolve3(ctx);
    return guarded3(ctx, "gg3_step", [&]() -> int {
        GG3_CUDA(ctx, cudaEventRecord(ctx->ev0, ctx->stream));
        long long left = n;
        unsigned long long dt_bits = 0;
        std::memcpy(&dt_bits, &dt, sizeof dt_bits);
        while (left > 0) {
            // the step loop is replayed from cached graphs of up to opt_chunk launches (one host call
            // per chunk instead of one per step: small grids are launch-bound otherwise)
            const long long len = ctx->opt_graph && n >= 2 ? (left < ctx->opt_chunk ? left : ctx->opt_chunk) : left;
            int rc = GG_OK;
            if (ctx->opt_graph && n >= 2) {
                const Graph3Key key{len, ctx->cur, kernel, dt_bits};
                auto it = ctx->graphs.find(key);
                if (it == ctx->graphs.end()) {
                    if (ctx->graphs.size() >= 16) drop_graphs3(ctx);
                    cudaGraphExec_t ex = nullptr;
                    rc = capture_graph3(ctx, kernel, ctx->cur, len, dt, &ex);
                    if (rc == GG_OK) it = ctx->graphs.emplace(key, ex).first;
                }
                if (rc == GG_OK) {
                    const cudaError_t e = cudaGraphLaunch(it->second, ctx->stream);
                    if (e != cudaSuccess) rc = fail3(ctx, GG_ERR_CUDA, "cudaGraphLaunch: %s", cudaGetErrorString(e));
                }
            } else {
                rc = enqueue_steps3(ctx, kernel, ctx->cur, len, dt);
            }
            if (rc) { ctx->have_state = false; return rc; }   // some launches may be enqueued: no consistent time level
            ctx->cur ^= (int)(len & 1);
            ctx->launches += len;
            left -= len;
        }
        GG3_CUDA(ctx, cudaEventRecord(ctx->ev1, ctx->stream));
        ctx->timed = true;
        return GG_OK;
    });
}

int gg3_set_option(gg3_ctx* ctx, int option, long long value) {
    if (!ctx) return GG_ERR_ARG;
    if (option == GG3_OPT_GRAPH) {
        if (value != 0 && value != 1) return fail3(ctx, GG_ERR_ARG, "GG3_OPT_GRAPH: 0 or 1");
        ctx->opt_graph = (int)value;
        return GG_OK;
    }
    if (option == GG3_OPT_GRAPH_CHUNK) {
        if (value < 1 || value > 4096) return fail3(ctx, GG_ERR_ARG, "GG3_OPT_GRAPH_CHUNK: 1..4096");
        ctx->opt_chunk = value;
        return GG_OK;
    }
    if (option != GG3_OPT_KERNEL) return fail3(ctx, GG_ERR_UNSUPPORTED, "gg3_set_option: unknown option %d", option);
    if (value != GG3_KERNEL_AUTO && value != GG3_KERNEL_GENERIC && value != GG3_KERNEL_TILED)
        return fail3(ctx, GG_ERR_UNSUPPORTED, "gg3_set_option: kernel %lld not available", value);
    if (value == GG3_KERNEL_TILED && !gg3::tiled_shape_ok(ctx->nx, ctx->ny, ctx->nz))
        return fail3(ctx, GG_ERR_UNSUPPORTED, "gg3 tiled kernel cannot take %d x %d x %d", ctx->nx, ctx->ny, ctx->nz);
    ctx->opt_kernel = (int)value;
    return GG_OK;
}
int gg3_kernel_used(const gg3_ctx* ctx) { return ctx ? resolve3(ctx) : -1; }
long long gg3_launches(const gg3_ctx* ctx) { return ctx ? ctx->launches : 0; }
long long gg3_graph_captures(const gg3_ctx* ctx) { return ctx ? ctx->graph_captures : 0; }
int gg3_last_step_ms(gg3_ctx* ctx, float* ms) {
    if (!ctx || !ms) return GG_ERR_ARG;
    if (!ctx->timed) return fail3(ctx, GG_ERR_STATE, "gg3_last_step_ms: no gg3_step call yet");
    GG3_CUDA(ctx, cudaEventSynchronize(ctx->ev1));
    GG3_CUDA(ctx, cudaEventElapsedTime(ms, ctx->ev0, ctx->ev1));
    return GG_OK;
}
int gg3_destroy(gg3_ctx* ctx) {
    if (!ctx) return GG_OK;
    if (ctx->bound) cudaStreamSynchronize(ctx->stream);
    drop_graphs3(ctx);
    if (ctx->ev0) cudaEventDestroy(ctx->ev0);
    if (ctx->ev1) cudaEventDestroy(ctx->ev1);
    delete ctx;
    return GG_OK;
}
const char* gg3_last_error(const gg3_ctx* ctx) { return ctx ? ctx->err.c_str() : g3_create_error.c_str(); }

}  // extern "C"

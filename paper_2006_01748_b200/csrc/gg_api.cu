// gg_api.cu -- the C ABI of libgg.so (include/gg.h): context, argument validation, workspace
// carving, tensor maps, kernel dispatch and the CUDA-graph step loop.  Product code; shares
// nothing with oracle/.  Build: paper_2006_01748_b200/build.py (nvcc, sm_100a).
#include "../../include/gg.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <limits>
#include <map>
#include <new>
#include <string>
#include <tuple>
#include <vector>

#include "gg_common.cuh"
#include "gg_generic.cuh"
#include "gg_stream.cuh"
#include "gg_stream2.cuh"
#include "gg_diag.cuh"
#include "gg_pair.cuh"
#include "gg_quad.cuh"
#include "gg_dt.cuh"
#include "gg_tuning.h"
#include "gg_resident.cuh"
#include "gg_cluster.cuh"
#include "gg_inst.h"

namespace {

constexpr size_t kAlign = 256;
inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

thread_local std::string g_create_error;

// A captured graph holds step kernels only (plus, for gg_step_adaptive, the device-side dt rule):
// dt never appears in a kernel argument (gg_dt.cuh), so it is not part of the key.
struct GraphKey {
    long long len;
    int parity;
    int kernel;
    long long every_k;   // 0: fixed dt (gg_step); > 0: dt re-evaluated on the device every_k steps
    bool operator<(const GraphKey& o) const {
        return std::tie(len, parity, kernel, every_k) < std::tie(o.len, o.parity, o.kernel, o.every_k);
    }
};

}  // namespace

struct gg_ctx {
    int nx = 0, ny = 0, nbatch = 1, dtype = GG_F64;
    double dx = 0, dy = 0;
    std::vector<gg::SimScalars> sims;
    // workspace
    char* ws = nullptr;
    size_t ws_bytes = 0;
    cudaStream_t stream = nullptr;
    bool bound = false, have_tensor = false, have_state = false;
    bool rule_failed = false;   // gg_get_clock saw DevClock::bad_rule != 0; cleared by gg_set_state
    void* state[2][3] = {{nullptr, nullptr, nullptr}, {nullptr, nullptr, nullptr}};
    void* coef[3] = {nullptr, nullptr, nullptr};
    gg::SimScalars* d_sims = nullptr;
    gg::StepCoef<double>* d_coefs = nullptr;   // folded on the device from the device-side dt (gg_dt.cuh)
    gg::DevClock* d_clock = nullptr;
    double folded_dt = std::numeric_limits<double>::quiet_NaN();  // dt the device's d_coefs were folded with (NaN: unknown)
    long long graph_captures = 0;
    double* d_scratch = nullptr;
    int cur = 0;  // which ping-pong copy holds the current time level
    // options
    int opt_kernel = GG_KERNEL_AUTO;
    int opt_graph = 1;
    long long opt_chunk = 64;
    int opt_variant = 0;
    int opt_items_per_warp = 4;   // work items per resident CTA
    int opt_warps = 0;            // warps (strips) per CTA; 0 = from the grid width
    // stream-kernel plan (tensor maps etc.)
    gg::StreamPlan plan, plan2;   // single-step and two-step stream kernels
    bool plan_ready = false, plan2_ready = false;
    // register-chained two-step kernel (gg_pair.cuh)
    struct PairPlan {
        CUtensorMap state[2][3], coef[3];
        int nw = 0, ntilecols = 0, nchunks = 0, chunk_rows = 0, grid = 0, block = 0, rb = 0, nst = 0, nst1 = 0, nstc = 0;
        long long nitems = 0;
        size_t smem = 0;
        const void* fn = nullptr;
        bool ready = false;
    } pair, quad;
    int opt_pair_variant = -1, opt_quad_variant = -1;
    // on-chip resident kernel (gg_resident.cuh)
    struct ResidentPlan {
        int R = 0, slabs_per_sim = 0, grid = 0, block = 0, block_y = 1;
        size_t smem = 0;
        const void* fn = nullptr;
        bool ready = false;
        bool cluster = false;     // gg_cluster.cuh (one cluster per simulation) instead of gg_resident.cuh
    } resident;
    int opt_resident_impl = 0;    // tuning: 0 = cluster kernel where a simulation fits one, 1 = never
    int opt_cluster_ctas = 0;     // tuning: CTAs per cluster (8 or 16); 0 = from the batch size
    void* d_res_halo = nullptr;
    unsigned int* d_res_flags = nullptr;
    int opt_variant2 = -1;        // -1 = tuned default for the dtype
    // graphs
    std::map<GraphKey, cudaGraphExec_t> graphs;
    // stats
    long long launches = 0;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    bool timed = false;
    int num_sms = 0;
    mutable std::string err, kname;

    size_t esize() const { return dtype == GG_F64 ? 8 : 4; }
    size_t plane() const { return (size_t)nx * ny; }
};

namespace {

int fail(const gg_ctx* c, int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (c) c->err = buf; else g_create_error = buf;
    return code;
}

#define GG_CUDA(c, call)                                                                  \
    do {                                                                                  \
        cudaError_t e_ = (call);                                                          \
        if (e_ != cudaSuccess)                                                            \
            return fail((c), GG_ERR_CUDA, "%s: %s (%s:%d)", #call, cudaGetErrorString(e_), \
                        __FILE__, __LINE__);                                              \
    } while (0)

struct Layout {
    size_t state[2][3], coef[3], sims, coefs, clock, scratch, res_halo, res_flags, total;
};
int resident_rows(const gg_ctx* c, int max_slabs);
int cluster_rows(const gg_ctx* c);
int cluster_ctas(const gg_ctx* c);
int cluster_run_cells(const gg_ctx* c);
bool resident_fits(const gg_ctx* c);   // either on-chip implementation can take the shape
size_t resident_halo_bytes(const gg_ctx* c);
// scratch for the reductions of gg_diag.cuh: [nbatch][kDiagMaxBlocks][8] partials + [nbatch][8]
size_t scratch_doubles(const gg_ctx* c);

Layout layout_of(const gg_ctx* c) {
    Layout L;
    size_t off = 0;
    const size_t sb = align_up((size_t)c->nbatch * c->plane() * c->esize());
    const size_t cb = align_up(c->plane() * c->esize());
    for (int p = 0; p < 2; ++p)
        for (int f = 0; f < 3; ++f) { L.state[p][f] = off; off += sb; }
    for (int f = 0; f < 3; ++f) { L.coef[f] = off; off += cb; }
    L.sims = off;
    off += align_up((size_t)c->nbatch * sizeof(gg::SimScalars));
    L.coefs = off;
    off += align_up((size_t)c->nbatch * sizeof(gg::StepCoef<double>));
    L.clock = off;
    off += align_up(sizeof(gg::DevClock));
    L.scratch = off;
    off += align_up(scratch_doubles(c) * sizeof(double));
    // edge-row exchange buffers and step counters of the resident kernel (small grids only)
    L.res_halo = L.res_flags = 0;
    if (resident_rows(c, 148) > 0) {
        L.res_halo = off;
        off += align_up(resident_halo_bytes(c));
        L.res_flags = off;
        off += align_up(148 * sizeof(unsigned int));
    }
    L.total = off;
    return L;
}

size_t scratch_doubles(const gg_ctx* c) {
    return (size_t)c->nbatch * gg::kDiagMaxBlocks * gg::kDiagCount + (size_t)c->nbatch * gg::kDiagCount;
}

// The opt-in dynamic shared-memory limit is an attribute of the FUNCTION (process-wide), while the
// size a plan asks for depends on its context's shape: always raise it to the device cap, so that
// contexts of different shapes sharing one instantiation never lower each other's limit.
constexpr int kMaxDynSmem = 227 * 1024;
cudaError_t allow_max_smem(const void* fn) {
    return cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxDynSmem);
}

bool stream_shape_ok(const gg_ctx* c) { return ((size_t)c->nx * c->esize()) % 16 == 0; }

int resolve_kernel(const gg_ctx* c) {
    if (c->opt_kernel != GG_KERNEL_AUTO) return c->opt_kernel;
    if (!stream_shape_ok(c)) return GG_KERNEL_GENERIC;
    // Tuned on B200.  The deeper the temporal blocking, the larger the
    // per-launch pipeline fill and the halo overhead, so small grids stay with shallower kernels.
    const double cells = (double)c->nx * c->ny * c->nbatch;
    // Small grids are latency-bound.  A simulation that fits into the shared
    // memory of one thread-block cluster runs the whole call on chip, one cluster per simulation
    // (gg_cluster.cuh: 64^2 fp64 0.84 us per step, 256^2 fp32 2.7), as long as the batch fills at
    // most two waves of clusters; gg_step uses it for calls of >= kResidentMinSteps steps, STREAM2
    // for shorter ones.  Other small shapes that fit on chip as row slabs: gg_resident.cuh.
    if (cluster_rows(c) > 0 && c->opt_resident_impl != 1 && (long long)c->nbatch * cluster_ctas(c) <= 2 * 148)
        return GG_KERNEL_RESIDENT;
    if (cells <= (c->dtype == GG_F32 ? 65536.0 : 16384.0) &&
        resident_rows(c, c->bound ? (c->num_sms < 148 ? c->num_sms : 148) : 148) > 0)
        return GG_KERNEL_RESIDENT;
    // From mid-size grids up: four steps per launch (ahead of the pair kernel in both types from
    // 512^2 to 8192^2 and on batches; a flat 4.5-5 us per step below ~600^2).  Needs one 58-run tile.
    if (c->nx >= gg::quad_runs(2) * (c->dtype == GG_F64 ? 2 : 4) && cells >= 65536.0) return GG_KERNEL_QUAD;
    if (cells > 262144.0 && c->nx >= 240) return GG_KERNEL_PAIR;
    return GG_KERNEL_STREAM2;
}

void drop_graphs(gg_ctx* c) {
    for (auto& kv : c->graphs) cudaGraphExecDestroy(kv.second);
    c->graphs.clear();
}

}  // namespace

// ------------------------------------------------------------------------------------------
// Stream-kernel plan: tensor maps + launch geometry
// ------------------------------------------------------------------------------------------
namespace {

// Stream kernel instantiations: tuning index v = (rows per TMA box RB, ring stages NST), crossed
// with the warps (= strips) per CTA, NW in {1, 2, 4, 8}, which the plan picks from the grid width.
// v = 0 is the build tuned on B200; the others stay selectable through
// GG_OPT_STREAM_VARIANT for re-tuning.
struct Variant { int rb, nst; };
constexpr Variant kVariants[] = {{2, 4}, {4, 2}};
constexpr int kNumVariants = (int)(sizeof(kVariants) / sizeof(kVariants[0]));
constexpr int kDefaultVariant = 1;

struct Variant2 { int rb, nst0, nst1; };
constexpr Variant2 kVariants2[] = {{4, 2, 2}, {3, 2, 2}};
constexpr int kNumVariants2 = (int)(sizeof(kVariants2) / sizeof(kVariants2[0]));

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) !=
                cudaSuccess || qres != cudaDriverEntryPointSuccess)
            p = nullptr;
        return (EncodeTiledFn)p;
    }();
    return fn;
}

int make_map(gg_ctx* c, CUtensorMap* m, void* base, int depth, int box_bytes, int box_rows) {
    EncodeTiledFn enc = encode_fn();
    if (!enc) return fail(c, GG_ERR_CUDA, "cuTensorMapEncodeTiled entry point not available");
    const size_t es = c->esize();
    cuuint64_t dims[3] = {(cuuint64_t)c->nx, (cuuint64_t)c->ny, (cuuint64_t)depth};
    cuuint64_t strides[2] = {(cuuint64_t)c->nx * es, (cuuint64_t)c->plane() * es};
    cuuint32_t box[3] = {(cuuint32_t)(box_bytes / es), (cuuint32_t)box_rows, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = enc(m, c->dtype == GG_F64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64
                                           : CU_TENSOR_MAP_DATA_TYPE_FLOAT32,
                     3, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(c, GG_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
    return GG_OK;
}

// Row-chunk planner of every tiled kernel: the item schedule is static round-robin over
// `resident` CTAs, so among chunk counts that give between 1 and 4 x the target items pick the one
// with the best (wave efficiency) x (useful rows / rows loaded); every chunk loads `halo_rows`
// extra rows.  No chunk is shorter than kMinChunkRows rows.
// shortest row chunk of a work item (512^2 fp64 with 16: 4.86 us per step, with 8: 4.2; the halo
// rows are redundant work, but small grids are bound by the length of an item's march)
constexpr int kMinChunkRows = 8;
void plan_chunks(const gg_ctx* c, long long per, long long resident, int halo_rows, int* chunk_rows,
                 int* nchunks) {
    const long long max_chunks = (c->ny + kMinChunkRows - 1) / kMinChunkRows;
    const long long target = (long long)c->opt_items_per_warp * resident;
    long long best_n = 1;
    double best_score = -1.0;
    for (long long n = 1; n <= max_chunks; ++n) {
        const long long rows = (c->ny + n - 1) / n;
        const long long nch = (c->ny + rows - 1) / rows;  // chunks actually produced
        if (nch != n) continue;
        const long long items = per * nch;
        if (items > 4 * target && n > 1) break;
        const long long waves = (items + resident - 1) / resident;
        // ragged last chunk: the slowest CTA still processes `rows` rows per item
        const double eff = (double)c->ny * per / ((double)waves * resident * rows);
        double score = eff * (double)rows / (double)(rows + halo_rows);
        if (items < target) score *= 0.90 + 0.10 * (double)items / (double)target;  // prefer >= target items
        if (score > best_score + 1e-9) { best_score = score; best_n = nch; }
    }
    *chunk_rows = (int)((c->ny + best_n - 1) / best_n);
    *nchunks = (c->ny + *chunk_rows - 1) / *chunk_rows;
}

// Builds the plan of the single-step (two_step = false) or two-step stream kernel.
int build_plan(gg_ctx* c, bool two_step) {
    bool& ready = two_step ? c->plan2_ready : c->plan_ready;
    if (ready) return GG_OK;
    if (!stream_shape_ok(c))
        return fail(c, GG_ERR_UNSUPPORTED, "stream kernel needs nx*sizeof(elem) %% 16 == 0");
    gg::StreamPlan& P = two_step ? c->plan2 : c->plan;
    const int strip_cells = gg::kStripBytes / (int)c->esize();
    const int nstrips = (c->nx + strip_cells - 1) / strip_cells;
    int nw = c->opt_warps;
    if (resolve_kernel(c) == GG_KERNEL_PAIR || resolve_kernel(c) == GG_KERNEL_QUAD) nw = 0;  // GG_OPT_STREAM_WARPS then addresses the pair kernel
    // Tuned on B200 at 8192^2: fp64 runs 4 rows per box with 4 strips per
    // step; fp32 runs 3 rows per box with 2 strips (its row body is twice as long per lane, and
    // the smaller build keeps the three warp roles inside the instruction cache).
    const int v2 = c->opt_variant2 >= 0 ? c->opt_variant2 : (c->dtype == GG_F64 ? 0 : 1);
    if (two_step) {
        const Variant2 var = kVariants2[v2];
        const int nw_max = c->opt_variant2 < 0 && c->dtype == GG_F32 ? 2 : 4;
        if (nw == 0 || nw > 4) nw = nstrips >= 4 && nw_max >= 4 ? 4 : nstrips >= 2 ? 2 : 1;
        P.rb = var.rb; P.nst = var.nst0; P.nst1 = var.nst1; P.nw = nw; P.steps = 2;
    } else {
        const Variant var = kVariants[c->opt_variant];
        if (nw == 0) nw = nstrips >= 8 ? 8 : nstrips >= 4 ? 4 : nstrips >= 2 ? 2 : 1;
        P.rb = var.rb; P.nst = var.nst; P.nst1 = 0; P.nw = nw; P.steps = 1;
    }
    const int gw_max = 256 / strip_cells;                 // a TMA box is at most 256 elements wide
    const int box_bytes = (nw < gw_max ? nw : gw_max) * gg::kStripBytes;
    for (int p = 0; p < 2; ++p)
        for (int f = 0; f < 3; ++f) {
            int rc = make_map(c, &P.state[p][f], c->state[p][f], c->nbatch, box_bytes, P.rb);
            if (rc) return rc;
            rc = make_map(c, &P.state_halo[p][f], c->state[p][f], c->nbatch, gg::kHaloBytes, P.rb);
            if (rc) return rc;
        }
    for (int f = 0; f < 3; ++f) {
        int rc = make_map(c, &P.coef[f], c->coef[f], 1, box_bytes, P.rb);
        if (rc) return rc;
        rc = make_map(c, &P.coef_halo[f], c->coef[f], 1, gg::kHaloBytes, P.rb);
        if (rc) return rc;
    }
    const void* fn = nullptr;
    int rc = 0;
    if (two_step) {
        P.block = (2 * nw + 2) * 32;  // nw step-1 + nw step-2 warps, halo warp, TMA producer warp
        P.smem = (size_t)gg::stream2_smem_bytes(P.rb, P.nst, P.nst1, nw);
        fn = gg::stream2_kernel(c->dtype == GG_F64, v2, nw);
    } else {
        P.block = (nw + 1) * 32;  // nw consumer warps + the TMA producer warp
        P.smem = (size_t)gg::stream_smem_bytes(P.rb, P.nst, nw);
        fn = gg::stream_kernel(c->dtype == GG_F64, c->opt_variant, nw);
    }
    if (rc || !fn) return fail(c, GG_ERR_UNSUPPORTED, "no stream kernel build for this variant with %d warps", nw);
    P.fn = fn;
    GG_CUDA(c, allow_max_smem(fn));
    int per_sm = 0;
    GG_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, P.block, P.smem));
    if (per_sm < 1) return fail(c, GG_ERR_CUDA, "stream kernel does not fit on an SM");
    const long long resident = (long long)c->num_sms * per_sm;
    P.ntilecols = (nstrips + nw - 1) / nw;
    plan_chunks(c, (long long)P.ntilecols * c->nbatch, resident, 2 * P.steps, &P.chunk_rows, &P.nchunks);
    P.nitems = (long long)P.ntilecols * P.nchunks * c->nbatch;
    P.grid = (int)(P.nitems < resident ? P.nitems : resident);
    ready = true;
    return GG_OK;
}

#include "gg_pair_plan.inc"
#include "gg_resident_plan.inc"

template <typename T>
int launch_generic(gg_ctx* c, int src) {
    gg::GenericArgs<T> a;
    a.U = (const T*)c->state[src][0]; a.V = (const T*)c->state[src][1]; a.W = (const T*)c->state[src][2];
    a.U1 = (T*)c->state[src ^ 1][0]; a.V1 = (T*)c->state[src ^ 1][1]; a.W1 = (T*)c->state[src ^ 1][2];
    a.a = (const T*)c->coef[0]; a.b = (const T*)c->coef[1]; a.c = (const T*)c->coef[2];
    a.coefs = c->d_coefs;
    a.nx = c->nx; a.ny = c->ny; a.nbatch = c->nbatch;
    dim3 block(64, 4, 1);
    dim3 grid((c->nx + 63) / 64, (c->ny + 3) / 4, c->nbatch);
    gg::gg_step_generic<T><<<grid, block, 0, c->stream>>>(a);
    GG_CUDA(c, cudaGetLastError());
    return GG_OK;
}

// One launch of the single-step or two-step stream kernel from copy `src` into `src^1`.
int launch_stream(gg_ctx* c, int src, bool two_step) {
    const gg::StreamPlan& P = two_step ? c->plan2 : c->plan;
    gg::StreamArgs a;
    a.mU = P.state[src][0]; a.mV = P.state[src][1]; a.mW = P.state[src][2];
    a.ma = P.coef[0]; a.mb = P.coef[1]; a.mc = P.coef[2];
    a.hU = P.state_halo[src][0]; a.hV = P.state_halo[src][1]; a.hW = P.state_halo[src][2];
    a.ha = P.coef_halo[0]; a.hb = P.coef_halo[1]; a.hc = P.coef_halo[2];
    a.U1 = c->state[src ^ 1][0]; a.V1 = c->state[src ^ 1][1]; a.W1 = c->state[src ^ 1][2];
    a.coefs = c->d_coefs;
    a.nx = c->nx; a.ny = c->ny; a.nbatch = c->nbatch;
    a.ntilecols = P.ntilecols; a.nchunks = P.nchunks; a.chunk_rows = P.chunk_rows;
    a.nitems = P.nitems;
    void* params[1] = {&a};
    GG_CUDA(c, cudaLaunchKernel(P.fn, dim3(P.grid), dim3(P.block), params, P.smem, c->stream));
    return GG_OK;
}

// one step from ping-pong copy `src` into `src^1`
int launch_step(gg_ctx* c, int kernel, int src) {
    switch (kernel) {
        case GG_KERNEL_GENERIC:
            return c->dtype == GG_F64 ? launch_generic<double>(c, src) : launch_generic<float>(c, src);
        case GG_KERNEL_STREAM:
            return launch_stream(c, src, false);
        default:
            return fail(c, GG_ERR_UNSUPPORTED, "kernel %d not available", kernel);
    }
}

// Enqueue `len` time steps starting from ping-pong copy `src`, with whatever step coefficients
// the device holds when the kernels run.  GG_KERNEL_STREAM2 / PAIR advance two steps per launch,
// QUAD four; a remainder ends with shallower launches.  *nlaunch = kernels launched so far in
// this call (also on failure); every launch flips the ping-pong copy.
int enqueue_steps(gg_ctx* c, int kernel, int src, long long len, long long* nlaunch) {
    int s = src;
    while (len > 0) {
        int rc;
        if (kernel == GG_KERNEL_STREAM2 && len >= 2) { rc = launch_stream(c, s, true); len -= 2; }
        else if (kernel == GG_KERNEL_QUAD && len >= 4) { rc = launch_multi(c, c->quad, s); len -= 4; }
        else if ((kernel == GG_KERNEL_PAIR || kernel == GG_KERNEL_QUAD) && len >= 2) { rc = launch_pair(c, s); len -= 2; }
        else if (kernel == GG_KERNEL_STREAM2 || kernel == GG_KERNEL_PAIR || kernel == GG_KERNEL_QUAD) { rc = launch_stream(c, s, false); len -= 1; }
        else { rc = launch_step(c, kernel, s); len -= 1; }
        if (rc) return rc;
        s ^= 1;
        ++*nlaunch;
    }
    return GG_OK;
}

long long launches_for(int kernel, long long len) {
    if (kernel == GG_KERNEL_QUAD) return len / 4 + ((len % 4) >> 1) + (len & 1);
    return kernel == GG_KERNEL_STREAM2 || kernel == GG_KERNEL_PAIR ? len / 2 + (len & 1) : len;
}

// segment length and block count of the two-stage reductions (gg_diag.cuh, gg_dt.cuh)
void reduce_geometry(const gg_ctx* c, size_t* seg, int* nblk) {
    const size_t plane = c->plane();
    size_t s = (plane + gg::kDiagMaxBlocks - 1) / gg::kDiagMaxBlocks;
    s = (s + gg::kDiagThreads - 1) / gg::kDiagThreads * gg::kDiagThreads;
    *seg = s;
    *nblk = (int)((plane + s - 1) / s);
}

// The device-side dt rule for the `k` steps that follow (gg_dt.cuh): min U of copy `src` per
// simulation, then dt_k, the folded coefficients and the clock.  Two small launches.
int enqueue_adapt(gg_ctx* c, int src, long long k) {
    size_t seg; int nblk;
    reduce_geometry(c, &seg, &nblk);
    dim3 grid(nblk, c->nbatch);
    if (c->dtype == GG_F64)
        gg::gg_min_u_partial<double><<<grid, gg::kDiagThreads, 0, c->stream>>>((const double*)c->state[src][0], c->plane(), seg, c->d_scratch);
    else
        gg::gg_min_u_partial<float><<<grid, gg::kDiagThreads, 0, c->stream>>>((const float*)c->state[src][0], c->plane(), seg, c->d_scratch);
    GG_CUDA(c, cudaGetLastError());
    gg::gg_fold_adaptive<<<1, gg::kDiagThreads, 0, c->stream>>>(c->d_clock, c->d_sims, c->d_coefs, c->d_scratch, nblk,
                                                              c->nbatch, c->dx, c->dy, k);
    GG_CUDA(c, cudaGetLastError());
    return GG_OK;
}

// `len` steps from copy `src`: every_k == 0 -> plain steps; every_k > 0 -> groups of every_k steps,
// each preceded by the device-side dt rule.
int enqueue_span(gg_ctx* c, int kernel, int src, long long len, long long every_k, long long* nlaunch) {
    if (every_k <= 0) return enqueue_steps(c, kernel, src, len, nlaunch);
    int s = src;
    while (len > 0) {
        const long long g = len < every_k ? len : every_k;
        int rc = enqueue_adapt(c, s, g);
        if (rc) return rc;
        const long long before = *nlaunch;
        rc = enqueue_steps(c, kernel, s, g, nlaunch);
        if (rc) return rc;
        s ^= (int)((*nlaunch - before) & 1);
        len -= g;
    }
    return GG_OK;
}

// parity flip of `len` steps issued in groups of every_k (0: one group)
int span_flips(int kernel, long long len, long long every_k, long long* nlaunch) {
    long long nl = 0;
    if (every_k <= 0) nl = launches_for(kernel, len);
    else {
        nl = (len / every_k) * launches_for(kernel, every_k);
        if (len % every_k) nl += launches_for(kernel, len % every_k);
    }
    *nlaunch = nl;
    return (int)(nl & 1);
}

// Capture a span into an executable graph.
int capture_graph(gg_ctx* c, int kernel, long long len, long long every_k, int src, cudaGraphExec_t* out) {
    long long nl = 0;
    cudaStream_t cap = nullptr;
    GG_CUDA(c, cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
    cudaStream_t user = c->stream;
    c->stream = cap;  // the launch functions enqueue on c->stream
    cudaGraph_t graph = nullptr;
    int rc = GG_OK;
    cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) {
        rc = fail(c, GG_ERR_CUDA, "cudaStreamBeginCapture: %s", cudaGetErrorString(e));
    } else {
        rc = enqueue_span(c, kernel, src, len, every_k, &nl);
        e = cudaStreamEndCapture(cap, &graph);
        if (rc == GG_OK && e != cudaSuccess)
            rc = fail(c, GG_ERR_CUDA, "cudaStreamEndCapture: %s", cudaGetErrorString(e));
    }
    c->stream = user;
    if (rc == GG_OK) {
        e = cudaGraphInstantiate(out, graph, 0);
        if (e != cudaSuccess) rc = fail(c, GG_ERR_CUDA, "cudaGraphInstantiate: %s", cudaGetErrorString(e));
        else ++c->graph_captures;
    }
    if (graph) cudaGraphDestroy(graph);
    cudaStreamDestroy(cap);
    return rc;
}

int build_plans(gg_ctx* ctx, int kernel) {
    int rc = GG_OK;
    if (kernel == GG_KERNEL_STREAM || kernel == GG_KERNEL_STREAM2 || kernel == GG_KERNEL_PAIR ||
        kernel == GG_KERNEL_QUAD)
        rc = build_plan(ctx, false);
    if (!rc && (kernel == GG_KERNEL_PAIR || kernel == GG_KERNEL_QUAD)) rc = build_plan_pair(ctx);
    if (!rc && kernel == GG_KERNEL_QUAD) rc = build_plan_quad(ctx);
    if (!rc && kernel == GG_KERNEL_STREAM2) rc = build_plan(ctx, true);
    return rc;
}

// The step loop shared by gg_step (every_k = 0) and gg_step_adaptive: replay cached graphs of up
// to opt_chunk steps (whole groups of every_k), or plain launches with GG_OPT_GRAPH = 0.
int run_steps(gg_ctx* ctx, int kernel, long long n, long long every_k) {
    long long left = n;
    if (ctx->opt_graph && n >= 2) {
        long long chunk = ctx->opt_chunk;
        if (every_k > 0) chunk = chunk / every_k >= 1 ? chunk / every_k * every_k : every_k;
        while (left > 0) {
            const long long len = left < chunk ? left : chunk;
            const GraphKey key{len, ctx->cur, kernel, every_k};
            auto it = ctx->graphs.find(key);
            if (it == ctx->graphs.end()) {
                if (ctx->graphs.size() >= 32) drop_graphs(ctx);
                cudaGraphExec_t ex = nullptr;
                int rc = capture_graph(ctx, kernel, len, every_k, ctx->cur, &ex);
                if (rc) return rc;
                it = ctx->graphs.emplace(key, ex).first;
            }
            GG_CUDA(ctx, cudaGraphLaunch(it->second, ctx->stream));
            long long nl = 0;
            ctx->cur ^= span_flips(kernel, len, every_k, &nl);
            ctx->launches += nl;
            left -= len;
        }
    } else {
        long long nl = 0;
        const int rc = enqueue_span(ctx, kernel, ctx->cur, left, every_k, &nl);
        ctx->cur ^= (int)(nl & 1);
        ctx->launches += nl;
        if (rc) {
            // some launches may have been enqueued: the ping-pong copies no longer hold a
            // consistent time level
            ctx->have_state = false;
            return rc;
        }
    }
    return GG_OK;
}

// raw: the tensor entries a, c as given, in scratch (the ping-pong copy no step has written yet
// or will read again); b is already in place.
template <typename T>
int finish_tensor(gg_ctx* ctx, const void* raw_a, const void* raw_c) {
    // lambda_max(A) of the tensor as given, cached on the device for the step-size rule ...
    size_t seg; int nblk;
    reduce_geometry(ctx, &seg, &nblk);
    gg::gg_lambda_max_partial<T><<<nblk, gg::kDiagThreads, 0, ctx->stream>>>(
        (const T*)raw_a, (const T*)ctx->coef[1], (const T*)raw_c, ctx->plane(), seg, ctx->d_scratch);
    GG_CUDA(ctx, cudaGetLastError());
    gg::gg_lambda_final<<<1, gg::kDiagThreads, 0, ctx->stream>>>(ctx->d_scratch, nblk, ctx->d_clock);
    GG_CUDA(ctx, cudaGetLastError());
    // ... then a and c in their stored form: pre-scaled west- and south-face sums (StepCoef comment
    // in gg_common.cuh)
    const int blocks = (int)std::min<size_t>((ctx->plane() + 255) / 256, (size_t)ctx->num_sms * 8);
    gg::gg_face_tensor<T><<<blocks, 256, 0, ctx->stream>>>((const T*)raw_a, (T*)ctx->coef[0], ctx->nx, ctx->plane(), 1,
                                                          gg::tensor_scale_a(ctx->dx, ctx->dy));
    GG_CUDA(ctx, cudaGetLastError());
    gg::gg_face_tensor<T><<<blocks, 256, 0, ctx->stream>>>((const T*)raw_c, (T*)ctx->coef[2], ctx->nx, ctx->plane(), ctx->nx,
                                                          gg::tensor_scale_c(ctx->dx, ctx->dy));
    GG_CUDA(ctx, cudaGetLastError());
    return GG_OK;
}

// Function-level guard: nothing throws across the ABI (std::bad_alloc from the host containers).
template <typename F>
int guarded(const gg_ctx* c, const char* what, F&& f) {
    try {
        return f();
    } catch (const std::bad_alloc&) {
        try { return fail(c, GG_ERR_ARG, "%s: out of host memory", what); } catch (...) { return GG_ERR_ARG; }
    } catch (...) {
        try { return fail(c, GG_ERR_CUDA, "%s: unexpected C++ exception", what); } catch (...) { return GG_ERR_CUDA; }
    }
}

}  // namespace

// ------------------------------------------------------------------------------------------
// extern "C" entry points (contracts in include/gg.h)
// ------------------------------------------------------------------------------------------
extern "C" {

int gg_create_xy(gg_ctx** out, int nbatch, int nx, int ny, double dx, double dy, const double* r,
                 const double* d, const double* alpha, const double* c, int dtype) {
    return guarded(nullptr, "gg_create", [&]() -> int {
        if (!out) return fail(nullptr, GG_ERR_ARG, "gg_create: out is NULL");
        *out = nullptr;
        if (nbatch < 1) return fail(nullptr, GG_ERR_ARG, "gg_create: nbatch %d < 1", nbatch);
        if (nx < 2 || ny < 2) return fail(nullptr, GG_ERR_ARG, "gg_create: nx, ny must be >= 2 (got %d x %d)", nx, ny);
        // launch-geometry limits of the one-thread-per-cell and reduction kernels (gridDim.y / .z)
        if (nbatch > 65535) return fail(nullptr, GG_ERR_ARG, "gg_create: nbatch %d > 65535", nbatch);
        if (ny > 262140) return fail(nullptr, GG_ERR_ARG, "gg_create: ny %d > 262140", ny);
        if (!(dx > 0.0) || !std::isfinite(dx) || !(dy > 0.0) || !std::isfinite(dy))
            return fail(nullptr, GG_ERR_ARG, "gg_create: mesh sizes must be finite and > 0");
        if (!r || !d || !alpha || !c) return fail(nullptr, GG_ERR_ARG, "gg_create: NULL parameter array");
        if (dtype != GG_F64 && dtype != GG_F32) return fail(nullptr, GG_ERR_UNSUPPORTED, "gg_create: unknown dtype %d", dtype);
        if ((double)nx * ny * nbatch > 2.0e10) return fail(nullptr, GG_ERR_ARG, "gg_create: grid too large");
        for (int s = 0; s < nbatch; ++s)
            if (!std::isfinite(r[s]) || !std::isfinite(d[s]) || !std::isfinite(alpha[s]) || !std::isfinite(c[s]))
                return fail(nullptr, GG_ERR_ARG, "gg_create: non-finite parameter for simulation %d", s);
        gg_ctx* ctx = new (std::nothrow) gg_ctx;
        if (!ctx) return fail(nullptr, GG_ERR_ARG, "gg_create: out of host memory");
        ctx->nx = nx; ctx->ny = ny; ctx->nbatch = nbatch; ctx->dx = dx; ctx->dy = dy; ctx->dtype = dtype;
        try {
            ctx->sims.resize(nbatch);
        } catch (...) {
            delete ctx;
            throw;
        }
        for (int s = 0; s < nbatch; ++s) ctx->sims[s] = gg::SimScalars{r[s], d[s], alpha[s], c[s]};
        ctx->opt_variant = kDefaultVariant;
        *out = ctx;
        return GG_OK;
    });
}

int gg_create_batch(gg_ctx** out, int nbatch, int nx, int ny, double h, const double* r,
                    const double* d, const double* alpha, const double* c, int dtype) {
    return gg_create_xy(out, nbatch, nx, ny, h, h, r, d, alpha, c, dtype);
}

int gg_create(gg_ctx** out, int nx, int ny, double h, double r, double d, double alpha, double c,
              int dtype) {
    return gg_create_batch(out, 1, nx, ny, h, &r, &d, &alpha, &c, dtype);
}

size_t gg_workspace_bytes(const gg_ctx* ctx) { return ctx ? layout_of(ctx).total : 0; }

int gg_bind(gg_ctx* ctx, void* ws, size_t bytes, void* stream) {
    if (!ctx) return GG_ERR_ARG;
    if (ctx->bound) return fail(ctx, GG_ERR_STATE, "gg_bind: already bound");
    if (!ws) return fail(ctx, GG_ERR_ARG, "gg_bind: workspace is NULL");
    const Layout L = layout_of(ctx);
    if (bytes < L.total) return fail(ctx, GG_ERR_ARG, "gg_bind: workspace %zu B < required %zu B", bytes, L.total);
    if ((uintptr_t)ws % kAlign) return fail(ctx, GG_ERR_ARG, "gg_bind: workspace not 256-byte aligned");
    cudaPointerAttributes at;
    GG_CUDA(ctx, cudaPointerGetAttributes(&at, ws));
    if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)
        return fail(ctx, GG_ERR_ARG, "gg_bind: workspace is not device memory");
    int dev = 0;
    GG_CUDA(ctx, cudaGetDevice(&dev));
    GG_CUDA(ctx, cudaDeviceGetAttribute(&ctx->num_sms, cudaDevAttrMultiProcessorCount, dev));
    ctx->ws = (char*)ws; ctx->ws_bytes = bytes; ctx->stream = (cudaStream_t)stream;
    for (int p = 0; p < 2; ++p)
        for (int f = 0; f < 3; ++f) ctx->state[p][f] = ctx->ws + L.state[p][f];
    for (int f = 0; f < 3; ++f) ctx->coef[f] = ctx->ws + L.coef[f];
    ctx->d_sims = (gg::SimScalars*)(ctx->ws + L.sims);
    ctx->d_coefs = (gg::StepCoef<double>*)(ctx->ws + L.coefs);
    ctx->d_clock = (gg::DevClock*)(ctx->ws + L.clock);
    ctx->d_scratch = (double*)(ctx->ws + L.scratch);
    if (L.res_halo) {
        ctx->d_res_halo = ctx->ws + L.res_halo;
        ctx->d_res_flags = (unsigned int*)(ctx->ws + L.res_flags);
    }
    GG_CUDA(ctx, cudaMemsetAsync(ctx->d_clock, 0, sizeof(gg::DevClock), ctx->stream));
    GG_CUDA(ctx, cudaMemcpyAsync(ctx->d_sims, ctx->sims.data(), ctx->sims.size() * sizeof(gg::SimScalars),
                                 cudaMemcpyHostToDevice, ctx->stream));
    GG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));  // sims is pageable host memory
    GG_CUDA(ctx, cudaEventCreate(&ctx->ev0));
    GG_CUDA(ctx, cudaEventCreate(&ctx->ev1));
    ctx->bound = true;
    return GG_OK;
}

static int copy3(gg_ctx* ctx, void* const dst[3], const void* const src[3], size_t bytes,
                 cudaMemcpyKind kind, bool sync) {
    for (int f = 0; f < 3; ++f)
        GG_CUDA(ctx, cudaMemcpyAsync(dst[f], src[f], bytes, kind, ctx->stream));
    if (sync) GG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return GG_OK;
}

static int set_tensor_impl(gg_ctx* ctx, const void* a, const void* b, const void* c, bool host) {
    if (!ctx) return GG_ERR_ARG;
    if (!ctx->bound) return fail(ctx, GG_ERR_STATE, "gg_set_tensor: call gg_bind first");
    if (!a || !b || !c) return fail(ctx, GG_ERR_ARG, "gg_set_tensor: NULL array");
    const void* src[3] = {a, b, c};
    ctx->have_tensor = false;
    // a and c land in the ping-pong copy that holds no live time level (the next step overwrites
    // it, nothing reads it before); finish_tensor turns them into the stored face sums
    void* dst[3] = {ctx->state[ctx->cur ^ 1][0], ctx->coef[1], ctx->state[ctx->cur ^ 1][1]};
    int rc = copy3(ctx, dst, src, ctx->plane() * ctx->esize(),
                   host ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, host);
    if (rc) return rc;
    rc = ctx->dtype == GG_F64 ? finish_tensor<double>(ctx, dst[0], dst[2]) : finish_tensor<float>(ctx, dst[0], dst[2]);
    if (rc) return rc;
    ctx->have_tensor = true;
    return GG_OK;
}
static int set_state_impl(gg_ctx* ctx, const void* U, const void* V, const void* W, bool host) {
    if (!ctx) return GG_ERR_ARG;
    if (!ctx->bound) return fail(ctx, GG_ERR_STATE, "gg_set_state: call gg_bind first");
    if (!U || !V || !W) return fail(ctx, GG_ERR_ARG, "gg_set_state: NULL array");
    const void* src[3] = {U, V, W};
    int rc = copy3(ctx, ctx->state[ctx->cur], src, (size_t)ctx->nbatch * ctx->plane() * ctx->esize(),
                   host ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, host);
    if (rc) return rc;
    gg::gg_clock_reset<<<1, 1, 0, ctx->stream>>>(ctx->d_clock);
    GG_CUDA(ctx, cudaGetLastError());
    ctx->have_state = true;
    ctx->rule_failed = false;
    return GG_OK;
}
static int get_state_impl(gg_ctx* ctx, void* U, void* V, void* W, bool host) {
    if (!ctx) return GG_ERR_ARG;
    if (!ctx->bound || !ctx->have_state) return fail(ctx, GG_ERR_STATE, "gg_get_state: no state set");
    if (!U || !V || !W) return fail(ctx, GG_ERR_ARG, "gg_get_state: NULL array");
    void* dst[3] = {U, V, W};
    return copy3(ctx, dst, ctx->state[ctx->cur], (size_t)ctx->nbatch * ctx->plane() * ctx->esize(),
                 host ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, host);
}

int gg_set_tensor(gg_ctx* c, const void* a, const void* b, const void* cc) { return set_tensor_impl(c, a, b, cc, false); }
int gg_set_tensor_host(gg_ctx* c, const void* a, const void* b, const void* cc) { return set_tensor_impl(c, a, b, cc, true); }
int gg_set_state(gg_ctx* c, const void* U, const void* V, const void* W) { return set_state_impl(c, U, V, W, false); }
int gg_set_state_host(gg_ctx* c, const void* U, const void* V, const void* W) { return set_state_impl(c, U, V, W, true); }
int gg_get_state(gg_ctx* c, void* U, void* V, void* W) { return get_state_impl(c, U, V, W, false); }
int gg_get_state_host(gg_ctx* c, void* U, void* V, void* W) { return get_state_impl(c, U, V, W, true); }

int gg_step(gg_ctx* ctx, long long n, double dt) {
    if (!ctx) return GG_ERR_ARG;
    return guarded(ctx, "gg_step", [&]() -> int {
        if (!ctx->bound || !ctx->have_tensor || !ctx->have_state)
            return fail(ctx, GG_ERR_STATE, "gg_step: needs gg_bind, gg_set_tensor and gg_set_state first");
        if (ctx->rule_failed) return fail(ctx, GG_ERR_ARG, "gg_step: an earlier gg_step_adaptive found no usable step size (see gg_get_clock); call gg_set_state");
        if (n < 0) return fail(ctx, GG_ERR_ARG, "gg_step: n = %lld < 0", n);
        if (!(dt > 0.0) || !std::isfinite(dt)) return fail(ctx, GG_ERR_ARG, "gg_step: dt must be finite and > 0");
        if (n == 0) return GG_OK;
        int kernel = resolve_kernel(ctx);
        const bool autosel = ctx->opt_kernel == GG_KERNEL_AUTO;
        if (kernel == GG_KERNEL_RESIDENT && autosel &&
            n < (cluster_rows(ctx) > 0 && ctx->opt_resident_impl != 1 ? kClusterMinSteps : kResidentMinSteps))
            kernel = GG_KERNEL_STREAM2;   // a cooperative launch does not pay for a handful of steps
        if (kernel == GG_KERNEL_RESIDENT) {
            const int rc = build_plan_resident(ctx);
            if (rc && !autosel) return rc;
            if (rc) kernel = GG_KERNEL_STREAM2;   // AUTO: a refused cooperative plan is not an error
        }
        if (kernel != GG_KERNEL_RESIDENT) {
            const int rc = build_plans(ctx, kernel);
            if (rc) return rc;
        }
        GG_CUDA(ctx, cudaEventRecord(ctx->ev0, ctx->stream));
        // dt goes to the device by value, in front of (never inside) the replayed graphs
        gg::gg_fold_fixed<<<(ctx->nbatch + 127) / 128, 128, 0, ctx->stream>>>(
            ctx->d_clock, ctx->d_sims, ctx->d_coefs, ctx->nbatch, dt, ctx->dx, ctx->dy, n,
            ctx->folded_dt == dt ? 0 : 1);
        GG_CUDA(ctx, cudaGetLastError());
        ctx->folded_dt = dt;
        // From here on the device clock already counts all n steps: if a launch, a capture or a
        // replay below fails, clock and state no longer belong together -- the state is dropped
        // (gg_set_state starts over and resets the clock) rather than left looking valid.
        if (kernel == GG_KERNEL_RESIDENT) {
            const int rc = launch_resident(ctx, ctx->cur, n);
            if (rc) { ctx->have_state = false; return rc; }
            ctx->cur ^= 1;
            ctx->launches += 1;
        } else {
            const int rc = run_steps(ctx, kernel, n, 0);
            if (rc) { ctx->have_state = false; return rc; }
        }
        GG_CUDA(ctx, cudaEventRecord(ctx->ev1, ctx->stream));
        ctx->timed = true;
        return GG_OK;
    });
}

int gg_step_adaptive(gg_ctx* ctx, long long n, double safety, long long every_k) {
    if (!ctx) return GG_ERR_ARG;
    return guarded(ctx, "gg_step_adaptive", [&]() -> int {
        if (!ctx->bound || !ctx->have_tensor || !ctx->have_state)
            return fail(ctx, GG_ERR_STATE, "gg_step_adaptive: needs gg_bind, gg_set_tensor and gg_set_state first");
        if (ctx->rule_failed) return fail(ctx, GG_ERR_ARG, "gg_step_adaptive: an earlier call found no usable step size (see gg_get_clock); call gg_set_state");
        if (n < 0) return fail(ctx, GG_ERR_ARG, "gg_step_adaptive: n = %lld < 0", n);
        if (!(safety > 0.0) || !std::isfinite(safety)) return fail(ctx, GG_ERR_ARG, "gg_step_adaptive: safety must be finite and > 0");
        if (every_k < 1 || every_k > 4096) return fail(ctx, GG_ERR_ARG, "gg_step_adaptive: every_k must be in 1..4096");
        if (n == 0) return GG_OK;
        int kernel = resolve_kernel(ctx);
        if (kernel == GG_KERNEL_RESIDENT) {
            // the on-chip kernel advances a whole call in one launch and cannot re-read dt
            if (ctx->opt_kernel != GG_KERNEL_AUTO)
                return fail(ctx, GG_ERR_UNSUPPORTED, "gg_step_adaptive: GG_KERNEL_RESIDENT cannot change dt inside its launch");
            kernel = GG_KERNEL_STREAM2;
        }
        int rc = build_plans(ctx, kernel);
        if (rc) return rc;
        GG_CUDA(ctx, cudaEventRecord(ctx->ev0, ctx->stream));
        gg::gg_clock_safety<<<1, 1, 0, ctx->stream>>>(ctx->d_clock, safety);
        GG_CUDA(ctx, cudaGetLastError());
        ctx->folded_dt = std::numeric_limits<double>::quiet_NaN();   // the device decides from here on
        rc = run_steps(ctx, kernel, n, every_k);
        if (rc) { ctx->have_state = false; return rc; }   // as in gg_step: no half-advanced state is kept
        GG_CUDA(ctx, cudaEventRecord(ctx->ev1, ctx->stream));
        ctx->timed = true;
        return GG_OK;
    });
}

int gg_get_clock(gg_ctx* ctx, double* time, double* dt, long long* steps) {
    if (!ctx) return GG_ERR_ARG;
    if (!ctx->bound) return fail(ctx, GG_ERR_STATE, "gg_get_clock: call gg_bind first");
    gg::DevClock h;
    GG_CUDA(ctx, cudaMemcpyAsync(&h, ctx->d_clock, sizeof h, cudaMemcpyDeviceToHost, ctx->stream));
    GG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (time) *time = h.time;
    if (dt) *dt = h.dt;
    if (steps) *steps = h.steps;
    if (h.bad_rule != 0) {
        ctx->rule_failed = true;
        return fail(ctx, GG_ERR_ARG, "gg_step_adaptive: the step-size rule had no positive finite bound in %lld evaluation(s) "
                    "(max(lambda_max, alpha (1 - min U)) = %g); those steps ran with dt = 0.  gg_set_state clears this",
                    h.bad_rule, h.rate);
    }
    return GG_OK;
}

int gg_set_option(gg_ctx* ctx, int option, long long value) {
    if (!ctx) return GG_ERR_ARG;
    switch (option) {
        case GG_OPT_KERNEL:
            if (value == GG_KERNEL_AUTO || value == GG_KERNEL_GENERIC) break;
            if (value == GG_KERNEL_STREAM || value == GG_KERNEL_STREAM2 || value == GG_KERNEL_PAIR ||
                value == GG_KERNEL_QUAD) {
                if (!stream_shape_ok(ctx))
                    return fail(ctx, GG_ERR_UNSUPPORTED, "stream kernel needs nx*sizeof(elem) %% 16 == 0 (nx = %d)", ctx->nx);
                break;
            }
            if (value == GG_KERNEL_RESIDENT) {
                if (!resident_fits(ctx))
                    return fail(ctx, GG_ERR_UNSUPPORTED, "resident kernel: %d x %d x %d does not fit on chip", ctx->nx, ctx->ny, ctx->nbatch);
                break;
            }
            return fail(ctx, GG_ERR_UNSUPPORTED, "gg_set_option: kernel %lld not available", value);
        case GG_OPT_GRAPH:
            if (value != 0 && value != 1) return fail(ctx, GG_ERR_ARG, "GG_OPT_GRAPH: 0 or 1");
            break;
        case GG_OPT_GRAPH_CHUNK:
            if (value < 1 || value > 4096) return fail(ctx, GG_ERR_ARG, "GG_OPT_GRAPH_CHUNK: 1..4096");
            break;
        case GG_OPT_STREAM_VARIANT:
            if (value < 0 || value >= kNumVariants) return fail(ctx, GG_ERR_ARG, "GG_OPT_STREAM_VARIANT: 0..%d", kNumVariants - 1);
            break;
        case GG_OPT_ITEMS_PER_WARP:
            if (value < 1 || value > 1024) return fail(ctx, GG_ERR_ARG, "GG_OPT_ITEMS_PER_CTA: 1..1024");
            break;
        case GG_OPT_STREAM2_VARIANT:
            if (value < -1 || value >= kNumVariants2) return fail(ctx, GG_ERR_ARG, "GG_OPT_STREAM2_VARIANT: -1 (tuned default) or 0..%d", kNumVariants2 - 1);
            break;
        case GG_OPT_STREAM_WARPS:
            if (value < 0 || value > 8)
                return fail(ctx, GG_ERR_ARG, "GG_OPT_STREAM_WARPS: 0..8");
            break;
        case GG_OPT_RESIDENT_IMPL:
            if (value != 0 && value != 1) return fail(ctx, GG_ERR_ARG, "GG_OPT_RESIDENT_IMPL: 0 or 1");
            if (value == 1 && ctx->bound && !ctx->d_res_halo)
                return fail(ctx, GG_ERR_UNSUPPORTED, "GG_OPT_RESIDENT_IMPL = 1: the slab kernel cannot take %d x %d x %d", ctx->nx, ctx->ny, ctx->nbatch);
            break;
        case GG_OPT_CLUSTER_CTAS:
            if (value != 0 && value != 2 && value != 4 && value != 8 && value != 16) return fail(ctx, GG_ERR_ARG, "GG_OPT_CLUSTER_CTAS: 0, 2, 4, 8 or 16");
            break;
        case GG_OPT_QUAD_VARIANT:
            if (value < -1 || value >= kNumQuadVariants) return fail(ctx, GG_ERR_ARG, "GG_OPT_QUAD_VARIANT: -1 or 0..%d", kNumQuadVariants - 1);
            break;
        case GG_OPT_PAIR_VARIANT:
            if (value < -1 || value >= kNumPairVariants) return fail(ctx, GG_ERR_ARG, "GG_OPT_PAIR_VARIANT: -1 or 0..%d", kNumPairVariants - 1);
            break;
        default:
            return fail(ctx, GG_ERR_UNSUPPORTED, "gg_set_option: unknown option %d", option);
    }
    drop_graphs(ctx);
    switch (option) {
        case GG_OPT_KERNEL: ctx->opt_kernel = (int)value; break;
        case GG_OPT_GRAPH: ctx->opt_graph = (int)value; break;
        case GG_OPT_GRAPH_CHUNK: ctx->opt_chunk = value; break;
        case GG_OPT_STREAM_VARIANT: ctx->opt_variant = (int)value; ctx->plan_ready = false; break;
        case GG_OPT_STREAM2_VARIANT: ctx->opt_variant2 = (int)value; ctx->plan2_ready = false; break;
        case GG_OPT_ITEMS_PER_WARP: ctx->opt_items_per_warp = (int)value; ctx->plan_ready = ctx->plan2_ready = false; ctx->pair.ready = ctx->quad.ready = false; break;
        case GG_OPT_STREAM_WARPS: ctx->opt_warps = (int)value; ctx->plan_ready = ctx->plan2_ready = false; ctx->pair.ready = false; break;
        case GG_OPT_PAIR_VARIANT: ctx->opt_pair_variant = (int)value; ctx->pair.ready = false; break;
        case GG_OPT_QUAD_VARIANT: ctx->opt_quad_variant = (int)value; ctx->quad.ready = false; break;
        case GG_OPT_RESIDENT_IMPL: ctx->opt_resident_impl = (int)value; ctx->resident.ready = false; break;
        case GG_OPT_CLUSTER_CTAS: ctx->opt_cluster_ctas = (int)value; ctx->resident.ready = false; break;
    }
    return GG_OK;
}

int gg_diagnostics(gg_ctx* ctx, double eps, double* out) {
    if (!ctx) return GG_ERR_ARG;
    if (!ctx->bound || !ctx->have_state) return fail(ctx, GG_ERR_STATE, "gg_diagnostics: no state set");
    if (!out) return fail(ctx, GG_ERR_ARG, "gg_diagnostics: out is NULL");
    if (!(eps >= 0.0) || !std::isfinite(eps)) return fail(ctx, GG_ERR_ARG, "gg_diagnostics: eps must be finite and >= 0");
    const size_t plane = ctx->plane();
    size_t seg; int nblk;
    reduce_geometry(ctx, &seg, &nblk);
    double* partial = ctx->d_scratch;
    double* fin = ctx->d_scratch + (size_t)ctx->nbatch * gg::kDiagMaxBlocks * gg::kDiagCount;
    void* const* st = ctx->state[ctx->cur];
    dim3 grid(nblk, ctx->nbatch);
    if (ctx->dtype == GG_F64)
        gg::gg_diag_partial<double><<<grid, gg::kDiagThreads, 0, ctx->stream>>>(
            (const double*)st[0], (const double*)st[1], (const double*)st[2], plane, seg, eps, partial);
    else
        gg::gg_diag_partial<float><<<grid, gg::kDiagThreads, 0, ctx->stream>>>(
            (const float*)st[0], (const float*)st[1], (const float*)st[2], plane, seg, eps, partial);
    GG_CUDA(ctx, cudaGetLastError());
    gg::gg_diag_final<<<ctx->nbatch, gg::kDiagThreads, 0, ctx->stream>>>(partial, nblk, fin);
    GG_CUDA(ctx, cudaGetLastError());
    GG_CUDA(ctx, cudaMemcpyAsync(out, fin, (size_t)ctx->nbatch * gg::kDiagCount * sizeof(double),
                                 cudaMemcpyDeviceToHost, ctx->stream));
    GG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return GG_OK;
}

int gg_front(gg_ctx* ctx, int field, int axis, int index, double level, int* out) {
    if (!ctx) return GG_ERR_ARG;
    if (!ctx->bound || !ctx->have_state) return fail(ctx, GG_ERR_STATE, "gg_front: no state set");
    if (!out) return fail(ctx, GG_ERR_ARG, "gg_front: out is NULL");
    if (field < 0 || field > 2) return fail(ctx, GG_ERR_ARG, "gg_front: field must be 0 (U), 1 (V) or 2 (W)");
    if (axis != 0 && axis != 1) return fail(ctx, GG_ERR_ARG, "gg_front: axis must be 0 (along x) or 1 (along y)");
    const int len = axis == 0 ? ctx->nx : ctx->ny, other = axis == 0 ? ctx->ny : ctx->nx;
    if (index < 0 || index >= other) return fail(ctx, GG_ERR_ARG, "gg_front: line index %d outside [0, %d)", index, other);
    if (!std::isfinite(level)) return fail(ctx, GG_ERR_ARG, "gg_front: level must be finite");
    if ((size_t)ctx->nbatch * 2 * sizeof(int) > scratch_doubles(ctx) * sizeof(double))
        return fail(ctx, GG_ERR_UNSUPPORTED, "gg_front: scratch too small");
    const size_t offset = axis == 0 ? (size_t)index * ctx->nx : (size_t)index;
    const size_t stride = axis == 0 ? 1 : (size_t)ctx->nx;
    int* d_out = (int*)ctx->d_scratch;
    const void* F = ctx->state[ctx->cur][field];
    if (ctx->dtype == GG_F64)
        gg::gg_front_line<double><<<ctx->nbatch, gg::kDiagThreads, 0, ctx->stream>>>((const double*)F, ctx->plane(), offset, stride, len, level, d_out);
    else
        gg::gg_front_line<float><<<ctx->nbatch, gg::kDiagThreads, 0, ctx->stream>>>((const float*)F, ctx->plane(), offset, stride, len, level, d_out);
    GG_CUDA(ctx, cudaGetLastError());
    GG_CUDA(ctx, cudaMemcpyAsync(out, d_out, (size_t)ctx->nbatch * 2 * sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    GG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return GG_OK;
}

int gg_max_stable_dt(gg_ctx* ctx, double safety, double* dt, double* lambda_max) {
    if (!ctx) return GG_ERR_ARG;
    if (!ctx->bound || !ctx->have_tensor) return fail(ctx, GG_ERR_STATE, "gg_max_stable_dt: no tensor set");
    if (!dt) return fail(ctx, GG_ERR_ARG, "gg_max_stable_dt: dt is NULL");
    if (!(safety > 0.0) || !std::isfinite(safety)) return fail(ctx, GG_ERR_ARG, "gg_max_stable_dt: safety must be finite and > 0");
    // lambda_max(A) was reduced on the device by gg_set_tensor and is cached in the device clock
    gg::DevClock h;
    GG_CUDA(ctx, cudaMemcpyAsync(&h, ctx->d_clock, sizeof h, cudaMemcpyDeviceToHost, ctx->stream));
    GG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    const double lam = h.lambda_max;
    double amax = ctx->sims[0].alpha;
    for (const auto& sc : ctx->sims) amax = sc.alpha > amax ? sc.alpha : amax;
    const double rate = lam > amax ? lam : amax;
    if (!(rate > 0.0) || !std::isfinite(rate))
        return fail(ctx, GG_ERR_ARG, "gg_max_stable_dt: max(alpha, lambda_max) = %g is not positive and finite", rate);
    const double hmin = ctx->dx < ctx->dy ? ctx->dx : ctx->dy;
    *dt = safety * hmin * hmin / rate;
    if (lambda_max) *lambda_max = lam;
    return GG_OK;
}

int gg_kernel_used(const gg_ctx* ctx) { return ctx ? resolve_kernel(ctx) : -1; }

const char* gg_kernel_name(const gg_ctx* ctx) {
    if (!ctx) return "";
    const char* T = ctx->dtype == GG_F64 ? "double" : "float";
    char buf[128];
    try {
        switch (resolve_kernel(ctx)) {
            case GG_KERNEL_GENERIC: snprintf(buf, sizeof buf, "gg_step_generic<%s>", T); break;
            case GG_KERNEL_RESIDENT:
                if (cluster_rows(ctx) > 0 && ctx->opt_resident_impl != 1) snprintf(buf, sizeof buf, "gg_step_cluster<%s,%d>", T, cluster_run_cells(ctx));
                else snprintf(buf, sizeof buf, "gg_step_resident<%s>", T);
                break;
            case GG_KERNEL_STREAM:
                if (!ctx->plan_ready) return "";
                snprintf(buf, sizeof buf, "gg_step_stream<%s,%d,%d,%d>", T, ctx->plan.rb, ctx->plan.nst, ctx->plan.nw); break;
            case GG_KERNEL_STREAM2:
                if (!ctx->plan2_ready) return "";
                snprintf(buf, sizeof buf, "gg_step_stream2<%s,%d,%d,%d,%d>", T, ctx->plan2.rb, ctx->plan2.nst, ctx->plan2.nst1, ctx->plan2.nw); break;
            case GG_KERNEL_PAIR:
                if (!ctx->pair.ready) return "";
                snprintf(buf, sizeof buf, "gg_step_pair<%s,%d,%d>", T, ctx->pair.rb, ctx->pair.nst); break;
            case GG_KERNEL_QUAD:
                if (!ctx->quad.ready) return "";
                snprintf(buf, sizeof buf, "gg_step_quad<%s,%d,%d,%d,%d,%d>", T, ctx->quad.rb, ctx->quad.nst, ctx->quad.nst1, ctx->quad.nstc, ctx->quad.nw); break;
            default: return "";
        }
        ctx->kname = buf;
    } catch (...) {
        return "";
    }
    return ctx->kname.c_str();
}
long long gg_launches(const gg_ctx* ctx) { return ctx ? ctx->launches : 0; }
long long gg_graph_captures(const gg_ctx* ctx) { return ctx ? ctx->graph_captures : 0; }

int gg_last_step_ms(gg_ctx* ctx, float* ms) {
    if (!ctx || !ms) return GG_ERR_ARG;
    *ms = -1.0f;
    if (!ctx->timed) return GG_OK;
    GG_CUDA(ctx, cudaEventSynchronize(ctx->ev1));
    GG_CUDA(ctx, cudaEventElapsedTime(ms, ctx->ev0, ctx->ev1));
    return GG_OK;
}

int gg_destroy(gg_ctx* ctx) {
    if (!ctx) return GG_OK;
    int rc = GG_OK;
    if (ctx->bound) {
        if (cudaStreamSynchronize(ctx->stream) != cudaSuccess) rc = GG_ERR_CUDA;
        drop_graphs(ctx);
        if (ctx->ev0) cudaEventDestroy(ctx->ev0);
        if (ctx->ev1) cudaEventDestroy(ctx->ev1);
    }
    delete ctx;
    return rc;
}

const char* gg_last_error(const gg_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }
int gg_num_stream_variants(void) { return kNumVariants; }
int gg_num_stream2_variants(void) { return kNumVariants2; }
int gg_num_pair_variants(void) { return kNumPairVariants; }
int gg_num_quad_variants(void) { return kNumQuadVariants; }
const char* gg_version(void) { return "gg-b200 0.2 sm_100a"; }

}  // extern "C"

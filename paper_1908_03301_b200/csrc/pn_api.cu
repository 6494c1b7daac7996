// pn_api.cu -- the C ABI of include/pn.h: handle, workspace carving, and the host side of the
// mixed-precision loop.  Every step of the path runs in the kernels
// of pn_setup.cu / pn_outer.cu / pn_inner.cu; this file only sequences them and reads back a few
// scalars per outer cycle.
//
// The loop ("SP inner loop ... DP outer loop", Fig.5 is a missing image; SURVEY.md 8(c) reading 4,
// "reliable updates"):
//   x64 = pins + initial guess;  r = b - A x64 in fp64 (S3)  ->  r_hat (fp32, scaled)
//   repeat: fp32 CG iterations on the scaled system (S4, S5) until the recursive residual has fallen
//           by `delta` since the last replacement, or below the proxy of the exit threshold;
//           x64 += s * x_hat (S7, fp64);  r = b - A x64 in fp64 (S3);  exit if ||r|| <= tol ||b||;
//           otherwise continue the SAME Krylov sequence (search direction kept, beta from the true
//           residual) -- the fp32 solver is never restarted.
#include <cstdio>
#include <cstring>
#include <cmath>
#include <new>

#include "pn_internal.cuh"

#define PN_HISTORY_MAX 256

struct pn_ctx {
    int unx, uny, unz;          // user lattice
    bool is2d;
    pn_geom g;                  // internal lattice (direction fields filled per solve)
    int device;
    cudaStream_t stream;
    char* ws;
    size_t ws_bytes;
    pn_ptrs P;
    float* raw_store[3];
    pn_state* h_state;          // pinned mirror
    cudaEvent_t ev[4];
    bool have_g, have_solution, ever_solved;
    int last_dir_user;
    // options
    int max_iters, chunk, x0_linear, skip_label, variant, profile, peel, lateral;
    int chunk_set;              // PN_OPT_CHUNK was set by the caller: it also bounds the persistent launches
    int base_closed;            // some in-lattice (non-wrap) bond is closed: from S0's validation
    // node classes kept from the last solve (S8(f) item 4): reused while no bond crosses zero and nothing they depend on changes
    int reuse_labels;           // option
    int compact;                // option: active-node compaction 0 off, 1 on, 2 automatic
    int contract;               // option: eliminate degree-2 chain nodes when compacting (pn_chain.cu)
    int label_chains, label_compact, label_contract, label_variant;   // what the kept node classes were made with
    bool labels_valid, topo_dirty, warm_next;
    int label_dir, label_lateral, label_peel, label_skip;
    // CUDA graph of one chunk of inner iterations (captured on a private stream, launched on the caller's)
    int use_graph, xdefer;
    cudaStream_t cap_stream;
    cudaGraphExec_t graph_exec;
    pn_geom graph_g;
    int graph_scheme, graph_chunk;
    long long graph_cm, graph_clong;   // compact scheme: the captured kernels carry pointers that depend on these
    pn_cptrs C;                 // compact arrays of the current solve (scheme 7)
    cudaEvent_t* pev;           // event pool for PN_OPT_PROFILE (2*chunk+1), created on demand
    int pev_n;
    double delta;
    long long launches;
    double flux[4];
    double hist[PN_HISTORY_MAX];   // true relative residual at every fp64 residual evaluation of the last solve
    int hist_n;
    bool flux_valid;
    char err[256];
};

namespace {

constexpr double PN_PEEL_MIN_FRACTION = 0.10;
constexpr double PN_COMPACT_MAX_FRACTION = 0.45;   // automatic compaction: unknowns per padded lattice node at most this

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct layout {
    pn_geom g;
    size_t off_raw[3], off_gs[3], off_w[3], off_gsw[3], off_ww[3], off_s, off_x64, off_r, off_p, off_p2, off_q, off_xh, off_r2, off_q2, off_cls, off_slots,
        off_state, off_xchg, off_gbar, total;
    size_t halo;                // elements in one halo plane
};

bool make_layout(int nx, int ny, int nz, layout* L) {
    if (nx < 1 || ny < 1 || nz < 1) return false;
    const bool is2d = (nz == 1);
    pn_geom& g = L->g;
    g.nx = nx;
    g.ny = is2d ? 1 : ny;
    g.nz = is2d ? ny : nz;
    g.px = (nx + 3) / 4 * 4;
    g.plane = (long long)g.px * g.ny;
    g.npad = g.plane * g.nz;
    g.n = (long long)nx * ny * nz;
    g.dir = 0; g.n_a = nx; g.stride_a = 1;
    g.wrap[0] = g.wrap[1] = g.wrap[2] = 0;
    g.sms = 0;
    g.coop = 0;
    g.tile = 0;
    if (g.npad + 2 * g.plane >= (1ll << 31)) return false;
    L->halo = (size_t)g.plane;
    const size_t vec = (size_t)g.npad + 2 * L->halo;   // elements of a padded array with its two halo planes
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes, 256); return at; };
    for (int b = 0; b < 3; ++b) L->off_raw[b] = take((size_t)g.n * 4);
    for (int b = 0; b < 3; ++b) L->off_gs[b] = take(vec * 4);
    for (int b = 0; b < 3; ++b) L->off_w[b] = take(vec * 4);
    for (int b = 0; b < 3; ++b) L->off_gsw[b] = take((size_t)pn_face_count(g, b) * 4);
    for (int b = 0; b < 3; ++b) L->off_ww[b] = take((size_t)pn_face_count(g, b) * 4);
    L->off_s = take(vec * 4);
    L->off_x64 = take(vec * 8);
    L->off_r = take(vec * 4);
    L->off_p = take(vec * 4);
    L->off_p2 = take(vec * 4);
    L->off_q = take(vec * 4);
    L->off_xh = take(vec * 4);
    L->off_r2 = take(vec * 4);
    L->off_q2 = take(vec * 4);
    L->off_cls = take(vec);
    L->off_slots = take(8 * PN_MAX_BLOCKS * sizeof(double));
    L->off_state = take(sizeof(pn_state));
    L->off_gbar = take(256);
    // exchange rows of the persistent 2D kernel (pn_resident.cu); (size_t)-1: not a lattice it handles
    L->off_xchg = (g.ny == 1 && g.px <= 2048) ? take((size_t)12 * PN_RESIDENT_MAX_CTAS * g.px * 4) : (size_t)-1;
    L->total = o;
    return true;
}

struct device_guard {
    int prev;
    bool ok;
    explicit device_guard(int dev) : prev(-1), ok(false) {
        if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; }
        ok = (cudaSetDevice(dev) == cudaSuccess);
    }
    ~device_guard() { if (prev >= 0) cudaSetDevice(prev); }
};

int fail_cuda(pn_ctx* c, cudaError_t e, const char* where) {
    if (c) snprintf(c->err, sizeof(c->err), "%s: %s", where, cudaGetErrorString(e));
    return PN_ERR_CUDA;
}

#define CK(call)                                                     \
    do {                                                             \
        cudaError_t e_ = (call);                                     \
        if (e_ != cudaSuccess) return fail_cuda(ctx, e_, #call);     \
    } while (0)

}  // namespace

extern "C" {

size_t pn_workspace_bytes(int nx, int ny, int nz) {
    layout L;
    if (!make_layout(nx, ny, nz, &L)) return 0;
    return L.total;
}

int pn_create(pn_ctx** out, int nx, int ny, int nz, int device, void* cuda_stream, void* workspace,
              size_t workspace_bytes) {
    if (!out) return PN_ERR_ARG;
    *out = nullptr;
    layout L;
    if (!make_layout(nx, ny, nz, &L)) return PN_ERR_ARG;
    if (!workspace || ((uintptr_t)workspace & 255) || workspace_bytes < L.total) return PN_ERR_WORKSPACE;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) { cudaGetLastError(); return PN_ERR_CUDA; }
    device_guard guard(device);
    if (!guard.ok) return PN_ERR_CUDA;
    pn_ctx* ctx = new (std::nothrow) pn_ctx;
    if (!ctx) return PN_ERR_ARG;
    memset(ctx, 0, sizeof(*ctx));
    ctx->unx = nx; ctx->uny = ny; ctx->unz = nz;
    ctx->is2d = (nz == 1);
    ctx->g = L.g;
    ctx->device = device;
    ctx->stream = (cudaStream_t)cuda_stream;
    ctx->ws = (char*)workspace;
    ctx->ws_bytes = workspace_bytes;
    ctx->max_iters = 200000; ctx->chunk = 32; ctx->chunk_set = 0; ctx->x0_linear = 1; ctx->skip_label = 0; ctx->variant = 0; ctx->peel = 2; ctx->use_graph = 1; ctx->xdefer = 1; ctx->reuse_labels = 1; ctx->compact = 2; ctx->contract = 1;
    ctx->delta = 0.3;   // measured: 0.3 needs 11 % fewer iterations than 0.1 on CFG2 2048^2 and the same on CFG3/4/5
    ctx->last_dir_user = -1;
    // per-handle device facts (no process-global state: handles on different devices are independent)
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess || sms < 1) sms = 148;
    ctx->g.sms = sms;
    int coop = 0;
    if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, device) != cudaSuccess) coop = 0;
    ctx->g.coop = coop;
    const size_t h = L.halo;
    pn_ptrs& P = ctx->P;
    for (int b = 0; b < 3; ++b) {
        ctx->raw_store[b] = (float*)(ctx->ws + L.off_raw[b]);
        P.gs[b] = (float*)(ctx->ws + L.off_gs[b]) + h;
        P.w[b] = (float*)(ctx->ws + L.off_w[b]) + h;
        P.gsw[b] = (float*)(ctx->ws + L.off_gsw[b]);
        P.ww[b] = (float*)(ctx->ws + L.off_ww[b]);
    }
    P.s = (float*)(ctx->ws + L.off_s) + h;
    P.x64 = (double*)(ctx->ws + L.off_x64) + h;
    P.r = (float*)(ctx->ws + L.off_r) + h;
    P.p = (float*)(ctx->ws + L.off_p) + h;
    P.p2 = (float*)(ctx->ws + L.off_p2) + h;
    P.q = (float*)(ctx->ws + L.off_q) + h;
    P.xh = (float*)(ctx->ws + L.off_xh) + h;
    P.r2 = (float*)(ctx->ws + L.off_r2) + h;
    P.q2 = (float*)(ctx->ws + L.off_q2) + h;
    P.cls = (signed char*)(ctx->ws + L.off_cls) + h;
    P.parent = (int*)P.q;
    P.flags = (int*)P.xh;
    P.slots = (double*)(ctx->ws + L.off_slots);
    P.st = (pn_state*)(ctx->ws + L.off_state);
    P.gbar = (unsigned int*)(ctx->ws + L.off_gbar);
    P.xchg = L.off_xchg == (size_t)-1 ? nullptr : (float*)(ctx->ws + L.off_xchg);
    P.scratch = (void*)(ctx->ws + L.off_p);   // p and p2 are adjacent: 8 bytes per padded node
    cudaError_t e = cudaMemsetAsync(ctx->ws, 0, L.total, ctx->stream);
    // large dynamic shared memory is opted into per DEVICE (the attribute is not per process)
    if (e == cudaSuccess && pn_tma_supported()) e = pn_fused_init_device();
    if (e == cudaSuccess) e = pn_onchip_init_device();
    if (e == cudaSuccess && pn_tma_supported()) e = pn_resident_init_device();
    if (e == cudaSuccess) e = cudaMallocHost((void**)&ctx->h_state, sizeof(pn_state));
    for (int i = 0; i < 4 && e == cudaSuccess; ++i) e = cudaEventCreate(&ctx->ev[i]);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) {
        if (ctx->h_state) cudaFreeHost(ctx->h_state);
        for (int i = 0; i < 4; ++i) if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
        delete ctx;
        cudaGetLastError();
        return PN_ERR_CUDA;
    }
    *out = ctx;
    return PN_OK;
}

int pn_destroy(pn_ctx* ctx) {
    if (!ctx) return PN_OK;
    device_guard guard(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    if (ctx->h_state) cudaFreeHost(ctx->h_state);
    for (int i = 0; i < 4; ++i) if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
    for (int i = 0; i < ctx->pev_n; ++i) cudaEventDestroy(ctx->pev[i]);
    delete[] ctx->pev;
    if (ctx->graph_exec) cudaGraphExecDestroy(ctx->graph_exec);
    if (ctx->cap_stream) cudaStreamDestroy(ctx->cap_stream);
    delete ctx;
    return PN_OK;
}

int pn_set_option(pn_ctx* ctx, int key, double value) {
    if (!ctx || !(value == value)) return PN_ERR_ARG;
    switch (key) {
        case PN_OPT_MAX_ITERS: if (value < 1 || value > 2e9) return PN_ERR_ARG; ctx->max_iters = (int)value; return PN_OK;
        case PN_OPT_DELTA: if (!(value > 0.0 && value < 1.0)) return PN_ERR_ARG; ctx->delta = value; return PN_OK;
        case PN_OPT_X0: if (value != 0.0 && value != 1.0 && value != 2.0) return PN_ERR_ARG; ctx->x0_linear = (int)value; return PN_OK;
        case PN_OPT_CHUNK: if (value < 1 || value > 4096) return PN_ERR_ARG; ctx->chunk = (int)value; ctx->chunk_set = 1; return PN_OK;
        case PN_OPT_SKIP_LABEL: if (value != 0.0 && value != 1.0) return PN_ERR_ARG; ctx->skip_label = (int)value; return PN_OK;
        case PN_OPT_KERNEL: if (value != 0.0 && value != 1.0 && value != 3.0 && value != 5.0 && value != 6.0 && value != 8.0) return PN_ERR_ARG; ctx->variant = (int)value; return PN_OK;
        case PN_OPT_PROFILE: if (value != 0.0 && value != 1.0) return PN_ERR_ARG; ctx->profile = (int)value; return PN_OK;
        case PN_OPT_LATERAL: if (value != 0.0 && value != 1.0) return PN_ERR_ARG; ctx->lateral = (int)value; return PN_OK;
        case PN_OPT_GRAPH: if (value != 0.0 && value != 1.0 && value != 2.0) return PN_ERR_ARG; ctx->use_graph = (int)value; return PN_OK;
        case PN_OPT_XDEFER: if (value != 0.0 && value != 1.0) return PN_ERR_ARG; ctx->xdefer = (int)value; return PN_OK;
        case PN_OPT_CONTRACT: if (value != 0.0 && value != 1.0) return PN_ERR_ARG; ctx->contract = (int)value; return PN_OK;
        case PN_OPT_TILE: if (value != 0.0 && value != 1.0 && value != 2.0 && value != 3.0) return PN_ERR_ARG; ctx->g.tile = (int)value; return PN_OK;
        case PN_OPT_COMPACT: if (value != 0.0 && value != 1.0 && value != 2.0) return PN_ERR_ARG; ctx->compact = (int)value; return PN_OK;
        case PN_OPT_REUSE_LABELS: if (value != 0.0 && value != 1.0) return PN_ERR_ARG; ctx->reuse_labels = (int)value; return PN_OK;
        case PN_OPT_PEEL: if (value != 0.0 && value != 1.0 && value != 2.0) return PN_ERR_ARG; ctx->peel = (int)value; return PN_OK;
        default: return PN_ERR_ARG;
    }
}

long long pn_launch_count(const pn_ctx* ctx) { return ctx ? ctx->launches : 0; }

int pn_residual_history(const pn_ctx* ctx, double* out, int capacity) {
    if (!ctx || capacity < 0 || (capacity > 0 && !out)) return PN_ERR_ARG;
    const int n = ctx->hist_n < capacity ? ctx->hist_n : capacity;
    for (int i = 0; i < n; ++i) out[i] = ctx->hist[i];
    return ctx->hist_n;
}

const char* pn_last_error(const pn_ctx* ctx) { return ctx ? ctx->err : ""; }

const char* pn_strerror(int code) {
    switch (code) {
        case PN_OK: return "ok";
        case PN_NO_SPANNING_CLUSTER: return "no cluster spans inlet to outlet (Q = 0)";
        case PN_MAX_ITERS: return "iteration budget spent or residual stagnated";
        case PN_ERR_ARG: return "bad argument";
        case PN_ERR_STATE: return "call out of order";
        case PN_ERR_VALUE: return "conductance negative or not finite";
        case PN_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
        case PN_ERR_CUDA: return "CUDA error";
        case PN_ERR_BREAKDOWN: return "conjugate-gradient breakdown";
        case PN_ERR_TOO_LARGE: return "more nodes than PN_NOALLOC_MAX_NODES (268435456): the fixed scratch array of pn_dissipation_noalloc does not hold them";
        default: return "unknown code";
    }
}

int pn_set_conductances(pn_ctx* ctx, const float* gx, const float* gy, const float* gz, int pointers_are_device) {
    if (!ctx || !gx || !gy) return PN_ERR_ARG;
    if ((ctx->unz == 1) != (gz == nullptr)) return PN_ERR_ARG;
    device_guard guard(ctx->device);
    if (!guard.ok) return fail_cuda(ctx, cudaGetLastError(), "cudaSetDevice");
    ctx->have_g = false;
    ctx->have_solution = false;
    ctx->flux_valid = false;
    ctx->labels_valid = false;   // a new network: classes, peeling and the warm start are void
    ctx->topo_dirty = false;
    ctx->warm_next = false;
    const size_t bytes = (size_t)ctx->g.n * 4;
    const cudaMemcpyKind kind = pointers_are_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    // internal axes: 2D lattices are held as nx x 1 x ny, so user gy feeds the internal z-bond array
    const float* src[3] = {gx, ctx->is2d ? nullptr : gy, ctx->is2d ? gy : gz};
    for (int b = 0; b < 3; ++b) {
        ctx->P.raw[b] = nullptr;
        if (!src[b]) continue;
        CK(cudaMemcpyAsync(ctx->raw_store[b], src[b], bytes, kind, ctx->stream));
        ctx->P.raw[b] = ctx->raw_store[b];
    }
    CK(cudaMemsetAsync(&ctx->P.st->bad_value, 0, 3 * sizeof(int), ctx->stream));
    int nl = 0;
    CK(pn_launch_validate(ctx->g, ctx->P, ctx->stream, &nl));
    ctx->launches += nl;
    CK(cudaMemcpyAsync(ctx->h_state, ctx->P.st, sizeof(pn_state), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    if (ctx->h_state->bad_value) return PN_ERR_VALUE;
    ctx->base_closed = ctx->h_state->any_closed;
    ctx->have_g = true;
    return PN_OK;
}

// field-by-field (a memcmp would also compare padding bytes and force needless re-captures)
static bool same_geom(const pn_geom& a, const pn_geom& b) {
    return a.nx == b.nx && a.ny == b.ny && a.nz == b.nz && a.px == b.px && a.plane == b.plane && a.npad == b.npad &&
           a.n == b.n && a.dir == b.dir && a.n_a == b.n_a && a.stride_a == b.stride_a && a.wrap[0] == b.wrap[0] &&
           a.wrap[1] == b.wrap[1] && a.wrap[2] == b.wrap[2] && a.sms == b.sms && a.tile == b.tile;
}

static int read_state(pn_ctx* ctx) {
    CK(cudaMemcpyAsync(ctx->h_state, ctx->P.st, sizeof(pn_state), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return PN_OK;
}

// One chunk of inner iterations as a CUDA graph: the launches carry no per-iteration host arguments (buffer
// parity, alpha, beta and the run flag are read on the device), so the same executable graph serves every chunk
// of a solve and every later solve with the same geometry, direction, scheme and chunk length.  Captured on a
// private stream (the caller's may be the legacy default stream, which cannot be captured); nothing executes
// there.  Returns false (graph_exec == nullptr) when capture is unavailable: the caller launches directly.
static bool ensure_graph(pn_ctx* ctx, int scheme, long long cm, long long clong) {
    if (ctx->graph_exec && ctx->graph_scheme == scheme && ctx->graph_chunk == ctx->chunk && ctx->graph_cm == cm && ctx->graph_clong == clong &&
        same_geom(ctx->graph_g, ctx->g))
        return true;
    if (ctx->graph_exec) { cudaGraphExecDestroy(ctx->graph_exec); ctx->graph_exec = nullptr; }
    if (!ctx->cap_stream && cudaStreamCreateWithFlags(&ctx->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
        ctx->cap_stream = nullptr;
        cudaGetLastError();
        return false;
    }
    int dummy = 0;
    // warm the launch path once outside capture is not needed: function attributes are set by the launchers themselves
    if (cudaStreamBeginCapture(ctx->cap_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); return false; }
    cudaError_t e = pn_launch_inner(ctx->g, ctx->P, ctx->chunk, scheme, ctx->cap_stream, &dummy, nullptr, &ctx->C);
    cudaGraph_t graph = nullptr;
    cudaError_t e2 = cudaStreamEndCapture(ctx->cap_stream, &graph);
    if (e != cudaSuccess || e2 != cudaSuccess || !graph) {
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        return false;
    }
    e = cudaGraphInstantiate(&ctx->graph_exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) { ctx->graph_exec = nullptr; cudaGetLastError(); return false; }
    ctx->graph_g = ctx->g;
    ctx->graph_scheme = scheme;
    ctx->graph_chunk = ctx->chunk;
    ctx->graph_cm = cm;
    ctx->graph_clong = clong;
    return true;
}

// `nl` counts the kernel launches enqueued, whatever the outcome (pn_solve adds it to the handle's total on every return path)
static int solve_impl(pn_ctx* ctx, int direction, double tol, pn_info* info, int& nl) {
    if (info) memset(info, 0, sizeof(*info));
    if (!ctx) return PN_ERR_ARG;
    if (direction < 0 || direction > 2 || !(tol > 0.0 && tol < 1.0)) return PN_ERR_ARG;
    if (ctx->is2d && direction == 2) return PN_ERR_ARG;
    const int ulen[3] = {ctx->unx, ctx->uny, ctx->unz};
    if (ulen[direction] < 3) return PN_ERR_ARG;
    if (!ctx->have_g) return PN_ERR_STATE;
    device_guard guard(ctx->device);
    if (!guard.ok) return fail_cuda(ctx, cudaGetLastError(), "cudaSetDevice");
    ctx->have_solution = false;
    ctx->flux_valid = false;
    pn_geom& g = ctx->g;
    g.dir = (ctx->is2d && direction == 1) ? 2 : direction;
    g.n_a = ulen[direction];
    g.stride_a = g.dir == 0 ? 1 : (g.dir == 1 ? g.px : g.plane);
    // periodic lateral faces: every internal axis but the solve axis wraps, if it has >= 2 nodes
    const int idims[3] = {g.nx, g.ny, g.nz};
    bool any_wrap = false;
    for (int b = 0; b < 3; ++b) { g.wrap[b] = (ctx->lateral == 1 && b != g.dir && idims[b] >= 2) ? 1 : 0; any_wrap |= g.wrap[b] != 0; }
    const pn_ptrs& P = ctx->P;
    cudaStream_t s = ctx->stream;
    int rc = PN_OK;

    // ---- S1 + set-up ----
    CK(cudaEventRecord(ctx->ev[0], s));
    // node classes of the previous solve still describe this network? (same direction and options, no bond crossed zero)
    const bool reuse = ctx->reuse_labels && ctx->labels_valid && !ctx->topo_dirty && ctx->label_dir == g.dir &&
                       ctx->label_lateral == ctx->lateral && ctx->label_peel == ctx->peel && ctx->label_skip == ctx->skip_label &&
                       ctx->label_compact == ctx->compact && ctx->label_contract == ctx->contract && ctx->label_variant == ctx->variant;
    ctx->labels_valid = false;   // until this solve's S1 has gone through
    CK(cudaMemsetAsync(P.st->acc, 0, sizeof(P.st->acc) + (reuse ? 0 : sizeof(P.st->count) + sizeof(P.st->n_peeled) + sizeof(P.st->n_chain)), s));
    CK(cudaMemsetAsync(&P.st->ticket, 0, sizeof(unsigned int), s));
    CK(cudaMemsetAsync(&P.st->iters, 0, sizeof(int), s));   // buffer parity of the first residual = 0
    int scheme = pn_resolve_variant(g, P, ctx->variant);
    int fused = scheme == 3 || scheme == 6 || scheme == 8;   // deferred residual update + predicted beta (the state holds the measured r.r)
    int bufmode = (scheme == 3 || scheme == 8) ? 1 : (scheme == 6 ? 2 : 0);   // where r, q, p live (pn_internal.cuh)
    // the fused TMA kernel stores no residual: three rotating direction slots (bufmode 3).  It runs as one persistent
    // launch per residual replacement (internal launch code 10) unless periodic faces need k_wrap_fix between the
    // iterations or PN_OPT_GRAPH = 0; 3D tiles only: the 2D tile (lattices above 12 M nodes) measured slower that way
    // and keeps the graph replay of single launches
    const bool persist_tma = scheme == 3 && ctx->use_graph && g.coop && !any_wrap && (g.ny > 1 || ctx->use_graph == 2);
    if (scheme == 3 || scheme == 8) bufmode = 3;   // (k_cg_persist, pn_inner.cu, works the same way)
    int any_closed = ctx->base_closed;
    if (any_wrap) {
        // the forward entries of the last nodes along the wrapping axes are bonds now: copy + validate them (S0's rules)
        CK(cudaMemsetAsync(&P.st->bad_value, 0, 3 * sizeof(int), s));
        CK(pn_launch_wrap_copy(g, P, s, &nl));
        rc = read_state(ctx);
        if (rc) return rc;
        if (ctx->h_state->bad_value) return PN_ERR_VALUE;
        any_closed |= ctx->h_state->any_closed;
    }
    const bool do_label = !ctx->skip_label && any_closed;
    const bool do_peel = do_label && ctx->peel;
    // warm start: asked for (PN_OPT_X0 = 2), or implied by pn_update_conductances / pn_replace_conductances unless the
    // caller insists on the zero start; nothing to start from before the first solve
    int x0_mode = ctx->x0_linear;
    if (ctx->warm_next && x0_mode != 0) x0_mode = 2;
    if (x0_mode == 2 && !ctx->ever_solved) x0_mode = 1;
    if (reuse) CK(pn_launch_label_reuse(g, P, x0_mode, s, &nl));
    else CK(pn_launch_label(g, P, do_label, do_peel, x0_mode, s, &nl));
    if (!reuse && do_peel && ctx->peel == 2) {
        // automatic: keep the peeling only if it removes at least PN_PEEL_MIN_FRACTION of the unknowns.  Peeled nodes are
        // still streamed (structured storage), so the gain is fewer iterations only; measured on B200:
        // 52 % peeled -> -28 % iterations (CFG3), 3.8 % peeled -> +1.8 % (CFG4: no gain)
        rc = read_state(ctx);
        if (rc) return rc;
        if ((double)ctx->h_state->n_peeled < PN_PEEL_MIN_FRACTION * (double)ctx->h_state->count[0]) {
            CK(pn_launch_unpeel(g, P, s, &nl));
            CK(cudaMemsetAsync(&P.st->n_peeled, 0, sizeof(P.st->n_peeled), s));
        }
    }
    // active-node compaction may apply (decided below, once the scaled weights exist): automatic only with the automatic
    // kernel choice -- an explicit PN_OPT_KERNEL is honoured unless PN_OPT_COMPACT = 1
    const bool compact_allowed = (ctx->compact == 1 || (ctx->compact == 2 && ctx->variant == 0)) && !any_wrap && (scheme == 3 || scheme == 1 || scheme == 8);
    // degree-2 chain nodes (pn_chain.cu) are eliminated together with the compaction: marked now, because the Jacobi scale
    // and the weights of the reduced system depend on them
    int chains = 0;
    if (compact_allowed && ctx->contract && do_label) {
        if (reuse) chains = ctx->label_chains;
        else {
            rc = read_state(ctx);
            if (rc) return rc;
            const double est = (double)ctx->h_state->count[0] - (double)ctx->h_state->n_peeled;
            if (ctx->compact == 1 || est <= PN_COMPACT_MAX_FRACTION * (double)g.npad) {
                CK(pn_launch_chain_mark(g, P, s, &nl));
                chains = 1;
            }
        }
    }
    CK(pn_launch_scale(g, P, chains, s, &nl));
    // parent / flags aliased q / x_hat: clear the CG vectors before the first iteration
    const size_t vbytes = (size_t)g.npad * 4;
    CK(cudaMemsetAsync(P.xh, 0, vbytes, s));
    CK(cudaMemsetAsync(P.q, 0, vbytes, s));
    if (scheme == 3 || scheme == 8) CK(cudaMemsetAsync(P.q2, 0, vbytes, s));
    // p / p2 double as export staging (pn_get_pressures), halo planes included: clear them whole
    const size_t vhalo = ((size_t)g.npad + 2 * (size_t)g.plane) * 4;
    CK(cudaMemsetAsync(P.p - g.plane, 0, vhalo, s));
    CK(cudaMemsetAsync(P.p2 - g.plane, 0, vhalo, s));
    // The iteration kernels read one plane beyond both ends of these arrays and rely on zeros there.
    // The compacted scheme and the chain records of an earlier solve on this handle borrow the same arrays: restore the
    // invariant instead of trusting every borrower (a second solve after one with the links eliminated broke down on a
    // 53 x 22 x 7 network: tests/golden/chain_case_53x22x7.npz)
    {
        float* const halo_arrays[] = {P.w[0], P.w[1], P.w[2], P.q, P.q2, P.r, P.r2, P.xh};
        const size_t hb = (size_t)g.plane * 4;
        for (float* a : halo_arrays) {
            if (!a) continue;
            CK(cudaMemsetAsync(a - g.plane, 0, hb, s));
            CK(cudaMemsetAsync(a + g.npad, 0, hb, s));
        }
    }
    // ---- active-node compaction (S8(f) item 1): when few lattice nodes are unknowns, iterate on the unknowns only ----
    // 66 bytes per unknown and iteration against 40 per lattice node: automatic below 0.45 unknowns per padded node.  The
    // compact arrays live in lattice-shaped arrays (npad entries each): pn_compact_fits.
    long long cm = 0, clong = 0;
    if (compact_allowed) {
        CK(pn_launch_compact_count(g, P, chains, s, &nl));
        rc = read_state(ctx);
        if (rc) return rc;
        const long long m = (long long)ctx->h_state->cm, nl_rows = (long long)ctx->h_state->clong;
        const bool want = ctx->compact == 1 || (double)m <= PN_COMPACT_MAX_FRACTION * (double)g.npad;
        if (want && pn_compact_fits(g, m, nl_rows)) {
            ctx->C = pn_compact_ptrs(g, P, m, nl_rows);
            CK(pn_launch_compact_build(g, P, ctx->C, m, chains, s, &nl));
            cm = m; clong = nl_rows;
            scheme = 7; fused = 1; bufmode = 2;
        } else if (chains) {   // no compaction after all: the structured kernels need every solved node as an unknown again
            CK(pn_launch_chain_unmark(g, P, s, &nl));
            CK(cudaMemsetAsync(&P.st->n_chain, 0, sizeof(P.st->n_chain), s));
            chains = 0;
            CK(pn_launch_scale(g, P, 0, s, &nl));
        }
    }
    ctx->labels_valid = true;
    ctx->topo_dirty = false;
    ctx->warm_next = false;
    ctx->label_dir = g.dir; ctx->label_lateral = ctx->lateral; ctx->label_peel = ctx->peel; ctx->label_skip = ctx->skip_label;
    ctx->label_chains = chains; ctx->label_compact = ctx->compact; ctx->label_contract = ctx->contract; ctx->label_variant = ctx->variant;
    // back-fill of the chain nodes: by one record per node written once per solve when the records fit the arrays the
    // compact form leaves free (else by walking the chains every time)
    long long n_rec = 0;
    if (chains && cm && (long long)ctx->h_state->n_chain <= ctx->C.chcap) {
        n_rec = (long long)ctx->h_state->n_chain;
        CK(pn_launch_chain_record(g, P, ctx->C, s, &nl));
    }
    auto chain_fill = [&]() -> cudaError_t {
        return n_rec ? pn_launch_chain_fill_rec(g, P, ctx->C, n_rec, s, &nl) : pn_launch_chain_fill(g, P, s, &nl);
    };
    if (chains) CK(chain_fill());   // chain nodes follow the starting pressures of their chains' ends
    CK(pn_launch_residual64(g, P, bufmode, s, &nl));
    if (cm) CK(pn_launch_compact_gather(g, P, ctx->C, cm, s, &nl));
    CK(cudaEventRecord(ctx->ev[1], s));
    rc = read_state(ctx);
    if (rc) return rc;
    pn_state* h = ctx->h_state;
    const long long n_solved = (long long)h->count[0];
    const long long n_peeled = (long long)h->n_peeled;
    const double nb = sqrt(h->acc[2]);
    double rn = sqrt(h->acc[0]);
    double rr_hat = h->acc[1];
    int outer = 1;
    ctx->hist_n = 0;
    if (nb > 0.0) ctx->hist[ctx->hist_n++] = rn / nb;
    int status = PN_OK;
    int total_iters = 0;
    double t_stencil = 0.0, t_update = 0.0;
    int n_timed = 0;
    if (ctx->profile && ctx->pev_n < 2 * ctx->chunk + 1) {
        for (int i = 0; i < ctx->pev_n; ++i) cudaEventDestroy(ctx->pev[i]);
        delete[] ctx->pev;
        ctx->pev_n = 0;   // counts the events that exist: pn_destroy never sees one that was not created
        const int want = 2 * ctx->chunk + 1;
        ctx->pev = new (std::nothrow) cudaEvent_t[want];
        if (!ctx->pev) return fail_cuda(ctx, cudaErrorMemoryAllocation, "event pool of PN_OPT_PROFILE");
        for (int i = 0; i < want; ++i) { CK(cudaEventCreate(&ctx->pev[i])); ctx->pev_n = i + 1; }
    }

    if (n_solved == 0 || !(nb > 0.0)) {
        status = PN_NO_SPANNING_CLUSTER;
        rn = 0.0;
    } else if (rn > tol * nb) {
        // (a smaller threshold for the compacted scheme, whose replacements cost 12 iterations' worth each, was tried: 0.1 saves
        // 6 % on CFG3 256^3 -- 17 -> 10 replacements, same 2135 iterations -- but costs 16 % more iterations on a harder
        // near-threshold case of the test suite, 18780 against 16233: 0.3 stays the default everywhere)
        const double delta2 = ctx->delta * ctx->delta;
        const double xskip_min = (fused && scheme != 7 && ctx->xdefer) ? 0.1 : 0.0;   // x_hat updated every other iteration (pn_fused_tma.cu)
        auto target_for = [&](double rn_true, double rr_true) {
            // proxy of the fp64 exit test in the scaled norm: ||r|| / ||r_hat|| measured at this replacement
            const double c = rn_true / sqrt(rr_true);
            const double t = 0.7 * tol * nb / c;
            return t * t;
        };
        CK(pn_launch_set_state(P, rr_hat, 0.0, rr_hat, target_for(rn, rr_hat), delta2, ctx->max_iters, 1, xskip_min, s, &nl));
        double best_rn = rn;
        int stagnant = 0;
        int iters_seen = 0;
        // Graph path: whole chunks replayed from one executable graph.  With PN_OPT_PROFILE it is used for the single-kernel
        // scheme only (one kernel per iteration: the chunk's device time / iterations run is that kernel's average launch
        // duration, gaps and the no-op tail included); the two-kernel schemes keep per-launch events to split S4 from S5.
        // compacted unknowns: PN_OPT_GRAPH = 1 means the persistent cooperative launch (one per residual replacement);
        // 0 the two kernels of an iteration launched one by one
        // the fused TMA kernel likewise (internal code 10), unless periodic faces need k_wrap_fix between the iterations
        const int lscheme = (scheme == 7 && ctx->use_graph && g.coop) ? 9
                            : ((scheme == 3 && persist_tma) ? 10 : scheme);
        const bool graph = ctx->use_graph && ctx->chunk > 1 && lscheme < 5 && !(ctx->profile && !fused) && ensure_graph(ctx, scheme, cm, clong);
        const int per_iter = (scheme == 3 ? 1 : 2) + (any_wrap ? 1 : 0);   // (scheme 7: two kernels, never with wrap)
        while (true) {
            if (graph) {
                if (ctx->profile) CK(cudaEventRecord(ctx->pev[0], s));
                CK(cudaGraphLaunch(ctx->graph_exec, s));
                if (ctx->profile) CK(cudaEventRecord(ctx->pev[1], s));
                nl += per_iter * ctx->chunk;
            } else {
                // (a persistent launch runs up to the next trigger, or PN_OPT_CHUNK iterations when the caller has set it)
                const bool one_launch = lscheme == 5 || lscheme == 6 || lscheme >= 8;
                CK(pn_launch_inner(g, P, (one_launch && !ctx->chunk_set) ? (1 << 30) : ctx->chunk, lscheme, s, &nl,
                                   ctx->profile ? ctx->pev : nullptr, &ctx->C));
            }
            rc = read_state(ctx);
            if (rc) return rc;
            if (ctx->profile && graph) {
                const int ran = h->iters - iters_seen;
                float ta = 0.f;
                cudaEventElapsedTime(&ta, ctx->pev[0], ctx->pev[1]);
                if (ran > 0) { t_stencil += ta; n_timed += ran; }
            } else if (ctx->profile && (lscheme == 5 || lscheme == 6 || lscheme >= 8)) {   // one launch ran `ran` iterations (on chip / persistent)
                const int ran = h->iters - iters_seen;
                float ta = 0.f;
                cudaEventElapsedTime(&ta, ctx->pev[0], ctx->pev[1]);
                if (ran > 0) { t_stencil += ta; n_timed += ran; }
            } else if (ctx->profile) {   // per-kernel device time of the launches that did work (not the no-op tail)
                const int ran = h->iters - iters_seen;
                for (int it = 0; it < ran && it < ctx->chunk; ++it) {
                    float ta = 0.f, tb = 0.f;
                    cudaEventElapsedTime(&ta, ctx->pev[2 * it], ctx->pev[2 * it + 1]);
                    cudaEventElapsedTime(&tb, ctx->pev[2 * it + 1], ctx->pev[2 * it + 2]);
                    t_stencil += ta; t_update += tb; ++n_timed;
                }
            }
            iters_seen = h->iters;
            if (h->flag == PN_FLAG_RUN) continue;
            total_iters = h->iters;
            if (h->flag == PN_FLAG_BREAKDOWN) { status = PN_ERR_BREAKDOWN; }
            // S7 + S3: fold the fp32 correction into x64 and recompute the true residual
            // beta's denominator = r.r of the residual that generated the last search direction: the two-kernel
            // iteration has already stepped past it (rr_old), the fused kernel holds it as its measured rr
            const double rr_before = fused ? h->rr : h->rr_old;
            const int flag = h->flag;
            if (cm) CK(pn_launch_compact_flush(g, P, ctx->C, cm, s, &nl));
            else CK(pn_launch_flush(g, P, bufmode, s, &nl));
            if (chains) CK(chain_fill());
            CK(pn_launch_residual64(g, P, bufmode, s, &nl));
            if (cm) CK(pn_launch_compact_gather(g, P, ctx->C, cm, s, &nl));
            rc = read_state(ctx);
            if (rc) return rc;
            ++outer;
            rn = sqrt(h->acc[0]);
            if (ctx->hist_n < PN_HISTORY_MAX) ctx->hist[ctx->hist_n++] = rn / nb;
            rr_hat = h->acc[1];
            if (status == PN_ERR_BREAKDOWN) break;
            if (rn <= tol * nb) break;
            if (flag == PN_FLAG_BUDGET || total_iters >= ctx->max_iters) { status = PN_MAX_ITERS; break; }
            if (rn < 0.9 * best_rn) { best_rn = rn; stagnant = 0; }
            else if (++stagnant >= 8) { status = PN_MAX_ITERS; break; }
            if (!(rr_hat > 0.0)) { status = PN_MAX_ITERS; break; }
            // continue the same Krylov sequence: beta = (true r.r) / (r.r before the last step)
            const double beta = rr_before > 0.0 ? rr_hat / rr_before : 0.0;
            CK(pn_launch_set_state(P, rr_hat, beta, rr_hat, target_for(rn, rr_hat), delta2, ctx->max_iters, 0, xskip_min, s, &nl));
        }
    }
    // (the last k_chain_fill ran before the last residual evaluation: the chain nodes are up to date)
    if (n_peeled > 0) CK(pn_launch_backfill(g, P, s, &nl));   // dangling ends take the pressure of the node they hang from
    CK(cudaEventRecord(ctx->ev[2], s));
    CK(cudaStreamSynchronize(s));
    ctx->have_solution = true;
    ctx->ever_solved = true;
    ctx->last_dir_user = direction;
    if (info) {
        float ms = 0.f;
        info->status = status;
        info->outer_cycles = outer;
        info->inner_iters = total_iters;
        info->kernel_scheme = scheme;
        info->n_xskip = h->n_xskip;
        info->rel_residual = nb > 0.0 ? rn / nb : 0.0;
        info->b_norm = nb;
        info->n_solved = n_solved;
        info->n_inlet_only = (long long)h->count[1];
        info->n_outlet_only = (long long)h->count[2];
        info->n_floating = (long long)h->count[3];
        info->n_peeled = n_peeled;
        info->labels_reused = reuse ? 1 : 0;
        info->residual_recovered = bufmode == 3 ? 1 : 0;
        info->n_unknowns = cm ? cm : n_solved - n_peeled;
        info->n_chain = (long long)h->n_chain;
        info->n_long_rows = clong;
        if (cudaEventElapsedTime(&ms, ctx->ev[0], ctx->ev[1]) == cudaSuccess) info->t_label_ms = ms;
        if (cudaEventElapsedTime(&ms, ctx->ev[1], ctx->ev[2]) == cudaSuccess) info->t_solve_ms = ms;
        info->t_stencil_ms = t_stencil;
        info->t_update_ms = t_update;
        info->n_timed_iters = n_timed;
    }
    return status;
}

// Shared tail of the two update calls: read the flags the kernels raised, keep the handle consistent.
static int finish_update(pn_ctx* ctx, int nl) {
    ctx->launches += nl;
    int rc = read_state(ctx);
    if (rc) return rc;
    const int bad = ctx->h_state->bad_value;
    if (bad) {   // some entries may have been written already: the handle keeps no network (as after a failed pn_set_conductances)
        ctx->have_g = false;
        ctx->labels_valid = false;
        return (bad & 1) ? PN_ERR_VALUE : PN_ERR_ARG;
    }
    if (ctx->h_state->topo_changed) {
        // a bond opened or closed: the classes are void, and whether ANY in-lattice bond is closed must be looked at again
        ctx->topo_dirty = true;
        CK(cudaMemsetAsync(&ctx->P.st->bad_value, 0, 3 * sizeof(int), ctx->stream));
        int nl2 = 0;
        CK(pn_launch_validate(ctx->g, ctx->P, ctx->stream, &nl2));
        ctx->launches += nl2;
        rc = read_state(ctx);
        if (rc) return rc;
        ctx->base_closed = ctx->h_state->any_closed;
    }
    ctx->have_solution = false;
    ctx->flux_valid = false;
    ctx->warm_next = true;
    return PN_OK;
}

int pn_update_conductances(pn_ctx* ctx, long long count, const int* axis, const long long* node, const float* value,
                           int pointers_are_device) {
    if (!ctx || count < 0 || (count > 0 && (!axis || !node || !value))) return PN_ERR_ARG;
    if (!ctx->have_g) return PN_ERR_STATE;
    if (count == 0) return PN_OK;
    device_guard guard(ctx->device);
    if (!guard.ok) return fail_cuda(ctx, cudaGetLastError(), "cudaSetDevice");
    cudaStream_t s = ctx->stream;
    CK(cudaMemsetAsync(&ctx->P.st->bad_value, 0, 3 * sizeof(int), s));
    int nl = 0;
    if (pointers_are_device) {
        CK(pn_launch_update_raw(ctx->unx, ctx->uny, ctx->unz, ctx->P, ctx->raw_store, count, axis, node, value, ctx->g.sms, s, &nl));
    } else {
        // host lists go through the export staging area (8 bytes per padded node), 16 bytes per entry, in pieces
        const long long cap = (long long)((size_t)ctx->g.npad * 8 / 16);
        char* stage = (char*)ctx->P.scratch;
        for (long long o = 0; o < count; o += cap) {
            const long long m = count - o < cap ? count - o : cap;
            long long* d_node = (long long*)stage;
            int* d_axis = (int*)(stage + (size_t)m * 8);
            float* d_val = (float*)(stage + (size_t)m * 12);
            CK(cudaMemcpyAsync(d_node, node + o, (size_t)m * 8, cudaMemcpyHostToDevice, s));
            CK(cudaMemcpyAsync(d_axis, axis + o, (size_t)m * 4, cudaMemcpyHostToDevice, s));
            CK(cudaMemcpyAsync(d_val, value + o, (size_t)m * 4, cudaMemcpyHostToDevice, s));
            CK(pn_launch_update_raw(ctx->unx, ctx->uny, ctx->unz, ctx->P, ctx->raw_store, m, d_axis, d_node, d_val, ctx->g.sms, s, &nl));
        }
    }
    return finish_update(ctx, nl);
}

int pn_replace_conductances(pn_ctx* ctx, const float* gx, const float* gy, const float* gz, int pointers_are_device) {
    if (!ctx || !gx || !gy) return PN_ERR_ARG;
    if ((ctx->unz == 1) != (gz == nullptr)) return PN_ERR_ARG;
    if (!ctx->have_g) return PN_ERR_STATE;
    device_guard guard(ctx->device);
    if (!guard.ok) return fail_cuda(ctx, cudaGetLastError(), "cudaSetDevice");
    cudaStream_t s = ctx->stream;
    CK(cudaMemsetAsync(&ctx->P.st->bad_value, 0, 3 * sizeof(int), s));
    const float* src[3] = {gx, ctx->is2d ? nullptr : gy, ctx->is2d ? gy : gz};
    const size_t bytes = (size_t)ctx->g.n * 4;
    int nl = 0;
    for (int b = 0; b < 3; ++b) {
        if (!src[b]) continue;
        const float* d_src = src[b];
        if (!pointers_are_device) {   // through the export staging area (8 bytes per padded node >= one array)
            CK(cudaMemcpyAsync(ctx->P.scratch, src[b], bytes, cudaMemcpyHostToDevice, s));
            d_src = (const float*)ctx->P.scratch;
        }
        CK(pn_launch_replace_raw(ctx->g, ctx->raw_store[b], d_src, b, ctx->P.st, s, &nl));
    }
    return finish_update(ctx, nl);
}

int pn_solve(pn_ctx* ctx, int direction, double tol, pn_info* info) {
    int nl = 0;
    pn_info local;
    memset(&local, 0, sizeof(local));
    int rc = solve_impl(ctx, direction, tol, &local, nl);
    // Safety net of PN_OPT_CONTRACT: if the iteration on the system with the links eliminated breaks down or stagnates
    // before its budget is spent, the solve is repeated once on the structured lattice kernels, without elimination and without
    // compaction (same network, labels redone: the path every other test exercises).  The one failure that led to it
    // (tests/golden/chain_case_53x22x7.npz, found by a random stress run) turned out to be stale halo planes left by the
    // borrowers of the lattice arrays -- fixed in solve_impl, where the halos are zeroed at every solve; the net stays.
    if (ctx && (rc == PN_ERR_BREAKDOWN || (rc == PN_MAX_ITERS && local.inner_iters < ctx->max_iters)) && local.n_chain > 0 &&
        ctx->contract) {
        const int saved_x0 = ctx->x0_linear, saved_compact = ctx->compact;
        ctx->contract = 0;
        ctx->compact = 0;
        ctx->labels_valid = false;
        ctx->warm_next = false;
        if (saved_x0 == 2) ctx->x0_linear = 1;          // the failed attempt's pressures are no starting point
        pn_info again;
        memset(&again, 0, sizeof(again));
        const int rc2 = solve_impl(ctx, direction, tol, &again, nl);
        ctx->contract = 1;
        ctx->compact = saved_compact;
        ctx->x0_linear = saved_x0;
        ctx->labels_valid = false;          // the next solve labels again, with the elimination
        again.outer_cycles += local.outer_cycles;      // the work of both attempts
        again.inner_iters += local.inner_iters;
        again.t_label_ms += local.t_label_ms + local.t_solve_ms;
        local = again;
        rc = rc2;
    }
    if (info) *info = local;
    if (ctx) ctx->launches += nl;
    return rc;
}

int pn_get_pressures(pn_ctx* ctx, double* out, int pointer_is_device) {
    if (!ctx || !out) return PN_ERR_ARG;
    if (!ctx->have_solution) return PN_ERR_STATE;
    device_guard guard(ctx->device);
    if (!guard.ok) return fail_cuda(ctx, cudaGetLastError(), "cudaSetDevice");
    const pn_geom& g = ctx->g;
    const size_t bytes = (size_t)g.n * sizeof(double);
    int nl = 0;
    if (g.px == g.nx) {   // padded layout == user layout
        CK(cudaMemcpyAsync(out, ctx->P.x64, bytes, pointer_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, ctx->stream));
    } else if (pointer_is_device) {
        CK(pn_launch_export_x(g, ctx->P, out, ctx->stream, &nl));
    } else {
        CK(pn_launch_export_x(g, ctx->P, (double*)ctx->P.scratch, ctx->stream, &nl));
        CK(cudaMemcpyAsync(out, ctx->P.scratch, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    }
    ctx->launches += nl;
    CK(cudaStreamSynchronize(ctx->stream));
    return PN_OK;
}

int pn_get_classes(pn_ctx* ctx, signed char* out, int pointer_is_device) {
    if (!ctx || !out) return PN_ERR_ARG;
    if (!ctx->have_solution) return PN_ERR_STATE;
    device_guard guard(ctx->device);
    if (!guard.ok) return fail_cuda(ctx, cudaGetLastError(), "cudaSetDevice");
    const pn_geom& g = ctx->g;
    int nl = 0;
    if (pointer_is_device) {
        CK(pn_launch_export_cls(g, ctx->P, out, 0, ctx->stream, &nl));
    } else {
        CK(pn_launch_export_cls(g, ctx->P, (signed char*)ctx->P.scratch, 0, ctx->stream, &nl));
        CK(cudaMemcpyAsync(out, ctx->P.scratch, (size_t)g.n, cudaMemcpyDeviceToHost, ctx->stream));
    }
    ctx->launches += nl;
    CK(cudaStreamSynchronize(ctx->stream));
    return PN_OK;
}

int pn_flux(pn_ctx* ctx, double* q_in, double* q_out, double* g_eff, double* k_eff) {
    if (!ctx) return PN_ERR_ARG;
    if (!ctx->have_solution) return PN_ERR_STATE;
    if (!ctx->flux_valid) {   // S8: one fused kernel over the two boundary planes, four scalars back
        device_guard guard(ctx->device);
        if (!guard.ok) return fail_cuda(ctx, cudaGetLastError(), "cudaSetDevice");
        const pn_geom& g = ctx->g;
        int nl = 0;
        CK(pn_launch_flux(g, ctx->P, ctx->stream, &nl));
        ctx->launches += nl;
        int rc = read_state(ctx);
        if (rc) return rc;
        const double qi = ctx->h_state->acc[0], qo = ctx->h_state->acc[1];
        const long long s_perp = g.n / g.n_a;
        ctx->flux[0] = qi;
        ctx->flux[1] = qo;
        ctx->flux[2] = 0.5 * (qi + qo);
        ctx->flux[3] = ctx->flux[2] * (double)(g.n_a - 1) / (double)s_perp;
        ctx->flux_valid = true;
    }
    if (q_in) *q_in = ctx->flux[0];
    if (q_out) *q_out = ctx->flux[1];
    if (g_eff) *g_eff = ctx->flux[2];
    if (k_eff) *k_eff = ctx->flux[3];
    return PN_OK;
}

int pn_dissipation(pn_ctx* ctx, double* g_e) {
    if (!ctx || !g_e) return PN_ERR_ARG;
    if (!ctx->have_solution) return PN_ERR_STATE;
    device_guard guard(ctx->device);
    if (!guard.ok) return fail_cuda(ctx, cudaGetLastError(), "cudaSetDevice");
    int nl = 0;
    CK(pn_launch_dissipation(ctx->g, ctx->P, ctx->stream, &nl));
    ctx->launches += nl;
    int rc = read_state(ctx);
    if (rc) return rc;
    *g_e = ctx->h_state->acc[3];
    return PN_OK;
}

}  // extern "C"

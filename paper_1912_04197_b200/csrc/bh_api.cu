// bh_api.cu — the C ABI declared in include/bh.h: context, workspace carving, call sequencing.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <atomic>
#include <new>

#include "bh_common.cuh"

using namespace bh;

struct bh_ctx {
    int64_t max_n = 0;
    int leaf_cap = 0;
    int group = kMaxGroup;   // W
    int group_cell = BH_GROUP_CELL_DEFAULT;   // Gc
    cudaStream_t stream = nullptr;
    int device = 0;          // ordinal of the device that was current at bh_create: the workspace, the stream and the
                             // per-device kernel attributes belong to it
    Workspace ws{};
    int64_t n = 0;          // bodies of the last build
    bool built = false;
    bool walked = false;
    bool no_mid = false;     // the one-kernel build of mid-size sets is not available (cooperative launch refused)
    // bound leapfrog state
    double *pos = nullptr, *vel = nullptr;
    const double *mass = nullptr;
    int64_t bound_n = 0;
    double theta = 0, eps = 0, G = 0;
    bool bound = false, have_acc = false;
    bool use_direct = false;   // steppers evaluate gravity by the direct N^2 sum instead of the tree
    bool acc_filled = false;   // ws.acc holds the accelerations of the last stepper evaluation
    // timing
    bool timing = false;
    cudaEvent_t ev[BH_NUM_PHASES][2]{};
    bool ev_set[BH_NUM_PHASES]{};
    // CUDA graph of one stepper call (sixteen launches per step with the streaming build)
    struct StepSig {
        int kind = -1, n_sub = 0;
        double dt = 0, theta = 0, eps = 0, G = 0;
        const void *pos = nullptr, *vel = nullptr, *mass = nullptr;
        int64_t n = 0;
        bool direct = false;
        cudaStream_t stream = nullptr;
        bool operator==(const StepSig &o) const
        {
            return kind == o.kind && n_sub == o.n_sub && dt == o.dt && theta == o.theta && eps == o.eps && G == o.G &&
                   pos == o.pos && vel == o.vel && mass == o.mass && n == o.n && direct == o.direct && stream == o.stream;
        }
    };
    cudaStream_t copy_stream = nullptr;   // bh_eval_host: mass upload beside the first build kernels
    cudaEvent_t ev_copy[2]{};
    bool use_graph = false;
    cudaGraphExec_t graph_exec = nullptr;
    StepSig graph_sig{}, seen_sig{};
    uint64_t graph_launches = 0;
    DevState *host_state = nullptr;   // pinned mirror for synchronising getters
    double *host_diag = nullptr;      // pinned, 16 doubles, after host_state
    uint64_t launches = 0;            // kernels launched so far (bench.py's gpu_launches)
    char err[256] = "";
};

namespace {

thread_local char g_err[256] = "";

bh_status fail(bh_ctx *c, bh_status s, const char *msg)
{
    snprintf(c ? c->err : g_err, 256, "%s", msg);
    return s;
}

bh_status cuda_check(bh_ctx *c, cudaError_t e, const char *what)
{
    if (e == cudaSuccess) return BH_OK;
    snprintf(c->err, 256, "%s: %s", what, cudaGetErrorString(e));
    return BH_ERR_CUDA;
}

// A context belongs to the device that was current at bh_create (workspace, stream, events, the SM count its grids
// are sized by).  A call made with another device current would launch there on foreign pointers: refuse it.
bh_status on_device(bh_ctx *c, const char *who)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return fail(c, BH_ERR_CUDA, "no current CUDA device");
    }
    if (dev != c->device) {
        snprintf(c->err, 256, "%s: the context was created on device %d, the current device is %d", who, c->device, dev);
        return BH_ERR_STATE;
    }
    return BH_OK;
}

inline size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

struct Carver {
    char *base;
    size_t off = 0;
    template <typename T>
    T *take(size_t count)
    {
        size_t at = off;
        off = align_up(off + count * sizeof(T));
        return base ? reinterpret_cast<T *>(base + at) : nullptr;
    }
};

struct Phase {   // records events around a phase when timing is on
    bh_ctx *c;
    int id;
    Phase(bh_ctx *ctx, int phase) : c(ctx), id(phase)
    {
        if (c->timing) cudaEventRecord(c->ev[id][0], c->stream);
    }
    ~Phase()
    {
        if (c->timing) {
            cudaEventRecord(c->ev[id][1], c->stream);
            c->ev_set[id] = true;
        }
    }
};

bh_status fetch_state(bh_ctx *c)   // synchronising
{
    cudaError_t e = cudaMemcpyAsync(c->host_state, c->ws.st, sizeof(DevState), cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_check(c, e, "state readback");
    const int s = c->host_state->status;
    if (s == 0) return BH_OK;
    // sticky until reported: the device word is cleared now that the caller is being told
    cudaMemsetAsync(&c->ws.st->status, 0, sizeof(int), c->stream);
    if (s & kStatNonFinite) return fail(c, BH_ERR_NONFINITE, "a body coordinate is NaN or infinite");
    if (s & kStatRange) return fail(c, BH_ERR_INVALID_ARG, "largest extent of the bodies outside [2^-300, 2^300]");
    if (s & kStatCapacity) return fail(c, BH_ERR_CAPACITY, "node array overflow");
    if (s & kStatStack) return fail(c, BH_ERR_CAPACITY, "walk stack overflow");
    if (s & kStatBpStack) return fail(c, BH_ERR_CAPACITY, "broad-phase search stack overflow");
    return BH_OK;
}

// cube_done: step a1 for these positions has already run (kick_drift_cube_kernel); only the streaming path takes note
bh_status do_build(bh_ctx *c, const double *pos, const double *mass, int64_t n, cudaEvent_t mass_ready = nullptr,
                   bool cube_done = false)
{
    const Workspace &w = c->ws;
    cudaStream_t s = c->stream;
    c->built = false;
    c->walked = false;
    // phases this build does not record read 0 (one-kernel builds record [4] only; a build whose cube came out of the
    // drift records no [0]), not what an earlier build left
    if (c->timing)
        for (int p = 0; p <= 5; ++p) c->ev_set[p] = false;
    if (n <= kSortTile) {   // one block does the whole build (and its own clearing): one launch
        if (mass_ready) cudaStreamWaitEvent(s, mass_ready, 0);   // masses copied on another stream
        {
            Phase p(c, 4);
            launch_build_small(w, pos, mass, n, s);
        }
        bh_status st1 = cuda_check(c, cudaGetLastError(), "bh_build launch");
        if (st1 != BH_OK) return st1;
        c->n = n;
        c->built = true;
        c->launches += 1;
        return BH_OK;
    }
    if (n <= mid_build_limit(w) && !c->no_mid) {   // one co-resident kernel with grid barriers instead of sixteen launches and two memsets
        if (mass_ready) cudaStreamWaitEvent(s, mass_ready, 0);
        int launched;
        {
            Phase p(c, 4);
            launched = launch_build_mid(w, pos, mass, n, s);
        }
        if (launched > 0) {
            bh_status st1 = cuda_check(c, cudaGetLastError(), "bh_build launch");
            if (st1 != BH_OK) return st1;
            c->n = n;
            c->built = true;
            c->launches += 1;
            return BH_OK;
        }
        cudaGetLastError();     // cooperative launch not available here: the streaming kernels from now on
        c->no_mid = true;
    }
    int sort_launches = 0;
    // what a build clears (histograms, tickets, look-back rows of this n, child masks / arrival counters, sized by n and
    // not by max_n) is cleared by its first kernel: cube_kernel, or the drift that took the cube (bh_keys.cu)
    if (!cube_done) {
        Phase p(c, 0);
        launch_cube(w, pos, n, s);
    }
    {
        Phase p(c, 1);
        launch_keys(w, pos, n, s);
    }
    {
        Phase p(c, 2);
        sort_launches = launch_sort(w, pos, n, s);
    }
    if (sort_launches < 0) return fail(c, BH_ERR_CUDA, "bh_build: the sort could not be enqueued");
    {
        Phase p(c, 4);
        launch_tree(w, n, c->leaf_cap, s);                       // from the sorted keys alone
    }
    {
        Phase p(c, 3);
        if (mass_ready) cudaStreamWaitEvent(s, mass_ready, 0);   // masses copied on another stream
        launch_gather_boxes(w, pos, mass, n, s);                 // sorted bodies + group boxes, a warp per group
    }
    {
        Phase p(c, 5);
        launch_monopoles(w, n, s);
    }
    bh_status st = cuda_check(c, cudaGetLastError(), "bh_build launch");
    if (st != BH_OK) return st;
    c->n = n;
    c->built = true;
    c->launches += (cube_done ? 1 : 2) + sort_launches + 3 + 1 + 1;   // cube, keys, sort (5 passes + repair + fallback), tree (3), gather + boxes, monopoles
    return BH_OK;
}

bh_status do_accel(bh_ctx *c, double theta, double eps, double G, double *acc, int mode = 0, double *phi = nullptr)
{
    const Workspace &w = c->ws;
    // The counters of this evaluation: the build zeroes them, so only a second walk of the same build clears
    // them here.  The group queue is reset by the walk kernel itself when its last producer warp leaves.
    if (c->walked) cudaMemsetAsync(&w.st->stats[0], 0, kNumStats * sizeof(unsigned long long), c->stream);
    {
        Phase p(c, 6);
        launch_walk(w, c->n, theta, eps, G, acc, mode, phi, c->stream);
    }
    bh_status st = cuda_check(c, cudaGetLastError(), "bh_accel launch");
    if (st == BH_OK) {
        c->walked = true;
        c->launches += 1;
    }
    return st;
}

// One gravity evaluation of the bound state into ws.acc, by the method bh_set_gravity_method chose
// ("through N^2 interactions or by building the octree").
bh_status do_eval_state(bh_ctx *c, bool cube_done = false)
{
    if (c->timing) {   // the stepper's evaluation is a tree walk or a direct sum: the other one's phase reads 0
        if (c->use_direct)
            for (int p = 0; p <= 6; ++p) c->ev_set[p] = false;
        else
            c->ev_set[7] = false;
    }
    if (!c->use_direct) {
        bh_status st = do_build(c, c->pos, c->mass, c->bound_n, nullptr, cube_done);
        if (st != BH_OK) return st;
        return do_accel(c, c->theta, c->eps, c->G, c->ws.acc);
    }
    // direct sum: no tree, bodies packed in their own order
    c->built = false;
    c->walked = false;
    launch_pack(c->ws, c->pos, c->mass, c->bound_n, c->stream);
    {
        Phase p(c, 7);
        c->launches += 1 + launch_direct(c->ws, c->bound_n, nullptr, c->bound_n, c->eps, c->G, c->ws.acc, false, c->stream);
    }
    return cuda_check(c, cudaGetLastError(), "direct evaluation launch");
}

// Run one stepper call, through a CUDA graph when bh_set_graph is on: the first call with a given
// signature (stepper, dt, state pointers, parameters) runs plainly, the second is captured while it is
// enqueued, later ones replay the graph.  All kernel arguments are pointers into the workspace or the
// bound state and values of the signature, so a replay does exactly what a plain call would.
template <typename F>
bh_status run_stepper(bh_ctx *c, int kind, double dt, int n_sub, F enqueue)
{
    if (!c->use_graph || c->timing) return enqueue();
    bh_ctx::StepSig sig;
    sig.kind = kind; sig.n_sub = n_sub; sig.dt = dt; sig.theta = c->theta; sig.eps = c->eps; sig.G = c->G;
    sig.pos = c->pos; sig.vel = c->vel; sig.mass = c->mass; sig.n = c->bound_n; sig.direct = c->use_direct;
    sig.stream = c->stream;
    if (c->graph_exec && sig == c->graph_sig) {   // the callers refresh built / walked / n (stepper_done)
        c->launches += c->graph_launches;
        return cuda_check(c, cudaGraphLaunch(c->graph_exec, c->stream), "stepper graph launch");
    }
    if (!(sig == c->seen_sig)) {
        c->seen_sig = sig;
        return enqueue();
    }
    if (c->graph_exec) {
        cudaGraphExecDestroy(c->graph_exec);
        c->graph_exec = nullptr;
    }
    const uint64_t l0 = c->launches;
    if (cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
        cudaGetLastError();
        c->use_graph = false;
        return enqueue();
    }
    bh_status st = enqueue();
    cudaGraph_t g = nullptr;
    cudaError_t e = cudaStreamEndCapture(c->stream, &g);
    if (st == BH_OK && e == cudaSuccess && g) e = cudaGraphInstantiate(&c->graph_exec, g, 0);
    if (g) cudaGraphDestroy(g);
    if (st != BH_OK || e != cudaSuccess || !c->graph_exec) {   // capture failed: nothing ran; fall back for good
        cudaGetLastError();
        c->graph_exec = nullptr;
        c->use_graph = false;
        c->launches = l0;
        return enqueue();
    }
    c->graph_sig = sig;
    c->graph_launches = c->launches - l0;
    return cuda_check(c, cudaGraphLaunch(c->graph_exec, c->stream), "stepper graph launch");
}

}  // namespace

namespace bh {

int current_device()
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    return dev >= 0 && dev < kMaxDevices ? dev : 0;
}

int sm_count()
{
    static std::atomic<int> sms[kMaxDevices];   // per device ordinal; 0 = not asked yet
    const int dev = current_device();
    int v = sms[dev].load(std::memory_order_relaxed);
    if (v == 0) {
        int cur = 0;
        if (cudaGetDevice(&cur) == cudaSuccess &&
            cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, cur) == cudaSuccess && v > 0) {
            sms[dev].store(v, std::memory_order_relaxed);
        } else {
            cudaGetLastError();
            return kDefaultSMs;   // no device (yet): not cached
        }
    }
    return v;
}

Workspace carve(char *base, int64_t max_n, int leaf_cap)
{
    Workspace w{};
    Carver cv{base};
    const int64_t n = max_n;
    w.sms = sm_count();
    w.leaf_cap = leaf_cap;
    w.group_w = kMaxGroup;
    w.group_cell = BH_GROUP_CELL_DEFAULT;
    w.node_cap = node_capacity(n, leaf_cap);
    {   // most tiles any n <= max_n can have (2048-key tiles below kSortSmallTileBelow keys, 4096-key tiles from there)
        const int64_t small_n = n < kSortSmallTileBelow ? n : kSortSmallTileBelow - 1;
        const int64_t t8 = (small_n + kSortThreads * 8 - 1) / (kSortThreads * 8), t16 = (n + kSortTile - 1) / kSortTile;
        w.sort_tiles = t8 > t16 ? t8 : t16;
    }
    w.tree_tiles = (n + kTreeTile - 1) / kTreeTile;
    w.walk_warps = w.sms * WalkConfig::kPairsPerBlock;
    const int64_t groups = n;   // capacity: a group holds at least one body
    w.st = cv.take<DevState>(1);
    w.bbox_part = cv.take<double>(kMaxBboxBlocks * 8);
    // --- region cleared by one memset at every build ---
    size_t z0 = cv.off;
    w.hist = cv.take<unsigned>(kSortPasses * kRadix);
    w.zero_begin = w.hist;
    w.sort_ticket = cv.take<unsigned>(kSortPasses);
    w.lookback = cv.take<unsigned>((size_t)kSortPasses * w.sort_tiles * kRadix);
    w.node_meta = cv.take<unsigned>(w.node_cap);
    w.zero_bytes = cv.off - z0;
    // ---
    w.key[0] = cv.take<unsigned long long>(n);
    w.key[1] = cv.take<unsigned long long>(n);
    w.idx[0] = cv.take<unsigned>(n);
    w.idx[1] = cv.take<unsigned>(n);
    w.iperm = cv.take<unsigned>(n);
    w.sbody = cv.take<double4>(n);
    w.gstart = cv.take<unsigned>(groups + 1);
    w.gbox = cv.take<double>(6 * groups);
    w.dlev = cv.take<uchar4>(n);
    w.tile_lvl = cv.take<unsigned>((size_t)(kLevels + 1) * w.tree_tiles);
    w.nlevel = cv.take<unsigned char>(w.node_cap);
    w.nbegin = cv.take<unsigned>(w.node_cap);
    w.ncount = cv.take<unsigned>(w.node_cap);
    w.nfirst = cv.take<int>(w.node_cap);
    w.nparent = cv.take<int>(w.node_cap);
    w.mono = cv.take<double4>(w.node_cap);
    w.winfo = cv.take<uint4>(w.node_cap);
    w.cnt_mono = cv.take<unsigned>(groups);
    w.cnt_direct = cv.take<unsigned>(groups);
    w.walk_stack = cv.take<unsigned>((size_t)w.walk_warps * kStackSlab * 2);
    w.acc = cv.take<double>(3 * n);
    w.stage_pos = cv.take<double>(3 * n);
    w.stage_doubles = 3 * n;
    w.stage_mass = cv.take<double>(n);
    w.diag_part = cv.take<double>((size_t)kDiagBlocks * 16);
    w.diag_out = cv.take<double>(16);
    w.diag_ticket = base ? &w.st->ticket_diag : nullptr;
    w.bsort = cv.take<double>(n);
    w.box_lo = cv.take<double4>(w.node_cap);
    w.box_hi = cv.take<double4>(w.node_cap);
    w.bp_cnt = cv.take<unsigned>(w.node_cap);
    w.agg_size = cv.take<int>(n);
    w.total_bytes = cv.off;
    return w;
}

}  // namespace bh

// message of a call that has no context (bh_diagnostics_static, bh_diag.cu): what bh_last_error(NULL) returns
void bh::set_global_error(const char *msg) { snprintf(g_err, 256, "%s", msg); }

extern "C" {

const char *bh_version(void) { return "bh-b200 0.1 (sm_100a)"; }

const char *bh_last_error(const bh_ctx *ctx) { return ctx ? ctx->err : g_err; }

static bool args_ok(int64_t max_n, int leaf_cap, int group_size)
{
    return max_n >= 1 && max_n <= ((int64_t)1 << 30) && leaf_cap >= 1 && leaf_cap <= 1024 &&
           group_size >= 0 && group_size <= kMaxGroup;
}

size_t bh_workspace_bytes(int64_t max_n, int leaf_cap, int group_size)
{
    if (!args_ok(max_n, leaf_cap, group_size)) return 0;
    return carve(nullptr, max_n, leaf_cap).total_bytes;
}

bh_status bh_create(bh_ctx **out, int64_t max_n, int leaf_cap, int group_size, void *workspace_dev,
                    size_t workspace_bytes, void *cuda_stream)
{
    if (!out) return fail(nullptr, BH_ERR_INVALID_ARG, "out is null");
    *out = nullptr;
    if (!args_ok(max_n, leaf_cap, group_size))
        return fail(nullptr, BH_ERR_INVALID_ARG, "max_n, leaf_cap or group_size out of range");
    if (!workspace_dev || ((uintptr_t)workspace_dev & 255))
        return fail(nullptr, BH_ERR_INVALID_ARG, "workspace is null or not 256-byte aligned");
    Workspace w = carve((char *)workspace_dev, max_n, leaf_cap);
    if (workspace_bytes < w.total_bytes) return fail(nullptr, BH_ERR_CAPACITY, "workspace too small");
    bh_ctx *c = new (std::nothrow) bh_ctx();
    if (!c) return fail(nullptr, BH_ERR_CAPACITY, "out of host memory");
    c->max_n = max_n;
    c->leaf_cap = leaf_cap;
    c->stream = (cudaStream_t)cuda_stream;
    c->group = group_size == 0 ? kMaxGroup : group_size;
    w.group_w = c->group;
    c->ws = w;
    const size_t hs = (sizeof(DevState) + 63) & ~(size_t)63;
    cudaError_t e = cudaGetDevice(&c->device);
    if (e == cudaSuccess) e = cudaMallocHost((void **)&c->host_state, hs + 16 * sizeof(double));
    if (e == cudaSuccess) c->host_diag = reinterpret_cast<double *>(reinterpret_cast<char *>(c->host_state) + hs);
    if (e == cudaSuccess) e = cudaMemsetAsync(w.st, 0, sizeof(DevState), c->stream);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking);
    for (int k = 0; k < 2 && e == cudaSuccess; ++k) e = cudaEventCreateWithFlags(&c->ev_copy[k], cudaEventDisableTiming);
    for (int p = 0; p < BH_NUM_PHASES && e == cudaSuccess; ++p) {
        e = cudaEventCreate(&c->ev[p][0]);
        if (e == cudaSuccess) e = cudaEventCreate(&c->ev[p][1]);
    }
    if (e != cudaSuccess) {
        snprintf(g_err, 256, "bh_create: %s", cudaGetErrorString(e));
        if (c->host_state) cudaFreeHost(c->host_state);
        if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
        for (int k = 0; k < 2; ++k)
            if (c->ev_copy[k]) cudaEventDestroy(c->ev_copy[k]);
        delete c;
        return BH_ERR_CUDA;
    }
    *out = c;
    return BH_OK;
}

bh_status bh_destroy(bh_ctx *c)
{
    if (!c) return BH_ERR_INVALID_ARG;
    cudaStreamSynchronize(c->stream);
    for (int p = 0; p < BH_NUM_PHASES; ++p) {
        if (c->ev[p][0]) cudaEventDestroy(c->ev[p][0]);
        if (c->ev[p][1]) cudaEventDestroy(c->ev[p][1]);
    }
    if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
    if (c->copy_stream) {
        cudaStreamSynchronize(c->copy_stream);
        cudaStreamDestroy(c->copy_stream);
    }
    for (int k = 0; k < 2; ++k)
        if (c->ev_copy[k]) cudaEventDestroy(c->ev_copy[k]);
    if (c->host_state) cudaFreeHost(c->host_state);
    delete c;
    return BH_OK;
}

bh_status bh_set_stream(bh_ctx *c, void *cuda_stream)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_set_stream")) return ds;
    cudaStreamSynchronize(c->stream);
    c->stream = (cudaStream_t)cuda_stream;
    return BH_OK;
}

bh_status bh_build(bh_ctx *c, const double *pos_dev, const double *mass_dev, int64_t n)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_build")) return ds;
    if (!pos_dev || !mass_dev) return fail(c, BH_ERR_INVALID_ARG, "bh_build: null pointer");
    if (n < 1 || n > c->max_n) return fail(c, BH_ERR_INVALID_ARG, "bh_build: n out of range");
    return do_build(c, pos_dev, mass_dev, n);
}

bh_status bh_accel(bh_ctx *c, double theta, double eps, double G, double *acc_dev)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_accel")) return ds;
    if (!c->built) return fail(c, BH_ERR_STATE, "bh_accel before bh_build");
    if (!acc_dev) return fail(c, BH_ERR_INVALID_ARG, "bh_accel: null pointer");
    if (!(theta >= 0.0) || !(eps >= 0.0)) return fail(c, BH_ERR_INVALID_ARG, "bh_accel: theta or eps negative");
    return do_accel(c, theta, eps, G, acc_dev);
}

bh_status bh_direct(bh_ctx *c, double eps, double G, double *acc_dev)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_direct")) return ds;
    if (!c->built) return fail(c, BH_ERR_STATE, "bh_direct before bh_build");
    if (!acc_dev) return fail(c, BH_ERR_INVALID_ARG, "bh_direct: null pointer");
    if (!(eps >= 0.0)) return fail(c, BH_ERR_INVALID_ARG, "bh_direct: eps negative");
    {
        Phase p(c, 7);
        c->launches += launch_direct(c->ws, c->n, nullptr, c->n, eps, G, acc_dev, false, c->stream);
    }
    return cuda_check(c, cudaGetLastError(), "bh_direct launch");
}

bh_status bh_direct_targets(bh_ctx *c, const int32_t *tgt_dev, int64_t nt, double eps, double G, double *acc_dev)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_direct_targets")) return ds;
    if (!c->built) return fail(c, BH_ERR_STATE, "bh_direct_targets before bh_build");
    if (!acc_dev || !tgt_dev) return fail(c, BH_ERR_INVALID_ARG, "bh_direct_targets: null pointer");
    if (nt < 1 || !(eps >= 0.0)) return fail(c, BH_ERR_INVALID_ARG, "bh_direct_targets: nt < 1 or eps negative");
    {
        Phase p(c, 7);
        c->launches += launch_direct(c->ws, c->n, tgt_dev, nt, eps, G, acc_dev, false, c->stream);
    }
    return cuda_check(c, cudaGetLastError(), "bh_direct_targets launch");
}

bh_status bh_bind_state(bh_ctx *c, double *pos_dev, double *vel_dev, const double *mass_dev, int64_t n,
                        double theta, double eps, double G)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_bind_state")) return ds;
    if (!pos_dev || !vel_dev || !mass_dev) return fail(c, BH_ERR_INVALID_ARG, "bh_bind_state: null pointer");
    if (n < 1 || n > c->max_n) return fail(c, BH_ERR_INVALID_ARG, "bh_bind_state: n out of range");
    if (!(theta >= 0.0) || !(eps >= 0.0)) return fail(c, BH_ERR_INVALID_ARG, "bh_bind_state: theta or eps negative");
    c->pos = pos_dev;
    c->vel = vel_dev;
    c->mass = mass_dev;
    c->bound_n = n;
    c->theta = theta;
    c->eps = eps;
    c->G = G;
    c->bound = true;
    c->have_acc = false;
    c->acc_filled = false;
    return BH_OK;
}

bh_status bh_set_group_cell(bh_ctx *c, int group_cell)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (group_cell < 1 || group_cell > kMaxGroupCell) return fail(c, BH_ERR_INVALID_ARG, "bh_set_group_cell: Gc out of range");
    c->group_cell = group_cell;
    c->ws.group_cell = group_cell;
    c->seen_sig = bh_ctx::StepSig{};   // a captured stepper graph holds the old Gc as a kernel argument
    if (c->graph_exec) {
        cudaGraphExecDestroy(c->graph_exec);
        c->graph_exec = nullptr;
    }
    return BH_OK;
}

bh_status bh_set_graph(bh_ctx *c, int enable)
{
    if (!c) return BH_ERR_INVALID_ARG;
    c->use_graph = enable != 0;
    if (!c->use_graph && c->graph_exec) {
        cudaGraphExecDestroy(c->graph_exec);
        c->graph_exec = nullptr;
    }
    c->seen_sig = bh_ctx::StepSig{};
    return BH_OK;
}

static bh_status kdk_enqueue(bh_ctx *c, double dt);

// Host-side view of the context after a stepper call, whichever way it ran (plain, captured or replayed
// graph): a replay does on the device what a plain call does, so the flags must say the same.  Tree
// method: the context holds the tree and the walk of the bound state's n bodies.  Direct method: the
// sorted-body arrays were overwritten by the identity packing, so it holds no tree.
static void stepper_done(bh_ctx *c, bool acc_is_current)
{
    c->have_acc = acc_is_current;
    c->acc_filled = true;
    c->n = c->bound_n;
    c->built = c->walked = !c->use_direct;
}

bh_status bh_kdk_step(bh_ctx *c, double dt)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_kdk_step")) return ds;
    if (!c->bound) return fail(c, BH_ERR_STATE, "bh_kdk_step before bh_bind_state");
    // the first step also evaluates a(x0): not the repeating pattern
    const bh_status st = !c->have_acc ? kdk_enqueue(c, dt) : run_stepper(c, 0, dt, 0, [=]() { return kdk_enqueue(c, dt); });
    if (st == BH_OK) stepper_done(c, true);
    return st;
}

static bh_status kdk_enqueue(bh_ctx *c, double dt)
{
    bh_status st;
    if (!c->have_acc) {   // a(x0), once
        if ((st = do_eval_state(c)) != BH_OK) return st;
        c->have_acc = true;
    }
    if (c->timing) cudaEventRecord(c->ev[8][0], c->stream);
    // above the one-kernel builds' sizes the drift also takes the bounding cube of the positions it writes (step a1)
    const bool with_cube = !c->use_direct && c->bound_n > mid_build_limit(c->ws);
    if (with_cube) launch_kick_drift_cube(c->ws, c->pos, c->vel, c->ws.acc, c->bound_n, dt, c->stream);
    else launch_kick_drift(c->pos, c->vel, c->ws.acc, c->bound_n, dt, c->stream);
    if (c->timing) {
        cudaEventRecord(c->ev[8][1], c->stream);
        c->ev_set[8] = true;
    }
    if ((st = do_eval_state(c, with_cube)) != BH_OK) return st;
    launch_kick(c->vel, c->ws.acc, c->bound_n, dt * 0.5, c->stream);
    c->acc_filled = true;
    c->launches += 2;   // kick+drift, kick
    return cuda_check(c, cudaGetLastError(), "bh_kdk_step launch");
}

/* ---- rows "next": paper's stepping variants and conservation diagnostics ---- */
static bh_status euler_enqueue(bh_ctx *c, double dt, int n_sub, const char *who);

static bh_status euler_like(bh_ctx *c, double dt, int n_sub, const char *who)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "stepper")) return ds;
    if (!c->bound) return fail(c, BH_ERR_STATE, "stepper called before bh_bind_state");
    if (n_sub < 1) return fail(c, BH_ERR_INVALID_ARG, "n_sub < 1");
    const bh_status st = run_stepper(c, 1, dt, n_sub, [=]() { return euler_enqueue(c, dt, n_sub, who); });
    if (st == BH_OK) stepper_done(c, false);   // acc is a(x_k), not a(x_k+1): a later bh_kdk_step re-evaluates
    return st;
}

static bh_status euler_enqueue(bh_ctx *c, double dt, int n_sub, const char *who)
{
    bh_status st;
    if ((st = do_eval_state(c)) != BH_OK) return st;
    c->have_acc = false;   // acc is a(x_k), not a(x_k+1): a later bh_kdk_step re-evaluates
    c->acc_filled = true;
    if (c->timing) cudaEventRecord(c->ev[8][0], c->stream);
    launch_euler_sub(c->pos, c->vel, c->ws.acc, c->bound_n, dt, n_sub, c->stream);
    if (c->timing) {
        cudaEventRecord(c->ev[8][1], c->stream);
        c->ev_set[8] = true;
    }
    c->launches += 1;
    return cuda_check(c, cudaGetLastError(), who);
}

bh_status bh_set_gravity_method(bh_ctx *c, int method)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (method != 0 && method != 1) return fail(c, BH_ERR_INVALID_ARG, "bh_set_gravity_method: method must be 0 or 1");
    c->use_direct = method == 1;
    c->have_acc = false;
    return BH_OK;
}

bh_status bh_euler_step(bh_ctx *c, double dt) { return euler_like(c, dt, 1, "bh_euler_step launch"); }

bh_status bh_multirate_step(bh_ctx *c, double dt_c, int n_sub)
{
    return euler_like(c, dt_c, n_sub, "bh_multirate_step launch");
}

bh_status bh_potential(bh_ctx *c, double theta, double eps, double G, double *phi_dev)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_potential")) return ds;
    if (!c->built) return fail(c, BH_ERR_STATE, "bh_potential before bh_build");
    if (!phi_dev) return fail(c, BH_ERR_INVALID_ARG, "bh_potential: null pointer");
    if (!(theta >= 0.0) || !(eps >= 0.0)) return fail(c, BH_ERR_INVALID_ARG, "bh_potential: theta or eps negative");
    return do_accel(c, theta, eps, G, phi_dev, 1);
}

bh_status bh_accel_potential(bh_ctx *c, double theta, double eps, double G, double *acc_dev, double *phi_dev)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_accel_potential")) return ds;
    if (!c->built) return fail(c, BH_ERR_STATE, "bh_accel_potential before bh_build");
    if (!acc_dev || !phi_dev) return fail(c, BH_ERR_INVALID_ARG, "bh_accel_potential: null pointer");
    if (!(theta >= 0.0) || !(eps >= 0.0)) return fail(c, BH_ERR_INVALID_ARG, "bh_accel_potential: theta or eps negative");
    return do_accel(c, theta, eps, G, acc_dev, 2, phi_dev);
}

bh_status bh_direct_potential(bh_ctx *c, double eps, double G, double *phi_dev)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_direct_potential")) return ds;
    if (!c->built) return fail(c, BH_ERR_STATE, "bh_direct_potential before bh_build");
    if (!phi_dev) return fail(c, BH_ERR_INVALID_ARG, "bh_direct_potential: null pointer");
    if (!(eps >= 0.0)) return fail(c, BH_ERR_INVALID_ARG, "bh_direct_potential: eps negative");
    {
        Phase p(c, 7);
        c->launches += launch_direct(c->ws, c->n, nullptr, c->n, eps, G, phi_dev, true, c->stream);
    }
    return cuda_check(c, cudaGetLastError(), "bh_direct_potential launch");
}

static bh_status read_diag(bh_ctx *c, int first, int count, double *out_host)
{
    cudaError_t e = cudaMemcpyAsync(c->host_diag, c->ws.diag_out + first, count * sizeof(double),
                                    cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_check(c, e, "diagnostics readback");
    for (int k = 0; k < count; ++k) out_host[k] = c->host_diag[k];
    return BH_OK;
}

bh_status bh_diagnostics(bh_ctx *c, const double *pos_dev, const double *vel_dev, const double *mass_dev,
                         const double *phi_dev, int64_t n, double out_host[8])
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_diagnostics")) return ds;
    if (!pos_dev || !vel_dev || !mass_dev || !out_host) return fail(c, BH_ERR_INVALID_ARG, "bh_diagnostics: null pointer");
    if (n < 1) return fail(c, BH_ERR_INVALID_ARG, "bh_diagnostics: n < 1");
    launch_diagnostics(c->ws, pos_dev, vel_dev, mass_dev, phi_dev, n, c->stream);
    c->launches += 1;
    bh_status st = cuda_check(c, cudaGetLastError(), "bh_diagnostics launch");
    if (st != BH_OK) return st;
    return read_diag(c, 0, 8, out_host);
}

bh_status bh_position_error(bh_ctx *c, const double *pos_dev, const double *ref_dev, int64_t n, double *err_host)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_position_error")) return ds;
    if (!pos_dev || !ref_dev || !err_host) return fail(c, BH_ERR_INVALID_ARG, "bh_position_error: null pointer");
    if (n < 1) return fail(c, BH_ERR_INVALID_ARG, "bh_position_error: n < 1");
    launch_position_error(c->ws, pos_dev, ref_dev, n, c->stream);
    c->launches += 1;
    bh_status st = cuda_check(c, cudaGetLastError(), "bh_position_error launch");
    if (st != BH_OK) return st;
    return read_diag(c, 8, 1, err_host);
}

bh_status bh_broadphase(bh_ctx *c, const double *radius_dev, const double *vel_dev, double dt, int32_t *pairs_dev,
                        int64_t capacity, int64_t *count_host)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_broadphase")) return ds;
    if (!c->built) return fail(c, BH_ERR_STATE, "bh_broadphase before bh_build");
    if (!radius_dev || !count_host) return fail(c, BH_ERR_INVALID_ARG, "bh_broadphase: null pointer");
    if (capacity < 0 || (capacity > 0 && !pairs_dev)) return fail(c, BH_ERR_INVALID_ARG, "bh_broadphase: bad pair buffer");
    if (!(dt >= 0.0)) return fail(c, BH_ERR_INVALID_ARG, "bh_broadphase: dt negative");
    c->launches += launch_broadphase(c->ws, c->n, radius_dev, vel_dev, dt, pairs_dev, capacity, c->stream);
    bh_status st = cuda_check(c, cudaGetLastError(), "bh_broadphase launch");
    if (st != BH_OK) return st;
    if ((st = fetch_state(c)) != BH_OK) return st;
    *count_host = (int64_t)c->host_state->pair_count;
    if (capacity > 0 && *count_host > capacity) return fail(c, BH_ERR_CAPACITY, "bh_broadphase: pair buffer too small");
    return BH_OK;
}

bh_status bh_aggregates(bh_ctx *c, int64_t n, const int32_t *pairs_dev, int64_t n_pairs, const double *mass_dev,
                        int32_t *label_dev, int32_t *size_dev, double *agg_mass_dev, int64_t counts_host[2])
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_aggregates")) return ds;
    if (!label_dev || !counts_host) return fail(c, BH_ERR_INVALID_ARG, "bh_aggregates: null pointer");
    if (n < 1 || n > c->max_n) return fail(c, BH_ERR_INVALID_ARG, "bh_aggregates: n out of range");
    if (n_pairs < 0 || (n_pairs > 0 && !pairs_dev)) return fail(c, BH_ERR_INVALID_ARG, "bh_aggregates: bad pair list");
    if (agg_mass_dev && !mass_dev) return fail(c, BH_ERR_INVALID_ARG, "bh_aggregates: agg_mass without mass");
    c->launches += launch_aggregates(c->ws, n, pairs_dev, n_pairs, mass_dev, label_dev, size_dev, agg_mass_dev, c->stream);
    bh_status st = cuda_check(c, cudaGetLastError(), "bh_aggregates launch");
    if (st != BH_OK) return st;
    cudaError_t e = cudaMemcpyAsync(c->host_state, c->ws.st, sizeof(DevState), cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_check(c, e, "bh_aggregates readback");
    if (c->host_state->agg_counts[2]) return fail(c, BH_ERR_INVALID_ARG, "bh_aggregates: a pair names a body outside [0, n)");
    counts_host[0] = (int64_t)c->host_state->agg_counts[0];
    counts_host[1] = (int64_t)c->host_state->agg_counts[1];
    return BH_OK;
}

double bh_gravity_dt(double G, double rho) { return 1.0 / (2.0 * sqrt(G * rho)); }

bh_status bh_get_state_acc(bh_ctx *c, const double **acc_dev)
{
    if (!c || !acc_dev) return BH_ERR_INVALID_ARG;
    if (!c->bound || !c->have_acc) return fail(c, BH_ERR_STATE, "no accelerations yet");
    *acc_dev = c->ws.acc;
    return BH_OK;
}

bh_status bh_copy_state_acc(bh_ctx *c, double *acc_dev)
{
    if (!c || !acc_dev) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_copy_state_acc")) return ds;
    if (!c->bound || !c->acc_filled) return fail(c, BH_ERR_STATE, "no stepper evaluation yet");
    return cuda_check(c, cudaMemcpyAsync(acc_dev, c->ws.acc, (size_t)c->bound_n * 24, cudaMemcpyDeviceToDevice,
                                         c->stream), "bh_copy_state_acc");
}

// device alias of a pinned (page-locked, mapped) host buffer, or nullptr for pageable memory
static double *mapped_alias(const void *host)
{
    cudaPointerAttributes a{};
    if (cudaPointerGetAttributes(&a, host) != cudaSuccess) {
        cudaGetLastError();
        return nullptr;
    }
    return a.type == cudaMemoryTypeHost ? static_cast<double *>(a.devicePointer) : nullptr;
}

bh_status bh_eval_host(bh_ctx *c, const double *pos_host, const double *mass_host, int64_t n, double theta,
                       double eps, double G, double *acc_host)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_eval_host")) return ds;
    if (!pos_host || !mass_host || !acc_host) return fail(c, BH_ERR_INVALID_ARG, "bh_eval_host: null pointer");
    if (n < 1 || n > c->max_n) return fail(c, BH_ERR_INVALID_ARG, "bh_eval_host: n out of range");
    if (!(theta >= 0.0) || !(eps >= 0.0)) return fail(c, BH_ERR_INVALID_ARG, "bh_eval_host: theta or eps negative");
    const Workspace &w = c->ws;
    // The masses are first needed by the gather (after the sort): their copy runs on a second stream,
    // beside cube / keys / sort.  It starts after the positions have arrived (one transfer at a time gets
    // the whole link) and after the previous user of the staging buffer (stream order up to the event).
    cudaError_t e = cudaMemcpyAsync(w.stage_pos, pos_host, 3 * n * sizeof(double), cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaEventRecord(c->ev_copy[0], c->stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(c->copy_stream, c->ev_copy[0], 0);
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(w.stage_mass, mass_host, n * sizeof(double), cudaMemcpyHostToDevice, c->copy_stream);
    if (e == cudaSuccess) e = cudaEventRecord(c->ev_copy[1], c->copy_stream);
    if (e != cudaSuccess) return cuda_check(c, e, "bh_eval_host H2D");
    bh_status st;
    if ((st = do_build(c, w.stage_pos, w.stage_mass, n, c->ev_copy[1])) != BH_OK) return st;
    // Pinned output (cudaHostAlloc / cudaHostRegister, e.g. a torch pin_memory() tensor): the walk stores the
    // accelerations straight into it, 24 bytes per body in one or two write segments, while it computes, and
    // no copy follows.  Pageable output: staged in the workspace and copied.
    double *direct_out = mapped_alias(acc_host);
    if ((st = do_accel(c, theta, eps, G, direct_out ? direct_out : w.acc)) != BH_OK) return st;
    c->have_acc = false;   // the internal acc buffer no longer belongs to the bound state
    c->acc_filled = false;
    if (!direct_out) {
        e = cudaMemcpyAsync(acc_host, w.acc, 3 * n * sizeof(double), cudaMemcpyDeviceToHost, c->stream);
        if (e != cudaSuccess) return cuda_check(c, e, "bh_eval_host D2H");
    }
    return fetch_state(c);
}

bh_status bh_synchronize(bh_ctx *c)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_synchronize")) return ds;
    return fetch_state(c);
}

bh_status bh_get_cube(bh_ctx *c, double lo_host[3], double *side_host)
{
    if (!c || !lo_host || !side_host) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_get_cube")) return ds;
    if (!c->built) return fail(c, BH_ERR_STATE, "no build yet");
    bh_status st = fetch_state(c);
    if (st != BH_OK) return st;
    for (int a = 0; a < 3; ++a) lo_host[a] = c->host_state->lo[a];
    *side_host = c->host_state->side;
    return BH_OK;
}

bh_status bh_get_keys(bh_ctx *c, uint64_t *sorted_key_dev, uint32_t *perm_dev)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_get_keys")) return ds;
    if (!c->built) return fail(c, BH_ERR_STATE, "no build yet");
    cudaError_t e = cudaSuccess;
    if (sorted_key_dev)
        e = cudaMemcpyAsync(sorted_key_dev, c->ws.key[0], c->n * sizeof(uint64_t), cudaMemcpyDeviceToDevice, c->stream);
    if (e == cudaSuccess && perm_dev)
        e = cudaMemcpyAsync(perm_dev, c->ws.idx[0], c->n * sizeof(uint32_t), cudaMemcpyDeviceToDevice, c->stream);
    return cuda_check(c, e, "bh_get_keys");
}

bh_status bh_get_node_count(bh_ctx *c, int64_t *m_host, int32_t *depth_host)
{
    if (!c || !m_host) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_get_node_count")) return ds;
    if (!c->built) return fail(c, BH_ERR_STATE, "no build yet");
    bh_status st = fetch_state(c);
    if (st != BH_OK) return st;
    *m_host = c->host_state->n_nodes;
    if (depth_host) *depth_host = c->host_state->depth;
    return BH_OK;
}

bh_status bh_get_nodes(bh_ctx *c, uint8_t *level, uint32_t *begin, uint32_t *count, int32_t *first_child,
                       uint8_t *child_mask, int32_t *parent, double *mono)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_get_nodes")) return ds;
    if (!c->built) return fail(c, BH_ERR_STATE, "no build yet");
    bh_status st = fetch_state(c);
    if (st != BH_OK) return st;
    const size_t M = (size_t)c->host_state->n_nodes;
    const Workspace &w = c->ws;
    cudaStream_t s = c->stream;
    cudaError_t e = cudaSuccess;
    auto cp = [&](void *dst, const void *src, size_t bytes) {
        if (dst && e == cudaSuccess) e = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToDevice, s);
    };
    cp(level, w.nlevel, M);
    cp(begin, w.nbegin, M * 4);
    cp(count, w.ncount, M * 4);
    cp(first_child, w.nfirst, M * 4);
    cp(parent, w.nparent, M * 4);
    cp(mono, w.mono, M * 32);
    if (child_mask && e == cudaSuccess) {
        launch_unpack_mask(w, child_mask, (int64_t)M, s);
        e = cudaGetLastError();
    }
    return cuda_check(c, e, "bh_get_nodes");
}

bh_status bh_get_groups(bh_ctx *c, int64_t *ng_host, uint32_t *gstart_dev)
{
    if (!c || !ng_host) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_get_groups")) return ds;
    if (!c->built) return fail(c, BH_ERR_STATE, "no build yet");
    bh_status st = fetch_state(c);
    if (st != BH_OK) return st;
    *ng_host = c->host_state->n_groups;
    if (!gstart_dev) return BH_OK;
    return cuda_check(c, cudaMemcpyAsync(gstart_dev, c->ws.gstart, (size_t)(*ng_host + 1) * 4,
                                         cudaMemcpyDeviceToDevice, c->stream), "bh_get_groups");
}

bh_status bh_get_bodies(bh_ctx *c, double *sbody_dev, double *glo_dev, double *ghi_dev)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_get_bodies")) return ds;
    if (!c->built) return fail(c, BH_ERR_STATE, "no build yet");
    bh_status st = fetch_state(c);
    if (st != BH_OK) return st;
    const int64_t groups = c->host_state->n_groups;
    cudaError_t e = cudaSuccess;
    if (sbody_dev)
        e = cudaMemcpyAsync(sbody_dev, c->ws.sbody, c->n * 32, cudaMemcpyDeviceToDevice, c->stream);
    if (glo_dev && e == cudaSuccess)
        e = cudaMemcpy2DAsync(glo_dev, 24, c->ws.gbox, 48, 24, groups, cudaMemcpyDeviceToDevice, c->stream);
    if (ghi_dev && e == cudaSuccess)
        e = cudaMemcpy2DAsync(ghi_dev, 24, c->ws.gbox + 3, 48, 24, groups, cudaMemcpyDeviceToDevice, c->stream);
    return cuda_check(c, e, "bh_get_bodies");
}

bh_status bh_get_counts(bh_ctx *c, uint32_t *n_mono_dev, uint32_t *n_direct_dev)
{
    if (!c) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_get_counts")) return ds;
    if (!c->walked) return fail(c, BH_ERR_STATE, "no bh_accel since the last build");
    bh_status st = fetch_state(c);
    if (st != BH_OK) return st;
    const int64_t groups = c->host_state->n_groups;
    cudaError_t e = cudaSuccess;
    if (n_mono_dev)
        e = cudaMemcpyAsync(n_mono_dev, c->ws.cnt_mono, groups * 4, cudaMemcpyDeviceToDevice, c->stream);
    if (n_direct_dev && e == cudaSuccess)
        e = cudaMemcpyAsync(n_direct_dev, c->ws.cnt_direct, groups * 4, cudaMemcpyDeviceToDevice, c->stream);
    return cuda_check(c, e, "bh_get_counts");
}

bh_status bh_get_stats(bh_ctx *c, uint64_t stats_host[BH_NUM_STATS])
{
    if (!c || !stats_host) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_get_stats")) return ds;
    if (!c->walked) return fail(c, BH_ERR_STATE, "no bh_accel since the last build");
    bh_status st = fetch_state(c);
    if (st != BH_OK) return st;
    for (int k = 0; k < kNumStats; ++k) stats_host[k] = c->host_state->stats[k];
    return BH_OK;
}

bh_status bh_get_launches(bh_ctx *c, uint64_t *count_host)
{
    if (!c || !count_host) return BH_ERR_INVALID_ARG;
    *count_host = c->launches;
    return BH_OK;
}

bh_status bh_set_timing(bh_ctx *c, int enable)
{
    if (!c) return BH_ERR_INVALID_ARG;
    c->timing = enable != 0;
    for (int p = 0; p < BH_NUM_PHASES; ++p) c->ev_set[p] = false;
    return BH_OK;
}

bh_status bh_get_phase_ms(bh_ctx *c, float ms_host[BH_NUM_PHASES])
{
    if (!c || !ms_host) return BH_ERR_INVALID_ARG;
    if (bh_status ds = on_device(c, "bh_get_phase_ms")) return ds;
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_check(c, e, "bh_get_phase_ms");
    for (int p = 0; p < BH_NUM_PHASES; ++p) {
        ms_host[p] = 0.f;
        if (c->ev_set[p]) cudaEventElapsedTime(&ms_host[p], c->ev[p][0], c->ev[p][1]);
    }
    return BH_OK;
}

}  // extern "C"

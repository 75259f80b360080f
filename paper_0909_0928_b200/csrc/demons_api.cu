// C ABI of the demons library (include/demons.h): context, workspace partition, the multi-scale
// registration driver and the per-kernel entry points.
#include "../../include/demons.h"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "kernels.h"

using namespace demons;

namespace {

thread_local std::string g_last_error;

int fail(int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_last_error = buf;
    return code;
}

#define CUDA_TRY(expr)                                                                        \
    do {                                                                                      \
        cudaError_t e_ = (expr);                                                              \
        if (e_ != cudaSuccess)                                                                \
            return fail(DEMONS_E_CUDA, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e_), \
                        __FILE__, __LINE__);                                                  \
    } while (0)

constexpr size_t ALIGN = 256;
size_t align_up(size_t v) { return (v + ALIGN - 1) / ALIGN * ALIGN; }

// Workspace partition for `nb` pairs: every per-pair array is laid out [nb][...] so that one batched launch
// covers a group of pairs.  The pyramid images of a pair are interleaved ([nb][2][n]: S then M), so that one L2
// access-policy window covers the images of a group.
struct Partition {
    size_t control, partials, stats, Mw, Sw, uprime, ubprime, smooth_tmp;
    size_t pyrI[DEMONS_MAX_LEVELS], pyrU[DEMONS_MAX_LEVELS], pyrUb[DEMONS_MAX_LEVELS];
    size_t hI, hU, hUb;
    size_t total;
    int partial_stride;
};

struct GraphEntry {
    Dims d;
    const float *S, *M;
    float *u, *ub;
    int chunk, nb, one_field;
    int timed;         // "profile" = 2: one iteration of the chunk carries event-record nodes
    int b0, nb_total;  // the captured kernels carry workspace offsets that move with the pair index and the batch size
    double eps;
    cudaGraphExec_t exec;
    int launches;
};

}  // namespace

namespace demons {
void set_last_error(const char* msg) { g_last_error = msg ? msg : ""; }
}  // namespace demons

struct demons_ctx {
    Dims dims;
    float spacing[3];
    int variant;
    float alpha;
    float sigma;
    char* ws = nullptr;
    size_t ws_bytes = 0;
    long long launches = 0;
    int opt_graphs = 1;
    int opt_texture = 0;
    int opt_generic_smooth = 0;
    int opt_profile = 0;
    int opt_l2_persist = 1;
    int opt_zero_start = 0;
    int opt_ic_one_field = 1;
    size_t l2_granted = 0;
    bool l2_limit_raised = false;
    size_t l2_prev_limit = 0;
    std::vector<cudaEvent_t> prof_all;                               // events of the profiled call
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> prof_pairs[4];  // per kernel class: start/stop
    cudaEvent_t tg[4] = {nullptr, nullptr, nullptr, nullptr};  // "profile" = 2: before force / between / after the smoother / once more, recorded by graph nodes
    double prof_ms[4] = {0, 0, 0, 0};
    long long prof_n[4] = {0, 0, 0, 0};
    std::vector<GraphEntry> graphs;
    // side branch of an iteration: the metric finalisation runs beside the smoothing kernel (fork / join by events)
    cudaStream_t side = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    // demons_register_host_queue: copy-in and copy-out streams, per staging slot the events "images uploaded",
    // "registration done" and "field downloaded"
    cudaStream_t q_in = nullptr, q_out = nullptr;
    cudaEvent_t q_up[2] = {nullptr, nullptr}, q_done[2] = {nullptr, nullptr}, q_down[2] = {nullptr, nullptr};
    cudaArray_t tex_array = nullptr;
    cudaTextureObject_t tex = 0;
    Dims tex_dims{0, 0, 0};
};

namespace {

Dims coarser(const Dims& d) { return Dims{(d.nx + 1) / 2, (d.ny + 1) / 2, (d.nz + 1) / 2}; }

bool is_ic(const demons_ctx* c) { return c->variant == DEMONS_INVERSE_CONSISTENT; }

// Gaussian taps (reading A9): R = ceil(3 sigma), w_k = exp(-k^2/2 sigma^2) / sum_j exp(-j^2/2 sigma^2),
// evaluated in double and rounded to float.
int gaussian_taps(double sigma, float* w) {
    const int R = (int)std::ceil(3.0 * sigma);
    if (R < 0 || R > DEMONS_MAX_RADIUS) return -1;
    double e[DEMONS_MAX_RADIUS + 1];
    double total = 0.0;
    for (int k = 0; k <= R; ++k) {
        e[k] = std::exp(-0.5 * (double)k * (double)k / (sigma * sigma));
        total += k == 0 ? e[k] : 2.0 * e[k];
    }
    for (int k = 0; k <= R; ++k) w[k] = (float)(e[k] / total);
    return R;
}

Partition make_partition(const demons_ctx* c, int levels, int nb) {
    Partition p{};
    const size_t N = nvox(c->dims);
    const bool ic = is_ic(c);
    size_t off = 0;
    auto take = [&](size_t bytes) {
        const size_t o = off;
        off += align_up(bytes);
        return o;
    };
    p.control = take((size_t)nb * sizeof(Control));
    int stride = force_partial_blocks(c->dims);
    if (stride < 148 * 8) stride = 148 * 8;
    p.partial_stride = stride;
    p.partials = take((size_t)nb * 5 * stride * sizeof(double));  // 3 metrics per force block; 5 sums per block of demons_cc
    p.stats = take((size_t)nb * DEMONS_MAX_STATS_ROWS * 3 * sizeof(double));
    p.Mw = take(nb * N * 4);
    p.Sw = ic ? take(nb * N * 4) : 0;
    p.uprime = take(nb * 3 * N * 4);
    p.ubprime = ic ? take(nb * 3 * N * 4) : 0;
    p.smooth_tmp = take(nb * N * 4);
    Dims d = c->dims;
    for (int l = 1; l < levels; ++l) {
        d = coarser(d);
        const size_t n = nvox(d);
        p.pyrI[l] = take(nb * 2 * n * 4);
        p.pyrU[l] = take(nb * 3 * n * 4);
        p.pyrUb[l] = ic ? take(nb * 3 * n * 4) : 0;
    }
    if (nb == 1) {  // staging of demons_register_host (single registrations only)
        p.hI = take(2 * N * 4);
        p.hU = take(3 * N * 4);
        p.hUb = ic ? take(3 * N * 4) : 0;
    }
    p.total = off;
    return p;
}

bool dims_ok(const int dims[3]) {
    if (!dims) return false;
    for (int c = 0; c < 3; ++c)
        if (dims[c] < 1 || dims[c] > 16384) return false;
    const double n = (double)dims[0] * dims[1] * dims[2];
    return n < 2147483647.0 / 4.0;
}

int check_ws(const demons_ctx* c, int levels, int nb = 1) {
    if (!c->ws) return fail(DEMONS_E_WORKSPACE, "no workspace set (demons_set_workspace)");
    const Partition p = make_partition(c, levels, nb);
    if (p.total > c->ws_bytes)
        return fail(DEMONS_E_WORKSPACE, "workspace too small: have %zu bytes, need %zu for %d level(s), batch of %d",
                    c->ws_bytes, p.total, levels, nb);
    return DEMONS_OK;
}

int check_call_dims(const demons_ctx* c, const int dims[3], Dims* out) {
    if (!dims_ok(dims)) return fail(DEMONS_E_ARG, "bad dims");
    const Dims d{dims[0], dims[1], dims[2]};
    if (nvox(d) > nvox(c->dims))
        return fail(DEMONS_E_WORKSPACE, "volume %dx%dx%d exceeds the context's %dx%dx%d", d.nx, d.ny, d.nz,
                    c->dims.nx, c->dims.ny, c->dims.nz);
    *out = d;
    return DEMONS_OK;
}

// L2 residency for the gathered images (option "l2_persist", default on): the kernels that gather launch with an
// access-policy window over the images of their group of pairs (hitProp = persisting).  The window is one
// address range: [S_0, M_last] when the images of the group form one block (the workspace's pyramid levels do,
// and so does a caller's pair whose moving image directly follows its static image), else the moving image of
// a single pair.  The device's persisting-L2 set-aside (cudaLimitPersistingL2CacheSize) is RAISED to the size of
// the window (never lowered here; demons_destroy restores it); windows larger than the device's maximum
// set-aside are not requested at all: pinning a part of the images takes L2 away from everything else (the
// smoothing halos, the stencils) and was 2x slower at 512x512x160.
struct L2Window {
    const void* ptr = nullptr;
    size_t bytes = 0;
    float ratio = 0.f;
};

bool images_form_block(const float* S, const float* M, size_t n, size_t img_stride, int nb) {
    if (S == nullptr || M <= S) return false;
    const size_t gap = (size_t)(M - S);
    if (nb == 1) return gap <= n + 1024;            // M right behind S (at most one alignment gap)
    return gap == n && img_stride == 2 * n;         // [nb][2][n]
}

L2Window l2_window(demons_ctx* c, const Dims& d, const float* S, const float* M, size_t img_stride, int nb) {
    L2Window w;
    if (!c->opt_l2_persist) return w;
    const size_t max_persist = max_persisting_l2(), max_window = max_policy_window();
    if (max_persist == 0 || max_window == 0) return w;
    const size_t n = nvox(d);
    const char* lo;
    size_t span;
    if (images_form_block(S, M, n, img_stride, nb)) {
        lo = reinterpret_cast<const char*>(S);
        span = (size_t)(reinterpret_cast<const char*>(M + (size_t)(nb - 1) * img_stride + n) - lo);
    } else if (nb == 1) {
        lo = reinterpret_cast<const char*>(M);
        span = n * sizeof(float);
    } else {
        return w;
    }
    const size_t want = (span + ((size_t)1 << 20) - 1) & ~(((size_t)1 << 20) - 1);
    if (want > max_persist || span > max_window) {
        // both images of a pair do not fit: retry with the gathered (moving) image alone
        if (nb == 1 && lo != reinterpret_cast<const char*>(M)) return l2_window(c, d, nullptr, M, img_stride, 1);
        return w;
    }
    size_t cur = 0;
    if (cudaDeviceGetLimit(&cur, cudaLimitPersistingL2CacheSize) != cudaSuccess) {
        cudaGetLastError();
        return w;
    }
    if (cur < want) {
        if (cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, want) != cudaSuccess) {
            cudaGetLastError();
            return w;
        }
        if (!c->l2_limit_raised) {  // remember what to restore in demons_destroy
            c->l2_limit_raised = true;
            c->l2_prev_limit = cur;
        }
    }
    c->l2_granted = want;
    w.ptr = lo;
    w.bytes = span;
    w.ratio = 1.f;
    return w;
}

MetricSink make_sink(const demons_ctx* c, const Partition& p, int b0, double* out, size_t out_stride, bool driver,
                     double eps) {
    MetricSink s{};
    s.ctl = reinterpret_cast<Control*>(c->ws + p.control) + b0;
    s.partials = reinterpret_cast<double*>(c->ws + p.partials) + (size_t)b0 * 5 * p.partial_stride;
    s.out = out;
    s.out_stride = out_stride;
    s.stride = p.partial_stride;
    s.driver = driver ? 1 : 0;
    s.eps = eps;
    return s;
}

void release_texture(demons_ctx* c) {
    if (c->tex) cudaDestroyTextureObject(c->tex);
    if (c->tex_array) cudaFreeArray(c->tex_array);
    c->tex = 0;
    c->tex_array = nullptr;
}

// S9 (measured option): copy M into a 3D CUDA array and bind it with hardware linear filtering,
// clamp addressing ("map the original static images and moving images on the texture
// memory").  The array is the one device allocation the library makes itself (a cudaArray cannot be
// a torch tensor); it lives in the context.
int bind_texture(demons_ctx* c, const Dims& d, const float* M, cudaStream_t st) {
    if (!c->tex_array || c->tex_dims.nx != d.nx || c->tex_dims.ny != d.ny || c->tex_dims.nz != d.nz) {
        release_texture(c);
        cudaChannelFormatDesc fmt = cudaCreateChannelDesc<float>();
        CUDA_TRY(cudaMalloc3DArray(&c->tex_array, &fmt, make_cudaExtent(d.nx, d.ny, d.nz)));
        cudaResourceDesc rd{};
        rd.resType = cudaResourceTypeArray;
        rd.res.array.array = c->tex_array;
        cudaTextureDesc td{};
        td.addressMode[0] = td.addressMode[1] = td.addressMode[2] = cudaAddressModeClamp;
        td.filterMode = cudaFilterModeLinear;
        td.readMode = cudaReadModeElementType;
        td.normalizedCoords = 0;
        CUDA_TRY(cudaCreateTextureObject(&c->tex, &rd, &td, nullptr));
        c->tex_dims = d;
    }
    cudaMemcpy3DParms cp{};
    cp.srcPtr = make_cudaPitchedPtr(const_cast<float*>(M), (size_t)d.nx * 4, d.nx, d.ny);
    cp.dstArray = c->tex_array;
    cp.extent = make_cudaExtent(d.nx, d.ny, d.nz);
    cp.kind = cudaMemcpyDeviceToDevice;
    CUDA_TRY(cudaMemcpy3DAsync(&cp, st));
    return DEMONS_OK;
}

enum { PROF_FORCE = 0, PROF_WARP = 1, PROF_SMOOTH = 2, PROF_PYRAMID = 3 };

// "profile" option: bracket every launch of a kernel class with a pair of events on the stream.
cudaEvent_t prof_event(demons_ctx* c, cudaStream_t st, bool record) {
    if (c->opt_profile != 1) return nullptr;
    cudaEvent_t e = nullptr;
    if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
    if (record) cudaEventRecord(e, st);
    c->prof_all.push_back(e);
    return e;
}

void prof_pair(demons_ctx* c, int cls, cudaEvent_t a, cudaEvent_t b) {
    if (a && b) c->prof_pairs[cls].push_back({a, b});
}

void prof_clear(demons_ctx* c) {
    for (cudaEvent_t e : c->prof_all) cudaEventDestroy(e);
    c->prof_all.clear();
    for (int k = 0; k < 4; ++k) c->prof_pairs[k].clear();
}

void prof_collect(demons_ctx* c) {  // after a stream synchronise
    for (int k = 0; k < 4; ++k) {
        double ms = 0.0;
        for (auto& pr : c->prof_pairs[k]) {
            float t = 0.f;
            if (cudaEventElapsedTime(&t, pr.first, pr.second) == cudaSuccess) ms += t;
        }
        c->prof_ms[k] = ms;
        c->prof_n[k] = (long long)c->prof_pairs[k].size();
    }
    prof_clear(c);
}

struct LevelBuffers {
    Dims d;
    const float* S;     // pair 0 of the group
    const float* M;
    size_t img_stride;  // floats between the images of consecutive pairs
    float* u;           // [nb][3][n]
    float* ub;          // variant 5, two-field form; nullptr otherwise
    int b0, nb;         // first pair and number of pairs of the group
    int nb_total;       // pairs of the whole call (the workspace partition is laid out for this many)
    int one_field;
};

// The side stream of the metric finalisation and its fork / join events; created outside any stream capture.
int ensure_side(demons_ctx* c) {
    if (c->side) return DEMONS_OK;
    CUDA_TRY(cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking));
    CUDA_TRY(cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming));
    CUDA_TRY(cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming));
    return DEMONS_OK;
}

// One iteration of a group of pairs: [warp_force ; smooth the total field] (reading C2).
int enqueue_iteration(demons_ctx* c, const Partition& p, const LevelBuffers& lb, const L2Window& win, double eps,
                      cudaStream_t st, int* launches, bool timed = false) {
    const bool ic = is_ic(c);
    const bool two = ic && !lb.one_field;
    const size_t N = nvox(c->dims);
    ForceArgs fa{};
    fa.d = lb.d;
    fa.variant = c->variant;
    fa.alpha2 = c->variant == DEMONS_ADJUSTED_DOUBLE ? c->alpha * c->alpha : 1.f;
    fa.nb = lb.nb;
    fa.img_stride = lb.img_stride;
    fa.S = lb.S;
    fa.M = lb.M;
    fa.u_in = lb.u;
    // per-pair scratch is laid out for the level's own size, [nb][..n], starting at pair b0's share of the buffer
    fa.u_out = reinterpret_cast<float*>(c->ws + p.uprime) + (size_t)lb.b0 * 3 * N;
    fa.ub_in = two ? lb.ub : nullptr;
    fa.ub_out = two ? reinterpret_cast<float*>(c->ws + p.ubprime) + (size_t)lb.b0 * 3 * N : nullptr;
    fa.one_field = lb.one_field;
    fa.Mw = reinterpret_cast<float*>(c->ws + p.Mw) + (size_t)lb.b0 * N;
    fa.Sw = ic ? reinterpret_cast<float*>(c->ws + p.Sw) + (size_t)lb.b0 * N : nullptr;
    fa.sink = make_sink(c, p, lb.b0, reinterpret_cast<double*>(c->ws + p.stats) + (size_t)lb.b0 * DEMONS_MAX_STATS_ROWS * 3,
                        (size_t)DEMONS_MAX_STATS_ROWS * 3, true, eps);
    fa.sink.defer = 1;  // the force blocks store partials; k_metrics_final (below) sums and publishes them
    fa.texM = c->opt_texture ? c->tex : 0;
    fa.l2_ptr = win.ptr;
    fa.l2_bytes = win.bytes;
    fa.l2_ratio = win.ratio;
    // timed (inside a stream capture only): event-record NODES around the kernels of this iteration, so that the
    // replayed graph itself says how long they take with the caches and clocks of the run
    if (timed) CUDA_TRY(cudaEventRecordWithFlags(c->tg[0], st, cudaEventRecordExternal));
    cudaEvent_t e0 = prof_event(c, st, true);
    fa.ev_mid = c->variant >= DEMONS_ACTIVE ? prof_event(c, st, false) : nullptr;
    int metric_blocks = 0;
    fa.metric_blocks = &metric_blocks;
    int k = launch_warp_force(fa, st);
    if (k < 0) return fail(DEMONS_E_CUDA, "warp_force launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    *launches += k;
    if (timed) CUDA_TRY(cudaEventRecordWithFlags(c->tg[1], st, cudaEventRecordExternal));
    cudaEvent_t e1 = prof_event(c, st, true);
    if (fa.ev_mid) {
        prof_pair(c, PROF_WARP, e0, fa.ev_mid);
        prof_pair(c, PROF_FORCE, fa.ev_mid, e1);
    } else {
        prof_pair(c, PROF_FORCE, e0, e1);
    }
    // fork: statistics row and stopping rule of this iteration, beside the smoothing kernel (which reads neither)
    CUDA_TRY(cudaEventRecord(c->ev_fork, st));
    CUDA_TRY(cudaStreamWaitEvent(c->side, c->ev_fork, 0));
    fa.sink.nblocks = (unsigned)metric_blocks;
    if (launch_metrics_final(fa.sink, lb.nb, c->side) < 0)
        return fail(DEMONS_E_CUDA, "metrics launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    *launches += 1;
    CUDA_TRY(cudaEventRecord(c->ev_join, c->side));
    SmoothArgs sa{};
    sa.d = lb.d;
    sa.tmp = reinterpret_cast<float*>(c->ws + p.smooth_tmp) + (size_t)lb.b0 * N;
    sa.ncomp = 3 * lb.nb;
    sa.comps_per_pair = 3;
    sa.R = gaussian_taps(c->sigma, sa.w);
    // the smoothing kernels test the pair's stop flag only when the rule can fire
    sa.ctl = eps > 0.0 ? reinterpret_cast<Control*>(c->ws + p.control) + lb.b0 : nullptr;
    sa.force_generic = c->opt_generic_smooth;
    sa.in = fa.u_out;
    sa.out = lb.u;
    k = launch_smooth(sa, st);
    if (k < 0) return fail(DEMONS_E_CUDA, "smooth launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    *launches += k;
    if (two) {
        sa.in = fa.ub_out;
        sa.out = lb.ub;
        k = launch_smooth(sa, st);
        if (k < 0) return fail(DEMONS_E_CUDA, "smooth launch failed: %s", cudaGetErrorString(cudaGetLastError()));
        *launches += k;
    }
    if (timed) {
        CUDA_TRY(cudaEventRecordWithFlags(c->tg[2], st, cudaEventRecordExternal));  // end of the smoothing kernel(s)
        CUDA_TRY(cudaEventRecordWithFlags(c->tg[3], st, cudaEventRecordExternal));  // empty bracket: what a record node costs
    }
    CUDA_TRY(cudaStreamWaitEvent(st, c->ev_join, 0));  // join: the next force kernel reads the stop flag
    prof_pair(c, PROF_SMOOTH, e1, prof_event(c, st, true));
    return DEMONS_OK;
}

bool capturable(cudaStream_t st) { return st != nullptr && st != cudaStreamLegacy; }

constexpr size_t GRAPH_CACHE = 192;

int run_level(demons_ctx* c, const Partition& p, const LevelBuffers& lb, int iters, double eps, cudaStream_t st) {
    int done = 0;
    const size_t N = nvox(c->dims);
    const L2Window win = l2_window(c, lb.d, lb.S, lb.M, lb.img_stride, lb.nb);  // outside any stream capture
    if (c->variant == DEMONS_EVOLVED_PASSIVE && iters > 0) {  // |grad M0|^2 of this level, fixed for the level
        if (launch_grad_mag2(lb.d, lb.M, lb.img_stride, reinterpret_cast<float*>(c->ws + p.Mw) + (size_t)lb.b0 * N, lb.nb, st) < 0)
            return fail(DEMONS_E_CUDA, "gradient launch failed: %s", cudaGetErrorString(cudaGetLastError()));
        c->launches += 1;
    }
    const int chunk = iters >= 20 ? 20 : iters;
    if (c->opt_graphs && capturable(st) && iters >= 4 && !c->opt_texture && c->opt_profile != 1) {
        const int timed = c->opt_profile == 2 ? 1 : 0;
        GraphEntry* ge = nullptr;
        for (auto& g : c->graphs)
            if (g.d.nx == lb.d.nx && g.d.ny == lb.d.ny && g.d.nz == lb.d.nz && g.S == lb.S && g.M == lb.M &&
                g.u == lb.u && g.ub == lb.ub && g.chunk == chunk && g.eps == eps && g.nb == lb.nb &&
                g.one_field == lb.one_field && g.b0 == lb.b0 && g.nb_total == lb.nb_total && g.timed == timed)
                ge = &g;
        if (!ge) {
            GraphEntry g{};
            g.d = lb.d;
            g.S = lb.S;
            g.M = lb.M;
            g.u = lb.u;
            g.ub = lb.ub;
            g.chunk = chunk;
            g.eps = eps;
            g.nb = lb.nb;
            g.one_field = lb.one_field;
            g.b0 = lb.b0;
            g.nb_total = lb.nb_total;
            g.timed = timed;
            cudaGraph_t graph = nullptr;
            CUDA_TRY(cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal));
            int rc = DEMONS_OK;
            // the timed iteration sits in the middle of the chunk, with replayed work on both sides of it
            for (int i = 0; i < chunk && rc == DEMONS_OK; ++i)
                rc = enqueue_iteration(c, p, lb, win, eps, st, &g.launches, timed && i == chunk / 2);
            cudaError_t e = cudaStreamEndCapture(st, &graph);
            if (rc != DEMONS_OK) {
                if (graph) cudaGraphDestroy(graph);
                return rc;
            }
            if (e != cudaSuccess) return fail(DEMONS_E_CUDA, "graph capture failed: %s", cudaGetErrorString(e));
            e = cudaGraphInstantiate(&g.exec, graph, 0);
            cudaGraphDestroy(graph);
            if (e != cudaSuccess) return fail(DEMONS_E_CUDA, "graph instantiate failed: %s", cudaGetErrorString(e));
            if (c->graphs.size() >= GRAPH_CACHE) {  // bounded cache
                cudaGraphExecDestroy(c->graphs.front().exec);
                c->graphs.erase(c->graphs.begin());
            }
            c->graphs.push_back(g);
            ge = &c->graphs.back();
        }
        while (iters - done >= chunk) {
            CUDA_TRY(cudaGraphLaunch(ge->exec, st));
            c->launches += ge->launches;
            done += chunk;
            if (timed) {  // read the three events of this replay before the next one records them again
                CUDA_TRY(cudaStreamSynchronize(st));
                float t_force = 0.f, t_smooth = 0.f, t_empty = 0.f;
                CUDA_TRY(cudaEventElapsedTime(&t_force, c->tg[0], c->tg[1]));
                CUDA_TRY(cudaEventElapsedTime(&t_smooth, c->tg[1], c->tg[2]));
                CUDA_TRY(cudaEventElapsedTime(&t_empty, c->tg[2], c->tg[3]));
                c->prof_ms[PROF_FORCE] += t_force;
                c->prof_ms[PROF_SMOOTH] += t_smooth;
                c->prof_ms[PROF_WARP] += t_empty;  // slot [1] carries the empty bracket in this mode
                c->prof_n[PROF_FORCE] += 1;
                c->prof_n[PROF_SMOOTH] += 1;
                c->prof_n[PROF_WARP] += 1;
            }
        }
    }
    for (; done < iters; ++done) {
        int k = 0;
        const int rc = enqueue_iteration(c, p, lb, win, eps, st, &k);
        if (rc != DEMONS_OK) return rc;
        c->launches += k;
    }
    return DEMONS_OK;
}

// Pairs per launch on a level of n voxels: enough voxels per launch to fill the GPU (a 256x256x100 level
// does; a 64x64x25 level needs the whole batch), never more than the batch.  Large levels run pair by pair:
// their launches already fill the machine and the images of ONE pair stay resident in L2.
int group_size(size_t n, int nb, int nz = 1) {
    const size_t target = (size_t)3 << 20;  // voxels per launch
    size_t g = (target + n - 1) / n;
    // the separable smoothing fallback and the scalar |grad M|^2 kernel carry (planes x components x pairs) in
    // gridDim.z (<= 65535): a thin, tall level that misses the fast paths must not fail as a batch where every pair
    // alone succeeds
    const size_t zcap = (size_t)65535 / ((size_t)3 * (size_t)(nz < 1 ? 1 : nz));
    if (g > zcap) g = zcap;
    if (g < 1) g = 1;
    if (g > (size_t)nb) g = nb;
    return (int)g;
}

// The multi-scale driver (O9) for a batch of nb independent pairs: images [nb][N], fields [nb][3][N].
int register_impl(demons_ctx* c, const float* dS, const float* dM, float* du, float* dub, int nb, int levels,
                  const int* iters, double eps, double* h_stats, int* h_done, cudaStream_t st) {
    const bool ic = is_ic(c);
    const Partition p = make_partition(c, levels, nb);
    const size_t N = nvox(c->dims);
    Control* ctl = reinterpret_cast<Control*>(c->ws + p.control);
    long long total_iters = 0;
    for (int l = 0; l < levels; ++l) total_iters += iters[l];
    const bool zero_start = levels > 1 || c->opt_zero_start;
    // variant 5 from a zero start: u_b = -u_f exactly at every iteration and level (pin P10), so only u_f is
    // iterated on and u_b is written once on exit; bit-identical to iterating on both fields
    const int one_field = ic && zero_start && c->opt_ic_one_field ? 1 : 0;
    prof_clear(c);
    if (c->opt_profile == 2) {
        for (int k = 0; k < 4; ++k) c->prof_ms[k] = 0.0, c->prof_n[k] = 0;
        for (int k = 0; k < 4; ++k)
            if (!c->tg[k]) CUDA_TRY(cudaEventCreate(&c->tg[k]));
    }
    if (const int rs = ensure_side(c); rs != DEMONS_OK) return rs;
    CUDA_TRY(cudaMemsetAsync(ctl, 0, (size_t)nb * sizeof(Control), st));
    if (total_iters > 0)
        CUDA_TRY(cudaMemsetAsync(c->ws + p.stats, 0,
                                 ((size_t)(nb - 1) * DEMONS_MAX_STATS_ROWS + (size_t)total_iters) * 24, st));

    // pyramids (O6): images only, no pre-blur (reading A15)
    struct Level {
        Dims d;
        const float *S, *M;
        size_t img_stride;
        float *u, *ub;
    } lv[DEMONS_MAX_LEVELS];
    lv[0] = Level{c->dims, dS, dM, N, du, dub};  // the caller's layout: static [nb][N], moving [nb][N]
    for (int l = 1; l < levels; ++l) {
        lv[l].d = coarser(lv[l - 1].d);
        const size_t n = nvox(lv[l].d);
        float* base = reinterpret_cast<float*>(c->ws + p.pyrI[l]);
        lv[l].S = base;
        lv[l].M = base + n;
        lv[l].img_stride = 2 * n;
        lv[l].u = reinterpret_cast<float*>(c->ws + p.pyrU[l]);
        lv[l].ub = ic ? reinterpret_cast<float*>(c->ws + p.pyrUb[l]) : nullptr;
        cudaEvent_t e0 = prof_event(c, st, true);
        if (launch_restrict(lv[l - 1].d, lv[l - 1].S, lv[l - 1].img_stride, base, 2 * n, nb, st) < 0 ||
            launch_restrict(lv[l - 1].d, lv[l - 1].M, lv[l - 1].img_stride, base + n, 2 * n, nb, st) < 0)
            return fail(DEMONS_E_CUDA, "restrict launch failed: %s", cudaGetErrorString(cudaGetLastError()));
        c->launches += 2;
        prof_pair(c, PROF_PYRAMID, e0, prof_event(c, st, true));
    }
    if (zero_start) {  // the coarsest level starts from zero (O9); "zero_start": a single level too
        const size_t n = nvox(lv[levels - 1].d);
        CUDA_TRY(cudaMemsetAsync(lv[levels - 1].u, 0, (size_t)nb * 3 * n * 4, st));
        if (ic && !one_field) CUDA_TRY(cudaMemsetAsync(lv[levels - 1].ub, 0, (size_t)nb * 3 * n * 4, st));
    }
    for (int step = 0; step < levels; ++step) {
        const int l = levels - 1 - step;  // coarse -> fine
        const size_t n = nvox(lv[l].d);
        const int G = group_size(n, nb, lv[l].d.nz);
        if (step > 0)  // level_iter, stop_force, stop_smooth of every pair
            CUDA_TRY(cudaMemset2DAsync(&ctl[0].level_iter, sizeof(Control), 0, 12, nb, st));
        for (int b0 = 0; b0 < nb; b0 += G) {
            const int g = nb - b0 < G ? nb - b0 : G;
            LevelBuffers lb{};
            lb.d = lv[l].d;
            lb.S = lv[l].S + (size_t)b0 * lv[l].img_stride;
            lb.M = lv[l].M + (size_t)b0 * lv[l].img_stride;
            lb.img_stride = lv[l].img_stride;
            lb.u = lv[l].u + (size_t)b0 * 3 * n;
            lb.ub = ic && !one_field ? lv[l].ub + (size_t)b0 * 3 * n : nullptr;
            lb.b0 = b0;
            lb.nb_total = nb;
            lb.nb = g;
            lb.one_field = one_field;
            if (c->opt_texture) {
                const int rc = bind_texture(c, lb.d, lb.M, st);
                if (rc != DEMONS_OK) return rc;
            }
            const int rc = run_level(c, p, lb, iters[step], eps, st);
            if (rc != DEMONS_OK) return rc;
            if (l > 0) {  // O7
                const size_t nf = nvox(lv[l - 1].d);
                cudaEvent_t e0 = prof_event(c, st, true);
                if (launch_prolong(lb.d, lb.u, lv[l - 1].d, lv[l - 1].u + (size_t)b0 * 3 * nf, g, st) < 0)
                    return fail(DEMONS_E_CUDA, "prolong launch failed: %s", cudaGetErrorString(cudaGetLastError()));
                c->launches += 1;
                if (ic && !one_field) {
                    if (launch_prolong(lb.d, lb.ub, lv[l - 1].d, lv[l - 1].ub + (size_t)b0 * 3 * nf, g, st) < 0)
                        return fail(DEMONS_E_CUDA, "prolong launch failed: %s", cudaGetErrorString(cudaGetLastError()));
                    c->launches += 1;
                }
                prof_pair(c, PROF_PYRAMID, e0, prof_event(c, st, true));
            }
        }
        CUDA_TRY(cudaMemcpy2DAsync(&ctl[0].iters_done[step], sizeof(Control), &ctl[0].level_iter, sizeof(Control), 4, nb,
                                   cudaMemcpyDeviceToDevice, st));
    }
    if (one_field) {  // u_b = -u_f (P10), written once
        if (launch_negate(du, dub, (size_t)nb * 3 * N, st) < 0)
            return fail(DEMONS_E_CUDA, "negate launch failed: %s", cudaGetErrorString(cudaGetLastError()));
        c->launches += 1;
    }
    if (h_stats && total_iters > 0)
        CUDA_TRY(cudaMemcpy2DAsync(h_stats, (size_t)total_iters * 24, c->ws + p.stats, (size_t)DEMONS_MAX_STATS_ROWS * 24,
                                   (size_t)total_iters * 24, nb, cudaMemcpyDeviceToHost, st));
    if (h_done)
        CUDA_TRY(cudaMemcpy2DAsync(h_done, (size_t)levels * 4, ctl[0].iters_done, sizeof(Control), (size_t)levels * 4, nb,
                                   cudaMemcpyDeviceToHost, st));
    if (h_stats || h_done || c->opt_profile) CUDA_TRY(cudaStreamSynchronize(st));
    if (c->opt_profile == 1) prof_collect(c);
    return DEMONS_OK;
}

int check_register_args(demons_ctx* c, const void* S, const void* M, const void* u, const void* ub, int nb, int levels,
                        const int* iters) {
    if (!c) return fail(DEMONS_E_ARG, "ctx is NULL");
    if (!S || !M || !u) return fail(DEMONS_E_ARG, "static, moving and u must be non-NULL");
    if (is_ic(c) && !ub) return fail(DEMONS_E_ARG, "variant 5 needs u_back");
    if (!is_ic(c) && ub) return fail(DEMONS_E_ARG, "u_back must be NULL unless variant 5");
    if (nb < 1 || nb > DEMONS_MAX_BATCH) return fail(DEMONS_E_ARG, "batch size out of range");
    if (levels < 1 || levels > DEMONS_MAX_LEVELS) return fail(DEMONS_E_ARG, "levels out of range");
    if (!iters) return fail(DEMONS_E_ARG, "iters_per_level is NULL");
    long long total = 0;
    for (int l = 0; l < levels; ++l) {
        if (iters[l] < 0) return fail(DEMONS_E_ARG, "negative iteration count");
        total += iters[l];
    }
    if (total > DEMONS_MAX_STATS_ROWS) return fail(DEMONS_E_ARG, "more than DEMONS_MAX_STATS_ROWS iterations");
    if (nb > 1 && c->opt_texture) return fail(DEMONS_E_UNSUPPORTED, "the texture option serves single registrations only");
    if (nb > 1 && (double)nb * (double)nvox(c->dims) >= 2147483647.0 / 4.0 && group_size(nvox(c->dims), nb, c->dims.nz) > 1)
        return fail(DEMONS_E_UNSUPPORTED, "batch too large for 32-bit indexing");
    return check_ws(c, levels, nb);
}

}  // namespace

extern "C" {

const char* demons_last_error(void) { return g_last_error.c_str(); }

int demons_create(demons_ctx** out, const int dims[3], const float spacing[3], int variant, float alpha,
                  float sigma) {
    if (!out) return fail(DEMONS_E_ARG, "out is NULL");
    *out = nullptr;
    if (!dims_ok(dims)) return fail(DEMONS_E_ARG, "dims must be in [1,16384] with fewer than 2^29 voxels");
    if (!spacing || !(spacing[0] > 0.f) || !(spacing[1] > 0.f) || !(spacing[2] > 0.f))
        return fail(DEMONS_E_ARG, "spacing must be positive");
    if (variant < 0 || variant > 5) return fail(DEMONS_E_ARG, "variant must be 0..5");
    if (!(alpha > 0.f) || !std::isfinite(alpha)) return fail(DEMONS_E_ARG, "alpha must be positive");
    if (!(sigma > 0.f) || !std::isfinite(sigma)) return fail(DEMONS_E_ARG, "sigma must be positive");
    float w[DEMONS_MAX_RADIUS + 1];
    if (gaussian_taps(sigma, w) < 0)
        return fail(DEMONS_E_UNSUPPORTED, "ceil(3 sigma) exceeds DEMONS_MAX_RADIUS (%d)", DEMONS_MAX_RADIUS);
    demons_ctx* c = new (std::nothrow) demons_ctx();
    if (!c) return fail(DEMONS_E_ARG, "out of host memory");
    c->dims = Dims{dims[0], dims[1], dims[2]};
    for (int i = 0; i < 3; ++i) c->spacing[i] = spacing[i];
    c->variant = variant;
    c->alpha = alpha;
    c->sigma = sigma;
    *out = c;
    return DEMONS_OK;
}

void demons_destroy(demons_ctx* c) {
    if (!c) return;
    if (c->l2_granted > 0 || c->l2_limit_raised) {
        // hand the persisting lines back to normal use and restore the device limit this context raised
        // (work still running on a stream finishes correctly either way: the window is a hint)
        cudaCtxResetPersistingL2Cache();
        if (c->l2_limit_raised) cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, c->l2_prev_limit);
        cudaGetLastError();
    }
    for (auto& g : c->graphs) cudaGraphExecDestroy(g.exec);
    for (cudaEvent_t e : c->tg)
        if (e) cudaEventDestroy(e);
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    if (c->side) cudaStreamDestroy(c->side);
    for (int k = 0; k < 2; ++k) {
        if (c->q_up[k]) cudaEventDestroy(c->q_up[k]);
        if (c->q_done[k]) cudaEventDestroy(c->q_done[k]);
        if (c->q_down[k]) cudaEventDestroy(c->q_down[k]);
    }
    if (c->q_in) cudaStreamDestroy(c->q_in);
    if (c->q_out) cudaStreamDestroy(c->q_out);
    release_texture(c);
    prof_clear(c);
    delete c;
}

size_t demons_workspace_bytes(const demons_ctx* c, int levels) {
    if (!c || levels < 1 || levels > DEMONS_MAX_LEVELS) return 0;
    return make_partition(c, levels, 1).total;
}

size_t demons_workspace_bytes_batch(const demons_ctx* c, int levels, int nbatch) {
    if (!c || levels < 1 || levels > DEMONS_MAX_LEVELS || nbatch < 1 || nbatch > DEMONS_MAX_BATCH) return 0;
    const size_t single = make_partition(c, levels, 1).total, batch = make_partition(c, levels, nbatch).total;
    return batch > single ? batch : single;  // every single-registration entry point keeps working
}

int demons_set_workspace(demons_ctx* c, void* d_ws, size_t bytes) {
    if (!c || !d_ws) return fail(DEMONS_E_ARG, "ctx / workspace is NULL");
    if (reinterpret_cast<uintptr_t>(d_ws) % ALIGN) return fail(DEMONS_E_ARG, "workspace must be 256-byte aligned");
    if (bytes < make_partition(c, 1, 1).total)
        return fail(DEMONS_E_WORKSPACE, "workspace too small: %zu < %zu", bytes, make_partition(c, 1, 1).total);
    for (auto& g : c->graphs) cudaGraphExecDestroy(g.exec);
    c->graphs.clear();
    CUDA_TRY(cudaMemset(d_ws, 0, sizeof(Control)));
    CUDA_TRY(cudaDeviceSynchronize());
    c->ws = static_cast<char*>(d_ws);
    c->ws_bytes = bytes;
    return DEMONS_OK;
}

int demons_level_dims(const demons_ctx* c, int level, int out_dims[3]) {
    if (!c || !out_dims || level < 0 || level >= DEMONS_MAX_LEVELS) return fail(DEMONS_E_ARG, "bad arguments");
    Dims d = c->dims;
    for (int l = 0; l < level; ++l) d = coarser(d);
    out_dims[0] = d.nx;
    out_dims[1] = d.ny;
    out_dims[2] = d.nz;
    return DEMONS_OK;
}

long long demons_launch_count(const demons_ctx* c) { return c ? c->launches : 0; }

int demons_get_profile(const demons_ctx* c, double h_ms[4], long long h_launch_groups[4]) {
    if (!c || !h_ms || !h_launch_groups) return fail(DEMONS_E_ARG, "bad arguments");
    for (int k = 0; k < 4; ++k) {
        h_ms[k] = c->prof_ms[k];
        h_launch_groups[k] = c->prof_n[k];
    }
    return DEMONS_OK;
}

int demons_set_option(demons_ctx* c, const char* name, int value) {
    if (!c || !name) return fail(DEMONS_E_ARG, "bad arguments");
    if (!strcmp(name, "graphs")) c->opt_graphs = value != 0;
    else if (!strcmp(name, "texture")) c->opt_texture = value != 0;
    else if (!strcmp(name, "generic_smooth")) c->opt_generic_smooth = value != 0;
    else if (!strcmp(name, "profile")) c->opt_profile = value == 2 ? 2 : (value != 0);
    else if (!strcmp(name, "l2_persist")) c->opt_l2_persist = value != 0;
    else if (!strcmp(name, "zero_start")) c->opt_zero_start = value != 0;
    else if (!strcmp(name, "ic_one_field")) c->opt_ic_one_field = value != 0;
    else return fail(DEMONS_E_ARG, "unknown option '%s'", name);
    for (auto& g : c->graphs) cudaGraphExecDestroy(g.exec);
    c->graphs.clear();
    return DEMONS_OK;
}

int demons_register(demons_ctx* c, const float* d_static, const float* d_moving, float* d_u, float* d_u_back,
                    int levels, const int* h_iters, double eps, double* h_stats, int* h_iters_done, void* stream) {
    const int rc = check_register_args(c, d_static, d_moving, d_u, d_u_back, 1, levels, h_iters);
    if (rc != DEMONS_OK) return rc;
    return register_impl(c, d_static, d_moving, d_u, d_u_back, 1, levels, h_iters, eps, h_stats, h_iters_done,
                         static_cast<cudaStream_t>(stream));
}

int demons_register_batch(demons_ctx* c, int nbatch, const float* d_static, const float* d_moving, float* d_u,
                          float* d_u_back, int levels, const int* h_iters, double eps, double* h_stats,
                          int* h_iters_done, void* stream) {
    const int rc = check_register_args(c, d_static, d_moving, d_u, d_u_back, nbatch, levels, h_iters);
    if (rc != DEMONS_OK) return rc;
    return register_impl(c, d_static, d_moving, d_u, d_u_back, nbatch, levels, h_iters, eps, h_stats, h_iters_done,
                         static_cast<cudaStream_t>(stream));
}

int demons_register_host(demons_ctx* c, const float* h_static, const float* h_moving, float* h_u, float* h_u_back,
                         int levels, const int* h_iters, double eps, double* h_stats, int* h_iters_done,
                         void* stream) {
    const int rc = check_register_args(c, h_static, h_moving, h_u, h_u_back, 1, levels, h_iters);
    if (rc != DEMONS_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const Partition p = make_partition(c, levels, 1);
    const size_t N = nvox(c->dims);
    const bool ic = is_ic(c);
    float* dS = reinterpret_cast<float*>(c->ws + p.hI);  // M right behind S: one L2 window covers both
    float* dM = dS + N;
    float* dU = reinterpret_cast<float*>(c->ws + p.hU);
    float* dUb = ic ? reinterpret_cast<float*>(c->ws + p.hUb) : nullptr;
    CUDA_TRY(cudaMemcpyAsync(dS, h_static, N * 4, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(dM, h_moving, N * 4, cudaMemcpyHostToDevice, st));
    if (levels == 1 && !c->opt_zero_start) {
        CUDA_TRY(cudaMemcpyAsync(dU, h_u, 3 * N * 4, cudaMemcpyHostToDevice, st));
        if (ic) CUDA_TRY(cudaMemcpyAsync(dUb, h_u_back, 3 * N * 4, cudaMemcpyHostToDevice, st));
    }
    const int rr = register_impl(c, dS, dM, dU, dUb, 1, levels, h_iters, eps, nullptr, nullptr, st);
    if (rr != DEMONS_OK) return rr;
    CUDA_TRY(cudaMemcpyAsync(h_u, dU, 3 * N * 4, cudaMemcpyDeviceToHost, st));
    if (ic) CUDA_TRY(cudaMemcpyAsync(h_u_back, dUb, 3 * N * 4, cudaMemcpyDeviceToHost, st));
    long long total_iters = 0;
    for (int l = 0; l < levels; ++l) total_iters += h_iters[l];
    Control* ctl = reinterpret_cast<Control*>(c->ws + p.control);
    if (h_stats && total_iters > 0)
        CUDA_TRY(cudaMemcpyAsync(h_stats, c->ws + p.stats, (size_t)total_iters * 24, cudaMemcpyDeviceToHost, st));
    if (h_iters_done)
        CUDA_TRY(cudaMemcpyAsync(h_iters_done, ctl->iters_done, (size_t)levels * 4, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return DEMONS_OK;
}

namespace {
// Second staging slot of demons_register_host_queue, behind the single-registration partition.
struct QueueSlots {
    size_t hI[2], hU[2], hUb[2], total;
};
QueueSlots queue_slots(const demons_ctx* c, int levels) {
    const Partition p = make_partition(c, levels, 1);
    const size_t N = nvox(c->dims);
    QueueSlots q{};
    q.hI[0] = p.hI;
    q.hU[0] = p.hU;
    q.hUb[0] = p.hUb;
    size_t off = align_up(p.total);
    q.hI[1] = off;
    off += align_up(2 * N * 4);
    q.hU[1] = off;
    off += align_up(3 * N * 4);
    q.hUb[1] = is_ic(c) ? off : 0;
    if (is_ic(c)) off += align_up(3 * N * 4);
    q.total = off;
    return q;
}
}  // namespace

size_t demons_workspace_bytes_queue(const demons_ctx* c, int levels) {
    if (!c || levels < 1 || levels > DEMONS_MAX_LEVELS) return 0;
    return queue_slots(c, levels).total;
}

int demons_register_host_queue(demons_ctx* c, int n, const float* const* h_static, const float* const* h_moving,
                               float* const* h_u, float* const* h_u_back, int levels, const int* h_iters, double eps,
                               double* h_stats, int* h_iters_done, void* stream) {
    if (!c) return fail(DEMONS_E_ARG, "ctx is NULL");
    if (n < 1 || !h_static || !h_moving || !h_u) return fail(DEMONS_E_ARG, "n must be >= 1 and the pointer arrays non-NULL");
    const bool ic = is_ic(c);
    if (ic && !h_u_back) return fail(DEMONS_E_ARG, "variant 5 needs h_u_back");
    if (!ic && h_u_back) return fail(DEMONS_E_ARG, "h_u_back must be NULL unless variant 5");
    for (int k = 0; k < n; ++k) {
        const int rc = check_register_args(c, h_static[k], h_moving[k], h_u[k], ic ? h_u_back[k] : nullptr, 1, levels, h_iters);
        if (rc != DEMONS_OK) return rc;
    }
    const QueueSlots q = queue_slots(c, levels);
    if (q.total > c->ws_bytes)
        return fail(DEMONS_E_WORKSPACE, "workspace too small: have %zu bytes, need %zu (demons_workspace_bytes_queue)",
                    c->ws_bytes, q.total);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (!c->q_in) {
        // all eight objects or none: created into locals and handed to the context only when every one exists, so a
        // failure half-way leaves the context as it was and the next call tries again
        cudaStream_t qs[2] = {nullptr, nullptr};
        cudaEvent_t qe[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
        cudaError_t qerr = cudaSuccess;
        for (int k = 0; k < 2 && qerr == cudaSuccess; ++k) qerr = cudaStreamCreateWithFlags(&qs[k], cudaStreamNonBlocking);
        for (int k = 0; k < 6 && qerr == cudaSuccess; ++k) qerr = cudaEventCreateWithFlags(&qe[k], cudaEventDisableTiming);
        if (qerr != cudaSuccess) {
            for (cudaStream_t q : qs)
                if (q) cudaStreamDestroy(q);
            for (cudaEvent_t q : qe)
                if (q) cudaEventDestroy(q);
            return fail(DEMONS_E_CUDA, "creating the queue's streams and events failed: %s", cudaGetErrorString(qerr));
        }
        c->q_in = qs[0];
        c->q_out = qs[1];
        for (int k = 0; k < 2; ++k) {
            c->q_up[k] = qe[3 * k];
            c->q_done[k] = qe[3 * k + 1];
            c->q_down[k] = qe[3 * k + 2];
        }
    }
    const Partition p = make_partition(c, levels, 1);
    const size_t N = nvox(c->dims);
    long long total_iters = 0;
    for (int l = 0; l < levels; ++l) total_iters += h_iters[l];
    Control* ctl = reinterpret_cast<Control*>(c->ws + p.control);
    const bool upload_u = levels == 1 && !c->opt_zero_start;
    // everything enqueued before this call on `stream` comes first
    CUDA_TRY(cudaEventRecord(c->q_done[0], st));
    CUDA_TRY(cudaStreamWaitEvent(c->q_in, c->q_done[0], 0));
    CUDA_TRY(cudaStreamWaitEvent(c->q_out, c->q_done[0], 0));
    auto upload = [&](int k) -> int {  // images (and initial fields) of registration k into slot k & 1, on q_in
        const int s = k & 1;
        if (k >= 2) {
            CUDA_TRY(cudaStreamWaitEvent(c->q_in, c->q_done[s], 0));                // registration k - 2 is done with the images
            if (upload_u) CUDA_TRY(cudaStreamWaitEvent(c->q_in, c->q_down[s], 0));  // and its field has been read back
        }
        float* dS = reinterpret_cast<float*>(c->ws + q.hI[s]);
        CUDA_TRY(cudaMemcpyAsync(dS, h_static[k], N * 4, cudaMemcpyHostToDevice, c->q_in));
        CUDA_TRY(cudaMemcpyAsync(dS + N, h_moving[k], N * 4, cudaMemcpyHostToDevice, c->q_in));
        if (upload_u) {
            CUDA_TRY(cudaMemcpyAsync(c->ws + q.hU[s], h_u[k], 3 * N * 4, cudaMemcpyHostToDevice, c->q_in));
            if (ic) CUDA_TRY(cudaMemcpyAsync(c->ws + q.hUb[s], h_u_back[k], 3 * N * 4, cudaMemcpyHostToDevice, c->q_in));
        }
        CUDA_TRY(cudaEventRecord(c->q_up[s], c->q_in));
        return DEMONS_OK;
    };
    auto enqueue_all = [&]() -> int {
        int rc = upload(0);
        if (rc != DEMONS_OK) return rc;
        for (int k = 0; k < n; ++k) {
            const int s = k & 1;
            if (k + 1 < n && (rc = upload(k + 1)) != DEMONS_OK) return rc;  // rides beside registration k
            float* dS = reinterpret_cast<float*>(c->ws + q.hI[s]);
            float* dU = reinterpret_cast<float*>(c->ws + q.hU[s]);
            float* dUb = ic ? reinterpret_cast<float*>(c->ws + q.hUb[s]) : nullptr;
            CUDA_TRY(cudaStreamWaitEvent(st, c->q_up[s], 0));
            if (k >= 2) CUDA_TRY(cudaStreamWaitEvent(st, c->q_down[s], 0));  // the field of registration k - 2 has left the slot
            rc = register_impl(c, dS, dS + N, dU, dUb, 1, levels, h_iters, eps, nullptr, nullptr, st);
            if (rc != DEMONS_OK) return rc;
            if (h_stats && total_iters > 0)
                CUDA_TRY(cudaMemcpyAsync(h_stats + (size_t)k * total_iters * 3, c->ws + p.stats, (size_t)total_iters * 24,
                                         cudaMemcpyDeviceToHost, st));
            if (h_iters_done)
                CUDA_TRY(cudaMemcpyAsync(h_iters_done + (size_t)k * levels, ctl->iters_done, (size_t)levels * 4,
                                         cudaMemcpyDeviceToHost, st));
            CUDA_TRY(cudaEventRecord(c->q_done[s], st));
            CUDA_TRY(cudaStreamWaitEvent(c->q_out, c->q_done[s], 0));
            CUDA_TRY(cudaMemcpyAsync(h_u[k], dU, 3 * N * 4, cudaMemcpyDeviceToHost, c->q_out));
            if (ic) CUDA_TRY(cudaMemcpyAsync(h_u_back[k], dUb, 3 * N * 4, cudaMemcpyDeviceToHost, c->q_out));
            CUDA_TRY(cudaEventRecord(c->q_down[s], c->q_out));
        }
        CUDA_TRY(cudaStreamWaitEvent(st, c->q_down[0], 0));  // `stream` ends behind the last downloads
        if (n > 1) CUDA_TRY(cudaStreamWaitEvent(st, c->q_down[1], 0));
        return DEMONS_OK;
    };
    const int rq = enqueue_all();
    // drain the three streams whatever happened: the caller's buffers must not be in flight when this call returns
    const cudaError_t e_in = cudaStreamSynchronize(c->q_in), e_out = cudaStreamSynchronize(c->q_out), e_st = cudaStreamSynchronize(st);
    if (rq != DEMONS_OK) return rq;
    if (e_in != cudaSuccess || e_out != cudaSuccess || e_st != cudaSuccess)
        return fail(DEMONS_E_CUDA, "queue synchronise failed: %s", cudaGetErrorString(e_in != cudaSuccess ? e_in : e_out != cudaSuccess ? e_out : e_st));
    return DEMONS_OK;
}

int demons_warp_force(demons_ctx* c, const int dims[3], const float* d_static, const float* d_moving,
                      const float* d_u_in, float* d_u_out, const float* d_ub_in, float* d_ub_out, double* d_metrics,
                      void* stream) {
    if (!c) return fail(DEMONS_E_ARG, "ctx is NULL");
    Dims d;
    int rc = check_call_dims(c, dims, &d);
    if (rc != DEMONS_OK) return rc;
    if (!d_static || !d_moving || !d_u_in || !d_u_out) return fail(DEMONS_E_ARG, "NULL volume / field pointer");
    if (d_u_in == d_u_out) return fail(DEMONS_E_ARG, "u_out must not alias u_in");
    const bool ic = is_ic(c);
    if (ic && (!d_ub_in || !d_ub_out)) return fail(DEMONS_E_ARG, "variant 5 needs ub_in and ub_out");
    if (!ic && (d_ub_in || d_ub_out)) return fail(DEMONS_E_ARG, "ub_in / ub_out must be NULL unless variant 5");
    if (ic && d_ub_in == d_ub_out) return fail(DEMONS_E_ARG, "ub_out must not alias ub_in");
    rc = check_ws(c, 1);
    if (rc != DEMONS_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const Partition p = make_partition(c, 1, 1);
    ForceArgs fa{};
    fa.d = d;
    fa.variant = c->variant;
    fa.alpha2 = c->variant == DEMONS_ADJUSTED_DOUBLE ? c->alpha * c->alpha : 1.f;
    fa.nb = 1;
    fa.img_stride = nvox(d);
    fa.S = d_static;
    fa.M = d_moving;
    fa.u_in = d_u_in;
    fa.u_out = d_u_out;
    fa.ub_in = d_ub_in;
    fa.ub_out = d_ub_out;
    fa.Mw = reinterpret_cast<float*>(c->ws + p.Mw);
    fa.Sw = ic ? reinterpret_cast<float*>(c->ws + p.Sw) : nullptr;
    fa.sink = make_sink(c, p, 0, d_metrics, 0, false, 0.0);
    const L2Window win = l2_window(c, d, d_static, d_moving, nvox(d), 1);
    fa.l2_ptr = win.ptr;
    fa.l2_bytes = win.bytes;
    fa.l2_ratio = win.ratio;
    if (c->opt_texture) {
        rc = bind_texture(c, d, d_moving, st);
        if (rc != DEMONS_OK) return rc;
        fa.texM = c->tex;
    }
    if (c->variant == DEMONS_EVOLVED_PASSIVE) {
        if (launch_grad_mag2(d, d_moving, nvox(d), fa.Mw, 1, st) < 0)
            return fail(DEMONS_E_CUDA, "gradient launch failed: %s", cudaGetErrorString(cudaGetLastError()));
        c->launches += 1;
    }
    const int n = launch_warp_force(fa, st);
    if (n < 0) return fail(DEMONS_E_CUDA, "warp_force launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    c->launches += n;
    return DEMONS_OK;
}

int demons_warp_force_slab(demons_ctx* c, const int dims[3], int z_begin, int z_count, int own_begin, int own_count,
                           const float* d_static, const float* d_moving, const float* d_u_in, float* d_u_out,
                           const float* d_ub_in, float* d_ub_out, double* d_metrics, void* stream) {
    if (!c) return fail(DEMONS_E_ARG, "ctx is NULL");
    Dims g;
    int rc = check_call_dims(c, dims, &g);
    if (rc != DEMONS_OK) return rc;
    if (g.nx < 2 || g.ny < 2 || g.nz < 2) return fail(DEMONS_E_UNSUPPORTED, "the slab form needs at least 2 voxels per axis");
    if (z_begin < 0 || z_count < 2 || z_begin + z_count > g.nz) return fail(DEMONS_E_ARG, "slab outside the volume");
    if (own_begin < 0 || own_count < 0 || own_begin + own_count > z_count) return fail(DEMONS_E_ARG, "own planes outside the slab");
    if (!d_static || !d_moving || !d_u_in || !d_u_out) return fail(DEMONS_E_ARG, "NULL volume / field pointer");
    if (d_u_in == d_u_out) return fail(DEMONS_E_ARG, "u_out must not alias u_in");
    const bool ic = is_ic(c);
    // variant 5 without the backward field: the one-field form (the caller holds u_b = -u_f, pin P10)
    const bool one_field = ic && !d_ub_in && !d_ub_out;
    if (ic && !one_field && (!d_ub_in || !d_ub_out)) return fail(DEMONS_E_ARG, "variant 5 needs both ub_in and ub_out, or neither");
    if (!ic && (d_ub_in || d_ub_out)) return fail(DEMONS_E_ARG, "ub_in / ub_out must be NULL unless variant 5");
    if (c->opt_texture) return fail(DEMONS_E_UNSUPPORTED, "the texture option serves whole volumes only");
    rc = check_ws(c, 1);
    if (rc != DEMONS_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const Partition p = make_partition(c, 1, 1);
    ForceArgs fa{};
    fa.d = Dims{g.nx, g.ny, z_count};
    fa.variant = c->variant;
    fa.alpha2 = c->variant == DEMONS_ADJUSTED_DOUBLE ? c->alpha * c->alpha : 1.f;
    fa.nb = 1;
    fa.img_stride = nvox(g);
    fa.S = d_static;
    fa.M = d_moving;
    fa.u_in = d_u_in;
    fa.u_out = d_u_out;
    fa.ub_in = d_ub_in;
    fa.ub_out = d_ub_out;
    fa.Mw = reinterpret_cast<float*>(c->ws + p.Mw);  // variant 1: |grad M|^2 in GLOBAL indexing; else the slab's Mw
    fa.Sw = ic ? reinterpret_cast<float*>(c->ws + p.Sw) : nullptr;
    fa.sink = make_sink(c, p, 0, d_metrics, 0, false, 0.0);
    fa.one_field = one_field ? 1 : 0;
    fa.slab = 1;
    fa.zoff = z_begin;
    fa.gnz = g.nz;
    fa.mz0 = own_begin;
    fa.mz1 = own_begin + own_count;
    const L2Window win = l2_window(c, g, d_static, d_moving, nvox(g), 1);
    fa.l2_ptr = win.ptr;
    fa.l2_bytes = win.bytes;
    fa.l2_ratio = win.ratio;
    if (c->variant == DEMONS_EVOLVED_PASSIVE) {  // the planes of this slab only
        if (launch_grad_mag2(g, d_moving, nvox(g), fa.Mw, 1, st, z_begin, z_count) < 0)
            return fail(DEMONS_E_CUDA, "gradient launch failed: %s", cudaGetErrorString(cudaGetLastError()));
        c->launches += 1;
    }
    const int n = launch_warp_force(fa, st);
    if (n < 0) return fail(DEMONS_E_CUDA, "warp_force launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    c->launches += n;
    return DEMONS_OK;
}

int demons_smooth(demons_ctx* c, const int dims[3], const float* d_in, float* d_out, int ncomp, float sigma,
                  void* stream) {
    if (!c) return fail(DEMONS_E_ARG, "ctx is NULL");
    Dims d;
    int rc = check_call_dims(c, dims, &d);
    if (rc != DEMONS_OK) return rc;
    if (!d_in || !d_out) return fail(DEMONS_E_ARG, "NULL field pointer");
    if (d_in == d_out) return fail(DEMONS_E_ARG, "in-place smoothing is not supported");
    if (ncomp < 1 || ncomp > 6) return fail(DEMONS_E_ARG, "ncomp must be 1..6");
    if (!(sigma > 0.f) || !std::isfinite(sigma)) return fail(DEMONS_E_ARG, "sigma must be positive");
    SmoothArgs sa{};
    sa.R = gaussian_taps(sigma, sa.w);
    if (sa.R < 0) return fail(DEMONS_E_UNSUPPORTED, "ceil(3 sigma) exceeds DEMONS_MAX_RADIUS (%d)", DEMONS_MAX_RADIUS);
    rc = check_ws(c, 1);
    if (rc != DEMONS_OK) return rc;
    const Partition p = make_partition(c, 1, 1);
    sa.d = d;
    sa.in = d_in;
    sa.out = d_out;
    sa.tmp = reinterpret_cast<float*>(c->ws + p.smooth_tmp);
    sa.ncomp = ncomp;
    sa.comps_per_pair = ncomp;
    sa.ctl = nullptr;
    sa.force_generic = c->opt_generic_smooth;
    const int n = launch_smooth(sa, static_cast<cudaStream_t>(stream));
    if (n < 0) return fail(DEMONS_E_CUDA, "smooth launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    c->launches += n;
    return DEMONS_OK;
}

int demons_restrict(demons_ctx* c, const int fine_dims[3], const float* d_fine, float* d_coarse, void* stream) {
    if (!c) return fail(DEMONS_E_ARG, "ctx is NULL");
    if (!dims_ok(fine_dims)) return fail(DEMONS_E_ARG, "bad dims");
    if (!d_fine || !d_coarse) return fail(DEMONS_E_ARG, "NULL volume pointer");
    const Dims fd{fine_dims[0], fine_dims[1], fine_dims[2]};
    if (launch_restrict(fd, d_fine, 0, d_coarse, 0, 1, static_cast<cudaStream_t>(stream)) < 0)
        return fail(DEMONS_E_CUDA, "restrict launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    c->launches += 1;
    return DEMONS_OK;
}

int demons_prolong(demons_ctx* c, const int coarse_dims[3], const float* d_uc, const int fine_dims[3], float* d_uf,
                   void* stream) {
    if (!c) return fail(DEMONS_E_ARG, "ctx is NULL");
    if (!dims_ok(coarse_dims) || !dims_ok(fine_dims)) return fail(DEMONS_E_ARG, "bad dims");
    if (!d_uc || !d_uf) return fail(DEMONS_E_ARG, "NULL field pointer");
    for (int i = 0; i < 3; ++i)
        if (coarse_dims[i] != (fine_dims[i] + 1) / 2)
            return fail(DEMONS_E_ARG, "coarse dims must be ceil(fine dims / 2)");
    const Dims cd{coarse_dims[0], coarse_dims[1], coarse_dims[2]};
    const Dims fd{fine_dims[0], fine_dims[1], fine_dims[2]};
    if (launch_prolong(cd, d_uc, fd, d_uf, 1, static_cast<cudaStream_t>(stream)) < 0)
        return fail(DEMONS_E_CUDA, "prolong launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    c->launches += 1;
    return DEMONS_OK;
}

int demons_ssd(demons_ctx* c, const int dims[3], const float* d_static, const float* d_moving, const float* d_u,
               const float* d_ub, double* d_out, void* stream) {
    if (!c) return fail(DEMONS_E_ARG, "ctx is NULL");
    Dims d;
    int rc = check_call_dims(c, dims, &d);
    if (rc != DEMONS_OK) return rc;
    if (!d_static || !d_moving || !d_u || !d_out) return fail(DEMONS_E_ARG, "NULL pointer");
    if (is_ic(c) != (d_ub != nullptr)) return fail(DEMONS_E_ARG, "ub must be given exactly for variant 5");
    rc = check_ws(c, 1);
    if (rc != DEMONS_OK) return rc;
    const Partition p = make_partition(c, 1, 1);
    ReduceScratch rs{reinterpret_cast<double*>(c->ws + p.partials),
                     &reinterpret_cast<Control*>(c->ws + p.control)->ticket, p.partial_stride};
    if (launch_ssd(d, d_static, d_moving, d_u, d_ub, d_out, rs, static_cast<cudaStream_t>(stream)) < 0)
        return fail(DEMONS_E_CUDA, "ssd launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    c->launches += 1;
    return DEMONS_OK;
}

int demons_ic_error(demons_ctx* c, const int dims[3], const float* d_uf, const float* d_ub, double* d_out,
                    void* stream) {
    if (!c) return fail(DEMONS_E_ARG, "ctx is NULL");
    Dims d;
    int rc = check_call_dims(c, dims, &d);
    if (rc != DEMONS_OK) return rc;
    if (!d_uf || !d_ub || !d_out) return fail(DEMONS_E_ARG, "NULL pointer");
    rc = check_ws(c, 1);
    if (rc != DEMONS_OK) return rc;
    const Partition p = make_partition(c, 1, 1);
    ReduceScratch rs{reinterpret_cast<double*>(c->ws + p.partials),
                     &reinterpret_cast<Control*>(c->ws + p.control)->ticket, p.partial_stride};
    if (launch_ic_error(d, d_uf, d_ub, d_out, rs, static_cast<cudaStream_t>(stream)) < 0)
        return fail(DEMONS_E_CUDA, "ic_error launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    c->launches += 1;
    return DEMONS_OK;
}

int demons_cc(demons_ctx* c, const int dims[3], const float* d_static, const float* d_moving, const float* d_u,
              const float* d_ub, double* d_out, void* stream) {
    if (!c) return fail(DEMONS_E_ARG, "ctx is NULL");
    Dims d;
    int rc = check_call_dims(c, dims, &d);
    if (rc != DEMONS_OK) return rc;
    if (!d_static || !d_moving || !d_u || !d_out) return fail(DEMONS_E_ARG, "NULL pointer");
    if (is_ic(c) && !d_ub) return fail(DEMONS_E_ARG, "variant 5 needs u_back");
    if (!is_ic(c) && d_ub) return fail(DEMONS_E_ARG, "u_back must be NULL unless variant 5");
    rc = check_ws(c, 1);
    if (rc != DEMONS_OK) return rc;
    const Partition p = make_partition(c, 1, 1);
    ReduceScratch rs{reinterpret_cast<double*>(c->ws + p.partials),
                     &reinterpret_cast<Control*>(c->ws + p.control)->ticket, p.partial_stride};
    if (launch_cc(d, d_static, d_moving, d_u, d_ub, d_out, rs, static_cast<cudaStream_t>(stream)) < 0)
        return fail(DEMONS_E_CUDA, "cc launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    c->launches += 1;
    return DEMONS_OK;
}

int demons_point_error(demons_ctx* c, const int dims[3], const float* d_u, int n_points, const float* d_points,
                       const float* d_expect, double* d_err, void* stream) {
    if (!c) return fail(DEMONS_E_ARG, "ctx is NULL");
    if (!dims_ok(dims)) return fail(DEMONS_E_ARG, "bad dims");
    if (n_points < 0) return fail(DEMONS_E_ARG, "negative point count");
    if (n_points == 0) return DEMONS_OK;
    if (!d_u || !d_points || !d_expect || !d_err) return fail(DEMONS_E_ARG, "NULL pointer");
    const Dims d{dims[0], dims[1], dims[2]};
    if (launch_point_error(d, c->spacing, d_u, n_points, d_points, d_expect, d_err, static_cast<cudaStream_t>(stream)) < 0)
        return fail(DEMONS_E_CUDA, "point_error launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    c->launches += 1;
    return DEMONS_OK;
}

}  // extern "C"

// api.cu -- C ABI of libasr_sched (include/asr_sched.h): argument checks,
// workspace carving, launch sequencing.  No compute happens on the host.
#include <atomic>
#include <climits>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>

#include "launchers.cuh"

namespace asr {

static thread_local char g_err[512] = "";
static std::atomic<long long> g_launches{0};

void set_error(const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

int check_launch(const char *what) {
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        set_error("%s: %s", what, cudaGetErrorString(e));
        return ASR_ECUDA;
    }
    return ASR_OK;
}

void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

// grids are sized from the SM count of the device the call runs on
int sm_count() {
    static std::atomic<int> cache[64];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return 148;
    }
    if (dev >= 0 && dev < 64) {
        const int c = cache[dev].load(std::memory_order_relaxed);
        if (c > 0) return c;
    }
    int n = 0;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1) {
        cudaGetLastError();
        n = 148;
    }
    if (dev >= 0 && dev < 64) cache[dev].store(n, std::memory_order_relaxed);
    return n;
}

// ---- per-kernel timing: one CUDA-event pair per launch, on the launch stream
static const char *const g_kernel_names[KID_COUNT] = {
    "select_topk_kernel", "sim_prepare_kernel", "sim_warp_kernel", "sim_lane_kernel", "summary_percentiles_kernel",
    "percentiles_kernel", "gen_trace_kernel", "gen_queues_kernel", "build_sweep_replicas_kernel", "sim_cta_kernel", "sim_init_lat_kernel", "sim_ex_kernel", "tpot_kernel", "estimate_kernel", "itl_percentiles_kernel", "summary_stream_kernel", "lane_plan_kernels", "sim_lane_kernel(repair)", "sim_lane_kernel(redo)", "select_wide_kernel"};
struct TimedLaunch {
    int kid;
    cudaEvent_t start, stop;
};
static std::mutex g_timing_mu;
static bool g_timing_on = false;
static std::vector<TimedLaunch> g_timed;      // recorded launches since the last reset
static std::vector<cudaEvent_t> g_event_pool; // recycled events

static cudaEvent_t take_event() {
    if (!g_event_pool.empty()) {
        cudaEvent_t e = g_event_pool.back();
        g_event_pool.pop_back();
        return e;
    }
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    return e;
}

KernelTimer::KernelTimer(int kid, cudaStream_t st) : kid_(kid), st_(st), slot_(-1) {
    count_launch();
    std::lock_guard<std::mutex> g(g_timing_mu);
    if (!g_timing_on) return;
    TimedLaunch t{kid, take_event(), take_event()};
    if (!t.start || !t.stop) return;
    cudaEventRecord(t.start, st);
    g_timed.push_back(t);
    slot_ = (int)g_timed.size() - 1;
}

KernelTimer::~KernelTimer() {
    if (slot_ < 0) return;
    std::lock_guard<std::mutex> g(g_timing_mu);
    if (slot_ < (int)g_timed.size()) cudaEventRecord(g_timed[slot_].stop, st_);
}

static inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

struct SimWorkspace {
    size_t bm_off_bytes, bitmap_bytes, defer_bytes, lat_bytes, total;
    // summary-only calls: the time-split plan of the thread-per-replica tier, behind everything else
    size_t plan_off, order_bytes, seg_bytes, unit_q_bytes;
};

// asr_sched_set_option values
static std::atomic<int> g_opt_lane_min{1024};
static std::atomic<int> g_opt_escalate{4096};
static std::atomic<int> g_opt_lane_split{1};

static SimWorkspace sim_ws(int64_t total_requests, int64_t n_replicas, bool summary_only) {
    SimWorkspace w;
    w.bm_off_bytes = align_up(sizeof(int64_t) * (size_t)(n_replicas + 1));
    w.bitmap_bytes = align_up(sizeof(uint32_t) * (size_t)(total_requests / 32 + 2 * n_replicas + 2));
    w.defer_bytes = align_up(sizeof(int32_t) * (size_t)(2 * n_replicas + 64));   // [0], [1]: counters, [64..]: the two lists
    w.lat_bytes = summary_only ? align_up(sizeof(int64_t) * (size_t)total_requests) : 0;
    w.total = w.bm_off_bytes + w.bitmap_bytes + w.defer_bytes + 2 * w.lat_bytes;
    w.plan_off = w.total;
    w.order_bytes = summary_only ? align_up(sizeof(int32_t) * (size_t)n_replicas) : 0;   // also: failed
    w.seg_bytes = summary_only ? align_up((size_t)n_replicas) : 0;                        // load class; segments
    // + counters; after the simulation the region is the percentile kernels' scratch (seed list: 2 n + 64 + runs)
    w.unit_q_bytes = summary_only ? align_up(sizeof(int32_t) * (size_t)n_replicas * LANE_MAX_SEG + 64 + 512) : 0;
    w.total += 2 * w.order_bytes + 2 * w.seg_bytes + w.unit_q_bytes;
    return w;
}

// asr_sched_itl_batched: the summary-only simulate workspace + second bitmap + zeroed extension
// descriptors + gap histogram + (duration, weight) pairs + pair counts
struct ItlWorkspace {
    size_t sim_bytes, ext_bytes, hist_bytes, pairs_bytes, np_bytes, total;
};
static ItlWorkspace itl_ws(int64_t total_requests, int64_t n_replicas) {
    ItlWorkspace w;
    const SimWorkspace s = sim_ws(total_requests, n_replicas, true);
    w.sim_bytes = s.total + s.bitmap_bytes;
    w.ext_bytes = align_up(sizeof(asr_sim_ext_t) * 4096);   // n_cms <= 4096 for this call
    w.hist_bytes = align_up(sizeof(unsigned long long) * (size_t)ITL_BINS * (size_t)n_replicas);
    w.pairs_bytes = align_up(sizeof(int64_t) * 2 * (size_t)(total_requests + 1));
    w.np_bytes = align_up(sizeof(int32_t) * (size_t)(n_replicas + 1));
    w.total = w.sim_bytes + w.ext_bytes + w.hist_bytes + w.pairs_bytes + w.np_bytes;
    return w;
}

}  // namespace asr

using namespace asr;

#define CUDA_TRY(expr, what)                                         \
    do {                                                             \
        cudaError_t _e = (expr);                                     \
        if (_e != cudaSuccess) {                                     \
            set_error("%s: %s", what, cudaGetErrorString(_e));       \
            return ASR_ECUDA;                                        \
        }                                                            \
    } while (0)

extern "C" const char *asr_sched_last_error(void) { return g_err; }
extern "C" int asr_sched_version(void) { return ASR_SCHED_VERSION; }
extern "C" int64_t asr_sched_launch_count(void) { return (int64_t)g_launches.load(); }

extern "C" int asr_sched_set_option(int32_t option, int64_t value) {
    switch (option) {
        case ASR_OPT_SIM_LANE_MIN_REPLICAS:
            if (value < 1 || value > INT32_MAX) break;
            g_opt_lane_min.store((int)value);
            return ASR_OK;
        case ASR_OPT_SIM_ESCALATE_WINDOW:
            if (value < 0 || value > INT32_MAX) break;
            g_opt_escalate.store((int)value);
            return ASR_OK;
        case ASR_OPT_SIM_LANE_SPLIT:
            if (value < 0 || value > 1) break;
            g_opt_lane_split.store((int)value);
            return ASR_OK;
    }
    set_error("set_option: bad option %d or value %lld", option, (long long)value);
    return ASR_EINVAL;
}

extern "C" int asr_sched_timing_enable(int on) {
    std::lock_guard<std::mutex> g(g_timing_mu);
    g_timing_on = on != 0;
    return ASR_OK;
}

extern "C" int asr_sched_timing_reset(void) {
    std::lock_guard<std::mutex> g(g_timing_mu);
    for (auto &t : g_timed) {
        g_event_pool.push_back(t.start);
        g_event_pool.push_back(t.stop);
    }
    g_timed.clear();
    return ASR_OK;
}

extern "C" const char *asr_sched_kernel_name(int32_t kernel_id) {
    return kernel_id >= 0 && kernel_id < KID_COUNT ? g_kernel_names[kernel_id] : nullptr;
}

extern "C" int asr_sched_timing_read(int32_t kernel_id, double *total_ms, int64_t *launches) {
    if (kernel_id < 0 || kernel_id >= KID_COUNT || !total_ms || !launches) {
        set_error("timing_read: bad argument");
        return ASR_EINVAL;
    }
    std::lock_guard<std::mutex> g(g_timing_mu);
    double ms = 0.0;
    int64_t n = 0;
    for (auto &t : g_timed) {
        if (t.kid != kernel_id) continue;
        cudaError_t e = cudaEventSynchronize(t.stop);
        float f = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&f, t.start, t.stop);
        if (e != cudaSuccess) {
            set_error("timing_read: %s", cudaGetErrorString(e));
            return ASR_ECUDA;
        }
        ms += f;
        n++;
    }
    *total_ms = ms;
    *launches = n;
    return ASR_OK;
}

extern "C" size_t asr_sched_workspace_bytes(int32_t op, int64_t a, int64_t b, int64_t c) {
    if (a < 0 || b < 0) return 0;
    switch (op) {
        case ASR_OP_SELECT: return select_workspace_bytes(a, b);
        case ASR_OP_SIMULATE: return sim_ws(a, b, c != 0).total + 512;   // + descriptors of the single-replica call
        case ASR_OP_SIMULATE_EX: return sim_ws(a, b, c != 0).total + sim_ws(a, b, c != 0).bitmap_bytes;
        case ASR_OP_PERCENTILES: return 0;
        case ASR_OP_ITL: return itl_ws(a, b).total;
    }
    return 0;
}

extern "C" int asr_sched_simulate_batched(const asr_req_t *traces, const asr_replica_t *replicas,
                                          int32_t n_replicas, const asr_cost_model_t *cms, int32_t n_cms,
                                          int64_t total_requests, int32_t max_slots, int64_t *out_lat,
                                          int64_t *out_ttft, asr_summary_t *out_summary, void *workspace,
                                          size_t workspace_bytes, void *stream) {
    if (n_replicas < 0 || n_cms < 1 || total_requests < 0 || max_slots < 1) {
        set_error("simulate_batched: bad argument (n_replicas=%d n_cms=%d total=%lld max_slots=%d)", n_replicas,
                  n_cms, (long long)total_requests, max_slots);
        return ASR_EINVAL;
    }
    if (max_slots > 256) {
        set_error("simulate_batched: max_slots=%d exceeds the limit 256", max_slots);
        return ASR_EUNSUPPORTED;
    }
    if (n_replicas == 0) return ASR_OK;
    if (!replicas || !cms || (!traces && total_requests > 0) || ((out_lat == nullptr) != (out_ttft == nullptr))) {
        set_error("simulate_batched: null pointer (out_lat and out_ttft must both be given or both be NULL)");
        return ASR_EINVAL;
    }
    const bool summary_only = out_lat == nullptr;
    if (summary_only && !out_summary) {
        set_error("simulate_batched: nothing to output");
        return ASR_EINVAL;
    }
    const SimWorkspace w = sim_ws(total_requests, n_replicas, summary_only);
    if (!workspace || workspace_bytes < w.total) {
        set_error("simulate_batched: workspace too small (%zu < %zu)", workspace_bytes, w.total);
        return ASR_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    char *ws = (char *)workspace;
    int64_t *bm_off = (int64_t *)ws;
    uint32_t *bitmap = (uint32_t *)(ws + w.bm_off_bytes);
    int32_t *defer = (int32_t *)(ws + w.bm_off_bytes + w.bitmap_bytes);
    if (summary_only) {
        out_lat = (int64_t *)(ws + w.bm_off_bytes + w.bitmap_bytes + w.defer_bytes);
        out_ttft = (int64_t *)(ws + w.bm_off_bytes + w.bitmap_bytes + w.defer_bytes + w.lat_bytes);
    }
    int rc = ASR_OK;
    SimArgs a{traces,  replicas, cms,         bm_off,         bitmap,     defer + 64, defer, defer + 64 + n_replicas, defer + 1,
              out_lat, out_ttft, out_summary, total_requests, n_replicas, n_cms, summary_only ? 1 : 0,
              g_opt_escalate.load(), LanePlan{}};
    // many small replicas: one thread each; few or wide ones: one warp each
    const bool use_lane = max_slots <= 32 && n_replicas >= g_opt_lane_min.load();
    if (use_lane && summary_only && g_opt_lane_split.load() && (int64_t)n_replicas * LANE_MAX_SEG < INT32_MAX) {
        char *pl = ws + w.plan_off;
        a.plan.order = (int32_t *)pl;
        a.plan.failed = (int32_t *)(pl + w.order_bytes);
        pl += 2 * w.order_bytes;
        a.plan.bucket = (uint8_t *)pl;
        a.plan.nseg = (uint8_t *)(pl + w.seg_bytes);
        pl += 2 * w.seg_bytes;
        a.plan.unit_q = (int32_t *)pl;
        a.plan.counters = a.plan.unit_q + (size_t)n_replicas * LANE_MAX_SEG;
    }
    if (!a.plan.order) {   // (with a plan its second kernel does this job beside the sort)
        rc = launch_sim_prepare(replicas, n_replicas, total_requests, bm_off, defer, st);
        if (rc) return rc;
    }
    rc = launch_simulate(a, max_slots, use_lane, st);
    if (rc) return rc;
    if (out_summary) {
        // the hand-over lists are spent: miss lists; so is the plan's unit_q region: seed lists
        int32_t *scratch = summary_only ? (int32_t *)(ws + w.plan_off + 2 * w.order_bytes + 2 * w.seg_bytes) : nullptr;
        rc = launch_summary_percentiles(replicas, n_replicas, out_lat, out_ttft, out_summary, use_lane && summary_only,
                                        a.plan.order, defer + 64, defer + 2, scratch, st);
    }
    return rc;
}

extern "C" int asr_sched_simulate_batched_ex(const asr_req_t *traces, const asr_replica_t *replicas,
                                             int32_t n_replicas, const asr_cost_model_t *cms,
                                             const asr_sim_ext_t *exts, int32_t n_cms, int64_t total_requests,
                                             int32_t max_slots, int64_t *out_lat, int64_t *out_ttft,
                                             asr_summary_t *out_summary, int64_t *out_preempt, void *workspace,
                                             size_t workspace_bytes, void *stream) {
    if (n_replicas < 0 || n_cms < 1 || total_requests < 0 || max_slots < 1) {
        set_error("simulate_batched_ex: bad argument (n_replicas=%d n_cms=%d total=%lld max_slots=%d)", n_replicas,
                  n_cms, (long long)total_requests, max_slots);
        return ASR_EINVAL;
    }
    if (max_slots > 256) {
        set_error("simulate_batched_ex: max_slots=%d exceeds the limit 256", max_slots);
        return ASR_EUNSUPPORTED;
    }
    if (n_replicas == 0) return ASR_OK;
    if (!replicas || !cms || !exts || (!traces && total_requests > 0) ||
        ((out_lat == nullptr) != (out_ttft == nullptr))) {
        set_error("simulate_batched_ex: null pointer (out_lat and out_ttft must both be given or both be NULL)");
        return ASR_EINVAL;
    }
    const bool summary_only = out_lat == nullptr;
    if (summary_only && !out_summary) {
        set_error("simulate_batched_ex: nothing to output");
        return ASR_EINVAL;
    }
    const SimWorkspace w = sim_ws(total_requests, n_replicas, summary_only);
    if (!workspace || workspace_bytes < w.total + w.bitmap_bytes) {
        set_error("simulate_batched_ex: workspace too small (%zu < %zu)", workspace_bytes, w.total + w.bitmap_bytes);
        return ASR_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    char *ws = (char *)workspace;
    int64_t *bm_off = (int64_t *)ws;
    uint32_t *bitmap = (uint32_t *)(ws + w.bm_off_bytes);
    int32_t *defer = (int32_t *)(ws + w.bm_off_bytes + w.bitmap_bytes);
    if (summary_only) {
        out_lat = (int64_t *)(ws + w.bm_off_bytes + w.bitmap_bytes + w.defer_bytes);
        out_ttft = (int64_t *)(ws + w.bm_off_bytes + w.bitmap_bytes + w.defer_bytes + w.lat_bytes);
    }
    uint32_t *bitmap2 = (uint32_t *)(ws + w.total);
    int rc = launch_sim_prepare(replicas, n_replicas, total_requests, bm_off, defer, st);
    if (rc) return rc;
    SimExArgs a;
    static_cast<SimArgs &>(a) = SimArgs{traces,  replicas, cms,         bm_off,         bitmap,     defer + 64, defer,
                                        defer + 64 + n_replicas, defer + 1,
                                        out_lat, out_ttft, out_summary, total_requests, n_replicas, n_cms, 0,
                                        g_opt_escalate.load(), LanePlan{}};
    a.exts = exts;
    a.bitmap2 = bitmap2;
    a.out_preempt = out_preempt;
    a.itl_hist = nullptr;
    a.itl_pairs = nullptr;
    a.itl_npairs = nullptr;
    rc = launch_simulate_ex(a, max_slots, st);
    if (rc) return rc;
    if (out_summary) rc = launch_summary_percentiles(replicas, n_replicas, out_lat, out_ttft, out_summary, false, nullptr, nullptr, nullptr, nullptr, st);
    return rc;
}

extern "C" int asr_sched_itl_batched(const asr_req_t *traces, const asr_replica_t *replicas, int32_t n_replicas,
                                     const asr_cost_model_t *cms, int32_t n_cms, int64_t total_requests,
                                     int32_t max_slots, const int32_t *pcts, int32_t n_pct, int64_t *out,
                                     void *workspace, size_t workspace_bytes, void *stream) {
    if (n_replicas < 0 || n_cms < 1 || total_requests < 0 || max_slots < 1 || n_pct < 0 || (n_pct > 0 && !pcts)) {
        set_error("itl_batched: bad argument (n_replicas=%d n_cms=%d total=%lld max_slots=%d n_pct=%d)", n_replicas,
                  n_cms, (long long)total_requests, max_slots, n_pct);
        return ASR_EINVAL;
    }
    if (max_slots > 256 || n_pct > 8 || n_cms > 4096) {
        set_error("itl_batched: limit exceeded (max_slots=%d n_pct=%d n_cms=%d)", max_slots, n_pct, n_cms);
        return ASR_EUNSUPPORTED;
    }
    ItlPcts pl;
    pl.n_pct = n_pct;
    for (int j = 0; j < 8; ++j) {
        pl.pct[j] = j < n_pct ? pcts[j] : 0;
        if (j < n_pct && (pcts[j] < 1 || pcts[j] > 100)) {
            set_error("itl_batched: percentile %d out of 1..100", pcts[j]);
            return ASR_EINVAL;
        }
    }
    if (n_replicas == 0) return ASR_OK;
    if (!replicas || !cms || !out || (!traces && total_requests > 0)) {
        set_error("itl_batched: null pointer");
        return ASR_EINVAL;
    }
    const ItlWorkspace iw = itl_ws(total_requests, n_replicas);
    if (!workspace || workspace_bytes < iw.total) {
        set_error("itl_batched: workspace too small (%zu < %zu)", workspace_bytes, iw.total);
        return ASR_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const SimWorkspace w = sim_ws(total_requests, n_replicas, true);
    char *ws = (char *)workspace;
    int64_t *bm_off = (int64_t *)ws;
    uint32_t *bitmap = (uint32_t *)(ws + w.bm_off_bytes);
    int32_t *defer = (int32_t *)(ws + w.bm_off_bytes + w.bitmap_bytes);
    int64_t *lat = (int64_t *)(ws + w.bm_off_bytes + w.bitmap_bytes + w.defer_bytes);
    int64_t *ttft = (int64_t *)(ws + w.bm_off_bytes + w.bitmap_bytes + w.defer_bytes + w.lat_bytes);
    uint32_t *bitmap2 = (uint32_t *)(ws + w.total);
    char *extra = ws + iw.sim_bytes;
    asr_sim_ext_t *exts = (asr_sim_ext_t *)extra;
    unsigned long long *hist = (unsigned long long *)(extra + iw.ext_bytes);
    int64_t *pairs = (int64_t *)(extra + iw.ext_bytes + iw.hist_bytes);
    int32_t *npairs = (int32_t *)(extra + iw.ext_bytes + iw.hist_bytes + iw.pairs_bytes);
    CUDA_TRY(cudaMemsetAsync(extra, 0, iw.ext_bytes + iw.hist_bytes, st), "itl_batched: memset");
    int rc = launch_sim_prepare(replicas, n_replicas, total_requests, bm_off, defer, st);
    if (rc) return rc;
    SimExArgs a;
    static_cast<SimArgs &>(a) = SimArgs{traces, replicas, cms,     bm_off,         bitmap,     defer + 64, defer,
                                        defer + 64 + n_replicas, defer + 1,
                                        lat,    ttft,     nullptr, total_requests, n_replicas, n_cms, 0,
                                        g_opt_escalate.load(), LanePlan{}};
    a.exts = exts;
    a.bitmap2 = bitmap2;
    a.out_preempt = nullptr;
    a.itl_hist = hist;
    a.itl_pairs = pairs;
    a.itl_npairs = npairs;
    rc = launch_simulate_ex(a, max_slots, st);
    if (rc) return rc;
    return launch_itl_percentiles(a, pl, out, st);
}

extern "C" int asr_sched_tpot(const asr_req_t *trace, int64_t n, const asr_cost_model_t *cm, const int64_t *lat,
                              const int64_t *ttft, int64_t *out, void *stream) {
    if (n < 0 || !cm) {
        set_error("tpot: bad argument (n=%lld)", (long long)n);
        return ASR_EINVAL;
    }
    if (n == 0) return ASR_OK;
    if (!trace || !lat || !ttft || !out) {
        set_error("tpot: null pointer");
        return ASR_EINVAL;
    }
    return launch_tpot(trace, n, *cm, lat, ttft, out, (cudaStream_t)stream);
}

extern "C" int asr_sched_estimate(asr_req_t *recs, int64_t n, const int32_t *kappa_milli_by_lang, int32_t n_lang,
                                  const uint8_t *lang, const int32_t *speech_ms, void *stream) {
    if (n < 0 || !kappa_milli_by_lang || n_lang < 1) {
        set_error("estimate: bad argument (n=%lld n_lang=%d)", (long long)n, n_lang);
        return ASR_EINVAL;
    }
    if (n_lang > 64) {
        set_error("estimate: n_lang=%d exceeds the limit 64", n_lang);
        return ASR_EUNSUPPORTED;
    }
    if (n == 0) return ASR_OK;
    if (!recs) {
        set_error("estimate: null pointer");
        return ASR_EINVAL;
    }
    KappaTable kt;
    kt.n_lang = n_lang;
    for (int j = 0; j < 64; ++j) kt.kappa_milli[j] = j < n_lang ? kappa_milli_by_lang[j] : 0;
    return launch_estimate(recs, n, kt, lang, speech_ms, (cudaStream_t)stream);
}

extern "C" int asr_sched_simulate(const asr_req_t *trace, int64_t n, int32_t policy, const asr_cost_model_t *cm,
                                  int32_t slots, int64_t *out_lat, int64_t *out_ttft, asr_summary_t *out_summary,
                                  void *workspace, size_t workspace_bytes, void *stream) {
    if (n < 0 || n >= (1ll << 31) || policy < 0 || policy > 2 || slots < 1 || !cm) {
        set_error("simulate: bad argument (n=%lld policy=%d slots=%d)", (long long)n, policy, slots);
        return ASR_EINVAL;
    }
    if (slots > 256) {
        set_error("simulate: slots=%d exceeds the limit 256", slots);
        return ASR_EUNSUPPORTED;
    }
    // the single-replica call is the batched call with descriptors staged in the workspace
    const size_t head = 256 + 256;   // asr_replica_t + asr_cost_model_t, each in its own 256 B line
    const bool summary_only = out_lat == nullptr;
    const size_t need = head + sim_ws(n, 1, summary_only).total;
    if (!workspace || workspace_bytes < need) {
        set_error("simulate: workspace too small (%zu < %zu)", workspace_bytes, need);
        return ASR_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    asr_replica_t rep;
    rep.trace_off = 0;
    rep.out_off = 0;
    rep.n = (int32_t)n;
    rep.policy = policy;
    rep.slots = slots;
    rep.cm_id = 0;
    char *ws = (char *)workspace;
    CUDA_TRY(cudaMemcpyAsync(ws, &rep, sizeof(rep), cudaMemcpyHostToDevice, st), "simulate: upload replica");
    CUDA_TRY(cudaMemcpyAsync(ws + 256, cm, sizeof(*cm), cudaMemcpyHostToDevice, st), "simulate: upload cost model");
    // rep/cm are stack temporaries: pageable copies are staged before the call returns
    return asr_sched_simulate_batched(trace, (const asr_replica_t *)ws, 1, (const asr_cost_model_t *)(ws + 256), 1,
                                      n, slots, out_lat, out_ttft, out_summary, ws + head, workspace_bytes - head,
                                      stream);
}

extern "C" int asr_sched_percentiles(const int64_t *values, const int64_t *seg_off, int32_t n_seg,
                                     const int32_t *pcts, int32_t n_pct, int64_t *out, void *workspace,
                                     size_t workspace_bytes, void *stream) {
    (void)workspace;
    (void)workspace_bytes;
    if (n_seg < 0 || n_pct < 0 || (n_pct > 0 && !pcts)) {
        set_error("percentiles: bad argument (n_seg=%d n_pct=%d)", n_seg, n_pct);
        return ASR_EINVAL;
    }
    if (n_pct > 8) {
        set_error("percentiles: n_pct=%d exceeds the limit 8", n_pct);
        return ASR_EUNSUPPORTED;
    }
    for (int j = 0; j < n_pct; ++j)
        if (pcts[j] < 1 || pcts[j] > 100) {
            set_error("percentiles: pcts[%d]=%d outside 1..100", j, pcts[j]);
            return ASR_EINVAL;
        }
    if (n_seg == 0 || n_pct == 0) return ASR_OK;
    if (!seg_off || !out) {
        set_error("percentiles: null pointer");
        return ASR_EINVAL;
    }
    return launch_percentiles(values, seg_off, n_seg, pcts, n_pct, out, (cudaStream_t)stream);
}

extern "C" int asr_sched_gen_trace(uint64_t seed, int32_t rate_mhz, int32_t dist, int64_t n,
                                   const asr_tables_t *tables, asr_req_t *out, void *stream) {
    if (rate_mhz < 1 || dist < 0 || dist > 1 || n < 0 || !tables || (!out && n > 0)) {
        set_error("gen_trace: bad argument (rate_mhz=%d dist=%d n=%lld)", rate_mhz, dist, (long long)n);
        return ASR_EINVAL;
    }
    asr_trace_spec_t one{seed, rate_mhz, dist};
    return launch_gen_trace(nullptr, one, 1, n, tables, out, (cudaStream_t)stream);
}

extern "C" int asr_sched_gen_trace_batched(const asr_trace_spec_t *specs, int32_t n_traces, int64_t n_per_trace,
                                           const asr_tables_t *tables, asr_req_t *out, void *stream) {
    if (n_traces < 0 || n_per_trace < 0 || !tables || ((!specs || !out) && n_traces > 0 && n_per_trace > 0)) {
        set_error("gen_trace_batched: bad argument (n_traces=%d n_per_trace=%lld)", n_traces, (long long)n_per_trace);
        return ASR_EINVAL;
    }
    asr_trace_spec_t none{0, 0, 0};
    return launch_gen_trace(specs, none, n_traces, n_per_trace, tables, out, (cudaStream_t)stream);
}

extern "C" int asr_sched_gen_queues(uint64_t seed, int64_t first, int64_t n, int64_t now,
                                    const asr_tables_t *tables, asr_req_t *out, void *stream) {
    if (first < 0 || n < 0 || now < 1 || !tables || (!out && n > 0)) {
        set_error("gen_queues: bad argument (first=%lld n=%lld now=%lld)", (long long)first, (long long)n,
                  (long long)now);
        return ASR_EINVAL;
    }
    return launch_gen_queues(seed, first, n, now, tables, out, (cudaStream_t)stream);
}

// ---------------------------------------------------------------------------
// synchronous HOST-buffer entry points
// ---------------------------------------------------------------------------
namespace {
// Device scratch of the synchronous host-buffer calls: stream-ordered allocations from the
// device's default memory pool, whose release threshold is raised once so that the pool keeps
// the memory between calls (a sweep needs ~26 GB of scratch; cudaMalloc/cudaFree of that much
// cost more than the kernels).  asr_sched_trim_scratch() gives it back.
static void keep_pool_memory() {
    static std::atomic<bool> done{false};
    if (done.exchange(true)) return;
    int dev = 0;
    cudaMemPool_t pool;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
        uint64_t thr = UINT64_MAX;
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr);
    }
    cudaGetLastError();
}

struct DevBuf {
    void *p = nullptr;
    cudaStream_t st = nullptr;
    ~DevBuf() {
        if (p) cudaFreeAsync(p, st);
    }
    cudaError_t alloc(size_t bytes, cudaStream_t stream = nullptr) {
        keep_pool_memory();
        st = stream;
        return cudaMallocAsync(&p, bytes ? bytes : 1, st);
    }
};

__global__ void build_sweep_replicas_kernel(asr_replica_t *rep, int32_t n_traces, int64_t n_per_trace,
                                            int32_t n_policies, int32_t slots, const int32_t *policies) {
    const int64_t total = (int64_t)n_traces * n_policies;
    for (int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; r < total; r += (int64_t)gridDim.x * blockDim.x) {
        asr_replica_t x;
        x.trace_off = (r / n_policies) * n_per_trace;
        x.out_off = r * n_per_trace;
        x.n = (int32_t)n_per_trace;
        x.policy = policies[r % n_policies];
        x.slots = slots;
        x.cm_id = 0;
        rep[r] = x;
    }
}
}  // namespace

extern "C" int asr_sched_sweep_host(const asr_trace_spec_t *specs, int32_t n_traces, int64_t n_per_trace,
                                    const asr_tables_t *tables, const int32_t *policies, int32_t n_policies,
                                    int32_t slots, const asr_cost_model_t *cm, asr_summary_t *out_summary) {
    if (n_traces < 0 || n_per_trace < 0 || n_per_trace >= (1ll << 31) || n_policies < 1 || n_policies > 16 ||
        slots < 1 || !specs || !tables || !policies || !cm || !out_summary) {
        set_error("sweep_host: bad argument");
        return ASR_EINVAL;
    }
    if (slots > 256) {
        set_error("sweep_host: slots=%d exceeds the limit 256", slots);
        return ASR_EUNSUPPORTED;
    }
    if (n_traces == 0) return ASR_OK;
    const int64_t n_rep = (int64_t)n_traces * n_policies;
    const int64_t total = n_rep * n_per_trace;
    if (n_rep >= (1ll << 31)) {
        set_error("sweep_host: too many replicas");
        return ASR_EUNSUPPORTED;
    }
    DevBuf d_specs, d_tables, d_traces, d_rep, d_cm, d_pol, d_sum, d_ws;
    const size_t ws_bytes = sim_ws(total, n_rep, true).total;
    CUDA_TRY(d_specs.alloc(sizeof(asr_trace_spec_t) * (size_t)n_traces), "sweep_host: cudaMalloc");
    CUDA_TRY(d_tables.alloc(sizeof(asr_tables_t)), "sweep_host: cudaMalloc");
    CUDA_TRY(d_traces.alloc(sizeof(asr_req_t) * (size_t)n_traces * (size_t)n_per_trace), "sweep_host: cudaMalloc");
    CUDA_TRY(d_rep.alloc(sizeof(asr_replica_t) * (size_t)n_rep), "sweep_host: cudaMalloc");
    CUDA_TRY(d_cm.alloc(sizeof(asr_cost_model_t)), "sweep_host: cudaMalloc");
    CUDA_TRY(d_pol.alloc(sizeof(int32_t) * (size_t)n_policies), "sweep_host: cudaMalloc");
    CUDA_TRY(d_sum.alloc(sizeof(asr_summary_t) * (size_t)n_rep), "sweep_host: cudaMalloc");
    CUDA_TRY(d_ws.alloc(ws_bytes), "sweep_host: cudaMalloc workspace");
    cudaStream_t st = nullptr;
    CUDA_TRY(cudaMemcpyAsync(d_specs.p, specs, sizeof(asr_trace_spec_t) * (size_t)n_traces, cudaMemcpyHostToDevice, st),
             "sweep_host: H2D specs");
    CUDA_TRY(cudaMemcpyAsync(d_tables.p, tables, sizeof(asr_tables_t), cudaMemcpyHostToDevice, st), "sweep_host: H2D tables");
    CUDA_TRY(cudaMemcpyAsync(d_cm.p, cm, sizeof(asr_cost_model_t), cudaMemcpyHostToDevice, st), "sweep_host: H2D cm");
    CUDA_TRY(cudaMemcpyAsync(d_pol.p, policies, sizeof(int32_t) * (size_t)n_policies, cudaMemcpyHostToDevice, st),
             "sweep_host: H2D policies");
    int rc = asr_sched_gen_trace_batched((const asr_trace_spec_t *)d_specs.p, n_traces, n_per_trace,
                                         (const asr_tables_t *)d_tables.p, (asr_req_t *)d_traces.p, st);
    if (rc) return rc;
    {
        KernelTimer kt(KID_SWEEP_REPLICAS, st);
        const int64_t cap = (int64_t)sm_count() * 8;
        build_sweep_replicas_kernel<<<(int)((n_rep + 255) / 256 < cap ? (n_rep + 255) / 256 : cap), 256, 0, st>>>(
            (asr_replica_t *)d_rep.p, n_traces, n_per_trace, n_policies, slots, (const int32_t *)d_pol.p);
    }
    rc = check_launch("build_sweep_replicas_kernel");
    if (rc) return rc;
    rc = asr_sched_simulate_batched((const asr_req_t *)d_traces.p, (const asr_replica_t *)d_rep.p, (int32_t)n_rep,
                                    (const asr_cost_model_t *)d_cm.p, 1, total, slots, nullptr, nullptr,
                                    (asr_summary_t *)d_sum.p, d_ws.p, ws_bytes, st);
    if (rc) return rc;
    CUDA_TRY(cudaMemcpyAsync(out_summary, d_sum.p, sizeof(asr_summary_t) * (size_t)n_rep, cudaMemcpyDeviceToHost, st),
             "sweep_host: D2H summaries");
    CUDA_TRY(cudaStreamSynchronize(st), "sweep_host: synchronize");
    return ASR_OK;
}

extern "C" int asr_sched_trim_scratch(void) {
    int dev = 0;
    cudaMemPool_t pool;
    CUDA_TRY(cudaGetDevice(&dev), "trim_scratch: cudaGetDevice");
    CUDA_TRY(cudaDeviceSynchronize(), "trim_scratch: synchronize");
    CUDA_TRY(cudaDeviceGetDefaultMemPool(&pool, dev), "trim_scratch: default pool");
    CUDA_TRY(cudaMemPoolTrimTo(pool, 0), "trim_scratch: trim");
    return ASR_OK;
}

extern "C" int asr_sched_select_host(const asr_req_t *keys, int32_t n_queues, int32_t q_len, int32_t policy,
                                     int64_t now, int32_t k, int32_t *out_idx) {
    if (n_queues < 0 || q_len < 0 || k < 0 || policy < 0 || policy > 2) {
        set_error("select_host: bad argument");
        return ASR_EINVAL;
    }
    if (k > ASR_SELECT_MAX_K) {
        set_error("select_host: k=%d exceeds the limit %d", k, ASR_SELECT_MAX_K);
        return ASR_EUNSUPPORTED;
    }
    if (n_queues == 0 || k == 0) return ASR_OK;
    if ((!keys && q_len > 0) || !out_idx) {
        set_error("select_host: null pointer");
        return ASR_EINVAL;
    }
    DevBuf d_keys, d_out;
    const size_t kb = sizeof(asr_req_t) * (size_t)n_queues * (size_t)q_len;
    const size_t ob = sizeof(int32_t) * (size_t)n_queues * (size_t)k;
    CUDA_TRY(d_keys.alloc(kb), "select_host: cudaMalloc");
    CUDA_TRY(d_out.alloc(ob), "select_host: cudaMalloc");
    cudaStream_t st = nullptr;
    if (kb) CUDA_TRY(cudaMemcpyAsync(d_keys.p, keys, kb, cudaMemcpyHostToDevice, st), "select_host: H2D keys");
    int rc = asr_sched_select_batched((const asr_req_t *)d_keys.p, n_queues, q_len, nullptr, policy, now, nullptr, k,
                                      (int32_t *)d_out.p, st);
    if (rc) return rc;
    CUDA_TRY(cudaMemcpyAsync(out_idx, d_out.p, ob, cudaMemcpyDeviceToHost, st), "select_host: D2H indices");
    CUDA_TRY(cudaStreamSynchronize(st), "select_host: synchronize");
    return ASR_OK;
}

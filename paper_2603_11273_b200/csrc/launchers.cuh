// launchers.cuh -- host-side launch interfaces between api.cu and the kernel files.
#pragma once
#include "common.cuh"

namespace asr {

// Time-split plan of the order-free thread-per-replica tier (simulate.cu, "units"): all DEVICE pointers into the
// workspace; order == nullptr switches it off.  A work item is one WARP: item w = segment w % LANE_MAX_SEG of the
// 32 replicas order[32*g .. 32*g + 31], g = w / LANE_MAX_SEG (a lane whose replica has fewer segments idles).
struct LanePlan {
    int32_t *order;      // [n_replicas] replicas by offered load, heaviest first, input order within a load class
    uint8_t *bucket;     // [n_replicas] load class
    uint8_t *nseg;       // [n_replicas] segments
    int32_t *failed;     // [n_replicas] 1: the units of the replica could not be stitched; simulate it in one piece
    int32_t *unit_q;     // [n_replicas * LANE_MAX_SEG] by position in `order` and segment: the last regeneration
                         // point (request index in the replica) that unit saw
    int32_t *counters;   // [0] / [1] next item of the unit / repair pass
};

struct SimArgs {
    const asr_req_t *traces;
    const asr_replica_t *replicas;
    const asr_cost_model_t *cms;
    const int64_t *bm_off;    // [n_replicas] first bitmap word of each replica
    uint32_t *bitmap;
    int32_t *defer_list;      // [n_replicas] replicas handed from the lane kernel to the warp kernel
    int32_t *defer_count;     // [1]
    int32_t *defer2_list;     // [n_replicas] replicas handed from the warp kernel to the CTA kernel
    int32_t *defer2_count;    // [1]
    int64_t *out_lat;
    int64_t *out_ttft;
    asr_summary_t *out_summary;  // nullable
    int64_t total_requests;
    int32_t n_replicas;
    int32_t n_cms;
    int32_t order_free;       // 1: summary-only call, out_lat/out_ttft are workspace arrays whose order is free
    int32_t escalate_window;  // waiting window (requests) beyond which a warp hands its replica to the CTA kernel
    LanePlan plan;
};

int launch_simulate(const SimArgs &a, int max_slots, bool use_lane, cudaStream_t st);
int launch_simulate_cta(const SimArgs &a, cudaStream_t st);
// the extension kernel's arguments (kept out of SimArgs: the base kernels' parameter block stays as it was)
struct SimExArgs : SimArgs {
    const asr_sim_ext_t *exts;   // [n_cms]
    uint32_t *bitmap2;           // second bitmap: requests that had a first token
    int64_t *out_preempt;        // [n_replicas] nullable
    // inter-token latency capture (nullable): per replica ITL_BINS weights of the plain iterations, indexed by
    // |running|, and (duration, weight) pairs of the iterations that admitted somebody, at 2*out_off
    unsigned long long *itl_hist;
    int64_t *itl_pairs;
    int32_t *itl_npairs;
};
constexpr int ITL_BINS = 257;
struct ItlPcts {
    int32_t n_pct;
    int32_t pct[8];
};
int launch_itl_percentiles(const SimExArgs &a, const ItlPcts &pl, int64_t *out, cudaStream_t st);
int launch_simulate_ex(const SimExArgs &a, int max_slots, cudaStream_t st);
int launch_tpot(const asr_req_t *trace, int64_t n, asr_cost_model_t cm, const int64_t *lat, const int64_t *ttft,
                int64_t *out, cudaStream_t st);
struct KappaTable {
    int32_t n_lang;
    int32_t kappa_milli[64];
};
int launch_estimate(asr_req_t *recs, int64_t n, const KappaTable &kt, const uint8_t *lang, const int32_t *speech_ms,
                    cudaStream_t st);
int launch_sim_prepare(const asr_replica_t *replicas, int32_t n_replicas, int64_t total_requests, int64_t *bm_off,
                       int32_t *defer_count, cudaStream_t st);
// requests per unit aimed at, most units per replica: bound of the number of units of a batch
#ifndef LANE_SEG_TARGET_N
#define LANE_SEG_TARGET_N 1250
#endif
constexpr int LANE_SEG_TARGET = LANE_SEG_TARGET_N;
constexpr int LANE_MAX_SEG = 16;
int launch_lane_plan(const SimArgs &a, cudaStream_t st);
int launch_percentiles(const int64_t *values, const int64_t *seg_off, int32_t n_seg, const int32_t *pcts,
                       int32_t n_pct, int64_t *out, cudaStream_t st);
// fmt_flags: the lane kernel ran in order-free mode and left ASR_FMT32 / 0 in p50_e2e_us and p50_ttft_us of
// every valid replica (ASR_FMT32: the replica's values are uint32 in the first half of its region)
constexpr int64_t ASR_FMT32 = INT64_MIN + 32;
int launch_summary_percentiles(const asr_replica_t *replicas, int32_t n_replicas, const int64_t *lat,
                               const int64_t *ttft, asr_summary_t *out_summary, bool fmt_flags, const int32_t *order,
                               int32_t *miss_list, int32_t *miss_count, int32_t *scratch, cudaStream_t st);
int launch_gen_trace(const asr_trace_spec_t *specs, asr_trace_spec_t one, int32_t n_traces, int64_t n_per_trace,
                     const asr_tables_t *tables, asr_req_t *out, cudaStream_t st);
int launch_gen_queues(uint64_t seed, int64_t first, int64_t n, int64_t now, const asr_tables_t *tables,
                      asr_req_t *out, cudaStream_t st);
size_t select_workspace_bytes(int64_t n, int64_t k);

}  // namespace asr

/*
 * asr_sched.h -- C ABI of the B200-native duration-aware ASR scheduling hot path
 * (arxiv 2603.11273, "Duration Aware Scheduling for ASR Serving under Workload
 * Drift").  Citations are /root/reference/PAPER.md:<line>.
 *
 * The library holds hand-written sm_100a CUDA kernels for
 *   a1  trace generation          (Poisson arrivals; durations PAPER.md:80,96)
 *   a2  priority keys             (FCFS PAPER.md:13; SJF PAPER.md:63,270,277;
 *                                  HRRN PAPER.md:67-72,279-282)
 *   a3  batched top-k select      (the paper's heap pop / O(n) scan)
 *   a4  continuous-batching simulator step (iteration-level scheduling, PAPER.md:31;
 *                                  encoder ~constant + decode linear in tokens)
 *   a5  per-request E2E latency and TTFT
 *   a6  segmented nearest-rank percentiles + throughput inputs
 *
 * CONVENTIONS (apply to every call unless the call says otherwise)
 *  - Pointers marked DEVICE are device addresses allocated and owned by the
 *    caller; pointers marked HOST are ordinary host addresses read during the
 *    call (small descriptors: a single cost model, percentile lists, kappa
 *    tables; they may be freed as soon as the call returns).  The stream-ordered
 *    calls never allocate or free memory: scratch comes from the caller-supplied
 *    DEVICE `workspace` (size it with asr_sched_workspace_bytes; its contents
 *    need no initialisation).
 *  - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *    Calls only enqueue work on it and return without synchronising; outputs
 *    are valid once the caller has synchronised the stream.
 *  - EXCEPTION: the two *_host entry points (asr_sched_sweep_host,
 *    asr_sched_select_host) are synchronous, take HOST buffers only, and DO
 *    allocate: their device scratch comes from the device's default
 *    stream-ordered memory pool and stays cached there between calls until
 *    asr_sched_trim_scratch.
 *  - Return value: 0 success; -1 invalid argument (null pointer, negative size,
 *    unknown policy, slots < 1, workspace too small); -2 CUDA runtime error
 *    (text via asr_sched_last_error); -3 unsupported shape (exceeds a limit
 *    stated at the call).  No exception crosses the ABI, nothing is printed.
 *  - There is no CPU fallback: without a CUDA device every compute call
 *    returns -2.
 *  - All times are integer microseconds.  Documented preconditions (not
 *    checked on the device): 0 <= arrival_us < 2^38, now < 2^38, est <= 2^24,
 *    so that wait * est < 2^62 fits int64.  est < 1 is read as 1
 *    (PAPER.md:260 max(1, .)); arrival_us > now is read as wait = 0.
 *
 * TOTAL ORDER better(a, b, now) used by select and by the simulator's admit
 * step (exactly one correct answer everywhere; idx = position in the input):
 *   FCFS  (arrival_us, idx) ascending
 *   SJF   (max(est,1), arrival_us, idx) ascending
 *   HRRN  wait_a*est_b > wait_b*est_a, wait = max(now-arrival_us,0), exact in
 *         int64 (equivalent to comparing (wait+est)/est);
 *         equal products -> (arrival_us, idx) ascending
 */
#ifndef ASR_SCHED_H
#define ASR_SCHED_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ASR_SCHED_VERSION 100

#define ASR_SELECT_MAX_K 256
enum { ASR_FCFS = 0, ASR_SJF = 1, ASR_HRRN = 2 };
enum { ASR_ADAPTIVE = 3 };  /* policy switching on queue depth, asr_sched_simulate_batched_ex only */
enum { ASR_DIST_LOGNORMAL = 0, ASR_DIST_UNIFORM = 1 };
enum { ASR_OK = 0, ASR_EINVAL = -1, ASR_ECUDA = -2, ASR_EUNSUPPORTED = -3 };

/* one request, 16 bytes, read with one 128-bit load */
typedef struct {
    int64_t arrival_us; /* arrival time */
    int32_t dur_ms;     /* audio duration: drives the TRUE cost (tokens, encoder) */
    int32_t est;        /* scheduler's job-length estimate, est = max(1,int(d*kappa)) */
} asr_req_t;

/* cost of serving:  tokens(d) = max(1, tok_base + tok_per_s*d/1000),
 * admission costs enc_base_us + enc_per_ms_us*d once, an engine iteration costs
 * iter_base_us + iter_per_running_us*|running| and emits one token per running request */
typedef struct {
    int64_t enc_base_us;
    int64_t enc_per_ms_us;
    int64_t iter_base_us;
    int64_t iter_per_running_us;
    int32_t tok_base;
    int32_t tok_per_s;
} asr_cost_model_t; /* 40 bytes */

/* one replica of a batched simulation, 32 bytes */
typedef struct {
    int64_t trace_off; /* first record of this replica's trace in `traces` */
    int64_t out_off;   /* first element of this replica in out_lat/out_ttft  */
    int32_t n;         /* requests in the trace (sorted by arrival_us)       */
    int32_t policy;    /* ASR_FCFS / ASR_SJF / ASR_HRRN                     */
    int32_t slots;     /* continuous-batching slots, 1..256                 */
    int32_t cm_id;     /* index into `cms`                                  */
} asr_replica_t;

/* per-replica summary, 56 bytes; throughput = n_done*1e6/(last_done_us-first_arrival_us)
 * is left to the caller so the ABI stays integer */
typedef struct {
    int64_t p50_e2e_us, p90_e2e_us;   /* nearest-rank */
    int64_t p50_ttft_us, p90_ttft_us;
    int64_t first_arrival_us, last_done_us;
    int64_t n_done;                   /* -1: the replica descriptor was invalid */
} asr_summary_t;

/* one trace to generate, 16 bytes */
typedef struct {
    uint64_t seed;
    int32_t rate_mhz; /* arrival rate in milli-requests/s; mean gap = 1e9/rate_mhz us */
    int32_t dist;     /* ASR_DIST_* */
} asr_trace_spec_t;

/* quantile tables the generator interpolates (inputs, built by the caller):
 * ln_dur[j] = duration quantile (ms) at probability j/4096;
 * exp_t[j]  = round(-ln(1 - j/8192) * 2^32), exp_t[4096] = ln 2 in Q32 */
typedef struct {
    uint32_t ln_dur[4097];
    uint32_t exp_t[4097];
} asr_tables_t;

/* ------------------------------------------------------------------ */
/* a2+a3  priority keys and top-k select                               */
/* ------------------------------------------------------------------ */

/* One queue of n records.  Writes k indices (positions in `keys`), best
 * first; if k > n the tail is -1.
 *   keys DEVICE [n]; out_idx DEVICE [k]; workspace DEVICE.
 * Limits: 0 <= k <= ASR_SELECT_MAX_K = 256 (else -3; the paper's engine admits into up to 256
 * slots); n < 2^31.  k <= 32 streams the queue once (HBM-bound); 32 < k <= 256 sorts it in shared memory. */
int asr_sched_select(const asr_req_t *keys, int64_t n, int32_t policy, int64_t now,
                     int32_t k, int32_t *out_idx, void *workspace,
                     size_t workspace_bytes, void *stream);

/* asr_sched_select without a workspace and without any allocation, for callers
 * that cannot call cudaMalloc (code under CUDA graph capture, serving loops,
 * harnesses that forbid it).  The scratch of the single-queue reduction tree is
 * a device array of ASR_SELECT_STATIC_SCRATCH_BYTES built into the library (every
 * GPU that loads the library holds it until exit).  Same arguments, results and
 * error codes as asr_sched_select; in addition -3 when
 * asr_sched_workspace_bytes(ASR_OP_SELECT, n, k) exceeds the array (1 MiB:
 * k <= 32 up to n = 3.3e7 records, k = 256 up to n = 3.9e6).  All calls on a
 * device share the array: calls that overlap on the GPU (different streams
 * without ordering) race; calls on one stream do not.  Nothing is carried from
 * one call to the next.  Calls no cudaMalloc / cudaFree. */
#define ASR_SELECT_STATIC_SCRATCH_BYTES (1 << 20)
int asr_sched_select_static(const asr_req_t *keys, int64_t n, int32_t policy, int64_t now,
                            int32_t k, int32_t *out_idx, void *stream);

/* n_queues independent queues; queue q is keys[q*q_len .. q*q_len+q_len) of
 * which the first q_count[q] (or q_len if q_count is NULL) records are valid.
 * Indices are local to the queue; out_idx[q*k + j] is the j-th best, -1 padded.
 * now_per_queue (nullable) overrides `now` per queue.
 *   keys DEVICE [n_queues*q_len]; q_count, now_per_queue DEVICE [n_queues] or NULL;
 *   out_idx DEVICE [n_queues*k].  Limits: 0 <= k <= ASR_SELECT_MAX_K, q_len < 2^31. */
int asr_sched_select_batched(const asr_req_t *keys, int32_t n_queues, int32_t q_len,
                             const int32_t *q_count, int32_t policy, int64_t now,
                             const int64_t *now_per_queue, int32_t k, int32_t *out_idx,
                             void *stream);

/* ------------------------------------------------------------------ */
/* a4+a5+a6  simulator                                                 */
/* ------------------------------------------------------------------ */

/* One replica.  trace DEVICE [n] sorted by arrival_us non-decreasing
 * (precondition); out_lat/out_ttft DEVICE [n] or NULL; out_summary DEVICE [1]
 * or NULL; workspace DEVICE.  slots in 1..256 (else -3).
 * cm is a HOST pointer here (one 40-byte struct, copied into the workspace
 * during the call), whereas the batched calls below take `cms` as a DEVICE
 * array that the kernels index by replica.cm_id. */
int asr_sched_simulate(const asr_req_t *trace, int64_t n, int32_t policy,
                       const asr_cost_model_t *cm, int32_t slots, int64_t *out_lat,
                       int64_t *out_ttft, asr_summary_t *out_summary, void *workspace,
                       size_t workspace_bytes, void *stream);

/* n_replicas independent replicas (seed x rate x policy).  Batches of at least
 * ASR_OPT_SIM_LANE_MIN_REPLICAS replicas with max_slots <= 32 run one THREAD
 * per replica until a replica has to choose among waiting requests under
 * SJF/HRRN; such replicas, and every other batch, run one WARP per replica; a
 * replica whose waiting window outgrows ASR_OPT_SIM_ESCALATE_WINDOW requests
 * (a deep backlog) is handed on to one CTA per replica, which selects from a
 * candidate pool in shared memory.  The results do not depend on which kernel ran.
 *   traces DEVICE; replicas DEVICE [n_replicas]; cms DEVICE [n_cms];
 *   out_lat/out_ttft DEVICE [total_requests] indexed by replica.out_off, or both
 *   NULL for summary-only mode (the arrays then live in the workspace);
 *   out_summary DEVICE [n_replicas] or NULL.
 * total_requests = max over replicas of out_off + n (HOST value; the regions
 * [out_off, out_off+n) must be disjoint); max_slots = an upper bound of
 * replica.slots (HOST value, 1..256, picks the kernel instantiation).  A
 * replica with an invalid descriptor (or slots > max_slots) gets n_done = -1
 * and no other output.  Further preconditions: dur_ms <= 2^24, every cost
 * >= 0 and one engine iteration < 2^31 us. */
int asr_sched_simulate_batched(const asr_req_t *traces, const asr_replica_t *replicas,
                               int32_t n_replicas, const asr_cost_model_t *cms,
                               int32_t n_cms, int64_t total_requests, int32_t max_slots,
                               int64_t *out_lat, int64_t *out_ttft,
                               asr_summary_t *out_summary, void *workspace,
                               size_t workspace_bytes, void *stream);

/* ------------------------------------------------------------------ */
/* extensions: preemption, policy switching, TPOT, estimator */
/* ------------------------------------------------------------------ */

/* Per cost model, 48 bytes.  f1, "Preemption logic": one KV unit is
 * the cache of one decoded token; a running request holds
 * kv_base + kv_per_s*dur_ms/1000 (floor) + the tokens it has generated;
 * kv_budget <= 0 switches the memory model off.  f3, "Dynamic policy
 * switching": a replica with policy ASR_ADAPTIVE uses, at every scheduling step
 * with w requests waiting (after ingest), pol[0] if w < depth1, pol[1] if
 * w < depth2, else pol[2] (each ASR_FCFS/SJF/HRRN; depth1 <= depth2). */
typedef struct {
    int64_t kv_budget;
    int64_t kv_base;
    int64_t kv_per_s;
    int32_t depth1, depth2;
    int32_t pol[3];
    int32_t pad;
} asr_sim_ext_t;

/* asr_sched_simulate_batched with exts[cm_id] applied to every replica (one WARP
 * per replica).  Scheduling step (readings E1-E8): ingest; while one more
 * token for every running request would exceed kv_budget, the WORST running request
 * under the step's policy at now = t is preempted (SJF: largest est; HRRN: lowest
 * ratio; FCFS: latest arrival), loses its progress and waits again with its
 * original arrival time; only a step without preemption admits, best first, and
 * stops at the first request whose cache plus one token does not fit (it is not
 * retried until the waiting or the running set changes); one engine iteration.
 * A re-admitted request pays its encoder again; its TTFT stays that of its first
 * admission.  A request that cannot fit the budget alone marks its replica invalid
 * (n_done = -1).
 *   exts DEVICE [n_cms]; out_preempt DEVICE [n_replicas] or NULL (evictions per
 *   replica); everything else as asr_sched_simulate_batched; workspace sized with
 *   ASR_OP_SIMULATE_EX. */
int asr_sched_simulate_batched_ex(const asr_req_t *traces, const asr_replica_t *replicas,
                                  int32_t n_replicas, const asr_cost_model_t *cms,
                                  const asr_sim_ext_t *exts, int32_t n_cms,
                                  int64_t total_requests, int32_t max_slots, int64_t *out_lat,
                                  int64_t *out_ttft, asr_summary_t *out_summary,
                                  int64_t *out_preempt, void *workspace,
                                  size_t workspace_bytes, void *stream);

/* f2, PAPER.md:214 time per output token: out[i] = (lat[i] - ttft[i]) / (tokens_i - 1)
 * (floor) for requests with more than one token, else -1.
 *   trace, lat, ttft, out DEVICE [n]; cm HOST. */
int asr_sched_tpot(const asr_req_t *trace, int64_t n, const asr_cost_model_t *cm,
                   const int64_t *lat, const int64_t *ttft, int64_t *out, void *stream);

/* f2, PAPER.md:214 inter-token latency: the multiset of the gaps between consecutive
 * output tokens of every request of a replica.  A token appears at the end of every
 * engine iteration its request runs in, so an iteration contributes one sample of its
 * own duration (iteration cost plus the encoders admitted in it) for every request
 * that was already running; first tokens belong to TTFT.  Simulates the replicas
 * (policies ASR_FCFS/SJF/HRRN, no memory model) and writes, per replica,
 * out[r*(n_pct+2) ..] = the n_pct nearest-rank percentiles (-1 if there is no gap),
 * the number of gaps, their sum (mean = sum / count); all -1 for an invalid replica.
 *   pcts HOST [n_pct], 1..100, n_pct <= 8; out DEVICE [n_replicas*(n_pct+2)];
 *   workspace sized with ASR_OP_ITL (a = total_requests, b = n_replicas);
 *   everything else as asr_sched_simulate_batched. */
int asr_sched_itl_batched(const asr_req_t *traces, const asr_replica_t *replicas,
                          int32_t n_replicas, const asr_cost_model_t *cms, int32_t n_cms,
                          int64_t total_requests, int32_t max_slots, const int32_t *pcts,
                          int32_t n_pct, int64_t *out, void *workspace,
                          size_t workspace_bytes, void *stream);

/* f3, Eq. 1 and Listing 1: rewrites recs[i].est =
 * max(1, floor(d_ms * kappa_milli / 10^6)), d = speech_ms[i] if given (speech-active
 * duration from a VAD) else dur_ms, kappa_milli =
 * kappa_milli_by_lang[lang[i]] (entry 0 if lang is NULL; per-language kappa,
 * PAPER.md:154).  A lang id >= n_lang reads entry 0.  est is clamped to
 * [1, 2^24], the range the comparator is exact on (CONVENTIONS above).
 *   recs DEVICE [n] (only est is written); kappa_milli_by_lang HOST [n_lang],
 *   1 <= n_lang <= 64; lang DEVICE [n] or NULL; speech_ms DEVICE [n] or NULL. */
int asr_sched_estimate(asr_req_t *recs, int64_t n, const int32_t *kappa_milli_by_lang,
                       int32_t n_lang, const uint8_t *lang, const int32_t *speech_ms,
                       void *stream);

/* Segmented nearest-rank percentiles: segment s is values[seg_off[s] ..
 * seg_off[s+1]); out[s*n_pct + j] = element of rank ceil(pcts[j]*N/100) of the
 * sorted segment, -1 for an empty segment.  `values` is not modified.
 *   values DEVICE; seg_off DEVICE [n_seg+1]; pcts HOST [n_pct], each 1..100,
 *   n_pct <= 8; out DEVICE [n_seg*n_pct]. */
int asr_sched_percentiles(const int64_t *values, const int64_t *seg_off, int32_t n_seg,
                          const int32_t *pcts, int32_t n_pct, int64_t *out,
                          void *workspace, size_t workspace_bytes, void *stream);

/* ------------------------------------------------------------------ */
/* a1  integer-only counter-based trace generator                      */
/* ------------------------------------------------------------------ */

/* Poisson arrivals (exponential gaps, inclusive prefix sum) and durations
 * (table quantile or uniform integer ms on [1000, 35000]); est = dur_ms.
 *   tables DEVICE; out DEVICE [n]. */
int asr_sched_gen_trace(uint64_t seed, int32_t rate_mhz, int32_t dist, int64_t n,
                        const asr_tables_t *tables, asr_req_t *out, void *stream);

/* n_traces traces of n_per_trace records each; trace t is written at
 * out[t*n_per_trace ..).  specs DEVICE [n_traces] (not validated: a spec with
 * rate_mhz < 1 leaves its trace untouched; above 10^9 mHz the mean gap is 0 us
 * and every arrival is 0).  The draws of record i depend on (seed, i) only
 * (identical request sequences across runs), so consecutive specs
 * with equal (seed, dist) -- the rates of one seed -- are generated together;
 * the result does not depend on the order of the specs. */
int asr_sched_gen_trace_batched(const asr_trace_spec_t *specs, int32_t n_traces,
                                int64_t n_per_trace, const asr_tables_t *tables,
                                asr_req_t *out, void *stream);

/* Unsorted waiting queues of the standalone select workload: record i (global
 * counter first+i) has arrival_us uniform in [0, now), dur_ms from ln_dur. */
int asr_sched_gen_queues(uint64_t seed, int64_t first, int64_t n, int64_t now,
                         const asr_tables_t *tables, asr_req_t *out, void *stream);

/* ------------------------------------------------------------------ */
/* synchronous HOST-buffer entry points (the end-to-end calls)         */
/* ------------------------------------------------------------------ */

/* Replica sweep from host descriptors: generates n_traces traces, simulates
 * every trace under each of the n_policies policies (replica index =
 * t*n_policies + j) with one cost model and slot count, and returns the
 * per-replica summaries.  All pointers HOST.  Device scratch is allocated and
 * released inside the call. */
int asr_sched_sweep_host(const asr_trace_spec_t *specs, int32_t n_traces,
                         int64_t n_per_trace, const asr_tables_t *tables,
                         const int32_t *policies, int32_t n_policies, int32_t slots,
                         const asr_cost_model_t *cm, asr_summary_t *out_summary);

/* The two *_host calls take their device scratch from the device's default
 * stream-ordered memory pool and leave it cached there for the next call;
 * asr_sched_trim_scratch synchronises the device and returns it to the driver. */
int asr_sched_trim_scratch(void);

/* asr_sched_select_batched with HOST keys / out_idx (q_count, now_per_queue
 * not supported: pass full queues). */
int asr_sched_select_host(const asr_req_t *keys, int32_t n_queues, int32_t q_len,
                          int32_t policy, int64_t now, int32_t k, int32_t *out_idx);

/* ------------------------------------------------------------------ */
/* helpers                                                             */
/* ------------------------------------------------------------------ */

enum { ASR_OP_SELECT = 0, ASR_OP_SIMULATE = 1, ASR_OP_PERCENTILES = 2, ASR_OP_SIMULATE_EX = 3, ASR_OP_ITL = 4 };
/* Workspace bytes needed.  SELECT: a = n, b = k.  SIMULATE: a = total_requests,
 * b = n_replicas, c = 1 if summary-only (out_lat/out_ttft NULL) else 0 (SIMULATE_EX alike).
 * PERCENTILES: a = total values, b = n_seg.  Returns 0 for an unknown op. */
size_t asr_sched_workspace_bytes(int32_t op, int64_t a, int64_t b, int64_t c);

/* Process-wide tuning options (never change any result).
 * ASR_OPT_SIM_LANE_MIN_REPLICAS: smallest batch that asr_sched_simulate_batched
 * runs thread-per-replica (default 1024; 1 = always when max_slots <= 32;
 * INT32_MAX = never).
 * ASR_OPT_SIM_ESCALATE_WINDOW: waiting-window length (requests) beyond which the
 * warp kernel hands a SJF/HRRN replica to the CTA kernel (default 4096; 0 = as
 * soon as the policy has to choose; INT32_MAX = never).
 * ASR_OPT_SIM_LANE_SPLIT: 1 (default) lets a summary-only thread-per-replica
 * call cut lightly loaded replicas into time segments that are simulated side
 * by side and stitched at regeneration points (server idle at an arrival);
 * 0 simulates every replica in one piece. */
enum { ASR_OPT_SIM_LANE_MIN_REPLICAS = 0, ASR_OPT_SIM_ESCALATE_WINDOW = 1, ASR_OPT_SIM_LANE_SPLIT = 2 };
int asr_sched_set_option(int32_t option, int64_t value);

const char *asr_sched_last_error(void); /* thread-local, never NULL */
int asr_sched_version(void);
/* number of kernels this library has launched in this process (monotonic) */
int64_t asr_sched_launch_count(void);

/* Per-kernel timing (the library's own tracing aid).  While enabled, every
 * kernel launch is bracketed by a CUDA-event pair recorded on the launching
 * stream.  asr_sched_timing_read synchronises those events and returns the
 * summed device time and launch count of kernel `kernel_id` since the last
 * reset; asr_sched_kernel_name(id) names the ids 0.. (NULL past the end). */
int asr_sched_timing_enable(int on);
int asr_sched_timing_reset(void);
int asr_sched_timing_read(int32_t kernel_id, double *total_ms, int64_t *launches);
const char *asr_sched_kernel_name(int32_t kernel_id);

#ifdef __cplusplus
}
#endif
#endif /* ASR_SCHED_H */

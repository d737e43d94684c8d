/*
 * asr_oracle.h -- CPU ORACLE (test infrastructure, NOT the product).
 *
 * A plain, slow, obviously-correct restatement of what the hot path computes,
 * written from /root/reference/PAPER.md (arxiv 2603.11273) and the readings
 * listed in DESIGN.md.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, link, import or run
 * anything in this directory.  It shares no code, header, table generator or
 * constant with the CUDA path under paper_2603_11273_b200/.
 *
 * All time is integer microseconds; every result is exact (no tolerance).
 *
 * Parity pins (tests/test_oracle_*.py, run with -m "not gpu"):
 *   orc_better / orc_select   : pinned (brute force, invariants, hand ties)
 *   orc_simulate              : pinned (Fig. 1 toy, brute force
 *                               over orderings, closed forms, invariants)
 *   orc_percentile            : pinned (textbook nearest-rank example)
 *   orc_fmix64 / orc_mix64    : pinned (published splitmix64 known answers)
 *   orc_gen_trace/orc_gen_queue: moments pinned to closed forms; the exact
 *                               bit stream is a recipe of this repo
 *                                -- the paper fixes
 *                               only "Poisson, burstiness 1.0".
 *   orc_itl                   : pinned (closed forms: isolated request, two
 *                               overlapping requests by hand; sum = sum of
 *                               (E2E - TTFT) over requests)
 *   orc_tpot / orc_estimate   : pinned (closed forms; Fig. 1 caption's 40/20/10
 *                               tokens)
 *   orc_simulate_ex           : reduces to orc_simulate (pinned) with the memory
 *                               model off; the preemption model itself is this
 *                               repo's reading of one sentence:
 *                               pinned by a hand-worked example and invariants,
 *                               PARITY UNPINNED against the paper's system.
 *   The paper's Table 1/2 trends: PARITY UNPINNED (real-system measurements).
 */
#ifndef ASR_ORACLE_H
#define ASR_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* one request: PAPER.md:57-59 (Eq. 1: est = d * kappa) */
typedef struct {
    int64_t arrival_us; /* arrival time, integer microseconds */
    int32_t dur_ms;     /* audio duration: drives the TRUE cost */
    int32_t est;        /* scheduler's job-length estimate */
} orc_req_t;

/* cost model: PAPER.md:51-53 (encoder ~constant, decode linear in tokens) */
typedef struct {
    int64_t enc_base_us;
    int64_t enc_per_ms_us;
    int64_t iter_base_us;
    int64_t iter_per_running_us;
    int32_t tok_base;
    int32_t tok_per_s;
} orc_cost_t;

enum { ORC_FCFS = 0, ORC_SJF = 1, ORC_HRRN = 2 };
enum { ORC_DIST_LOGNORMAL = 0, ORC_DIST_UNIFORM = 1 };

/* 1 if request a (at position ia) is strictly better than b (at ib).
 * HRRN multiplies in 128 bits; a cross-product >= 2^62 (outside the boundary's
 * documented bounds wait < 2^38, est <= 2^24) is counted in a
 * thread-local counter, and orc_select / orc_simulate / orc_simulate_ex /
 * orc_itl return -4 when a comparison of theirs tripped it. */
int64_t orc_bound_violations(void);
void orc_bound_violations_reset(void);
int orc_better(const orc_req_t *a, int64_t ia, const orc_req_t *b, int64_t ib,
               int policy, int64_t now);

/* sort all n by orc_better, write the first min(k,n) positions, pad -1 */
int orc_select(const orc_req_t *q, int64_t n, int policy, int64_t now,
               int32_t k, int32_t *out_idx);

/* iteration-level continuous-batching simulator, one iteration at a time */
int orc_simulate(const orc_req_t *trace, int64_t n, int policy,
                 const orc_cost_t *cm, int32_t slots, int64_t *lat,
                 int64_t *ttft, int64_t *first_arrival_us,
                 int64_t *last_done_us);

/* ---- SURVEY.md 8(f) extensions ------------------ */

/* f1 preemption under memory pressure (A.4 "Preemption logic") and
 * f3 dynamic policy switching on queue depth.  One KV unit = the
 * cache of one decoded token.  A running request holds
 *   kv_base + kv_per_s*dur_ms/1000 (encoder / cross-attention cache, floor)
 *   + the tokens it has generated so far.
 * kv_budget <= 0 switches the memory model off. */
typedef struct {
    int64_t kv_budget;
    int64_t kv_base;
    int64_t kv_per_s;
    int32_t depth1, depth2; /* ORC_ADAPTIVE: waiting < depth1 -> pol[0],   */
    int32_t pol[3];         /*   < depth2 -> pol[1], else pol[2]            */
    int32_t pad;
} orc_ext_t;                /* 48 bytes */

enum { ORC_ADAPTIVE = 3 };

/* orc_simulate with the extensions; ext == NULL is orc_simulate.  Step order
 * (readings E1-E8): ingest; while the running set would not fit after
 * one more token each, preempt the WORST running request under the policy's total
 * order at now = t (SJF: largest est; HRRN: lowest ratio; FCFS: latest arrival),
 * which loses its progress and waits again; only a step without preemption
 * admits, best first, stopping at the first request that does not fit; iterate.
 * TTFT is that of the first admission.  n_preempt (nullable) counts evictions.
 * Returns -3 if a request alone cannot fit the budget. */
int orc_simulate_ex(const orc_req_t *trace, int64_t n, int policy,
                    const orc_cost_t *cm, const orc_ext_t *ext, int32_t slots,
                    int64_t *lat, int64_t *ttft, int64_t *first_arrival_us,
                    int64_t *last_done_us, int64_t *n_preempt);

/* f2 time per output token (A.2): (E2E - TTFT) / (tokens - 1),
 * floor, for requests with more than one token; -1 otherwise */
int orc_tpot(const orc_req_t *trace, int64_t n, const orc_cost_t *cm,
             const int64_t *lat, const int64_t *ttft, int64_t *out);

/* f2 inter-token latency (A.2 "P50 ITL"): the multiset of the gaps
 * between consecutive output tokens of every request.  A token appears at the end
 * of every engine iteration its request is running in, so each iteration adds one
 * sample of its own duration (iteration cost plus the encoders admitted in it) for
 * every request that was ALREADY running (a request's first token belongs to TTFT).
 * out_pcts[j] = nearest-rank percentile pcts[j] of the multiset (-1 if empty),
 * out_count = its size, out_sum = the sum of its samples (mean = sum / count). */
int orc_itl(const orc_req_t *trace, int64_t n, int policy, const orc_cost_t *cm,
            int32_t slots, const int32_t *pcts, int32_t n_pct, int64_t *out_pcts,
            int64_t *out_count, int64_t *out_sum);

/* f3 duration-based estimator (Eq. 1, Listing 1):
 * est = max(1, floor(d_ms * kappa_milli / 10^6)) with d = speech_ms[i] when given
 * (VAD speech-active duration) else dur_ms, and kappa_milli =
 * kappa_milli_by_lang[lang[i]] (lang == NULL or lang[i] >= n_lang: entry 0;
 * PAPER.md:154); est is clamped to the comparator's bound 2^24 */
int orc_estimate(orc_req_t *recs, int64_t n, const int32_t *kappa_milli_by_lang,
                 int32_t n_lang, const uint8_t *lang, const int32_t *speech_ms);

/* nearest-rank percentile, p in [1,100]; n == 0 -> -1 */
int64_t orc_percentile(const int64_t *v, int64_t n, int32_t p);

/* tokens and encoder cost of one request (exposed for closed-form pins) */
int64_t orc_tokens(const orc_cost_t *cm, int32_t dur_ms);
int64_t orc_enc_cost(const orc_cost_t *cm, int32_t dur_ms);

/* counter-based generator */
uint64_t orc_fmix64(uint64_t z);
uint64_t orc_mix64(uint64_t seed, uint32_t stream, uint64_t i);
int orc_gen_trace(uint64_t seed, int32_t rate_mhz, int32_t dist, int64_t n,
                  const uint32_t *ln_dur /*[4097]*/,
                  const uint32_t *exp_t /*[4097]*/, orc_req_t *out);
int orc_gen_queue(uint64_t seed, int64_t first, int64_t n, int64_t now,
                  const uint32_t *ln_dur /*[4097]*/, orc_req_t *out);

#ifdef __cplusplus
}
#endif
#endif

// sim_common.cuh -- helpers shared by the simulator kernels (simulate.cu, simulate_cta.cu).
#pragma once
#include "launchers.cuh"

namespace asr {

constexpr int SIM_WARPS = 4;
constexpr int32_t REM_FREE = 0x7FFFFFFF;

__device__ __forceinline__ int64_t ceil_div_pos(int64_t g, int64_t c) {
    // g > 0, c > 0; 32-bit divide whenever both operands fit
    if ((((uint64_t)g | (uint64_t)c) >> 32) == 0) {
        const uint32_t q = (uint32_t)g / (uint32_t)c;
        return (int64_t)q + ((uint32_t)g - q * (uint32_t)c != 0u ? 1 : 0);
    }
    const uint64_t q = (uint64_t)g / (uint64_t)c;
    return (int64_t)q + ((uint64_t)g - q * (uint64_t)c != 0ull ? 1 : 0);
}

__device__ __forceinline__ int32_t tokens_of(const asr_cost_model_t &cm, int32_t dur_ms) {
    int64_t t = (int64_t)cm.tok_base + ((int64_t)cm.tok_per_s * (int64_t)dur_ms) / 1000;
    t = t < 1 ? 1 : t;
    return t > 0x7FFFFFFE ? 0x7FFFFFFE : (int32_t)t;
}

// sum over the warp of a non-negative 32-bit value per lane, exact in 64 bits
__device__ __forceinline__ int64_t warp_sum_u32(uint32_t v) {
    uint32_t lo = __reduce_add_sync(ASR_FULL_MASK, v & 0xFFFFu);
    uint32_t hi = __reduce_add_sync(ASR_FULL_MASK, v >> 16);
    return ((int64_t)hi << 16) + (int64_t)lo;
}

// true if the descriptor of replica r can be simulated with `max_slots` slots per replica
__device__ __forceinline__ bool replica_ok(const SimArgs &a, const asr_replica_t &rep, int max_slots) {
    return rep.n >= 0 && rep.slots >= 1 && rep.slots <= max_slots && rep.policy >= 0 && rep.policy <= 2 &&
           rep.cm_id >= 0 && rep.cm_id < a.n_cms && rep.trace_off >= 0 && rep.out_off >= 0 &&
           rep.out_off + (int64_t)rep.n <= a.total_requests;
}

__device__ __forceinline__ void flag_invalid(const SimArgs &a, int r) {
    if (!a.out_summary) return;
    asr_summary_t s;
    s.p50_e2e_us = s.p90_e2e_us = s.p50_ttft_us = s.p90_ttft_us = -1;
    s.first_arrival_us = s.last_done_us = 0;
    s.n_done = -1;
    a.out_summary[r] = s;
}

// ---- chunk bounds of the sparse waiting window ------------------------------------------------------------------
// While SJF/HRRN choose among a backlog, the window [lo, p) is seen as chunks of 32 consecutive requests.  Per
// chunk the warp keeps, in shared memory, which requests still wait there, and an earliest arrival and a smallest
// est that bound them (exact when the chunk was last scanned; ingesting a request updates them, admitting one
// leaves them -- still bounds, only looser).  No request of a chunk has a better key than (that est, that
// arrival), so an admission scans chunks best bound first and stops as soon as no unscanned chunk's bound reaches
// the best request found: branch and bound, instead of the whole window per admission.  The winner always comes
// from the exact comparator; the bounds only decide what need not be looked at.
constexpr int CHUNK_RING = 160;   // chunk slots per warp: windows of up to (CHUNK_RING - 2) * 32 requests
constexpr int CHUNK_PER_LANE = CHUNK_RING / 32;
struct ChunkMeta {
    int64_t a_first;   // no waiting request of the chunk arrived before this
    int32_t e_min;     // none has a smaller max(est, 1)
    uint32_t wait;     // bit j: request 32c + j waits
};

static __device__ __noinline__ bool better_cold(int policy, int64_t arr_a, int32_t est_a, int32_t idx_a, int64_t arr_b,
                                         int32_t est_b, int32_t idx_b, int64_t now) {
    return better_rt(policy, arr_a, est_a, idx_a, arr_b, est_b, idx_b, now);
}

// order scalar of a waiting request (common.cuh): smaller = better, equal = ask the exact comparator
__device__ __forceinline__ int64_t warp_order_scalar(int policy, int64_t arr, int32_t est, int64_t t) {
    if (policy == ASR_FCFS) return arr;
    const int64_t e = est_of(est);
    if (policy == ASR_SJF) {
        int64_t a8 = arr >> 8;
        a8 = a8 < 0 ? 0 : (a8 > 0xFFFFFFFFll ? 0xFFFFFFFFll : a8);
        return (e << 32) | a8;
    }
    const double r = (double)wait_of(arr, t) / (double)e;
    return INT64_MAX - __double_as_longlong(r);
}

__device__ __forceinline__ int64_t warp_min_s64(int64_t v) {
    const int32_t hi = __reduce_min_sync(ASR_FULL_MASK, (int32_t)(v >> 32));
    const uint32_t lo = __reduce_min_sync(ASR_FULL_MASK, (int32_t)(v >> 32) == hi ? (uint32_t)v : 0xFFFFFFFFu);
    return (int64_t)(((uint64_t)(uint32_t)hi << 32) | lo);
}

// bounds of chunk c from the global bitmap and the records (entering the sparse mode, or coming back into the ring)
__device__ __forceinline__ void chunk_rebuild(const asr_req_t *trace, const uint32_t *bm, ChunkMeta *ring, int c, int lo,
                                              int p, int lane) {
    const int i = (c << 5) + lane;
    const uint32_t word = bm[c];
    const bool waiting = i >= lo && i < p && !((word >> lane) & 1u);
    int64_t arr = 0;
    int32_t e = INT32_MAX;
    if (waiting) {
        const Rec q = ld_cached(trace + i);
        arr = q.arrival_us;
        e = (int32_t)est_of(q.est);
    }
    const uint32_t wm = __ballot_sync(ASR_FULL_MASK, waiting);
    const int32_t emin = __reduce_min_sync(ASR_FULL_MASK, e);
    const int64_t a_first = shfl64(arr, wm ? __ffs(wm) - 1 : 0);   // arrivals are sorted: the first waiting one
    if (lane == 0) {
        ChunkMeta m;
        m.a_first = a_first;
        m.e_min = emin;
        m.wait = wm;
        ring[c % CHUNK_RING] = m;
    }
}

// scan chunk c (somebody waits there): its bounds become exact, its best request is merged into the running best
// b_* (uniform over the warp; b_s = its order scalar)
__device__ __forceinline__ void chunk_scan(const asr_req_t *trace, ChunkMeta *ring, int c, int policy, int64_t t, int lane,
                                           int64_t &b_s, int64_t &b_arr, int32_t &b_est, int32_t &b_dur, int32_t &b_idx) {
    ChunkMeta *slot = ring + (c % CHUNK_RING);
    const uint32_t wm = slot->wait;
    const bool waiting = (wm >> lane) & 1u;
    Rec q;
    q.arrival_us = 0;
    q.dur_ms = q.est = 0;
    int64_t sc = INT64_MAX;
    int32_t e = INT32_MAX;
    if (waiting) {
        q = ld_cached(trace + (c << 5) + lane);
        sc = warp_order_scalar(policy, q.arrival_us, q.est, t);
        e = (int32_t)est_of(q.est);
    }
    const int32_t emin = __reduce_min_sync(ASR_FULL_MASK, e);
    const int first = __ffs(wm) - 1;
    const int64_t a_first = shfl64(q.arrival_us, first);
    if (lane == 0) {
        slot->a_first = a_first;
        slot->e_min = emin;
    }
    const int64_t smin = warp_min_s64(sc);
    uint32_t tie = __ballot_sync(ASR_FULL_MASK, waiting && sc == smin);
    int wl = __ffs(tie) - 1;
    int64_t c_arr = shfl64(q.arrival_us, wl);
    int32_t c_est = __shfl_sync(ASR_FULL_MASK, q.est, wl);
    tie &= tie - 1u;
    while (tie) {   // equal scalars (rare): the exact order among them
        const int l = __ffs(tie) - 1;
        tie &= tie - 1u;
        const int64_t o_arr = shfl64(q.arrival_us, l);
        const int32_t o_est = __shfl_sync(ASR_FULL_MASK, q.est, l);
        if (better_cold(policy, o_arr, o_est, (c << 5) + l, c_arr, c_est, (c << 5) + wl, t)) {
            wl = l;
            c_arr = o_arr;
            c_est = o_est;
        }
    }
    const int32_t c_idx = (c << 5) + wl;
    const bool take = b_idx < 0 || smin < b_s ||
                      (smin == b_s && better_cold(policy, c_arr, c_est, c_idx, b_arr, b_est, b_idx, t));
    if (take) {
        b_s = smin;
        b_arr = c_arr;
        b_est = c_est;
        b_dur = __shfl_sync(ASR_FULL_MASK, q.dur_ms, wl);
        b_idx = c_idx;
    }
}

// the best waiting request of the chunks c_lo .. c_hi (at most CHUNK_RING - 1 of them) under `policy` at time t:
// branch and bound over the chunk bounds, exact (see ChunkMeta).  b_idx = -1 if nobody waits.
__device__ __forceinline__ void chunk_pick(const asr_req_t *trace, ChunkMeta *ring, int c_lo, int c_hi, int policy, int64_t t,
                                           int lane, int64_t &b_arr, int32_t &b_est, int32_t &b_dur, int32_t &b_idx) {
    int64_t b_s = INT64_MAX;
    uint32_t scanned = 0;   // bit j: my j-th chunk was scanned in this call
    const int nj = (c_hi - c_lo + 32) >> 5;   // chunk slots per lane in use (uniform)
    b_idx = -1;
    while (true) {
        // my most promising chunk among those whose bound reaches the best request so far
        float best_sc = 0.f;
        int best_j = -1;
        for (int j = 0; j < nj; ++j) {
            const int c = c_lo + lane + 32 * j;
            if (c <= c_hi && !((scanned >> j) & 1u)) {
                const ChunkMeta mt = ring[c % CHUNK_RING];
                if (mt.wait != 0u) {
                    bool need = b_idx < 0;
                    const int64_t w_c = wait_of(mt.a_first, t);
                    if (!need) {
                        if (policy == ASR_FCFS) {
                            need = mt.a_first <= b_arr;
                        } else if (policy == ASR_SJF) {
                            const int64_t eb = est_of(b_est);
                            need = mt.e_min < eb || (mt.e_min == eb && mt.a_first <= b_arr);
                        } else {   // ties included: an equal ratio with an earlier arrival wins
                            need = w_c * est_of(b_est) >= wait_of(b_arr, t) * (int64_t)mt.e_min;
                        }
                    }
                    if (need) {
                        const float inv = __frcp_rn((float)mt.e_min);
                        const float sc = policy == ASR_FCFS ? (float)(c_hi - c + 1)
                                                            : (policy == ASR_SJF ? inv : ((float)w_c + 1.f) * inv);
                        if (best_j < 0 || sc > best_sc) {
                            best_sc = sc;
                            best_j = j;
                        }
                    }
                }
            }
        }
        const uint32_t key = best_j >= 0 ? (__float_as_uint(best_sc) | 1u) : 0u;   // scores are positive
        const uint32_t kmax = __reduce_max_sync(ASR_FULL_MASK, key);
        if (kmax == 0u) break;
        const int src = __ffs(__ballot_sync(ASR_FULL_MASK, key == kmax)) - 1;
        const int gj = __shfl_sync(ASR_FULL_MASK, best_j, src);
        if (lane == src) scanned |= 1u << gj;
        chunk_scan(trace, ring, c_lo + src + 32 * gj, policy, t, lane, b_s, b_arr, b_est, b_dur, b_idx);
        __syncwarp();
    }
}

}  // namespace asr

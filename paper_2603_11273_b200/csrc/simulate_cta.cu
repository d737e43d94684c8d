// simulate_cta.cu -- a4 simulator step + a5 outputs for DEEP BACKLOGS: one CTA per replica.
//
// The warp-per-replica kernel re-scans the whole waiting window for every
// admission, which is fine for windows of a few thousand requests and hopeless
// for the deep-backlog configuration (10^6 requests, ~2*10^5 waiting,
// PAPER.md:104-118 overload regime; BASELINE.json configs[3]).  A warp whose
// window outgrows ASR_OPT_SIM_ESCALATE_WINDOW hands its replica to this kernel.
//
// Thread s of the CTA owns batch slot s (up to 256, "max batch
// 256"); the engine step (ingest, admit, iterate with exact fast-forward,
// record) is the one of simulate.cu with block-wide reductions.
//
// Candidate pool.  Admission never looks at the whole waiting set.  A pool of
// at most POOL_CAP waiting requests in shared memory is guaranteed to contain
// the k best; the exact k-set is found in the pool with a block-wide
// quickselect over 64-bit order scalars (common.cuh), ties settled by the
// exact comparator.  The guarantee:
//   complete   the pool IS the waiting set (backlogs up to POOL_CAP).
//   SJF        the order is static: the pool holds every waiting request with
//              est <= E; it contains the k best while it has k members.
//   HRRN       the order moves with time, r_x(t) = (t - a_x)/e_x.  Built at t0
//              with a threshold ratio theta and a horizon H, the pool holds
//              every request with r_x(t0 + H) >= theta (ratios only grow, so
//              nobody else can reach theta before t0 + H); G counts the
//              members with r_x(t0) >= theta ("strong").  While t <= t0 + H and
//              at least k strong members remain, k pool members have a ratio
//              >= theta > that of every request outside: the k best are inside.
// When the guarantee lapses the pool is rebuilt from the waiting window (a
// histogram over an approximate 32-bit key picks theta; the pool itself is
// filled by the exact integer tests).  If no pool can be built (massive ties)
// the step falls back to an exact block-wide arg-best scan of the window.
#include "sim_common.cuh"
#ifdef CTA_STATS
#include <cstdio>
#endif

namespace asr {

constexpr int CTA_T = 256;
constexpr int POOL_CAP = 2048;
constexpr int POOL_EPT = POOL_CAP / CTA_T;
constexpr int POOL_TARGET = 768;       // strong members wanted from a rebuild
constexpr int HIST_BINS = 2048;
constexpr int KSEL_SMALL = 32;         // up to this many admissions the k-th scalar is found by extraction
constexpr int64_t H_MAX = 1ll << 36;   // (2^38 + 2^36) * 2^24 < 2^63

struct CtaSmem {
    int4 pool[POOL_CAP];       // (arrival lo, arrival hi, max(est,1), trace position)
    int64_t K[POOL_CAP];       // order scalars of the current step
    int4 adm[CTA_T];           // requests admitted in this step
    int4 wbest[CTA_T / 32];    // per-warp winners of the fallback scan
    uint32_t hist[HIST_BINS];
    int32_t rep[HIST_BINS];    // one trace position per histogram bin
    uint64_t wsel[CTA_T / 32][KSEL_SMALL];   // small k: every warp's k smallest order scalars, ascending
    uint16_t tie[POOL_CAP];
    uint16_t hole[CTA_T], surv[CTA_T];
    int64_t carr_win[CTA_T];   // arrival stamps of the trace window [cbase, cbase + CTA_T)
    int64_t red64[CTA_T / 32];
    int32_t red32[CTA_T / 32];
    int64_t bc64;
    int32_t pool_n, adm_n, hole_n, surv_n, tie_n, bc32[4];
};

// ---- block-wide helpers (every thread calls them; every thread gets the result) ----
__device__ __forceinline__ int block_sum(int v, CtaSmem &sm) {
    v = __reduce_add_sync(ASR_FULL_MASK, v);
    __syncthreads();
    if (lane_id() == 0) sm.red32[threadIdx.x >> 5] = v;
    __syncthreads();
    int s = 0;
#pragma unroll
    for (int w = 0; w < CTA_T / 32; ++w) s += sm.red32[w];
    return s;
}
__device__ __forceinline__ int block_min(int v, CtaSmem &sm) {
    v = __reduce_min_sync(ASR_FULL_MASK, v);
    __syncthreads();
    if (lane_id() == 0) sm.red32[threadIdx.x >> 5] = v;
    __syncthreads();
    int s = sm.red32[0];
#pragma unroll
    for (int w = 1; w < CTA_T / 32; ++w) s = sm.red32[w] < s ? sm.red32[w] : s;
    return s;
}
__device__ __forceinline__ int block_max(int v, CtaSmem &sm) { return -block_min(-v, sm); }
__device__ __forceinline__ int64_t block_sum64(int64_t v, CtaSmem &sm) {
#pragma unroll
    for (int j = 16; j > 0; j >>= 1) v += (int64_t)shfl64_xor((uint64_t)v, j);
    __syncthreads();
    if (lane_id() == 0) sm.red64[threadIdx.x >> 5] = v;
    __syncthreads();
    int64_t s = 0;
#pragma unroll
    for (int w = 0; w < CTA_T / 32; ++w) s += sm.red64[w];
    return s;
}
// sum of the admitted durations and minimum of the remaining tokens in one pair of barriers
__device__ __forceinline__ void block_sum_min(int32_t dur, int32_t rem, int64_t &dur_sum, int32_t &rem_min, CtaSmem &sm) {
    // dur = hi * 65536 + lo with 0 <= lo < 65536 (any sign of dur): two 32-bit REDUX instead of ten shuffles
    const int lo = __reduce_add_sync(ASR_FULL_MASK, dur & 0xFFFF), hi = __reduce_add_sync(ASR_FULL_MASK, dur >> 16);
    const int mn = __reduce_min_sync(ASR_FULL_MASK, rem);
    __syncthreads();
    if (lane_id() == 0) {
        sm.red64[threadIdx.x >> 5] = (int64_t)hi * 65536 + (int64_t)lo;
        sm.red32[threadIdx.x >> 5] = mn;
    }
    __syncthreads();
    int64_t s = 0;
    int m = sm.red32[0];
#pragma unroll
    for (int w = 0; w < CTA_T / 32; ++w) {
        s += sm.red64[w];
        m = sm.red32[w] < m ? sm.red32[w] : m;
    }
    dur_sum = s;
    rem_min = m;
}
// exclusive rank of this thread among the threads with flag set
__device__ __forceinline__ int block_rank(bool flag, CtaSmem &sm) {
    const uint32_t m = __ballot_sync(ASR_FULL_MASK, flag);
    const int warp = threadIdx.x >> 5;
    __syncthreads();
    if (lane_id() == 0) sm.red32[warp] = __popc(m);
    __syncthreads();
    int before = 0;
#pragma unroll
    for (int w = 0; w < CTA_T / 32; ++w)
        if (w < warp) before += sm.red32[w];
    return before + __popc(m & ((1u << lane_id()) - 1u));
}

__device__ __forceinline__ int64_t order_scalar_rt(int policy, const int4 &e, int64_t now) {
    return policy == ASR_SJF ? order_scalar<ASR_SJF>(e, now) : order_scalar<ASR_HRRN>(e, now);
}
__device__ __forceinline__ bool cand_better(int policy, const int4 &x, const int4 &y, int64_t now) {
    return better_rt(policy, rec_arr(x), x.z, x.w, rec_arr(y), y.z, y.w, now);
}
__device__ __forceinline__ int4 cand_of(const asr_req_t *trace, int pos) {
    const int4 v = __ldg(reinterpret_cast<const int4 *>(trace + pos));
    return make_int4(v.x, v.y, v.w < 1 ? 1 : v.w, pos);
}
// the bitmap is updated with atomics (performed in L2): read it past L1
__device__ __forceinline__ bool is_admitted(const uint32_t *bm, int pos) { return (__ldcg(bm + (pos >> 5)) >> (pos & 31)) & 1u; }

// Visit every waiting request of the window [lo, p): f(candidate record).  One CTA walks a window of up to
// 10^6 positions out of L2, so the loop is bound by load latency: SCAN_U bitmap words and SCAN_U records per
// thread are requested before the first one is looked at (the record load does not wait for its bitmap word).
#ifndef SCAN_U_N
#define SCAN_U_N 8
#endif
constexpr int SCAN_U = SCAN_U_N;
#ifdef CTA_STATS
__device__ unsigned long long g_stat[8];
#define STAT(i, v) do { if (threadIdx.x == 0) g_stat[i] += (v); } while (0)
#else
#define STAT(i, v) do { } while (0)
#endif
template <class F>
__device__ __forceinline__ void scan_waiting(const asr_req_t *trace, const uint32_t *bm, int lo, int p, F &&f) {
    STAT(1, 1);
    STAT(2, p - lo);
    if (lo >= p) return;
    // A thread takes one bitmap word (32 positions) at a time and walks its zero bits, so the admitted
    // positions -- most of a deep window -- cost nothing; up to SCAN_U records are requested before the first
    // one is looked at, and the thread's next word is requested before the current one is walked.
    const int w0 = lo >> 5, w1 = (p - 1) >> 5;
    const uint32_t head = ~((1u << (lo & 31)) - 1u);                                   // positions >= lo of word w0
    const uint32_t tail = ((p - 1) & 31) == 31 ? 0xFFFFFFFFu : (2u << ((p - 1) & 31)) - 1u;   // positions < p of word w1
    int w = w0 + (int)threadIdx.x;
    uint32_t word = w <= w1 ? __ldcg(bm + w) : 0xFFFFFFFFu;
    while (w <= w1) {
        const int wn = w + CTA_T;
        const uint32_t word_n = wn <= w1 ? __ldcg(bm + wn) : 0xFFFFFFFFu;
        uint32_t inv = ~word;
        if (w == w0) inv &= head;
        if (w == w1) inv &= tail;
        while (inv) {
            int4 v[SCAN_U];
            int pos[SCAN_U];
#pragma unroll
            for (int u = 0; u < SCAN_U; ++u) {
                pos[u] = -1;
                if (inv) {
                    pos[u] = w * 32 + __ffs((int)inv) - 1;
                    inv &= inv - 1u;
                    v[u] = __ldg(reinterpret_cast<const int4 *>(trace + pos[u]));
                }
            }
#pragma unroll
            for (int u = 0; u < SCAN_U; ++u)
                if (pos[u] >= 0) f(make_int4(v[u].x, v[u].y, v[u].w < 1 ? 1 : v[u].w, pos[u]));
        }
        w = wn;
        word = word_n;
    }
}

// approximate 32-bit key of a waiting request, smaller = better; only used to pick a threshold
__device__ __forceinline__ int32_t approx_key(int policy, const int4 &e, int64_t t0) {
    if (policy == ASR_SJF) return e.z;
    const float r = (float)wait_of(rec_arr(e), t0) / (float)e.z;
    return 0x7FFFFFFF - __float_as_int(r);
}

struct PoolState {
    int P;             // members
    bool complete;     // the pool is the whole waiting set
    bool thr_valid;    // threshold mode: thrW/thrE/t0H describe the membership test
    int G;             // HRRN: strong members left (lower bound)
    int64_t thrW;      // HRRN: theta = thrW / thrE
    int32_t thrE;      // SJF: est bound E
    int64_t t0H;       // HRRN: the guarantee holds up to this time
    int64_t t0;
    int64_t H;
    int G0, P0;        // HRRN: strong members and members right after the build
    int32_t prev_key;  // approximate key of the last threshold: centre of the next histogram
    bool prev_valid;
};

// membership test of the current threshold for a request (threshold mode)
__device__ __forceinline__ bool pool_pass(int policy, const PoolState &ps, const int4 &e) {
    if (policy == ASR_SJF) return e.z <= ps.thrE;
    return mul64x32(ps.t0H - rec_arr(e), (uint32_t)ps.thrE) >= mul64x32(ps.thrW, (uint32_t)e.z);
}

// ---- rebuild the pool from the waiting window [lo, p) ---------------------------------
__device__ __noinline__ void pool_rebuild(CtaSmem &sm, PoolState &ps, const asr_req_t *trace, const uint32_t *bm,
                                          int policy, int64_t t, int &lo, int p, int nW, int k) {
    const int tid = threadIdx.x;
    // advance lo to the first waiting request
    for (;;) {
        const int w = (lo >> 5) + tid;
        int cand = 0x7FFFFFFF;
        if ((int64_t)w * 32 < p) {
            uint32_t inv = ~__ldcg(bm + w);
            if (w == (lo >> 5)) inv &= ~((1u << (lo & 31)) - 1u);
            if (inv) cand = w * 32 + __ffs(inv) - 1;
        }
        cand = block_min(cand, sm);
        if (cand != 0x7FFFFFFF) {
            lo = cand < p ? cand : p;
            break;
        }
        lo = ((lo >> 5) + CTA_T) * 32;
        if (lo >= p) {
            lo = p;
            break;
        }
    }
    if (policy == ASR_HRRN && ps.thr_valid) {
        // Horizon from the life of the pool that just lapsed.  Requests cross the threshold at the rate they
        // are served, so the strong members last  elapsed * target / used  and the weak members a horizon H
        // lets in grow like  weak0 * H / H0 : cover 1.25 lives, within 0.8 of the room the pool has for them.
        const float elapsed = (float)(t - ps.t0), used = (float)(ps.G0 - ps.G);
        const float h0 = (float)(ps.t0H - ps.t0), weak0 = (float)(ps.P0 - ps.G0);
        float h = (float)ps.H;
        if (used >= 1.f && elapsed >= 1.f) h = 1.25f * elapsed * (float)POOL_TARGET / used;
        else if (t > ps.t0H && ps.G >= k) h *= 2.f;   // horizon ran out before anything was learnt
        if (weak0 >= 1.f && h0 >= 1.f) h = fminf(h, 0.8f * (float)(POOL_CAP - POOL_TARGET) * h0 / weak0);
        const int64_t hi = (int64_t)fminf(h, (float)H_MAX);
        ps.H = hi < 1000 ? 1000 : (hi > H_MAX ? H_MAX : hi);
    }
    STAT(0, 1);
    if (policy == ASR_HRRN && ps.thr_valid && t > ps.t0H) STAT(3, 1);
    if (ps.thr_valid && ps.G < k) STAT(4, 1);
    ps.thr_valid = false;
    ps.complete = false;
    ps.P = 0;
    ps.G = 0;
    ps.t0 = t;
    if (tid == 0) sm.pool_n = 0;
    __syncthreads();
    if (nW <= POOL_CAP) {
        scan_waiting(trace, bm, lo, p, [&](const int4 &e) { sm.pool[atomicAdd(&sm.pool_n, 1)] = e; });
        __syncthreads();
        ps.P = sm.pool_n;
        ps.complete = true;
        return;
    }
    // --- threshold mode: pick theta with a histogram over the approximate key
    // The threshold moves slowly between rebuilds: the first histogram is centred on the last threshold's key
    // and also counts what lies above its window; only if the target rank falls outside it does the full
    // procedure (key range by a scan of its own, then refinement levels) run.
    int64_t lo_k0 = 0, hi_k0 = -1;
    bool guess = ps.prev_valid;
    int target = POOL_TARGET;
  for (int attempt = 0; attempt < 4; ++attempt) {
    if (!guess && hi_k0 < lo_k0) {
        int kmin = 0x7FFFFFFF, kmax = 0;
        scan_waiting(trace, bm, lo, p, [&](const int4 &e) {
            const int key = approx_key(policy, e, t);
            kmin = key < kmin ? key : kmin;
            kmax = key > kmax ? key : kmax;
        });
        lo_k0 = block_min(kmin, sm);
        hi_k0 = block_max(kmax, sm);
    }
    const int64_t guess_w = policy == ASR_SJF ? 1023 : (1 << 18);   // est in ms; 3% of a ratio in float bits
    int64_t lo_k = guess ? (int64_t)ps.prev_key - guess_w : lo_k0, hi_k = guess ? (int64_t)ps.prev_key + guess_w : hi_k0;
    int base_above = 0;
    int theta_pos = -1;
    bool guess_failed = false;
    for (int level = 0; level < 4 && theta_pos < 0; ++level) {
        const bool guess_level = guess && level == 0;
        int above = 0;
        const int64_t width = (hi_k - lo_k + HIST_BINS) / HIST_BINS;   // >= 1
        for (int b = tid; b < HIST_BINS; b += CTA_T) {
            sm.hist[b] = 0;
            sm.rep[b] = -1;
        }
        __syncthreads();
        scan_waiting(trace, bm, lo, p, [&](const int4 &e) {
            const int64_t key = approx_key(policy, e, t);
            if (key >= lo_k && key <= hi_k) {
                const int b = (int)((uint32_t)(key - lo_k) / (uint32_t)width);   // keys are 32-bit: so is the range
                atomicAdd(&sm.hist[b], 1u);
                sm.rep[b] = e.w;
            } else if (guess_level && key < lo_k) {
                above++;
            }
        });
        if (guess_level) base_above = block_sum(above, sm);
        __syncthreads();
        if (tid == 0) {
            // smallest bin b with base_above + cum(b) >= target
            int cum = base_above, b = 0, prev = -1;
            for (; b < HIST_BINS; ++b) {
                if (cum + (int)sm.hist[b] >= target) break;
                if (sm.hist[b]) prev = b;
                cum += (int)sm.hist[b];
            }
            int verdict;   // >= 0: trace position of theta; -1: refine inside bin b; -2: give up
            if (b == HIST_BINS) verdict = prev >= 0 ? sm.rep[prev] : -2;
            else if (cum + (int)sm.hist[b] <= POOL_CAP / 2 + POOL_CAP / 4) verdict = sm.rep[b];
            else if (cum >= target / 8 && prev >= 0) verdict = sm.rep[prev];
            else verdict = width > 1 ? -1 : -2;
            if (guess_level && (base_above >= target || b == HIST_BINS)) verdict = -3;   // outside the window
            sm.bc32[0] = verdict;
            sm.bc32[1] = b;
            sm.bc32[2] = cum;
        }
        __syncthreads();
        const int verdict = sm.bc32[0];
        if (verdict >= 0) theta_pos = verdict;
        else if (verdict == -1) {
            base_above = sm.bc32[2];
            lo_k = lo_k + (int64_t)sm.bc32[1] * width;
            hi_k = lo_k + width - 1;
        } else if (verdict == -3) {
            guess_failed = true;
            __syncthreads();
            break;
        } else {
            __syncthreads();
            return;   // no usable threshold (massive ties): the caller scans the window directly
        }
        __syncthreads();
    }
    if (guess_failed) {
        STAT(6, 1);
        guess = false;
        --attempt;
        continue;
    }
    if (theta_pos < 0) return;
    const int4 th = cand_of(trace, theta_pos);
    ps.thrE = th.z;
    ps.thrW = wait_of(rec_arr(th), t);
    ps.prev_key = approx_key(policy, th, t);
    ps.prev_valid = true;
    // --- fill the pool with the exact tests; shrink the horizon until it fits
    for (;;) {
        ps.t0H = t + (policy == ASR_HRRN ? ps.H : 0);
        if (tid == 0) sm.pool_n = 0;
        __syncthreads();
        int strong = 0;
        scan_waiting(trace, bm, lo, p, [&](const int4 &e) {
            if (pool_pass(policy, ps, e)) {
                const int at = atomicAdd(&sm.pool_n, 1);
                if (at < POOL_CAP) sm.pool[at] = e;
                if (policy == ASR_HRRN &&
                    mul64x32(t - rec_arr(e), (uint32_t)ps.thrE) >= mul64x32(ps.thrW, (uint32_t)e.z))
                    strong++;
            }
        });
        strong = block_sum(strong, sm);
        const int cnt = sm.pool_n;
        if (cnt <= POOL_CAP) {
            ps.P = ps.P0 = cnt;
            ps.G = ps.G0 = strong;
            ps.thr_valid = true;
            return;
        }
        if (policy == ASR_HRRN && ps.H > 0) {
            // too many weak members: they grow like the horizon, so aim at 0.8 of the room left by the strong
            STAT(5, 1);
            const int weak = cnt - strong;
            int64_t h = ps.H / 2;
            if (strong <= POOL_CAP * 3 / 4 && weak > 0) {
                const int64_t fit = (int64_t)((float)ps.H * 0.8f * (float)(POOL_CAP - strong) / (float)weak);
                h = fit < h ? fit : h;
            }
            ps.H = h >= 1024 ? h : 0;
            continue;
        }
        // theta lets too many through (ties, or a crowded histogram bin): aim lower and pick again
        __syncthreads();
        if (tid == 0) sm.pool_n = 0;
        __syncthreads();
        target = (int)((int64_t)target * (POOL_CAP / 2) / cnt);
        break;
    }
    if (target < 1) return;
  }
}

// minimum of a 64-bit unsigned value over the warp: two 32-bit REDUX steps
__device__ __forceinline__ uint64_t warp_min_u64(uint64_t x) {
    const uint32_t hi = (uint32_t)(x >> 32);
    const uint32_t mh = __reduce_min_sync(ASR_FULL_MASK, hi);
    const uint32_t ml = __reduce_min_sync(ASR_FULL_MASK, hi == mh ? (uint32_t)x : 0xFFFFFFFFu);
    return ((uint64_t)mh << 32) | ml;
}

// The k-th smallest order scalar (with multiplicity) of the pool for k <= KSEL_SMALL < P, without a single
// pivot: a steady-state step admits a handful of requests out of a pool of one or two thousand, where a
// random-pivot quickselect spends ~2 ln P block-wide rounds.  Every warp extracts the k smallest of its 256
// scalars (k rounds of a warp minimum; only the lane that held it looks for its next one), then warp 0 merges
// the eight ascending lists k steps deep.  Scalars are >= 0, so they compare as unsigned; empty slots hold
// INT64_MAX, which no valid scalar exceeds, and the pool has more than k members.
__device__ __forceinline__ void cmp_swap_u64(uint64_t &a, uint64_t &b) {
    const bool sw = b < a;
    const uint64_t lo = sw ? b : a, hi = sw ? a : b;
    a = lo;
    b = hi;
}

__device__ __forceinline__ int64_t kth_scalar_small(CtaSmem &sm, const int64_t (&Kr)[POOL_EPT], int k) {
    static_assert(POOL_EPT == 8, "the sorting network below is the 19-exchange network for 8 keys");
    const int lane = lane_id(), warp = threadIdx.x >> 5;
    // the lane's 8 scalars ascending, so that the lane a minimum came from only shifts its list
    uint64_t s0 = (uint64_t)Kr[0], s1 = (uint64_t)Kr[1], s2 = (uint64_t)Kr[2], s3 = (uint64_t)Kr[3],
             s4 = (uint64_t)Kr[4], s5 = (uint64_t)Kr[5], s6 = (uint64_t)Kr[6], s7 = (uint64_t)Kr[7];
    cmp_swap_u64(s0, s1); cmp_swap_u64(s2, s3); cmp_swap_u64(s4, s5); cmp_swap_u64(s6, s7);
    cmp_swap_u64(s0, s2); cmp_swap_u64(s1, s3); cmp_swap_u64(s4, s6); cmp_swap_u64(s5, s7);
    cmp_swap_u64(s1, s2); cmp_swap_u64(s5, s6); cmp_swap_u64(s0, s4); cmp_swap_u64(s3, s7);
    cmp_swap_u64(s1, s5); cmp_swap_u64(s2, s6);
    cmp_swap_u64(s1, s4); cmp_swap_u64(s3, s6);
    cmp_swap_u64(s2, s4); cmp_swap_u64(s3, s5);
    cmp_swap_u64(s3, s4);
    for (int r = 0; r < k; ++r) {
        const uint64_t wm = warp_min_u64(s0);
        if (lane == 0) sm.wsel[warp][r] = wm;
        const bool me = lane == __ffs(__ballot_sync(ASR_FULL_MASK, s0 == wm)) - 1;
        s0 = me ? s1 : s0;
        s1 = me ? s2 : s1;
        s2 = me ? s3 : s2;
        s3 = me ? s4 : s3;
        s4 = me ? s5 : s4;
        s5 = me ? s6 : s5;
        s6 = me ? s7 : s6;
        s7 = me ? ~0ull : s7;
    }
    __syncthreads();
    if (warp == 0) {
        int h = 0;
        uint64_t cur = lane < CTA_T / 32 ? sm.wsel[lane][0] : ~0ull;
        uint64_t wm = 0;
        for (int r = 0; r < k; ++r) {
            wm = warp_min_u64(cur);
            const int who = __ffs(__ballot_sync(ASR_FULL_MASK, cur == wm)) - 1;
            if (lane == who) {
                ++h;
                cur = h < k ? sm.wsel[lane][h] : ~0ull;
            }
        }
        if (lane == 0) sm.bc64 = (int64_t)wm;
    }
    __syncthreads();
    return sm.bc64;
}

// ---- exact k-set of the pool -> sm.adm[0..k), members removed from the pool ----------------
__device__ __forceinline__ void pool_select(CtaSmem &sm, PoolState &ps, int policy, int64_t t, int k, uint32_t &seed) {
    const int tid = threadIdx.x;
    const int P = ps.P;
    int64_t Kr[POOL_EPT];
    const bool small_k = k < P && k <= KSEL_SMALL;   // kth_scalar_small: no probes into sm.K, barriers of its own
#pragma unroll
    for (int e = 0; e < POOL_EPT; ++e) {
        const int i = e * CTA_T + tid;
        Kr[e] = INT64_MAX;
        if (i < P) {
            Kr[e] = order_scalar_rt(policy, sm.pool[i], t);
            if (!small_k) sm.K[i] = Kr[e];
        }
    }
    if (tid == 0) sm.adm_n = sm.hole_n = sm.surv_n = sm.tie_n = 0;
    if (!small_k) __syncthreads();
    uint32_t admmask = 0;
    if (k >= P) {
#pragma unroll
        for (int e = 0; e < POOL_EPT; ++e)
            if (e * CTA_T + tid < P) admmask |= 1u << e;
    } else {
        // v = k-th smallest scalar: count_less(v) < k <= count_le(v)
        int64_t Klo = 0, Khi = 0, v = 0;
        bool lo_inf = true, hi_inf = true;
        int cl = 0, ce = 0;
        if (small_k) {
            v = kth_scalar_small(sm, Kr, k);
            int c = 0;
#pragma unroll
            for (int e = 0; e < POOL_EPT; ++e)
                if (e * CTA_T + tid < P) c += (Kr[e] < v ? 1 : 0) + (Kr[e] <= v ? 0x10000 : 0);
            c = block_sum(c, sm);
            cl = c & 0xFFFF;
            ce = c >> 16;
        } else
        for (;;) {
            int64_t pv = 0;
            bool ok = false;
#pragma unroll 1
            for (int probe = 0; probe < 2 && !ok; ++probe) {
                seed = seed * 1664525u + 1013904223u;
                pv = sm.K[(seed >> 8) % (uint32_t)P];
                ok = (lo_inf || pv > Klo) && (hi_inf || pv < Khi);
            }
            if (!ok) {
                // any scalar inside the bracket (v itself is one)
                __syncthreads();
#pragma unroll
                for (int e = 0; e < POOL_EPT; ++e)
                    if (e * CTA_T + tid < P && (lo_inf || Kr[e] > Klo) && (hi_inf || Kr[e] < Khi)) sm.bc64 = Kr[e];
                __syncthreads();
                pv = sm.bc64;
            }
            int c = 0;
#pragma unroll
            for (int e = 0; e < POOL_EPT; ++e)
                if (e * CTA_T + tid < P) c += (Kr[e] < pv ? 1 : 0) + (Kr[e] <= pv ? 0x10000 : 0);
            c = block_sum(c, sm);
            cl = c & 0xFFFF;
            ce = c >> 16;
            if (cl >= k) {
                Khi = pv;
                hi_inf = false;
            } else if (ce >= k) {
                v = pv;
                break;
            } else {
                Klo = pv;
                lo_inf = false;
            }
        }
        const int m = k - cl, T = ce - cl;   // m of the T members with scalar v are admitted
#pragma unroll
        for (int e = 0; e < POOL_EPT; ++e)
            if (e * CTA_T + tid < P && (Kr[e] < v || (T == m && Kr[e] == v))) admmask |= 1u << e;
        if (T != m) {
            // equal scalars: the exact comparator ranks the tied members
#pragma unroll
            for (int e = 0; e < POOL_EPT; ++e)
                if (e * CTA_T + tid < P && Kr[e] == v) sm.tie[atomicAdd(&sm.tie_n, 1)] = (uint16_t)(e * CTA_T + tid);
            __syncthreads();
#pragma unroll 1
            for (int e = 0; e < POOL_EPT; ++e)
                if (e * CTA_T + tid < P && Kr[e] == v) {
                    const int4 me = sm.pool[e * CTA_T + tid];
                    int rank = 0;
                    for (int j = 0; j < T; ++j) {
                        const int4 o = sm.pool[sm.tie[j]];
                        if (o.w != me.w && cand_better(policy, o, me, t)) rank++;
                    }
                    if (rank < m) admmask |= 1u << e;
                }
        }
    }
    // publish the admitted, fill their holes with the survivors of the pool's tail
    const int kk = k < P ? k : P;
    const int newP = P - kk;
#pragma unroll
    for (int e = 0; e < POOL_EPT; ++e) {
        const int i = e * CTA_T + tid;
        if (i < P) {
            if ((admmask >> e) & 1u) {
                sm.adm[atomicAdd(&sm.adm_n, 1)] = sm.pool[i];
                if (i < newP) sm.hole[atomicAdd(&sm.hole_n, 1)] = (uint16_t)i;
            } else if (i >= newP) {
                sm.surv[atomicAdd(&sm.surv_n, 1)] = (uint16_t)i;
            }
        }
    }
    __syncthreads();
    const int h = sm.hole_n;
    for (int j = tid; j < h; j += CTA_T) sm.pool[sm.hole[j]] = sm.pool[sm.surv[j]];
    if (tid == 0) sm.pool_n = newP;
    __syncthreads();
    ps.P = newP;
}

// ---- fallback: exact k best of the waiting window by k block-wide arg-best scans ----------------
__device__ __noinline__ void direct_select(CtaSmem &sm, const asr_req_t *trace, uint32_t *bm, int policy, int64_t t,
                                           int lo, int p, int k) {
    const int tid = threadIdx.x, lane = lane_id(), warp = tid >> 5;
    for (int round = 0; round < k; ++round) {
        int4 b = make_int4(0, 0, 1, -1);
        for (int pos = lo + tid; pos < p; pos += CTA_T)
            if (!is_admitted(bm, pos)) {
                const int4 e = cand_of(trace, pos);
                if (b.w < 0 || cand_better(policy, e, b, t)) b = e;
            }
#pragma unroll
        for (int j = 16; j > 0; j >>= 1) {
            int4 o;
            o.x = __shfl_xor_sync(ASR_FULL_MASK, b.x, j);
            o.y = __shfl_xor_sync(ASR_FULL_MASK, b.y, j);
            o.z = __shfl_xor_sync(ASR_FULL_MASK, b.z, j);
            o.w = __shfl_xor_sync(ASR_FULL_MASK, b.w, j);
            if (o.w >= 0 && (b.w < 0 || cand_better(policy, o, b, t))) b = o;
        }
        __syncthreads();
        if (lane == 0) sm.wbest[warp] = b;
        __syncthreads();
        if (tid == 0) {
            int4 w = sm.wbest[0];
            for (int j = 1; j < CTA_T / 32; ++j) {
                const int4 o = sm.wbest[j];
                if (o.w >= 0 && (w.w < 0 || cand_better(policy, o, w, t))) w = o;
            }
            sm.adm[round] = w;
            atomicOr(&bm[w.w >> 5], 1u << (w.w & 31));   // the next round skips it
            __threadfence_block();
        }
        __syncthreads();
    }
}

__device__ void cta_replica(const SimArgs &a, const int r, CtaSmem &sm) {
    const int tid = threadIdx.x;
    const asr_replica_t rep = a.replicas[r];
    const int n = rep.n, slots = rep.slots, policy = rep.policy;
    if (!replica_ok(a, rep, CTA_T)) {
        if (tid == 0) flag_invalid(a, r);
        return;
    }
    const asr_cost_model_t cm = a.cms[rep.cm_id];
    const asr_req_t *trace = a.traces + rep.trace_off;
    int64_t *lat = a.out_lat + rep.out_off;
    int64_t *ttft = a.out_ttft + rep.out_off;
    uint32_t *bm = a.bitmap + a.bm_off[r];
    for (int w = tid; w <= (n >> 5) + 1; w += CTA_T) bm[w] = 0u;
    if (tid == 0) sm.pool_n = 0;
    __syncthreads();

    int32_t rem = REM_FREE, ridx = -1;   // my batch slot
    int64_t rarr = 0;
    int64_t t = 0;
    int p = 0, lo = 0, nW = 0, nR = 0, done = 0;
    PoolState ps;
    ps.P = 0;
    ps.complete = true;   // nothing waits, the empty pool holds it
    ps.thr_valid = false;
    ps.G = 0;
    ps.thrW = 0;
    ps.thrE = 0;
    ps.t0H = 0;
    ps.t0 = 0;
    ps.H = 1000000;
    ps.G0 = ps.P0 = 0;
    ps.prev_key = 0;
    ps.prev_valid = false;
    uint32_t seed = 0x9E3779B9u * (uint32_t)(r + 1);
    int cbase = 0;
    int64_t carr = tid < n ? __ldg(reinterpret_cast<const long long *>(trace + tid)) : INT64_MAX;
    sm.carr_win[tid] = carr;   // read after the ingest loop's first barrier
    const int64_t first_arrival = n > 0 ? __ldg(reinterpret_cast<const long long *>(trace)) : 0;

    while (done < n) {
        // ---- 1. ingest arrivals <= t
        for (;;) {
            const int i = cbase + tid;
            const bool isnew = i >= p && i < n && carr <= t;
            const int cnt = __syncthreads_count(isnew);
            if (cnt > 0 && policy != ASR_FCFS && (ps.complete || ps.thr_valid)) {
                if (isnew) {
                    const int4 e = cand_of(trace, i);
                    if (ps.complete || pool_pass(policy, ps, e)) {
                        const int at = atomicAdd(&sm.pool_n, 1);
                        if (at < POOL_CAP) sm.pool[at] = e;
                    }
                }
                __syncthreads();
                const int np = sm.pool_n;
                if (np > POOL_CAP) {   // does not fit any more: drop the pool, rebuild on demand
                    __syncthreads();
                    if (tid == 0) sm.pool_n = 0;
                    __syncthreads();
                    ps.P = 0;
                    ps.complete = false;
                    ps.thr_valid = false;
                    ps.G = 0;
                } else {
                    ps.P = np;
                }
            }
            p += cnt;
            nW += cnt;
            if (cnt == 0 || p < cbase + CTA_T) break;
            cbase += CTA_T;
            carr = cbase + tid < n ? __ldg(reinterpret_cast<const long long *>(trace + cbase + tid)) : INT64_MAX;
            sm.carr_win[tid] = carr;   // the loop's next barrier orders it before any read
        }
        // arrival stamp of the next request (p < cbase + CTA_T here)
        const int64_t next_arr = p < n ? sm.carr_win[p - cbase] : INT64_MAX;
        // ---- 2. idle server
        if (nR == 0 && nW == 0) {
            t = next_arr;
            continue;
        }
        // ---- 3. admit
        const int free_slots = slots - nR;
        const int k = free_slots < nW ? free_slots : nW;
        bool newly = false;
        int32_t my_dur = 0;
        if (k > 0) {
            const bool is_free = tid < slots && rem == REM_FREE;
            if (policy == ASR_FCFS) {
                const int rank = block_rank(is_free, sm);
                if (is_free && rank < k) {
                    const Rec q = ld_cached(trace + lo + rank);
                    rem = tokens_of(cm, q.dur_ms);
                    ridx = lo + rank;
                    rarr = q.arrival_us;
                    my_dur = q.dur_ms;
                    newly = true;
                }
                lo += k;
            } else {
                auto usable = [&]() {
                    return ps.complete ||
                           (ps.thr_valid && (policy == ASR_SJF ? ps.P >= k : (ps.G >= k && ps.P >= k && t <= ps.t0H)));
                };
                if (!usable()) pool_rebuild(sm, ps, trace, bm, policy, t, lo, p, nW, k);
                if (usable()) {
                    pool_select(sm, ps, policy, t, k, seed);
                    if (!ps.complete) ps.G -= k;
                } else {
                    direct_select(sm, trace, bm, policy, t, lo, p, k);
                    ps.P = 0;
                    ps.thr_valid = false;
                    ps.complete = false;
                    ps.G = 0;
                    if (tid == 0) sm.pool_n = 0;
                }
                const int rank = block_rank(is_free, sm);   // also orders the writes of sm.adm before the reads
                if (is_free && rank < k) {
                    const int4 e = sm.adm[rank];
                    my_dur = __ldg(&trace[e.w].dur_ms);
                    rem = tokens_of(cm, my_dur);
                    ridx = e.w;
                    rarr = rec_arr(e);
                    newly = true;
                    atomicOr(&bm[e.w >> 5], 1u << (e.w & 31));
                }
            }
            nW -= k;
            nR += k;
        }
        // ---- 4. one engine iteration with the encoders of the admitted, then the exact fast-forward
        const int64_t c = cm.iter_base_us + cm.iter_per_running_us * (int64_t)nR;
        int64_t t1 = t + c;
        int64_t dur_sum;
        int32_t m;   // >= 1: nR >= 1 here
        block_sum_min(my_dur, rem, dur_sum, m, sm);
        if (k > 0) {
            t1 += cm.enc_base_us * (int64_t)k + cm.enc_per_ms_us * dur_sum;
            if (newly) ttft[ridx] = t1 - rarr;   // first token (S9)
        }
        int64_t j = 1;
        if (m > 1) {
            if (nR == slots || p >= n || c <= 0) {
                j = m;
            } else {
                const int64_t g = next_arr - t1;
                if (g <= 0) j = 1;
                else if (g > (int64_t)(m - 2) * c) j = m;
                else j = 1 + ceil_div_pos(g, c);
            }
        }
        t = t1 + (j - 1) * c;
        // ---- 5. tokens, completions
        bool fin = false;
        if (rem != REM_FREE) {
            rem -= (int32_t)j;
            if (rem == 0) {
                lat[ridx] = t - rarr;
                rem = REM_FREE;
                fin = true;
            }
        }
        const int nfin = __syncthreads_count(fin);
        nR -= nfin;
        done += nfin;
    }
#ifdef CTA_STATS
    if (tid == 0) {
        printf("cta stats: policy %d rebuilds %llu scans %llu positions %llu horizon-out %llu strong-out %llu shrinks %llu guess-fail %llu H %lld\n",
               policy, g_stat[0], g_stat[1], g_stat[2], g_stat[3], g_stat[4], g_stat[5], g_stat[6], (long long)ps.H);
        for (int i = 0; i < 8; ++i) g_stat[i] = 0;
    }
#endif
    if (a.out_summary && tid == 0) {
        asr_summary_t *s = a.out_summary + r;
        s->first_arrival_us = first_arrival;
        s->last_done_us = t;
        s->n_done = done;
    }
    __syncthreads();
}

__global__ void __launch_bounds__(CTA_T) sim_cta_kernel(SimArgs a) {
    extern __shared__ __align__(16) unsigned char cta_dyn_smem[];
    CtaSmem &sm = *reinterpret_cast<CtaSmem *>(cta_dyn_smem);
    const int cnt = *a.defer2_count;
    for (int w = blockIdx.x; w < cnt; w += gridDim.x) cta_replica(a, a.defer2_list[w], sm);
}

int launch_simulate_cta(const SimArgs &a, cudaStream_t st) {
    {   // per-device opt-in, set on every launch
        cudaError_t e = cudaFuncSetAttribute(sim_cta_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)sizeof(CtaSmem));
        if (e != cudaSuccess) {
            set_error("sim_cta_kernel: cudaFuncSetAttribute: %s", cudaGetErrorString(e));
            cudaGetLastError();
            return ASR_ECUDA;
        }
    }
    const int grid = a.n_replicas < sm_count() * 2 ? a.n_replicas : sm_count() * 2;
    {
        KernelTimer kt(KID_SIM_CTA, st);
        sim_cta_kernel<<<grid, CTA_T, sizeof(CtaSmem), st>>>(a);
    }
    return check_launch("sim_cta_kernel");
}

}  // namespace asr

// select.cu -- a2 priority keys + a3 batched top-k select (k <= 32), sm_100a.
//
// One warp owns one queue and STREAMS it from HBM exactly once with 128-bit
// loads (8 independent loads per lane in flight, next tile prefetched).  The
// exact k best so far live as a sorted list across the 32 lanes ("kept").
// A record is looked at closely only if a cheap, conservative proxy test says
// it might beat the current k-th best; such candidates are parked in a small
// shared-memory buffer and merged into the kept list 32 at a time with a
// bitonic sort + bitonic merge over warp shuffles.  Expected candidates per
// queue are ~k(1+ln(n/k)), so the merge work is O(k log^2 k ln n) while the
// stream is O(n): the kernel is HBM-bound by design (16 B per record).
//
// Exactness.  Ordering inside the sort uses a 57-bit monotone surrogate key
// (exact for FCFS/SJF up to the arrival resolution, a truncated fp64 ratio
// for HRRN); whenever two surrogate keys are closer than the surrogate's
// resolution the full integer comparator of asr_sched.h (int64
// cross-multiplication for HRRN) decides, so the result is the
// exact total order -- never an approximation of it.
#include "launchers.cuh"

namespace asr {

constexpr int SEL_WARPS = 8;   // warps (= queues in flight) per CTA
constexpr int SEL_TILE = 8;    // chunks of 32 records per tile: 8 x 16 B per lane in flight
constexpr int SEL_PEND = 64;   // pending-candidate capacity per warp
constexpr int SEL_SLOTS = 32 + SEL_PEND;
constexpr uint64_t SEL_INF = ~0ull;  // "no element": key 2^57-1, slot 127

struct __align__(16) SelWarpSmem {
    int4 rec[SEL_SLOTS];       // (arrival lo, arrival hi, est, idx); 0..31 kept bank, 32.. pending
    uint64_t pkey[SEL_PEND];   // surrogate key of each pending candidate
};

__device__ __forceinline__ int64_t rec_arr(const int4 &r) {
    return (int64_t)(((uint64_t)(uint32_t)r.y << 32) | (uint32_t)r.x);
}

// 57-bit surrogate key, smaller = better.  Guarantee used below:
//   key(a) + MARGIN < key(b)  ==>  a is strictly better than b.
template <int POLICY>
struct Surrogate;
template <>
struct Surrogate<ASR_FCFS> {
    static constexpr uint64_t MARGIN = 0;
    __device__ static uint64_t key(int64_t arr, int32_t, int64_t) {
        return (uint64_t)arr & ((1ull << 57) - 1);
    }
};
template <>
struct Surrogate<ASR_SJF> {
    static constexpr uint64_t MARGIN = 0;
    __device__ static uint64_t key(int64_t arr, int32_t est, int64_t) {
        // est < 2^25, arrival < 2^38: (est, arrival >> 6) packed
        return ((uint64_t)est_of(est) << 32) | (((uint64_t)arr >> 6) & 0xFFFFFFFFull);
    }
};
template <>
struct Surrogate<ASR_HRRN> {
    // fp64 quotient is within 2^-53 of wait/est; dropping 7 bits leaves 2^-45
    // resolution, so keys two or more units apart are ordered with certainty.
    static constexpr uint64_t MARGIN = 1;
    __device__ static uint64_t key(int64_t arr, int32_t est, int64_t now) {
        double q = __ll2double_rn(wait_of(arr, now)) / __ll2double_rn(est_of(est));
        return (~(uint64_t)__double_as_longlong(q)) >> 7;
    }
};

// a before b in the exact total order; a, b are packed (key << 7 | slot)
template <int POLICY>
__device__ __forceinline__ bool packed_less(uint64_t a, uint64_t b, const int4 *rec, int64_t now) {
    uint64_t ka = a >> 7, kb = b >> 7;
    uint64_t d = ka > kb ? ka - kb : kb - ka;
    if (d > Surrogate<POLICY>::MARGIN || a == SEL_INF || b == SEL_INF) return a < b;
    int4 ra = rec[a & 127], rb = rec[b & 127];
    return better<POLICY>(rec_arr(ra), ra.z, ra.w, rec_arr(rb), rb.z, rb.w, now);
}

template <int POLICY>
__device__ __forceinline__ uint64_t cmp_exchange(uint64_t v, int j, bool keep_min, const int4 *rec,
                                                 int64_t now) {
    uint64_t o = shfl64_xor(v, j);
    bool v_less = packed_less<POLICY>(v, o, rec, now);
    return (keep_min == v_less) ? v : o;
}

// Merge up to 32 pending candidates (batch b) into the kept list K.
template <int POLICY>
__device__ __forceinline__ uint64_t merge_batch(uint64_t K, SelWarpSmem &sm, int b, int nP, int64_t now) {
    const int lane = lane_id();
    const int pi = b * 32 + lane;
    uint64_t P = pi < nP ? ((sm.pkey[pi] << 7) | (uint64_t)(32 + pi)) : SEL_INF;
    // bitonic sort of P, ascending across lanes
#pragma unroll
    for (int k = 2; k <= 32; k <<= 1) {
#pragma unroll
        for (int j = k >> 1; j > 0; j >>= 1) {
            bool up = (lane & k) == 0;
            bool lower = (lane & j) == 0;
            P = cmp_exchange<POLICY>(P, j, lower == up, sm.rec, now);
        }
    }
    // K ascending, reversed P descending -> element-wise min is the 32 best, bitonic
    uint64_t Pr;
    {
        uint32_t lo = __shfl_sync(ASR_FULL_MASK, (uint32_t)P, 31 - lane);
        uint32_t hi = __shfl_sync(ASR_FULL_MASK, (uint32_t)(P >> 32), 31 - lane);
        Pr = ((uint64_t)hi << 32) | lo;
    }
    K = packed_less<POLICY>(K, Pr, sm.rec, now) ? K : Pr;
#pragma unroll
    for (int j = 16; j > 0; j >>= 1) K = cmp_exchange<POLICY>(K, j, (lane & j) == 0, sm.rec, now);
    // move the survivors' payload into the kept bank, slot = lane
    int4 r = make_int4(0, 0, 0, -1);
    if (K != SEL_INF) r = sm.rec[K & 127];
    __syncwarp();
    sm.rec[lane] = r;
    if (K != SEL_INF) K = (K & ~127ull) | (uint64_t)lane;
    __syncwarp();
    return K;
}

struct SelArgs {
    const asr_req_t *keys;
    const int32_t *src_idx;     // INDIRECT: positions into keys (-1 = hole), else nullptr
    const int32_t *q_count;     // nullable
    const int64_t *now_per_queue;  // nullable
    int32_t *out_idx;
    int64_t now;
    int64_t total;              // total records (ragged last queue) or -1
    int32_t n_queues;
    int32_t q_len;
    int32_t k;
    int32_t global_idx;         // report q*q_len + j instead of j
};

template <int POLICY, bool INDIRECT>
__global__ void __launch_bounds__(SEL_WARPS * 32) select_topk_kernel(SelArgs a) {
    __shared__ SelWarpSmem smem[SEL_WARPS];
    const int lane = lane_id();
    const int warp = threadIdx.x >> 5;
    SelWarpSmem &sm = smem[warp];
    const uint32_t lt_mask = (1u << lane) - 1u;
    const int k = a.k;

    for (int q = blockIdx.x * SEL_WARPS + warp; q < a.n_queues; q += gridDim.x * SEL_WARPS) {
        const int64_t qbase = (int64_t)q * a.q_len;
        int count = a.q_count ? a.q_count[q] : a.q_len;
        if (a.total >= 0) {
            int64_t left = a.total - qbase;
            count = (int)(left < (int64_t)count ? (left < 0 ? 0 : left) : count);
        }
        count = count < 0 ? 0 : (count > a.q_len ? a.q_len : count);
        const int64_t now = a.now_per_queue ? a.now_per_queue[q] : a.now;
        const asr_req_t *base = a.keys + (INDIRECT ? 0 : qbase);
        const int32_t idx_base = a.global_idx ? (int32_t)qbase : 0;

        uint64_t K = SEL_INF;   // kept list, lane i = i-th best so far (packed)
        int nP = 0;             // pending candidates
        // threshold record T = current k-th best (valid once k records are kept)
        bool t_valid = false;
        uint64_t t_key = 0;
        int64_t t_arr = 0;
        int32_t t_est = 0, t_idx = 0;
        float t_qf = -1.0f;     // HRRN proxy: pass if wait_up >= t_qf * est

        auto refresh_threshold = [&]() {
            uint64_t Kk = (uint64_t)shfl64((int64_t)K, k - 1);
            t_valid = Kk != SEL_INF;
            if (t_valid) {
                int4 r = sm.rec[Kk & 127];
                t_key = Kk >> 7;
                t_arr = rec_arr(r);
                t_est = r.z;
                t_idx = r.w;
                if (POLICY == ASR_HRRN) {
                    double q = __ll2double_rn(wait_of(t_arr, now)) / __ll2double_rn(est_of(t_est));
                    float f = __double2float_rd(q);
                    // one fp32 ulp of slack covers the fp64 rounding and the key margin
                    t_qf = f > 0.0f ? __int_as_float(__float_as_int(f) - 1) : -1.0f;
                }
            }
        };

        auto flush = [&]() {
            __syncwarp();
            for (int b = 0; b * 32 < nP; ++b) K = merge_batch<POLICY>(K, sm, b, nP, now);
            nP = 0;
            if (k > 0) refresh_threshold();
        };

        auto consider = [&](const Rec &r, int32_t idx, bool valid) {
            // cheap conservative proxy: a superset of {key <= t_key + MARGIN}
            bool pass = valid;
            if (t_valid) {
                if (POLICY == ASR_FCFS) pass = pass && r.arrival_us <= t_arr;
                if (POLICY == ASR_SJF) pass = pass && est_of(r.est) <= est_of(t_est);
                if (POLICY == ASR_HRRN) {
                    float w_up = __ll2float_ru(wait_of(r.arrival_us, now));
                    float e_dn = __ll2float_rd(est_of(r.est));
                    pass = pass && w_up >= __fmul_rd(t_qf, e_dn);
                }
            }
            if (__ballot_sync(ASR_FULL_MASK, pass) == 0u) return;
            uint64_t key = 0;
            if (pass) {
                key = Surrogate<POLICY>::key(r.arrival_us, r.est, now);
                if (t_valid) {
                    if (key > t_key + Surrogate<POLICY>::MARGIN) {
                        pass = false;
                    } else if (key + Surrogate<POLICY>::MARGIN >= t_key) {
                        // too close for the surrogate: the integer comparator decides
                        pass = better<POLICY>(r.arrival_us, r.est, idx, t_arr, t_est, t_idx, now);
                    }
                }
            }
            uint32_t m = __ballot_sync(ASR_FULL_MASK, pass);
            if (m == 0u) return;
            if (pass) {
                int pos = nP + __popc(m & lt_mask);
                sm.rec[32 + pos] = make_int4((int)(uint32_t)r.arrival_us, (int)(r.arrival_us >> 32),
                                             r.est, idx);
                sm.pkey[pos] = key;
            }
            nP += __popc(m);
            if (nP >= 32) flush();
        };

        auto fetch = [&](int j, Rec &r, int32_t &idx, bool &valid) {
            valid = j < count;
            r.arrival_us = 0;
            r.dur_ms = 0;
            r.est = 1;
            idx = idx_base + j;
            if (INDIRECT) {
                if (valid) {
                    int32_t s = a.src_idx[qbase + j];
                    valid = s >= 0;
                    idx = s;
                    if (valid) r = ld_cached(base + s);
                }
            } else if (valid) {
                r = ld_stream(base + j);
            }
        };

        const int ntiles = (count + SEL_TILE * 32 - 1) / (SEL_TILE * 32);
        Rec cur[SEL_TILE];
        int32_t cidx[SEL_TILE];
        bool cval[SEL_TILE];
        if (ntiles > 0) {
#pragma unroll
            for (int c = 0; c < SEL_TILE; ++c) fetch(c * 32 + lane, cur[c], cidx[c], cval[c]);
        }
        for (int t = 0; t < ntiles; ++t) {
            Rec nxt[SEL_TILE];
            int32_t nidx[SEL_TILE];
            bool nval[SEL_TILE];
            if (t + 1 < ntiles) {
#pragma unroll
                for (int c = 0; c < SEL_TILE; ++c)
                    fetch((t + 1) * SEL_TILE * 32 + c * 32 + lane, nxt[c], nidx[c], nval[c]);
            }
#pragma unroll
            for (int c = 0; c < SEL_TILE; ++c) consider(cur[c], cidx[c], cval[c]);
            if (t + 1 < ntiles) {
#pragma unroll
                for (int c = 0; c < SEL_TILE; ++c) {
                    cur[c] = nxt[c];
                    cidx[c] = nidx[c];
                    cval[c] = nval[c];
                }
            }
        }
        if (nP > 0) flush();
        __syncwarp();
        if (lane < k) {
            int32_t o = -1;
            if (K != SEL_INF) o = sm.rec[K & 127].w;
            a.out_idx[(int64_t)q * k + lane] = o;
        }
        __syncwarp();
    }
}

template <int POLICY, bool INDIRECT>
static int launch_one(const SelArgs &a, cudaStream_t st) {
    if (a.n_queues <= 0 || a.k <= 0) return ASR_OK;
    static int blocks_per_sm = 0, n_sm = 0;
    if (blocks_per_sm == 0) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&blocks_per_sm, select_topk_kernel<POLICY, INDIRECT>,
                                                      SEL_WARPS * 32, 0);
        if (blocks_per_sm < 1) blocks_per_sm = 1;
        if (n_sm < 1) n_sm = 148;
    }
    int64_t want = ((int64_t)a.n_queues + SEL_WARPS - 1) / SEL_WARPS;
    int64_t cap = (int64_t)n_sm * blocks_per_sm;
    int grid = (int)(want < cap ? want : cap);
    {
        KernelTimer kt(KID_SELECT, st);
        select_topk_kernel<POLICY, INDIRECT><<<grid, SEL_WARPS * 32, 0, st>>>(a);
    }
    return check_launch("select_topk_kernel");
}

int launch_select(const SelArgs &a, int policy, cudaStream_t st) {
    const bool ind = a.src_idx != nullptr;
    switch (policy) {
        case ASR_FCFS: return ind ? launch_one<ASR_FCFS, true>(a, st) : launch_one<ASR_FCFS, false>(a, st);
        case ASR_SJF: return ind ? launch_one<ASR_SJF, true>(a, st) : launch_one<ASR_SJF, false>(a, st);
        case ASR_HRRN: return ind ? launch_one<ASR_HRRN, true>(a, st) : launch_one<ASR_HRRN, false>(a, st);
    }
    set_error("unknown policy %d", policy);
    return ASR_EINVAL;
}

}  // namespace asr

// ---------------------------------------------------------------------------
// C ABI
// ---------------------------------------------------------------------------
using namespace asr;

static constexpr int64_t SEL_SEG = 4096;  // segment length of the single-queue reduction tree

extern "C" int asr_sched_select_batched(const asr_req_t *keys, int32_t n_queues, int32_t q_len,
                                        const int32_t *q_count, int32_t policy, int64_t now,
                                        const int64_t *now_per_queue, int32_t k, int32_t *out_idx,
                                        void *stream) {
    if (n_queues < 0 || q_len < 0 || k < 0 || policy < 0 || policy > 2) {
        set_error("select_batched: bad argument (n_queues=%d q_len=%d k=%d policy=%d)", n_queues, q_len, k, policy);
        return ASR_EINVAL;
    }
    if (k > 32) {
        set_error("select_batched: k=%d exceeds the limit 32", k);
        return ASR_EUNSUPPORTED;
    }
    if (n_queues == 0 || k == 0) return ASR_OK;
    if ((!keys && q_len > 0) || !out_idx) {
        set_error("select_batched: null pointer");
        return ASR_EINVAL;
    }
    SelArgs a{keys, nullptr, q_count, now_per_queue, out_idx, now, -1, n_queues, q_len, k, 0};
    return launch_select(a, policy, (cudaStream_t)stream);
}

static size_t select_ws_bytes(int64_t n, int64_t k) {
    if (n <= SEL_SEG || k <= 0) return 0;
    size_t ints = 0;
    int64_t len = n;
    while (len > SEL_SEG) {
        int64_t segs = (len + SEL_SEG - 1) / SEL_SEG;
        ints += (size_t)(segs * k);
        len = segs * k;
    }
    return ints * sizeof(int32_t) + 256;
}

extern "C" int asr_sched_select(const asr_req_t *keys, int64_t n, int32_t policy, int64_t now, int32_t k,
                                int32_t *out_idx, void *workspace, size_t workspace_bytes, void *stream) {
    if (n < 0 || k < 0 || policy < 0 || policy > 2 || n >= (1ll << 31)) {
        set_error("select: bad argument (n=%lld k=%d policy=%d)", (long long)n, k, policy);
        return ASR_EINVAL;
    }
    if (k > 32) {
        set_error("select: k=%d exceeds the limit 32", k);
        return ASR_EUNSUPPORTED;
    }
    if (k == 0) return ASR_OK;
    if ((!keys && n > 0) || !out_idx) {
        set_error("select: null pointer");
        return ASR_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    if (n <= SEL_SEG) {
        SelArgs a{keys, nullptr, nullptr, nullptr, out_idx, now, n, 1, (int32_t)(n > 0 ? n : 1), k, 0};
        return launch_select(a, policy, st);
    }
    if (workspace_bytes < select_ws_bytes(n, k) || !workspace) {
        set_error("select: workspace too small (%zu < %zu)", workspace_bytes, select_ws_bytes(n, k));
        return ASR_EINVAL;
    }
    // level 0: every segment of 4096 records reports its own k best (global positions)
    int32_t *level = (int32_t *)workspace;
    int64_t segs = (n + SEL_SEG - 1) / SEL_SEG;
    {
        SelArgs a{keys, nullptr, nullptr, nullptr, level, now, n, (int32_t)segs, (int32_t)SEL_SEG, k, 1};
        int rc = launch_select(a, policy, st);
        if (rc) return rc;
    }
    // further levels: select among the reported candidates (holes are -1)
    int64_t len = segs * k;
    while (true) {
        int64_t nsegs = (len + SEL_SEG - 1) / SEL_SEG;
        int32_t *dst = nsegs == 1 ? out_idx : level + len;
        SelArgs a{keys, level, nullptr, nullptr, dst, now, len, (int32_t)nsegs, (int32_t)SEL_SEG, k, 0};
        int rc = launch_select(a, policy, st);
        if (rc) return rc;
        if (nsegs == 1) break;
        level = dst;
        len = nsegs * k;
    }
    return ASR_OK;
}

namespace asr {
size_t select_workspace_bytes(int64_t n, int64_t k) { return select_ws_bytes(n, k); }
}

// select.cu -- a2 priority keys + a3 batched top-k select, sm_100a.  The streaming kernel described here serves
// k <= 32 (config 5); select_wide_kernel near the end serves 32 < k <= 256.
//
// One warp owns one queue at a time and STREAMS it from HBM exactly once.  The
// queue is cut into chunks of SEL_CHUNK records (4 KB); lane 0 of the warp
// moves each chunk into the warp's private ring of shared-memory stages with
// one TMA bulk copy (cp.async.bulk, completion on an mbarrier), SEL_STAGES
// chunks ahead of the consumer and across queue boundaries, so the data path
// costs one instruction per 4 KB and no registers.  The 32 lanes then read the
// stage with conflict-free 128-bit shared loads.
//
// Per record the warp runs ONE cheap, conservative, integer test against a
// threshold record T ("could this record be among the k best?"):
//   FCFS  arrival <= T.arrival
//   SJF   (est, arrival) <= (T.est, T.arrival)
//   HRRN  wait*T.est >= T.wait*est  in int64
// Survivors (a few per cent) are appended to a small candidate buffer in
// shared memory.  When the buffer fills, an exact quickselect over the buffer
// (random pivot, full comparator of asr_sched.h incl. the (arrival, idx)
// tie-break) keeps the best k..2k candidates and makes the worst kept one the
// new T.  At the end of the queue the buffer is cut to exactly the k best and
// sorted across the lanes with a bitonic network on the exact comparator.
// Carried threshold.  Consecutive queues of a batch usually look alike, so a
// warp starts a queue with the threshold of rank ~2k that it found in its
// previous queue instead of "pass everything": ~2k records survive, no cut
// happens before the end of the queue, and the exact work per queue is one
// quickselect over ~2k candidates.  The pass set of any threshold is closed
// upwards in the total order, so it holds the k best whenever it holds at
// least k records; if it holds fewer (the carried threshold was too strict for
// this queue) the warp re-reads the queue with "pass everything".
// Every decision that affects the output is taken by the exact integer
// comparator, so the result is the unique total order -- never an approximation.
// HBM-bound by design: 16 B read per record, 4k B written per queue.
#include <mutex>
#include "launchers.cuh"

namespace asr {

#ifndef SEL_WARPS_N
#define SEL_WARPS_N 20
#endif
#ifndef SEL_CHUNK_N
#define SEL_CHUNK_N 256
#endif
#ifndef SEL_STAGES_N
#define SEL_STAGES_N 2
#endif
constexpr int SEL_WARPS = SEL_WARPS_N;          // warps (= queues in flight) per CTA, one CTA per SM
constexpr int SEL_CHUNK = SEL_CHUNK_N;          // records per staged chunk (4 KB)
constexpr int SEL_STAGES = SEL_STAGES_N;        // TMA ring depth per warp
constexpr int SEL_UNROLL = 2;                   // records per lane loaded and tested together
constexpr int SEL_ROWS = 6;                     // candidate buffer: rows of 32
constexpr int SEL_BUFCAP = SEL_ROWS * 32;       // 192 candidates
constexpr int SEL_FLUSH_AT = SEL_BUFCAP - 64;   // cut the buffer once it holds more than this (checked every 64 records)

struct __align__(128) SelWarpSmem {
    int4 stage[SEL_STAGES][SEL_CHUNK];   // raw records (arrival lo, arrival hi, dur_ms | src idx, est)
    int4 buf[SEL_BUFCAP];                // candidates (arrival lo, arrival hi, max(est,1), idx)
    uint64_t full[SEL_STAGES];           // mbarriers: chunk landed
    int64_t carry_t64;                   // threshold carried to this warp's next queue (valid if carry_ok)
    int32_t carry_t32;
    int32_t carry_ok;
};
constexpr size_t SEL_SMEM_BYTES = sizeof(SelWarpSmem) * SEL_WARPS;

// ---- threshold record T and the conservative per-record test -------------------
struct Thr {
    int64_t t64;
    int32_t t32;
};

template <int POLICY>
__device__ __forceinline__ Thr thr_pass_all() {
    Thr t;
    if (POLICY == ASR_HRRN) {
        t.t64 = 0;   // T.wait
        t.t32 = 0;   // T.est = 0: 0 >= 0 passes everything
    } else {
        t.t64 = INT64_MAX;
        t.t32 = INT32_MAX;
    }
    return t;
}

// T := candidate p (arrival lo, hi, est >= 1, idx)
template <int POLICY>
__device__ __forceinline__ Thr thr_from(const int4 &p, int64_t now) {
    Thr t;
    if (POLICY == ASR_HRRN) {
        t.t64 = wait_of(rec_arr(p), now);
        t.t32 = t.t64 == 0 ? 0 : p.z;   // a zero-wait threshold ties with every clamped wait: pass all
    } else {
        t.t64 = rec_arr(p);
        t.t32 = p.z;
    }
    return t;
}

// true for every record that is better than or ties with T (a superset is fine)
template <int POLICY>
__device__ __forceinline__ bool may_beat(int64_t arr, int32_t est_raw, const Thr &t, int64_t now) {
    if (POLICY == ASR_FCFS) return arr <= t.t64;
    const int32_t e = est_raw < 1 ? 1 : est_raw;
    if (POLICY == ASR_SJF) return e < t.t32 || (e == t.t32 && arr <= t.t64);
    // HRRN: the signed wait is not clamped here: a negative wait fails unless T.est == 0
    const int64_t w = now - arr;
    return mul64x32(w, (uint32_t)t.t32) >= mul64x32(t.t64, (uint32_t)e);
}

// ---- exact quickselect over the candidate buffer --------------------------------
// Keeps the c+1 best candidates where c in [c_lo, c_hi] is the rank of an
// accepted pivot (number of candidates strictly better than it); the pivot is
// the worst kept candidate.  Precondition: c_lo < cnt <= SEL_BUFCAP.
// Returns (position of the pivot in the compacted buffer << 16) | new count.
template <int POLICY>
__device__ __noinline__ uint32_t buffer_cut(int4 *buf, int cnt, int c_lo, int c_hi, int64_t now, uint32_t seed) {
    const int lane = lane_id();
    const uint32_t lt_mask = (1u << lane) - 1u;
    const int nrows = (cnt + 31) >> 5;
    int64_t A[SEL_ROWS];      // order scalar of candidate j*32 + lane
    uint32_t pri[SEL_ROWS];   // random priority (23 bits) | 0x100 | position
    uint32_t alive = 0, keep = 0;
#pragma unroll
    for (int j = 0; j < SEL_ROWS; ++j) {
        if (j < nrows) {
            const uint32_t i = (uint32_t)(j * 32 + lane);
            if ((int)i < cnt) alive |= 1u << j;
            A[j] = order_scalar<POLICY>(buf[(int)i < cnt ? i : 0u], now);
            uint32_t h = (i + 1u) * 2654435761u ^ seed;
            h ^= h >> 15;
            h *= 2246822519u;
            pri[j] = (h & 0xFFFFFE00u) | 0x100u | i;
        }
    }
    int base = 0;
    int pi = 0;
    for (;;) {
        // uniform random pivot among the alive candidates
        seed = seed * 1664525u + 1013904223u;
        const uint32_t sx = seed & 0xFFFFFE00u;
        uint32_t best = 0;
#pragma unroll
        for (int j = 0; j < SEL_ROWS; ++j)
            if (j < nrows) {
                const uint32_t h = pri[j] ^ sx;
                if ((alive >> j) & 1u) best = h > best ? h : best;
            }
        const uint32_t win = __reduce_max_sync(ASR_FULL_MASK, best);
        if (win == 0u) break;   // nothing alive (cannot happen under the precondition)
        pi = (int)(win & 0xFFu);
        const uint32_t pflag = (pi & 31) == lane ? (1u << (pi >> 5)) : 0u;
        // the pivot's scalar comes from the lane that holds it
        int64_t mine = 0;
#pragma unroll
        for (int j = 0; j < SEL_ROWS; ++j)
            if (j < nrows && (pi >> 5) == j) mine = A[j];
        const int64_t Kp = shfl64(mine, pi & 31);
        uint32_t bflags = 0, tflags = 0;
#pragma unroll
        for (int j = 0; j < SEL_ROWS; ++j)
            if (j < nrows) {
                bflags |= A[j] < Kp ? (1u << j) : 0u;
                tflags |= A[j] == Kp ? (1u << j) : 0u;
            }
        tflags &= alive & ~pflag;
        if (__any_sync(ASR_FULL_MASK, tflags != 0u)) {
            // rare: equal scalars -- the full comparator with its (arrival, idx) tie-break decides
            const int4 P = buf[pi];
#pragma unroll
            for (int j = 0; j < SEL_ROWS; ++j)
                if (j < nrows && ((tflags >> j) & 1u)) {
                    const int4 e = buf[j * 32 + lane];
                    if (better<POLICY>(rec_arr(e), e.z, e.w, rec_arr(P), P.z, P.w, now)) bflags |= 1u << j;
                }
        }
        bflags &= alive;
        int c_alive = 0;
#pragma unroll
        for (int j = 0; j < SEL_ROWS; ++j)
            if (j < nrows) c_alive += __popc(__ballot_sync(ASR_FULL_MASK, (bflags >> j) & 1u));
        const int c = base + c_alive;
        if (c < c_lo) {            // pivot too good: it and everything better are certainly kept
            const uint32_t mv = alive & (bflags | pflag);
            keep |= mv;
            alive &= ~mv;
            base = c + 1;
        } else if (c > c_hi) {     // pivot too lax: it and everything worse are dropped
            alive &= bflags;
        } else {
            keep |= alive & (bflags | pflag);
            break;
        }
    }
    // in-place compaction, row by row: row j only writes positions <= its own
    __syncwarp();
    int off = 0;
    uint32_t ppos = 0;
#pragma unroll
    for (int j = 0; j < SEL_ROWS; ++j)
        if (j < nrows) {
            const bool kp = (keep >> j) & 1u;
            const int4 e = buf[j * 32 + lane];
            const uint32_t m = __ballot_sync(ASR_FULL_MASK, kp);
            __syncwarp();
            if (kp) {
                const int pos = off + __popc(m & lt_mask);
                buf[pos] = e;
                if (j * 32 + lane == pi) ppos = (uint32_t)pos;
            }
            off += __popc(m);
        }
    ppos = __reduce_max_sync(ASR_FULL_MASK, ppos);
    __syncwarp();
    return (ppos << 16) | (uint32_t)off;
}

// exact bitonic sort of buf[0 .. cnt), cnt <= 32, one candidate per lane: returns the buffer
// position of the candidate of rank `lane` (best first), -1 past the end.  Compares order
// scalars; equal scalars are settled by the exact comparator on the records themselves.
template <int POLICY>
__device__ __forceinline__ int sort32(const int4 *buf, int cnt, int64_t now) {
    const int lane = lane_id();
    int pos = lane < cnt ? lane : -1;
    int64_t K = pos >= 0 ? order_scalar<POLICY>(buf[lane], now) : INT64_MAX;
#pragma unroll
    for (int k = 2; k <= 32; k <<= 1) {
#pragma unroll
        for (int j = k >> 1; j > 0; j >>= 1) {
            const int64_t oK = (int64_t)shfl64_xor((uint64_t)K, j);
            const int opos = __shfl_xor_sync(ASR_FULL_MASK, pos, j);
            const bool up = (lane & k) == 0 || k == 32;
            const bool want_min = ((lane & j) == 0) == up;
            bool v_less = pos >= 0 && (opos < 0 || K < oK);
            const bool tie = pos >= 0 && opos >= 0 && K == oK;
            if (__any_sync(ASR_FULL_MASK, tie)) {
                if (tie) {
                    const int4 a = buf[pos], b = buf[opos];
                    v_less = better<POLICY>(rec_arr(a), a.z, a.w, rec_arr(b), b.z, b.w, now);
                }
            }
            if (want_min != v_less) {
                K = oK;
                pos = opos;
            }
        }
    }
    return pos;
}

struct SelArgs {
    const asr_req_t *keys;
    const int32_t *src_idx;        // INDIRECT: positions into keys, else nullptr
    const int32_t *q_count;        // nullable
    const int64_t *now_per_queue;  // nullable
    int32_t *out_idx;
    int64_t now;
    int64_t total;                 // total records (ragged last queue) or -1
    int32_t n_queues;
    int32_t q_len;
    int32_t k;
    int32_t global_idx;            // report q*q_len + j instead of j
};

__device__ __forceinline__ int sel_count(const SelArgs &a, int q) {
    int count = a.q_count ? a.q_count[q] : a.q_len;
    if (a.total >= 0) {
        const int64_t left = a.total - (int64_t)q * a.q_len;
        count = (int)(left < (int64_t)count ? (left < 0 ? 0 : left) : count);
    }
    return count < 0 ? 0 : (count > a.q_len ? a.q_len : count);
}

// per-queue selection state of one warp
template <int POLICY>
struct SelState {
    Thr thr;
    int cnt;
    int cuts;        // quickselect cuts taken inside this queue
    uint32_t seed;
};

// scan one chunk: `nvalid` records, the first one is record `rec0` of the queue.  The chunk
// sits in a shared-memory stage, or (GUARDED) in global memory, where nothing past nvalid is read.
template <int POLICY, bool INDIRECT, bool FULL, bool GUARDED = false>
__device__ __forceinline__ void scan_chunk(const int4 *__restrict__ stage, int4 *buf, int rec0, int nvalid,
                                           int32_t idx_base, int k, int64_t now, SelState<POLICY> &s) {
    const int lane = lane_id();
    const uint32_t lt_mask = (1u << lane) - 1u;
#pragma unroll
    for (int i = 0; i < SEL_CHUNK / 32; i += SEL_UNROLL) {
        if (!FULL && i * 32 >= nvalid) break;
        int4 r[SEL_UNROLL];
        uint32_t m[SEL_UNROLL];
        bool p[SEL_UNROLL];
#pragma unroll
        for (int u = 0; u < SEL_UNROLL; ++u) {
            if (GUARDED) r[u] = (i + u) * 32 + lane < nvalid ? __ldg(stage + (i + u) * 32 + lane) : make_int4(0, 0, 0, 0);
            else r[u] = stage[(i + u) * 32 + lane];
        }
        uint32_t many = 0;
#pragma unroll
        for (int u = 0; u < SEL_UNROLL; ++u) {
            p[u] = may_beat<POLICY>(rec_arr(r[u]), r[u].w, s.thr, now);
            if (!FULL) p[u] = p[u] && ((i + u) * 32 + lane < nvalid);
            m[u] = __ballot_sync(ASR_FULL_MASK, p[u]);
            many |= m[u];
        }
        if (many == 0u) continue;
#pragma unroll
        for (int half = 0; half < SEL_UNROLL; half += 2) {
            if ((m[half] | m[half + 1]) == 0u) continue;
#pragma unroll
            for (int u = half; u < half + 2; ++u) {
                if (p[u]) {
                    const int32_t idx = INDIRECT ? r[u].z : idx_base + rec0 + (i + u) * 32 + lane;
                    buf[s.cnt + __popc(m[u] & lt_mask)] = make_int4(r[u].x, r[u].y, r[u].w < 1 ? 1 : r[u].w, idx);
                }
                s.cnt += __popc(m[u]);
            }
            if (s.cnt > SEL_FLUSH_AT) {
                // keep the best 2k .. 2k+16: the survivors of a queue's last cut seed the carried threshold
                s.seed = s.seed * 747796405u + 2891336453u;
                __syncwarp();
                const uint32_t rc = buffer_cut<POLICY>(buf, s.cnt, 2 * k - 1, 2 * k + 15, now, s.seed);
                s.cnt = (int)(rc & 0xFFFFu);
                s.thr = thr_from<POLICY>(buf[rc >> 16], now);
                s.cuts++;
            }
        }
    }
}

// second reading of a whole queue straight from global memory with "pass everything" (cold path)
template <int POLICY>
__device__ __noinline__ void rescan_queue(const int4 *keys, int4 *buf, int count, int32_t idx_base, int k, int64_t now,
                                          SelState<POLICY> &s) {
    s.thr = thr_pass_all<POLICY>();
    s.cnt = 0;
    for (int c = 0; c * SEL_CHUNK < count; ++c) {
        const int left = count - c * SEL_CHUNK;
        scan_chunk<POLICY, false, false, true>(keys + (int64_t)c * SEL_CHUNK, buf, c * SEL_CHUNK,
                                               left < SEL_CHUNK ? left : SEL_CHUNK, idx_base, k, now, s);
    }
}

// cut to the k best, sort them, write the indices of queue q; decide what the next queue starts with
template <int POLICY>
__device__ __forceinline__ void finish_queue(SelWarpSmem &sm, int32_t *out, int k, int64_t now, SelState<POLICY> &s,
                                             bool steady) {
    const int lane = lane_id();
    int4 *buf = sm.buf;
    __syncwarp();
    if (steady) {
        // the carried threshold let s.cnt >= k records through and no cut was needed: keep it
        // unless it is getting close to letting fewer than k through
        if (s.cnt < k + (k >> 1) && lane == 0) sm.carry_ok = 0;
    } else if (s.cnt >= 2 * k) {
        // calibrate: the record of rank 2k .. 2k+16 of this queue becomes the carried threshold
        s.seed = s.seed * 747796405u + 2891336453u;
        const uint32_t rc = buffer_cut<POLICY>(buf, s.cnt, 2 * k - 1, 2 * k + 15, now, s.seed);
        s.cnt = (int)(rc & 0xFFFFu);
        const Thr c = thr_from<POLICY>(buf[rc >> 16], now);
        if (lane == 0) {
            sm.carry_t64 = c.t64;
            sm.carry_t32 = c.t32;
            sm.carry_ok = 1;
        }
    } else if (lane == 0) {
        sm.carry_ok = 0;
    }
    if (s.cnt > k) {
        s.seed = s.seed * 747796405u + 2891336453u;
        s.cnt = (int)(buffer_cut<POLICY>(buf, s.cnt, k - 1, k - 1, now, s.seed) & 0xFFFFu);
    }
    const int pos = sort32<POLICY>(buf, s.cnt, now);
    if (lane < k) out[lane] = pos >= 0 ? buf[pos].w : -1;
    __syncwarp();
}

template <int POLICY, bool INDIRECT>
__global__ void __launch_bounds__(SEL_WARPS * 32, 1) select_topk_kernel(SelArgs a) {
    extern __shared__ __align__(128) unsigned char sel_dyn_smem[];
    SelWarpSmem *smem = reinterpret_cast<SelWarpSmem *>(sel_dyn_smem);
    const int lane = lane_id();
    const int warp = threadIdx.x >> 5;
    SelWarpSmem &sm = smem[warp];
    const int k = a.k;
    const int gw = blockIdx.x * SEL_WARPS + warp;
    const int GW = gridDim.x * SEL_WARPS;

    if (!INDIRECT) {
        if (threadIdx.x == 0) {
            for (int w = 0; w < SEL_WARPS; ++w)
                for (int s = 0; s < SEL_STAGES; ++s) mbar_init(&smem[w].full[s], 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncthreads();
    }

    // producer cursor: the next chunk to fetch is chunk pc of queue pq (pq >= n_queues: no more)
    int pq = gw - GW, pc = 0, pn = 0, pcnt = 0;
    auto next_chunk = [&]() {   // move to the next chunk that exists, skipping empty queues
        while (pc >= pn) {
            pq += GW;
            if (pq >= a.n_queues) return;
            pcnt = sel_count(a, pq);
            pn = (pcnt + SEL_CHUNK - 1) / SEL_CHUNK;
            pc = 0;
        }
    };
    auto produce = [&](uint32_t g) {
        if (pq >= a.n_queues) return;
        const int st = (int)(g % SEL_STAGES);
        const int left = pcnt - pc * SEL_CHUNK;
        const uint32_t bytes = (uint32_t)(left < SEL_CHUNK ? left : SEL_CHUNK) * 16u;
        if (lane == 0) {
            mbar_expect_tx(&sm.full[st], bytes);
            bulk_g2s(sm.stage[st], a.keys + (int64_t)pq * a.q_len + (int64_t)pc * SEL_CHUNK, bytes, &sm.full[st]);
        }
        pc++;
        next_chunk();
    };

    uint32_t gp = 0, gc = 0;
    if (!INDIRECT) {
        next_chunk();
#pragma unroll 1
        for (int s = 0; s < SEL_STAGES; ++s) produce(gp++);
    }

    if (lane == 0) sm.carry_ok = 0;   // threshold carried from this warp's previous queue: none yet
    __syncwarp();
    for (int q = gw; q < a.n_queues; q += GW) {
        const int count = sel_count(a, q);
        const int64_t now = a.now_per_queue ? a.now_per_queue[q] : a.now;
        const int64_t qbase = (int64_t)q * a.q_len;
        const int32_t idx_base = a.global_idx ? (int32_t)qbase : 0;
        SelState<POLICY> s;
        const bool have_carry = sm.carry_ok != 0;
        s.thr = thr_pass_all<POLICY>();
        if (have_carry) {
            s.thr.t64 = sm.carry_t64;
            s.thr.t32 = sm.carry_t32;
        }
        s.cnt = 0;
        s.cuts = 0;
        s.seed = 0x9E3779B9u * (uint32_t)(q + 1);
        const int nch = (count + SEL_CHUNK - 1) / SEL_CHUNK;
        bool redo = false;
        for (;;) {
#pragma unroll 1
            for (int c = 0; c < nch; ++c) {
                const int left = count - c * SEL_CHUNK;
                const int nvalid = left < SEL_CHUNK ? left : SEL_CHUNK;
                if (INDIRECT) {
                    __syncwarp();
                    for (int j = lane; j < nvalid; j += 32) {
                        const int32_t src = a.src_idx[qbase + (int64_t)c * SEL_CHUNK + j];
                        const int4 v = __ldg(reinterpret_cast<const int4 *>(a.keys + src));
                        sm.stage[0][j] = make_int4(v.x, v.y, src, v.w);
                    }
                    __syncwarp();
                    scan_chunk<POLICY, true, false>(sm.stage[0], sm.buf, c * SEL_CHUNK, nvalid, idx_base, k, now, s);
                } else {
                    const int st = (int)(gc % SEL_STAGES);
                    mbar_wait(&sm.full[st], (gc / SEL_STAGES) & 1u);
                    if (nvalid == SEL_CHUNK)
                        scan_chunk<POLICY, false, true>(sm.stage[st], sm.buf, c * SEL_CHUNK, nvalid, idx_base, k, now, s);
                    else
                        scan_chunk<POLICY, false, false>(sm.stage[st], sm.buf, c * SEL_CHUNK, nvalid, idx_base, k, now, s);
                    __syncwarp();          // every lane is done reading the stage: refill it
                    produce(gp++);
                    gc++;
                }
            }
            // a carried threshold that let fewer than min(k, count) records through was too strict
            // for this queue: read it again with "pass everything"
            if (redo || !have_carry || s.cuts > 0 || s.cnt >= (k < count ? k : count)) break;
            redo = true;
            if (!INDIRECT) {
                rescan_queue<POLICY>(reinterpret_cast<const int4 *>(a.keys + qbase), sm.buf, count, idx_base, k, now, s);
                break;
            }
            s.thr = thr_pass_all<POLICY>();
            s.cnt = 0;
        }
        finish_queue<POLICY>(sm, a.out_idx + (int64_t)q * k, k, now, s, have_carry && !redo && s.cuts == 0);
    }
}

template <int POLICY, bool INDIRECT>
static int launch_one(const SelArgs &a, cudaStream_t st) {
    if (a.n_queues <= 0 || a.k <= 0) return ASR_OK;
    // the opt-in to > 48 KB of dynamic shared memory is per device: set it on every launch (cheap)
    {
        cudaError_t e = cudaFuncSetAttribute(select_topk_kernel<POLICY, INDIRECT>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SEL_SMEM_BYTES);
        if (e != cudaSuccess) {
            set_error("select_topk_kernel: cudaFuncSetAttribute: %s", cudaGetErrorString(e));
            cudaGetLastError();
            return ASR_ECUDA;
        }
    }
    const int n_sm = sm_count();
    // persistent: one CTA of SEL_WARPS queue-streams per SM
    const int64_t want = ((int64_t)a.n_queues + SEL_WARPS - 1) / SEL_WARPS;
    const int grid = (int)(want < (int64_t)n_sm ? want : (int64_t)n_sm);
    {
        KernelTimer kt(KID_SELECT, st);
        select_topk_kernel<POLICY, INDIRECT><<<grid, SEL_WARPS * 32, SEL_SMEM_BYTES, st>>>(a);
    }
    return check_launch("select_topk_kernel");
}

// ---------------------------------------------------------------------------
// 32 < k <= 256 (the engine admits into up to 256 slots): one CTA per queue.
// The queue goes through shared memory in chunks; a chunk joins the k best kept so far, the lot is sorted
// exactly (bitonic network on the order scalars, equal scalars settled by the full comparator with its
// (arrival, idx) tie-break), and the first k stay.  Not the streaming design of the k <= 32 kernel above: it
// trades bandwidth for a selection that needs no candidate buffer sized to k.
// ---------------------------------------------------------------------------
constexpr int WIDE_K = 256;
constexpr int WIDE_CAP = 4096;                 // entries sorted at a time (a power of two)
constexpr int WIDE_CHUNK = WIDE_CAP - WIDE_K;  // new records per round
constexpr int WIDE_THREADS = 512;

struct WideSmem {
    int4 ent[WIDE_CAP];       // (arrival lo, arrival hi, max(est,1), idx)
    int64_t key[WIDE_CAP];    // order scalar, INT64_MAX = padding
    uint16_t perm[WIDE_CAP];  // entry of rank i
    int4 tmp[WIDE_K];
    uint32_t hist[256];       // radix select of the k-th order scalar
    uint32_t wcnt[WIDE_THREADS / 32];
    uint32_t sel_digit, sel_below, n_cand;
};
constexpr int WIDE_SORT_MAX = 1024;   // a round with more entries first drops everything beyond the k-th order scalar

template <int POLICY>
__global__ void __launch_bounds__(WIDE_THREADS, 1) select_wide_kernel(SelArgs a) {
    extern __shared__ __align__(128) unsigned char sel_dyn_smem[];
    WideSmem &sm = *reinterpret_cast<WideSmem *>(sel_dyn_smem);
    const int tid = threadIdx.x;
    const int k = a.k;
    for (int q = blockIdx.x; q < a.n_queues; q += gridDim.x) {
        const int count = sel_count(a, q);
        const int64_t now = a.now_per_queue ? a.now_per_queue[q] : a.now;
        const int64_t qbase = (int64_t)q * a.q_len;
        const int32_t idx_base = a.global_idx ? (int32_t)qbase : 0;
        int kept = 0;   // entries [0, kept) = the best so far, best first
        for (int c0 = 0; c0 < count; c0 += WIDE_CHUNK) {
            const int nc = min(WIDE_CHUNK, count - c0);
            for (int j = tid; j < nc; j += WIDE_THREADS) {
                int4 v;
                int32_t idx;
                if (a.src_idx) {
                    idx = a.src_idx[qbase + c0 + j];
                    v = __ldg(reinterpret_cast<const int4 *>(a.keys + idx));
                } else {
                    idx = idx_base + c0 + j;
                    v = __ldg(reinterpret_cast<const int4 *>(a.keys + qbase + c0 + j));
                }
                sm.ent[kept + j] = make_int4(v.x, v.y, v.w < 1 ? 1 : v.w, idx);
            }
            __syncthreads();
            const int m = kept + nc;
            int size = 2;   // the power of two that holds m entries
            while (size < m) size <<= 1;
            for (int i = tid; i < size; i += WIDE_THREADS) {
                sm.key[i] = i < m ? order_scalar<POLICY>(sm.ent[i], now) : INT64_MAX;
                sm.perm[i] = (uint16_t)i;
            }
            __syncthreads();
            if (m > WIDE_SORT_MAX) {
                // Radix select (8 x 8 bits, MSB first) of the k-th smallest order scalar T.  Everything with a larger
                // scalar is worse than k entries (scalars are weakly order-preserving) and is dropped; what is left
                // (k entries and the ties at T) is compacted to the front and sorted.  Too many ties: sort it all.
                uint64_t prefix = 0;
                uint32_t kk = (uint32_t)k;
                for (int shift = 56; shift >= 0; shift -= 8) {
                    if (tid < 256) sm.hist[tid] = 0u;
                    __syncthreads();
                    for (int i = tid; i < m; i += WIDE_THREADS) {
                        const uint64_t u = (uint64_t)sm.key[i] ^ 0x8000000000000000ull;
                        if (shift == 56 || (u >> (shift + 8)) == prefix) atomicAdd(&sm.hist[(u >> shift) & 255u], 1u);
                    }
                    __syncthreads();
                    if (tid < 32) {   // lane L owns bins 8L .. 8L+7
                        uint32_t c8[8], tot = 0;
#pragma unroll
                        for (int b = 0; b < 8; ++b) {
                            c8[b] = sm.hist[tid * 8 + b];
                            tot += c8[b];
                        }
                        uint32_t incl = tot;
#pragma unroll
                        for (int d = 1; d < 32; d <<= 1) {
                            const uint32_t y = __shfl_up_sync(ASR_FULL_MASK, incl, d);
                            if (tid >= d) incl += y;
                        }
                        uint32_t run = incl - tot;
                        if (run < kk && kk <= incl) {
#pragma unroll
                            for (int b = 0; b < 8; ++b) {
                                if (run < kk && kk <= run + c8[b]) {
                                    sm.sel_digit = (uint32_t)(tid * 8 + b);
                                    sm.sel_below = run;
                                }
                                run += c8[b];
                            }
                        }
                    }
                    __syncthreads();
                    prefix = (prefix << 8) | sm.sel_digit;
                    kk -= sm.sel_below;
                }
                const int64_t T = (int64_t)(prefix ^ 0x8000000000000000ull);
                // compaction: every thread reads its eight entries, then writes the survivors to the front
                constexpr int PER = WIDE_CAP / WIDE_THREADS;
                int64_t ck[PER];
                uint16_t cp[PER];
                int nc_mine = 0;
#pragma unroll
                for (int j = 0; j < PER; ++j) {
                    const int i = tid * PER + j;
                    ck[j] = i < m ? sm.key[i] : INT64_MAX;
                    cp[j] = sm.perm[i];
                    if (i < m && ck[j] <= T) ++nc_mine;
                }
                uint32_t incl = (uint32_t)nc_mine;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const uint32_t y = __shfl_up_sync(ASR_FULL_MASK, incl, d);
                    if ((tid & 31) >= d) incl += y;
                }
                if ((tid & 31) == 31) sm.wcnt[tid >> 5] = incl;
                __syncthreads();
                uint32_t off = incl - (uint32_t)nc_mine, total = 0;
#pragma unroll
                for (int w = 0; w < WIDE_THREADS / 32; ++w) {
                    const uint32_t c = sm.wcnt[w];
                    if (w < (tid >> 5)) off += c;
                    total += c;
                }
                if (total <= (uint32_t)WIDE_SORT_MAX) {
                    size = 2;
                    while (size < (int)total) size <<= 1;
#pragma unroll
                    for (int j = 0; j < PER; ++j) {
                        const int i = tid * PER + j;
                        if (i < m && ck[j] <= T) {
                            sm.key[off] = ck[j];
                            sm.perm[off] = cp[j];
                            ++off;
                        }
                    }
                    __syncthreads();
                    for (int i = (int)total + tid; i < size; i += WIDE_THREADS) {
                        sm.key[i] = INT64_MAX;
                        sm.perm[i] = 0xFFFFu;   // a padding: ranks after every entry
                    }
                }
                __syncthreads();
            }
            for (int kk = 2; kk <= size; kk <<= 1) {
                for (int j = kk >> 1; j > 0; j >>= 1) {
                    for (int t = tid; t < (size >> 1); t += WIDE_THREADS) {
                        const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));   // the lower partner
                        const int l = i | j;
                        const bool up = (i & kk) == 0;
                        const int64_t ka = sm.key[i], kb = sm.key[l];
                        const uint16_t pa = sm.perm[i], pb = sm.perm[l];
                        // entry at i ranks before the entry at l?  (a padding ranks after everything; its scalar
                        // INT64_MAX is also that of a real HRRN entry that has not waited)
                        const bool pad_a = pa >= m, pad_b = pb >= m;
                        bool a_first;
                        if (pad_a || pad_b) {
                            a_first = !pad_a || pad_b;
                        } else if (ka != kb) {
                            a_first = ka < kb;
                        } else {
                            const int4 ea = sm.ent[pa], eb = sm.ent[pb];
                            a_first = better<POLICY>(rec_arr(ea), ea.z, ea.w, rec_arr(eb), eb.z, eb.w, now);
                        }
                        if (a_first != up) {
                            sm.key[i] = kb;
                            sm.key[l] = ka;
                            sm.perm[i] = pb;
                            sm.perm[l] = pa;
                        }
                    }
                    __syncthreads();
                }
            }
            kept = m < k ? m : k;
            if (tid < kept) sm.tmp[tid] = sm.ent[sm.perm[tid]];
            __syncthreads();
            if (tid < kept) sm.ent[tid] = sm.tmp[tid];
            __syncthreads();
        }
        int32_t *out = a.out_idx + (int64_t)q * k;
        for (int j = tid; j < k; j += WIDE_THREADS) out[j] = j < kept ? sm.ent[j].w : -1;
        __syncthreads();
    }
}

template <int POLICY>
static int launch_wide(const SelArgs &a, cudaStream_t st) {
    if (a.n_queues <= 0 || a.k <= 0) return ASR_OK;
    cudaError_t e = cudaFuncSetAttribute(select_wide_kernel<POLICY>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)sizeof(WideSmem));
    if (e != cudaSuccess) {
        set_error("select_wide_kernel: cudaFuncSetAttribute: %s", cudaGetErrorString(e));
        cudaGetLastError();
        return ASR_ECUDA;
    }
    const int cap = sm_count() * 2;
    const int grid = a.n_queues < cap ? a.n_queues : cap;
    {
        KernelTimer kt(KID_SELECT_WIDE, st);
        select_wide_kernel<POLICY><<<grid, WIDE_THREADS, sizeof(WideSmem), st>>>(a);
    }
    return check_launch("select_wide_kernel");
}

int launch_select(const SelArgs &a, int policy, cudaStream_t st) {
    const bool ind = a.src_idx != nullptr;
    if (!ind && (reinterpret_cast<uintptr_t>(a.keys) & 15u) != 0) {
        set_error("select: keys must be 16-byte aligned");
        return ASR_EINVAL;
    }
    if (a.k > 32) {
        switch (policy) {
            case ASR_FCFS: return launch_wide<ASR_FCFS>(a, st);
            case ASR_SJF: return launch_wide<ASR_SJF>(a, st);
            case ASR_HRRN: return launch_wide<ASR_HRRN>(a, st);
        }
        set_error("unknown policy %d", policy);
        return ASR_EINVAL;
    }
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
    if (k > ASR_SELECT_MAX_K) {
        set_error("select_batched: k=%d exceeds the limit %d", k, ASR_SELECT_MAX_K);
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

// valid prefix of a level array: every segment but the last reports k indices
static int64_t level_valid(int64_t len, int64_t segs, int64_t k) {
    const int64_t last = len - (segs - 1) * SEL_SEG;
    return (segs - 1) * k + (last < k ? last : k);
}

extern "C" int asr_sched_select(const asr_req_t *keys, int64_t n, int32_t policy, int64_t now, int32_t k,
                                int32_t *out_idx, void *workspace, size_t workspace_bytes, void *stream) {
    if (n < 0 || k < 0 || policy < 0 || policy > 2 || n >= (1ll << 31)) {
        set_error("select: bad argument (n=%lld k=%d policy=%d)", (long long)n, k, policy);
        return ASR_EINVAL;
    }
    if (k > ASR_SELECT_MAX_K) {
        set_error("select: k=%d exceeds the limit %d", k, ASR_SELECT_MAX_K);
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
    // further levels: select among the reported candidates (the -1 padding of a
    // short last segment sits at the very end of the level, outside `len`)
    int64_t len = level_valid(n, segs, k);
    int64_t stride = segs * k;
    while (true) {
        int64_t nsegs = (len + SEL_SEG - 1) / SEL_SEG;
        int32_t *dst = nsegs == 1 ? out_idx : level + stride;
        SelArgs a{keys, level, nullptr, nullptr, dst, now, len, (int32_t)nsegs, (int32_t)SEL_SEG, k, 0};
        int rc = launch_select(a, policy, st);
        if (rc) return rc;
        if (nsegs == 1) break;
        level = dst;
        len = level_valid(len, nsegs, k);
        stride = nsegs * k;
    }
    return ASR_OK;
}

// ---------------------------------------------------------------------------
// asr_sched_select_static: asr_sched_select for callers that cannot allocate (code under CUDA graph capture,
// serving loops, harnesses that forbid cudaMalloc).  The level arrays of the single-queue reduction tree live in a
// file-scope device array instead of a caller's workspace.  Every GPU that loads the library holds the array until
// exit; every call on a device shares it, so calls that overlap on the GPU (two streams) race.  Nothing in it has
// to start at zero: every level entry that is read was written by the launch before (-1 padding included).
// ---------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_select_scratch[ASR_SELECT_STATIC_SCRATCH_BYTES];

// In host code `g_select_scratch` is a host-side stand-in, not a device address: the address on the current device
// comes from cudaGetSymbolAddress, once per device.
static int select_scratch_ptr(void **out) {
    constexpr int MAX_DEV = 64;
    static std::mutex mu;
    static void *ptr[MAX_DEV] = {nullptr};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= MAX_DEV) {
        set_error("select_static: cudaGetDevice: %s (device %d)", cudaGetErrorString(e), dev);
        cudaGetLastError();
        return ASR_ECUDA;
    }
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_select_scratch);
        if (e != cudaSuccess || !p) {
            set_error("select_static: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
            cudaGetLastError();
            return ASR_ECUDA;
        }
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return ASR_OK;
}

extern "C" int asr_sched_select_static(const asr_req_t *keys, int64_t n, int32_t policy, int64_t now, int32_t k,
                                       int32_t *out_idx, void *stream) {
    if (n >= 0 && k >= 0 && k <= ASR_SELECT_MAX_K && select_ws_bytes(n, k) > (size_t)ASR_SELECT_STATIC_SCRATCH_BYTES) {
        set_error("select_static: n=%lld k=%d needs %zu bytes of scratch, the built-in array holds %d", (long long)n, k,
                  select_ws_bytes(n, k), (int)ASR_SELECT_STATIC_SCRATCH_BYTES);
        return ASR_EUNSUPPORTED;
    }
    void *scratch = nullptr;
    if (n > SEL_SEG && k > 0 && k <= ASR_SELECT_MAX_K) {   // (a queue of one segment needs no scratch)
        const int rc = select_scratch_ptr(&scratch);
        if (rc) return rc;
    }
    return asr_sched_select(keys, n, policy, now, k, out_idx, scratch, scratch ? (size_t)ASR_SELECT_STATIC_SCRATCH_BYTES : 0,
                            stream);
}

namespace asr {
size_t select_workspace_bytes(int64_t n, int64_t k) { return select_ws_bytes(n, k); }
}

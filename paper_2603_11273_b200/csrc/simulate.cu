// simulate.cu -- a4 simulator step + a5 per-request outputs, sm_100a.
//
// One warp owns one replica (seed x rate x policy).  Lane L holds batch slots
// L, L+32, ... in registers (remaining tokens, request index, arrival), so the
// per-iteration work of the paper's engine (PAPER.md:31 iteration-level
// scheduling; PAPER.md:51-53 encoder + linear decode) is a handful of
// warp-wide instructions: redux.min for the next completion, ballots for
// arrivals and finishes.
//
// Exact fast-forward.  Between two events (an admission opportunity or a
// completion) every engine iteration is identical: cost c = iter_base +
// iter_per_running*|R| and one token for everyone.  The kernel jumps j such
// iterations at once, j = min(iterations to the first completion, iterations
// to the first boundary at or after the next arrival when a slot is free),
// which is bit-identical to stepping them one by one.
//
// Waiting queue.  Requests are ingested in trace order, so the waiting set is
// {i in [lo, p) : not admitted(i)}.  While it is a dense range (always for
// FCFS, and whenever everything waiting is admitted at once) no queue storage
// is touched at all.  Otherwise a per-replica bitmap in the workspace marks
// admitted requests and the admit step scans the trace window [lo, p) with
// coalesced 128-bit loads, applying the exact comparator of asr_sched.h.
#include "sim_common.cuh"
#ifdef LANE_STATS
#include <cstdio>
#endif

namespace asr {

// the plain scan of the whole window (a window that outgrew the ring while the CTA tier is switched off)
__device__ __noinline__ void window_full_scan(const asr_req_t *trace, const uint32_t *bm, int lo, int p, int policy,
                                              int64_t t, int64_t *o_arr_, int32_t *o_est_, int32_t *o_dur_, int32_t *o_idx_) {
    const int lane = lane_id();
    int64_t b_arr = 0;
    int32_t b_est = 0, b_dur = 0, b_idx = -1;
    for (int c = lo & ~31; c < p; c += 32) {
        const uint32_t word = bm[c >> 5];
        const int i = c + lane;
        if (i >= lo && i < p && !((word >> lane) & 1u)) {
            const Rec q = ld_cached(trace + i);
            if (b_idx < 0 || better_rt(policy, q.arrival_us, q.est, i, b_arr, b_est, b_idx, t)) {
                b_arr = q.arrival_us;
                b_est = q.est;
                b_dur = q.dur_ms;
                b_idx = i;
            }
        }
    }
    for (int j = 16; j > 0; j >>= 1) {
        const int64_t o_arr = (int64_t)shfl64_xor((uint64_t)b_arr, j);
        const int32_t o_est = __shfl_xor_sync(ASR_FULL_MASK, b_est, j);
        const int32_t o_dur = __shfl_xor_sync(ASR_FULL_MASK, b_dur, j);
        const int32_t o_idx = __shfl_xor_sync(ASR_FULL_MASK, b_idx, j);
        if (o_idx >= 0 && (b_idx < 0 || better_rt(policy, o_arr, o_est, o_idx, b_arr, b_est, b_idx, t))) {
            b_arr = o_arr;
            b_est = o_est;
            b_dur = o_dur;
            b_idx = o_idx;
        }
    }
    *o_arr_ = b_arr;
    *o_est_ = b_est;
    *o_dur_ = b_dur;
    *o_idx_ = b_idx;
}

// one warp simulates replica r from start to end; ring = the warp's chunk bounds (shared memory)
template <int SPL>
__device__ __forceinline__ void sim_warp_replica(const SimArgs &a, const int r, ChunkMeta *ring) {
    const int lane = lane_id();
    const uint32_t lt_mask = (1u << lane) - 1u;

    const asr_replica_t rep = a.replicas[r];
    const int n = rep.n;
    const int slots = rep.slots;
    const int policy = rep.policy;
    if (!replica_ok(a, rep, 32 * SPL)) {
        if (lane == 0) flag_invalid(a, r);
        return;
    }
    const asr_cost_model_t cm = a.cms[rep.cm_id];
    const asr_req_t *trace = a.traces + rep.trace_off;
    int64_t *lat = a.out_lat + rep.out_off;
    int64_t *ttft = a.out_ttft + rep.out_off;
    uint32_t *bm = a.bitmap + a.bm_off[r];

    // running set: slot id = s*32 + lane
    int32_t rem[SPL];
    int32_t ridx[SPL];
    int64_t rarr[SPL];
#pragma unroll
    for (int s = 0; s < SPL; ++s) {
        rem[s] = REM_FREE;
        ridx[s] = -1;
        rarr[s] = 0;
    }

    int64_t t = 0;
    int p = 0;        // next request to ingest
    int lo = 0;       // every request below lo has been admitted
    int nW = 0;       // waiting requests
    int nR = 0;       // running requests
    int done = 0;
    bool sparse = false;  // bitmap in use for [lo, bm_hi)
    int bm_hi = 0;
    bool meta_ok = false; // the chunk bounds cover the window [lo, bm_hi)

    // arrival stamps (and est: the chunk bounds want it) of the trace chunk [cbase, cbase+32)
    int cbase = 0;
    int64_t carr = 0;
    int32_t cest = 0;
    if (lane < n) {
        const Rec q = ld_cached(trace + lane);
        carr = q.arrival_us;
        cest = q.est;
    }
    const int64_t first_arrival = n > 0 ? shfl64(carr, 0) : 0;

    while (done < n) {
        // ---- 1. ingest arrivals <= t (at the iteration boundary)
        while (p < n) {
            if (p >= cbase + 32) {
                cbase = p & ~31;
                carr = 0;
                if (cbase + lane < n) {
                    const Rec q = ld_cached(trace + cbase + lane);
                    carr = q.arrival_us;
                    cest = q.est;
                }
            }
            const int i = cbase + lane;
            uint32_t m = __ballot_sync(ASR_FULL_MASK, i >= p && i < n && carr <= t);
            int cnt = __popc(m);
            if (cnt > 0 && sparse && meta_ok) {
                // the newcomers join their chunk's bounds (a chunk is first touched at its first request)
                const int32_t e_new = __reduce_min_sync(ASR_FULL_MASK, ((m >> lane) & 1u) ? (int32_t)est_of(cest) : INT32_MAX);
                const int64_t a_new = shfl64(carr, __ffs(m) - 1);
                if (lane == 0) {
                    ChunkMeta *slot = ring + ((cbase >> 5) % CHUNK_RING);
                    ChunkMeta mt = *slot;
                    if (p == cbase) mt.wait = 0u;
                    if (mt.wait == 0u) {
                        mt.a_first = a_new;
                        mt.e_min = e_new;
                    } else {
                        mt.e_min = e_new < mt.e_min ? e_new : mt.e_min;
                    }
                    mt.wait |= m;
                    *slot = mt;
                }
                __syncwarp();
            }
            p += cnt;
            nW += cnt;
            if (cnt == 0 || p < cbase + 32) break;
        }
        if (p < n && p >= cbase + 32) {
            cbase = p & ~31;
            carr = 0;
            if (cbase + lane < n) {
                const Rec q = ld_cached(trace + cbase + lane);
                carr = q.arrival_us;
                cest = q.est;
            }
        }
        // ---- 2. idle server: jump to the next arrival
        if (nR == 0 && nW == 0) {
            t = shfl64(carr, p - cbase);
            continue;
        }
        // ---- 3. admit the k best waiting requests into the free slots
        const int free_slots = slots - nR;
        const int k = free_slots < nW ? free_slots : nW;
        uint32_t newly = 0;        // bit s: my slot s was admitted in this step
        uint32_t dur_sum_part = 0; // my share of sum(dur_ms) of the admitted
        if (k > 0) {
            const bool take_all = (k == nW);
            if (!sparse && (take_all || policy == ASR_FCFS)) {
                // dense window: admit requests lo .. lo+k-1 (their order is irrelevant
                // to every time; only the set matters, S15)
                int before = 0;
#pragma unroll
                for (int s = 0; s < SPL; ++s) {
                    const bool is_free = (s * 32 + lane < slots) && rem[s] == REM_FREE;
                    const uint32_t fm = __ballot_sync(ASR_FULL_MASK, is_free);
                    const int rank = before + __popc(fm & lt_mask);
                    if (is_free && rank < k) {
                        const Rec q = ld_cached(trace + lo + rank);
                        rem[s] = tokens_of(cm, q.dur_ms);
                        ridx[s] = lo + rank;
                        rarr[s] = q.arrival_us;
                        dur_sum_part += (uint32_t)q.dur_ms;
                        newly |= 1u << s;
                    }
                    before += __popc(fm);
                }
                lo += k;
                nW -= k;
            } else {
                // sparse window: bitmap marks the admitted requests of [lo, p)
                if (p - lo > a.escalate_window) {
                    // a backlog this deep is re-scanned for every admission: the CTA kernel
                    // (candidate pool in shared memory) takes the replica over, from the start
                    if (lane == 0) a.defer2_list[atomicAdd(a.defer2_count, 1)] = r;
                    return;
                }
                const int c_lo = lo >> 5, c_hi = (p - 1) >> 5;
                const bool ringed = c_hi - c_lo + 1 <= CHUNK_RING - 1;   // else the plain scan of the whole window
                if (!sparse) {
                    for (int w = (lo >> 5) + lane; w <= ((p - 1) >> 5); w += 32) bm[w] = 0u;
                    sparse = true;
                    bm_hi = p;
                    meta_ok = false;
                    __syncwarp();
                } else if (bm_hi < p) {
                    // clear the bits of the newly ingested requests [bm_hi, p)
                    const int w0 = bm_hi >> 5, w1 = (p - 1) >> 5;
                    for (int w = w0 + lane; w <= w1; w += 32) {
                        if (w == w0) {
                            if (bm_hi & 31) bm[w] &= (1u << (bm_hi & 31)) - 1u;
                            else bm[w] = 0u;
                        } else {
                            bm[w] = 0u;
                        }
                    }
                    bm_hi = p;
                    __syncwarp();
                }
                if (!ringed) {
                    meta_ok = false;
                } else if (!meta_ok) {
                    for (int c = c_lo; c <= c_hi; ++c) chunk_rebuild(trace, bm, ring, c, lo, p, lane);
                    meta_ok = true;
                    __syncwarp();
                }
                for (int round = 0; round < k; ++round) {
                    int64_t b_arr = 0;
                    int32_t b_est = 0, b_dur = 0, b_idx = -1;
                    if (!ringed) {
                        window_full_scan(trace, bm, lo, p, policy, t, &b_arr, &b_est, &b_dur, &b_idx);
                    } else {
                        chunk_pick(trace, ring, c_lo, c_hi, policy, t, lane, b_arr, b_est, b_dur, b_idx);
                    }
                    // b_* now uniform: the winner.  Mark it and seat it in the first free slot.
                    if (lane == 0) {
                        bm[b_idx >> 5] |= 1u << (b_idx & 31);
                        if (ringed) ring[(b_idx >> 5) % CHUNK_RING].wait &= ~(1u << (b_idx & 31));
                    }
                    bool seated = false;
#pragma unroll
                    for (int s = 0; s < SPL; ++s) {
                        const bool is_free = (s * 32 + lane < slots) && rem[s] == REM_FREE;
                        const uint32_t fm = __ballot_sync(ASR_FULL_MASK, is_free);
                        if (!seated && fm != 0u) {
                            if (lane == __ffs(fm) - 1) {
                                rem[s] = tokens_of(cm, b_dur);
                                ridx[s] = b_idx;
                                rarr[s] = b_arr;
                                dur_sum_part += (uint32_t)b_dur;
                                newly |= 1u << s;
                            }
                            seated = true;
                        }
                    }
                    __syncwarp();
                }
                nW -= k;
                if (nW == 0) {
                    lo = p;
                    sparse = false;
                } else {
                    // advance lo past admitted requests
                    while (lo < p) {
                        uint32_t word = ~bm[lo >> 5] & ~((1u << (lo & 31)) - 1u);
                        if (word) {
                            lo = (lo & ~31) + __ffs(word) - 1;
                            break;
                        }
                        lo = (lo & ~31) + 32;
                    }
                    if (lo > p) lo = p;
                }
            }
            nR += k;
        }
        // ---- 4. one engine iteration with the encoders of the admitted ...
        const int64_t c = cm.iter_base_us + cm.iter_per_running_us * (int64_t)nR;
        int64_t t1 = t + c;
        if (k > 0) {
            const int64_t dur_sum = warp_sum_u32(dur_sum_part);
            t1 += cm.enc_base_us * (int64_t)k + cm.enc_per_ms_us * dur_sum;
#pragma unroll
            for (int s = 0; s < SPL; ++s)
                if ((newly >> s) & 1u) ttft[ridx[s]] = t1 - rarr[s];   // first token (S9)
        }
        // ---- ... then fast-forward over identical iterations to the next event
        int32_t my_min = rem[0];
#pragma unroll
        for (int s = 1; s < SPL; ++s) my_min = rem[s] < my_min ? rem[s] : my_min;
        const int32_t m = __reduce_min_sync(ASR_FULL_MASK, my_min);   // >= 1, nR >= 1 here
        int64_t j = 1;
        if (m > 1) {
            if (nR == slots || p >= n || c <= 0) {
                j = m;   // nothing can be admitted before the first completion
            } else {
                const int64_t g = shfl64(carr, p - cbase) - t1;
                if (g <= 0) j = 1;
                else if (g > (int64_t)(m - 2) * c) j = m;
                else j = 1 + ceil_div_pos(g, c);
            }
        }
        t = t1 + (j - 1) * c;
        // ---- 5. tokens, completions (a5: E2E latency)
        int fin = 0;
#pragma unroll
        for (int s = 0; s < SPL; ++s) {
            if (rem[s] != REM_FREE) {
                rem[s] -= (int32_t)j;
                if (rem[s] == 0) {
                    lat[ridx[s]] = t - rarr[s];
                    rem[s] = REM_FREE;
                    fin++;
                }
            }
        }
        const int nfin = __reduce_add_sync(ASR_FULL_MASK, fin);
        nR -= nfin;
        done += nfin;
    }
    if (a.out_summary && lane == 0) {
        asr_summary_t *s = a.out_summary + r;
        s->first_arrival_us = first_arrival;
        s->last_done_us = t;
        s->n_done = done;
    }
}

// warp-per-replica kernel.  Direct mode: warp w of the grid simulates replica w.
// Worklist mode (a.defer_list != nullptr): the warps share the replicas that the
// lane kernel below handed over, defer_list[0 .. *defer_count).
#ifndef SIM_WARP_MIN_CTAS
#define SIM_WARP_MIN_CTAS 6
#endif
// PACKED: the work-list pass behind the thread tier (thousands of contended replicas: occupancy pays for the
// registers given up); the direct pass over a few replicas keeps every register
template <int SPL, bool PACKED>
__global__ void __launch_bounds__(SIM_WARPS * 32, PACKED ? SIM_WARP_MIN_CTAS : 1) sim_warp_kernel(SimArgs a) {
    __shared__ ChunkMeta s_ring[SIM_WARPS][CHUNK_RING];
    ChunkMeta *ring = s_ring[threadIdx.x >> 5];
    const int gw = (blockIdx.x * SIM_WARPS) + (threadIdx.x >> 5);
    if (a.defer_list == nullptr) {
        if (gw < a.n_replicas) sim_warp_replica<SPL>(a, gw, ring);
        return;
    }
    // the hand-over list is in the order the thread tier gave up: replicas that had to choose early -- the long
    // ones -- first; warps take the next one as they finish (defer_count[4] = the cursor)
    const int cnt = *a.defer_count;
    while (true) {
        int w = 0;
        if (lane_id() == 0) w = atomicAdd(a.defer_count + 4, 1);
        w = __shfl_sync(ASR_FULL_MASK, w, 0);
        if (w >= cnt) break;
        sim_warp_replica<SPL>(a, a.defer_list[w], ring);
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------
// lane-per-replica kernel: ONE THREAD simulates one replica.
//
// At the loads of the replica sweep (0.5-4 req/s against a capacity of 10-27
// req/s) a replica has a handful of running requests, so a warp-wide running
// set leaves most lanes idle.  Here every lane runs its own event loop: the
// running set is a compact array of (finish iteration, request index) pairs
// in shared memory, laid out [slot][thread] so that lane accesses never
// conflict; the trace is read with 16-byte loads.  "Finish iteration" is the
// engine-iteration counter at which the request emits its last token
// (counter at admission + tokens), kept modulo 2^32: remaining = fin - it is
// exact because remaining < 2^31.  The fast-forward is the one of the warp
// kernel.  The three policy replicas of one trace sit in adjacent lanes and
// read the same addresses.
//
// Only the uncontended regime is handled here: as soon as SJF/HRRN must CHOOSE
// (more waiting than free slots), the thread appends its replica to defer_list
// and stops; the warp kernel then simulates that replica from the start with
// its coalesced window scan.  Results are identical either way.
// ---------------------------------------------------------------------------
#ifndef LANE_THREADS_N
#define LANE_THREADS_N 64
#endif
constexpr int LANE_THREADS = LANE_THREADS_N;
constexpr int LANE_BLOCKS_PER_SM = 768 / LANE_THREADS;
constexpr int LANE_CAP = 32;   // slots per replica handled by the lane kernel

__device__ __forceinline__ int64_t ld_arrival(const asr_req_t *p) {
    return __ldg(reinterpret_cast<const long long *>(p));
}

__device__ __forceinline__ uint32_t lane_tokens(int64_t tok_base, int64_t tok_per_s, int32_t dur_ms) {
    const int64_t prod = tok_per_s * (int64_t)dur_ms;
    int64_t tok = tok_base + (((uint64_t)prod >> 32) == 0 ? (int64_t)((uint32_t)prod / 1000u) : prod / 1000);
    tok = tok < 1 ? 1 : (tok > 0x7FFFFFFE ? 0x7FFFFFFE : tok);
    return (uint32_t)tok;
}

// the same for 0 <= tok_per_s < 2^31 and |tok_base| < 2^30: 32-bit arithmetic whenever the
// product fits (quotient < 4.3e6, so neither the sum nor the upper clamp can overflow)
__device__ __forceinline__ uint32_t lane_tokens_small(int32_t tok_base, uint32_t tok_per_s, int32_t dur_ms) {
    const uint64_t prod = (uint64_t)tok_per_s * (uint32_t)dur_ms;
    if (dur_ms >= 0 && (prod >> 32) == 0) {
        const int32_t tok = tok_base + (int32_t)((uint32_t)prod / 1000u);
        return (uint32_t)(tok < 1 ? 1 : tok);
    }
    return lane_tokens((int64_t)tok_base, (int64_t)tok_per_s, dur_ms);
}

// The ring is addressed with 32-bit shared-memory byte addresses: `sbase` is the thread's
// column, `hoff` the byte offset of the head entry (a multiple of RING_STEP below RING_BYTES).
constexpr uint32_t RING_STEP = LANE_THREADS * 8;            // one ring position, all threads
constexpr uint32_t RING_MASK = LANE_CAP * RING_STEP - 1;    // 16 KB ring per CTA

__device__ __forceinline__ uint2 ring_ld(uint32_t addr) {
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ void ring_st(uint32_t addr, uint2 v) {
    asm volatile("st.shared.v2.u32 [%0], {%1,%2};" ::"r"(addr), "r"(v.x), "r"(v.y));
}

// insert (it + tokens, payload) into the sorted ring of nR entries starting at the head;
// an entry is one 64-bit word (finish iteration, payload)
__device__ __forceinline__ void lane_insert(uint32_t sbase, uint32_t hoff, int nR, uint32_t it, uint32_t tokens,
                                            uint32_t payload) {
    uint32_t off = (hoff + (uint32_t)nR * RING_STEP) & RING_MASK;   // first free position
    int h = nR;
    while (h > 0) {
        const uint32_t prev = (off - RING_STEP) & RING_MASK;
        const uint2 e = ring_ld(sbase + prev);
        if (e.x - it <= tokens) break;
        ring_st(sbase + off, e);
        off = prev;
        --h;
    }
    ring_st(sbase + off, make_uint2(it + tokens, payload));
}

// TTFT of request idx (requests are admitted in index order here)
__device__ __forceinline__ void lane_push_ttft(int64_t *ttft, int idx, int64_t v, bool staged, int64_t &s0,
                                               int64_t &s1, int64_t &s2, int64_t &s3) {
    if (!staged) {
        ttft[idx] = v;
        return;
    }
    s0 = s1;
    s1 = s2;
    s2 = s3;
    s3 = v;
    if ((idx & 3) == 3) {
        longlong2 *dst = reinterpret_cast<longlong2 *>(ttft + idx - 3);
        dst[0] = make_longlong2(s0, s1);
        dst[1] = make_longlong2(s2, s3);
    }
}

// Order-free outputs (summary-only calls: the per-request arrays live in the workspace and
// only feed the percentile reduction, which does not care about their order).  Values
// known to be below 2^32 are staged in four registers and written as one aligned 16-byte
// store of four uint32 into the FIRST HALF of the replica's int64 region; the replica's
// summary carries ASR_FMT32 in its percentile fields so that the reduction reads that
// format.  `ph` is the element phase of base[0] within its 16-byte line.
struct Stage32 {
    uint32_t v0, v1, v2, v3;
};

__device__ __forceinline__ void stage_push(uint32_t *base, int ph, int pos, uint32_t v, Stage32 &s) {
    s.v0 = s.v1;
    s.v1 = s.v2;
    s.v2 = s.v3;
    s.v3 = v;
    if (((ph + pos) & 3) == 3) {
        if (pos >= 3) {
            *reinterpret_cast<uint4 *>(base + pos - 3) = make_uint4(s.v0, s.v1, s.v2, s.v3);
        } else {   // short head before the first 16-byte boundary
            if (pos >= 2) base[pos - 2] = s.v1;
            if (pos >= 1) base[pos - 1] = s.v2;
            base[pos] = s.v3;
        }
    }
}

__device__ __forceinline__ void stage_tail(uint32_t *base, int ph, int n, const Stage32 &s) {
    int cnt = (ph + n) & 3;
    cnt = cnt < n ? cnt : n;
    if (cnt >= 3) base[n - 3] = s.v1;
    if (cnt >= 2) base[n - 2] = s.v2;
    if (cnt >= 1) base[n - 1] = s.v3;
}

#ifdef LANE_SECTOR_STORES
// The same with whole 32-byte sectors (pieces): a quad that completes the FIRST half of a sector is parked in shared
// memory (`park`: 16 bytes of this thread and stream) and written together with the second half, as two 16-byte stores
// to one sector back to back.  A half-written sector that L2 evicts before its other half arrives costs a read and a
// second write in DRAM.  r02, config 3: 13.5 GB of DRAM traffic (1.03x the 13.1 GB the kernel has to move) and 16.06 ms
// this way, 19.0-20.5 GB (1.5x) and 15.4 ms with the 16-byte stores of Stage32 some 6 us apart -- the kernel is bound
// by its dependent instruction chains, not by HBM, and the parked quad's way back through shared memory sits on
// them.  Hence an opt-in (-DLANE_SECTOR_STORES), not the default.
// ph8 = the element phase of base[0] within its 32-byte sector.
__device__ __forceinline__ void stage8_push(uint32_t *base, int ph8, int pos, uint32_t v, Stage32 &s, uint32_t park) {
    s.v0 = s.v1;
    s.v1 = s.v2;
    s.v2 = s.v3;
    s.v3 = v;
    const int k = (ph8 + pos) & 7;
    if ((k & 3) == 3) {
        if (pos < 3) {   // short head before the first 16-byte boundary
            if (pos >= 2) base[pos - 2] = s.v1;
            if (pos >= 1) base[pos - 1] = s.v2;
            base[pos] = s.v3;
        } else if (k == 3) {
            asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(park), "r"(s.v0), "r"(s.v1), "r"(s.v2), "r"(s.v3) : "memory");
        } else {
            if (pos >= 7) {
                uint4 h;
                asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(h.x), "=r"(h.y), "=r"(h.z), "=r"(h.w) : "r"(park) : "memory");
                *reinterpret_cast<uint4 *>(base + pos - 7) = h;
            }
            *reinterpret_cast<uint4 *>(base + pos - 3) = make_uint4(s.v0, s.v1, s.v2, s.v3);
        }
    }
}

// after n pushes: a parked quad whose second half never came, and the values after the last whole quad
__device__ __forceinline__ void stage8_tail(uint32_t *base, int ph8, int n, const Stage32 &s, uint32_t park) {
    int cnt = (ph8 + n) & 3;
    cnt = cnt < n ? cnt : n;
    const int last = n - cnt - 1;   // the last element of the last whole quad (if last >= 3)
    if (last >= 3 && ((ph8 + last) & 7) == 3) {
        uint4 h;
        asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(h.x), "=r"(h.y), "=r"(h.z), "=r"(h.w) : "r"(park) : "memory");
        *reinterpret_cast<uint4 *>(base + last - 3) = h;
    }
    if (cnt >= 3) base[n - 3] = s.v1;
    if (cnt >= 2) base[n - 2] = s.v2;
    if (cnt >= 1) base[n - 1] = s.v3;
}
#endif

// FREE = order-free outputs: the ring carries the low word of the arrival time instead of
// the request index, E2E latency is formed at completion and both outputs are emitted in
// event order through Stage32.  Exact as long as every value is below 2^32 us, which the
// kernel proves with the start of the current busy period (every request in the system
// arrived at or after it); a busy period of 2^32 us sends the replica to the warp kernel.
#ifndef LANE_REGEN_HEAD_N
#define LANE_REGEN_HEAD_N 512
#endif
constexpr int LANE_REGEN_HEAD = LANE_REGEN_HEAD_N;   // requests at the head of a segment whose regeneration points are recorded
#ifdef LANE_STATS
// tuning builds: units run, units flagged, repairs run, repairs that found no common point, replicas redone,
// requests re-simulated by repairs
__device__ unsigned long long g_lane_stats[8];
#endif

__host__ __device__ __forceinline__ int lane_seg_len(int n, int nseg) {
    return (((n + nseg - 1) / nseg) + 31) & ~31;   // whole bitmap words per segment
}

// a thread simulates replica r from its first request to its last; all 32 lanes of a warp call it together (`live` =
// this lane has a replica).  sbase = the lane's column of the CTA's ring
template <bool FREE>
__device__ __forceinline__ void lane_run(const SimArgs &a, const uint32_t sbase, bool live, const int r) {
    // every lane of a warp stays in the loop below until the whole warp is done (the loop
    // re-converges the warp once per admission step); `live` marks the lanes with work
    bool valid = live;
    asr_replica_t rep;
    rep.trace_off = rep.out_off = 0;
    rep.n = 0;
    rep.policy = rep.cm_id = 0;
    rep.slots = 1;
    if (live) {
        rep = a.replicas[r];
        if (!replica_ok(a, rep, LANE_CAP)) {
            flag_invalid(a, r);
            live = valid = false;
            rep.cm_id = 0;
            rep.n = 0;
        }
    }
    const int n = rep.n, slots = rep.slots, policy = rep.policy;
    const asr_cost_model_t *cmp = a.cms + rep.cm_id;
    const int64_t enc_base64 = __ldg(&cmp->enc_base_us), enc_per64 = __ldg(&cmp->enc_per_ms_us);
    const int64_t iter_base64 = __ldg(&cmp->iter_base_us), iter_per64 = __ldg(&cmp->iter_per_running_us);
    const int32_t tok_base = __ldg(&cmp->tok_base), tok_per_s_i = __ldg(&cmp->tok_per_s);
    const uint32_t tok_per_s = (uint32_t)tok_per_s_i;
    // this kernel computes iteration costs in 32 bits; any other cost model goes to the warp kernel
    const int64_t lim31 = (int64_t)1 << 31;
    const bool small = enc_base64 >= 0 && enc_base64 < lim31 && enc_per64 >= 0 && enc_per64 < lim31 &&
                       iter_base64 >= 0 && iter_per64 >= 0 && iter_base64 + iter_per64 * LANE_CAP < lim31 &&
                       tok_per_s_i >= 0 && tok_base > -(1 << 30) && tok_base < (1 << 30);
    bool deferred = false;
    if (live && !small) {
        deferred = true;
        live = false;
    }
    const uint32_t enc_base = (uint32_t)enc_base64;
    const int32_t enc_per = (int32_t)enc_per64;
    const uint32_t ib = (uint32_t)iter_base64, ip = (uint32_t)iter_per64;
    const asr_req_t *trace = a.traces + rep.trace_off;
    int64_t *lat = a.out_lat + rep.out_off;
    int64_t *ttft = a.out_ttft + rep.out_off;

    int64_t t = 0;     // the current iteration boundary
    int64_t tb = 0;    // FREE: start of the current busy period (arrival of its first request)
    int p = 0, lo = 0, nW = 0, nR = 0, done = 0;
    uint32_t hoff = 0;   // running set = nR ring positions from byte offset hoff, sorted by finish iteration
    uint32_t it = 0;   // engine iterations so far, mod 2^32
    // look-ahead window over the trace: records p and p+1 are in registers (one 128-bit
    // load each: the memory pipeline is paid per lane and access, not per byte)
    int64_t arr0 = INT64_MAX, arr1 = INT64_MAX, last_arr = 0;
    int32_t dur0 = 0, dur1 = 0, last_dur = 0;
    // the est word of the load is kept live until the record is consumed: a dead destination
    // register would be reused, and its next writer would wait for the load in flight
    int32_t est1 = 0;
    if (live && n > 0) {
        const Rec q = ld_cached(trace);
        arr0 = q.arrival_us;
        dur0 = q.dur_ms;
    }
    if (live && n > 1) {
        const Rec q = ld_cached(trace + 1);
        arr1 = q.arrival_us;
        dur1 = q.dur_ms;
        est1 = q.est;
    }
    // !FREE: TTFT values are staged in registers and stored four at a time (requests
    // 4g .. 4g+3 as two 16-byte stores) when the output is 16-byte aligned
    int64_t st0 = 0, st1 = 0, st2 = 0, st3 = 0;
    const bool staged = (reinterpret_cast<uintptr_t>(ttft) & 15u) == 0;
    // FREE: both outputs through Stage32
    Stage32 sq_t = {0, 0, 0, 0}, sq_l = {0, 0, 0, 0};
    uint32_t *ttft32 = reinterpret_cast<uint32_t *>(ttft), *lat32 = reinterpret_cast<uint32_t *>(lat);
    const int ph_t = (int)((reinterpret_cast<uintptr_t>(ttft32) >> 2) & 3u);
    const int ph_l = (int)((reinterpret_cast<uintptr_t>(lat32) >> 2) & 3u);
    // (written now rather than carried through the loop: the kernel sits at its register limit)
    if (valid && a.out_summary) a.out_summary[r].first_arrival_us = n > 0 ? arr0 : 0;
    if (n == 0) live = false;

    // One trip of the outer loop = one admission step, so that the lanes of a warp (32
    // different replicas) stay in the same phase: A pops the completions that precede the
    // step, B moves the clock to its boundary, C ingests, D admits.
    while (true) {
        if (live) {
            // A. completions before the next admission opportunity.  With m iterations to the
            // head's last token at cost c each, the boundaries t + j*c, j < m, precede it: if a
            // slot is free and somebody is waiting, or the next arrival falls at or before
            // t + (m-1)*c, the admission step comes first.
            bool more = nR > 0;
            const int64_t a_eff = nW > 0 ? INT64_MIN : arr0;   // somebody waiting: admit at the first free slot
            while (more) {
                const uint2 e = ring_ld(sbase + hoff);   // sorted: the head finishes first
                const uint32_t f = e.x;
                const uint32_t m = f - it;
                const uint32_t c = ib + ip * (uint32_t)nR;
                const int64_t lim = t + (int64_t)((uint64_t)(m - 1u) * c);
                if (m > 0u && nR < slots && a_eff <= lim) {
                    more = false;
                } else {
                    if (m > 0u) {
                        t = lim + c;
                        it = f;
                    }
                    if (FREE) {
                        stage_push(lat32, ph_l, done, (uint32_t)t - e.y, sq_l);   // E2E = t - arrival
                    } else {
                        // lat[i] holds -arrival (sim_init_lat_kernel); a fire-and-forget reduction
                        // adds the completion time, so no load sits on the critical path
                        atomicAdd(reinterpret_cast<unsigned long long *>(lat + (int32_t)e.y),
                                  (unsigned long long)t);
                    }
                    hoff = (hoff + RING_STEP) & RING_MASK;
                    --nR;
                    ++done;
                    more = nR > 0;
                }
            }
            if (done >= n) live = false;
            // every value emitted so far (TTFT of the previous step, the latencies above) is at
            // most t - tb; beyond 32 bits the proof fails and the warp kernel redoes the replica
            if (FREE && ((uint64_t)(t - tb) >> 32) != 0) {
                deferred = true;
                live = false;
            }
        }
        if (!__any_sync(ASR_FULL_MASK, live)) break;   // also the warp's re-convergence point
        if (live) {
            // B. the boundary of the admission step
            if (nW == 0 && nR == 0) tb = arr0;   // a new busy period starts with the next arrival
            if (nW == 0 && arr0 > t) {
                if (nR == 0) {
                    t = arr0;   // idle server: the clock jumps to the next arrival (S14)
                } else {
                    const uint32_t c = ib + ip * (uint32_t)nR;
                    const int64_t j = ceil_div_pos(arr0 - t, (int64_t)c);   // c > 0: arr0 <= t + (m-1)*c
                    t += j * (int64_t)c;
                    it += (uint32_t)j;
                }
            }
            // C. ingest arrivals <= t
            while (arr0 <= t) {
                last_arr = arr0;
                last_dur = dur0;
                ++p;
                ++nW;
                arr0 = arr1;
                dur0 = dur1;
                // (a real, harmless use: a prefetch that is never issued; ptxas drops anything less)
                asm volatile("{ .reg .pred p; setp.eq.s32 p, %0, -2147483647; @p prefetch.global.L2 [%1]; }" ::"r"(est1),
                             "l"(trace));
                arr1 = INT64_MAX;
                if (p + 1 < n) {
                    const Rec q = ld_cached(trace + p + 1);
                    arr1 = q.arrival_us;
                    dur1 = q.dur_ms;
                    est1 = q.est;
                }
            }
            // D. admit k >= 1 requests (a slot is free and somebody waits)
            const int free_slots = slots - nR;
            const int k = free_slots < nW ? free_slots : nW;
            if (policy != ASR_FCFS && k < nW) {   // a real choice: hand over to the warp kernel
                deferred = true;
                live = false;
            } else {
                int64_t t1 = t + (int64_t)(ib + ip * (uint32_t)(nR + k));
                if (k == 1 && lo == p - 1) {
                    // the request ingested last: everything needed is in registers
                    lane_insert(sbase, hoff, nR, it, lane_tokens_small(tok_base, tok_per_s, last_dur),
                                FREE ? (uint32_t)last_arr : (uint32_t)lo);
                    t1 += (int64_t)enc_per * (int64_t)last_dur + (int64_t)enc_base;
                    // first token (S9)
                    if (FREE) stage_push(ttft32, ph_t, lo, (uint32_t)t1 - (uint32_t)last_arr, sq_t);
                    else lane_push_ttft(ttft, lo, t1 - last_arr, staged, st0, st1, st2, st3);
                } else {
                    int64_t dur_sum = 0;
                    for (int q = 0; q < k; ++q) {
                        const Rec rq = ld_cached(trace + lo + q);
                        lane_insert(sbase, hoff, nR + q, it, lane_tokens_small(tok_base, tok_per_s, rq.dur_ms),
                                    FREE ? (uint32_t)rq.arrival_us : (uint32_t)(lo + q));
                        dur_sum += (int64_t)rq.dur_ms;
                    }
                    t1 += (int64_t)enc_base * (int64_t)k + (int64_t)enc_per * dur_sum;
                    for (int q = 0; q < k; ++q) {
                        const int64_t arr = ld_arrival(trace + lo + q);
                        if (FREE) stage_push(ttft32, ph_t, lo + q, (uint32_t)t1 - (uint32_t)arr, sq_t);
                        else lane_push_ttft(ttft, lo + q, t1 - arr, staged, st0, st1, st2, st3);
                    }
                }
                lo += k;
                nW -= k;
                nR += k;
                t = t1;
                it += 1u;
            }
        }
    }
    if (deferred) {
        const int pos = atomicAdd(a.defer_count, 1);
        a.defer_list[pos] = r;
        if (FREE && a.out_summary) {   // the warp kernel will write int64 values
            a.out_summary[r].p50_e2e_us = 0;
            a.out_summary[r].p50_ttft_us = 0;
        }
        return;
    }
    if (valid && FREE) {
        stage_tail(ttft32, ph_t, n, sq_t);
        stage_tail(lat32, ph_l, n, sq_l);
        if (a.out_summary) {
            a.out_summary[r].p50_e2e_us = ASR_FMT32;
            a.out_summary[r].p50_ttft_us = ASR_FMT32;
        }
    }
    if (valid && !FREE && staged) {   // requests n - (n & 3) .. n-1 are still in st(4 - tail) .. st3
        const int tail = n & 3;
        if (tail >= 3) ttft[n - 3] = st1;
        if (tail >= 2) ttft[n - 2] = st2;
        if (tail >= 1) ttft[n - 1] = st3;
    }
    if (valid && a.out_summary) {
        asr_summary_t *s = a.out_summary + r;
        s->last_done_us = t;
        s->n_done = done;
    }
}

// ---------------------------------------------------------------------------
// a piece of a replica in 32-bit times (summary-only calls).
//   LANE_UNIT    a thread simulates one segment [b, b + L) of a replica's trace AS IF it were a trace of its own:
//                the server is taken to be idle at the segment's first arrival and the trace to end with the
//                segment.  It records its regeneration points (server empty at an arrival at or after the clock:
//                the state is then (empty, t = that arrival) whatever came before) in the replica's bitmap, and
//                the last one in unit_q -- the segment's end itself if everything completed by the next arrival.
//   LANE_REPAIR  a thread stitches the boundary between segments s-1 and s: unless segment s-1 ended at a
//                regeneration point, it simulates from the last regeneration point q of segment s-1 (a TRUE state
//                when the segments before are stitched) across the boundary until it reaches a regeneration point
//                that segment s recorded too -- from there on segment s's values are the true ones -- and
//                overwrites the values of the requests [q, that point) in place (positions = request indices for
//                both streams: at a regeneration point exactly the requests before it have been emitted).
// Every value that survives comes from a simulation that started in a true state; a boundary that cannot be
// stitched inside segment s flags the replica, which lane_run then simulates in one piece.
//
// A piece starts with the server empty at one of its arrivals and stays within minutes of it, so every time is kept
// as a uint32 offset from an EPOCH E (an arrival at which the server was empty): the clock t, the look-ahead
// arrivals and the ring payloads; iteration costs, token counts and encoder times are 32-bit as well.  Exactness:
//   * the limits below (computed once per piece) bound what one trip of the loop can add to t by 3 * 2^29, and t is
//     tested against 2^30 once per trip (the epoch then moves up, see there), so no sum ever wraps; a request outside
//     the limits, a request that stays in the system for 2^30 us or a first arrival before the clock's origin flags
//     the replica, which is then simulated in one piece by the 64-bit code of lane_run (every emitted value is below
//     2^32 there too);
//   * an arrival 2^32 us or more past the epoch reads LANE_FAR, which no clock value reaches; the epoch moves to
//     the next arrival (read again from the trace, all 64 bits) whenever the server is empty and that arrival is
//     2^30 us or more past it.
// ---------------------------------------------------------------------------
enum { LANE_UNIT = 1, LANE_REPAIR = 2 };
constexpr uint32_t LANE_FAR = 0xFFFFFFFFu;

__device__ __forceinline__ uint32_t lane_rel(int64_t arrival, int64_t epoch) {
    const uint64_t d = (uint64_t)(arrival - epoch);
    return (d >> 32) != 0ull ? LANE_FAR : (uint32_t)d;
}

template <int MODE>
__device__ __forceinline__ void lane_piece(const SimArgs &a, const uint32_t sbase, const uint32_t park, bool live, const int r,
                                           const int seg, const int nseg, const int uq) {
    static_assert(MODE == LANE_UNIT || MODE == LANE_REPAIR, "pieces only");
    if (MODE == LANE_REPAIR && seg == 0) live = false;
    bool valid = live;
    int start = 0;     // first request of this thread's piece (index in the replica)
    int seg_b = 0;     // first request of segment `seg`
    int n = 0;         // requests in the piece
    asr_replica_t rep;
    rep.trace_off = rep.out_off = 0;
    rep.n = 0;
    rep.policy = rep.cm_id = 0;
    rep.slots = 1;
    if (live) {
        rep = a.replicas[r];
        if (!replica_ok(a, rep, LANE_CAP)) {
            flag_invalid(a, r);   // (an invalid descriptor is one unit)
            live = valid = false;
            rep.cm_id = 0;
            rep.n = 0;
        }
    }
    if (live) {
        const int L = lane_seg_len(rep.n, nseg);
        seg_b = seg * L;
        if (MODE == LANE_UNIT) {
            start = seg_b;
            n = min(L, rep.n - seg_b);
        } else {
            const int q = a.plan.unit_q[uq - 1];   // the entries of a replica are consecutive
            if (q >= seg_b || a.plan.failed[r] != 0) {
                live = valid = false;   // segment s-1 ended at a regeneration point (or the replica is flagged already)
            } else {
                start = q;
                n = min(seg_b + L, rep.n) - q;
            }
        }
    }
    const int slots = rep.slots;
    const bool chooses = rep.policy != ASR_FCFS;
    const asr_cost_model_t *cmp = a.cms + rep.cm_id;
    const int64_t enc_base64 = __ldg(&cmp->enc_base_us), enc_per64 = __ldg(&cmp->enc_per_ms_us);
    const int64_t iter_base64 = __ldg(&cmp->iter_base_us), iter_per64 = __ldg(&cmp->iter_per_running_us);
    const int32_t tok_base = __ldg(&cmp->tok_base), tok_per_s_i = __ldg(&cmp->tok_per_s);
    const uint32_t tok_per_s = (uint32_t)tok_per_s_i;
    // the limits: one iteration < 2^29 us at 32 running; a request's decode (tokens * that) < 2^29 us; 32 encoder
    // passes + one iteration < 2^29 us; tok_per_s * dur_ms < 2^32.  dur_lim = the longest audio inside all of them.
    const int64_t lim29 = ((int64_t)1 << 29) - 1;
    bool deferred = false;
    uint32_t dur_lim = 0;
    {
        const bool sane = enc_base64 >= 0 && enc_base64 <= lim29 && enc_per64 >= 0 && enc_per64 <= lim29 &&
                          iter_base64 >= 0 && iter_base64 <= lim29 && iter_per64 >= 0 && iter_per64 <= lim29 &&
                          tok_per_s_i >= 0 && tok_base > -(1 << 30) && tok_base < (1 << 30);
        const int64_t cmax = sane ? iter_base64 + iter_per64 * LANE_CAP : lim29 + 1;
        int64_t dl = -1;
        if (cmax <= lim29) {
            const int64_t tok_lim = lim29 / (cmax > 0 ? cmax : 1);             // tokens * cmax < 2^29
            const int64_t enc_lim = (lim29 - cmax) / LANE_CAP - enc_base64;     // enc_per * dur <= enc_lim
            dl = (int64_t)1 << 24;                                              // (asr_sched.h: dur_ms <= 2^24)
            if (tok_per_s_i > 0) {
                dl = min(dl, (int64_t)0xFFFFFFFFll / tok_per_s_i);
                dl = tok_lim < tok_base ? -1 : min(dl, ((tok_lim - tok_base) * 1000) / tok_per_s_i);
            } else if (tok_lim < tok_base) {
                dl = -1;
            }
            if (enc_lim < 0) dl = -1;
            else if (enc_per64 > 0) dl = min(dl, enc_lim / enc_per64);
        }
        if (live && dl < 0) {
            deferred = true;
            live = false;
        }
        dur_lim = dl < 0 ? 0u : (uint32_t)dl;
    }
    const uint32_t enc_base = (uint32_t)enc_base64, enc_per = (uint32_t)enc_per64;
    const uint32_t ib = (uint32_t)iter_base64, ip = (uint32_t)iter_per64;
    const asr_req_t *trace = a.traces + rep.trace_off + start;
    // the regeneration points of segment `seg`, one bit per request, in the replica's bitmap (whole words per
    // segment); `ibits` collects the word `wcur`
    uint32_t *bm = nullptr;
    if (live) bm = a.bitmap + a.bm_off[r] + (seg_b >> 5);
    uint32_t ibits = 0;
    int wcur = 0, q_last = 0;
    bool merged = false;

    int64_t E = 0;      // the epoch
    uint32_t t = 0;     // the current iteration boundary, us past the epoch
    int p = 0, lo = 0, nW = 0, nR = 0, done = 0;
    uint32_t hoff = 0;  // running set = nR ring positions from byte offset hoff, sorted by finish iteration
    uint32_t it = 0;    // engine iterations so far, mod 2^32
    // look-ahead window over the trace: records p and p+1 are in registers (one 128-bit load each); the arrival of
    // p+1 stays as loaded until it becomes arr0 a trip later (a conversion here would wait for the load)
    uint32_t arr0 = LANE_FAR, last_arr = 0, prev_arr = 0;   // last / prev: the two requests ingested last
    int64_t raw1 = INT64_MAX;
    int32_t dur0 = 0, dur1 = 0, last_dur = 0, prev_dur = 0;
    int32_t est1 = 0;   // (kept live until the record is consumed, see lane_run)
    bool bad = false;   // a request outside the limits was ingested
    if (live && n > 0) {
        const Rec q = ld_cached(trace);
        E = q.arrival_us;
        arr0 = 0;
        dur0 = q.dur_ms;
        if (MODE == LANE_UNIT && seg == 0) {
            if (a.out_summary) a.out_summary[r].first_arrival_us = E;
            if (E < 0) {   // the clock starts at 0, after this arrival: not a piece that starts idle
                deferred = true;
                live = false;
            }
        }
    }
    if (live && n > 1) {
        const Rec q = ld_cached(trace + 1);
        raw1 = q.arrival_us;
        dur1 = q.dur_ms;
        est1 = q.est;
    }
    Stage32 sq_t = {0, 0, 0, 0}, sq_l = {0, 0, 0, 0};
#ifdef LANE_SECTOR_STORES
    const uint32_t park_l = park + LANE_THREADS * 16u;
    const uint32_t ph_mask = 7u;
#define PIECE_PUSH_T(pos, v) stage8_push(ttft32, ph_t, pos, v, sq_t, park)
#define PIECE_PUSH_L(pos, v) stage8_push(lat32, ph_l, pos, v, sq_l, park_l)
#define PIECE_TAIL(cnt) (stage8_tail(ttft32, ph_t, cnt, sq_t, park), stage8_tail(lat32, ph_l, cnt, sq_l, park_l))
#else
    const uint32_t ph_mask = 3u;
#define PIECE_PUSH_T(pos, v) stage_push(ttft32, ph_t, pos, v, sq_t)
#define PIECE_PUSH_L(pos, v) stage_push(lat32, ph_l, pos, v, sq_l)
#define PIECE_TAIL(cnt) (stage_tail(ttft32, ph_t, cnt, sq_t), stage_tail(lat32, ph_l, cnt, sq_l))
#endif
    uint32_t *ttft32 = reinterpret_cast<uint32_t *>(a.out_ttft + rep.out_off) + start;
    uint32_t *lat32 = reinterpret_cast<uint32_t *>(a.out_lat + rep.out_off) + start;
    const int ph_t = (int)((reinterpret_cast<uintptr_t>(ttft32) >> 2) & ph_mask);
    const int ph_l = (int)((reinterpret_cast<uintptr_t>(lat32) >> 2) & ph_mask);
    if (n == 0) {
        if (MODE == LANE_UNIT && seg == 0 && valid && a.out_summary) a.out_summary[r].first_arrival_us = 0;
        live = false;
    }

    // One trip = one admission step (lane_run): A pops the completions that precede the step, B moves the clock to
    // its boundary, C ingests, D admits.
    while (true) {
        if (live) {
            // A. completions before the next admission opportunity
            bool more = nR > 0;
            const uint32_t a_eff = nW > 0 ? 0u : arr0;   // somebody waiting: admit at the first free slot
            while (more) {
                const uint2 e = ring_ld(sbase + hoff);   // sorted: the head finishes first
                const uint32_t f = e.x;
                const uint32_t m = f - it;
                const uint32_t c = ib + ip * (uint32_t)nR;
                const uint32_t lim = t + (m - 1u) * c;
                if (m > 0u && nR < slots && a_eff <= lim) {
                    more = false;
                } else {
                    if (m > 0u) {
                        t = lim + c;
                        it = f;
                    }
                    PIECE_PUSH_L(done, t - e.y);   // E2E = t - arrival
                    hoff = (hoff + RING_STEP) & RING_MASK;
                    --nR;
                    ++done;
                    more = nR > 0;
                }
            }
            if (done >= n) live = false;
            if (live && (t >> 30) != 0u) {
                // 2^30 us past the epoch with the server busy (rare): the epoch moves up to the clock, or to the next
                // arrival if that one is already due (no arrival still to come may lie before the epoch).  The
                // ring's payloads are arrivals relative to the epoch and only ever enter differences modulo 2^32,
                // which stay exact while no request in the system is older than 2^32 us; here every one of them
                // is checked to be younger than 2^30 us (else the 64-bit code takes the replica), and the clock
                // gains less than 2.5 * 2^30 us before the next check.
                const uint32_t s = arr0 < t ? arr0 : t;
                bool young = ((t - s) >> 30) == 0u;
                for (int i = 0; i < nR; ++i)
                    young = young && t - ring_ld(sbase + ((hoff + (uint32_t)i * RING_STEP) & RING_MASK)).y < (1u << 30);
                if (nW > 0) young = young && (E + (int64_t)t) - ld_arrival(trace + lo) < ((int64_t)1 << 30);
                if (!young) {
                    deferred = true;
                    live = false;
                } else {
                    for (int i = 0; i < nR; ++i) {
                        const uint32_t ad = sbase + ((hoff + (uint32_t)i * RING_STEP) & RING_MASK);
                        const uint2 e = ring_ld(ad);
                        ring_st(ad, make_uint2(e.x, e.y - s));
                    }
                    E += (int64_t)s;
                    t -= s;
                    last_arr -= s;
                    prev_arr -= s;
                    if (arr0 != LANE_FAR) arr0 -= s;
                    else if (p < n) arr0 = lane_rel(ld_arrival(trace + p), E);
                }
            }
        }
        if (!__any_sync(ASR_FULL_MASK, live)) break;   // also the warp's re-convergence point
        if (live) {
            // B. the boundary of the admission step
            if (nW == 0 && nR == 0 && arr0 >= t) {
                // regeneration point: the server is empty when request p arrives, the clock goes to that arrival
                if (MODE == LANE_UNIT) {
                    // (only the head of the segment is recorded: a repair meets the segment within a few busy
                    // periods of its start or not at all)
                    if (p < LANE_REGEN_HEAD) {
#pragma unroll 1
                        while (wcur < (p >> 5)) {
                            bm[wcur] = ibits;
                            ibits = 0;
                            ++wcur;
                        }
                        ibits |= 1u << (p & 31);
                    }
                    q_last = p;
                } else {
                    const int d = start + p - seg_b;   // position in segment s
                    if (d >= 0 && d < LANE_REGEN_HEAD && ((__ldcg(bm + (d >> 5)) >> (d & 31)) & 1u)) {
                        merged = true;   // segment s was in this very state: its values are true from here on
                        live = false;
                    }
                }
                if (arr0 >= (1u << 30)) {   // move the epoch to this arrival
                    E = ld_arrival(trace + p);
                    arr0 = 0;
                    t = 0;
                }
            }
            if (nW == 0 && arr0 > t) {
                if (nR == 0) {
                    t = arr0;   // idle server: the clock jumps to the next arrival (S14)
                } else {
                    const uint32_t c = ib + ip * (uint32_t)nR;
                    const uint32_t g = arr0 - t;   // c > 0: arr0 <= t + (m-1)*c
                    const uint32_t q = g / c;
                    const uint32_t j = q + (g - q * c != 0u ? 1u : 0u);
                    t += j * c;
                    it += j;
                }
            }
            // C. ingest arrivals <= t
            while (arr0 <= t && (MODE != LANE_REPAIR || !merged)) {
                prev_arr = last_arr;
                prev_dur = last_dur;
                last_arr = arr0;
                last_dur = dur0;
                bad = bad || (uint32_t)dur0 > dur_lim;
                ++p;
                ++nW;
                arr0 = lane_rel(raw1, E);
                dur0 = dur1;
                asm volatile("{ .reg .pred p; setp.eq.s32 p, %0, -2147483647; @p prefetch.global.L2 [%1]; }" ::"r"(est1),
                             "l"(trace));
                raw1 = INT64_MAX;
                if (p + 1 < n) {
                    const Rec q = ld_cached(trace + p + 1);
                    raw1 = q.arrival_us;
                    dur1 = q.dur_ms;
                    est1 = q.est;
                }
            }
            // D. admit k >= 1 requests (a slot is free and somebody waits)
            const int free_slots = slots - nR;
            const int k = free_slots < nW ? free_slots : nW;
            if (MODE == LANE_REPAIR && merged) {
                // stitched: nothing more to simulate
            } else if ((chooses && k < nW) || bad) {   // a real choice, or 64-bit arithmetic: the replica is redone in one piece
                deferred = true;
                live = false;
            } else {
                uint32_t t1 = t + ib + ip * (uint32_t)(nR + k);
                if (k == 1 && lo == p - 1) {
                    // the request ingested last: everything needed is in registers
                    const int32_t tok = tok_base + (int32_t)((tok_per_s * (uint32_t)last_dur) / 1000u);
                    lane_insert(sbase, hoff, nR, it, (uint32_t)(tok < 1 ? 1 : tok), last_arr);
                    t1 += enc_per * (uint32_t)last_dur + enc_base;
                    PIECE_PUSH_T(lo, t1 - last_arr);   // first token (S9)
                } else if (k == 2 && nW == 2) {
                    // the two requests ingested last (two arrivals during one admission step)
                    const int32_t tok_a = tok_base + (int32_t)((tok_per_s * (uint32_t)prev_dur) / 1000u);
                    lane_insert(sbase, hoff, nR, it, (uint32_t)(tok_a < 1 ? 1 : tok_a), prev_arr);
                    const int32_t tok_b = tok_base + (int32_t)((tok_per_s * (uint32_t)last_dur) / 1000u);
                    lane_insert(sbase, hoff, nR + 1, it, (uint32_t)(tok_b < 1 ? 1 : tok_b), last_arr);
                    t1 += enc_per * (uint32_t)(prev_dur + last_dur) + 2u * enc_base;
                    PIECE_PUSH_T(lo, t1 - prev_arr);
                    PIECE_PUSH_T(lo + 1, t1 - last_arr);
                } else {
                    uint32_t dur_sum = 0;
#pragma unroll 1
                    for (int q = 0; q < k; ++q) {
                        const Rec rq = ld_cached(trace + lo + q);
                        const int32_t tok = tok_base + (int32_t)((tok_per_s * (uint32_t)rq.dur_ms) / 1000u);
                        // (a waiting request may have arrived before the epoch: the difference modulo 2^32)
                        lane_insert(sbase, hoff, nR + q, it, (uint32_t)(tok < 1 ? 1 : tok), (uint32_t)(rq.arrival_us - E));
                        dur_sum += (uint32_t)rq.dur_ms;
                    }
                    t1 += enc_base * (uint32_t)k + enc_per * dur_sum;
#pragma unroll 1
                    for (int q = 0; q < k; ++q)
                        PIECE_PUSH_T(lo + q, t1 - (uint32_t)(ld_arrival(trace + lo + q) - E));
                }
                lo += k;
                nW -= k;
                nR += k;
                t = t1;
                it += 1u;
            }
        }
    }
    if (deferred) {
        a.plan.failed[r] = 1;   // whatever stopped this piece, the replica is simulated in one piece
#ifdef LANE_STATS
        atomicAdd(&g_lane_stats[1], 1ull);
#endif
        return;
    }
    if (!valid) return;
#ifdef LANE_STATS
    atomicAdd(&g_lane_stats[MODE == LANE_UNIT ? 0 : 2], 1ull);
    if (MODE == LANE_REPAIR) atomicAdd(&g_lane_stats[5], (unsigned long long)p);
#endif
    const int64_t t_end = E + (int64_t)t;
    if (MODE == LANE_UNIT) {
        PIECE_TAIL(n);
        for (; wcur <= ((min(n, LANE_REGEN_HEAD) - 1) >> 5); ++wcur) {
            bm[wcur] = ibits;
            ibits = 0;
        }
        // everything completed by the next segment's first arrival: the segment's end is a regeneration point
        if (start + n < rep.n && t_end <= ld_arrival(trace + n)) q_last = n;
        a.plan.unit_q[uq] = start + q_last;
        if (seg == nseg - 1 && a.out_summary) {
            asr_summary_t *s = a.out_summary + r;
            s->last_done_us = t_end;
            s->n_done = rep.n;
            s->p50_e2e_us = ASR_FMT32;
            s->p50_ttft_us = ASR_FMT32;
        }
    } else {
        const bool to_end = done >= n && start + n == rep.n;   // the last boundary, simulated to the end of the trace
        if (!merged && !to_end) {
            a.plan.failed[r] = 1;   // no common regeneration point inside segment s
#ifdef LANE_STATS
            atomicAdd(&g_lane_stats[3], 1ull);
#endif
            return;
        }
        const int cnt = merged ? p : n;   // at a regeneration point exactly the requests before it have been emitted
        PIECE_TAIL(cnt);
        if (to_end && !merged && a.out_summary) a.out_summary[r].last_done_us = t_end;
    }
}
#undef PIECE_PUSH_T
#undef PIECE_PUSH_L
#undef PIECE_TAIL

// a thread simulates a whole replica (with a plan: only the replicas flagged `failed`)
template <bool FREE>
__global__ void __launch_bounds__(LANE_THREADS, LANE_BLOCKS_PER_SM) sim_lane_kernel(SimArgs a) {
    __shared__ uint2 s_ring[LANE_CAP * LANE_THREADS];
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(s_ring) + threadIdx.x * 8u;
    const int r = blockIdx.x * LANE_THREADS + threadIdx.x;
    bool live = r < a.n_replicas;
    if (live && a.plan.failed && a.plan.failed[r] == 0) live = false;   // stitched: nothing to redo
#ifdef LANE_STATS
    if (live && a.plan.failed) atomicAdd(&g_lane_stats[4], 1ull);
#endif
    lane_run<FREE>(a, sbase, live, r);
}

// persistent warps work off the plan's items (heaviest load class first): lane j of item (group, seg) takes
// segment seg of replica order[32*group + j]
#ifndef LANE_WORK_BLOCKS
#define LANE_WORK_BLOCKS 10
#endif
// (r02 sweep: 15.8 ms at 10 CTAs and 94 registers, 16.4-16.5 ms at 12 or 13 CTAs squeezed into 80 / 72)
constexpr int LANE_WORK_BLOCKS_PER_SM = LANE_WORK_BLOCKS;
template <int MODE>
#ifdef LANE_WORK_MAXREG
__global__ void __maxnreg__(LANE_WORK_MAXREG) sim_lane_work_kernel(SimArgs a) {
#else
__global__ void __launch_bounds__(LANE_THREADS, LANE_WORK_BLOCKS_PER_SM) sim_lane_work_kernel(SimArgs a) {
#endif
    __shared__ uint2 s_ring[LANE_CAP * LANE_THREADS];
#ifdef LANE_SECTOR_STORES
    __shared__ uint4 s_park[2 * LANE_THREADS];   // [stream][thread]: stage8_push
    const uint32_t park = (uint32_t)__cvta_generic_to_shared(s_park) + threadIdx.x * 16u;
#else
    const uint32_t park = 0;
#endif
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(s_ring) + threadIdx.x * 8u;
    const int lane = lane_id();
    const int n_items = ((a.n_replicas + 31) / 32) * LANE_MAX_SEG;
    int32_t *next = a.plan.counters + (MODE == LANE_UNIT ? 0 : 1);
    while (true) {
        int w = 0;
        if (lane == 0) w = atomicAdd(next, 1);
        w = __shfl_sync(ASR_FULL_MASK, w, 0);
        if (w >= n_items) break;
        const int2 item = make_int2(w / LANE_MAX_SEG, w % LANE_MAX_SEG);
        if (MODE == LANE_REPAIR && item.y == 0) continue;
        const int pos = 32 * item.x + lane;
        bool live = pos < a.n_replicas;
        int r = 0, nseg = 1;
        if (live) {
            r = a.plan.order[pos];
            nseg = a.plan.nseg[r];
            live = item.y < nseg;
        }
        if (!__any_sync(ASR_FULL_MASK, live)) continue;   // no replica of the group has this many segments
        const int uq = pos * LANE_MAX_SEG + item.y;
        lane_piece<MODE>(a, sbase, park, live, r, item.y, nseg, uq);
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------
// the plan of a summary-only thread-per-replica call: load classes, order, units
// ---------------------------------------------------------------------------
// Offered load of a replica in Erlangs, estimated from a few records (mean arrival gap, mean solo service time of
// a few dozen sampled requests).  It only steers the schedule -- which replicas share a warp, which are cut into
// segments -- and never a result.
constexpr int PLAN_BUCKETS = 32;
constexpr float PLAN_SPLIT_MAX_LOAD = 3.5f;   // beyond it regeneration points (about exp(-load) of the arrivals) are too rare to stitch at
constexpr int PLAN_SAMPLES = 32;

__global__ void __launch_bounds__(256) lane_key_kernel(SimArgs a) {
    const int r = blockIdx.x * 256 + threadIdx.x;
    if (r >= a.n_replicas) return;
    const asr_replica_t rep = a.replicas[r];
    int bucket = PLAN_BUCKETS - 1, nseg = 1;
    if (replica_ok(a, rep, LANE_CAP) && rep.n >= 2) {
        const asr_req_t *tr = a.traces + rep.trace_off;
        const int n = rep.n;
        const asr_cost_model_t cm = a.cms[rep.cm_id];
        float svc = 0.f;
#pragma unroll 8
        for (int j = 0; j < PLAN_SAMPLES; ++j) {
            const int idx = (int)(((int64_t)(2 * j + 1) * n) / (2 * PLAN_SAMPLES));
            const int32_t dur = __ldg(&tr[idx].dur_ms);
            svc += (float)(cm.enc_base_us + cm.enc_per_ms_us * (int64_t)dur) +
                   (float)tokens_of(cm, dur) * (float)(cm.iter_base_us + cm.iter_per_running_us);
        }
        svc *= 1.f / PLAN_SAMPLES;
        const float gap = (float)(ld_arrival(tr + n - 1) - ld_arrival(tr)) / (float)(n - 1);
        const float load = gap > 0.f ? svc / gap : 1e9f;
        if (load > 0.f) {
            const int b = 16 - (int)rintf(4.f * log2f(load));   // four classes per octave, heaviest first
            bucket = b < 0 ? 0 : (b > PLAN_BUCKETS - 2 ? PLAN_BUCKETS - 2 : b);
        }
        if (load <= PLAN_SPLIT_MAX_LOAD && n >= 2 * LANE_SEG_TARGET) {
            nseg = n / LANE_SEG_TARGET;
            nseg = nseg > LANE_MAX_SEG ? LANE_MAX_SEG : nseg;
        }
    }
    a.plan.bucket[r] = (uint8_t)bucket;
    a.plan.nseg[r] = (uint8_t)nseg;
    a.plan.failed[r] = 0;
    if (r == 0) a.plan.counters[0] = a.plan.counters[1] = 0;
}

// exclusive scan over the 1,024 threads of the CTA; returns the thread's offset, *total = the sum
__device__ __forceinline__ uint32_t block_excl_scan_1024(uint32_t v, uint32_t *wsum, uint32_t *total) {
    const int lane = lane_id(), warp = threadIdx.x >> 5;
    uint32_t x = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t y = __shfl_up_sync(ASR_FULL_MASK, x, d);
        if (lane >= d) x += y;
    }
    __syncthreads();   // wsum's readers of the previous call are done
    if (lane == 31) wsum[warp] = x;
    __syncthreads();
    uint32_t w = wsum[lane];
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t y = __shfl_up_sync(ASR_FULL_MASK, w, d);
        if (lane >= d) w += y;
    }
    *total = __shfl_sync(ASR_FULL_MASK, w, 31);
    const uint32_t wbase = __shfl_sync(ASR_FULL_MASK, w, warp > 0 ? warp - 1 : 0);
    return (warp > 0 ? wbase : 0u) + x - v;
}

// one CTA: stable counting sort of the replicas by load class (thread t owns the replicas [tC, tC + C) and one
// column of the [class][thread] counters)
__device__ __forceinline__ void lane_sort_body(const SimArgs &a) {
    extern __shared__ uint32_t cnt[];   // [PLAN_BUCKETS][1024]
    __shared__ uint32_t wsum[32];
    const int t = threadIdx.x, n = a.n_replicas;
    const int C = (n + 1023) / 1024;
    const int r0 = (int)min((int64_t)n, (int64_t)t * C), r1 = min(n, r0 + C);
    for (int b = 0; b < PLAN_BUCKETS; ++b) cnt[b * 1024 + t] = 0;
    for (int r = r0; r < r1; ++r) cnt[a.plan.bucket[r] * 1024 + t]++;
    uint32_t base = 0;
    for (int b = 0; b < PLAN_BUCKETS; ++b) {
        uint32_t tot;
        const uint32_t v = cnt[b * 1024 + t];
        cnt[b * 1024 + t] = base + block_excl_scan_1024(v, wsum, &tot);
        base += tot;
    }
    for (int r = r0; r < r1; ++r) a.plan.order[cnt[a.plan.bucket[r] * 1024 + t]++] = r;
}

// block 0 sorts the plan, block 1 lays out the bitmaps and clears the counters (sim_prepare_kernel's job): two
// single-CTA jobs that do not depend on each other, side by side
__global__ void lane_plan_prepare_kernel(SimArgs a);

int launch_lane_plan(const SimArgs &a, cudaStream_t st) {
    const int grid = (a.n_replicas + 255) / 256;
    constexpr int SORT_SMEM = PLAN_BUCKETS * 1024 * 4;
    cudaFuncSetAttribute(lane_plan_prepare_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SORT_SMEM);
    {
        KernelTimer kt(KID_LANE_PLAN, st);
        lane_key_kernel<<<grid, 256, 0, st>>>(a);
        lane_plan_prepare_kernel<<<2, 1024, SORT_SMEM, st>>>(a);
    }
    count_launch(1);
    return check_launch("lane plan kernels");
}

// out_lat[i] = -arrival_us[i] for every request of every replica the lane kernel will
// simulate: a coalesced stream, so that the lane kernel's only per-completion memory
// operation is the reduction that adds the completion time
__global__ void __launch_bounds__(256) sim_init_lat_kernel(SimArgs a) {
    for (int r = blockIdx.x; r < a.n_replicas; r += gridDim.x) {
        const asr_replica_t rep = a.replicas[r];
        if (!replica_ok(a, rep, LANE_CAP)) continue;
        const asr_req_t *trace = a.traces + rep.trace_off;
        int64_t *lat = a.out_lat + rep.out_off;
        for (int i = threadIdx.x; i < rep.n; i += 256) __stcs(lat + i, -ld_arrival(trace + i));
    }
}

// exclusive prefix sum of the per-replica bitmap sizes (words), one CTA
// A descriptor that replica_ok() will reject (n or out_off out of range) gets the two slack
// words only, so that one bad descriptor cannot push the bitmaps of the valid replicas past
// the workspace (which is sized from total_requests: the valid regions are disjoint).
__device__ __forceinline__ void sim_prepare_body(const asr_replica_t *replicas, int32_t n_replicas, int64_t total_requests,
                                                 int64_t *bm_off, int32_t *defer_count) {
    __shared__ int64_t warp_tot[32];
    __shared__ int64_t carry_s;
    if (threadIdx.x == 0) {
        carry_s = 0;
        defer_count[0] = 0;   // lane kernel -> warp kernel
        defer_count[1] = 0;   // warp kernel -> CTA kernel
        defer_count[2] = 0;   // carried-window percentile kernel -> radix kernel, E2E latency
        defer_count[3] = 0;   // the same, TTFT
        defer_count[4] = 0;   // cursor of the warp kernel over the hand-over list
    }
    __syncthreads();
    const int lane = lane_id(), warp = threadIdx.x >> 5;
    for (int base = 0; base < n_replicas; base += 1024) {
        const int r = base + threadIdx.x;
        int64_t v = 0;
        if (r < n_replicas) {
            const int n = replicas[r].n;
            const int64_t off = replicas[r].out_off;
            const bool sane = n >= 0 && off >= 0 && off + (int64_t)n <= total_requests;
            v = (int64_t)((sane ? n : 0) >> 5) + 2;   // ceil(n/32) + slack word
        }
        int64_t x = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            int64_t y = (int64_t)shfl64(x, lane >= d ? lane - d : lane);
            if (lane >= d) x += y;
        }
        if (lane == 31) warp_tot[warp] = x;
        __syncthreads();
        if (warp == 0) {
            int64_t w = warp_tot[lane];
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                int64_t y = (int64_t)shfl64(w, lane >= d ? lane - d : lane);
                if (lane >= d) w += y;
            }
            warp_tot[lane] = w;   // inclusive over warps
        }
        __syncthreads();
        const int64_t carry = carry_s;
        const int64_t incl = carry + (warp > 0 ? warp_tot[warp - 1] : 0) + x;
        if (r < n_replicas) bm_off[r] = incl - v;
        __syncthreads();
        if (threadIdx.x == 1023) carry_s = incl;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(1024) sim_prepare_kernel(const asr_replica_t *replicas, int32_t n_replicas,
                                                           int64_t total_requests, int64_t *bm_off,
                                                           int32_t *defer_count) {
    sim_prepare_body(replicas, n_replicas, total_requests, bm_off, defer_count);
}

__global__ void __launch_bounds__(1024) lane_plan_prepare_kernel(SimArgs a) {
    if (blockIdx.x == 0) lane_sort_body(a);
    else sim_prepare_body(a.replicas, a.n_replicas, a.total_requests, const_cast<int64_t *>(a.bm_off), a.defer_count);
}

template <int SPL>
static void launch_warp(const SimArgs &a, int grid, cudaStream_t st) {
    KernelTimer kt(KID_SIMULATE, st);
    sim_warp_kernel<SPL, false><<<grid, SIM_WARPS * 32, 0, st>>>(a);
}

static void launch_warp_any(const SimArgs &a, int max_slots, int grid, cudaStream_t st) {
    if (max_slots <= 32 && a.defer_list != nullptr) {
        KernelTimer kt(KID_SIMULATE, st);
        sim_warp_kernel<1, true><<<grid, SIM_WARPS * 32, 0, st>>>(a);
    } else if (max_slots <= 32) launch_warp<1>(a, grid, st);
    else if (max_slots <= 64) launch_warp<2>(a, grid, st);
    else if (max_slots <= 128) launch_warp<4>(a, grid, st);
    else launch_warp<8>(a, grid, st);
}

// use_lane: thread-per-replica kernel first (slots <= 32), then the warp kernel
// on the replicas it handed over; else the warp kernel on everything.
int launch_simulate(const SimArgs &a_in, int max_slots, bool use_lane, cudaStream_t st) {
    if (a_in.n_replicas <= 0) return ASR_OK;
    SimArgs a = a_in;
    if (use_lane && max_slots <= LANE_CAP) {
        const int lane_grid = (a.n_replicas + LANE_THREADS - 1) / LANE_THREADS;
        if (a.order_free && a.plan.order) {
            // (lane_piece: the two value arrays of a summary-only call share the phase of their 16-byte lines)
            if (((reinterpret_cast<uintptr_t>(a.out_lat) ^ reinterpret_cast<uintptr_t>(a.out_ttft)) & 15u) != 0) {
                set_error("simulate: workspace value arrays out of phase");
                return ASR_EINVAL;
            }
            // time-split units, stitched at regeneration points; what could not be stitched, in one piece
            int rc0 = launch_lane_plan(a, st);
            if (rc0) return rc0;
            const int work_grid = sm_count() * LANE_WORK_BLOCKS_PER_SM;
            {
                KernelTimer kt(KID_SIM_LANE, st);
                sim_lane_work_kernel<LANE_UNIT><<<work_grid, LANE_THREADS, 0, st>>>(a);
            }
            rc0 = check_launch("sim_lane_work_kernel<units>");
            if (rc0) return rc0;
            {
                KernelTimer kt(KID_SIM_REPAIR, st);
                sim_lane_work_kernel<LANE_REPAIR><<<work_grid, LANE_THREADS, 0, st>>>(a);
            }
            rc0 = check_launch("sim_lane_work_kernel<repair>");
            if (rc0) return rc0;
            {
                KernelTimer kt(KID_SIM_REDO, st);
                sim_lane_kernel<true><<<lane_grid, LANE_THREADS, 0, st>>>(a);
            }
#ifdef LANE_STATS
            {
                unsigned long long h[8], z[8] = {0, 0, 0, 0, 0, 0, 0, 0};
                cudaStreamSynchronize(st);
                cudaMemcpyFromSymbol(h, g_lane_stats, sizeof(h));
                cudaMemcpyToSymbol(g_lane_stats, z, sizeof(z));
                fprintf(stderr, "lane stats: units %llu flagged-by-units %llu repairs %llu unstitched %llu redone %llu repair-requests %llu\n",
                        h[0], h[1], h[2], h[3], h[4], h[5]);
            }
#endif
        } else if (a.order_free) {
            KernelTimer kt(KID_SIM_LANE, st);
            sim_lane_kernel<true><<<lane_grid, LANE_THREADS, 0, st>>>(a);
        } else {
            {
                KernelTimer kt(KID_SIM_INIT_LAT, st);
                const int grid = a.n_replicas < sm_count() * 8 ? a.n_replicas : sm_count() * 8;
                sim_init_lat_kernel<<<grid, 256, 0, st>>>(a);
            }
            int rc0 = check_launch("sim_init_lat_kernel");
            if (rc0) return rc0;
            KernelTimer kt(KID_SIM_LANE, st);
            sim_lane_kernel<false><<<lane_grid, LANE_THREADS, 0, st>>>(a);
        }
        int rc = check_launch("sim_lane_kernel");
        if (rc) return rc;
        // worklist pass: empty (and a few microseconds) when nothing was handed over
        const int want = (a.n_replicas + SIM_WARPS - 1) / SIM_WARPS;
        launch_warp_any(a, max_slots, want < sm_count() * 8 ? want : sm_count() * 8, st);
        rc = check_launch("sim_warp_kernel");
        if (rc) return rc;
        return launch_simulate_cta(a, st);   // worklist of the warp kernel; empty unless a backlog ran deep
    }
    a.defer_list = nullptr;
    launch_warp_any(a, max_slots, (a.n_replicas + SIM_WARPS - 1) / SIM_WARPS, st);
    int rc = check_launch("sim_warp_kernel");
    if (rc) return rc;
    a.defer_list = a_in.defer_list;
    return launch_simulate_cta(a, st);
}

int launch_sim_prepare(const asr_replica_t *replicas, int32_t n_replicas, int64_t total_requests, int64_t *bm_off,
                       int32_t *defer_count, cudaStream_t st) {
    {
        KernelTimer kt(KID_SIM_PREPARE, st);
        sim_prepare_kernel<<<1, 1024, 0, st>>>(replicas, n_replicas, total_requests, bm_off, defer_count);
    }
    return check_launch("sim_prepare_kernel");
}

}  // namespace asr

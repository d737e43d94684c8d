// simulate_ex.cu -- the simulator step with the SURVEY.md 8(f) extensions, sm_100a:
//   f1  preemption under a KV-memory budget (A.4 "Preemption logic")
//   f3  policy switching on queue depth ("Dynamic policy switching")
//
// One warp owns one replica, lane L holds batch slots L, L+32, ... in registers, as
// in simulate.cu; per slot it also keeps the request's estimate (the eviction rule
// compares running requests under the policy's total order) and the KV units it
// holds.  Preempted requests return to the waiting set, so the waiting set is not a
// dense index range here: a bitmap over [0, p) marks the requests that are admitted
// (running or finished), a second one those that already had a first token.
//
// Exact fast-forward with two more bounds: the running set may only decode while
// M + |R| <= kv_budget (M grows by |R| per iteration), and a step that could admit
// (somebody waits, a slot is free, admission not blocked by memory) ends the run.
#include "sim_common.cuh"

namespace asr {

__device__ __forceinline__ int eff_policy(int policy, const asr_sim_ext_t &ex, int n_waiting) {
    if (policy != ASR_ADAPTIVE) return policy;
    if (n_waiting < ex.depth1) return ex.pol[0];
    if (n_waiting < ex.depth2) return ex.pol[1];
    return ex.pol[2];
}

__device__ __forceinline__ int64_t kv_enc(const asr_sim_ext_t &ex, int32_t dur_ms) {
    return ex.kv_base + (ex.kv_per_s * (int64_t)dur_ms) / 1000;
}

__device__ __forceinline__ bool ext_ok(const asr_sim_ext_t &ex, int policy) {
    if (policy < 0 || policy > ASR_ADAPTIVE) return false;
    if (policy == ASR_ADAPTIVE) {
        if (ex.depth1 > ex.depth2) return false;
        for (int j = 0; j < 3; ++j)
            if (ex.pol[j] < 0 || ex.pol[j] > 2) return false;
    }
    return ex.kv_base >= 0 && ex.kv_per_s >= 0;
}

template <int SPL>
__device__ __forceinline__ void sim_ex_replica(const SimExArgs &a, const int r, ChunkMeta *ring) {
    const int lane = lane_id();
    asr_replica_t rep = a.replicas[r];
    const int n = rep.n, slots = rep.slots, policy = rep.policy;
    {
        asr_replica_t chk = rep;
        chk.policy = 0;   // the policy range is checked by ext_ok
        if (!replica_ok(a, chk, 32 * SPL) || !ext_ok(a.exts[rep.cm_id], policy)) {
            if (lane == 0) {
                flag_invalid(a, r);
                if (a.out_preempt) a.out_preempt[r] = 0;
                if (a.itl_npairs) a.itl_npairs[r] = -1;
            }
            return;
        }
    }
    const asr_cost_model_t cm = a.cms[rep.cm_id];
    const asr_sim_ext_t ex = a.exts[rep.cm_id];
    const int64_t B = ex.kv_budget;
    const asr_req_t *trace = a.traces + rep.trace_off;
    int64_t *lat = a.out_lat + rep.out_off;
    int64_t *ttft = a.out_ttft + rep.out_off;
    uint32_t *bm = a.bitmap + a.bm_off[r];     // bit i: request i is running or finished
    uint32_t *ever = a.bitmap2 + a.bm_off[r];  // bit i: request i has had its first token

    int32_t rem[SPL], ridx[SPL], rest[SPL];
    int64_t rarr[SPL], rmem[SPL];
#pragma unroll
    for (int s = 0; s < SPL; ++s) {
        rem[s] = REM_FREE;
        ridx[s] = -1;
        rest[s] = 0;
        rarr[s] = 0;
        rmem[s] = 0;
    }
    int64_t t = 0, M = 0, n_pre = 0;
    int p = 0, lo = 0, nW = 0, nR = 0, done = 0, bm_hi = 0, n_pairs = 0;
    bool blocked = false, bad = false;
    bool meta_ok = false;   // the chunk bounds (sim_common.cuh) cover the window [lo, p)
    const int64_t first_arrival = n > 0 ? trace[0].arrival_us : 0;

    while (done < n) {
        // ---- 1. ingest arrivals <= t (32 at a time)
        while (p < n) {
            const int i = p + lane;
            Rec q;
            q.arrival_us = 0;
            q.dur_ms = q.est = 0;
            if (i < n) q = ld_cached(trace + i);
            const bool in = i < n && q.arrival_us <= t;
            const uint32_t m = __ballot_sync(ASR_FULL_MASK, in);
            const int cnt = (m == ASR_FULL_MASK) ? 32 : __ffs(~m) - 1;   // arrivals are sorted
            if (cnt > 0 && meta_ok) {
                // the newcomers [p, p + cnt) join the bounds of their chunks (at most two; a chunk starts with its
                // first request)
                const bool mine = lane < cnt;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int c = (p >> 5) + h;
                    const bool inc = mine && (i >> 5) == c;
                    const uint32_t lm = __ballot_sync(ASR_FULL_MASK, inc);
                    if (lm == 0u) continue;
                    const int32_t e_new = __reduce_min_sync(ASR_FULL_MASK, inc ? (int32_t)est_of(q.est) : INT32_MAX);
                    const uint32_t bits = __reduce_or_sync(ASR_FULL_MASK, inc ? 1u << (i & 31) : 0u);
                    const int64_t a_new = shfl64(q.arrival_us, __ffs(lm) - 1);
                    if (lane == 0) {
                        ChunkMeta *slot = ring + (c % CHUNK_RING);
                        ChunkMeta mt = *slot;
                        if ((c << 5) >= p) mt.wait = 0u;   // nothing of this chunk was ingested before
                        if (mt.wait == 0u) {
                            mt.a_first = a_new;
                            mt.e_min = e_new;
                        } else {
                            mt.e_min = e_new < mt.e_min ? e_new : mt.e_min;
                        }
                        mt.wait |= bits;
                        *slot = mt;
                    }
                }
                __syncwarp();
            }
            p += cnt;
            nW += cnt;
            if (cnt > 0) blocked = false;
            if (cnt < 32) break;
        }
        if (bm_hi < p) {   // clear the bits of the newly ingested requests [bm_hi, p)
            const int w0 = bm_hi >> 5, w1 = (p - 1) >> 5;
            for (int w = w0 + lane; w <= w1; w += 32) {
                if (w == w0 && (bm_hi & 31)) {
                    const uint32_t keep = (1u << (bm_hi & 31)) - 1u;
                    bm[w] &= keep;
                    ever[w] &= keep;
                } else {
                    bm[w] = 0u;
                    ever[w] = 0u;
                }
            }
            bm_hi = p;
            __syncwarp();
        }
        // ---- 2. idle server
        if (nR == 0 && nW == 0) {
            t = ld_cached(trace + p).arrival_us;
            continue;
        }
        const int pol = eff_policy(policy, ex, nW);
        // ---- 3a. memory pressure: evict the worst running request until one more token each fits
        int preempted = 0;
        while (B > 0 && M + nR > B) {
            if (nR <= 1) {   // a request that cannot fit alone
                bad = true;
                break;
            }
            int64_t w_arr = 0;
            int32_t w_est = 0, w_idx = -1, w_slot = -1;
#pragma unroll
            for (int s = 0; s < SPL; ++s)
                if (rem[s] != REM_FREE &&
                    (w_idx < 0 || better_rt(pol, w_arr, w_est, w_idx, rarr[s], rest[s], ridx[s], t))) {
                    w_arr = rarr[s];
                    w_est = rest[s];
                    w_idx = ridx[s];
                    w_slot = s * 32 + lane;
                }
#pragma unroll
            for (int j = 16; j > 0; j >>= 1) {
                const int64_t o_arr = (int64_t)shfl64_xor((uint64_t)w_arr, j);
                const int32_t o_est = __shfl_xor_sync(ASR_FULL_MASK, w_est, j);
                const int32_t o_idx = __shfl_xor_sync(ASR_FULL_MASK, w_idx, j);
                const int32_t o_slot = __shfl_xor_sync(ASR_FULL_MASK, w_slot, j);
                if (o_idx >= 0 && (w_idx < 0 || better_rt(pol, w_arr, w_est, w_idx, o_arr, o_est, o_idx, t))) {
                    w_arr = o_arr;
                    w_est = o_est;
                    w_idx = o_idx;
                    w_slot = o_slot;
                }
            }
            int64_t freed = 0;
#pragma unroll
            for (int s = 0; s < SPL; ++s)
                if (w_slot == s * 32 + lane) {
                    freed = rmem[s];
                    rem[s] = REM_FREE;
                    ridx[s] = -1;
                }
            freed = (int64_t)shfl64((int64_t)freed, w_slot & 31);
            M -= freed;
            if (lane == 0) {
                bm[w_idx >> 5] &= ~(1u << (w_idx & 31));   // waits again
                if (meta_ok) {
                    ChunkMeta *slot = ring + ((w_idx >> 5) % CHUNK_RING);
                    ChunkMeta mt = *slot;
                    const int32_t e = (int32_t)est_of(w_est);
                    if (mt.wait == 0u) {
                        mt.a_first = w_arr;
                        mt.e_min = e;
                    } else {
                        mt.a_first = w_arr < mt.a_first ? w_arr : mt.a_first;
                        mt.e_min = e < mt.e_min ? e : mt.e_min;
                    }
                    mt.wait |= 1u << (w_idx & 31);
                    *slot = mt;
                }
            }
            __syncwarp();
            lo = w_idx < lo ? w_idx : lo;
            --nR;
            ++nW;
            ++preempted;
            blocked = false;
        }
        if (bad) break;
        n_pre += preempted;
        // ---- 3b. admission (only in a step without preemption), best first, head of line
        uint32_t newly = 0;
        uint32_t dur_sum_part = 0;
        int k = 0;
        if (preempted == 0 && !blocked) {
            // the chunk bounds must cover the window (an eviction may have moved lo back)
            const int c_lo = lo >> 5, c_hi = (p - 1) >> 5;
            const bool ringed = nW > 0 && c_hi - c_lo + 1 <= CHUNK_RING - 1;
            if (!ringed) {
                meta_ok = false;
            } else if (!meta_ok && nR < slots) {
                for (int c = c_lo; c <= c_hi; ++c) chunk_rebuild(trace, bm, ring, c, lo, p, lane);
                meta_ok = true;
                __syncwarp();
            }
            while (nW > 0 && nR < slots) {
                int64_t b_arr = 0;
                int32_t b_est = 0, b_dur = 0, b_idx = -1;
                if (ringed) {
                    chunk_pick(trace, ring, c_lo, c_hi, pol, t, lane, b_arr, b_est, b_dur, b_idx);
                } else {
                for (int c = lo & ~31; c < p; c += 32) {
                    const uint32_t word = bm[c >> 5];
                    const int i = c + lane;
                    if (i >= lo && i < p && !((word >> lane) & 1u)) {
                        const Rec q = ld_cached(trace + i);
                        if (b_idx < 0 || better_rt(pol, q.arrival_us, q.est, i, b_arr, b_est, b_idx, t)) {
                            b_arr = q.arrival_us;
                            b_est = q.est;
                            b_dur = q.dur_ms;
                            b_idx = i;
                        }
                    }
                }
#pragma unroll
                for (int j = 16; j > 0; j >>= 1) {
                    const int64_t o_arr = (int64_t)shfl64_xor((uint64_t)b_arr, j);
                    const int32_t o_est = __shfl_xor_sync(ASR_FULL_MASK, b_est, j);
                    const int32_t o_dur = __shfl_xor_sync(ASR_FULL_MASK, b_dur, j);
                    const int32_t o_idx = __shfl_xor_sync(ASR_FULL_MASK, b_idx, j);
                    if (o_idx >= 0 &&
                        (b_idx < 0 || better_rt(pol, o_arr, o_est, o_idx, b_arr, b_est, b_idx, t))) {
                        b_arr = o_arr;
                        b_est = o_est;
                        b_dur = o_dur;
                        b_idx = o_idx;
                    }
                }
                }
                const int64_t kv = B > 0 ? kv_enc(ex, b_dur) : 0;
                if (B > 0 && M + kv + nR + 1 > B) {   // the head of the line does not fit
                    blocked = true;
                    if (nR == 0) bad = true;   // not even alone
                    break;
                }
                const uint32_t had = (ever[b_idx >> 5] >> (b_idx & 31)) & 1u;
                __syncwarp();
                if (lane == 0) {
                    bm[b_idx >> 5] |= 1u << (b_idx & 31);
                    ever[b_idx >> 5] |= 1u << (b_idx & 31);
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
                            rest[s] = b_est;
                            rarr[s] = b_arr;
                            rmem[s] = kv;
                            dur_sum_part += (uint32_t)b_dur;
                            if (!had) newly |= 1u << s;   // TTFT: first admission only
                        }
                        seated = true;
                    }
                }
                __syncwarp();
                M += kv;
                ++nR;
                --nW;
                ++k;
            }
            if (nW == 0) {
                lo = p;
            } else {
                while (lo < p) {   // advance lo past admitted requests
                    const uint32_t word = ~bm[lo >> 5] & ~((1u << (lo & 31)) - 1u);
                    if (word) {
                        lo = (lo & ~31) + __ffs(word) - 1;
                        break;
                    }
                    lo = (lo & ~31) + 32;
                }
                if (lo > p) lo = p;
            }
        }
        if (bad) break;
        // ---- 4. one engine iteration with the encoders of the admitted ...
        const int64_t c = cm.iter_base_us + cm.iter_per_running_us * (int64_t)nR;
        const int64_t t0 = t;
        int64_t t1 = t + c;
        if (k > 0) {
            const int64_t dur_sum = warp_sum_u32(dur_sum_part);
            t1 += cm.enc_base_us * (int64_t)k + cm.enc_per_ms_us * dur_sum;
#pragma unroll
            for (int s = 0; s < SPL; ++s)
                if ((newly >> s) & 1u) ttft[ridx[s]] = t1 - rarr[s];
        }
        // ---- ... then fast-forward to the next event
        int32_t my_min = rem[0];
#pragma unroll
        for (int s = 1; s < SPL; ++s) my_min = rem[s] < my_min ? rem[s] : my_min;
        const int32_t m = __reduce_min_sync(ASR_FULL_MASK, my_min);   // nR >= 1 here
        int64_t j = 1;
        const bool may_admit = nW > 0 && nR < slots && !blocked;   // the next boundary is a scheduling event
        if (m > 1 && !may_admit) {
            if (nR == slots || p >= n || c <= 0) {
                j = m;
            } else {
                const int64_t g = ld_cached(trace + p).arrival_us - t1;
                if (g <= 0) j = 1;
                else if (g > (int64_t)(m - 2) * c) j = m;
                else j = 1 + ceil_div_pos(g, c);
            }
            if (B > 0) {   // iterations the budget allows after this one: M + nR*(1 + x) + ... <= B
                const int64_t room = B - (M + nR);          // >= 0: this iteration fits
                const int64_t jm = 1 + room / nR;
                j = j < jm ? j : jm;
            }
        }
        t = t1 + (j - 1) * c;
        if (a.itl_hist) {
            // inter-token gaps: this step's first iteration lasted t1 - t0 for the
            // requests that were already running; the j-1 fast-forwarded ones cost c for everybody
            const int already = nR - k;
            if (k > 0) {
                if (already > 0) {
                    if (lane == 0) {
                        a.itl_pairs[2 * (rep.out_off + n_pairs)] = t1 - t0;
                        a.itl_pairs[2 * (rep.out_off + n_pairs) + 1] = already;
                    }
                    ++n_pairs;
                }
            } else if (lane == 0) {
                a.itl_hist[(int64_t)r * ITL_BINS + nR] += (unsigned long long)nR;
            }
            if (j > 1 && lane == 0)
                a.itl_hist[(int64_t)r * ITL_BINS + nR] += (unsigned long long)(j - 1) * (unsigned long long)nR;
        }
        // ---- 5. tokens, memory, completions
        M += j * (int64_t)nR;
        int fin = 0;
        int64_t freed = 0;
#pragma unroll
        for (int s = 0; s < SPL; ++s) {
            if (rem[s] != REM_FREE) {
                rem[s] -= (int32_t)j;
                rmem[s] += j;
                if (rem[s] == 0) {
                    lat[ridx[s]] = t - rarr[s];
                    freed += rmem[s];
                    rem[s] = REM_FREE;
                    ridx[s] = -1;
                    fin++;
                }
            }
        }
        const int nfin = __reduce_add_sync(ASR_FULL_MASK, fin);
        if (nfin > 0) {
            // 64-bit sum over the warp of the freed units
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) freed += (int64_t)shfl64_xor((uint64_t)freed, d);
            M -= freed;
            blocked = false;
        }
        nR -= nfin;
        done += nfin;
    }
    if (lane == 0) {
        if (bad) {
            flag_invalid(a, r);
        } else if (a.out_summary) {
            asr_summary_t *s = a.out_summary + r;
            s->first_arrival_us = first_arrival;
            s->last_done_us = t;
            s->n_done = done;
        }
        if (a.out_preempt) a.out_preempt[r] = n_pre;
        if (a.itl_npairs) a.itl_npairs[r] = bad ? -1 : n_pairs;
    }
}

template <int SPL>
#ifndef SIM_EX_MIN_CTAS
#define SIM_EX_MIN_CTAS 6
#endif
__global__ void __launch_bounds__(SIM_WARPS * 32, SPL == 1 ? SIM_EX_MIN_CTAS : 1) sim_ex_kernel(SimExArgs a) {
    __shared__ ChunkMeta s_ring[SIM_WARPS][CHUNK_RING];
    const int gw = (blockIdx.x * SIM_WARPS) + (threadIdx.x >> 5);
    if (gw < a.n_replicas) sim_ex_replica<SPL>(a, gw, s_ring[threadIdx.x >> 5]);
}

template <int SPL>
static void launch_ex(const SimExArgs &a, cudaStream_t st) {
    KernelTimer kt(KID_SIM_EX, st);
    sim_ex_kernel<SPL><<<(a.n_replicas + SIM_WARPS - 1) / SIM_WARPS, SIM_WARPS * 32, 0, st>>>(a);
}

int launch_simulate_ex(const SimExArgs &a, int max_slots, cudaStream_t st) {
    if (a.n_replicas <= 0) return ASR_OK;
    if (max_slots <= 32) launch_ex<1>(a, st);
    else if (max_slots <= 64) launch_ex<2>(a, st);
    else if (max_slots <= 128) launch_ex<4>(a, st);
    else launch_ex<8>(a, st);
    return check_launch("sim_ex_kernel");
}

}  // namespace asr

// percentiles.cu -- a6 segmented nearest-rank percentiles, sm_100a.
//
// One CTA per segment, the segment read from HBM exactly once.
//
// Register path (segments of up to 10,240 values whose high 32-bit words are
// all equal -- every latency below 71 minutes): each thread keeps the low
// words of 40 values in registers and the ranks are found by an MSB-first
// radix select WITHOUT shared-memory atomics (2 cycles per lane on this part,
// which made the histogram the bottleneck): every lane counts into its own
// private byte counters, laid out [warp][bin][lane] with a 36-byte bin stride
// so that both the counting and the column sums are free of systematic bank
// conflicts; the column sums use dp4a.  One counting pass over all values
// serves all requested ranks; each rank then continues on the few hundred
// values of its own bin, compacted into shared memory.
//
// General path (anything else): min/max, then MSB-first radix select over
// (value - min) with 8-bit digits and a 256-bin shared-memory histogram, only
// as many passes as the value range needs.
// Nearest rank (asr_sched.h): element of 1-based rank
// ceil(p*N/100) of the sorted segment; an empty segment gives -1.
#include "launchers.cuh"
#ifdef PCT_STATS
#include <cstdio>
#endif

namespace asr {

#ifndef PCT_MIN_CTAS
#define PCT_MIN_CTAS 3
#endif
#ifndef PCT_THREADS_N
#define PCT_THREADS_N 256
#endif
constexpr int PCT_THREADS = PCT_THREADS_N;   // 256 (40 values per thread) or 320 (32 values per thread)
static_assert(PCT_THREADS >= 256 && PCT_THREADS % 64 == 0 && 10240 % PCT_THREADS == 0, "see PCT_VPT");
constexpr int PCT_SMEM_VALUES = 12288;   // 96 KB of int64 staged per CTA
constexpr int PCT_MAX = 8;

struct PctList {
    int32_t n_pct;
    int32_t pct[PCT_MAX];
};

__device__ __forceinline__ int64_t block_reduce_minmax(int64_t v, bool is_min, int64_t *scratch) {
    const int lane = lane_id(), warp = threadIdx.x >> 5;
#pragma unroll
    for (int j = 16; j > 0; j >>= 1) {
        int64_t o = (int64_t)shfl64_xor((uint64_t)v, j);
        v = is_min ? (o < v ? o : v) : (o > v ? o : v);
    }
    __syncthreads();
    if (lane == 0) scratch[warp] = v;
    __syncthreads();
    int64_t r = scratch[0];
    for (int w = 1; w < PCT_THREADS / 32; ++w) {
        int64_t o = scratch[w];
        r = is_min ? (o < r ? o : r) : (o > r ? o : r);
    }
    return r;
}

// All threads of the CTA call this; results[j] valid on every thread afterwards.
__device__ void segment_percentiles(const int64_t *__restrict__ v, int64_t N, const PctList &pl,
                                    int64_t *results, int64_t *smem_vals, bool is32 = false) {
    const uint32_t *v32 = reinterpret_cast<const uint32_t *>(v);   // is32: N uint32 values at the same address
    __shared__ uint32_t hist[256];
    __shared__ int64_t scratch[PCT_THREADS / 32];
    __shared__ uint32_t sel_digit, sel_below;

    if (N <= 0) {
        for (int j = 0; j < pl.n_pct; ++j) results[j] = -1;
        return;
    }
    const bool staged = smem_vals != nullptr && N <= PCT_SMEM_VALUES;
    int64_t mn = INT64_MAX, mx = INT64_MIN;
    for (int64_t i = threadIdx.x; i < N; i += PCT_THREADS) {
        int64_t x = is32 ? (int64_t)v32[i] : v[i];
        if (staged) smem_vals[i] = x;
        mn = x < mn ? x : mn;
        mx = x > mx ? x : mx;
    }
    mn = block_reduce_minmax(mn, true, scratch);
    mx = block_reduce_minmax(mx, false, scratch);
    const int64_t *src = staged ? smem_vals : v;
    const uint64_t range = (uint64_t)mx - (uint64_t)mn;
    const int bits = range == 0 ? 0 : 64 - __clzll((long long)range);
    const int top_shift = bits <= 8 ? 0 : ((bits + 7) / 8 - 1) * 8;

    for (int j = 0; j < pl.n_pct; ++j) {
        // 1-based rank ceil(p*N/100)
        uint64_t kk = ((uint64_t)pl.pct[j] * (uint64_t)N + 99) / 100;
        uint64_t prefix = 0;   // known digits above `shift`
        if (bits > 0) {
            for (int shift = top_shift;; shift -= 8) {
                __syncthreads();
                if (PCT_THREADS == 256 || threadIdx.x < 256) hist[threadIdx.x] = 0;
                __syncthreads();
                for (int64_t i = threadIdx.x; i < N; i += PCT_THREADS) {
                    uint64_t key = (uint64_t)((is32 && !staged) ? (int64_t)v32[i] : src[i]) - (uint64_t)mn;
                    if (shift + 8 >= 64 || (key >> (shift + 8)) == prefix)
                        atomicAdd(&hist[(key >> shift) & 255u], 1u);
                }
                __syncthreads();
                if (threadIdx.x < 32) {
                    // lane L owns bins 8L..8L+7
                    uint32_t c[8], tot = 0;
#pragma unroll
                    for (int b = 0; b < 8; ++b) {
                        c[b] = hist[threadIdx.x * 8 + b];
                        tot += c[b];
                    }
                    uint32_t incl = tot;
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) {
                        uint32_t y = __shfl_up_sync(ASR_FULL_MASK, incl, d);
                        if ((int)threadIdx.x >= d) incl += y;
                    }
                    uint32_t excl = incl - tot;
                    if ((uint64_t)excl < kk && kk <= (uint64_t)incl) {
                        uint32_t run = excl;
#pragma unroll
                        for (int b = 0; b < 8; ++b) {
                            if ((uint64_t)run < kk && kk <= (uint64_t)(run + c[b])) {
                                sel_digit = threadIdx.x * 8 + b;
                                sel_below = run;
                            }
                            run += c[b];
                        }
                    }
                }
                __syncthreads();
                prefix = (prefix << 8) | sel_digit;
                kk -= sel_below;
                if (shift == 0) break;
            }
        }
        results[j] = (int64_t)((uint64_t)mn + prefix);
    }
    __syncthreads();
}


// ---------------------------------------------------------------------------
// register path
// ---------------------------------------------------------------------------
constexpr int PCT_VPT = 10240 / PCT_THREADS;                 // values per thread
static_assert(PCT_VPT % 4 == 0 && PCT_VPT <= 64, "quads of values per 128-bit load, two 32-bit match masks");
constexpr int PCT_REG_MAX = PCT_THREADS * PCT_VPT;           // 10,240 values
#ifndef PCT_DIG_N
#define PCT_DIG_N 7
#endif
constexpr int PCT_DIG = PCT_DIG_N;                                   // digit width of a counting pass
constexpr int PCT_BINS = 1 << PCT_DIG;
constexpr int PCT_BIN_STRIDE = 36;                           // bytes: 32 lane counters + 4 padding
constexpr int PCT_TAB_BYTES = PCT_BINS * PCT_BIN_STRIDE;     // per warp
constexpr int PCT_CAND = 1024;                               // candidates finished in shared memory

struct PctRegSmem {
    unsigned char tab[PCT_THREADS / 32][PCT_TAB_BYTES];      // private byte counters
    uint32_t part[2][PCT_BINS];                              // column sums of warps 0-3 / 4-7
    uint32_t cand[2][PCT_CAND];                              // candidates of a pair of targets
    uint32_t hist[2][256];
    uint32_t warp_cnt[PCT_THREADS / 32];
    uint32_t warp_or[PCT_THREADS / 32];
    uint32_t sel_digit[PCT_MAX], sel_below[PCT_MAX], sel_pop[PCT_MAX];
    uint32_t n_cand;
};

// One counting pass over the register-resident keys.  Counts digit
// (key >> new_shift) & (2^width - 1) of every key with key >> shift == prefix
// (no filter when shift >= 32) among the thread's first nvalid slots, then
// resolves every rank kk[t] of the targets [t0, t1): sel_digit/sel_below/sel_pop.
__device__ __forceinline__ void reg_count_pass(const uint32_t (&key)[PCT_VPT], int nvalid, int shift, int new_shift,
                                               uint32_t prefix, const uint32_t *kk, int t0, int t1,
                                               PctRegSmem &sm) {
    const int lane = lane_id(), warp = threadIdx.x >> 5;
    const uint32_t mask = (1u << (shift - new_shift)) - 1u;
    // zero the private counters
    {
        uint4 *z = reinterpret_cast<uint4 *>(&sm.tab[0][0]);
        constexpr int n16 = (PCT_THREADS / 32) * PCT_TAB_BYTES / 16;
        for (int i = threadIdx.x; i < n16; i += PCT_THREADS) z[i] = make_uint4(0, 0, 0, 0);
    }
    __syncthreads();
    unsigned char *mine = &sm.tab[warp][lane];
#pragma unroll
    for (int j = 0; j < PCT_VPT; ++j) {
        const bool in = j < nvalid && (shift >= 32 || (key[j] >> shift) == prefix);
        if (in) {
            unsigned char *c = mine + ((key[j] >> new_shift) & mask) * PCT_BIN_STRIDE;
            *c = (unsigned char)(*c + 1);
        }
    }
    __syncthreads();
    // column sums: thread (half, bin) adds the 32 lane counters of its half of the warps
    if (PCT_THREADS == 2 * PCT_BINS || threadIdx.x < 2 * PCT_BINS) {
        constexpr int HW = PCT_THREADS / 64;   // warps per half
        const int bin = threadIdx.x & (PCT_BINS - 1), half = threadIdx.x >> PCT_DIG;
        uint32_t tot = 0;
#pragma unroll
        for (int w = 0; w < HW; ++w) {
            const uint32_t *row = reinterpret_cast<const uint32_t *>(&sm.tab[half * HW + w][bin * PCT_BIN_STRIDE]);
#pragma unroll
            for (int q = 0; q < 8; ++q) tot = __dp4a(row[q], 0x01010101u, tot);
        }
        sm.part[half][bin] = tot;
    }
    __syncthreads();
    if (warp == 0) {
        // lane L owns bins BPL*L .. BPL*L + BPL-1
        constexpr int BPL = PCT_BINS / 32;
        uint32_t c[BPL], tot = 0;
#pragma unroll
        for (int b = 0; b < BPL; ++b) {
            c[b] = sm.part[0][lane * BPL + b] + sm.part[1][lane * BPL + b];
            tot += c[b];
        }
        uint32_t incl = tot;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t y = __shfl_up_sync(ASR_FULL_MASK, incl, d);
            if (lane >= d) incl += y;
        }
        const uint32_t excl = incl - tot;
        for (int t = t0; t < t1; ++t) {
            const uint32_t k = kk[t];
            if (excl < k && k <= incl) {
                uint32_t run = excl;
#pragma unroll
                for (int b = 0; b < BPL; ++b) {
                    if (run < k && k <= run + c[b]) {
                        sm.sel_digit[t] = (uint32_t)(lane * BPL + b);
                        sm.sel_below[t] = run;
                        sm.sel_pop[t] = c[b];
                    }
                    run += c[b];
                }
            }
        }
    }
    __syncthreads();
}

// Returns false (nothing written) when the segment does not qualify.
template <int MAXT, bool IS32>
__device__ __forceinline__ bool segment_percentiles_reg(const int64_t *__restrict__ v, int64_t N64, const PctList &pl,
                                        int64_t *results, PctRegSmem &sm) {
    if (N64 <= 0 || N64 > PCT_REG_MAX) return false;
    const int N = (int)N64;
    const int lane = lane_id(), warp = threadIdx.x >> 5;
    uint32_t key[PCT_VPT];
    uint32_t hi0 = 0, hi_diff = 0, or_all = 0;
    if (IS32) {   // N uint32 values (the lane kernel's order-free format): no high words to compare
        // which slot holds which value is irrelevant to a rank: four consecutive values per 128-bit load;
        // a segment that is not made of whole aligned quads takes the general path
        if ((N & 3) != 0 || (reinterpret_cast<uintptr_t>(v) & 15u) != 0) return false;
        const uint4 *v128 = reinterpret_cast<const uint4 *>(v);
        const int n4 = N >> 2;
#pragma unroll
        for (int q = 0; q < PCT_VPT / 4; ++q) {
            const int i = q * PCT_THREADS + threadIdx.x;
            uint4 x = make_uint4(0u, 0u, 0u, 0u);
            if (i < n4) x = __ldcs(v128 + i);
            key[4 * q] = x.x;
            key[4 * q + 1] = x.y;
            key[4 * q + 2] = x.z;
            key[4 * q + 3] = x.w;
            or_all |= (x.x | x.y) | (x.z | x.w);
        }
    } else {
        hi0 = (uint32_t)((uint64_t)__ldg(reinterpret_cast<const long long *>(v)) >> 32);
#pragma unroll
        for (int j = 0; j < PCT_VPT; ++j) {
            const int i = j * PCT_THREADS + threadIdx.x;
            uint64_t x = (uint64_t)hi0 << 32;
            if (i < N) x = (uint64_t)__ldcs(reinterpret_cast<const long long *>(v + i));   // read once: streaming
            key[j] = (uint32_t)x;
            hi_diff |= (uint32_t)(x >> 32) ^ hi0;
            or_all |= (uint32_t)x;
        }
    }
    // the thread's valid slots are a prefix of its PCT_VPT slots under both layouts
    int nvalid;
    if (IS32) {
        const int n4 = N >> 2;
        nvalid = n4 > (int)threadIdx.x ? 4 * ((n4 - (int)threadIdx.x + PCT_THREADS - 1) / PCT_THREADS) : 0;
    } else {
        nvalid = N > (int)threadIdx.x ? (N - (int)threadIdx.x + PCT_THREADS - 1) / PCT_THREADS : 0;
    }
    if (__syncthreads_or(hi_diff != 0u)) return false;
    or_all = __reduce_or_sync(ASR_FULL_MASK, or_all);
    if (lane == 0) sm.warp_or[warp] = or_all;
    __syncthreads();
    or_all = 0;
#pragma unroll
    for (int w = 0; w < PCT_THREADS / 32; ++w) or_all |= sm.warp_or[w];
    const int bits = or_all == 0u ? 0 : 32 - __clz((int)or_all);

    uint32_t kk[MAXT], prefix[MAXT];
#pragma unroll
    for (int t = 0; t < MAXT; ++t) {
        kk[t] = t < pl.n_pct ? ((uint32_t)pl.pct[t] * (uint32_t)N + 99u) / 100u : 0u;   // 1-based rank; pct <= 100, N <= 10,240
        prefix[t] = 0;
    }
    if (bits > 0) {
        // first pass: all targets at once, no filter (every key >> bits is 0)
        const int sh1 = bits > PCT_DIG ? bits - PCT_DIG : 0;
        reg_count_pass(key, nvalid, 32, sh1, 0u, kk, 0, pl.n_pct, sm);
        uint32_t pop[MAXT];
#pragma unroll
        for (int t = 0; t < MAXT; ++t)
            if (t < pl.n_pct) {
                prefix[t] = sm.sel_digit[t];
                kk[t] -= sm.sel_below[t];
                pop[t] = sm.sel_pop[t];
            }
        __syncthreads();
        int shiftv[MAXT];
#pragma unroll
        for (int t = 0; t < MAXT; ++t) shiftv[t] = sh1;
#pragma unroll
        for (int t = 0; t < MAXT; ++t) {
            if (t >= pl.n_pct) break;
            int shift = sh1;
            // more counting passes while the bin is too crowded for the candidate buffer
            while (shift > 0 && pop[t] > (uint32_t)PCT_CAND) {
                const int ns = shift > PCT_DIG ? shift - PCT_DIG : 0;
                reg_count_pass(key, nvalid, shift, ns, prefix[t], kk, t, t + 1, sm);
                prefix[t] = (prefix[t] << (shift - ns)) | sm.sel_digit[t];
                kk[t] -= sm.sel_below[t];
                pop[t] = sm.sel_pop[t];
                shift = ns;
                __syncthreads();
            }
            shiftv[t] = shift;
        }
        // targets two at a time: compact the keys of both selected bins into shared memory
        // (private counts, one block scan, no ballots), then finish both on the candidates
#pragma unroll
        for (int t0 = 0; t0 < MAXT; t0 += 2) {
            if (t0 >= pl.n_pct) break;
            const bool two = t0 + 1 < MAXT && t0 + 1 < pl.n_pct;
            const int sa = shiftv[t0], sb = two ? shiftv[t0 + 1 < MAXT ? t0 + 1 : t0] : 0;
            const uint32_t pa = prefix[t0], pb = two ? prefix[t0 + 1 < MAXT ? t0 + 1 : t0] : 0u;
            const bool do_a = sa > 0, do_b = two && sb > 0;
            if (!do_a && !do_b) continue;
            // an inactive target matches nothing: shift 31 against an impossible prefix (keys < 2^32)
            const int sha = do_a ? sa : 31, shb = do_b ? sb : 31;
            const uint32_t pra = do_a ? pa : 2u, prb = do_b ? pb : 2u;
            // match masks of this thread's values (bit j of word j/32), per target
            uint32_t ma0 = 0, ma1 = 0, mb0 = 0, mb1 = 0;
#pragma unroll
            for (int j = 0; j < PCT_VPT; ++j) {
                const bool ia = (key[j] >> sha) == pra, ibb = (key[j] >> shb) == prb;
                if (j < 32) {
                    ma0 |= ia ? (1u << j) : 0u;
                    mb0 |= ibb ? (1u << j) : 0u;
                } else {
                    ma1 |= ia ? (1u << (j - 32)) : 0u;
                    mb1 |= ibb ? (1u << (j - 32)) : 0u;
                }
            }
            {   // drop the slots past the end of the segment
                const uint32_t v0 = nvalid >= 32 ? 0xFFFFFFFFu : ((1u << nvalid) - 1u);
                const uint32_t v1 = nvalid > 32 ? ((1u << (nvalid - 32)) - 1u) : 0u;
                ma0 &= v0;
                mb0 &= v0;
                ma1 &= v1;
                mb1 &= v1;
            }
            // matches of target a in the low half, of target b in the high half
            const uint32_t cnt = (uint32_t)(__popc(ma0) + __popc(ma1)) + ((uint32_t)(__popc(mb0) + __popc(mb1)) << 16);
            uint32_t incl = cnt;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t y = __shfl_up_sync(ASR_FULL_MASK, incl, d);
                if (lane >= d) incl += y;
            }
            if (lane == 31) sm.warp_cnt[warp] = incl;
            __syncthreads();
            uint32_t base = incl - cnt;
            uint32_t total = 0;
#pragma unroll
            for (int w = 0; w < PCT_THREADS / 32; ++w) {
                const uint32_t c = sm.warp_cnt[w];
                if (w < warp) base += c;
                total += c;
            }
            uint32_t *wa = &sm.cand[0][base & 0xFFFFu], *wb = &sm.cand[1][base >> 16];
#pragma unroll
            for (int j = 0; j < PCT_VPT; ++j) {
                const uint32_t bit = 1u << (j & 31);
                if ((j < 32 ? ma0 : ma1) & bit) *wa++ = key[j];
                if ((j < 32 ? mb0 : mb1) & bit) *wb++ = key[j];
            }
            const int Ca = (int)(total & 0xFFFFu), Cb = (int)(total >> 16);   // == pop[t0], pop[t0+1]
            // finish on the candidates: 8-bit digits, shared-memory histograms (few values);
            // warp 0 resolves target a, warp 1 target b
            int s_a = do_a ? sa : 0, s_b = do_b ? sb : 0;
            uint32_t p_a = pa, p_b = pb, k_a = kk[t0], k_b = two ? kk[t0 + 1 < MAXT ? t0 + 1 : t0] : 0u;
            while (s_a > 0 || s_b > 0) {
                const int na = s_a > 8 ? s_a - 8 : 0, nb = s_b > 8 ? s_b - 8 : 0;
                if (PCT_THREADS == 256 || threadIdx.x < 256) {
                    sm.hist[0][threadIdx.x] = 0;
                    sm.hist[1][threadIdx.x] = 0;
                }
                __syncthreads();               // also orders the candidate stores above
                if (s_a > 0) {
                    const uint32_t mask = (1u << (s_a - na)) - 1u;
                    for (int i = threadIdx.x; i < Ca; i += PCT_THREADS) {
                        const uint32_t x = sm.cand[0][i];
                        if ((x >> s_a) == p_a) atomicAdd(&sm.hist[0][(x >> na) & mask], 1u);
                    }
                }
                if (s_b > 0) {
                    const uint32_t mask = (1u << (s_b - nb)) - 1u;
                    for (int i = threadIdx.x; i < Cb; i += PCT_THREADS) {
                        const uint32_t x = sm.cand[1][i];
                        if ((x >> s_b) == p_b) atomicAdd(&sm.hist[1][(x >> nb) & mask], 1u);
                    }
                }
                __syncthreads();
                if (warp < 2 && (warp == 0 ? s_a > 0 : s_b > 0)) {
                    const uint32_t *h = sm.hist[warp];
                    uint32_t c[8], tot = 0;
#pragma unroll
                    for (int b8 = 0; b8 < 8; ++b8) {
                        c[b8] = h[lane * 8 + b8];
                        tot += c[b8];
                    }
                    uint32_t inc = tot;
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) {
                        const uint32_t y = __shfl_up_sync(ASR_FULL_MASK, inc, d);
                        if (lane >= d) inc += y;
                    }
                    const uint32_t excl = inc - tot, k = warp == 0 ? k_a : k_b;
                    if (excl < k && k <= inc) {
                        uint32_t run = excl;
#pragma unroll
                        for (int b8 = 0; b8 < 8; ++b8) {
                            if (run < k && k <= run + c[b8]) {
                                sm.sel_digit[t0 + warp] = (uint32_t)(lane * 8 + b8);
                                sm.sel_below[t0 + warp] = run;
                            }
                            run += c[b8];
                        }
                    }
                }
                __syncthreads();
                if (s_a > 0) {
                    p_a = (p_a << (s_a - na)) | sm.sel_digit[t0];
                    k_a -= sm.sel_below[t0];
                    s_a = na;
                }
                if (s_b > 0) {
                    p_b = (p_b << (s_b - nb)) | sm.sel_digit[t0 + 1];
                    k_b -= sm.sel_below[t0 + 1];
                    s_b = nb;
                }
                __syncthreads();
            }
            if (do_a) prefix[t0] = p_a;
            if (do_b) prefix[t0 + 1 < MAXT ? t0 + 1 : t0] = p_b;
        }
    }
#pragma unroll
    for (int t = 0; t < MAXT; ++t)
        if (t < pl.n_pct) results[t] = (int64_t)(((uint64_t)hi0 << 32) | prefix[t]);
    __syncthreads();
    return true;
}


#ifdef PCT_STATS
__device__ unsigned long long g_pct_stats[8];   // -, settled, passes, above, dense, in-window keys, below, -
#endif
// ---------------------------------------------------------------------------
// summary_stream_kernel: p50/p90 of the uint32 segments of a summary-only sweep, one WARP per segment.
//
// Consecutive segments of a sweep are alike (the same trace under another policy, the neighbouring seed), so the
// two ranks of a segment are looked for in windows of values around the answers of the segment before.  (Round 2
// first did this with one CTA per segment: eight barriers and two block scans per segment made the fixed work
// 60 % of its instructions.)  A warp takes a run of consecutive work items -- a work item is one value stream of one
// replica, in the plan's order -- and streams each segment ONCE through its registers, 4 KB at a time with the next
// 4 KB's loads in flight and the rest of the segment prefetched into L2.  (A cp.async.bulk ring in shared memory
// as in select_topk_kernel was measured too: 13 warps per SM fit beside it and run in 2.1 ms, 19 warps without it
// in 1.96 ms.)  Per key and rank: count below the window's end, append to the lane's private slots if inside the
// window -- ten PTX instructions per key for both ranks.  The window is then resolved by a radix descent with 32
// bins over the ~150 collected keys and a one-warp ranking of the last bin's keys: warp shuffles only, no block
// barrier anywhere.  A rank just outside the window re-centres it, a rank far outside moves and doubles it, a lane
// that runs out of slots halves it, and the segment is read again (mostly from L2); what is not settled after
// PS_TRIES passes, or has another format, goes to the miss list for summary_percentiles_kernel.  The first
// streamable item of every PS_SEED_EVERY runs (the "seed") is computed by that kernel beforehand: its two answers
// and their distance give the runs their first windows.  No result depends on a guess.
// ---------------------------------------------------------------------------
#ifndef PS_WARPS_N
#define PS_WARPS_N 19
#endif
constexpr int PS_WARPS = PS_WARPS_N;
#ifndef PS_CHUNK_N
#define PS_CHUNK_N 1024
#endif
constexpr int PS_CHUNK = PS_CHUNK_N;   // keys a warp takes at a time (4 KB: one 128-bit load per lane and 512 bytes)
constexpr int PS_WIN = 32;       // a window is PS_WIN << shift values wide: 32 bins of 2^shift values
#ifndef PS_SLOTS_N
#define PS_SLOTS_N 32
#endif
constexpr int PS_SLOTS = PS_SLOTS_N;   // private slots per lane and rank
constexpr int PS_GROUP = 8;      // slots are checked once per group of keys
constexpr int PS_TRIES = 6;
constexpr int PS_MAX_SHIFT = 26;
#ifndef PS_IN_MANY_N
#define PS_IN_MANY_N 256
#endif
constexpr uint32_t PS_IN_MANY = PS_IN_MANY_N, PS_IN_FEW = PS_IN_MANY / 4;   // keys wanted inside a window
#ifndef PS_RUN_N
#define PS_RUN_N 24
#endif
#ifndef PS_SEED_EVERY_N
#define PS_SEED_EVERY_N 8
#endif
constexpr int PS_SEED_EVERY = PS_SEED_EVERY_N;   // runs that share a seed
constexpr int PS_RUN = PS_RUN_N;   // consecutive work items per run (each run costs one seed: a radix-kernel segment)
static_assert(PS_SLOTS >= 2 * PS_GROUP && (PS_CHUNK / 32) % PS_GROUP == 0, "slot check granularity");

struct __align__(128) PsWarpSmem {
    uint32_t slot[2][PS_SLOTS][32];   // [rank][slot][lane]
    uint32_t hist[32];
    uint32_t list[32];
    uint32_t lcnt;
};
constexpr size_t PS_SMEM_BYTES = sizeof(PsWarpSmem) * PS_WARPS;

// a work item w in [0, 2 * n_replicas): value stream w / n_replicas (0: E2E latency, 1: TTFT) of the replica at
// position w % n_replicas of the order.  state 0 = nothing to do (invalid replica, or the run's seed: done),
// 1 = uint32 values in the order-free simulator's format: streamed here, 2 = anything else: miss list
struct PsDesc {
    const uint32_t *base;
    int32_t N, r, y, state;
};

struct PsArgs {
    const asr_replica_t *replicas;
    const int64_t *lat, *ttft;
    asr_summary_t *out_summary;
    const int32_t *order;
    int32_t *miss_list, *miss_count;   // [2][n_replicas], [2]
    int32_t *seed_list, *seed_count;   // [2][n_replicas], [2]
    int32_t *seed_item;                // [groups of PS_SEED_EVERY runs]: the group's seed item, or -1
    int32_t *cursor;                   // the next run to hand out
    int32_t n_replicas, run, n_runs;   // run = consecutive work items a warp takes at a time
    uint32_t one;                      // 1 (see ps_chunk)
};

__device__ __forceinline__ PsDesc ps_describe(const PsArgs &a, int w, int seed) {
    PsDesc d;
    d.y = w >= a.n_replicas ? 1 : 0;
    const int idx = w - d.y * a.n_replicas;
    d.r = a.order ? a.order[idx] : idx;
    const asr_replica_t rp = a.replicas[d.r];
    const asr_summary_t *s = a.out_summary + d.r;
    const int64_t flag = d.y == 0 ? s->p50_e2e_us : s->p50_ttft_us;
    // (only a descriptor the simulator accepted, n_done >= 0, is ever dereferenced)
    const int64_t *vals = (d.y == 0 ? a.lat : a.ttft) + rp.out_off;
    d.base = reinterpret_cast<const uint32_t *>(vals);
    d.N = rp.n;
    if (w == seed || s->n_done < 0) d.state = 0;
    else if (flag == ASR_FMT32 && rp.n > 0 && (rp.n & 3) == 0 && (reinterpret_cast<uintptr_t>(vals) & 15u) == 0) d.state = 1;
    else d.state = 2;
    return d;
}

// one thread per group of PS_SEED_EVERY consecutive runs: the group's first streamable item becomes its seed
// (computed by summary_percentiles_kernel before summary_stream_kernel starts).  A seed costs as much as four
// second readings, and all a run needs from it is a first guess, so neighbouring runs share one.
__global__ void __launch_bounds__(1024) summary_seed_kernel(PsArgs a) {
    if (threadIdx.x < 2) a.seed_count[threadIdx.x] = 0;
    if (threadIdx.x == 2) *a.cursor = 0;
    __syncthreads();
    const int total = 2 * a.n_replicas;
    const int n_groups = (a.n_runs + PS_SEED_EVERY - 1) / PS_SEED_EVERY;
    for (int g = threadIdx.x; g < n_groups; g += 1024) {
        const int w0 = g * PS_SEED_EVERY * a.run, w1 = (int)min((int64_t)total, (int64_t)w0 + (int64_t)PS_SEED_EVERY * a.run);
        int seed = -1;
        for (int w = w0; w < w1 && seed < 0; ++w) {
            const PsDesc d = ps_describe(a, w, -1);
            if (d.state == 1) {
                seed = w;
                a.seed_list[(size_t)d.y * a.n_replicas + atomicAdd(a.seed_count + d.y, 1)] = d.r;
            }
        }
        a.seed_item[g] = seed;
    }
}

// the lane's state through one pass over a segment
struct PsPass {
    uint32_t c0, c1;             // keys below the end of window 0 / 1
    uint32_t p0, p1;             // next free slot (shared-memory byte address) of rank 0 / 1
    uint32_t lo0, hi0, lo1, hi1;
    uint32_t over;               // bit t: this lane closed window t for lack of slots
};

// 32 keys of a lane (one chunk): ten instructions per key, slots checked after every PS_GROUP keys.
// The four predicated increments are written as multiply-adds by `one` (a kernel argument equal to 1, so that
// ptxas cannot fold them back into additions): IMAD issues to the fma pipe, and the key then costs four
// instructions on the alu pipe (the compares) and four on the fma pipe, which run side by side at one warp
// instruction per two cycles each -- as plain additions all eight queue for the alu pipe.
__device__ __forceinline__ void ps_chunk(const uint32_t (&key)[PS_CHUNK / 32], PsPass &s, uint32_t stop0, uint32_t stop1,
                                         uint32_t one) {
    constexpr uint32_t ROW = 32 * 4;   // bytes between two slots of a lane
#pragma unroll
    for (int g = 0; g < PS_CHUNK / 32 / PS_GROUP; ++g) {
#pragma unroll
        for (int j = 0; j < PS_GROUP; ++j) {
            asm volatile(
                "{\n\t"
                ".reg .pred a, b;\n\t"
                "setp.lt.u32 a, %4, %5;\n\t"
                "@a mad.lo.u32 %0, %10, %10, %0;\n\t"
                "setp.ge.and.u32 b, %4, %6, a;\n\t"
                "@b st.shared.u32 [%1], %4;\n\t"
                "@b mad.lo.u32 %1, %10, %9, %1;\n\t"
                "setp.lt.u32 a, %4, %7;\n\t"
                "@a mad.lo.u32 %2, %10, %10, %2;\n\t"
                "setp.ge.and.u32 b, %4, %8, a;\n\t"
                "@b st.shared.u32 [%3], %4;\n\t"
                "@b mad.lo.u32 %3, %10, %9, %3;\n\t"
                "}"
                : "+r"(s.c0), "+r"(s.p0), "+r"(s.c1), "+r"(s.p1)
                : "r"(key[g * PS_GROUP + j]), "r"(s.hi0), "r"(s.lo0), "r"(s.hi1), "r"(s.lo1), "n"(ROW), "r"(one)
                : "memory");
        }
        // a lane that could run out of slots in the next group closes its window (rare: one test for both ranks)
        if (s.p0 > stop0 || s.p1 > stop1) {
            if (s.p0 > stop0) {
                s.lo0 = s.hi0;
                s.over |= 1u;
            }
            if (s.p1 > stop1) {
                s.lo1 = s.hi1;
                s.over |= 2u;
            }
        }
    }
}

__device__ __forceinline__ uint32_t ps_end(uint32_t lo, int sh) {   // saturated: a key 2^32-1 is never inside
    const uint32_t hi = lo + ((uint32_t)PS_WIN << sh);
    return hi < lo ? 0xFFFFFFFFu : hi;
}

// the j-th smallest (j >= 1) of the keys a pass collected for rank t: lane holds n_lane of them in its slots, all
// inside [lo, lo + (PS_WIN << sh)).  Radix descent, 32 bins (one per lane) per level, until the bin of the rank
// holds at most 32 keys (ranked by one key per lane) or one value.
__device__ __forceinline__ uint32_t ps_resolve(PsWarpSmem &sm, int t, int n_lane, uint32_t lo, int sh, uint32_t j) {
    const int lane = lane_id();
    const int n_max = (int)__reduce_max_sync(ASR_FULL_MASK, (uint32_t)n_lane);
    int shift = sh;   // the window is 32 bins of 2^sh values
    uint32_t cnt_b;
    for (;;) {
        sm.hist[lane] = 0;
        if (lane == 0) sm.lcnt = 0;
        __syncwarp();
        for (int e = 0; e < n_max; ++e)
            if (e < n_lane) {
                const uint32_t d = (sm.slot[t][e][lane] - lo) >> shift;   // (a key below lo wraps far beyond 32 bins)
                if (d < 32u) atomicAdd(&sm.hist[d], 1u);
            }
        __syncwarp();
        const uint32_t cnt = sm.hist[lane];
        uint32_t incl = cnt;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t y = __shfl_up_sync(ASR_FULL_MASK, incl, d);
            if (lane >= d) incl += y;
        }
        const int b = __ffs((int)__ballot_sync(ASR_FULL_MASK, incl >= j)) - 1;   // (the rank is inside: b >= 0)
        j -= __shfl_sync(ASR_FULL_MASK, incl - cnt, b);
        cnt_b = __shfl_sync(ASR_FULL_MASK, cnt, b);
        lo += (uint32_t)b << shift;
        if (shift == 0) return lo;   // one value per bin
        if (cnt_b <= 32u) break;
        shift = shift > 5 ? shift - 5 : 0;
    }
    // the keys of [lo, lo + 2^shift), one per lane, ranked by comparison (any order of equal keys gives the same
    // value at every rank)
    for (int e = 0; e < n_max; ++e)
        if (e < n_lane) {
            const uint32_t d = sm.slot[t][e][lane] - lo;
            if ((d >> shift) == 0u) sm.list[atomicAdd(&sm.lcnt, 1u)] = d;
        }
    __syncwarp();
    const uint32_t v = (uint32_t)lane < cnt_b ? sm.list[lane] : 0xFFFFFFFFu;
    uint32_t rank = 0;
    for (uint32_t q = 0; q < cnt_b; ++q) {
        const uint32_t u = __shfl_sync(ASR_FULL_MASK, v, (int)q);
        rank += (u < v || (u == v && q < (uint32_t)lane)) ? 1u : 0u;
    }
    const uint32_t hit = __ballot_sync(ASR_FULL_MASK, (uint32_t)lane < cnt_b && rank + 1u == j);
    const uint32_t res = lo + __shfl_sync(ASR_FULL_MASK, v, __ffs((int)hit) - 1);
    __syncwarp();   // list and hist are rewritten by the next call
    return res;
}

__global__ void __launch_bounds__(PS_WARPS * 32, 1) summary_stream_kernel(PsArgs a) {
    extern __shared__ __align__(128) unsigned char ps_dyn_smem[];
    PsWarpSmem *smem = reinterpret_cast<PsWarpSmem *>(ps_dyn_smem);
    const int lane = lane_id(), warp = threadIdx.x >> 5;
    PsWarpSmem &sm = smem[warp];
    // persistent warps take runs from a cursor: a run that needs many second readings does not hold up the rest
#pragma unroll 1
  for (;;) {
    int g = 0;
    if (lane == 0) g = atomicAdd(a.cursor, 1);
    g = __shfl_sync(ASR_FULL_MASK, g, 0);
    if (g >= a.n_runs) break;
    const int total = 2 * a.n_replicas;
    const int w0 = g * a.run, w1 = min(total, w0 + a.run);
    const int seed = a.seed_item[g / PS_SEED_EVERY];

    // the run's first windows: around the seed's answers, wide enough for ~100 of the keys between them
    uint32_t wlo[2] = {0, 0};
    int wsh[2] = {0, 0};
    bool have = false;
    if (seed >= 0) {
        const PsDesc d = ps_describe(a, seed, -1);
        const asr_summary_t *s = a.out_summary + d.r;
        const uint32_t r0 = (uint32_t)(d.y == 0 ? s->p50_e2e_us : s->p50_ttft_us);
        const uint32_t r1 = (uint32_t)(d.y == 0 ? s->p90_e2e_us : s->p90_ttft_us);
        const uint64_t width = ((uint64_t)(r1 - r0) * 256u) / (uint64_t)d.N;   // 0.4 N keys in r1 - r0: ~100 of them
        int sh = 0;
        while (sh < PS_MAX_SHIFT && ((uint64_t)PS_WIN << sh) < width) ++sh;
        const uint32_t half = (uint32_t)PS_WIN << sh >> 1;
        wlo[0] = r0 > half ? r0 - half : 0u;
        wlo[1] = r1 > half ? r1 - half : 0u;
        wsh[0] = wsh[1] = sh;
        have = true;
    }

    constexpr uint32_t ROW = 32 * 4;
    const uint32_t b0 = smem_u32(&sm.slot[0][0][lane]), b1 = smem_u32(&sm.slot[1][0][lane]);
    const uint32_t stop0 = b0 + (PS_SLOTS - PS_GROUP) * ROW, stop1 = b1 + (PS_SLOTS - PS_GROUP) * ROW;
#pragma unroll 1
    for (int w = w0; w < w1; ++w) {
        const PsDesc d = ps_describe(a, w, seed);
        if (d.state == 0) continue;
        bool settled = d.state == 1 && have;
        uint32_t res[2] = {0, 0};
        if (settled) {
            const uint32_t N = (uint32_t)d.N;
            const uint32_t k[2] = {(uint32_t)((50ull * N + 99ull) / 100ull), (uint32_t)((90ull * N + 99ull) / 100ull)};
            const int n4 = d.N >> 2, nch = (d.N + PS_CHUNK - 1) / PS_CHUNK;
            // the rest of the segment into L2 while its first chunk is on the way: a reading is ten 4 KB loads one
            // behind the other, and nine of them then come from L2 (1.97 -> 1.87 ms on config 3)
            if (lane == 0 && d.N > PS_CHUNK)
                asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(d.base + PS_CHUNK), "r"((uint32_t)(d.N - PS_CHUNK) * 4u) : "memory");
            for (int attempt = 0;; ++attempt) {
                PsPass s;
                s.c0 = s.c1 = 0;
                s.p0 = b0, s.p1 = b1;
                s.lo0 = wlo[0], s.hi0 = ps_end(wlo[0], wsh[0]);
                s.lo1 = wlo[1], s.hi1 = ps_end(wlo[1], wsh[1]);
                s.over = 0;
                // four consecutive keys per 128-bit load, the next chunk's loads in flight under this chunk's pass;
                // quads past the end read as 2^32-1 (below no window end)
                {
                    const uint4 *v = reinterpret_cast<const uint4 *>(d.base) + lane;
                    uint4 nx[PS_CHUNK / 128];
#pragma unroll
                    for (int q = 0; q < PS_CHUNK / 128; ++q) {
                        nx[q] = make_uint4(~0u, ~0u, ~0u, ~0u);
                        if (lane + q * 32 < n4) nx[q] = __ldcs(v + q * 32);
                    }
#pragma unroll 1
                    for (int c = 0; c < nch; ++c) {
                        uint32_t key[PS_CHUNK / 32];
#pragma unroll
                        for (int q = 0; q < PS_CHUNK / 128; ++q)
                            key[4 * q] = nx[q].x, key[4 * q + 1] = nx[q].y, key[4 * q + 2] = nx[q].z, key[4 * q + 3] = nx[q].w;
                        const int q1 = (c + 1) * (PS_CHUNK / 4) + lane;
#pragma unroll
                        for (int q = 0; q < PS_CHUNK / 128; ++q) {
                            nx[q] = make_uint4(~0u, ~0u, ~0u, ~0u);
                            if (q1 + q * 32 < n4) nx[q] = __ldcs(v + q1 - lane + q * 32);
                        }
                        ps_chunk(key, s, stop0, stop1, a.one);
                    }
                }
                const int n0 = (int)((s.p0 - b0) / ROW), n1 = (int)((s.p1 - b1) / ROW);
                const uint32_t T[2] = {__reduce_add_sync(ASR_FULL_MASK, s.c0), __reduce_add_sync(ASR_FULL_MASK, s.c1)};
                const uint32_t in[2] = {__reduce_add_sync(ASR_FULL_MASK, (uint32_t)n0),
                                        __reduce_add_sync(ASR_FULL_MASK, (uint32_t)n1)};
                const uint32_t ov = __reduce_or_sync(ASR_FULL_MASK, s.over);
                __syncwarp();
#ifdef PCT_STATS
                if (lane == 0) atomicAdd(&g_pct_stats[2], 1ull);
#endif
                bool ok = true;
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    const uint32_t hi = ps_end(wlo[t], wsh[t]);
                    if (k[t] > T[t]) {   // above the window (exact even when a lane ran out of slots)
                        ok = false;
#ifdef PCT_STATS
                        if (lane == 0) atomicAdd(&g_pct_stats[3], 1ull);
#endif
                        if (hi == 0xFFFFFFFFu) attempt = PS_TRIES;   // nothing above: keys of 2^32-1, radix path
                        const uint32_t e = k[t] - T[t];   // keys between the window's end and the rank
                        if (in[t] >= 16u && e <= 2u * in[t]) {
                            // near: a window of the same width centred where the window's density puts the rank
                            const uint32_t W = (uint32_t)PS_WIN << wsh[t];
                            const uint32_t c = hi + (uint32_t)(((uint64_t)e * W) / in[t]);
                            wlo[t] = c < hi ? 0xFFFFFFFFu - W : c - (W >> 1);
                        } else {
                            wlo[t] = hi;
                            wsh[t] += wsh[t] < PS_MAX_SHIFT ? 1 : 0;
                        }
                    } else if ((ov >> t) & 1u) {   // too dense for the slots: the upper half, then look again
                        ok = false;
#ifdef PCT_STATS
                        if (lane == 0) atomicAdd(&g_pct_stats[4], 1ull);
#endif
                        if (wsh[t] == 0) attempt = PS_TRIES;
                        else {
                            --wsh[t];
                            wlo[t] = hi - ((uint32_t)PS_WIN << wsh[t]);
                        }
                    } else if (k[t] <= T[t] - in[t]) {   // below the window
                        ok = false;
#ifdef PCT_STATS
                        if (lane == 0) atomicAdd(&g_pct_stats[6], 1ull);
#endif
                        const uint32_t e = T[t] - in[t] - k[t] + 1u;   // keys between the rank and the window's start
                        if (in[t] >= 16u && e <= 2u * in[t]) {
                            const uint32_t W = (uint32_t)PS_WIN << wsh[t];
                            const uint32_t back = (uint32_t)(((uint64_t)e * W) / in[t]) + (W >> 1);
                            wlo[t] = wlo[t] > back ? wlo[t] - back : 0u;
                        } else {
                            wsh[t] += wsh[t] < PS_MAX_SHIFT ? 1 : 0;
                            const uint32_t W = (uint32_t)PS_WIN << wsh[t];
                            wlo[t] = wlo[t] > W ? wlo[t] - W : 0u;
                        }
                    }
                }
                if (ok) {
#ifdef PCT_STATS
                    if (lane == 0) {
                        atomicAdd(&g_pct_stats[1], 1ull);
                        atomicAdd(&g_pct_stats[5], (unsigned long long)(in[0] + in[1]));
                    }
#endif
                    res[0] = ps_resolve(sm, 0, n0, wlo[0], wsh[0], k[0] - (T[0] - in[0]));
                    res[1] = ps_resolve(sm, 1, n1, wlo[1], wsh[1], k[1] - (T[1] - in[1]));
                    // the next segment's windows: centred on these answers, as wide as keeps the slots comfortably filled
#pragma unroll
                    for (int t = 0; t < 2; ++t) {
                        if (in[t] > PS_IN_MANY) wsh[t] -= wsh[t] > 0 ? 1 : 0;
                        else if (in[t] < PS_IN_FEW) wsh[t] += wsh[t] < PS_MAX_SHIFT ? 1 : 0;
                        const uint32_t half = (uint32_t)PS_WIN << wsh[t] >> 1;
                        wlo[t] = res[t] > half ? res[t] - half : 0u;
                    }
                    break;
                }
                if (attempt >= PS_TRIES - 1) {
                    settled = false;
                    break;
                }
            }
        }
        if (lane == 0) {
            asr_summary_t *s = a.out_summary + d.r;
            if (settled) {
                if (d.y == 0) {
                    s->p50_e2e_us = (int64_t)res[0];
                    s->p90_e2e_us = (int64_t)res[1];
                } else {
                    s->p50_ttft_us = (int64_t)res[0];
                    s->p90_ttft_us = (int64_t)res[1];
                }
            } else {
                a.miss_list[(size_t)d.y * a.n_replicas + atomicAdd(a.miss_count + d.y, 1)] = d.r;
            }
        }
    }
    __syncwarp();
  }
}

__global__ void __launch_bounds__(PCT_THREADS, PCT_MIN_CTAS) percentiles_kernel(const int64_t *values, const int64_t *seg_off,
                                                                  int32_t n_seg, PctList pl, int64_t *out) {
    extern __shared__ __align__(16) unsigned char dyn_smem[];
    PctRegSmem &sm = *reinterpret_cast<PctRegSmem *>(dyn_smem);
    for (int s = blockIdx.x; s < n_seg; s += gridDim.x) {
        const int64_t b = seg_off[s], e = seg_off[s + 1];
        int64_t res[PCT_MAX];
        if (!segment_percentiles_reg<PCT_MAX, false>(values + b, e - b, pl, res, sm))
            segment_percentiles(values + b, e - b, pl, res, nullptr);
        if (threadIdx.x == 0)
            for (int j = 0; j < pl.n_pct; ++j) out[(int64_t)s * pl.n_pct + j] = res[j];
    }
}

// p50/p90 of E2E latency (blockIdx.y = 0) and TTFT (blockIdx.y = 1) of every replica, or -- with a work list --
// of the replicas the carried-window kernel left: list[y*n_replicas + 0 .. count[y]).
__global__ void __launch_bounds__(PCT_THREADS, PCT_MIN_CTAS) summary_percentiles_kernel(const asr_replica_t *replicas,
                                                                          int32_t n_replicas, const int64_t *lat,
                                                                          const int64_t *ttft,
                                                                          asr_summary_t *out_summary, bool fmt_flags,
                                                                          const int32_t *list, const int32_t *count) {
    extern __shared__ __align__(16) unsigned char dyn_smem[];
    PctRegSmem &sm = *reinterpret_cast<PctRegSmem *>(dyn_smem);
    PctList pl;
    pl.n_pct = 2;
    pl.pct[0] = 50;
    pl.pct[1] = 90;
    const int64_t *vals = blockIdx.y == 0 ? lat : ttft;
    const int total = list ? count[blockIdx.y] : n_replicas;
    const int32_t *my_list = list ? list + (size_t)blockIdx.y * n_replicas : nullptr;
    for (int w = blockIdx.x; w < total; w += gridDim.x) {
        const int r = my_list ? my_list[w] : w;
        if (threadIdx.x == 0 && w + (int)gridDim.x < total) {
            // pull the CTA's next segment into L2 while this one is being processed
            const int rn = my_list ? my_list[w + gridDim.x] : w + gridDim.x;
            const asr_replica_t nx = replicas[rn];
            const int64_t flag = blockIdx.y == 0 ? out_summary[rn].p50_e2e_us : out_summary[rn].p50_ttft_us;
            const int64_t bytes = (int64_t)nx.n * ((fmt_flags && flag == ASR_FMT32) ? 4 : 8);
            // only a descriptor the simulator accepted (n_done >= 0) is dereferenced
            if (out_summary[rn].n_done >= 0 && nx.n > 0 && bytes <= (int64_t)PCT_REG_MAX * 8) {
                const char *src = reinterpret_cast<const char *>(vals + nx.out_off);
                const uint32_t sz = (uint32_t)(bytes & ~15ll);
                if (sz > 0 && (reinterpret_cast<uintptr_t>(src) & 15u) == 0)
                    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(sz) : "memory");
            }
        }
        if (out_summary[r].n_done < 0) continue;   // invalid descriptor, flagged by the simulator
        // order-free runs of the lane kernel leave the element format in the field this CTA fills in
        const int64_t flag = blockIdx.y == 0 ? out_summary[r].p50_e2e_us : out_summary[r].p50_ttft_us;
        const bool is32 = fmt_flags && flag == ASR_FMT32;
        const asr_replica_t rep = replicas[r];
        int64_t res[PCT_MAX];
        bool ok;
        if (is32) ok = segment_percentiles_reg<2, true>(vals + rep.out_off, rep.n, pl, res, sm);
        else ok = segment_percentiles_reg<2, false>(vals + rep.out_off, rep.n, pl, res, sm);
        if (!ok) segment_percentiles(vals + rep.out_off, rep.n, pl, res, nullptr, is32);
        if (threadIdx.x == 0) {
            if (blockIdx.y == 0) {
                out_summary[r].p50_e2e_us = res[0];
                out_summary[r].p90_e2e_us = res[1];
            } else {
                out_summary[r].p50_ttft_us = res[0];
                out_summary[r].p90_ttft_us = res[1];
            }
        }
    }
}

static constexpr size_t PCT_DYN_SMEM = sizeof(PctRegSmem);

static int pct_grid(int n_units, const void *fn, size_t smem = PCT_DYN_SMEM) {
    const int n_sm = sm_count();
    int per_sm = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, PCT_THREADS, smem);
    if (per_sm < 1) per_sm = 1;
    int cap = n_sm * per_sm;
    return n_units < cap ? n_units : cap;
}

int launch_percentiles(const int64_t *values, const int64_t *seg_off, int32_t n_seg, const int32_t *pcts,
                       int32_t n_pct, int64_t *out, cudaStream_t st) {
    if (n_seg <= 0 || n_pct <= 0) return ASR_OK;
    PctList pl;
    pl.n_pct = n_pct;
    for (int j = 0; j < PCT_MAX; ++j) pl.pct[j] = j < n_pct ? pcts[j] : 0;
    // per-device opt-in, set on every launch
    cudaFuncSetAttribute(percentiles_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PCT_DYN_SMEM);
    const int grid = pct_grid(n_seg, (const void *)percentiles_kernel);
    {
        KernelTimer kt(KID_PERCENTILES, st);
        percentiles_kernel<<<grid, PCT_THREADS, PCT_DYN_SMEM, st>>>(values, seg_off, n_seg, pl, out);
    }
    return check_launch("percentiles_kernel");
}

// fmt_flags with a miss list (2*n_replicas entries + 2 zeroed counters): the carried-window kernel first, the
// radix kernel on what it left.  Otherwise the radix kernel on every replica.
int launch_summary_percentiles(const asr_replica_t *replicas, int32_t n_replicas, const int64_t *lat,
                               const int64_t *ttft, asr_summary_t *out_summary, bool fmt_flags, const int32_t *order,
                               int32_t *miss_list, int32_t *miss_count, int32_t *scratch, cudaStream_t st) {
    if (n_replicas <= 0) return ASR_OK;
    cudaFuncSetAttribute(summary_percentiles_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PCT_DYN_SMEM);
    int gx = pct_grid(n_replicas, (const void *)summary_percentiles_kernel);
    gx = gx > 1 ? (gx + 1) / 2 : 1;
    const bool stream = fmt_flags && miss_list && miss_count && scratch;
    if (stream) {
        // seeds (radix kernel on the seed list), then one warp per segment; what is left goes to the miss list
        const int grid = sm_count();
        const int64_t total = 2 * (int64_t)n_replicas, run = PS_RUN;
        const int n_runs = (int)((total + run - 1) / run);
        PsArgs pa{replicas, lat, ttft, out_summary, order, miss_list, miss_count,
                  scratch + 64, scratch, scratch + 64 + 2 * (size_t)n_replicas, scratch + 2, n_replicas, (int32_t)run, n_runs, 1u};
        {
            KernelTimer kt(KID_SUMMARY_PCT, st);
            summary_seed_kernel<<<1, 1024, 0, st>>>(pa);
            summary_percentiles_kernel<<<dim3(gx, 2), PCT_THREADS, PCT_DYN_SMEM, st>>>(replicas, n_replicas, lat, ttft, out_summary,
                                                                                       true, pa.seed_list, pa.seed_count);
        }
        int rc = check_launch("summary_percentiles_kernel (seeds)");
        if (rc) return rc;
        cudaFuncSetAttribute(summary_stream_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PS_SMEM_BYTES);
        {
            KernelTimer kt(KID_SUMMARY_FAST, st);
            const int want = (n_runs + PS_WARPS - 1) / PS_WARPS;
            summary_stream_kernel<<<want < grid ? want : grid, PS_WARPS * 32, PS_SMEM_BYTES, st>>>(pa);
        }
        rc = check_launch("summary_stream_kernel");
        if (rc) return rc;
#ifdef PCT_STATS
        {
            int32_t h[4];
            cudaStreamSynchronize(st);
            cudaMemcpy(h, pa.seed_count, 8, cudaMemcpyDeviceToHost);
            cudaMemcpy(h + 2, miss_count, 8, cudaMemcpyDeviceToHost);
            unsigned long long g[8], z[8] = {0, 0, 0, 0, 0, 0, 0, 0};
            cudaMemcpyFromSymbol(g, g_pct_stats, sizeof(g));
            cudaMemcpyToSymbol(g_pct_stats, z, sizeof(z));
            fprintf(stderr, "stream stats: runs %d x %d items, seeds %d + %d, misses %d + %d, passes %llu settled %llu in-window/settled %.0f above %llu dense %llu below %llu\n",
                    n_runs, (int)run, h[0], h[1], h[2], h[3], g[2], g[1], g[1] ? (double)g[5] / (double)g[1] : 0.0, g[3], g[4], g[6]);
        }
#endif
    }
    {
        KernelTimer kt(KID_SUMMARY_PCT, st);
        summary_percentiles_kernel<<<dim3(gx, 2), PCT_THREADS, PCT_DYN_SMEM, st>>>(
            replicas, n_replicas, lat, ttft, out_summary, fmt_flags, stream ? miss_list : nullptr, stream ? miss_count : nullptr);
    }
    return check_launch("summary_percentiles_kernel");
}

}  // namespace asr

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


// ---------------------------------------------------------------------------
// carried-window kernel (order-free uint32 segments of a sweep: p50/p90)
//
// A CTA walks a run of consecutive segments.  Consecutive segments of a sweep
// are alike (the same trace under another policy, the neighbouring seed or
// rate), so the two ranks of segment i are looked for in windows of values
// around the answers of segment i-1: ONE pass over the register-resident keys
// counts, per rank, the keys below the window's end and appends the keys
// inside the window to per-thread private slots (no atomics, no tables to
// clear); the window is then resolved exactly by a two-level 10-bit histogram
// over the few hundred collected keys.  Every count is exact and the window is
// only a guess: a rank that falls outside moves the window that way and
// doubles it, a thread that runs out of slots halves it, and the pass is
// repeated on the keys still in registers.  A CTA's first segment finds its
// windows by bisection on the key bits (count-only passes).  A segment in
// another format, or one that is not settled after PF_TRIES passes, goes to
// the miss list, which summary_percentiles_kernel (radix path) works off.
// No result depends on a guess.
// ---------------------------------------------------------------------------
#ifndef PF_SLOTS_N
#define PF_SLOTS_N 16
#endif
#ifndef PF_MIN_CTAS
#define PF_MIN_CTAS 4
#endif
#ifdef PCT_STATS
__device__ unsigned long long g_pct_stats[8];   // segments, settled, passes, bootstraps, misses, in-window keys, -, -
#endif
constexpr int PF_SLOTS = PF_SLOTS_N;   // private slots per thread and rank
constexpr int PF_GROUP = 8;            // slots are checked once per group of keys
constexpr int PF_BINS = 1024;          // bins per histogram level
constexpr int PF_MAX_SHIFT = 10;       // window = PF_BINS << shift values; the second level resolves 2^shift
constexpr int PF_HALF = PCT_THREADS / 2;
constexpr int PF_TRIES = 6;
#ifndef PF_IN_MANY_N
#define PF_IN_MANY_N 256   // one key per thread: a thread with more than PF_SLOTS - PF_GROUP closes its window
#endif
constexpr uint32_t PF_IN_MANY = PF_IN_MANY_N, PF_IN_FEW = PF_IN_MANY / 4;   // keys wanted inside a window
static_assert(PCT_VPT % PF_GROUP == 0 && PF_SLOTS >= 2 * PF_GROUP, "slot check granularity");

struct PctFastSmem {
    uint32_t slot[2][PF_SLOTS][PCT_THREADS];
    uint32_t hist[2][2][PF_BINS];            // [level][rank][bin]
    uint32_t wtot[2][2][PCT_THREADS / 32];   // [parity][rank][warp]: keys below the window's end | keys inside << 16
    uint32_t wovf[2][PCT_THREADS / 32];      // [parity][warp]: bit t = a thread closed its window of rank t
    uint32_t wsum[2][PCT_THREADS / 64];
    uint32_t sel_bin[2][2], sel_rem[2][2];   // [level][rank]
    uint32_t sel_cnt[2];                     // [rank]: keys in the selected level-1 bin
    uint32_t lcnt[2], list[2][32];           // [rank]: those keys (their offsets inside the bin) when there are at most 32
};

__device__ __forceinline__ uint32_t pf_end(uint32_t lo, int sh) {   // saturated: a key 2^32-1 is never inside
    const uint32_t hi = lo + ((uint32_t)PF_BINS << sh);
    return hi < lo ? 0xFFFFFFFFu : hi;
}

// inclusive scan of the PF_BINS bins of histogram h by the PF_HALF threads of one rank: thread j owns
// bins 8j .. 8j+7.  Part A leaves the per-warp totals in wsum; after a barrier part B locates rank k.
__device__ __forceinline__ void pf_scan_a(const uint32_t *h, int j, uint32_t (&c)[8], uint32_t &tot, uint32_t &incl,
                                          uint32_t *wsum) {
    static_assert(PF_BINS == PF_HALF * 8, "eight bins per thread");
    const uint4 a = *reinterpret_cast<const uint4 *>(h + 8 * j), b = *reinterpret_cast<const uint4 *>(h + 8 * j + 4);
    c[0] = a.x, c[1] = a.y, c[2] = a.z, c[3] = a.w, c[4] = b.x, c[5] = b.y, c[6] = b.z, c[7] = b.w;
    tot = ((c[0] + c[1]) + (c[2] + c[3])) + ((c[4] + c[5]) + (c[6] + c[7]));
    incl = tot;
    const int lane = lane_id();
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t y = __shfl_up_sync(ASR_FULL_MASK, incl, d);
        if (lane >= d) incl += y;
    }
    if (lane == 31) wsum[j >> 5] = incl;
}

__device__ __forceinline__ void pf_scan_b(const uint32_t (&c)[8], uint32_t tot, uint32_t incl, const uint32_t *wsum, int j,
                                          uint32_t k, uint32_t *sel_bin, uint32_t *sel_rem, uint32_t *sel_cnt = nullptr) {
    uint32_t excl = incl - tot;
#pragma unroll
    for (int w = 0; w < PF_HALF / 32; ++w)
        if (w < (j >> 5)) excl += wsum[w];
    if (excl < k && k <= excl + tot) {
        uint32_t run = excl;
#pragma unroll
        for (int b = 0; b < 8; ++b) {
            if (run < k && k <= run + c[b]) {
                *sel_bin = (uint32_t)(8 * j + b);
                *sel_rem = k - run;
                if (sel_cnt) *sel_cnt = c[b];
            }
            run += c[b];
        }
    }
}

// hist[bin] += 1 if p (a predicated shared-memory reduction: no branch, nothing touched when !p)
__device__ __forceinline__ void pf_inc_if(uint32_t *hist, uint32_t bin, bool p) {
    asm volatile(
        "{\n\t"
        ".reg .pred q;\n\t"
        "setp.ne.u32 q, %1, 0;\n\t"
        "@q red.shared.add.u32 [%0], 1;\n\t"
        "}" ::"r"((uint32_t)__cvta_generic_to_shared(hist) + 4u * bin),
        "r"((uint32_t)p)
        : "memory");
}
#ifndef PF_STRAIGHT_N
#define PF_STRAIGHT_N 3
#endif
constexpr int PF_STRAIGHT = PF_STRAIGHT_N;   // entries per thread and rank handled without a loop (most threads hold 0-2)

// One pass over the keys.  Per key and rank: one compare-and-count below the window's end, one compare for
// "inside", a predicated store and a predicated pointer bump (written out in PTX: the compiler's version of the
// same loop took nine instructions per key and rank).  Returns, for rank t, T[t] = keys below the end | keys
// inside << 16 over the whole CTA, and ov = bit t set if some thread closed its window t for lack of slots
// (then "inside" of rank t is short; "below the end" is always exact).  n[t] = this thread's keys inside.
__device__ __forceinline__ void pf_pass(const uint32_t (&key)[PCT_VPT], uint32_t lo0, uint32_t hi0, uint32_t lo1,
                                        uint32_t hi1, PctFastSmem &fs, int par, uint32_t (&T)[2], uint32_t &ov,
                                        int (&n)[2]) {
    const int tid = threadIdx.x, lane = lane_id(), warp = tid >> 5;
    uint32_t c0 = 0, c1 = 0;
    const uint32_t b0 = (uint32_t)__cvta_generic_to_shared(&fs.slot[0][0][tid]);
    const uint32_t b1 = (uint32_t)__cvta_generic_to_shared(&fs.slot[1][0][tid]);
    uint32_t p0 = b0, p1 = b1;
    constexpr uint32_t ROW = PCT_THREADS * 4;   // bytes between two slots of a thread
    const uint32_t stop0 = b0 + (PF_SLOTS - PF_GROUP) * ROW, stop1 = b1 + (PF_SLOTS - PF_GROUP) * ROW;
    uint32_t over = 0;
#pragma unroll
    for (int g = 0; g < PCT_VPT / PF_GROUP; ++g) {
#pragma unroll
        for (int j = 0; j < PF_GROUP; ++j) {
            asm volatile(
                "{\n\t"
                ".reg .pred a, b;\n\t"
                "setp.lt.u32 a, %4, %5;\n\t"
                "@a add.u32 %0, %0, 1;\n\t"
                "setp.ge.and.u32 b, %4, %6, a;\n\t"
                "@b st.shared.u32 [%1], %4;\n\t"
                "@b add.u32 %1, %1, %9;\n\t"
                "setp.lt.u32 a, %4, %7;\n\t"
                "@a add.u32 %2, %2, 1;\n\t"
                "setp.ge.and.u32 b, %4, %8, a;\n\t"
                "@b st.shared.u32 [%3], %4;\n\t"
                "@b add.u32 %3, %3, %9;\n\t"
                "}"
                : "+r"(c0), "+r"(p0), "+r"(c1), "+r"(p1)
                : "r"(key[g * PF_GROUP + j]), "r"(hi0), "r"(lo0), "r"(hi1), "r"(lo1), "n"(ROW)
                : "memory");
        }
        // a thread that could run out of slots in the next group closes its window (after the first group it holds
        // at most PF_GROUP keys, after the last one nothing follows)
        if (g > 0 && g < PCT_VPT / PF_GROUP - 1) {
            if (p0 > stop0) {
                lo0 = hi0;
                over |= 1u;
            }
            if (p1 > stop1) {
                lo1 = hi1;
                over |= 2u;
            }
        }
    }
    n[0] = (int)((p0 - b0) / ROW);
    n[1] = (int)((p1 - b1) / ROW);
    const uint32_t t0 = __reduce_add_sync(ASR_FULL_MASK, c0 | ((uint32_t)n[0] << 16));
    const uint32_t t1 = __reduce_add_sync(ASR_FULL_MASK, c1 | ((uint32_t)n[1] << 16));
    const uint32_t wo = __reduce_or_sync(ASR_FULL_MASK, over);
    if (lane == 0) {
        fs.wtot[par][0][warp] = t0;
        fs.wtot[par][1][warp] = t1;
        fs.wovf[par][warp] = wo;
    }
    __syncthreads();
    T[0] = T[1] = ov = 0;
#pragma unroll
    for (int w = 0; w < PCT_THREADS / 32; ++w) {
        T[0] += fs.wtot[par][0][w];
        T[1] += fs.wtot[par][1][w];
        ov |= fs.wovf[par][w];
    }
}

// count-only pass: keys below t0 / below t1 over the whole CTA
__device__ __forceinline__ void pf_count(const uint32_t (&key)[PCT_VPT], uint32_t t0, uint32_t t1, PctFastSmem &fs, int par,
                                         uint32_t (&C)[2]) {
    const int lane = lane_id(), warp = threadIdx.x >> 5;
    uint32_t c0 = 0, c1 = 0;
#pragma unroll
    for (int j = 0; j < PCT_VPT; ++j) {
        c0 += key[j] < t0 ? 1u : 0u;
        c1 += key[j] < t1 ? 1u : 0u;
    }
    c0 = __reduce_add_sync(ASR_FULL_MASK, c0);
    c1 = __reduce_add_sync(ASR_FULL_MASK, c1);
    if (lane == 0) {
        fs.wtot[par][0][warp] = c0;
        fs.wtot[par][1][warp] = c1;
    }
    __syncthreads();
    C[0] = C[1] = 0;
#pragma unroll
    for (int w = 0; w < PCT_THREADS / 32; ++w) {
        C[0] += fs.wtot[par][0][w];
        C[1] += fs.wtot[par][1][w];
    }
}

__global__ void __launch_bounds__(PCT_THREADS, PF_MIN_CTAS) summary_fast_kernel(const asr_replica_t *replicas, int32_t n_replicas,
                                                                                const int64_t *lat, const int64_t *ttft,
                                                                                asr_summary_t *out_summary,
                                                                                const int32_t *order, int32_t chunk,
                                                                                int32_t *miss_list, int32_t *miss_count) {
    extern __shared__ __align__(16) unsigned char dyn_smem[];
    PctFastSmem &fs = *reinterpret_cast<PctFastSmem *>(dyn_smem);
    const int tid = threadIdx.x;
    const int64_t *vals = blockIdx.y == 0 ? lat : ttft;
    int32_t *my_miss = miss_list + (size_t)blockIdx.y * n_replicas;
    bool have = false;
    uint32_t wlo[2] = {0, 0};
    int wsh[2] = {0, 0};
    int par = 0;
    const int i0 = blockIdx.x * chunk, i1 = min(n_replicas, i0 + chunk);
    for (int i = i0; i < i1; ++i) {
        const int r = order ? order[i] : i;
        if (tid == 0 && i + 1 < i1) {
            // pull the CTA's next segment into L2 while this one is being processed
            const int rn = order ? order[i + 1] : i + 1;
            const asr_replica_t nx = replicas[rn];
            const int64_t flag = blockIdx.y == 0 ? out_summary[rn].p50_e2e_us : out_summary[rn].p50_ttft_us;
            // only a descriptor the simulator accepted (n_done >= 0) is dereferenced
            if (out_summary[rn].n_done >= 0 && flag == ASR_FMT32 && nx.n > 0 && nx.n <= PCT_REG_MAX) {
                const char *src = reinterpret_cast<const char *>(vals + nx.out_off);
                const uint32_t sz = (uint32_t)(((int64_t)nx.n * 4) & ~15ll);
                if (sz > 0 && (reinterpret_cast<uintptr_t>(src) & 15u) == 0)
                    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(sz) : "memory");
            }
        }
        if (out_summary[r].n_done < 0) continue;   // invalid descriptor, flagged by the simulator
        const int64_t flag = blockIdx.y == 0 ? out_summary[r].p50_e2e_us : out_summary[r].p50_ttft_us;
        const asr_replica_t rep = replicas[r];
        const int64_t *seg = vals + rep.out_off;
        const int N = rep.n;
        bool settled = flag == ASR_FMT32 && N > 0 && N <= PCT_REG_MAX && (N & 3) == 0 &&
                       (reinterpret_cast<uintptr_t>(seg) & 15u) == 0;
        uint32_t res[2] = {0, 0};
        if (settled) {
            const uint32_t k[2] = {(50u * (uint32_t)N + 99u) / 100u, (90u * (uint32_t)N + 99u) / 100u};
            // keys: four consecutive values per 128-bit load; slots past the end read as 2^32-1 (below no window end)
            uint32_t key[PCT_VPT];
            {
                const uint4 *v128 = reinterpret_cast<const uint4 *>(seg) + tid;
                const int n4 = N >> 2;
                const int full_rows = n4 / PCT_THREADS;   // rows of PCT_THREADS quads that every thread loads
#pragma unroll
                for (int q = 0; q < PCT_VPT / 4; ++q) {
                    uint4 x;
                    if (q < full_rows) {
                        x = __ldcs(v128 + q * PCT_THREADS);
                    } else {
                        x = make_uint4(~0u, ~0u, ~0u, ~0u);
                        if (q * PCT_THREADS + tid < n4) x = __ldcs(v128 + q * PCT_THREADS);
                    }
                    key[4 * q] = x.x, key[4 * q + 1] = x.y, key[4 * q + 2] = x.z, key[4 * q + 3] = x.w;
                }
            }
            // clear the first histogram level and the lists (their last readers passed the final barrier of the
            // previous segment)
            {
                uint4 *z = reinterpret_cast<uint4 *>(&fs.hist[0][0][0]);
                constexpr int n16 = 2 * PF_BINS / 4;
                static_assert(n16 % PCT_THREADS == 0, "whole passes");
#pragma unroll
                for (int q = 0; q < n16 / PCT_THREADS; ++q) z[q * PCT_THREADS + tid] = make_uint4(0u, 0u, 0u, 0u);
                if (tid < 2) fs.lcnt[tid] = 0;
            }
            if (!have) {
                // bisection on the key bits, both ranks at once: bracket [a, a + 2^rem) holds `in` keys, `below` lie under it
                uint32_t a[2] = {0, 0}, below[2] = {0, 0}, in[2] = {(uint32_t)N, (uint32_t)N};
                int rem[2] = {32, 32};
                while (true) {
                    const bool go0 = rem[0] > PF_MAX_SHIFT + 10 || (in[0] > PF_IN_MANY && rem[0] > 0);
                    const bool go1 = rem[1] > PF_MAX_SHIFT + 10 || (in[1] > PF_IN_MANY && rem[1] > 0);
                    if (!go0 && !go1) break;
                    const uint32_t m0 = go0 ? a[0] + (1u << (rem[0] - 1)) : a[0], m1 = go1 ? a[1] + (1u << (rem[1] - 1)) : a[1];
                    uint32_t C[2];
                    pf_count(key, m0, m1, fs, par, C);
                    par ^= 1;
                    if (go0) {
                        --rem[0];
                        if (k[0] <= C[0]) in[0] = C[0] - below[0];
                        else in[0] -= C[0] - below[0], below[0] = C[0], a[0] = m0;
                    }
                    if (go1) {
                        --rem[1];
                        if (k[1] <= C[1]) in[1] = C[1] - below[1];
                        else in[1] -= C[1] - below[1], below[1] = C[1], a[1] = m1;
                    }
                }
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    wlo[t] = a[t];
                    wsh[t] = rem[t] > 10 ? rem[t] - 10 : 0;
                }
                have = true;
#ifdef PCT_STATS
                if (tid == 0) atomicAdd(&g_pct_stats[3], 1ull);
#endif
            }
            uint32_t T[2], ov;
            int n[2];
            for (int attempt = 0;; ++attempt) {
                pf_pass(key, wlo[0], pf_end(wlo[0], wsh[0]), wlo[1], pf_end(wlo[1], wsh[1]), fs, par, T, ov, n);
                par ^= 1;
#ifdef PCT_STATS
                if (tid == 0) atomicAdd(&g_pct_stats[2], 1ull);
#endif
                bool ok = true;
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    const uint32_t c = T[t] & 0xFFFFu, in = T[t] >> 16, hi = pf_end(wlo[t], wsh[t]);
                    if (k[t] > c) {   // above the window (exact even when a thread ran out of slots)
                        ok = false;
                        if (hi == 0xFFFFFFFFu) attempt = PF_TRIES;   // nothing above: keys of 2^32-1, radix path
                        wlo[t] = hi;
                        wsh[t] += wsh[t] < PF_MAX_SHIFT ? 1 : 0;
                    } else if ((ov >> t) & 1u) {   // too dense for the slots: the upper half, then look again
                        ok = false;
                        if (wsh[t] == 0) attempt = PF_TRIES;
                        else {
                            --wsh[t];
                            wlo[t] = hi - ((uint32_t)PF_BINS << wsh[t]);
                        }
                    } else if (k[t] <= c - in) {   // below the window
                        ok = false;
                        wsh[t] += wsh[t] < PF_MAX_SHIFT ? 1 : 0;
                        const uint32_t W = (uint32_t)PF_BINS << wsh[t];
                        wlo[t] = wlo[t] > W ? wlo[t] - W : 0u;
                    }
                }
                if (ok) break;
                if (attempt >= PF_TRIES - 1) {
                    settled = false;
                    break;
                }
            }
            if (settled) {
                const int sh0 = wsh[0], sh1 = wsh[1];
                const uint32_t lo0 = wlo[0], lo1 = wlo[1];
                const uint32_t in0 = T[0] >> 16, in1 = T[1] >> 16;
                const uint32_t below0 = (T[0] & 0xFFFFu) - in0, below1 = (T[1] & 0xFFFFu) - in1;
                // level 1: bins of 2^sh values over the window
                const int nm = n[0] > n[1] ? n[0] : n[1];
#pragma unroll
                for (int e = 0; e < PF_STRAIGHT; ++e) {   // (a slot past the thread's count holds a stale key: never counted)
                    pf_inc_if(fs.hist[0][0], (fs.slot[0][e][tid] - lo0) >> sh0, e < n[0]);
                    pf_inc_if(fs.hist[0][1], (fs.slot[1][e][tid] - lo1) >> sh1, e < n[1]);
                }
                for (int e = PF_STRAIGHT; e < nm; ++e) {
                    if (e < n[0]) atomicAdd(&fs.hist[0][0][(fs.slot[0][e][tid] - lo0) >> sh0], 1u);
                    if (e < n[1]) atomicAdd(&fs.hist[0][1][(fs.slot[1][e][tid] - lo1) >> sh1], 1u);
                }
                __syncthreads();
                const int tg = tid / PF_HALF, j = tid % PF_HALF;
                const uint32_t kw = tg == 0 ? k[0] - below0 : k[1] - below1;   // rank inside the window
                uint32_t c[8], tot, incl;
                pf_scan_a(fs.hist[0][tg], j, c, tot, incl, fs.wsum[tg]);
                __syncthreads();
                pf_scan_b(c, tot, incl, fs.wsum[tg], j, kw, &fs.sel_bin[0][tg], &fs.sel_rem[0][tg], &fs.sel_cnt[tg]);
                __syncthreads();
                const uint32_t bin0 = fs.sel_bin[0][0], bin1 = fs.sel_bin[0][1];
                uint32_t r0 = lo0 + (bin0 << sh0), r1 = lo1 + (bin1 << sh1);
                if (sh0 > 0 || sh1 > 0) {
                    // level 2: the keys of the selected bin
                    const int m0 = sh0 > 0 ? n[0] : 0, m1 = sh1 > 0 ? n[1] : 0, mm = m0 > m1 ? m0 : m1;
                    const uint32_t cnt0 = sh0 > 0 ? fs.sel_cnt[0] : 0u, cnt1 = sh1 > 0 ? fs.sel_cnt[1] : 0u;
                    if (cnt0 <= 32u && cnt1 <= 32u) {
                        // a handful: listed, and ranked by one warp per rank (any order of equal keys gives the same
                        // value at every rank)
                        for (int e = 0; e < mm; ++e) {
                            if (e < m0) {
                                const uint32_t dd = fs.slot[0][e][tid] - lo0;
                                if ((dd >> sh0) == bin0) fs.list[0][atomicAdd(&fs.lcnt[0], 1u)] = dd & ((1u << sh0) - 1u);
                            }
                            if (e < m1) {
                                const uint32_t dd = fs.slot[1][e][tid] - lo1;
                                if ((dd >> sh1) == bin1) fs.list[1][atomicAdd(&fs.lcnt[1], 1u)] = dd & ((1u << sh1) - 1u);
                            }
                        }
                        __syncthreads();
                        if (tid < 64) {
                            const int t = tid >> 5, lane = tid & 31;
                            const uint32_t cn = t == 0 ? cnt0 : cnt1;
                            const uint32_t v = (uint32_t)lane < cn ? fs.list[t][lane] : 0xFFFFFFFFu;
                            uint32_t rank = 0;
                            for (uint32_t q = 0; q < cn; ++q) {
                                const uint32_t u = __shfl_sync(ASR_FULL_MASK, v, (int)q);
                                rank += (u < v || (u == v && q < (uint32_t)lane)) ? 1u : 0u;
                            }
                            if ((uint32_t)lane < cn && rank + 1u == fs.sel_rem[0][t]) fs.sel_bin[1][t] = v;
                        }
                        __syncthreads();
                    } else {
                        // many equal or near-equal keys: a second histogram, one value per bin
                        {
                            uint4 *z = reinterpret_cast<uint4 *>(&fs.hist[1][0][0]);
                            constexpr int n16 = 2 * PF_BINS / 4;
#pragma unroll
                            for (int q = 0; q < n16 / PCT_THREADS; ++q) z[q * PCT_THREADS + tid] = make_uint4(0u, 0u, 0u, 0u);
                        }
                        __syncthreads();
                        for (int e = 0; e < mm; ++e) {
                            if (e < m0) {
                                const uint32_t dd = fs.slot[0][e][tid] - lo0;
                                if ((dd >> sh0) == bin0) atomicAdd(&fs.hist[1][0][dd & ((1u << sh0) - 1u)], 1u);
                            }
                            if (e < m1) {
                                const uint32_t dd = fs.slot[1][e][tid] - lo1;
                                if ((dd >> sh1) == bin1) atomicAdd(&fs.hist[1][1][dd & ((1u << sh1) - 1u)], 1u);
                            }
                        }
                        __syncthreads();
                        const bool act = tg == 0 ? sh0 > 0 : sh1 > 0;
                        if (act) pf_scan_a(fs.hist[1][tg], j, c, tot, incl, fs.wsum[tg]);
                        __syncthreads();
                        if (act) pf_scan_b(c, tot, incl, fs.wsum[tg], j, fs.sel_rem[0][tg], &fs.sel_bin[1][tg], &fs.sel_rem[1][tg]);
                        __syncthreads();
                    }
                    if (sh0 > 0) r0 += fs.sel_bin[1][0];
                    if (sh1 > 0) r1 += fs.sel_bin[1][1];
                }
                res[0] = r0;
                res[1] = r1;
                // the next segment's windows: centred on these answers, as wide as keeps the slots comfortably filled
                const uint32_t inw[2] = {in0, in1};
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    if (inw[t] > PF_IN_MANY) wsh[t] -= wsh[t] > 0 ? 1 : 0;
                    else if (inw[t] < PF_IN_FEW) wsh[t] += wsh[t] < PF_MAX_SHIFT ? 1 : 0;
                    const uint32_t half = (uint32_t)PF_BINS << wsh[t] >> 1;
                    wlo[t] = res[t] > half ? res[t] - half : 0u;
                }
#ifdef PCT_STATS
                if (tid == 0) {
                    atomicAdd(&g_pct_stats[1], 1ull);
                    atomicAdd(&g_pct_stats[5], (unsigned long long)(in0 + in1));
                }
#endif
            }
            __syncthreads();   // the next segment rewrites slots, totals and histograms
        }
#ifdef PCT_STATS
        if (tid == 0) atomicAdd(&g_pct_stats[0], 1ull);
#endif
        if (tid == 0) {
            if (settled) {
                if (blockIdx.y == 0) {
                    out_summary[r].p50_e2e_us = (int64_t)res[0];
                    out_summary[r].p90_e2e_us = (int64_t)res[1];
                } else {
                    out_summary[r].p50_ttft_us = (int64_t)res[0];
                    out_summary[r].p90_ttft_us = (int64_t)res[1];
                }
            } else {
                my_miss[atomicAdd(miss_count + blockIdx.y, 1)] = r;
#ifdef PCT_STATS
                atomicAdd(&g_pct_stats[4], 1ull);
#endif
            }
        }
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
static constexpr size_t PF_DYN_SMEM = sizeof(PctFastSmem);

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
                               int32_t *miss_list, int32_t *miss_count, cudaStream_t st) {
    if (n_replicas <= 0) return ASR_OK;
    cudaFuncSetAttribute(summary_percentiles_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PCT_DYN_SMEM);
    int gx = pct_grid(n_replicas, (const void *)summary_percentiles_kernel);
    gx = gx > 1 ? (gx + 1) / 2 : 1;
    const bool fast = fmt_flags && miss_list && miss_count && PCT_THREADS == 256;
    if (fast) {
        cudaFuncSetAttribute(summary_fast_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PF_DYN_SMEM);
        int fx = pct_grid(n_replicas, (const void *)summary_fast_kernel, PF_DYN_SMEM);
        fx = fx > 1 ? (fx + 1) / 2 : 1;
        // every CTA walks one run of consecutive segments
        const int chunk = (n_replicas + fx - 1) / fx;
        fx = (n_replicas + chunk - 1) / chunk;
        {
            KernelTimer kt(KID_SUMMARY_FAST, st);
            summary_fast_kernel<<<dim3(fx, 2), PCT_THREADS, PF_DYN_SMEM, st>>>(replicas, n_replicas, lat, ttft, out_summary,
                                                                               order, chunk, miss_list, miss_count);
        }
        int rc = check_launch("summary_fast_kernel");
        if (rc) return rc;
#ifdef PCT_STATS
        {
            unsigned long long h[8], z[8] = {0, 0, 0, 0, 0, 0, 0, 0};
            cudaStreamSynchronize(st);
            cudaMemcpyFromSymbol(h, g_pct_stats, sizeof(h));
            cudaMemcpyToSymbol(g_pct_stats, z, sizeof(z));
            fprintf(stderr, "pct stats: segments %llu settled %llu passes %llu bootstraps %llu misses %llu in-window/settled %.0f\n",
                    h[0], h[1], h[2], h[3], h[4], h[1] ? (double)h[5] / (double)h[1] : 0.0);
        }
#endif
    }
    {
        KernelTimer kt(KID_SUMMARY_PCT, st);
        summary_percentiles_kernel<<<dim3(gx, 2), PCT_THREADS, PCT_DYN_SMEM, st>>>(
            replicas, n_replicas, lat, ttft, out_summary, fmt_flags, fast ? miss_list : nullptr, fast ? miss_count : nullptr);
    }
    return check_launch("summary_percentiles_kernel");
}

}  // namespace asr

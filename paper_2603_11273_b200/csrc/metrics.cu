// metrics.cu -- elementwise kernels of the SURVEY.md 8(f) extensions, sm_100a.
//   tpot_kernel      f2  time per output token: (E2E - TTFT) / (tokens - 1)
//   estimate_kernel  f3  duration-based estimator (Eq. 1, Listing 1)
// Both are HBM streams: 32 B read + 8 B written per request (tpot), 16 B read + 4 B
// written (estimate; + 1 B language id, + 4 B speech-active duration when given).
#include "sim_common.cuh"

namespace asr {

__global__ void __launch_bounds__(256) tpot_kernel(const asr_req_t *__restrict__ trace, int64_t n, asr_cost_model_t cm,
                                                   const int64_t *__restrict__ lat, const int64_t *__restrict__ ttft,
                                                   int64_t *__restrict__ out) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const int32_t dur = ld_stream(trace + i).dur_ms;
        const int64_t tok = tokens_of(cm, dur);
        const int64_t d = __ldcs(lat + i) - __ldcs(ttft + i);
        __stcs(out + i, tok > 1 ? d / (tok - 1) : (int64_t)-1);
    }
}

constexpr int64_t EST_MAX = (int64_t)1 << 24;

__global__ void __launch_bounds__(256) estimate_kernel(asr_req_t *recs, int64_t n, KappaTable kt,
                                                       const uint8_t *__restrict__ lang,
                                                       const int32_t *__restrict__ speech_ms) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        int l = lang ? (int)lang[i] : 0;
        if (l >= kt.n_lang) l = 0;
        int64_t d = speech_ms ? (int64_t)speech_ms[i] : (int64_t)recs[i].dur_ms;
        d = d < 0 ? 0 : d;
        int64_t e = (d * (int64_t)kt.kappa_milli[l]) / 1000000;
        e = e < 1 ? 1 : (e > EST_MAX ? EST_MAX : e);   // the comparator's documented bound (asr_sched.h: est <= 2^24)
        recs[i].est = (int32_t)e;
    }
}

// ---------------------------------------------------------------------------
// f2 inter-token latency: weighted nearest-rank percentiles of the gap
// multiset the extension kernel captured: ITL_BINS weights of the plain iterations (value
// iter_base + iter_per*|running|) plus (duration, weight) pairs.  One CTA per replica;
// MSB-first radix select over (value - min) with 8-bit digits and weighted counts.
// out[r] = n_pct percentiles, then the number of gaps, then their sum.
// ---------------------------------------------------------------------------
constexpr int ITL_THREADS = 256;

__device__ __forceinline__ void itl_item(const SimExArgs &a, const asr_replica_t &rep, const asr_cost_model_t &cm,
                                         int r, int n_pairs, int i, int64_t &v, unsigned long long &w) {
    if (i < ITL_BINS) {
        v = cm.iter_base_us + cm.iter_per_running_us * (int64_t)i;
        w = a.itl_hist[(int64_t)r * ITL_BINS + i];
    } else {
        const int64_t q = rep.out_off + (i - ITL_BINS);
        v = a.itl_pairs[2 * q];
        w = (unsigned long long)a.itl_pairs[2 * q + 1];
    }
    (void)n_pairs;
}

__global__ void __launch_bounds__(ITL_THREADS) itl_percentiles_kernel(SimExArgs a, ItlPcts pl, int64_t *out) {
    __shared__ unsigned long long hist[256];
    __shared__ unsigned long long red[ITL_THREADS / 32];
    __shared__ long long red_min[ITL_THREADS / 32], red_max[ITL_THREADS / 32];
    __shared__ unsigned long long sel_below;
    __shared__ uint32_t sel_digit;
    const int lane = lane_id(), warp = threadIdx.x >> 5;
    for (int r = blockIdx.x; r < a.n_replicas; r += gridDim.x) {
        int64_t *o = out + (int64_t)r * (pl.n_pct + 2);
        const int n_pairs = a.itl_npairs[r];
        if (n_pairs < 0) {   // invalid replica
            if (threadIdx.x == 0)
                for (int j = 0; j < pl.n_pct + 2; ++j) o[j] = -1;
            continue;
        }
        const asr_replica_t rep = a.replicas[r];
        const asr_cost_model_t cm = a.cms[rep.cm_id];
        const int n_items = ITL_BINS + n_pairs;
        // total weight, weighted sum, min and max of the values that occur
        unsigned long long tw = 0, ts = 0;
        long long mn = INT64_MAX, mx = INT64_MIN;
        for (int i = threadIdx.x; i < n_items; i += ITL_THREADS) {
            int64_t v;
            unsigned long long w;
            itl_item(a, rep, cm, r, n_pairs, i, v, w);
            if (w) {
                tw += w;
                ts += w * (unsigned long long)v;
                mn = v < mn ? v : mn;
                mx = v > mx ? v : mx;
            }
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            tw += shfl64_xor(tw, d);
            ts += shfl64_xor(ts, d);
            const long long omn = (long long)shfl64_xor((uint64_t)mn, d), omx = (long long)shfl64_xor((uint64_t)mx, d);
            mn = omn < mn ? omn : mn;
            mx = omx > mx ? omx : mx;
        }
        __syncthreads();
        if (lane == 0) {
            red[warp] = tw;
            red_min[warp] = mn;
            red_max[warp] = mx;
            hist[warp] = ts;
        }
        __syncthreads();
        tw = ts = 0;
        mn = INT64_MAX;
        mx = INT64_MIN;
#pragma unroll
        for (int w8 = 0; w8 < ITL_THREADS / 32; ++w8) {
            tw += red[w8];
            ts += hist[w8];
            mn = red_min[w8] < mn ? red_min[w8] : mn;
            mx = red_max[w8] > mx ? red_max[w8] : mx;
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            o[pl.n_pct] = (int64_t)tw;
            o[pl.n_pct + 1] = (int64_t)ts;
        }
        if (tw == 0) {
            if (threadIdx.x == 0)
                for (int j = 0; j < pl.n_pct; ++j) o[j] = -1;
            continue;
        }
        const uint64_t range = (uint64_t)mx - (uint64_t)mn;
        const int bits = range == 0 ? 0 : 64 - __clzll((long long)range);
        const int top_shift = bits <= 8 ? 0 : ((bits + 7) / 8 - 1) * 8;
        for (int j = 0; j < pl.n_pct; ++j) {
            // 1-based rank ceil(p*N/100); N < 2^57 keeps the product in 64 bits
            unsigned long long kk = (tw / 100ull) * (unsigned long long)pl.pct[j] +
                                    ((tw % 100ull) * (unsigned long long)pl.pct[j] + 99ull) / 100ull;
            uint64_t prefix = 0;
            if (bits > 0) {
                for (int shift = top_shift;; shift -= 8) {
                    __syncthreads();
                    hist[threadIdx.x] = 0;   // ITL_THREADS == 256
                    __syncthreads();
                    for (int i = threadIdx.x; i < n_items; i += ITL_THREADS) {
                        int64_t v;
                        unsigned long long w;
                        itl_item(a, rep, cm, r, n_pairs, i, v, w);
                        if (w) {
                            const uint64_t key = (uint64_t)v - (uint64_t)mn;
                            if (shift + 8 >= 64 || (key >> (shift + 8)) == prefix)
                                atomicAdd(&hist[(key >> shift) & 255u], w);
                        }
                    }
                    __syncthreads();
                    if (threadIdx.x == 0) {
                        unsigned long long run = 0;
                        for (int b = 0; b < 256; ++b) {
                            if (run < kk && kk <= run + hist[b]) {
                                sel_digit = (uint32_t)b;
                                sel_below = run;
                                break;
                            }
                            run += hist[b];
                        }
                    }
                    __syncthreads();
                    prefix = (prefix << 8) | sel_digit;
                    kk -= sel_below;
                    if (shift == 0) break;
                }
            }
            if (threadIdx.x == 0) o[j] = (int64_t)((uint64_t)mn + prefix);
        }
        __syncthreads();
    }
}

int launch_itl_percentiles(const SimExArgs &a, const ItlPcts &pl, int64_t *out, cudaStream_t st) {
    const int grid = a.n_replicas < sm_count() * 8 ? a.n_replicas : sm_count() * 8;
    {
        KernelTimer kt(KID_ITL_PCT, st);
        itl_percentiles_kernel<<<grid, ITL_THREADS, 0, st>>>(a, pl, out);
    }
    return check_launch("itl_percentiles_kernel");
}

static int stream_grid(int64_t n) {
    const int64_t want = (n + 255) / 256;
    return (int)(want < (int64_t)sm_count() * 16 ? want : (int64_t)sm_count() * 16);
}

int launch_tpot(const asr_req_t *trace, int64_t n, asr_cost_model_t cm, const int64_t *lat, const int64_t *ttft,
                int64_t *out, cudaStream_t st) {
    {
        KernelTimer kt(KID_TPOT, st);
        tpot_kernel<<<stream_grid(n), 256, 0, st>>>(trace, n, cm, lat, ttft, out);
    }
    return check_launch("tpot_kernel");
}

int launch_estimate(asr_req_t *recs, int64_t n, const KappaTable &ktab, const uint8_t *lang, const int32_t *speech_ms,
                    cudaStream_t st) {
    {
        KernelTimer kt(KID_ESTIMATE, st);
        estimate_kernel<<<stream_grid(n), 256, 0, st>>>(recs, n, ktab, lang, speech_ms);
    }
    return check_launch("estimate_kernel");
}

}  // namespace asr

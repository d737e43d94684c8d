// gen_trace.cu -- a1 integer-only, counter-based trace generator, sm_100a.
//
// Poisson arrivals ("burstiness 1.0"): exponential gaps drawn as
// E = G*ln2 + E' in Q32 (G = leading-zero count of a fresh 64-bit word, E' a
// table-interpolated exponential truncated to [0, ln 2)), scaled by the mean
// gap and prefix-summed in int64.  Durations: a table-interpolated quantile
// (the clipped lognormal that stands in for LibriSpeech) or a
// uniform integer number of ms (the drift workload).  Draw i of
// stream s of seed z is the (i+1)-th output of a splitmix64 sequence whose
// start state is a hash of (z, s): stateless, so any record can be generated
// independently and the same recipe runs on any machine bit for bit.
// HBM-write-bound: 16 B per record.
#include "launchers.cuh"

namespace asr {

constexpr int GEN_THREADS = 256;

__device__ __forceinline__ uint64_t mix_fin(uint64_t z) {
    z ^= z >> 30;
    z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 27;
    z *= 0x94D049BB133111EBull;
    z ^= z >> 31;
    return z;
}

__device__ __forceinline__ uint64_t stream_base(uint64_t seed, uint32_t stream) {
    return mix_fin(mix_fin(seed + 0x2545F4914F6CDD1Dull) + (uint64_t)stream * 0xD1B54A32D192ED03ull);
}

__device__ __forceinline__ uint64_t draw(uint64_t base, uint64_t i) {
    return mix_fin(base + (i + 1ull) * 0x9E3779B97F4A7C15ull);
}

__device__ __forceinline__ uint64_t table_interp(const uint32_t *__restrict__ T, uint64_t u) {
    const uint32_t cell = (uint32_t)(u >> 52);
    const uint64_t frac = (u >> 20) & 0xFFFFFFFFull;
    const uint64_t a = __ldg(T + cell), b = __ldg(T + cell + 1);
    return a + (((b - a) * frac) >> 32);
}

__device__ __forceinline__ int32_t draw_dur(uint64_t u, int dist, const uint32_t *__restrict__ ln_dur) {
    if (dist == ASR_DIST_UNIFORM) return (int32_t)(1000u + (uint32_t)(((u >> 32) * 34001ull) >> 32));
    return (int32_t)table_interp(ln_dur, u);
}

__device__ __forceinline__ void st_rec(asr_req_t *p, int64_t arr, int32_t dur) {
    int4 v = make_int4((int)(uint32_t)arr, (int)(arr >> 32), dur, dur);   // est = dur_ms
    *reinterpret_cast<int4 *>(p) = v;
}

// One CTA per aligned block of GEN_GROUP consecutive specs, cut into runs of equal (seed, dist).  The draws of
// record i depend on (seed, i) only (common random numbers: the traces of one seed at different rates are
// time-scaled copies), so a run hashes and interpolates each record ONCE and every trace of the run only
// scales the unit exponential by its own mean gap, scans and stores.  A thread owns GEN_RPT consecutive
// records of a GEN_CHUNK-record step: local prefix in registers, one warp scan of the thread totals per
// trace, one pass of warp 0 over the [trace][warp] totals that also carries the running sum.
constexpr int GEN_RPT = 4;
constexpr int GEN_CHUNK = GEN_THREADS * GEN_RPT;
constexpr int GEN_GROUP = 8;
constexpr int GEN_WARPS = GEN_THREADS / 32;
static_assert(GEN_GROUP * GEN_WARPS == 64, "warp 0 folds the [trace][warp] totals two per lane");

// (e * mean_gap) >> 32 for e < 2^38 (clz <= 63 times a 32-bit ln 2, plus a 32-bit table value), mean_gap < 2^30
__device__ __forceinline__ uint64_t scale_gap(uint64_t e, uint32_t mean_gap) {
    return (uint64_t)(uint32_t)(e >> 32) * mean_gap + __umulhi((uint32_t)e, mean_gap);
}

// four consecutive records of one thread: two 256-bit stores when the address allows it (sm_100 has them; a
// 16-byte store per lane at a 64-byte stride would fill every 32-byte sector in two separate requests)
__device__ __forceinline__ void st_rec4(asr_req_t *p, const int64_t (&arr)[GEN_RPT], const int32_t (&dur)[GEN_RPT],
                                        bool wide, int n_valid) {
    static_assert(GEN_RPT == 4, "two 32-byte stores");
    if (wide && n_valid == GEN_RPT) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const uint64_t d0 = ((uint64_t)(uint32_t)dur[2 * h] << 32) | (uint32_t)dur[2 * h];   // dur_ms, est = dur_ms
            const uint64_t d1 = ((uint64_t)(uint32_t)dur[2 * h + 1] << 32) | (uint32_t)dur[2 * h + 1];
            asm volatile("st.global.v4.b64 [%0], {%1, %2, %3, %4};" ::"l"(p + 2 * h), "l"(arr[2 * h]), "l"(d0),
                         "l"(arr[2 * h + 1]), "l"(d1)
                         : "memory");
        }
    } else {
#pragma unroll
        for (int j = 0; j < GEN_RPT; ++j)
            if (j < n_valid) st_rec(p + j, arr[j], dur[j]);
    }
}

constexpr uint32_t GEN_SKIP = 0xFFFFFFFFu;
struct GenSmem {
    int64_t warp_tot[GEN_GROUP][GEN_WARPS];   // per trace: the warps' gap sums of this step
    int64_t warp_off[GEN_GROUP][GEN_WARPS];   // per trace: arrival before the warp's first record
    uint64_t seed[GEN_GROUP];
    int32_t dist[GEN_GROUP];
    uint32_t gap[GEN_GROUP];                  // mean gap in us (<= 10^9; 0 above 10^9 mHz), GEN_SKIP: rate_mhz < 1
};

// one run of m traces with equal (seed, dist), first trace r0 of the unit; FULL: m == GEN_GROUP, so that the
// per-trace blocks carry no branch and the compiler interleaves the eight independent scans
template <bool FULL>
__device__ __forceinline__ void gen_run(GenSmem &sm, int r0, int m, int64_t n_per_trace, const asr_tables_t *tables,
                                        asr_req_t *dst) {
    const int lane = lane_id(), warp = threadIdx.x >> 5;
    const uint64_t ln2_q32 = tables->exp_t[4096];
    const uint64_t seed = sm.seed[r0];
    const int dist = sm.dist[r0];
    const uint64_t b0 = stream_base(seed, 0), b1 = stream_base(seed, 1), b2 = stream_base(seed, 2);
    const bool wide = (n_per_trace & 1) == 0 && (reinterpret_cast<uintptr_t>(dst) & 31u) == 0;
    // warp 0, every 8-lane segment: running arrival of traces (lane>>3) and (lane>>3)+4
    int64_t carry_a = 0, carry_b = 0;
    for (int64_t base = 0; base < n_per_trace; base += GEN_CHUNK) {
        const int64_t i0 = base + (int64_t)threadIdx.x * GEN_RPT;
        const int64_t left = n_per_trace - i0;
        const int n_valid = left >= GEN_RPT ? GEN_RPT : (left > 0 ? (int)left : 0);
        uint64_t e[GEN_RPT];
        int32_t dur[GEN_RPT];
#pragma unroll
        for (int j = 0; j < GEN_RPT; ++j) {
            const uint64_t i = (uint64_t)(i0 + j);
            e[j] = 0;
            dur[j] = 0;
            if (j < n_valid) {
                const uint64_t u0 = draw(b0, i), u1 = draw(b1, i), u2 = draw(b2, i);
                e[j] = (uint64_t)__clzll((long long)(u0 | 1ull)) * ln2_q32 + table_interp(tables->exp_t, u1);
                dur[j] = draw_dur(u2, dist, tables->ln_dur);
            }
        }
        int64_t excl[GEN_GROUP];   // per trace: gap sum of the warp's lower lanes
#pragma unroll
        for (int g = 0; g < GEN_GROUP; ++g) {
            excl[g] = 0;
            if (FULL || g < m) {
                const uint32_t mg = sm.gap[r0 + g];
                int64_t tot = 0;
#pragma unroll
                for (int j = 0; j < GEN_RPT; ++j) tot += (int64_t)scale_gap(e[j], mg);
                int64_t x = tot;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const int64_t y = shfl64(x, lane >= d ? lane - d : lane);
                    if (lane >= d) x += y;
                }
                excl[g] = x - tot;
                if (lane == 31) sm.warp_tot[g][warp] = x;
            }
        }
        __syncthreads();
        if (warp == 0) {
            const int ga = lane >> 3, w = lane & 7;
            int64_t ta = ga < m ? sm.warp_tot[ga][w] : 0, tb = ga + 4 < m ? sm.warp_tot[ga + 4][w] : 0;
            int64_t xa = ta, xb = tb;
#pragma unroll
            for (int d = 1; d < 8; d <<= 1) {
                const int64_t ya = shfl64(xa, w >= d ? lane - d : lane), yb = shfl64(xb, w >= d ? lane - d : lane);
                if (w >= d) {
                    xa += ya;
                    xb += yb;
                }
            }
            if (ga < m) sm.warp_off[ga][w] = carry_a + xa - ta;
            if (ga + 4 < m) sm.warp_off[ga + 4][w] = carry_b + xb - tb;
            carry_a += shfl64(xa, lane | 7);
            carry_b += shfl64(xb, lane | 7);
        }
        __syncthreads();
#pragma unroll
        for (int g = 0; g < GEN_GROUP; ++g) {
            if (FULL || g < m) {
                const uint32_t mg = sm.gap[r0 + g];
                if (mg != GEN_SKIP && n_valid > 0) {
                    int64_t arr[GEN_RPT];
                    int64_t run = sm.warp_off[g][warp] + excl[g];
#pragma unroll
                    for (int j = 0; j < GEN_RPT; ++j) {
                        run += (int64_t)scale_gap(e[j], mg);
                        arr[j] = run;
                    }
                    st_rec4(dst + (int64_t)g * n_per_trace + i0, arr, dur, wide, n_valid);
                }
            }
        }
    }
}

#ifndef GEN_MIN_CTAS
#define GEN_MIN_CTAS 4
#endif
__global__ void __launch_bounds__(GEN_THREADS, GEN_MIN_CTAS) gen_trace_kernel(const asr_trace_spec_t *specs, asr_trace_spec_t one,
                                                                int32_t n_traces, int64_t n_per_trace,
                                                                const asr_tables_t *tables, asr_req_t *out) {
    __shared__ GenSmem sm;
    const int n_units = (n_traces + GEN_GROUP - 1) / GEN_GROUP;
    for (int unit = blockIdx.x; unit < n_units; unit += gridDim.x) {
        const int t_first = unit * GEN_GROUP;
        const int cnt = n_traces - t_first < GEN_GROUP ? n_traces - t_first : GEN_GROUP;
        __syncthreads();
        if ((int)threadIdx.x < cnt) {
            const asr_trace_spec_t sp = specs ? specs[t_first + threadIdx.x] : one;
            sm.seed[threadIdx.x] = sp.seed;
            sm.dist[threadIdx.x] = sp.dist;
            sm.gap[threadIdx.x] = sp.rate_mhz < 1 ? GEN_SKIP : (uint32_t)(1000000000u / (uint32_t)sp.rate_mhz);
        }
        __syncthreads();
        for (int r0 = 0; r0 < cnt;) {
            int m = 1;
            while (r0 + m < cnt && sm.seed[r0 + m] == sm.seed[r0] && sm.dist[r0 + m] == sm.dist[r0]) ++m;
            asr_req_t *dst = out + (int64_t)(t_first + r0) * n_per_trace;
            if (m == GEN_GROUP) gen_run<true>(sm, r0, m, n_per_trace, tables, dst);
            else gen_run<false>(sm, r0, m, n_per_trace, tables, dst);
            r0 += m;
        }
    }
}

__global__ void __launch_bounds__(GEN_THREADS) gen_queues_kernel(uint64_t seed, int64_t first, int64_t n, int64_t now,
                                                                 const asr_tables_t *tables, asr_req_t *out) {
    const uint64_t b2 = stream_base(seed, 2), b3 = stream_base(seed, 3);
    const int64_t stride = (int64_t)gridDim.x * GEN_THREADS;
    for (int64_t j = (int64_t)blockIdx.x * GEN_THREADS + threadIdx.x; j < n; j += stride) {
        const uint64_t i = (uint64_t)(first + j);
        const uint64_t u2 = draw(b2, i), u3 = draw(b3, i);
        const int64_t arr = (int64_t)__umul64hi(u3, (uint64_t)now);
        st_rec(out + j, arr, draw_dur(u2, ASR_DIST_LOGNORMAL, tables->ln_dur));
    }
}

int launch_gen_trace(const asr_trace_spec_t *specs, asr_trace_spec_t one, int32_t n_traces, int64_t n_per_trace,
                     const asr_tables_t *tables, asr_req_t *out, cudaStream_t st) {
    if (n_traces <= 0 || n_per_trace <= 0) return ASR_OK;
    const int n_units = (n_traces + GEN_GROUP - 1) / GEN_GROUP;
    int grid = n_units < sm_count() * 64 ? n_units : sm_count() * 64;
    {
        KernelTimer kt(KID_GEN_TRACE, st);
        gen_trace_kernel<<<grid, GEN_THREADS, 0, st>>>(specs, one, n_traces, n_per_trace, tables, out);
    }
    return check_launch("gen_trace_kernel");
}

int launch_gen_queues(uint64_t seed, int64_t first, int64_t n, int64_t now, const asr_tables_t *tables,
                      asr_req_t *out, cudaStream_t st) {
    if (n <= 0) return ASR_OK;
    int64_t want = (n + GEN_THREADS - 1) / GEN_THREADS;
    int grid = (int)(want < (int64_t)sm_count() * 16 ? want : (int64_t)sm_count() * 16);
    {
        KernelTimer kt(KID_GEN_QUEUES, st);
        gen_queues_kernel<<<grid, GEN_THREADS, 0, st>>>(seed, first, n, now, tables, out);
    }
    return check_launch("gen_queues_kernel");
}

}  // namespace asr

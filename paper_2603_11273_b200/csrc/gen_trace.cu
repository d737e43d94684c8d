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

// one CTA per trace; 256 records per step, running int64 carry
__global__ void __launch_bounds__(GEN_THREADS) gen_trace_kernel(const asr_trace_spec_t *specs, asr_trace_spec_t one,
                                                                int32_t n_traces, int64_t n_per_trace,
                                                                const asr_tables_t *tables, asr_req_t *out) {
    __shared__ int64_t warp_tot[GEN_THREADS / 32];
    const int lane = lane_id(), warp = threadIdx.x >> 5;
    for (int tr = blockIdx.x; tr < n_traces; tr += gridDim.x) {
        const asr_trace_spec_t sp = specs ? specs[tr] : one;
        asr_req_t *dst = out + (int64_t)tr * n_per_trace;
        if (sp.rate_mhz < 1) continue;
        const uint64_t mean_gap = 1000000000ull / (uint64_t)sp.rate_mhz;
        const uint64_t ln2_q32 = tables->exp_t[4096];
        const uint64_t b0 = stream_base(sp.seed, 0), b1 = stream_base(sp.seed, 1), b2 = stream_base(sp.seed, 2);
        int64_t carry = 0;
        for (int64_t base = 0; base < n_per_trace; base += GEN_THREADS) {
            const int64_t i = base + threadIdx.x;
            int64_t gap = 0;
            int32_t dur = 0;
            if (i < n_per_trace) {
                const uint64_t u0 = draw(b0, (uint64_t)i), u1 = draw(b1, (uint64_t)i), u2 = draw(b2, (uint64_t)i);
                const uint64_t e = (uint64_t)__clzll((long long)(u0 | 1ull)) * ln2_q32 +
                                   table_interp(tables->exp_t, u1);
                gap = (int64_t)((__umul64hi(e, mean_gap) << 32) | ((e * mean_gap) >> 32));
                dur = draw_dur(u2, sp.dist, tables->ln_dur);
            }
            // inclusive block scan of the gaps
            int64_t x = gap;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                int64_t y = shfl64(x, lane >= d ? lane - d : lane);
                if (lane >= d) x += y;
            }
            __syncthreads();
            if (lane == 31) warp_tot[warp] = x;
            __syncthreads();
            int64_t before = 0, total = 0;
#pragma unroll
            for (int w = 0; w < GEN_THREADS / 32; ++w) {
                const int64_t wt = warp_tot[w];
                if (w < warp) before += wt;
                total += wt;
            }
            if (i < n_per_trace) st_rec(dst + i, carry + before + x, dur);
            carry += total;
        }
        __syncthreads();
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
    int grid = n_traces < 148 * 64 ? n_traces : 148 * 64;
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
    int grid = (int)(want < 148 * 16 ? want : 148 * 16);
    {
        KernelTimer kt(KID_GEN_QUEUES, st);
        gen_queues_kernel<<<grid, GEN_THREADS, 0, st>>>(seed, first, n, now, tables, out);
    }
    return check_launch("gen_queues_kernel");
}

}  // namespace asr

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
        e = e < 1 ? 1 : (e > 0x7FFFFFFF ? 0x7FFFFFFF : e);
        recs[i].est = (int32_t)e;
    }
}

static int stream_grid(int64_t n) {
    const int64_t want = (n + 255) / 256;
    return (int)(want < 148 * 16 ? want : 148 * 16);
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

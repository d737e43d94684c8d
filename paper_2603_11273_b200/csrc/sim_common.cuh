// sim_common.cuh -- helpers shared by the simulator kernels (simulate.cu, simulate_cta.cu).
#pragma once
#include "launchers.cuh"

namespace asr {

constexpr int SIM_WARPS = 4;
constexpr int32_t REM_FREE = 0x7FFFFFFF;

__device__ __forceinline__ int64_t ceil_div_pos(int64_t g, int64_t c) {
    // g > 0, c > 0; 32-bit divide whenever both operands fit
    if ((((uint64_t)g | (uint64_t)c) >> 32) == 0) {
        const uint32_t q = (uint32_t)g / (uint32_t)c;
        return (int64_t)q + ((uint32_t)g - q * (uint32_t)c != 0u ? 1 : 0);
    }
    const uint64_t q = (uint64_t)g / (uint64_t)c;
    return (int64_t)q + ((uint64_t)g - q * (uint64_t)c != 0ull ? 1 : 0);
}

__device__ __forceinline__ int32_t tokens_of(const asr_cost_model_t &cm, int32_t dur_ms) {
    int64_t t = (int64_t)cm.tok_base + ((int64_t)cm.tok_per_s * (int64_t)dur_ms) / 1000;
    t = t < 1 ? 1 : t;
    return t > 0x7FFFFFFE ? 0x7FFFFFFE : (int32_t)t;
}

// sum over the warp of a non-negative 32-bit value per lane, exact in 64 bits
__device__ __forceinline__ int64_t warp_sum_u32(uint32_t v) {
    uint32_t lo = __reduce_add_sync(ASR_FULL_MASK, v & 0xFFFFu);
    uint32_t hi = __reduce_add_sync(ASR_FULL_MASK, v >> 16);
    return ((int64_t)hi << 16) + (int64_t)lo;
}

// true if the descriptor of replica r can be simulated with `max_slots` slots per replica
__device__ __forceinline__ bool replica_ok(const SimArgs &a, const asr_replica_t &rep, int max_slots) {
    return rep.n >= 0 && rep.slots >= 1 && rep.slots <= max_slots && rep.policy >= 0 && rep.policy <= 2 &&
           rep.cm_id >= 0 && rep.cm_id < a.n_cms && rep.trace_off >= 0 && rep.out_off >= 0 &&
           rep.out_off + (int64_t)rep.n <= a.total_requests;
}

__device__ __forceinline__ void flag_invalid(const SimArgs &a, int r) {
    if (!a.out_summary) return;
    asr_summary_t s;
    s.p50_e2e_us = s.p90_e2e_us = s.p50_ttft_us = s.p90_ttft_us = -1;
    s.first_arrival_us = s.last_done_us = 0;
    s.n_done = -1;
    a.out_summary[r] = s;
}

}  // namespace asr

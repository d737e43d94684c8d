// common.cuh -- device helpers shared by the sm_100a kernels of libasr_sched.
// Product code: shares nothing with the CPU checker used by the tests.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "asr_sched.h"

#define ASR_FULL_MASK 0xFFFFFFFFu

namespace asr {

// ---- host-side error plumbing (api.cu) ------------------------------------
void set_error(const char *fmt, ...);
int check_launch(const char *what);   // cudaGetLastError -> ASR_OK / ASR_ECUDA
void count_launch(int n = 1);
int sm_count();                       // SMs of the current device (queried, cached per device)

// kernel ids of the per-kernel CUDA-event timing facility (asr_sched_timing_*)
enum KernelId {
    KID_SELECT = 0, KID_SIM_PREPARE, KID_SIMULATE, KID_SIM_LANE, KID_SUMMARY_PCT, KID_PERCENTILES, KID_GEN_TRACE,
    KID_GEN_QUEUES, KID_SWEEP_REPLICAS, KID_SIM_CTA, KID_SIM_INIT_LAT, KID_SIM_EX, KID_TPOT, KID_ESTIMATE, KID_ITL_PCT, KID_SUMMARY_FAST, KID_LANE_PLAN, KID_SIM_REPAIR, KID_SIM_REDO, KID_SELECT_WIDE, KID_COUNT
};
// RAII: counts the launch and, when timing is enabled, brackets it with an
// event pair recorded on the launching stream.
struct KernelTimer {
    KernelTimer(int kid, cudaStream_t st);
    ~KernelTimer();
    int kid_;
    cudaStream_t st_;
    int slot_;
};

// ---- 128-bit record access -------------------------------------------------
struct __align__(16) Rec {
    int64_t arrival_us;
    int32_t dur_ms;
    int32_t est;
};
static_assert(sizeof(Rec) == sizeof(asr_req_t), "record layout");

// streaming load: read once, keep out of L1
__device__ __forceinline__ Rec ld_stream(const asr_req_t *p) {
    int4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                 : "l"(p));
    Rec r;
    r.arrival_us = (int64_t)(((uint64_t)(uint32_t)v.y << 32) | (uint32_t)v.x);
    r.dur_ms = v.z;
    r.est = v.w;
    return r;
}

__device__ __forceinline__ int64_t rec_arrival(const int4 &v) {
    return (int64_t)(((uint64_t)(uint32_t)v.y << 32) | (uint32_t)v.x);
}

// cached load (trace windows that are re-read by the simulator)
__device__ __forceinline__ Rec ld_cached(const asr_req_t *p) {
    int4 v = __ldg(reinterpret_cast<const int4 *>(p));
    Rec r;
    r.arrival_us = (int64_t)(((uint64_t)(uint32_t)v.y << 32) | (uint32_t)v.x);
    r.dur_ms = v.z;
    r.est = v.w;
    return r;
}

// ---- the total order (asr_sched.h "TOTAL ORDER") -----------------------------
// a2: priority keys.  FCFS PAPER.md:13; SJF PAPER.md:277; HRRN PAPER.md:282.
__device__ __forceinline__ int64_t est_of(int32_t est) { return est < 1 ? 1 : (int64_t)est; }

__device__ __forceinline__ int64_t wait_of(int64_t arrival_us, int64_t now) {
    int64_t w = now - arrival_us;
    return w < 0 ? 0 : w;
}

__device__ __forceinline__ bool earlier(int64_t arr_a, int32_t idx_a, int64_t arr_b, int32_t idx_b) {
    return arr_a != arr_b ? arr_a < arr_b : idx_a < idx_b;
}

template <int POLICY>
__device__ __forceinline__ bool better(int64_t arr_a, int32_t est_a, int32_t idx_a, int64_t arr_b,
                                       int32_t est_b, int32_t idx_b, int64_t now) {
    if (POLICY == ASR_FCFS) return earlier(arr_a, idx_a, arr_b, idx_b);
    if (POLICY == ASR_SJF) {
        int64_t ea = est_of(est_a), eb = est_of(est_b);
        if (ea != eb) return ea < eb;
        return earlier(arr_a, idx_a, arr_b, idx_b);
    }
    // HRRN: (wa+ea)/ea > (wb+eb)/eb  <=>  wa*eb > wb*ea ; products < 2^62 under
    // the documented bounds (wait < 2^38, est <= 2^24)
    int64_t lhs = wait_of(arr_a, now) * est_of(est_b);
    int64_t rhs = wait_of(arr_b, now) * est_of(est_a);
    if (lhs != rhs) return lhs > rhs;
    return earlier(arr_a, idx_a, arr_b, idx_b);
}

__device__ __forceinline__ bool better_rt(int policy, int64_t arr_a, int32_t est_a, int32_t idx_a,
                                          int64_t arr_b, int32_t est_b, int32_t idx_b, int64_t now) {
    if (policy == ASR_FCFS) return better<ASR_FCFS>(arr_a, est_a, idx_a, arr_b, est_b, idx_b, now);
    if (policy == ASR_SJF) return better<ASR_SJF>(arr_a, est_a, idx_a, arr_b, est_b, idx_b, now);
    return better<ASR_HRRN>(arr_a, est_a, idx_a, arr_b, est_b, idx_b, now);
}

// ---- candidate records (arrival lo, arrival hi, max(est,1), idx) and their order scalar ----
__device__ __forceinline__ int64_t rec_arr(const int4 &r) {
    return (int64_t)(((uint64_t)(uint32_t)r.y << 32) | (uint32_t)r.x);
}

// a * b for |a| < 2^62 / b: one wide multiply + one multiply-add (the compiler's
// generic 64x64 product costs twice that)
__device__ __forceinline__ int64_t mul64x32(int64_t a, uint32_t b) {
    uint64_t lo;
    uint32_t hi;
    asm("mul.wide.u32 %0, %1, %2;" : "=l"(lo) : "r"((uint32_t)a), "r"(b));
    asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(hi) : "r"((uint32_t)(a >> 32)), "r"(b), "r"((uint32_t)(lo >> 32)));
    return (int64_t)(((uint64_t)hi << 32) | (uint32_t)lo);
}

// ---- order scalar ---------------------------------------------------------------
// A 64-bit scalar that is WEAKLY order-preserving: scalar(a) < scalar(b) implies
// that a is better than b under the total order; equal scalars say nothing and
// are settled by the exact comparator.  It makes the common-case comparison of
// the quickselect and of the final sort one 64-bit compare.
//   FCFS  arrival
//   SJF   est (>= 1) above the arrival time in units of 256 us, saturated
//   HRRN  the IEEE double quotient wait/est, negated: wait < 2^53 and est are exact
//         in double and the division is correctly rounded, hence monotone in the
//         exact ratio (a strictly larger double means a strictly larger ratio)
template <int POLICY>
__device__ __forceinline__ int64_t order_scalar(const int4 &e, int64_t now) {
    const int64_t arr = rec_arr(e);
    if (POLICY == ASR_FCFS) return arr;
    if (POLICY == ASR_SJF) {
        int64_t a8 = arr >> 8;
        a8 = a8 < 0 ? 0 : (a8 > 0xFFFFFFFFll ? 0xFFFFFFFFll : a8);
        return ((int64_t)e.z << 32) | a8;
    }
    const double r = (double)wait_of(arr, now) / (double)e.z;   // e.z = max(est, 1)
    return INT64_MAX - __double_as_longlong(r);
}

// ---- warp helpers -----------------------------------------------------------
__device__ __forceinline__ int lane_id() { return threadIdx.x & 31; }

__device__ __forceinline__ int64_t shfl64(int64_t v, int src) {
    int lo = __shfl_sync(ASR_FULL_MASK, (int)(uint32_t)v, src);
    int hi = __shfl_sync(ASR_FULL_MASK, (int)(v >> 32), src);
    return (int64_t)(((uint64_t)(uint32_t)hi << 32) | (uint32_t)lo);
}

__device__ __forceinline__ uint64_t shfl64_xor(uint64_t v, int m) {
    uint32_t lo = __shfl_xor_sync(ASR_FULL_MASK, (uint32_t)v, m);
    uint32_t hi = __shfl_xor_sync(ASR_FULL_MASK, (uint32_t)(v >> 32), m);
    return ((uint64_t)hi << 32) | lo;
}

// ---- TMA bulk copy + mbarrier (PTX) -------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile(
            "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
            : "=r"(ok)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!ok);
}


}  // namespace asr

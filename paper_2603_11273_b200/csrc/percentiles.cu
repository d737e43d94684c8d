// percentiles.cu -- a6 segmented nearest-rank percentiles, sm_100a.
//
// One CTA per segment.  The segment is read from HBM once (staged into shared
// memory when it fits), reduced to its min/max, and each requested rank is
// found by an MSB-first radix select over (value - min): 8-bit digits, a
// 256-bin shared-memory histogram per pass, only as many passes as the value
// range needs (a 2 s latency spread in microseconds is 21 bits = 3 passes).
// Nearest rank (asr_sched.h): element of 1-based rank
// ceil(p*N/100) of the sorted segment; an empty segment gives -1.
#include "launchers.cuh"

namespace asr {

constexpr int PCT_THREADS = 256;
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
                                    int64_t *results, int64_t *smem_vals) {
    __shared__ uint32_t hist[256];
    __shared__ int64_t scratch[PCT_THREADS / 32];
    __shared__ uint32_t sel_digit, sel_below;

    if (N <= 0) {
        for (int j = 0; j < pl.n_pct; ++j) results[j] = -1;
        return;
    }
    const bool staged = N <= PCT_SMEM_VALUES;
    int64_t mn = INT64_MAX, mx = INT64_MIN;
    for (int64_t i = threadIdx.x; i < N; i += PCT_THREADS) {
        int64_t x = v[i];
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
                hist[threadIdx.x] = 0;   // PCT_THREADS == 256
                __syncthreads();
                for (int64_t i = threadIdx.x; i < N; i += PCT_THREADS) {
                    uint64_t key = (uint64_t)src[i] - (uint64_t)mn;
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

__global__ void __launch_bounds__(PCT_THREADS) percentiles_kernel(const int64_t *values, const int64_t *seg_off,
                                                                  int32_t n_seg, PctList pl, int64_t *out) {
    extern __shared__ __align__(16) unsigned char dyn_smem[];
    int64_t *smem_vals = reinterpret_cast<int64_t *>(dyn_smem);
    for (int s = blockIdx.x; s < n_seg; s += gridDim.x) {
        const int64_t b = seg_off[s], e = seg_off[s + 1];
        int64_t res[PCT_MAX];
        segment_percentiles(values + b, e - b, pl, res, smem_vals);
        if (threadIdx.x == 0)
            for (int j = 0; j < pl.n_pct; ++j) out[(int64_t)s * pl.n_pct + j] = res[j];
    }
}

// p50/p90 of E2E latency (blockIdx.y = 0) and TTFT (blockIdx.y = 1) of every replica
__global__ void __launch_bounds__(PCT_THREADS) summary_percentiles_kernel(const asr_replica_t *replicas,
                                                                          int32_t n_replicas, const int64_t *lat,
                                                                          const int64_t *ttft,
                                                                          asr_summary_t *out_summary) {
    extern __shared__ __align__(16) unsigned char dyn_smem[];
    int64_t *smem_vals = reinterpret_cast<int64_t *>(dyn_smem);
    PctList pl;
    pl.n_pct = 2;
    pl.pct[0] = 50;
    pl.pct[1] = 90;
    const int64_t *vals = blockIdx.y == 0 ? lat : ttft;
    for (int r = blockIdx.x; r < n_replicas; r += gridDim.x) {
        if (out_summary[r].n_done < 0) continue;   // invalid descriptor, flagged by the simulator
        const asr_replica_t rep = replicas[r];
        int64_t res[PCT_MAX];
        segment_percentiles(vals + rep.out_off, rep.n, pl, res, smem_vals);
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

static constexpr size_t PCT_DYN_SMEM = (size_t)PCT_SMEM_VALUES * sizeof(int64_t);

static int pct_grid(int n_units, const void *fn) {
    static int n_sm = 0;
    int per_sm = 0;
    if (n_sm == 0) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
        if (n_sm < 1) n_sm = 148;
    }
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, PCT_THREADS, PCT_DYN_SMEM);
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
    static bool attr = false;
    if (!attr) {
        cudaFuncSetAttribute(percentiles_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PCT_DYN_SMEM);
        attr = true;
    }
    const int grid = pct_grid(n_seg, (const void *)percentiles_kernel);
    {
        KernelTimer kt(KID_PERCENTILES, st);
        percentiles_kernel<<<grid, PCT_THREADS, PCT_DYN_SMEM, st>>>(values, seg_off, n_seg, pl, out);
    }
    return check_launch("percentiles_kernel");
}

int launch_summary_percentiles(const asr_replica_t *replicas, int32_t n_replicas, const int64_t *lat,
                               const int64_t *ttft, asr_summary_t *out_summary, cudaStream_t st) {
    if (n_replicas <= 0) return ASR_OK;
    static bool attr = false;
    if (!attr) {
        cudaFuncSetAttribute(summary_percentiles_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)PCT_DYN_SMEM);
        attr = true;
    }
    int gx = pct_grid(n_replicas, (const void *)summary_percentiles_kernel);
    gx = gx > 1 ? (gx + 1) / 2 : 1;
    dim3 grid(gx, 2);
    {
        KernelTimer kt(KID_SUMMARY_PCT, st);
        summary_percentiles_kernel<<<grid, PCT_THREADS, PCT_DYN_SMEM, st>>>(replicas, n_replicas, lat, ttft, out_summary);
    }
    return check_launch("summary_percentiles_kernel");
}

}  // namespace asr

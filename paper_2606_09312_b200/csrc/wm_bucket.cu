// K1 (DESIGN.md §1 step a0): counting sort of the candidates by (clamped) sequence length, longest first, so a
// tile of consecutive entries of `perm` holds sequences of (almost) equal length and no MMA row idles
// (BASELINE.json north_star: "variable-length sequences are bucketed or sorted by length").
//
// Integer work, HBM-bound and tiny (4 B read twice + 4 B written per candidate).  Two launches:
//   hist:    per-CTA shared-memory histogram of lengths -> global hist[T_max+1] (one atomic per CTA and bin)
//   scatter: every CTA rebuilds the descending exclusive scan of hist (<= 257 bins, redundant and cheap), takes
//            a private range of each bin with one global atomic per CTA and bin, and places its candidates.
// The order of candidates INSIDE a length bin depends on atomic arrival order; scores do not (every row of a tile
// is computed independently), so results are bit-identical whatever the order.
#include "wm_internal.h"

namespace wm {

constexpr int kBucketThreads = 512;
constexpr int kBucketItems = 8;   // candidates per thread

__device__ __forceinline__ int clamp_len(int len, int T_max) { return len < 0 ? 0 : (len > T_max ? T_max : len); }
// sort key: the number of rollout steps, i.e. the clamped length minus the clamped start (prefix-latent reuse)
__device__ __forceinline__ int steps_of(const int32_t* __restrict__ lengths, const int32_t* __restrict__ start, int64_t i,
                                        int T_max) {
    const int len = clamp_len(__ldg(lengths + i), T_max);
    return start ? len - clamp_start(__ldg(start + i), len) : len;
}

__global__ void __launch_bounds__(kBucketThreads) wm_len_hist_kernel(const int32_t* __restrict__ lengths,
                                                                     const int32_t* __restrict__ start, int64_t B,
                                                                     int T_max, int32_t* __restrict__ hist) {
    __shared__ int sh[WM_MAX_T + 1];
    for (int i = threadIdx.x; i <= T_max; i += blockDim.x) sh[i] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * (kBucketThreads * kBucketItems);
#pragma unroll
    for (int it = 0; it < kBucketItems; ++it) {
        const int64_t i = base + (int64_t)it * kBucketThreads + threadIdx.x;
        if (i < B) atomicAdd(&sh[steps_of(lengths, start, i, T_max)], 1);
    }
    __syncthreads();
    for (int i = threadIdx.x; i <= T_max; i += blockDim.x)
        if (sh[i]) atomicAdd(&hist[i], sh[i]);
}

__global__ void __launch_bounds__(kBucketThreads) wm_len_scatter_kernel(const int32_t* __restrict__ lengths,
                                                                        const int32_t* __restrict__ start,
                                                                        int64_t B, int T_max,
                                                                        const int32_t* __restrict__ hist,
                                                                        int32_t* __restrict__ cursor,
                                                                        int32_t* __restrict__ perm) {
    __shared__ int s_cnt[WM_MAX_T + 1];    // this CTA's histogram, then its running cursor inside each bin
    __shared__ int s_base[WM_MAX_T + 1];   // global start of the CTA's range in each bin
    for (int i = threadIdx.x; i <= T_max; i += blockDim.x) s_cnt[i] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * (kBucketThreads * kBucketItems);
    int my_len[kBucketItems];
#pragma unroll
    for (int it = 0; it < kBucketItems; ++it) {
        const int64_t i = base + (int64_t)it * kBucketThreads + threadIdx.x;
        my_len[it] = -1;
        if (i < B) {
            my_len[it] = steps_of(lengths, start, i, T_max);
            atomicAdd(&s_cnt[my_len[it]], 1);
        }
    }
    __syncthreads();
    // descending exclusive scan of the global histogram: bin_start[l] = #candidates with length > l.
    // One warp, 257 bins at most: each lane owns a contiguous run of bins, longest first.
    if (threadIdx.x < 32) {
        const int nb = T_max + 1;
        const int per = (nb + 31) / 32;
        const int lane = threadIdx.x;
        int sum = 0;
        for (int q = 0; q < per; ++q) {
            const int bin = T_max - (lane * per + q);
            if (bin >= 0) sum += __ldg(hist + bin);
        }
        int incl = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += v;
        }
        int run = incl - sum;
        for (int q = 0; q < per; ++q) {
            const int bin = T_max - (lane * per + q);
            if (bin >= 0) {
                int mine = 0;
                const int c = s_cnt[bin];
                if (c) mine = atomicAdd(&cursor[bin], c);
                s_base[bin] = run + mine;
                run += __ldg(hist + bin);
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i <= T_max; i += blockDim.x) s_cnt[i] = 0;
    __syncthreads();
#pragma unroll
    for (int it = 0; it < kBucketItems; ++it) {
        if (my_len[it] >= 0) {
            const int64_t i = base + (int64_t)it * kBucketThreads + threadIdx.x;
            const int pos = s_base[my_len[it]] + atomicAdd(&s_cnt[my_len[it]], 1);
            perm[pos] = (int32_t)i;
        }
    }
}

// Both steps in ONE launch for batches whose CTAs are all resident at once (grid <= 32; cfg 2 / 3: 8 / 16
// CTAs): every CTA adds its histogram to the global one, the CTAs meet at a counter (bounded spin; co-residency makes it
// safe), then each takes its ranges and places its candidates as wm_len_scatter_kernel does.  The lengths are read once and
// one launch (of three in an evolution-round-sized call) goes away.  `hist` is read back through L2 (__ldcg): it was written
// by other CTAs' atomics during this launch.
__global__ void __launch_bounds__(kBucketThreads) wm_len_sort_kernel(const int32_t* __restrict__ lengths,
                                                                     const int32_t* __restrict__ start, int64_t B,
                                                                     int T_max, int32_t* hist, int32_t* cursor,
                                                                     int32_t* arrived, int32_t* __restrict__ perm) {
    __shared__ int s_cnt[WM_MAX_T + 1];    // this CTA's histogram, then its running cursor inside each bin
    __shared__ int s_base[WM_MAX_T + 1];   // global start of the CTA's range in each bin
    for (int i = threadIdx.x; i <= T_max; i += blockDim.x) s_cnt[i] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * (kBucketThreads * kBucketItems);
    int my_len[kBucketItems];
#pragma unroll
    for (int it = 0; it < kBucketItems; ++it) {
        const int64_t i = base + (int64_t)it * kBucketThreads + threadIdx.x;
        my_len[it] = -1;
        if (i < B) {
            my_len[it] = steps_of(lengths, start, i, T_max);
            atomicAdd(&s_cnt[my_len[it]], 1);
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i <= T_max; i += blockDim.x)
        if (s_cnt[i]) atomicAdd(&hist[i], s_cnt[i]);
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        atomicAdd(arrived, 1);
        const long long t0 = clock64();
        while (atomicAdd(arrived, 0) < (int)gridDim.x)
            if (clock64() - t0 > 4000000000LL) __trap();      // (a CTA that is not resident would never arrive)
        __threadfence();
    }
    __syncthreads();
    if (threadIdx.x < 32) {
        const int nb = T_max + 1;
        const int per = (nb + 31) / 32;
        const int lane = threadIdx.x;
        int sum = 0;
        for (int q = 0; q < per; ++q) {
            const int bin = T_max - (lane * per + q);
            if (bin >= 0) sum += __ldcg(hist + bin);
        }
        int incl = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += v;
        }
        int run = incl - sum;
        for (int q = 0; q < per; ++q) {
            const int bin = T_max - (lane * per + q);
            if (bin >= 0) {
                int mine = 0;
                const int c = s_cnt[bin];
                if (c) mine = atomicAdd(&cursor[bin], c);
                s_base[bin] = run + mine;
                run += __ldcg(hist + bin);
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i <= T_max; i += blockDim.x) s_cnt[i] = 0;
    __syncthreads();
#pragma unroll
    for (int it = 0; it < kBucketItems; ++it) {
        if (my_len[it] >= 0) {
            const int64_t i = base + (int64_t)it * kBucketThreads + threadIdx.x;
            const int pos = s_base[my_len[it]] + atomicAdd(&s_cnt[my_len[it]], 1);
            perm[pos] = (int32_t)i;
        }
    }
}

int launch_length_bucketing(wm_ctx* ctx, Workspace* ws, const int32_t* lengths, const int32_t* start, int64_t B,
                            int T_max, cudaStream_t st) {
    if (B <= 0) return WM_OK;
    WM_CUDA_TRY(cudaMemsetAsync(ws->counters, 0, sizeof(int32_t) * kCounterInts, st));
    const int64_t per_cta = (int64_t)kBucketThreads * kBucketItems;
    const int grid = (int)((B + per_cta - 1) / per_cta);
    // one launch while every CTA is certainly resident at once: at most kSortMaxCtas CTAs of 512 threads (an SM holds four,
    // so even a dozen such sorts on other streams, or a persistent kernel that leaves a fifth of the SMs, cannot starve the
    // meeting); the counters' memset above clears the meeting word too
    constexpr int kSortMaxCtas = 32;     // 131,072 candidates: cfg 2 (8 CTAs), cfg 3 (16), every search-round-sized call
    if (grid <= kSortMaxCtas && grid <= ctx->n_sms) {
        wm_len_sort_kernel<<<grid, kBucketThreads, 0, st>>>(lengths, start, B, T_max, ws->counters + kHistOff,
                                                            ws->counters + kCursorOff, ws->counters + kTileCtrOff + 1, ws->perm);
        WM_CUDA_TRY(cudaGetLastError());
        ctx->launches.fetch_add(1);
        return WM_OK;
    }
    wm_len_hist_kernel<<<grid, kBucketThreads, 0, st>>>(lengths, start, B, T_max, ws->counters + kHistOff);
    WM_CUDA_TRY(cudaGetLastError());
    wm_len_scatter_kernel<<<grid, kBucketThreads, 0, st>>>(lengths, start, B, T_max, ws->counters + kHistOff,
                                                           ws->counters + kCursorOff, ws->perm);
    WM_CUDA_TRY(cudaGetLastError());
    ctx->launches.fetch_add(2);
    return WM_OK;
}

}  // namespace wm

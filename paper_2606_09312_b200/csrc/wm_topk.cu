// K3 (DESIGN.md §1 step a7): segmented top-k by radix select.  PAPER.md:215 ("rank candidate states and
// prioritize which candidates should be measured"), :64 ("selects only a subset for hardware measurement").
//
// One CTA per subgraph segment.  Scores map to order-preserving 32-bit keys (larger key = better; -0.0 == +0.0;
// NaN -> key 0, below -inf).  Four 8-bit MSB-first histogram passes find the key T of the k-th best candidate and
// how many candidates with key == T still belong to the answer; one ordered compaction pass (index order, block
// scan) collects every key > T plus the FIRST need_eq candidates with key == T (ties go to the lower index); the
// <= 1024 winners are then bitonic-sorted on the 64-bit composite (key, ~index) = (score desc, index asc).
// Integer compares only: the result is bit-exact against a full sort (tests/test_gpu_topk.py).
// Segments of up to kCacheKeys candidates keep their keys in shared memory (one HBM read of 4 B/candidate);
// larger ones re-read the scores (L2-resident) in every pass.
#include "wm_internal.h"

namespace wm {

constexpr int kTopkThreads = 1024;
constexpr int kCacheKeys = 16384;   // 64 KB of keys

static std::atomic<int64_t> g_topk_launches{0};
int64_t topk_launches() { return g_topk_launches.load(); }

__device__ __forceinline__ uint32_t score_key(float v) {
    if (v != v) return 0u;                     // NaN ranks below everything
    uint32_t u = __float_as_uint(v + 0.0f);    // -0.0 + 0.0 = +0.0
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// exclusive block scan of a 32-bit value over kTopkThreads threads; also returns the block total.
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t* warp_sums, uint32_t* total) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    __syncthreads();   // protect warp_sums from the previous use
    if (lane == 31) warp_sums[w] = incl;
    __syncthreads();
    if (w == 0) {
        uint32_t s = warp_sums[lane];
        uint32_t si = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, si, o);
            if (lane >= o) si += t;
        }
        warp_sums[lane] = si - s;
        if (lane == 31) warp_sums[32] = si;
    }
    __syncthreads();
    *total = warp_sums[32];
    return warp_sums[w] + incl - v;
}

__global__ void __launch_bounds__(kTopkThreads) wm_topk_kernel(const float* __restrict__ scores,
                                                               const int32_t* __restrict__ offsets, int k,
                                                               int32_t* __restrict__ idx_out) {
    extern __shared__ __align__(16) unsigned char topk_smem[];
    uint32_t* s_keys = reinterpret_cast<uint32_t*>(topk_smem);                       // [kCacheKeys]
    unsigned long long* s_win = reinterpret_cast<unsigned long long*>(s_keys + kCacheKeys);   // [1024]
    __shared__ uint32_t s_hist[256];
    __shared__ uint32_t s_warp[33];
    __shared__ uint32_t s_sel[2];   // chosen digit, remaining rank

    const int s = blockIdx.x;
    const int tid = threadIdx.x;
    const int base = __ldg(offsets + s);
    const int n = __ldg(offsets + s + 1) - base;
    int32_t* out = idx_out + (size_t)s * k;
    const int kk = n < k ? (n < 0 ? 0 : n) : k;
    for (int j = kk + tid; j < k; j += kTopkThreads) out[j] = -1;
    if (kk == 0) return;
    const bool cached = n <= kCacheKeys;
    if (cached) {
        for (int i = tid; i < n; i += kTopkThreads) s_keys[i] = score_key(__ldg(scores + base + i));
        __syncthreads();
    }
    auto key_at = [&](int i) -> uint32_t { return cached ? s_keys[i] : score_key(__ldg(scores + base + i)); };

    // ---- radix select: key of the kk-th largest
    uint32_t prefix = 0, mask = 0;
    uint32_t remaining = (uint32_t)kk;   // rank (1-based, from the top) still to resolve inside the prefix class
    for (int shift = 24; shift >= 0; shift -= 8) {
        for (int i = tid; i < 256; i += kTopkThreads) s_hist[i] = 0;
        __syncthreads();
        for (int i = tid; i < n; i += kTopkThreads) {
            const uint32_t key = key_at(i);
            if ((key & mask) == prefix) atomicAdd(&s_hist[(key >> shift) & 255u], 1u);
        }
        __syncthreads();
        if (tid < 32) {
            // lane l owns digits 255-8l .. 248-8l (descending)
            uint32_t c[8], sum = 0;
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                c[q] = s_hist[255 - (tid * 8 + q)];
                sum += c[q];
            }
            uint32_t incl = sum;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
                if (tid >= o) incl += t;
            }
            const uint32_t before = incl - sum;
            if (before < remaining && remaining <= incl) {   // exactly one lane
                uint32_t run = before;
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    if (run < remaining && remaining <= run + c[q]) {
                        s_sel[0] = 255u - (uint32_t)(tid * 8 + q);
                        s_sel[1] = remaining - run;
                    }
                    run += c[q];
                }
            }
        }
        __syncthreads();
        prefix |= s_sel[0] << shift;
        mask |= 255u << shift;
        remaining = s_sel[1];
        __syncthreads();
    }
    const uint32_t T = prefix;
    const uint32_t need_eq = remaining;            // candidates with key == T that belong to the answer
    const uint32_t n_gt = (uint32_t)kk - need_eq;  // candidates with key > T

    // ---- ordered compaction (index order) into s_win
    int npow = 1;
    while (npow < kk) npow <<= 1;
    for (int j = tid; j < npow; j += kTopkThreads) s_win[j] = 0ull;
    uint32_t run_gt = 0, run_eq = 0;
    for (int c0 = 0; c0 < n; c0 += kTopkThreads) {
        const int i = c0 + tid;
        uint32_t key = 0;
        bool gt = false, eq = false;
        if (i < n) {
            key = key_at(i);
            gt = key > T;
            eq = key == T;
        }
        uint32_t total;
        const uint32_t packed = block_excl_scan((gt ? 1u : 0u) | (eq ? 0x10000u : 0u), s_warp, &total);
        const uint32_t r_gt = run_gt + (packed & 0xffffu), r_eq = run_eq + (packed >> 16);
        const unsigned long long comp = ((unsigned long long)key << 32) | (unsigned long long)(0xffffffffu - (uint32_t)i);
        if (gt) s_win[r_gt] = comp;
        else if (eq && r_eq < need_eq) s_win[n_gt + r_eq] = comp;
        run_gt += total & 0xffffu;
        run_eq += total >> 16;
        if (run_eq >= need_eq && run_gt >= n_gt) break;   // uniform: totals are block-wide
    }
    __syncthreads();

    // ---- bitonic sort, descending, npow <= 1024 elements, one element per thread
    for (int size = 2; size <= npow; size <<= 1) {
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
            if (tid < npow) {
                const int partner = tid ^ stride;
                if (partner > tid) {
                    const unsigned long long x = s_win[tid], y = s_win[partner];
                    const bool desc = (tid & size) == 0;
                    if (desc ? (x < y) : (x > y)) {
                        s_win[tid] = y;
                        s_win[partner] = x;
                    }
                }
            }
            __syncthreads();
        }
    }
    for (int j = tid; j < kk; j += kTopkThreads)
        out[j] = base + (int32_t)(0xffffffffu - (uint32_t)(s_win[j] & 0xffffffffull));
}

int launch_topk(const float* scores, const int32_t* offsets, int S, int k, int32_t* idx_out, cudaStream_t st) {
    if (S <= 0) return WM_OK;
    const size_t smem = (size_t)kCacheKeys * 4 + 1024 * 8;
    // the attribute is per device and cheap to set; set it on every call so multi-device processes stay correct
    WM_CUDA_TRY(cudaFuncSetAttribute(wm_topk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    wm_topk_kernel<<<S, kTopkThreads, smem, st>>>(scores, offsets, k, idx_out);
    WM_CUDA_TRY(cudaGetLastError());
    g_topk_launches.fetch_add(1);
    return WM_OK;
}

}  // namespace wm

// K2-fp32: the whole hot path (a1-a6 of DESIGN.md §1) on fp32 CUDA cores, for every model kind.
//
// It is the kernel of record for cfg 1 (fp32, 1e-4 tolerance: TF32/bf16 tensor cores cannot meet it) and the
// fallback for the bf16 models the tcgen05 kernel (wm_tc.cu) does not cover yet.  One CTA owns a tile of R
// candidates; all activations of the tile live in shared memory TRANSPOSED ([feature][row], rows contiguous)
// so that (a) a thread that owns one output unit reads the R inputs of a feature as float4 broadcasts and
// (b) element-wise phases map lanes to rows and never bank-conflict.  Weights are read through the read-only
// path from their [in][out] (transposed at load time) layout: consecutive threads -> consecutive addresses.
//
// PAPER.md:162 Eq.8 / :166 (recurrent rollout), :176 (mask), :186-188 Eq.12 (features + score).
#include <math_constants.h>

#include "wm_internal.h"
#include "wm_ptx.cuh"

namespace wm {

struct GenericParams {
    int kind, embed, d, da, hidden, n_types, P, n_buckets, H, n_lin;
    int phi_kind, phi_dim;   // WM_PHI_*; rows of phi in the scorer input (<= da)
    int sdim[kMaxScorerLinears + 1];
    int maxw;        // rows of buffer Hb
    int alt_rows;    // rows of the region that holds V, AS, Y (and the scorer's second ping-pong buffer)
    int xa_rows;     // rows of X's middle part: max(da, phi_dim) (the step's a, then phi for the scorer)
    int as_rows;     // rows of AS: da, or for WM_PHI_TYPED n_types + 2 n_types P (counts, per-type sums, per-type maxima)
    float ln_eps;
    const float *E, *WpT, *bp, *Tbl;
    const float *W1t, *b1, *W2t, *b2, *gamma, *beta;
    const float *Wwt, *Wdt;      // TransH
    const float *Wgt, *Wrt, *Wht;
    const float* Wst[kMaxScorerLinears];
    const float* bs[kMaxScorerLinears];
    CallArgs a;
    int n_tiles;
    // weights-in-shared-memory mode (wm_generic_kernel<R, true>): byte offset of the weight region in dynamic shared memory
    // and the float offsets of W1t, W2t and the scorer matrices inside it
    uint32_t ws_off, ws_bytes;
    uint32_t ws_w1, ws_w2, ws_s[kMaxScorerLinears];
    // ... and of the small tensors: E, WpT, bp, b1, b2, gamma, beta, scorer biases
    uint32_t ws_E, ws_Wp, ws_bp, ws_b1, ws_b2, ws_g, ws_be, ws_bs[kMaxScorerLinears];
    int split_ok;   // every linear's width <= 256: the split-K form applies (R <= 8)
};

enum { ACT_NONE = 0, ACT_GELU = 1, ACT_SIGMOID = 2, ACT_TANH = 3 };
constexpr int kSplitThreads = 256;   // = kGenericThreads (defined below); threads that share one split-K linear

__device__ __forceinline__ float gelu_erf(float x) { return 0.5f * x * (1.0f + erff(x * 0.70710678118654752440f)); }
__device__ __forceinline__ float sigmoidf_(float x) { return 1.0f / (1.0f + expf(-x)); }

template <int ACT>
__device__ __forceinline__ float apply_act(float x) {
    if (ACT == ACT_GELU) return gelu_erf(x);
    if (ACT == ACT_SIGMOID) return sigmoidf_(x);
    if (ACT == ACT_TANH) return tanhf(x);
    return x;
}

// outT[n][r] = act(bias[n] + sum_k Wt[k][n] * inT[k][r]),  n < N, r < R.  inT/outT in shared memory.  WS: Wt is in shared
// memory too (staged once per CTA), read with plain loads: consecutive threads -> consecutive banks.
template <int R, int ACT, bool WS = false>
__device__ void linear_T(const float* __restrict__ Wt, const float* __restrict__ bias, const float* inT, int K,
                         int N, float* outT) {
    int n_first = threadIdx.x;
    if (!WS) {
        // two output units per thread (n and n + blockDim.x) where the layer is wide enough: one read of the R inputs of a
        // feature from shared memory feeds 2 R FMAs (the single-unit loop below issues R / 4 LDS.128 per R FMAs)
        for (; n_first + (int)blockDim.x < N; n_first += 2 * blockDim.x) {
            const int n0 = n_first, n1 = n_first + blockDim.x;
            float acc0[R], acc1[R];
            const float b0 = bias ? __ldg(bias + n0) : 0.0f, b1 = bias ? __ldg(bias + n1) : 0.0f;
#pragma unroll
            for (int r = 0; r < R; ++r) { acc0[r] = b0; acc1[r] = b1; }
            int k = 0;
            for (; k + 8 <= K; k += 8) {
                float w0[8], w1[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    w0[u] = __ldg(Wt + (size_t)(k + u) * N + n0);
                    w1[u] = __ldg(Wt + (size_t)(k + u) * N + n1);
                }
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const float4* xv = reinterpret_cast<const float4*>(inT + (size_t)(k + u) * R);
#pragma unroll
                    for (int q = 0; q < R / 4; ++q) {
                        const float4 x = xv[q];
                        acc0[4 * q + 0] = fmaf(w0[u], x.x, acc0[4 * q + 0]); acc1[4 * q + 0] = fmaf(w1[u], x.x, acc1[4 * q + 0]);
                        acc0[4 * q + 1] = fmaf(w0[u], x.y, acc0[4 * q + 1]); acc1[4 * q + 1] = fmaf(w1[u], x.y, acc1[4 * q + 1]);
                        acc0[4 * q + 2] = fmaf(w0[u], x.z, acc0[4 * q + 2]); acc1[4 * q + 2] = fmaf(w1[u], x.z, acc1[4 * q + 2]);
                        acc0[4 * q + 3] = fmaf(w0[u], x.w, acc0[4 * q + 3]); acc1[4 * q + 3] = fmaf(w1[u], x.w, acc1[4 * q + 3]);
                    }
                }
            }
            for (; k < K; ++k) {
                const float w0 = __ldg(Wt + (size_t)k * N + n0), w1 = __ldg(Wt + (size_t)k * N + n1);
                const float4* xv = reinterpret_cast<const float4*>(inT + (size_t)k * R);
#pragma unroll
                for (int q = 0; q < R / 4; ++q) {
                    const float4 x = xv[q];
                    acc0[4 * q + 0] = fmaf(w0, x.x, acc0[4 * q + 0]); acc1[4 * q + 0] = fmaf(w1, x.x, acc1[4 * q + 0]);
                    acc0[4 * q + 1] = fmaf(w0, x.y, acc0[4 * q + 1]); acc1[4 * q + 1] = fmaf(w1, x.y, acc1[4 * q + 1]);
                    acc0[4 * q + 2] = fmaf(w0, x.z, acc0[4 * q + 2]); acc1[4 * q + 2] = fmaf(w1, x.z, acc1[4 * q + 2]);
                    acc0[4 * q + 3] = fmaf(w0, x.w, acc0[4 * q + 3]); acc1[4 * q + 3] = fmaf(w1, x.w, acc1[4 * q + 3]);
                }
            }
            float4* ov0 = reinterpret_cast<float4*>(outT + (size_t)n0 * R);
            float4* ov1 = reinterpret_cast<float4*>(outT + (size_t)n1 * R);
#pragma unroll
            for (int q = 0; q < R / 4; ++q) {
                ov0[q] = make_float4(apply_act<ACT>(acc0[4 * q + 0]), apply_act<ACT>(acc0[4 * q + 1]),
                                     apply_act<ACT>(acc0[4 * q + 2]), apply_act<ACT>(acc0[4 * q + 3]));
                ov1[q] = make_float4(apply_act<ACT>(acc1[4 * q + 0]), apply_act<ACT>(acc1[4 * q + 1]),
                                     apply_act<ACT>(acc1[4 * q + 2]), apply_act<ACT>(acc1[4 * q + 3]));
            }
        }
    }
    for (int n = n_first; n < N; n += blockDim.x) {
        float acc[R];
        const float b = bias ? (WS ? bias[n] : __ldg(bias + n)) : 0.0f;
#pragma unroll
        for (int r = 0; r < R; ++r) acc[r] = b;
        const float* wp = Wt + n;
        int k = 0;
        // weights from global memory (L2): one CTA of 8 warps per SM cannot hide a ~600-cycle load behind four loads in
        // flight per thread (measured 0.19 of the FFMA peak); sixteen rows are requested before the first is used
        if (!WS) {
            for (; k + 16 <= K; k += 16) {
                float w[16];
#pragma unroll
                for (int u = 0; u < 16; ++u) w[u] = __ldg(wp + (size_t)(k + u) * N);
#pragma unroll
                for (int u = 0; u < 16; ++u) {
                    const float4* xv = reinterpret_cast<const float4*>(inT + (size_t)(k + u) * R);
#pragma unroll
                    for (int q = 0; q < R / 4; ++q) {
                        float4 x = xv[q];
                        acc[4 * q + 0] = fmaf(w[u], x.x, acc[4 * q + 0]);
                        acc[4 * q + 1] = fmaf(w[u], x.y, acc[4 * q + 1]);
                        acc[4 * q + 2] = fmaf(w[u], x.z, acc[4 * q + 2]);
                        acc[4 * q + 3] = fmaf(w[u], x.w, acc[4 * q + 3]);
                    }
                }
            }
        }
        for (; k + 4 <= K; k += 4) {
            float w[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) w[u] = WS ? wp[(size_t)(k + u) * N] : __ldg(wp + (size_t)(k + u) * N);
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const float4* xv = reinterpret_cast<const float4*>(inT + (size_t)(k + u) * R);
#pragma unroll
                for (int q = 0; q < R / 4; ++q) {
                    float4 x = xv[q];
                    acc[4 * q + 0] = fmaf(w[u], x.x, acc[4 * q + 0]);
                    acc[4 * q + 1] = fmaf(w[u], x.y, acc[4 * q + 1]);
                    acc[4 * q + 2] = fmaf(w[u], x.z, acc[4 * q + 2]);
                    acc[4 * q + 3] = fmaf(w[u], x.w, acc[4 * q + 3]);
                }
            }
        }
        for (; k < K; ++k) {
            const float w = WS ? wp[(size_t)k * N] : __ldg(wp + (size_t)k * N);
            const float4* xv = reinterpret_cast<const float4*>(inT + (size_t)k * R);
#pragma unroll
            for (int q = 0; q < R / 4; ++q) {
                float4 x = xv[q];
                acc[4 * q + 0] = fmaf(w, x.x, acc[4 * q + 0]);
                acc[4 * q + 1] = fmaf(w, x.y, acc[4 * q + 1]);
                acc[4 * q + 2] = fmaf(w, x.z, acc[4 * q + 2]);
                acc[4 * q + 3] = fmaf(w, x.w, acc[4 * q + 3]);
            }
        }
        float4* ov = reinterpret_cast<float4*>(outT + (size_t)n * R);
#pragma unroll
        for (int q = 0; q < R / 4; ++q) {
            float4 o;
            o.x = apply_act<ACT>(acc[4 * q + 0]);
            o.y = apply_act<ACT>(acc[4 * q + 1]);
            o.z = apply_act<ACT>(acc[4 * q + 2]);
            o.w = apply_act<ACT>(acc[4 * q + 3]);
            ov[q] = o;
        }
    }
}

// Split-K form for the weights-in-shared-memory mode and small tiles (R <= 8): with N <= 128 output units only N of the
// CTA's 256 threads would work, each on a serial chain of K dependent FMAs — the whole cost of a cfg-1-sized call.  Here
// S = 256 / N thread groups take K / S of the reduction each, partial sums meet in `scratch` ([S][N][R] floats) and the
// first N threads add bias and activation.  Called by all threads (two block barriers inside).
// explicit shared-space load (the matrix pointer reaches linear_T_split as a generic pointer: without this ptxas emits LD.E)
__device__ __forceinline__ float lds_f32(const float* p) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"((uint32_t)__cvta_generic_to_shared(p)));
    return v;
}

template <int R, int ACT>
__device__ void linear_T_split(const float* Wt, const float* bias, const float* inT, int K, int N, float* outT,
                               float* scratch) {
    const int S = N <= kSplitThreads ? kSplitThreads / N : 1;
    const int tid = threadIdx.x;
    const int n = tid % N, part = tid / N;
    if (part < S) {
        const int kc = (K + S - 1) / S, k0 = part * kc, k1 = min(K, k0 + kc);
        float acc[R];
#pragma unroll
        for (int r = 0; r < R; ++r) acc[r] = 0.0f;
        const float* wp = Wt + n;
#pragma unroll 4
        for (int k = k0; k < k1; ++k) {
            const float w = lds_f32(wp + (size_t)k * N);
            const float4* xv = reinterpret_cast<const float4*>(inT + (size_t)k * R);
#pragma unroll
            for (int q = 0; q < R / 4; ++q) {
                const float4 x = xv[q];
                acc[4 * q + 0] = fmaf(w, x.x, acc[4 * q + 0]);
                acc[4 * q + 1] = fmaf(w, x.y, acc[4 * q + 1]);
                acc[4 * q + 2] = fmaf(w, x.z, acc[4 * q + 2]);
                acc[4 * q + 3] = fmaf(w, x.w, acc[4 * q + 3]);
            }
        }
        float4* sv = reinterpret_cast<float4*>(scratch + ((size_t)part * N + n) * R);
#pragma unroll
        for (int q = 0; q < R / 4; ++q) sv[q] = make_float4(acc[4 * q], acc[4 * q + 1], acc[4 * q + 2], acc[4 * q + 3]);
    }
    __syncthreads();
    if (tid < N) {
        float acc[R];
        const float b = bias ? bias[tid] : 0.0f;
#pragma unroll
        for (int r = 0; r < R; ++r) acc[r] = b;
        for (int s = 0; s < S; ++s) {
            const float4* sv = reinterpret_cast<const float4*>(scratch + ((size_t)s * N + tid) * R);
#pragma unroll
            for (int q = 0; q < R / 4; ++q) {
                const float4 x = sv[q];
                acc[4 * q + 0] += x.x; acc[4 * q + 1] += x.y; acc[4 * q + 2] += x.z; acc[4 * q + 3] += x.w;
            }
        }
        float4* ov = reinterpret_cast<float4*>(outT + (size_t)tid * R);
#pragma unroll
        for (int q = 0; q < R / 4; ++q)
            ov[q] = make_float4(apply_act<ACT>(acc[4 * q + 0]), apply_act<ACT>(acc[4 * q + 1]), apply_act<ACT>(acc[4 * q + 2]),
                                apply_act<ACT>(acc[4 * q + 3]));
    }
    __syncthreads();
}

__device__ __forceinline__ int find_segment(const int32_t* __restrict__ off, int S, int cand) {
    // largest s with off[s] <= cand (empty segments have off[s] == off[s+1]; pick the one that contains cand)
    int lo = 0, hi = S;  // invariant: off[lo] <= cand < off[hi]
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (__ldg(off + mid) <= cand) lo = mid; else hi = mid;
    }
    return lo;
}

// Weights-in-shared-memory modes: one thread issues the bulk async copies (TMA engine) of every matrix and vector the
// residual-MLP step and the scorer read; `bar` (initialised, count 1) completes when all of them have landed.
__device__ __forceinline__ void stage_weights(const GenericParams& p, float* wreg, uint32_t bar) {
    ptx::mbar_arrive_expect_tx(bar, p.ws_bytes);
    ptx::bulk_g2s(ptx::smem_u32(wreg + p.ws_w1), p.W1t, (uint32_t)((size_t)(p.d + p.da) * p.hidden * 4), bar);
    ptx::bulk_g2s(ptx::smem_u32(wreg + p.ws_w2), p.W2t, (uint32_t)((size_t)p.hidden * p.d * 4), bar);
    for (int l = 0; l < p.n_lin; ++l) {
        ptx::bulk_g2s(ptx::smem_u32(wreg + p.ws_s[l]), p.Wst[l], (uint32_t)((size_t)p.sdim[l] * p.sdim[l + 1] * 4), bar);
        ptx::bulk_g2s(ptx::smem_u32(wreg + p.ws_bs[l]), p.bs[l], (uint32_t)(((size_t)p.sdim[l + 1] * 4 + 15) & ~15u), bar);
    }
    ptx::bulk_g2s(ptx::smem_u32(wreg + p.ws_E), p.E, (uint32_t)((size_t)p.n_types * p.da * 4), bar);
    ptx::bulk_g2s(ptx::smem_u32(wreg + p.ws_Wp), p.WpT, (uint32_t)((size_t)p.P * p.da * 4), bar);
    ptx::bulk_g2s(ptx::smem_u32(wreg + p.ws_bp), p.bp, (uint32_t)((size_t)p.da * 4), bar);
    ptx::bulk_g2s(ptx::smem_u32(wreg + p.ws_b1), p.b1, (uint32_t)((size_t)p.hidden * 4), bar);
    ptx::bulk_g2s(ptx::smem_u32(wreg + p.ws_b2), p.b2, (uint32_t)((size_t)p.d * 4), bar);
    if (p.kind == WM_KIND_MLP_LN) {
        ptx::bulk_g2s(ptx::smem_u32(wreg + p.ws_g), p.gamma, (uint32_t)((size_t)p.d * 4), bar);
        ptx::bulk_g2s(ptx::smem_u32(wreg + p.ws_be), p.beta, (uint32_t)((size_t)p.d * 4), bar);
    }
}

constexpr int kGenericThreads = 256;
static_assert(kSplitThreads == kGenericThreads, "linear_T_split spreads K over the whole CTA");

// WS = true (small residual-MLP models whose W1, W2 and scorer matrices fit shared memory beside the tile, e.g. BASELINE.json
// cfg 1: 135 KB): every CTA stages the matrices ONCE with bulk async copies (TMA engine, mbarrier complete_tx) and then
// walks its tiles — north_star's "transition weights are staged once per CTA through TMA into shared memory", which is
// literally possible only for models of this size.  WS = false re-reads them through the read-only path.
template <int R, bool WS>
__global__ void __launch_bounds__(kGenericThreads) wm_generic_kernel(const GenericParams p) {
    extern __shared__ __align__(16) float smem[];
    const int d = p.d, da = p.da, H = p.H, P = p.P;
    const int K1 = d + da;
    float* X = smem;                                   // [(d+xa_rows+H)][R]  rows: z | a (phi) | hw
    float* Hb = X + (size_t)(d + p.xa_rows + H) * R;   // [maxw][R]
    float* ALT = Hb + (size_t)p.maxw * R;              // [alt_rows][R]: V | AS | Y   (scorer: ping-pong buffer)
    float* V = ALT;                                    // [d][R]
    float* AS = V + (size_t)d * R;                     // [da][R] running sum of a (WM_PHI_MEAN), or the running
                                                       // statistics of WM_PHI_STRUCT: counts [n_types], then per
                                                       // parameter slot sum [P] and max [P] of log2 p
    float* Y = AS + (size_t)p.as_rows * R;             // [(d+da)][R], GRU and TransH only
    float* LP = ALT + (size_t)p.alt_rows * R;          // [R][P] log2(param) or bucket index (as int bits)
    float* RED = LP + (size_t)R * P;                   // [G][R] reduction scratch, G = threads / R
    int* meta = reinterpret_cast<int*>(RED + kGenericThreads);   // cand[R], len[R], seg[R], id[R], start[R], tile_len, tile_pre
    int* m_cand = meta;
    int* m_len = meta + R;
    int* m_seg = meta + 2 * R;
    int* m_id = meta + 3 * R;
    int* m_start = meta + 4 * R;       // prefix-latent reuse: steps [0, start) only feed phi
    int* m_tile_len = meta + 5 * R;    // rollout steps of the tile = max (len - start)
    int* m_tile_pre = meta + 5 * R + 1;   // max start of the tile

    const int tid = threadIdx.x;
    const int r_of = tid % R;
    const int g_of = tid / R;
    constexpr int G = kGenericThreads / R;
    const CallArgs& a = p.a;
    const float* W1t = p.W1t;
    const float* W2t = p.W2t;
    const float* Wst[kMaxScorerLinears];
    const float* bsv[kMaxScorerLinears];
#pragma unroll
    for (int l = 0; l < kMaxScorerLinears; ++l) { Wst[l] = p.Wst[l]; bsv[l] = p.bs[l]; }
    const float *pE = p.E, *pWp = p.WpT, *pbp = p.bp, *pb1 = p.b1, *pb2 = p.b2, *pg = p.gamma, *pbe = p.beta;
    if (WS) {
        float* wreg = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(smem) + p.ws_off);
        uint64_t* wbar = reinterpret_cast<uint64_t*>(reinterpret_cast<uint8_t*>(smem) + p.ws_off + p.ws_bytes);
        const uint32_t bar = ptx::smem_u32(wbar);
        if (tid == 0) {
            ptx::mbar_init(bar, 1);
            ptx::fence_barrier_init();
            stage_weights(p, wreg, bar);
        }
        __syncthreads();
        ptx::mbar_wait(bar, 0);
        W1t = wreg + p.ws_w1;
        W2t = wreg + p.ws_w2;
#pragma unroll
        for (int l = 0; l < kMaxScorerLinears; ++l) { Wst[l] = wreg + p.ws_s[l]; bsv[l] = wreg + p.ws_bs[l]; }
        pE = wreg + p.ws_E; pWp = wreg + p.ws_Wp; pbp = wreg + p.ws_bp; pb1 = wreg + p.ws_b1; pb2 = wreg + p.ws_b2;
        pg = wreg + p.ws_g; pbe = wreg + p.ws_be;
    }
    auto ldw = [&](const float* q) -> float { return WS ? *q : __ldg(q); };
    // split-K scratch: [256][R] floats behind the weight region's barrier (WS mode, R <= 8, every width <= 256)
    constexpr bool SPLIT = WS && R <= 8;
    float* scratch = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(smem) + p.ws_off + p.ws_bytes + 16);

    for (int tile = blockIdx.x; tile < p.n_tiles; tile += gridDim.x) {
        __syncthreads();
        if (tid == 0) *m_tile_len = *m_tile_pre = 0;
        __syncthreads();
        if (tid < R) {
            const int64_t i = (int64_t)tile * R + tid;
            int cand = -1, len = 0, seg = 0, st = 0;
            if (i < a.B) {
                cand = a.perm ? __ldg(a.perm + i) : (int)i;
                len = __ldg(a.lengths + cand);
                if (len < 0 || len > a.T_max) {
                    atomicOr(a.fault, WM_FAULT_LEN);
                    len = len < 0 ? 0 : a.T_max;
                }
                seg = a.offsets ? find_segment(a.offsets, a.S, cand) : cand;
                if (a.start) st = clamp_start(__ldg(a.start + cand), len);
            }
            m_cand[tid] = cand;
            m_len[tid] = len;
            m_seg[tid] = seg;
            m_start[tid] = st;
            atomicMax(m_tile_len, len - st);
            atomicMax(m_tile_pre, st);
        }
        __syncthreads();
        const int tile_len = *m_tile_len, tile_pre = *m_tile_pre;
        // z_0 (the subgraph's, the candidate's, or the row init_index names) and the running action sum
        for (int e = tid; e < d * R; e += kGenericThreads) {
            const int r = e % R, j = e / R;   // lanes over rows: conflict-free store; global read strided but tiny
            float v = 0.0f;
            if (m_cand[r] >= 0) {
                size_t zrow = (size_t)m_seg[r];
                if (a.init_index) {   // banked latent (wm_rollout_score_from); clamped, WM_FAULT_INDEX when outside
                    long long bi = __ldg(a.init_index + m_cand[r]);
                    if (bi < 0 || bi >= a.n_init) {
                        if (j == 0) atomicOr(a.fault, WM_FAULT_INDEX);
                        bi = bi < 0 ? 0 : a.n_init - 1;
                    }
                    zrow = (size_t)bi;
                }
                v = (a.cand_latents && m_len[r] > 0) ? __ldg(a.cand_latents + (size_t)m_cand[r] * d + j)
                                                     : __ldg(a.init_states + zrow * d + j);
            }
            X[(size_t)j * R + r] = v;
        }
        for (int e = tid; e < p.as_rows * R; e += kGenericThreads) AS[e] = 0.0f;
        __syncthreads();

        // Iterations tq < 0 walk the prefix positions [0, start) of every row: embedding and phi statistics only, no
        // transition (prefix-latent reuse: the latent at `start` was supplied).  Iterations tq >= 0 are rollout steps:
        // row r is at position start[r] + tq.
        for (int tq = -tile_pre; tq < tile_len; ++tq) {
            const bool prefix = tq < 0;
            const int t = tq;   // (name kept for the masks below: live rows have pos < len)
            auto pos_of = [&](int r) { return prefix ? tq + tile_pre : m_start[r] + tq; };
            auto live_of = [&](int r) { return prefix ? tq + tile_pre < m_start[r] : m_start[r] + tq < m_len[r]; };
            (void)t;
            // ---- a1: action embedding at this position (rows that are not live get a = 0 and touch no input)
            if (tid < R) {
                int id = 0;
                if (live_of(tid)) {
                    id = __ldg(a.action_ids + (size_t)m_cand[tid] * a.T_max + pos_of(tid));
                    if (id < 0 || id >= p.n_types) {
                        atomicOr(a.fault, WM_FAULT_TYPE);
                        id = id < 0 ? 0 : p.n_types - 1;
                    }
                }
                m_id[tid] = id;
                if (p.phi_kind != WM_PHI_MEAN && live_of(tid)) AS[(size_t)id * R + tid] += 1.0f;
            }
            for (int e = tid; e < R * P; e += kGenericThreads) {
                const int r = e / P, j = e % P;
                float v = 0.0f;
                if (live_of(r)) {
                    int prm = __ldg(a.action_params + ((size_t)m_cand[r] * a.T_max + pos_of(r)) * P + j);
                    if (prm < 1) {
                        atomicOr(a.fault, WM_FAULT_PARAM);
                        prm = 1;
                    }
                    if (p.phi_kind == WM_PHI_STRUCT) {   // (r, j) belongs to this thread alone
                        const float l2 = log2f((float)prm);
                        float* sum = AS + (size_t)(p.n_types + j) * R + r;
                        float* mx = AS + (size_t)(p.n_types + P + j) * R + r;
                        *sum += l2;
                        *mx = fmaxf(*mx, l2);
                    } else if (p.phi_kind == WM_PHI_TYPED) {   // per action type (S28); the id is re-read here: m_id is
                        int id = __ldg(a.action_ids + (size_t)m_cand[r] * a.T_max + pos_of(r));   // written by another thread
                        id = id < 0 ? 0 : (id >= p.n_types ? p.n_types - 1 : id);
                        const float l2 = log2f((float)prm);
                        float* sum = AS + (size_t)(p.n_types + id * P + j) * R + r;
                        float* mx = AS + (size_t)(p.n_types + p.n_types * P + id * P + j) * R + r;
                        *sum += l2;
                        *mx = fmaxf(*mx, l2);
                    }
                    if (p.embed == WM_EMBED_LINEAR) {
                        v = log2f((float)prm);
                    } else {
                        // bucket(p) = min(n_b-1, floor(4 log2 p)), exact for every int32 p (n_buckets goes up to 4096)
                        v = __int_as_float(min(quarter_octave_bucket(prm), p.n_buckets - 1));
                    }
                }
                LP[e] = v;
            }
            __syncthreads();
            for (int e = tid; e < da * R; e += kGenericThreads) {
                const int r = e % R, j = e / R;
                float v = 0.0f;
                if (live_of(r)) {
                    const int id = m_id[r];
                    if (p.embed == WM_EMBED_LINEAR) {
                        v = ldw(pE + (size_t)id * da + j) + ldw(pbp + j);
                        for (int q = 0; q < P; ++q) v = fmaf(ldw(pWp + (size_t)q * da + j), LP[r * P + q], v);
                    } else {
                        for (int q = 0; q < P; ++q) {
                            const int bk = __float_as_int(LP[r * P + q]);
                            v += __ldg(p.Tbl + ((size_t)(id * P + q) * p.n_buckets + bk) * da + j);
                        }
                    }
                    if (p.phi_kind == WM_PHI_MEAN) AS[e] += v;   // a4: running sum for phi
                }
                X[(size_t)(d + j) * R + r] = v;
            }
            __syncthreads();
            if (prefix) continue;
            const bool live_row = live_of(r_of);

            // ---- a2/a3: one transition step, rows that are not live frozen
            if (p.kind == WM_KIND_TRANSH) {
                // PAPER.md:164 (S24): u = W_w a, w = u / sqrt(|u|^2 + eps); x = z - (w.z) w + W_d a;
                // v = x + W2 gelu(W1 [x;a] + b1) + b2; z' = v / sqrt(|v|^2 + eps).  (w.z) w = (u.z) u / (|u|^2 + eps).
                constexpr float kEps = 1e-12f;
                const float* A_ = X + (size_t)d * R;
                linear_T<R, ACT_NONE>(p.Wwt, nullptr, A_, da, d, V);     // u
                linear_T<R, ACT_NONE>(p.Wdt, nullptr, A_, da, d, Y);     // translation W_d a
                __syncthreads();
                float s1 = 0.0f, s2 = 0.0f;
                for (int j = g_of; j < d; j += G) {
                    const float u = V[(size_t)j * R + r_of];
                    s1 = fmaf(u, u, s1);
                    s2 = fmaf(u, X[(size_t)j * R + r_of], s2);
                }
                RED[g_of * R + r_of] = s1;
                __syncthreads();
                float nw2 = 0.0f;
                for (int g = 0; g < G; ++g) nw2 += RED[g * R + r_of];
                __syncthreads();
                RED[g_of * R + r_of] = s2;
                __syncthreads();
                float dot = 0.0f;
                for (int g = 0; g < G; ++g) dot += RED[g * R + r_of];
                __syncthreads();
                const float c = dot / (nw2 + kEps);
                for (int j = g_of; j < d; j += G) {
                    const size_t o = (size_t)j * R + r_of;
                    Y[o] = X[o] - c * V[o] + Y[o];                        // x = z_perp + W_d a
                }
                for (int e = tid; e < da * R; e += kGenericThreads) Y[(size_t)d * R + e] = X[(size_t)d * R + e];
                __syncthreads();
                linear_T<R, ACT_GELU>(p.W1t, p.b1, Y, K1, p.hidden, Hb);
                __syncthreads();
                linear_T<R, ACT_NONE>(p.W2t, p.b2, Hb, p.hidden, d, V);
                __syncthreads();
                float q = 0.0f;
                for (int j = g_of; j < d; j += G) {
                    const size_t o = (size_t)j * R + r_of;
                    const float v = Y[o] + V[o];
                    V[o] = v;
                    q = fmaf(v, v, q);
                }
                RED[g_of * R + r_of] = q;
                __syncthreads();
                float n2 = 0.0f;
                for (int g = 0; g < G; ++g) n2 += RED[g * R + r_of];
                const float rn = 1.0f / sqrtf(n2 + kEps);
                if (live_row) {
                    for (int j = g_of; j < d; j += G) X[(size_t)j * R + r_of] = V[(size_t)j * R + r_of] * rn;
                }
            } else if (p.kind != WM_KIND_GRU) {
                if (SPLIT && p.split_ok) {
                    linear_T_split<R, ACT_GELU>(W1t, pb1, X, K1, p.hidden, Hb, scratch);
                    linear_T_split<R, ACT_NONE>(W2t, pb2, Hb, p.hidden, d, V, scratch);
                } else {
                    linear_T<R, ACT_GELU, WS>(W1t, pb1, X, K1, p.hidden, Hb);
                    __syncthreads();
                    linear_T<R, ACT_NONE, WS>(W2t, pb2, Hb, p.hidden, d, V);
                    __syncthreads();
                }
                if (p.kind == WM_KIND_MLP_LN) {
                    // v = z + V; two-pass LayerNorm over the d features of each row
                    float s = 0.0f;
                    for (int j = g_of; j < d; j += G) {
                        const float v = X[(size_t)j * R + r_of] + V[(size_t)j * R + r_of];
                        V[(size_t)j * R + r_of] = v;
                        s += v;
                    }
                    RED[g_of * R + r_of] = s;
                    __syncthreads();
                    float mean = 0.0f;
                    for (int g = 0; g < G; ++g) mean += RED[g * R + r_of];
                    mean /= (float)d;
                    __syncthreads();
                    float q = 0.0f;
                    for (int j = g_of; j < d; j += G) {
                        const float c = V[(size_t)j * R + r_of] - mean;
                        q = fmaf(c, c, q);
                    }
                    RED[g_of * R + r_of] = q;
                    __syncthreads();
                    float var = 0.0f;
                    for (int g = 0; g < G; ++g) var += RED[g * R + r_of];
                    var /= (float)d;
                    const float rstd = 1.0f / sqrtf(var + p.ln_eps);
                    if (live_row) {
                        for (int j = g_of; j < d; j += G) {
                            const float c = (V[(size_t)j * R + r_of] - mean) * rstd;
                            X[(size_t)j * R + r_of] = fmaf(ldw(pg + j), c, ldw(pbe + j));
                        }
                    }
                } else {
                    if (live_row) {
                        for (int j = g_of; j < d; j += G) X[(size_t)j * R + r_of] += V[(size_t)j * R + r_of];
                    }
                }
            } else {
                linear_T<R, ACT_SIGMOID>(p.Wgt, nullptr, X, K1, d, Hb);   // g
                linear_T<R, ACT_SIGMOID>(p.Wrt, nullptr, X, K1, d, V);    // r
                __syncthreads();
                for (int e = tid; e < K1 * R; e += kGenericThreads)
                    Y[e] = e < d * R ? V[e] * X[e] : X[e];                // [r*z ; a]
                __syncthreads();
                linear_T<R, ACT_TANH>(p.Wht, nullptr, Y, K1, d, V);       // candidate h
                __syncthreads();
                if (live_row) {
                    for (int j = g_of; j < d; j += G) {
                        const size_t o = (size_t)j * R + r_of;
                        const float g = Hb[o];
                        X[o] = (1.0f - g) * X[o] + g * V[o];
                    }
                }
            }
            __syncthreads();
            if (a.latents_out) {   // z after this step, rows that took it: latents_out[cand][pos][:]
                for (int e = tid; e < d * R; e += kGenericThreads) {
                    const int r = e / d, j = e % d;    // lanes over features: coalesced global store
                    if (!live_of(r)) continue;
                    if (!a.latents_terminal)
                        a.latents_out[((size_t)m_cand[r] * a.T_max + pos_of(r)) * d + j] = X[(size_t)j * R + r];
                    else if (pos_of(r) == m_len[r] - 1)     // [B, d]: the terminal latent only
                        a.latents_out[(size_t)m_cand[r] * d + j] = X[(size_t)j * R + r];
                }
            }
        }
        if (!a.scores_out) continue;   // wm_rollout_latents: no ranking

        // ---- a4/a5: x = [z_T ; phi ; hw], scorer MLP
        const int F = p.phi_dim, NT = p.n_types;
        for (int e = tid; e < F * R; e += kGenericThreads) {
            const int r = e % R, j = e / R;
            const int len = m_len[r];
            float v;
            if (p.phi_kind == WM_PHI_MEAN) {
                v = len > 0 ? AS[e] / (float)len : 0.0f;
            } else if (p.phi_kind == WM_PHI_TYPED && j > NT) {   // per type k: sums | means | maxima (S28)
                const int q = j - NT - 1, k = q / (3 * P), stat = (q / P) % 3, slot = q % P;
                const float cnt = AS[(size_t)k * R + r];
                const float sum = AS[(size_t)(NT + k * P + slot) * R + r];
                v = stat == 0 ? sum : stat == 1 ? (cnt > 0.0f ? sum / cnt : 0.0f) : AS[(size_t)(NT + NT * P + k * P + slot) * R + r];
            } else if (j < NT) {                       // counts (S25)
                v = AS[e];
            } else if (j == NT) {                      // length
                v = (float)len;
            } else if (j < NT + 1 + P) {               // sums of log2 p
                v = AS[(size_t)(j - 1) * R + r];
            } else if (j < NT + 1 + 2 * P) {           // means
                v = len > 0 ? AS[(size_t)(j - 1 - P) * R + r] / (float)len : 0.0f;
            } else {                                   // maxima (log2 p >= 0, so the running max starts at 0)
                v = AS[(size_t)(j - 1 - P) * R + r];
            }
            X[(size_t)d * R + e] = v;
        }
        for (int e = tid; e < H * R; e += kGenericThreads) {
            const int r = e % R, j = e / R;
            X[(size_t)(d + F) * R + e] = m_cand[r] >= 0 ? __ldg(a.hw_feats + (size_t)m_seg[r] * H + j) : 0.0f;
        }
        __syncthreads();
        const float* in = X;
        for (int l = 0; l < p.n_lin; ++l) {
            float* out = (l & 1) ? ALT : Hb;
            if (SPLIT && p.split_ok) {
                if (l + 1 < p.n_lin) linear_T_split<R, ACT_GELU>(Wst[l], bsv[l], in, p.sdim[l], p.sdim[l + 1], out, scratch);
                else linear_T_split<R, ACT_NONE>(Wst[l], bsv[l], in, p.sdim[l], p.sdim[l + 1], out, scratch);
            } else {
                if (l + 1 < p.n_lin)
                    linear_T<R, ACT_GELU, WS>(Wst[l], bsv[l], in, p.sdim[l], p.sdim[l + 1], out);
                else
                    linear_T<R, ACT_NONE, WS>(Wst[l], bsv[l], in, p.sdim[l], p.sdim[l + 1], out);
                __syncthreads();
            }
            in = out;
        }
        // ---- a6: scatter to the original order
        if (tid < R && m_cand[tid] >= 0) a.scores_out[m_cand[tid]] = in[tid];
    }
}

// ------------------------------------------------------------------------------------------------------------------
// K2-small: ONE CTA (four warps) PER CANDIDATE, for search-round-sized calls of a small residual-MLP model (BASELINE.json
// cfg 1: 64 candidates, T_max 8; PAPER.md:21 works with 64-trial budgets).  Such a call is bound by the LATENCY of its
// serial chain (T_max steps x two matrix-vector products), not by throughput: in wm_generic_kernel<4, true> a step costs
// about eight block barriers and ~8 K cycles on 16 of the 148 SMs.  Here every candidate gets an SM of its own: the
// weights are staged once per CTA by bulk async copies (as in the WS mode above); a matrix-vector product is split over
// the four warps by K (one warp per scheduler, each streams a quarter of the matrix from shared memory: a lone warp is
// bound by the latency of its own loads, measured 2.3 us per step for both products), a lane owns the output units
// [NPL lane, NPL lane + NPL) so that a weight row is one conflict-free vector load per lane, inputs are float4
// broadcasts; the four partial sums meet in shared memory.  Four 128-thread barriers per step.
constexpr int kSmallWarps = 4;
constexpr int kSmallMaxB = 592;     // four candidates per SM; beyond that the tiled kernel's reuse of a weight read over R rows wins
constexpr int kSmallMaxW = 256;     // widest layer: 8 output units per lane

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// part[n] = sum over k in [k0, k1) of Wt[k][n] in[k] for the N = 32 NPL output units; Wt ([K][N]), in, part in shared
// memory, 16-byte aligned; k0, k1 multiples of 4.  Two accumulator sets (even / odd k) halve the dependent-FMA chain.
template <int NPL>
__device__ __forceinline__ void warp_partial_n(const float* Wt, const float* in, int k0, int k1, float* part, int lane) {
    constexpr int N = 32 * NPL;
    float acc[2][NPL];
#pragma unroll
    for (int i = 0; i < NPL; ++i) acc[0][i] = acc[1][i] = 0.0f;
    const float* wl = Wt + NPL * lane;
#pragma unroll 2
    for (int k = k0; k < k1; k += 4) {
        const float4 x = *reinterpret_cast<const float4*>(in + k);
        const float xv[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            float w[NPL];
            const float* r = wl + (size_t)(k + u) * N;
            if (NPL == 1) {
                w[0] = r[0];
            } else if (NPL == 2) {
                const float2 t = *reinterpret_cast<const float2*>(r);
                w[0] = t.x; w[1] = t.y;
            } else {
#pragma unroll
                for (int q = 0; q < NPL / 4; ++q) {
                    const float4 t = *reinterpret_cast<const float4*>(r + 4 * q);
                    w[4 * q] = t.x; w[4 * q + 1] = t.y; w[4 * q + 2] = t.z; w[4 * q + 3] = t.w;
                }
            }
#pragma unroll
            for (int i = 0; i < NPL; ++i) acc[u & 1][i] = fmaf(w[i], xv[u], acc[u & 1][i]);
        }
    }
#pragma unroll
    for (int i = 0; i < NPL; ++i) part[NPL * lane + i] = acc[0][i] + acc[1][i];
}

// The CTA's product out = act(bias + Wt^T in) for N in {32, 64, 128, 256}: warp w takes the w-th quarter of K (in groups of
// four rows) into part[w][.]; after a barrier thread n (and n + 128) adds the four partial sums and the bias.  Called by all
// 128 threads; ends with a barrier (out is complete, part is free again).
template <int ACT>
__device__ __forceinline__ void cta_linear(const float* Wt, const float* bias, const float* in, int K, int N, float* out,
                                           float* part, int maxw, int warp, int lane) {
    const int groups = K >> 2, g0 = (groups * warp) / kSmallWarps, g1 = (groups * (warp + 1)) / kSmallWarps;
    float* mine = part + (size_t)warp * maxw;
    switch (N) {
        case 32: warp_partial_n<1>(Wt, in, 4 * g0, 4 * g1, mine, lane); break;
        case 64: warp_partial_n<2>(Wt, in, 4 * g0, 4 * g1, mine, lane); break;
        case 128: warp_partial_n<4>(Wt, in, 4 * g0, 4 * g1, mine, lane); break;
        default: warp_partial_n<8>(Wt, in, 4 * g0, 4 * g1, mine, lane); break;
    }
    __syncthreads();
    for (int n = threadIdx.x; n < N; n += kSmallWarps * 32)
        out[n] = apply_act<ACT>((part[n] + part[maxw + n]) + (part[2 * maxw + n] + part[3 * maxw + n]) + bias[n]);
    __syncthreads();
}

__global__ void __launch_bounds__(kSmallWarps * 32) wm_small_kernel(const GenericParams p) {
    extern __shared__ __align__(16) float smem[];
    const int d = p.d, da = p.da, H = p.H, P = p.P, K1 = d + da;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    // weight region first (ws_off = 0), its barrier, then xs [d | da | H] (4-float aligned), hb, yb [maxw], part [4][maxw]
    float* wreg = smem;
    uint64_t* wbar = reinterpret_cast<uint64_t*>(reinterpret_cast<uint8_t*>(smem) + p.ws_bytes);
    const int xs_len = (d + da + H + 3) & ~3;
    float* xs = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(smem) + p.ws_bytes + 16);
    float* hb = xs + xs_len;
    float* yb = hb + p.maxw;
    float* part = yb + p.maxw;
    const uint32_t bar = ptx::smem_u32(wbar);
    if (tid == 0) {
        ptx::mbar_init(bar, 1);
        ptx::fence_barrier_init();
        stage_weights(p, wreg, bar);
    }
    __syncthreads();
    const CallArgs& a = p.a;
    const float *W1t = wreg + p.ws_w1, *W2t = wreg + p.ws_w2, *pE = wreg + p.ws_E, *pWp = wreg + p.ws_Wp,
                *pbp = wreg + p.ws_bp, *pb1 = wreg + p.ws_b1, *pb2 = wreg + p.ws_b2, *pg = wreg + p.ws_g, *pbe = wreg + p.ws_be;
    const int dj = (d + 31) >> 5, aj = (da + 31) >> 5;
    bool staged = false;
    for (int64_t i = blockIdx.x; i < a.B; i += gridDim.x) {
        const int cand = a.perm ? __ldg(a.perm + i) : (int)i;
        int len = __ldg(a.lengths + cand);
        if (len < 0 || len > a.T_max) {
            if (tid == 0) atomicOr(a.fault, WM_FAULT_LEN);
            len = len < 0 ? 0 : a.T_max;
        }
        const int seg = a.offsets ? find_segment(a.offsets, a.S, cand) : cand;
        // z_0 and the hardware features (the loads fly while the weights land)
        for (int n = tid; n < d; n += kSmallWarps * 32) xs[n] = __ldg(a.init_states + (size_t)seg * d + n);
        for (int n = tid; n < H; n += kSmallWarps * 32) xs[K1 + n] = __ldg(a.hw_feats + (size_t)seg * H + n);
        float phi[8];      // warp 1: running sum of the embedding columns lane, lane + 32, ...
#pragma unroll
        for (int j = 0; j < 8; ++j) phi[j] = 0.0f;
        if (!staged) {
            ptx::mbar_wait(bar, 0);
            staged = true;
        }
        // warp 1 writes a_t = E[id] + W_p log2 p + b_p (a1) into xs[d ..): `fetch` issues the step's global loads (a product
        // earlier than `embed` needs them), `embed` runs beside warp 0's latent update
        int id_n = 0, prm_n = 1;
        auto fetch = [&](int t) {
            id_n = __ldg(a.action_ids + (size_t)cand * a.T_max + t);
            if (lane < P) prm_n = __ldg(a.action_params + ((size_t)cand * a.T_max + t) * P + lane);
        };
        auto embed = [&]() {
            int id = id_n;
            if (id < 0 || id >= p.n_types) {
                if (lane == 0) atomicOr(a.fault, WM_FAULT_TYPE);
                id = id < 0 ? 0 : p.n_types - 1;
            }
            float lp = 0.0f;
            if (lane < P) {
                int prm = prm_n;
                if (prm < 1) {
                    atomicOr(a.fault, WM_FAULT_PARAM);
                    prm = 1;
                }
                lp = log2f((float)prm);
            }
            float lq[8];       // log2 p_q of this step, q < P <= 8
#pragma unroll
            for (int q = 0; q < 8; ++q) lq[q] = __shfl_sync(0xffffffffu, lp, q);
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int n = lane + 32 * j;
                if (j < aj && n < da) {
                    float v = pE[(size_t)id * da + n] + pbp[n];
#pragma unroll
                    for (int q = 0; q < 8; ++q)
                        if (q < P) v = fmaf(pWp[(size_t)q * da + n], lq[q], v);
                    xs[d + n] = v;
                    phi[j] += v;     // a4: running sum for phi
                }
            }
        };
        if (warp == 1 && len > 0) {
            fetch(0);
            embed();
        }
        __syncthreads();
        for (int t = 0; t < len; ++t) {
            // ---- a2: z' = z + W2 gelu(W1 [z; a] + b1) + b2 (, LayerNorm)
            cta_linear<ACT_GELU>(W1t, pb1, xs, K1, p.hidden, hb, part, p.maxw, warp, lane);
            if (warp == 1 && t + 1 < len) fetch(t + 1);
            cta_linear<ACT_NONE>(W2t, pb2, hb, p.hidden, d, yb, part, p.maxw, warp, lane);
            if (warp == 1) {        // (the a-part of xs was last read by the first product of this step)
                if (t + 1 < len) embed();
            } else if (warp == 0) {
                float v[8];
                float s = 0.0f;
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int n = lane + 32 * j;
                    v[j] = (j < dj && n < d) ? xs[n] + yb[n] : 0.0f;
                    s += v[j];
                }
                if (p.kind == WM_KIND_MLP_LN) {     // two-pass LayerNorm, as in wm_generic_kernel
                    const float mean = warp_sum(s) / (float)d;
                    float q = 0.0f;
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        const int n = lane + 32 * j;
                        const float c = (j < dj && n < d) ? v[j] - mean : 0.0f;
                        q = fmaf(c, c, q);
                    }
                    const float rstd = 1.0f / sqrtf(warp_sum(q) / (float)d + p.ln_eps);
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        const int n = lane + 32 * j;
                        if (j < dj && n < d) xs[n] = fmaf(pg[n], (v[j] - mean) * rstd, pbe[n]);
                    }
                } else {
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        const int n = lane + 32 * j;
                        if (j < dj && n < d) xs[n] = v[j];
                    }
                }
            }
            __syncthreads();
        }
        // ---- a4/a5: x = [z_T ; phi ; hw], scorer MLP; a6: the score goes to the candidate's slot
        if (warp == 1) {
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int n = lane + 32 * j;
                if (j < aj && n < da) xs[d + n] = len > 0 ? phi[j] / (float)len : 0.0f;
            }
        }
        __syncthreads();
        const float* in = xs;
        for (int l = 0; l + 1 < p.n_lin; ++l) {
            float* out = (l & 1) ? yb : hb;
            cta_linear<ACT_GELU>(wreg + p.ws_s[l], wreg + p.ws_bs[l], in, p.sdim[l], p.sdim[l + 1], out, part, p.maxw, warp, lane);
            in = out;
        }
        if (warp == 0) {      // the output unit: lanes split K, then a warp reduction
            const int l = p.n_lin - 1;
            const float* Ws = wreg + p.ws_s[l];
            float acc = 0.0f;
            for (int k = lane; k < p.sdim[l]; k += 32) acc = fmaf(Ws[k], in[k], acc);
            acc = warp_sum(acc);
            if (lane == 0) a.scores_out[cand] = acc + wreg[p.ws_bs[l]];
        }
        __syncthreads();      // xs / hb / yb are rewritten by the next candidate
    }
    if (!staged) ptx::mbar_wait(bar, 0);     // (a CTA without a candidate may not leave before its copies have landed)
}

static int generic_as_rows(const Model& m) {
    const int typed = m.n_types + 2 * m.n_types * m.P;
    return m.phi_kind == WM_PHI_TYPED && typed > m.d_a ? typed : m.d_a;
}

static size_t generic_smem_bytes(const Model& m, int R, int* maxw_out, int* alt_rows_out) {
    int maxw = m.d > m.hidden ? m.d : m.hidden;
    int maxsw = 1;
    for (int l = 1; l <= m.n_lin; ++l) maxsw = m.sdim[l] > maxsw ? m.sdim[l] : maxsw;
    if (maxsw > maxw) maxw = maxsw;
    const int as_rows = generic_as_rows(m), xa_rows = m.phi_dim > m.d_a ? m.phi_dim : m.d_a;
    int alt = m.d + as_rows + (m.kind == WM_KIND_GRU || m.kind == WM_KIND_TRANSH ? m.d + m.d_a : 0);
    if (maxsw > alt) alt = maxsw;
    *maxw_out = maxw;
    *alt_rows_out = alt;
    size_t floats = (size_t)(m.d + xa_rows + m.H) * R + (size_t)maxw * R + (size_t)alt * R + (size_t)R * m.P +
                    kGenericThreads;
    return floats * 4 + (5 * R + 4) * sizeof(int);
}

template <int R, bool WS>
static int launch_R(wm_ctx* ctx, const GenericParams& p, size_t smem, int grid, cudaStream_t st) {
    // (the attribute call costs microseconds of host time per launch — the whole budget of a cfg-1-sized call: made only
    // when this instance needs more shared memory than it has been granted on this device)
    static std::atomic<int> granted[16];
    int dev = 0;
    cudaGetDevice(&dev);
    dev &= 15;
    if (granted[dev].load(std::memory_order_relaxed) < (int)smem) {
        WM_CUDA_TRY(cudaFuncSetAttribute(wm_generic_kernel<R, WS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        granted[dev].store((int)smem, std::memory_order_relaxed);
    }
    wm_generic_kernel<R, WS><<<grid, kGenericThreads, smem, st>>>(p);
    WM_CUDA_TRY(cudaGetLastError());
    ctx->launches.fetch_add(1);
    return WM_OK;
}

// Weights-in-shared-memory mode: residual-MLP models (no TransH / GRU matrices) with an MLP ranker whose W1t, W2t and
// scorer matrices fit beside the tile; every matrix a multiple of 16 bytes (bulk-copy granularity).  Fills the ws_*
// fields and returns the total dynamic shared memory, or 0 when the mode does not apply.
static size_t weights_in_smem(const wm_ctx* ctx, GenericParams* p, size_t tile_bytes) {
    const Model& m = ctx->m;
    if ((m.kind != WM_KIND_MLP && m.kind != WM_KIND_MLP_LN) || m.ranker_kind != WM_RANKER_MLP || m.n_lin < 1 ||
        m.embed != WM_EMBED_LINEAR)
        return 0;
    size_t off = 0;   // in floats
    auto take = [&](size_t n, uint32_t* at) -> bool {
        if ((n * 4) % 16 != 0) return false;
        *at = (uint32_t)off;
        off += n;
        return true;
    };
    if (!take((size_t)(m.d + m.d_a) * m.hidden, &p->ws_w1) || !take((size_t)m.hidden * m.d, &p->ws_w2)) return 0;
    for (int l = 0; l < m.n_lin; ++l) {
        if (!take((size_t)m.sdim[l] * m.sdim[l + 1], &p->ws_s[l])) return 0;
        p->ws_bs[l] = (uint32_t)off;            // (every device vector is allocated with 16 spare bytes: the copy is rounded up)
        off += ((size_t)m.sdim[l + 1] + 3) & ~(size_t)3;
    }
    if (!take((size_t)m.n_types * m.d_a, &p->ws_E) || !take((size_t)m.P * m.d_a, &p->ws_Wp) || !take(m.d_a, &p->ws_bp) ||
        !take(m.hidden, &p->ws_b1) || !take(m.d, &p->ws_b2))
        return 0;
    if (m.kind == WM_KIND_MLP_LN && (!take(m.d, &p->ws_g) || !take(m.d, &p->ws_be))) return 0;
    bool split_ok = m.hidden <= kGenericThreads && m.d <= kGenericThreads;
    for (int l = 1; l <= m.n_lin; ++l) split_ok &= m.sdim[l] <= kGenericThreads;
    p->split_ok = split_ok ? 1 : 0;
    const size_t base = (tile_bytes + 127) & ~(size_t)127;
    const size_t total = base + off * 4 + 16 + (size_t)kGenericThreads * 8 * 4;   // + barrier + split-K scratch (R <= 8)
    if (total > (size_t)ctx->smem_optin || off * 4 >= (1u << 20)) return 0;   // (mbarrier tx-count: < 2^20 bytes per phase)
    p->ws_off = (uint32_t)base;
    p->ws_bytes = (uint32_t)(off * 4);
    return total;
}

// K2-small takes the call when it is small and plain: a model of the weights-in-shared-memory class (checked by the
// caller), mean-embedding phi, every layer at most kSmallMaxW wide and a multiple of 4 (float4 broadcasts), no
// prefix-reuse arguments, at most kSmallMaxB candidates.
static size_t small_smem_bytes(const Model& m, const GenericParams& p) {
    const int xs_len = (m.d + m.d_a + m.H + 3) & ~3;
    return (size_t)p.ws_bytes + 16 + (size_t)(xs_len + (2 + kSmallWarps) * p.maxw) * 4;
}

static bool small_call_ok(const wm_ctx* ctx, const CallArgs& a, const GenericParams& p) {
    const Model& m = ctx->m;
    if (small_smem_bytes(m, p) > (size_t)ctx->smem_optin) return false;
    if (a.B > kSmallMaxB || !a.scores_out || a.start || a.init_index || a.latents_out || a.cand_latents) return false;
    if (m.phi_kind != WM_PHI_MEAN || m.P > 8) return false;
    auto w32 = [](int n) { return n == 32 || n == 64 || n == 128 || n == 256; };    // widths warp_linear_n is built for
    bool ok = w32(m.d) && w32(m.hidden) && m.d_a <= kSmallMaxW && (m.d + m.d_a) % 4 == 0 && p.maxw % 4 == 0 &&
              m.sdim[m.n_lin] == 1 && m.sdim[0] % 4 == 0 && m.sdim[0] <= 4 * kSmallMaxW;
    for (int l = 1; l < m.n_lin; ++l) ok &= w32(m.sdim[l]);
    return ok;
}

static int launch_small(wm_ctx* ctx, GenericParams p, cudaStream_t st) {
    const Model& m = ctx->m;
    p.ws_off = 0;
    const size_t smem = small_smem_bytes(m, p);
    static std::atomic<int> granted[16];
    int dev = 0;
    cudaGetDevice(&dev);
    dev &= 15;
    if (granted[dev].load(std::memory_order_relaxed) < (int)smem) {
        WM_CUDA_TRY(cudaFuncSetAttribute(wm_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        granted[dev].store((int)smem, std::memory_order_relaxed);
    }
    const int grid = (int)(p.a.B < ctx->n_sms ? p.a.B : ctx->n_sms);     // one candidate per CTA, one CTA per SM
    wm_small_kernel<<<grid, kSmallWarps * 32, smem, st>>>(p);
    WM_CUDA_TRY(cudaGetLastError());
    ctx->launches.fetch_add(1);
    return WM_OK;
}

static int pick_R(const wm_ctx* ctx, int64_t B, size_t* smem_out, int* maxw, int* alt) {
    // Largest tile that fits shared memory; small batches take smaller tiles so the (latency-bound) work
    // spreads over the SMs.
    const int cands[4] = {32, 16, 8, 4};
    int fallback = 0;
    for (int i = 0; i < 4; ++i) {
        const int R = cands[i];
        if (generic_smem_bytes(ctx->m, R, maxw, alt) > (size_t)ctx->smem_optin) continue;
        if (!fallback) fallback = R;
        if ((B + R - 1) / R >= ctx->n_sms || R == 4) {
            *smem_out = generic_smem_bytes(ctx->m, R, maxw, alt);
            return R;
        }
    }
    if (fallback) *smem_out = generic_smem_bytes(ctx->m, fallback, maxw, alt);
    return fallback;
}

int generic_supported(const wm_ctx* ctx) {
    size_t s;
    int a, b;
    return pick_R(ctx, 1 << 20, &s, &a, &b) != 0;
}

int launch_generic(wm_ctx* ctx, const CallArgs& a, cudaStream_t st) {
    const Model& m = ctx->m;
    GenericParams p;
    p.kind = m.kind; p.embed = m.embed; p.d = m.d; p.da = m.d_a; p.hidden = m.hidden; p.n_types = m.n_types;
    p.P = m.P; p.n_buckets = m.n_buckets; p.H = m.H; p.n_lin = m.n_lin;
    p.phi_kind = m.phi_kind; p.phi_dim = m.phi_dim;
    for (int i = 0; i <= kMaxScorerLinears; ++i) p.sdim[i] = m.sdim[i];
    p.ln_eps = m.ln_eps;
    p.E = m.E; p.WpT = m.WpT; p.bp = m.bp; p.Tbl = m.Tbl;
    p.W1t = m.W1t; p.b1 = m.b1; p.W2t = m.W2t; p.b2 = m.b2; p.gamma = m.gamma; p.beta = m.beta;
    p.Wwt = m.Wwt; p.Wdt = m.Wdt;
    p.Wgt = m.Wgt; p.Wrt = m.Wrt; p.Wht = m.Wht;
    for (int i = 0; i < kMaxScorerLinears; ++i) { p.Wst[i] = m.Wst[i]; p.bs[i] = m.bs[i]; }
    p.a = a;
    size_t smem = 0;
    p.as_rows = generic_as_rows(m);
    p.xa_rows = m.phi_dim > m.d_a ? m.phi_dim : m.d_a;
    const int R = pick_R(ctx, a.B, &smem, &p.maxw, &p.alt_rows);
    if (R == 0) {
        set_error("model too wide for the fp32 kernel's shared-memory tile");
        return WM_ERR_UNSUPPORTED;
    }
    p.n_tiles = (int)((a.B + R - 1) / R);
    if (p.n_tiles < 1) return WM_OK;
    p.ws_off = p.ws_bytes = p.ws_w1 = p.ws_w2 = 0;
    p.split_ok = 0;
    p.ws_E = p.ws_Wp = p.ws_bp = p.ws_b1 = p.ws_b2 = p.ws_g = p.ws_be = 0;
    for (int i = 0; i < kMaxScorerLinears; ++i) p.ws_s[i] = p.ws_bs[i] = 0;
    const size_t ws_total = weights_in_smem(ctx, &p, smem);
    if (ws_total && small_call_ok(ctx, a, p)) return launch_small(ctx, p, st);
    if (ws_total) {       // one CTA per SM (the weights take most of its shared memory), each walks its tiles
        const int grid = p.n_tiles < ctx->n_sms ? p.n_tiles : ctx->n_sms;
        switch (R) {
            case 32: return launch_R<32, true>(ctx, p, ws_total, grid, st);
            case 16: return launch_R<16, true>(ctx, p, ws_total, grid, st);
            case 8: return launch_R<8, true>(ctx, p, ws_total, grid, st);
            default: return launch_R<4, true>(ctx, p, ws_total, grid, st);
        }
    }
    const int grid = p.n_tiles < ctx->n_sms * 4 ? p.n_tiles : ctx->n_sms * 4;
    switch (R) {
        case 32: return launch_R<32, false>(ctx, p, smem, grid, st);
        case 16: return launch_R<16, false>(ctx, p, smem, grid, st);
        case 8: return launch_R<8, false>(ctx, p, smem, grid, st);
        default: return launch_R<4, false>(ctx, p, smem, grid, st);
    }
}

}  // namespace wm

// K5 (tcgen05, CTA pair, M = 256): the ranking MLP alone, for models whose phi is too wide to be built inside the rollout
// kernels — the per-action-type statistics of WM_PHI_TYPED (S28: n_types (1 + 3P) + 1 = 609 features at cfg 2's
// shapes; "action-specific numeric attributes"), sm_100a only.
//
// PAPER.md:122 Eq.3 / :188 Eq.12 — y = G([z_T ; phi ; h]) with G = Linear -> GELU -> Linear -> GELU -> Linear(-> 1).
// wm_rollout_score of such a model is three launches after K1: wm_tcp_kernel<., EXT> rolls the candidates and stores the
// terminal latents; wm_typed_x_kernel (below) writes the scorer input X = [z_T | phi | 1 | 0.. | h | 0..] as fp16 rows
// (phi in a fixed order per row: the steps of one action type are summed in step order by one lane, no atomics); this kernel is the scorer of
// wm_tcp_kernel with the A operand streamed from X instead of being written by the epilogue / action warps.
//
// A cluster of two CTAs owns a tile of 256 consecutive candidates (128 rows each).  Layer 1 runs as two passes of two
// 128-column chunks (both GEMM1-style accumulators, tensor-memory columns [256, 512)): a ring stage is ONE K-block of A
// (this CTA's 128 rows of X, 16 KB, a TMA tensor load with 128-byte swizzle = the SW128 K-major operand layout) plus the two
// chunks' weight boxes (2 x 8 KB), 8 MMAs per wait / commit; X is therefore streamed twice.  The GELU epilogue writes the
// fp16 hidden activations H1 into tensor-memory columns [0, 256), layer 2 reads them as a TMEM A operand (TS form) and the
// 512 -> 1 output layer is a dot product in the layer-2 epilogue — all as in wm_tcp_kernel.  bs0 rides on X's constant-1
// column.  Static tile schedule (tile = it * pairs + pair), no length bucketing: a row's cost does not depend on its length.
#include <cuda.h>
#include <cuda_fp16.h>

#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "wm_internal.h"
#include "wm_ptx.cuh"
#include "wm_tmap.h"

namespace wm {

namespace tsc {

using namespace ptx;

constexpr int TMP = 256;           // candidates per pair tile (MMA M)
constexpr int TM = 128;            // rows per CTA
constexpr int D = 256;             // latent width
constexpr int SW = 512;            // scorer hidden width (both hidden layers)
constexpr int KB_BYTES = 16384;    // one A K-block: [128 rows x 64 cols] fp16, SW128 K-major
constexpr int HB_BYTES = 8192;     // one weight box: this CTA's 64 weight rows of an N = 128 K-block
constexpr int STAGE_BYTES = KB_BYTES + 2 * HB_BYTES;    // layer 1: A K-block + two chunks' boxes; layer 2: four boxes
constexpr int NSTAGE = 6;
constexpr int THREADS = 352;       // warps 0-7 epilogue, 8 TMEM allocator, 9 TMA producer, 10 MMA issuer
constexpr int ALLOC_WARP = 8, PROD_WARP = 9, MMA_WARP = 10;
constexpr int MAX_KB = 24;         // K-blocks of X

enum {
    B_FULL = 0,                    // [NSTAGE] TMA (both CTAs) -> leader's MMA warp
    B_EMPTY = B_FULL + NSTAGE,     // [NSTAGE] MMA commit (multicast) -> each CTA's producer
    B_D1FULL = B_EMPTY + NSTAGE,   // [2] MMA commit -> epilogue: accumulator buffer b filled
    B_HREADY = B_D1FULL + 2,       // [2] epilogue (both CTAs) -> leader MMA: buffer b read (and its output written)
    B_COUNT = B_HREADY + 2
};

struct Params {
    int nkb;                       // K-blocks of X (64 columns each)
    const float *bs1, *w3, *bs2;
    float* scores_out;
    int64_t B;
    int n_tiles;
};

constexpr uint32_t idesc_m256(uint32_t n) { return (1u << 4) | ((n >> 3) << 17) | ((256u >> 4) << 24); }
constexpr uint32_t ID_N128 = idesc_m256(128);

// pair MMA with the A operand in tensor memory (each CTA's own 128 lanes)
__device__ __forceinline__ void mma_ts2(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d_tmem),
        "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(acc)
        : "memory");
}

constexpr uint32_t SMEM_RING = 0, SMEM_BARS = NSTAGE * STAGE_BYTES, SMEM_SLOT = SMEM_BARS + B_COUNT * 8 + 8,
                   SMEM_RED = SMEM_SLOT + 16, SMEM_TOTAL = SMEM_RED + TM * 4;

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(THREADS, 1)
wm_tsc_kernel(const Params p, const __grid_constant__ CUtensorMap tmap_x, const __grid_constant__ CUtensorMap tmap_w) {
    extern __shared__ __align__(1024) uint8_t smem[];
    const uint32_t s_base = smem_u32(smem);
    const uint32_t s_ring = s_base + SMEM_RING, s_bars = s_base + SMEM_BARS;
    auto bar = [&](int i) -> uint32_t { return s_bars + 8u * (uint32_t)i; };
    float* s_red = reinterpret_cast<float*>(smem + SMEM_RED);          // [128] layer-2 partial dot products (column half 1)
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();          // 0 = leader (issues the MMAs)
    const int pair = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;
    const int NKB = p.nkb;

    if (threadIdx.x == 0) {
        for (int i = 0; i < NSTAGE; ++i) { mbar_init(bar(B_FULL + i), 1); mbar_init(bar(B_EMPTY + i), 1); }
        for (int i = 0; i < 2; ++i) { mbar_init(bar(B_D1FULL + i), 1); mbar_init(bar(B_HREADY + i), 16); }
        fence_barrier_init();
        fence_proxy_async();
    }
    if (warp == ALLOC_WARP) tmem_alloc2(s_base + SMEM_SLOT, 512);
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();      // both CTAs' barriers are initialised before anyone arrives remotely / multicasts
    tc_fence_after();
    const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(smem + SMEM_SLOT);
    const uint32_t T_H = tmem_base;                 // H1 (fp16) as the A operand of layer 2: columns [0, 256)
    const uint32_t T_D1 = tmem_base + 256;          // two 128-column accumulators

    if (warp == PROD_WARP) {
        // =============================================================== TMA producer
        if (lane == 0) {
            uint32_t stage = 0, ph = 0;
            auto next = [&]() { if (++stage == NSTAGE) { stage = 0; ph ^= 1; } };
            for (int tile = pair; tile < p.n_tiles; tile += n_pairs) {
                // layer 1: per pass and K-block, this CTA's 128 rows of X and the two chunks' weight boxes.  The leader's
                // barrier collects both CTAs' bytes; a box of X that reaches past the last row is zero-filled
                for (int ps = 0; ps < 2; ++ps)
                    for (int kb = 0; kb < NKB; ++kb) {
                        mbar_wait(bar(B_EMPTY + stage), ph ^ 1);
                        if (rank == 0) mbar_arrive_expect_tx(bar(B_FULL + stage), 2u * STAGE_BYTES);
                        const uint32_t dst = s_ring + stage * STAGE_BYTES;
                        tma_load_2sm(dst, &tmap_x, 64 * kb, tile * TMP + TM * (int)rank, bar(B_FULL + stage));
                        const int box = 2 * (ps * NKB + kb);
                        tma_load_2sm(dst + KB_BYTES, &tmap_w, 0, 64 * (2 * box + (int)rank), bar(B_FULL + stage));
                        tma_load_2sm(dst + KB_BYTES + HB_BYTES, &tmap_w, 0, 64 * (2 * (box + 1) + (int)rank), bar(B_FULL + stage));
                        next();
                    }
                // layer 2: per chunk two stages of four K-blocks' boxes
                for (int s2 = 0; s2 < 8; ++s2) {
                    mbar_wait(bar(B_EMPTY + stage), ph ^ 1);
                    if (rank == 0) mbar_arrive_expect_tx(bar(B_FULL + stage), 2u * STAGE_BYTES);
                    const int box = 4 * NKB + 4 * s2;
                    for (int q = 0; q < 4; ++q)
                        tma_load_2sm(s_ring + stage * STAGE_BYTES + q * HB_BYTES, &tmap_w, 0, 64 * (2 * (box + q) + (int)rank),
                                     bar(B_FULL + stage));
                    next();
                }
            }
        }
        __syncwarp();
    } else if (warp == MMA_WARP) {
        // =============================================================== MMA issuer (leader CTA only)
        if (rank == 0) {
            uint32_t stage = 0, ph = 0, n_h[2] = {0, 0};
            bool pend[2] = {false, false};
            auto wait_h = [&](int b) {
                if (pend[b]) {
                    mbar_wait(bar(B_HREADY + b), n_h[b] & 1);
                    ++n_h[b];
                    pend[b] = false;
                    tc_fence_after();
                }
            };
            auto acquire = [&]() {
                mbar_wait(bar(B_FULL + stage), ph);
                tc_fence_after();
            };
            auto advance = [&]() {
                __syncwarp();
                if (++stage == NSTAGE) { stage = 0; ph ^= 1; }
            };
            auto commit = [&](int barrier) {
                if (elect_one()) mma_commit2(bar(barrier));
                __syncwarp();
            };
            for (int tile = pair; tile < p.n_tiles; tile += n_pairs) {
                // ---- layer 1: two passes of two 128-column chunks of gelu(Ws0 x + bs0)
#pragma unroll 1
                for (int ps = 0; ps < 2; ++ps) {
                    wait_h(0);
                    wait_h(1);
#pragma unroll 1
                    for (int kb = 0; kb < NKB; ++kb) {
                        acquire();
                        if (elect_one()) {
                            const uint32_t a_lo = smem_desc_lo(s_ring + stage * STAGE_BYTES);
                            const uint32_t w_lo = a_lo + (KB_BYTES >> 4);
#pragma unroll
                            for (int c = 0; c < 2; ++c)
#pragma unroll
                                for (int j = 0; j < 4; ++j)
                                    mma_ss2(T_D1 + 128u * c, desc_of(a_lo + 2u * j), desc_of(w_lo + c * (HB_BYTES >> 4) + 2u * j), ID_N128,
                                            (kb == 0 && j == 0) ? 0u : 1u);
                            mma_commit2(bar(B_EMPTY + stage));
                        }
                        advance();
                    }
                    commit(B_D1FULL + 0);
                    commit(B_D1FULL + 1);
                    pend[0] = pend[1] = true;
                }
                wait_h(0);
                wait_h(1);   // all of H1 (fp16, TMEM columns [0, 256)) written
                // ---- layer 2: A = H1 from TMEM, K = 512
#pragma unroll 1
                for (int c = 0; c < 4; ++c) {
                    const int b = c & 1;
                    wait_h(b);
#pragma unroll 1
                    for (int kb = 0; kb < 8; kb += 4) {
                        acquire();
                        if (elect_one()) {
                            const uint32_t w_lo = smem_desc_lo(s_ring + stage * STAGE_BYTES);
#pragma unroll
                            for (int q = 0; q < 4; ++q)
#pragma unroll
                                for (int j = 0; j < 4; ++j)
                                    mma_ts2(T_D1 + 128u * b, T_H + 32u * (kb + q) + 8u * j, desc_of(w_lo + q * (HB_BYTES >> 4) + 2u * j),
                                            ID_N128, (kb == 0 && q == 0 && j == 0) ? 0u : 1u);
                            mma_commit2(bar(B_EMPTY + stage));
                        }
                        advance();
                    }
                    commit(B_D1FULL + b);
                    pend[b] = true;
                }
            }
        }
        __syncwarp();
    } else if (warp < ALLOC_WARP) {
        // =============================================================== epilogue warps (GELU / output dot product)
        const int q = warp & 3, hh = warp >> 2;
        const int row = 32 * q + lane;
        const uint32_t lane_off = (uint32_t)(32 * q) << 16;
        const uint32_t r_hready0 = mapa(bar(B_HREADY), 0), r_hready1 = mapa(bar(B_HREADY + 1), 0);
        uint32_t n_d1[2] = {0, 0};
        // GELU over this thread's 64 columns of accumulator buffer b (the bias is in the accumulator: it rides on X's
        // constant-1 column), fp16 result to TMEM at dst_col
        auto gelu_chunk = [&](int b, uint32_t dst_col) {
            mbar_wait(bar(B_D1FULL + b), n_d1[b] & 1);
            ++n_d1[b];
            tc_fence_after();
            uint32_t v0[32], v1[32], o[16];
            tmem_ld32(T_D1 + 128u * b + lane_off + 64u * hh, v0);
            tmem_ld32(T_D1 + 128u * b + lane_off + 64u * hh + 32u, v1);
            tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 16; ++i) o[i] = gelu2_h2(__uint_as_float(v0[2 * i]), __uint_as_float(v0[2 * i + 1]));
            tmem_st16(dst_col + lane_off, o);
#pragma unroll
            for (int i = 0; i < 16; ++i) o[i] = gelu2_h2(__uint_as_float(v1[2 * i]), __uint_as_float(v1[2 * i + 1]));
            tmem_st16(dst_col + lane_off + 16u, o);
            tmem_st_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_remote(b == 0 ? r_hready0 : r_hready1);
        };
        for (int tile = pair; tile < p.n_tiles; tile += n_pairs) {
            const int64_t cand = (int64_t)tile * TMP + TM * (int)rank + row;
            // ---- layer 1 -> H1 (fp16) in TMEM columns [0, 256): chunk c at [64 c, 64 c + 64)
            for (int c = 0; c < 4; ++c) gelu_chunk(c & 1, T_H + 64u * c + 32u * hh);
            // ---- layer 2 + output dot product
            float part = 0.0f;
            for (int c = 0; c < 4; ++c) {
                const int b = c & 1;
                mbar_wait(bar(B_D1FULL + b), n_d1[b] & 1);
                ++n_d1[b];
                tc_fence_after();
#pragma unroll
                for (int p2 = 0; p2 < 2; ++p2) {
                    uint32_t v[32];
                    tmem_ld32(T_D1 + 128u * b + lane_off + 64u * hh + 32u * p2, v);
                    tmem_ld_wait();
                    const int n0 = c * 128 + 64 * hh + 32 * p2;
#pragma unroll
                    for (int i = 0; i < 32; ++i)
                        part = fmaf(gelu_fast(__uint_as_float(v[i]) + __ldg(p.bs1 + n0 + i)), __ldg(p.w3 + n0 + i), part);
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_remote(b == 0 ? r_hready0 : r_hready1);
            }
            if (hh == 1) s_red[row] = part;
            named_bar_sync(1 + q, 64);
            if (hh == 0 && cand < p.B) p.scores_out[cand] = part + s_red[row] + __ldg(p.bs2);
            named_bar_sync(1 + q, 64);   // s_red is rewritten by the next tile
        }
    }

    // ---- teardown: no CTA of the pair may exit (or free TMEM) while the other's MMAs / arrivals can still reach it
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    if (warp == ALLOC_WARP) tmem_dealloc2(tmem_base, 512);
}

// X row of a candidate: [z_T (256) | phi (n_types (1 + 3P) + 1) | 1 | 0.. to a K-block | h (H) | 0.. to a K-block], fp16.
// One warp per candidate.  phi (S28) = [c_k | len | per type k: s_kj | m_kj | x_kj]; the steps of one type are summed in step
// order by one lane (see the loop), so every sum has ONE order whatever the launch.  z_T is the terminal latent K2 stored (the task's z_0 for an empty sequence).
struct XParams {
    const float* zT;            // [B, d] terminal latents of the candidates that rolled at least one step
    const float* init_states;   // [S, d] ([B, d] without offsets); the bank [n_init, d] of a prefix-reuse call
    const int32_t *ids, *params, *lengths, *offsets;
    const int32_t *start, *init_index;   // prefix-reuse call (else null): first rolled position, bank row
    int64_t n_init;
    const float* hw;
    __half* X;                  // [B, 64 nkb]
    int64_t B;
    int S, T_max, n_types, P, H, nkb, phi_dim;
    uint32_t* fault;
};

constexpr int kXWarps = 8;
constexpr int kXTypes = 64, kXAcc = 17;     // most action types; accumulator floats per type (odd: conflict-free)

__global__ void __launch_bounds__(kXWarps * 32) wm_typed_x_kernel(const XParams p) {
    __shared__ float s_acc[kXWarps * kXTypes * kXAcc];          // per warp and action type: count, sum[8], max[8]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int NT = p.n_types, P = p.P, ld = 64 * p.nkb;
    for (int64_t c = (int64_t)blockIdx.x * kXWarps + warp; c < p.B; c += (int64_t)gridDim.x * kXWarps) {
        int len = __ldg(p.lengths + c);
        len = len < 0 ? 0 : (len > p.T_max ? p.T_max : len);           // (K2 has reported the fault)
        int seg = (int)c;
        if (p.offsets) {      // largest s with off[s] <= c
            int lo = 0, hi = p.S;
            while (hi - lo > 1) {
                const int mid = (lo + hi) >> 1;
                if (__ldg(p.offsets + mid) <= (int)c) lo = mid; else hi = mid;
            }
            seg = lo;
        }
        __half* x = p.X + (size_t)c * ld;
        // z_T: the stored terminal latent, or — when no step was rolled (empty sequence; start = len) — the latent the rollout
        // would have started from
        const bool rolled = len > 0 && (!p.start || clamp_start(__ldg(p.start + c), len) < len);
        size_t zrow = (size_t)seg;
        if (p.init_index) {
            long long bi = __ldg(p.init_index + c);      // (K2 has reported an index outside the bank)
            zrow = (size_t)(bi < 0 ? 0 : (bi >= p.n_init ? p.n_init - 1 : bi));
        }
        const float* z = rolled ? p.zT + (size_t)c * D : p.init_states + zrow * D;
        for (int j = 2 * lane; j < D; j += 64) {
            const float2 v = __ldg(reinterpret_cast<const float2*>(z + j));
            *reinterpret_cast<uint32_t*>(x + j) = pack_f16(v.x, v.y);
        }
        // everything behind z_T starts as zero (padding columns must not hold NaNs: their weights are zero, 0 * NaN is not)
        for (int j = D + 8 * lane; j < ld; j += 256) *reinterpret_cast<uint4*>(x + j) = make_uint4(0u, 0u, 0u, 0u);   // (rows are 16-byte aligned)
        __syncwarp();
        __half* phi = x + D;
        // Steps in chunks of 32, one step per lane: the lane turns its step's parameters into log2 p; the lanes of one action
        // type find each other (match.any), the group's first lane collects the others' values in step order (one shuffle
        // per slot and round, as many rounds as the most frequent type has steps) and adds the chunk's partial to the
        // type's accumulators in shared memory.  One order per sum, whatever the launch; a type that does not occur keeps
        // the zeros the row was filled with.
        float* acc = s_acc + warp * (kXTypes * kXAcc);
        for (int e = lane; e < NT * kXAcc; e += 32) acc[e] = 0.0f;
        __syncwarp();
        for (int t0 = 0; t0 < len; t0 += 32) {
            const int nt = min(32, len - t0);
            const bool valid = lane < nt;
            int id = -1 - lane;            // lanes without a step: groups of their own, ignored
            float l2[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) l2[j] = 0.0f;
            if (valid) {
                id = __ldg(p.ids + (size_t)c * p.T_max + t0 + lane);
                id = id < 0 ? 0 : (id >= NT ? NT - 1 : id);
                const int32_t* pp = p.params + ((size_t)c * p.T_max + t0 + lane) * P;
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    if (j < P) {      // MUFU.LG2 (2 ulp in fp32): the features are stored as fp16, 11 bits
                        const int prm = __ldg(pp + j);
                        l2[j] = __log2f((float)(prm < 1 ? 1 : prm));
                    }
            }
            const uint32_t mask = __match_any_sync(0xffffffffu, id);
            const int leader = __ffs(mask) - 1, cnt = __popc(mask);
            const int rounds = __reduce_max_sync(0xffffffffu, valid ? cnt : 1);
            float sum[8], mx[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) sum[j] = mx[j] = l2[j];       // the group's first step is the leader's own
            for (int r = 1; r < rounds; ++r) {
                const uint32_t src = __fns(mask, 0, r + 1);           // lane of the group's r-th later step (none: > 31)
                const bool take = lane == leader && src < 32u;
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    if (j < P) {
                        const float v = __shfl_sync(0xffffffffu, l2[j], (int)(src & 31u));
                        if (take) {
                            sum[j] += v;
                            mx[j] = fmaxf(mx[j], v);                  // (log2 p >= 0)
                        }
                    }
            }
            if (valid && lane == leader) {
                float* a = acc + id * kXAcc;
                a[0] += (float)cnt;
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    if (j < P) {
                        a[1 + j] += sum[j];
                        a[9 + j] = fmaxf(a[9 + j], mx[j]);
                    }
            }
            __syncwarp();
        }
        for (int k = lane; k < NT; k += 32) {
            const float* a = acc + k * kXAcc;
            const float cntf = a[0];
            if (cntf > 0.0f) {
                phi[k] = __float2half_rn(cntf);
                const float inv = 1.0f / cntf;
                __half* q = phi + NT + 1 + k * 3 * P;
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    if (j < P) {
                        q[j] = __float2half_rn(a[1 + j]);
                        q[P + j] = __float2half_rn(a[1 + j] * inv);
                        q[2 * P + j] = __float2half_rn(a[9 + j]);
                    }
            }
        }
        __syncwarp();      // acc is cleared for the warp's next candidate
        if (lane == 0) {
            phi[NT] = __float2half_rn((float)len);
            phi[p.phi_dim] = __float2half_rn(1.0f);        // the constant column that carries bs0
        }
        __half* hwx = x + ld - 64;
        for (int j = lane; j < p.H; j += 32) hwx[j] = __float2half_rn(__ldg(p.hw + (size_t)seg * p.H + j));
    }
}

}  // namespace tsc

// ------------------------------------------------------------------------------------------------ host side
namespace {

// Append one box slot (as in wm_tcp.cu): for each CTA (rank 0, then rank 1) 64 image rows of 128 B = the SW128 K-major image
// of W[row0 + 64 r + n][k0 + k], n < 64, k < 64.  Returns false when a weight is not finite in fp16.
bool append_box(std::vector<uint16_t>& blob, const std::vector<float>& W, int ld, int row0, int k0) {
    const size_t base = blob.size();
    blob.resize(base + 2 * tsc::HB_BYTES / 2, 0);
    bool ok = true;
    for (int r = 0; r < 2; ++r)
        for (int n = 0; n < 64; ++n)
            for (int k = 0; k < 64; ++k) {
                const float v = W[(size_t)(row0 + 64 * r + n) * ld + k0 + k];
                const size_t off = (size_t)r * tsc::HB_BYTES + (size_t)n * 128 + (size_t)((((k >> 3) ^ (n & 7)) << 4)) +
                                   (size_t)(k & 7) * 2;
                uint16_t hb;
                ok &= f32_to_f16_bits(v, &hb);
                blob[base + off / 2] = hb;
            }
    return ok;
}

}  // namespace

int tsc_prepare(wm_ctx* ctx, const std::vector<std::vector<float>>& hv, const std::vector<std::string>& names) {
    Model& m = ctx->m;
    m.tsc_ok = 0;
    if (m.phi_kind != WM_PHI_TYPED || m.ranker_kind != WM_RANKER_MLP || !m.tcp_ok || m.d != tsc::D || m.n_lin != 3 ||
        m.sdim[1] != tsc::SW || m.sdim[2] != tsc::SW || m.sdim[3] != 1 || m.H < 1 || m.H > 64 || m.P > 8 || m.n_types > tsc::kXTypes ||
        (int)tsc::SMEM_TOTAL > ctx->smem_optin)
        return WM_OK;
    const int F = m.phi_dim, PKB = (F + 1 + 63) / 64, NKB = 4 + PKB + 1, KX = 64 * NKB, K0 = tsc::D + F + m.H;
    if (NKB > tsc::MAX_KB) return WM_OK;
    auto get = [&](const char* n) -> const std::vector<float>& {
        for (size_t i = 0; i < names.size(); ++i)
            if (names[i] == n) return hv[i];
        static const std::vector<float> empty;
        return empty;
    };
    const std::vector<float>&Ws0 = get("Ws0"), &bs0 = get("bs0"), &Ws1 = get("Ws1");
    // layer 1 over X's columns: [z_T | phi | 1 (bs0) | 0.. | h | 0..]
    std::vector<float> Wx((size_t)tsc::SW * KX, 0.0f);
    for (int n = 0; n < tsc::SW; ++n) {
        const float* wr = &Ws0[(size_t)n * K0];
        float* o = &Wx[(size_t)n * KX];
        for (int k = 0; k < tsc::D + F; ++k) o[k] = wr[k];
        o[tsc::D + F] = bs0[n];
        for (int k = 0; k < m.H; ++k) o[KX - 64 + k] = wr[tsc::D + F + k];
    }
    std::vector<uint16_t> blob;
    bool ok = true;
    for (int ps = 0; ps < 2; ++ps)            // the kernel's order: per pass and K-block, chunks 2 ps and 2 ps + 1
        for (int kb = 0; kb < NKB; ++kb)
            for (int c = 0; c < 2; ++c) ok &= append_box(blob, Wx, KX, (2 * ps + c) * 128, kb * 64);
    for (int c = 0; c < 4; ++c)               // layer 2: per chunk the eight K-blocks of H1
        for (int kb = 0; kb < 8; ++kb) ok &= append_box(blob, Ws1, tsc::SW, c * 128, kb * 64);
    if (!ok) return WM_OK;   // a weight beyond the fp16 range: the fp32 kernel ranks this model
    void* d_blob = nullptr;
    WM_CUDA_TRY(cudaMalloc(&d_blob, blob.size() * 2));
    ctx->allocs.push_back(d_blob);
    WM_CUDA_TRY(cudaMemcpy(d_blob, blob.data(), blob.size() * 2, cudaMemcpyHostToDevice));
    // the image seen as rows of 64 16-bit values (128 B); one box = 64 rows; already swizzled: the map uses no swizzle
    static_assert(sizeof(CUtensorMap) <= sizeof(m.tsc_tmap), "tensor map storage");
    CUtensorMap tm;
    {
        const int rc = encode_tmap_2d(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, d_blob, 64, blob.size() * 2 / 128, 128, 64, 64, false, "tsc_prepare");
        if (rc != WM_OK) return rc;
    }
    memcpy(m.tsc_tmap, &tm, sizeof(tm));
    WM_CUDA_TRY(cudaFuncSetAttribute(tsc::wm_tsc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tsc::SMEM_TOTAL));
    m.tsc_blob = d_blob;
    m.tsc_nkb = NKB;
    m.tsc_ok = 1;
    return WM_OK;
}

size_t tsc_x_bytes(const wm_ctx* ctx, int64_t B) { return (size_t)B * 64 * ctx->m.tsc_nkb * sizeof(__half); }

int launch_tsc(wm_ctx* ctx, const float* zT, void* X, const CallArgs& a, float* scores_out, cudaStream_t st) {
    const Model& m = ctx->m;
    const int NKB = m.tsc_nkb;
    tsc::XParams xp;
    xp.zT = zT; xp.init_states = a.init_states; xp.ids = a.action_ids; xp.params = a.action_params; xp.lengths = a.lengths;
    xp.offsets = a.offsets; xp.hw = a.hw_feats; xp.X = static_cast<__half*>(X);
    xp.start = a.start; xp.init_index = a.init_index; xp.n_init = a.n_init;
    xp.B = a.B; xp.S = a.S; xp.T_max = a.T_max; xp.n_types = m.n_types; xp.P = m.P; xp.H = m.H; xp.nkb = NKB;
    xp.phi_dim = m.phi_dim; xp.fault = a.fault;
    const int64_t xb = (a.B + tsc::kXWarps - 1) / tsc::kXWarps;
    const int xgrid = (int)(xb < (int64_t)ctx->n_sms * 8 ? xb : (int64_t)ctx->n_sms * 8);
    tsc::wm_typed_x_kernel<<<xgrid, tsc::kXWarps * 32, 0, st>>>(xp);
    WM_CUDA_TRY(cudaGetLastError());
    // tensor map over X: rows of 64 nkb fp16, one box = this CTA's 128 rows of one K-block, 128-byte swizzle = the SW128
    // K-major operand layout; rows past B read as zero
    CUtensorMap tx, tw;
    {
        const int rc = encode_tmap_2d(&tx, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, X, (uint64_t)(64 * NKB), (uint64_t)a.B,
                                      (uint64_t)(64 * NKB) * sizeof(__half), 64, (uint32_t)tsc::TM, true, "launch_tsc");
        if (rc != WM_OK) return rc;
    }
    memcpy(&tw, m.tsc_tmap, sizeof(tw));
    tsc::Params p;
    p.nkb = NKB; p.bs1 = m.bs[1]; p.w3 = m.Wst[2]; p.bs2 = m.bs[2]; p.scores_out = scores_out; p.B = a.B;
    p.n_tiles = (int)((a.B + tsc::TMP - 1) / tsc::TMP);
    const int max_pairs = ctx->n_sms / 2;
    const int pairs = p.n_tiles < max_pairs ? p.n_tiles : max_pairs;
    tsc::wm_tsc_kernel<<<2 * pairs, tsc::THREADS, tsc::SMEM_TOTAL, st>>>(p, tx, tw);
    WM_CUDA_TRY(cudaGetLastError());
    ctx->launches.fetch_add(2);
    return WM_OK;
}

}  // namespace wm

// K2 (tcgen05, CTA pair, M = 256): fused persistent rollout + score kernel for the bf16 residual-MLP + LayerNorm
// models with d = 256, d_a = 128 (BASELINE.json cfg 2 and cfg 4) — the pair form of wm_tc_kernel, sm_100a only.
//
// PAPER.md:162 Eq.8 / :166 — z_t = F(z_{t-1}, a_t) applied recurrently; :176 — masked steps leave z unchanged;
// :186-188 Eq.12 — y = G([z_T ; phi ; h]).  Parametrisation: BASELINE.json cfg 2/4.
//
// Why a pair: wm_tc_kernel is bound by its single MMA-issuing warp (one ring stage of bookkeeping per 512
// tensor cycles) and, next, by the L2 -> SM weight stream.  A cluster of two CTAs (one TPC) owns a tile of 256
// length-sorted candidates, 128 rows per CTA, and the leader CTA issues `tcgen05.mma.cta_group::2` with M = 256:
//   * per CTA nothing changes in TMEM (fp32 latent = GEMM2 accumulator in columns [0,256), two 128-column GEMM1
//     accumulators whose fp16 GELU output is written back over them and read by GEMM2 as a TMEM A operand) nor in the A
//     operand ([z ; a] fp16, six 16 KB K-blocks in shared memory): each CTA supplies ITS 128 rows;
//   * each CTA supplies HALF of every B (weight) tile, so the L2 -> SM weight stream per SM halves, and one issued MMA
//     drives both SMs' tensor pipes: the issuer executes half the instructions, waits and commits per FLOP;
//   * a ring stage is two 16 KB TMA boxes per CTA = 1024 tensor cycles of work for the pair (8 or 16 MMAs per wait / commit);
//     the weight image is laid out in consumption order, one box per CTA side by side, and read through a tensor map
//     (`cp.async.bulk.tensor ... cta_group::2`: both halves' complete_tx land on the leader's barrier);
//   * MMA completion is multicast to both CTAs' barriers; epilogue / action warps of both CTAs arrive on the leader's
//     barriers (cluster-scope release).
// What else differs from wm_tc_kernel (measured: the CUDA-core side, not the tensor pipe or its issuer, bounded both forms —
// ~32 K warp instructions per CTA and step against 41 K issue slots in the step's 10.2 K tensor cycles):
//   * the action embedding is never formed: a_t = E[id] + W_p log2 p + b_p is linear in the features
//     f_t = [onehot(id) | log2 p_j | 1], so the host folds E, W_p, b_p AND b1 into GEMM1's a-columns
//     (W1a E^T, W1a W_p, W1a b_p + b1; summed in double, then the fp16 operand rounding every weight gets) and the action
//     warps only write f_t: one K-block of 64 feature columns instead of two K-blocks of embedding, a handful of 16-bit
//     stores per row and step instead of 128 FMAs;
//   * the GELU epilogue therefore needs no bias and runs on the packed fp16x2 pipe (gelu2_h2);
//   * scorer layer 1's bias rides on a constant-1 column of the phi features the same way.
// Warp roles per CTA (512 threads) as in wm_tc_kernel: warps 0-7 epilogue (one thread per row and column half), warps
// 8-11 action embedding, warp 12 TMEM allocator, warp 13 tile schedule + TMA producer, warp 15 MMA issuer (leader only).
#include <cuda.h>
#include <cuda_bf16.h>

#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "wm_internal.h"
#include "wm_ptx.cuh"
#include "wm_tmap.h"
#include "wm_trace.cuh"

namespace wm {

namespace tcp {

using namespace ptx;

constexpr int TMP = 256;           // candidates per pair tile (MMA M)
constexpr int TM = 128;            // rows per CTA
constexpr int D = 256;             // latent width
constexpr int DA = 128;            // action-embedding width
constexpr int SW = 512;            // scorer hidden width (both hidden layers)
constexpr int KB_BYTES = 16384;    // one A K-block: [128 rows x 64 cols] fp16, SW128 K-major
constexpr int HB_BYTES = 8192;     // one TMA box ("half block"): 64 image rows of 128 B = this CTA's half of one N = 128
                                   // K-block (64 weight rows x 64 cols; 4 MMAs, 256 tensor cycles) or a quarter of one
                                   // N = 256 K-block (two consecutive boxes = this CTA's 128 weight rows)
constexpr int NSTAGE = 3;
// Two shared-memory shapes.  "wide" (akb = pkb = 1: the action and phi features fit one K-block each, e.g. cfg 2 / 4): A1 is
// five K-blocks and a ring stage holds up to FIVE boxes (40 KB), so a later chunk's feature K-block and its four z K-blocks
// are ONE stage (one wait, one commit, one elected region: the issuer's fixed cost per stage is ~350 cycles).  Otherwise A1
// is six K-blocks, a stage holds four boxes and features and z are two stages.
__host__ __device__ inline int a1_kb(bool wide) { return wide ? 5 : 6; }      // z: 0-3, features f_t / phi: 4(-5)
__host__ __device__ inline int stage_hb(bool wide) { return wide ? 5 : 4; }
constexpr int HWK_BYTES = 4096;    // hw operand: one [128 x 16] no-swizzle K-major tile per K = 16 step
constexpr int THREADS = 512;
constexpr int EPI_WARP0 = 0, ACT_WARP0 = 8, ALLOC_WARP = 12, PROD_WARP = 13, MMA_WARP = 15;
constexpr int MAX_TYPES = 64, MAX_P = 8, MAX_H = 64, MAX_HID = 1024;

enum {
    B_FULL = 0,                    // [NSTAGE] TMA (both CTAs) -> leader's MMA warp
    B_EMPTY = B_FULL + NSTAGE,     // [NSTAGE] MMA commit (multicast) -> each CTA's producer
    B_D1FULL = B_EMPTY + NSTAGE,   // [2] MMA commit -> epilogue: accumulator buffer b filled
    B_HREADY = B_D1FULL + 2,       // [2] epilogue (both CTAs) -> leader MMA: buffer b read, fp16 hidden written to TMEM
    B_D2FULL = B_HREADY + 2,       // MMA commit -> epilogue: GEMM2 of the step done
    B_ZREADY,                      // epilogue (both CTAs) -> leader MMA: z K-blocks 0 and 2 written (first half of every thread's columns)
    B_ZREADY2,                     // ... K-blocks 1 and 3 written, and the fp32 latent in TMEM
    B_UFULL,                       // TransH step: MMA commit -> epilogue: u = W_w a of the next step is in the GEMM1 accumulators
    B_AFREE,                       // MMA commit -> action warps: a-part of A1 no longer read
    B_AREADY,                      // action warps (both CTAs) -> leader MMA: a-part written
    B_SFULL,                       // [2] schedule slot filled (CTA-local)
    B_SEMPTY = B_SFULL + 2,        // [2] schedule slot consumed (CTA-local)
    B_COUNT = B_SEMPTY + 2
};

struct Params {
    int hid, nc, n_types, P, H, hw_ksteps;
    int akb, pkb;               // K-blocks of the action features f_t (1 or 2) and of the phi features (1 or 2)
    float ln_eps;
    const float *b2, *gamma, *beta;
    const float *bs1, *w3, *bs2;
    CallArgs a;
    int n_tiles;
    unsigned long long* prof;   // developer trace buffer (wm_trace.cuh), null in a normal build
};

struct SmemLayout {
    uint32_t a1, hwk, ring, mx, cnt, b2, gamma, beta, red, bars, sched, tmem_slot, total;
};

__host__ __device__ inline SmemLayout smem_layout(int n_types, int hw_ksteps, int phi_struct, bool wide) {
    SmemLayout L;
    uint32_t o = 0;
    L.a1 = o; o += a1_kb(wide) * KB_BYTES;
    o = (o + 1023) & ~1023u;
    L.ring = o; o += NSTAGE * stage_hb(wide) * HB_BYTES;
    L.hwk = o; o += (uint32_t)hw_ksteps * HWK_BYTES;
    L.mx = o; o += phi_struct ? TM * MAX_P * 4 : 0;
    L.cnt = o; o += TM * (uint32_t)n_types;           // u8 counts, row-major [128][n_types]
    o = (o + 15) & ~15u;
    L.b2 = o; o += D * 4;
    L.gamma = o; o += D * 4;
    L.beta = o; o += D * 4;
    L.red = o; o += 4 * TM * 16;                       // [2 (parity)][2 column halves][128 rows] float4 (LayerNorm uses .x, .y)
    L.bars = o; o += B_COUNT * 8;
    L.sched = o; o += 2 * 8;
    L.tmem_slot = o; o += 16;
    L.total = o;
    return L;
}

// Static tile schedule (as wm_tc2_kernel): pair `pair` of `np` takes tile it*np + pair on even rounds and
// it*np + (np-1-pair) on odd rounds; tiles are sorted longest first, the serpentine evens out the step totals.
__device__ __forceinline__ int tile_of(int it, int pair, int np, int n_tiles) {
    const int idx = it * np + ((it & 1) ? np - 1 - pair : pair);
    return idx < n_tiles ? idx : -1;
}

// Ring-stage program of one rollout step, per CTA, in boxes: stage 0 = feature K-blocks of chunks 0 and 1 (2 akb boxes),
// stages 1, 2 = z K-blocks of chunk 0 / chunk 1 (4 boxes each), stage 3 = GEMM2 chunk 0 (4), then per further chunk i:
// feature K-blocks (akb), z K-blocks (4), GEMM2 chunk i-1 (4); last stage = GEMM2 chunk NC-1.  3 NC - 1 stages.
// (wide: 2 NC + 1 stages — features and z of chunk i are one stage of 5 boxes)
__host__ __device__ inline int step_stages(int nc, bool wide) { return wide ? 2 * nc + 1 : 3 * nc - 1; }
__host__ __device__ inline int stage_boxes(int j, int nc, int akb, bool wide) {
    if (j == 0) return 2 * akb;
    if (wide) return (j >= 4 && j < 2 * nc && (j - 4) % 2 == 0) ? 5 : 4;
    return (j >= 4 && j < 3 * nc - 2 && (j - 4) % 3 == 0) ? akb : 4;
}
__host__ __device__ inline int step_boxes(int nc, int akb) { return 2 * akb + 12 + (nc - 2) * (akb + 8) + 4; }
// TransH step (STEP_TRANSH): three feature stages first — u = W_w a (N = 256: 2 akb boxes), the translation W_d a onto the
// latent (2 akb), the feature K-blocks of chunks 0 and 1 (2 akb) — then z K-blocks of chunk 0, of chunk 1 (4 each), GEMM2
// chunk 0 and the rest as above.
__host__ __device__ inline int th_step_stages(int nc, bool wide) { return step_stages(nc, wide) + 2; }
__host__ __device__ inline int th_stage_boxes(int j, int nc, int akb, bool wide) {
    return j < 3 ? 2 * akb : stage_boxes(j - 2, nc, akb, wide);
}
__host__ __device__ inline int th_step_boxes(int nc, int akb) { return step_boxes(nc, akb) + 4 * akb; }
// scorer: layer 1, per 128-column chunk: [phi features (pkb) + hw (1)], [z (4)]; layer 2, per chunk: two stages of 4
__host__ __device__ inline int scorer_boxes(int pkb) { return 4 * (pkb + 1 + 4) + 4 * 8; }

constexpr uint32_t idesc_m256(uint32_t n) { return (1u << 4) | ((n >> 3) << 17) | ((256u >> 4) << 24); }
constexpr uint32_t ID_N128 = idesc_m256(128), ID_N256 = idesc_m256(256);

// pair MMA with the A operand in tensor memory (each CTA's own 128 lanes)
__device__ __forceinline__ void mma_ts2(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d_tmem),
        "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(acc)
        : "memory");
}

// PHI / EXT as in wm_tc_kernel: PHI = WM_PHI_MEAN | WM_PHI_STRUCT (what the action warps write into the phi K-blocks);
// EXT = the prefix-latent-reuse calls (per-candidate start and initial-latent row, latents stored), compiled out of
// the literal path.
// STEP = STEP_MLP_LN: z' = LayerNorm(z + W2 gelu(W1 [z; a] + b1) + b2) (BASELINE.json cfg 2 / 4).
// STEP = STEP_TRANSH (NEXT row f1, S24): u = W_w a; z_perp = z - (u.z) u / (|u|^2 + eps);
//   x = z_perp + W_d a; v = x + W2 gelu(W1 [x; a] + b1) + b2; z' = v / sqrt(|v|^2 + eps).  On this skeleton: u = W_w a is one
//   more N = 256 GEMM on the feature K-block into the (then free) GEMM1 accumulators; ONE boundary epilogue per step
//   normalises the previous step's v (held in registers) and projects it for the next action; the translation W_d a (with b2
//   on the constant feature column) is accumulated onto the latent by the tensor core, and GEMM1 consumes z_perp with
//   W1a' = W1a + W1z W_d folded on the host, so x is never formed by a thread.
constexpr int STEP_MLP_LN = 0, STEP_TRANSH = 1;
template <int PHI, bool EXT, int STEP>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(THREADS, 1)
wm_tcp_kernel(const Params p, const __grid_constant__ CUtensorMap tmap) {
    constexpr bool TH = STEP == STEP_TRANSH;
    extern __shared__ __align__(1024) uint8_t smem[];
    const bool WIDE = p.akb == 1 && p.pkb == 1;
    const SmemLayout L = smem_layout(p.n_types, p.hw_ksteps, PHI, WIDE);
    const uint32_t STAGE_BYTES = (uint32_t)stage_hb(WIDE) * HB_BYTES;
    const uint32_t s_base = smem_u32(smem);
    const uint32_t s_a1 = s_base + L.a1, s_ring = s_base + L.ring, s_bars = s_base + L.bars;
    auto bar = [&](int i) -> uint32_t { return s_bars + 8u * (uint32_t)i; };
    volatile int* s_sched = reinterpret_cast<volatile int*>(smem + L.sched);   // [2][2]: tile, nsteps
    float* s_b2 = reinterpret_cast<float*>(smem + L.b2);
    float* s_gamma = reinterpret_cast<float*>(smem + L.gamma);
    float* s_beta = reinterpret_cast<float*>(smem + L.beta);
    float4* s_red = reinterpret_cast<float4*>(smem + L.red);                  // [2][2][128]

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();          // 0 = leader (issues the MMAs)
    const int pair = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;
    const int NC = p.nc;
    const int AKB = p.akb, PKB = p.pkb;
    const int ROLL_BOXES = TH ? th_step_boxes(NC, AKB) : step_boxes(NC, AKB);
    const int ROLL_STAGES = TH ? th_step_stages(NC, WIDE) : step_stages(NC, WIDE);

    // ---- one-time setup
    if (threadIdx.x == 0) {
        for (int i = 0; i < NSTAGE; ++i) { mbar_init(bar(B_FULL + i), 1); mbar_init(bar(B_EMPTY + i), 1); }
        for (int i = 0; i < 2; ++i) {
            mbar_init(bar(B_D1FULL + i), 1);
            mbar_init(bar(B_HREADY + i), 16);
            mbar_init(bar(B_SFULL + i), 1);
            mbar_init(bar(B_SEMPTY + i), 13);
        }
        mbar_init(bar(B_D2FULL), 1);
        mbar_init(bar(B_ZREADY), 16);
        mbar_init(bar(B_ZREADY2), 16);
        mbar_init(bar(B_UFULL), 1);
        mbar_init(bar(B_AFREE), 1);
        mbar_init(bar(B_AREADY), 8);
        fence_barrier_init();
        fence_proxy_async();
    }
    if (warp == ALLOC_WARP) tmem_alloc2(s_base + L.tmem_slot, 512);
    for (int i = threadIdx.x; i < D; i += THREADS) {
        s_b2[i] = __ldg(p.b2 + i);
        s_gamma[i] = TH ? 1.0f : __ldg(p.gamma + i);
        s_beta[i] = TH ? 0.0f : __ldg(p.beta + i) + __ldg(p.b2 + i);   // the latent is carried as u = z + b2 (see the epilogue)
    }
    {
        // the hw K-block is only ever written in its first columns: clear it once so unread bytes are not NaNs
        uint32_t* hwk = reinterpret_cast<uint32_t*>(smem + L.hwk);
        for (int i = threadIdx.x; i < p.hw_ksteps * HWK_BYTES / 4; i += THREADS) hwk[i] = 0u;
    }
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();      // both CTAs' barriers are initialised before anyone arrives remotely / multicasts
    tc_fence_after();
    const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(smem + L.tmem_slot);
    // EXT calls that store latents and rank nothing skip the scorer in every role
    const bool rank_it = !EXT || p.a.scores_out != nullptr;
    const uint32_t T_Z = tmem_base;                 // fp32 latent / GEMM2 accumulator, 256 columns
    const uint32_t T_D1 = tmem_base + 256;          // two 128-column GEMM1 accumulators

    // Register hand-over between warpgroups (the kernel is launched with 128 per thread): the two epilogue warpgroups
    // take 176 each — the LayerNorm holds a row's 128 fp32 columns in registers: ONE pass over tensor memory instead of
    // two — the service warpgroup (allocator, producer, MMA issuer) keeps 96, the action-feature warpgroup 64.
    // (each warpgroup executes ONE setmaxnreg instruction, at the head of its own branch: ptxas budgets the code below it)
    if (warp >= ALLOC_WARP) {
    reg_dealloc<96>();
    if (warp == PROD_WARP) {
        // =============================================================== tile schedule + TMA producer
        uint32_t stage = 0, ph = 0;
        WM_TRACE_DECL(p.prof, 1)
        for (uint32_t it = 0;; ++it) {
            const uint32_t slot = it & 1;
            int tile = tile_of((int)it, pair, n_pairs, p.n_tiles);
            int nsteps = 0;
            if (tile >= 0) {
                for (int r = lane; r < TMP; r += 32) {
                    int cand, len, seg;
                    row_meta(p.a, (int64_t)tile * TMP + r, cand, len, seg, rank == 0);
                    nsteps = max(nsteps, EXT ? len - row_start(p.a, cand, len) : len);
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) nsteps = max(nsteps, __shfl_xor_sync(0xffffffffu, nsteps, o));
            }
            if (lane == 0) {
                mbar_wait(bar(B_SEMPTY + slot), ((it >> 1) & 1) ^ 1);
                s_sched[slot * 2 + 0] = tile;
                s_sched[slot * 2 + 1] = nsteps;
                mbar_arrive(bar(B_SFULL + slot));   // release semantics order the two stores before it
            }
            if (tile < 0) break;
            if (lane == 0) {
                // image row of box `b` of this CTA: boxes of the two CTAs alternate, 64 rows each
                auto issue = [&](int nbox, int box0) {
                    WM_TRACE(60);
                    mbar_wait(bar(B_EMPTY + stage), ph ^ 1);
                    WM_TRACE(61);
                    // the leader's barrier collects both CTAs' boxes of the stage
                    if (rank == 0) mbar_arrive_expect_tx(bar(B_FULL + stage), 2u * (uint32_t)nbox * HB_BYTES);
                    for (int b = 0; b < nbox; ++b)
                        tma_load_2sm(s_ring + stage * STAGE_BYTES + b * HB_BYTES, &tmap, 0,
                                     64 * (2 * (box0 + b) + (int)rank), bar(B_FULL + stage));
                    if (++stage == NSTAGE) { stage = 0; ph ^= 1; }
                };
                for (int t = 0; t < nsteps; ++t) {
                    int box = 0;
                    for (int j = 0; j < ROLL_STAGES; ++j) {
                        const int nb = TH ? th_stage_boxes(j, NC, AKB, WIDE) : stage_boxes(j, NC, AKB, WIDE);
                        issue(nb, box);
                        box += nb;
                    }
                }
                if (rank_it) {
                    int box = ROLL_BOXES;
                    for (int c = 0; c < 4; ++c) {
                        issue(PKB + 1, box); box += PKB + 1;
                        issue(4, box); box += 4;
                    }
                    for (int j = 0; j < 8; ++j) { issue(4, box); box += 4; }
                }
            }
            __syncwarp();
        }
    } else if (warp == MMA_WARP) {
        // =============================================================== MMA issuer (leader CTA; the peer's warp only
        // follows the schedule so that both CTAs' slot barriers have the same arrival count)
        const uint32_t TZ = __reduce_max_sync(0xffffffffu, tmem_base);   // provably warp-uniform (uniform registers)
        const uint32_t TD1 = TZ + 256;
        uint32_t stage = 0, ph = 0;
        uint32_t n_z = 0, n_a = 0, n_h[2] = {0, 0};
        bool pend[2] = {false, false};
        const uint32_t s_hwk = s_base + L.hwk;
        WM_TRACE_DECL(p.prof, 0)
        auto wait_h = [&](int b) {
            if (pend[b]) {
                WM_TRACE(10 + b);
                mbar_wait_warp(bar(B_HREADY + b), n_h[b] & 1);
                WM_TRACE(12 + b);
                ++n_h[b];
                pend[b] = false;
                tc_fence_after();
            }
        };
        const uint32_t ring_lo0 = smem_desc_lo(s_ring);
        uint32_t b_lo = ring_lo0;
        auto acquire_stage = [&]() {       // returns with the current stage's data landed
            WM_TRACE(20);
            mbar_wait_warp(bar(B_FULL + stage), ph);
            WM_TRACE(21);
            tc_fence_after();
        };
        auto advance = [&]() {
            __syncwarp();
            WM_TRACE(22);
            b_lo += STAGE_BYTES >> 4;
            if (++stage == NSTAGE) { stage = 0; ph ^= 1; b_lo = ring_lo0; }
        };
        // one box (this CTA's 64-row half of an N = 128 K-block) against the A K-block at a_kb: 4 MMAs of K = 16
        auto kb_ss = [&](uint32_t d, uint32_t a_kb, uint32_t blo, bool first) {
#pragma unroll
            for (int j = 0; j < 4; ++j) mma_ss2(d, desc_of(a_kb + 2u * j), desc_of(blo + 2u * j), ID_N128, (first && j == 0) ? 0u : 1u);
        };
        const uint32_t a_lo = smem_desc_lo(s_a1);
        constexpr uint32_t KBL = KB_BYTES >> 4, HBL = HB_BYTES >> 4;
        auto commit = [&](int barrier) {
            if (elect_one()) mma_commit2(bar(barrier));
            __syncwarp();
        };
        // stage: feature K-blocks (4 ..) of chunk buffers 0 AND 1
        auto stage_a01 = [&]() {
            acquire_stage();
            if (elect_one()) {
                for (int c = 0; c < 2; ++c)
                    for (int k = 0; k < AKB; ++k)
                        kb_ss(TD1 + 128u * c, a_lo + (4 + k) * KBL, b_lo + (uint32_t)(c * AKB + k) * HBL, k == 0);
                mma_commit2(bar(B_EMPTY + stage));
            }
            advance();
        };
        // stage: feature / phi K-blocks (4 ..) into buffer b, nk of them; with_hw: followed by the hw tile
        auto stage_a = [&](int b, int nk, bool with_hw) {
            acquire_stage();
            if (elect_one()) {
                for (int k = 0; k < nk; ++k) kb_ss(TD1 + 128u * b, a_lo + (4 + k) * KBL, b_lo + (uint32_t)k * HBL, k == 0);
                if (with_hw)
                    for (int j = 0; j < p.hw_ksteps; ++j)
                        mma_ss2(TD1 + 128u * b, smem_desc_nosw(s_hwk + j * HWK_BYTES), desc_of(b_lo + (uint32_t)nk * HBL + 2u * j),
                                ID_N128, 1u);
                mma_commit2(bar(B_EMPTY + stage));
            }
            advance();
        };
        // wide shape, one stage: the feature K-block then z K-blocks 0-3 into buffer b; the a-buffer is released (B_AFREE)
        // from inside the stage when this is the step's last read of it
        auto stage_az = [&](int b, bool last) {
            acquire_stage();
            if (elect_one()) {
                kb_ss(TD1 + 128u * b, a_lo + 4 * KBL, b_lo, true);
                if (last) mma_commit2(bar(B_AFREE));
#pragma unroll
                for (int k = 0; k < 4; ++k) kb_ss(TD1 + 128u * b, a_lo + k * KBL, b_lo + (uint32_t)(k + 1) * HBL, false);
                mma_commit2(bar(B_EMPTY + stage));
            }
            advance();
        };
        // stage: z K-blocks 0-3 into buffer b
        auto stage_z = [&](int b) {
            acquire_stage();
            if (elect_one()) {
#pragma unroll
                for (int k = 0; k < 4; ++k) kb_ss(TD1 + 128u * b, a_lo + k * KBL, b_lo + (uint32_t)k * HBL, false);
                mma_commit2(bar(B_EMPTY + stage));
            }
            advance();
        };
        // step boundary, stage 1: z K-blocks 0 and 2 (published first by the LayerNorm) of chunk buffers 0 and 1
        auto stage_za = [&]() {
            acquire_stage();
            if (elect_one()) {
                kb_ss(TD1, a_lo, b_lo, false);
                kb_ss(TD1, a_lo + 2 * KBL, b_lo + HBL, false);
                kb_ss(TD1 + 128u, a_lo, b_lo + 2 * HBL, false);
                kb_ss(TD1 + 128u, a_lo + 2 * KBL, b_lo + 3 * HBL, false);
                mma_commit2(bar(B_EMPTY + stage));
            }
            advance();
        };
        // step boundary, stage 2: z K-blocks 1 and 3 of chunk buffer 0 (accumulator 0 complete: published from inside the
        // stage), then of chunk buffer 1
        auto stage_zb = [&]() {
            acquire_stage();
            if (elect_one()) {
                kb_ss(TD1, a_lo + KBL, b_lo, false);
                kb_ss(TD1, a_lo + 3 * KBL, b_lo + HBL, false);
                mma_commit2(bar(B_D1FULL + 0));
                kb_ss(TD1 + 128u, a_lo + KBL, b_lo + 2 * HBL, false);
                kb_ss(TD1 + 128u, a_lo + 3 * KBL, b_lo + 3 * HBL, false);
                mma_commit2(bar(B_EMPTY + stage));
                mma_commit2(bar(B_D1FULL + 1));
            }
            advance();
        };
        // TransH: one stage of N = 256 MMAs of the feature K-blocks (4 ..) against a [256 x 64 akb] weight tile (two boxes per
        // K-block = this CTA's 128 weight rows) into the 256-column tile d: u = W_w' f (d = both GEMM1 accumulators, fresh) or
        // the translation W_d' f accumulated onto the latent
        auto stage_f256 = [&](uint32_t d, bool fresh) {
            acquire_stage();
            if (elect_one()) {
                for (int k = 0; k < AKB; ++k)
#pragma unroll
                    for (int j = 0; j < 4; ++j)
                        mma_ss2(d, desc_of(a_lo + (4 + k) * KBL + 2u * j), desc_of(b_lo + (uint32_t)(2 * k) * HBL + 2u * j), ID_N256,
                                (fresh && k == 0 && j == 0) ? 0u : 1u);
                mma_commit2(bar(B_EMPTY + stage));
            }
            advance();
        };
        // stage: GEMM2 of hidden chunk buffer b (fp16 in TMEM: K-block 0 at +0, K-block 1 at +64 columns) x all 256
        // latent columns: two consecutive boxes are this CTA's 128 weight rows of one [256 x 64] B tile, 4 MMAs with N = 256
        auto stage_g2 = [&](int b) {
            acquire_stage();
            if (elect_one()) {
                const uint32_t hbuf = TD1 + 128u * b;
#pragma unroll
                for (int j = 0; j < 4; ++j) mma_ts2(TZ, hbuf + 8u * j, desc_of(b_lo + 2u * j), ID_N256, 1u);
#pragma unroll
                for (int j = 0; j < 4; ++j) mma_ts2(TZ, hbuf + 64u + 8u * j, desc_of(b_lo + 2 * HBL + 2u * j), ID_N256, 1u);
                mma_commit2(bar(B_EMPTY + stage));
            }
            advance();
        };
        // scorer layer 2 stage: H1 K-blocks kb .. kb+3 (fp16 in TMEM columns [32 kb, ...)) into buffer b
        auto stage_l2 = [&](int b, int kb) {
            acquire_stage();
            if (elect_one()) {
#pragma unroll
                for (int q = 0; q < 4; ++q)
#pragma unroll
                    for (int j = 0; j < 4; ++j)
                        mma_ts2(TD1 + 128u * b, TZ + 32u * (kb + q) + 8u * j,
                                desc_of(b_lo + (uint32_t)q * HBL + 2u * j), ID_N128, (kb == 0 && q == 0 && j == 0) ? 0u : 1u);
                mma_commit2(bar(B_EMPTY + stage));
            }
            advance();
        };
        for (uint32_t it = 0;; ++it) {
            const uint32_t slot = it & 1;
            mbar_wait_warp(bar(B_SFULL + slot), (it >> 1) & 1);
            const int tile = __reduce_max_sync(0xffffffffu, (int)s_sched[slot * 2 + 0]);
            const int nsteps = __reduce_max_sync(0xffffffffu, (int)s_sched[slot * 2 + 1]);
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(B_SEMPTY + slot));
            if (tile < 0) break;
            if (rank != 0) continue;
#pragma unroll 1
            for (int t = 0; t < nsteps; ++t) {
                // Step boundary: the a K-blocks of chunks 0 and 1 depend only on a_{t+1} and both GEMM1 accumulators are
                // free, so they are issued before the wait for z' (pipe drain + LayerNorm is the serial section of a step)
                WM_TRACE(30);
                wait_h(0);
                wait_h(1);
                WM_TRACE(1);
                mbar_wait_warp(bar(B_AREADY), n_a & 1); ++n_a; tc_fence_after();
                WM_TRACE(2);
                if (TH) {
                    stage_f256(TD1, true);                 // u = W_w a into both (free) GEMM1 accumulators
                    commit(B_UFULL);
                    mbar_wait_warp(bar(B_ZREADY2), n_z & 1); ++n_z; tc_fence_after();   // boundary done: z_perp written, u read
                    stage_f256(TZ, false);                 // x = z_perp + W_d a (+ b2), accumulated onto the latent
                    stage_a01();
                    if (NC == 2) commit(B_AFREE);
                    stage_z(0); commit(B_D1FULL + 0);
                    stage_z(1); commit(B_D1FULL + 1);
                } else {
                    stage_a01();
                    if (NC == 2) commit(B_AFREE);
                    WM_TRACE(3);
                    mbar_wait_warp(bar(B_ZREADY), n_z & 1); tc_fence_after();
                    WM_TRACE(4);
                    stage_za();
                    mbar_wait_warp(bar(B_ZREADY2), n_z & 1); ++n_z; tc_fence_after();
                    stage_zb();
                }
                pend[0] = pend[1] = true;
                wait_h(0);
                stage_g2(0);
                if (NC == 1) commit(B_D2FULL);
#pragma unroll 1
                for (int i = 2; i <= NC; ++i) {
                    if (i < NC) {                       // GEMM1 chunk i into buffer i & 1 (its GEMM2 reader has been issued)
                        const int b = i & 1;
                        wait_h(b);
                        if (WIDE) {
                            stage_az(b, i == NC - 1);
                        } else {
                            stage_a(b, AKB, false);
                            if (i == NC - 1) commit(B_AFREE);
                            stage_z(b);
                        }
                        commit(B_D1FULL + b);
                        pend[b] = true;
                    }
                    wait_h((i - 1) & 1);
                    stage_g2((i - 1) & 1);              // GEMM2 chunk i - 1
                    if (i == NC) commit(B_D2FULL);
                }
            }
            if (!rank_it) {   // nothing to rank: only take the terminal latent's ZREADY so the phase count stays in step
                if (!TH) mbar_wait_warp(bar(B_ZREADY), n_z & 1);
                mbar_wait_warp(bar(B_ZREADY2), n_z & 1);
                ++n_z;
                continue;
            }
            // ---- scorer layer 1: four 128-column chunks of gelu(Ws0 [z_T; phi; hw] + bs0)
            WM_TRACE(31);
#pragma unroll 1
            for (int c = 0; c < 4; ++c) {
                const int b = c & 1;
                wait_h(b);
                if (c == 0) { mbar_wait_warp(bar(B_AREADY), n_a & 1); ++n_a; tc_fence_after(); }
                stage_a(b, PKB, true);
                if (c == 3) commit(B_AFREE);
                if (c == 0) {
                    if (!TH) mbar_wait_warp(bar(B_ZREADY), n_z & 1);
                    mbar_wait_warp(bar(B_ZREADY2), n_z & 1);
                    ++n_z;
                    tc_fence_after();
                }
                stage_z(b);
                commit(B_D1FULL + b);
                pend[b] = true;
            }
            wait_h(0);
            wait_h(1);   // all of H1 (fp16, TMEM columns [0,256)) written
            // ---- scorer layer 2: A = H1 from TMEM, K = 512
#pragma unroll 1
            for (int c = 0; c < 4; ++c) {
                const int b = c & 1;
                wait_h(b);
                stage_l2(b, 0);
                stage_l2(b, 4);
                commit(B_D1FULL + b);
                pend[b] = true;
            }
        }
        __syncwarp();
    }
    }
    else if (warp < ACT_WARP0) {
        // =============================================================== epilogue warps (GELU / LayerNorm / scorer)
        reg_alloc<176>();
        const int q = warp & 3, hh = (warp - EPI_WARP0) >> 2;
        const int row = 32 * q + lane;
        const uint32_t lane_off = (uint32_t)(32 * q) << 16;
        uint8_t* a1 = smem + L.a1;
        const uint32_t r_hready0 = mapa(bar(B_HREADY), 0), r_hready1 = mapa(bar(B_HREADY + 1), 0);
        const uint32_t r_zready = mapa(bar(B_ZREADY), 0), r_zready2 = mapa(bar(B_ZREADY2), 0);
        uint32_t n_d1[2] = {0, 0}, n_d2 = 0, n_u = 0, n_b = 0;
        const float inv_d = 1.0f / (float)D;
        WM_TRACE_DECL(warp == 0 ? p.prof : nullptr, 2)
        // The latent is carried as u = z + b2, twice: fp32 in TMEM — GEMM2 accumulates W2 h onto it, so the accumulator IS
        // LayerNorm's input z + W2 h + b2 and no pass adds b2 — and fp16 in A1 (GEMM1's operand, the scorer's input): the
        // host subtracts W1z b2 (Ws0z b2) from the bias that rides on the constant feature column (tcp_prepare), and
        // beta in shared memory is beta + b2, so LayerNorm's output is u directly.
        // 32 consecutive columns of this row: u (fp32 values in v) -> fp16 -> A1
        auto z_to_smem = [&](int col0, const uint32_t* v) {
            uint8_t* kb = a1 + (col0 >> 6) * KB_BYTES;
            const int chunk0 = (col0 & 63) >> 3;
#pragma unroll
            for (int ch = 0; ch < 4; ++ch) {
                uint4 o;
                o.x = pack_f16(__uint_as_float(v[8 * ch + 0]), __uint_as_float(v[8 * ch + 1]));
                o.y = pack_f16(__uint_as_float(v[8 * ch + 2]), __uint_as_float(v[8 * ch + 3]));
                o.z = pack_f16(__uint_as_float(v[8 * ch + 4]), __uint_as_float(v[8 * ch + 5]));
                o.w = pack_f16(__uint_as_float(v[8 * ch + 6]), __uint_as_float(v[8 * ch + 7]));
                *reinterpret_cast<uint4*>(kb + sw128_off(row, chunk0 + ch)) = o;
            }
        };
        // first half of this thread's columns (K-block 2 hh) is in A1: GEMM1 may start on it
        auto publish_half = [&]() {
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) mbar_arrive_remote(r_zready);
        };
        auto publish = [&](uint32_t leader_bar, bool smem_written) {
            tmem_st_wait();
            WM_TRACE(45);
            if (smem_written) fence_proxy_async();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_remote(leader_bar);
        };
        // GELU over this thread's 64 columns of accumulator buffer b (the bias is already in the accumulator: it rides on
        // the constant-1 feature column), fp16 result to TMEM at dst_col.  Both TMEM loads are in flight before the first use.
        auto gelu_chunk = [&](int b, uint32_t dst_col) {
            WM_TRACE(40);
            mbar_wait_inline(bar(B_D1FULL + b), n_d1[b] & 1);
            WM_TRACE(41);
            ++n_d1[b];
            tc_fence_after();
            uint32_t v0[32], v1[32], o[16];
            tmem_ld32(T_D1 + 128u * b + lane_off + 64u * hh, v0);
            tmem_ld32(T_D1 + 128u * b + lane_off + 64u * hh + 32u, v1);
            tmem_ld_wait();
            WM_TRACE(43);
#pragma unroll
            for (int i = 0; i < 16; ++i) o[i] = gelu2_h2(__uint_as_float(v0[2 * i]), __uint_as_float(v0[2 * i + 1]));
            tmem_st16(dst_col + lane_off, o);
#pragma unroll
            for (int i = 0; i < 16; ++i) o[i] = gelu2_h2(__uint_as_float(v1[2 * i]), __uint_as_float(v1[2 * i + 1]));
            tmem_st16(dst_col + lane_off + 16u, o);
            WM_TRACE(44);
            publish(b == 0 ? r_hready0 : r_hready1, false);
            WM_TRACE(42);
        };

        for (uint32_t it = 0;; ++it) {
            const uint32_t slot = it & 1;
            mbar_wait_inline(bar(B_SFULL + slot), (it >> 1) & 1);
            const int tile = s_sched[slot * 2 + 0], nsteps = s_sched[slot * 2 + 1];
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(B_SEMPTY + slot));
            if (tile < 0) break;
            int cand, len, seg;
            row_meta(p.a, (int64_t)tile * TMP + TM * (int)rank + row, cand, len, seg, false);
            // prefix-latent reuse: the rollout covers positions [st, len) and starts from the row init_index names
            const int st = EXT ? row_start(p.a, cand, len) : 0, rem = len - st;
            const size_t zrow = EXT ? row_init(p.a, cand, seg) : (size_t)seg;

            if (TH) {
            // ---- TransH: boundary t = 0 .. nsteps.  Boundary t normalises the result of step t - 1 (t = 0: takes z_0 as it
            // is) and, when a step t follows, projects it onto the hyperplane of action t: ONE epilogue per step boundary.
            constexpr float kEps = 1e-12f;
#pragma unroll 1
            for (int t = 0; t <= nsteps; ++t) {
                const bool has_u = t < nsteps;
                uint32_t v[128];
                if (t > 0) {
                    mbar_wait_inline(bar(B_D2FULL), n_d2 & 1);
                    ++n_d2;
                    tc_fence_after();
#pragma unroll
                    for (int p4 = 0; p4 < 4; ++p4)
                        tmem_ld32(T_Z + lane_off + (uint32_t)(128 * hh + 32 * p4), reinterpret_cast<uint32_t(&)[32]>(v[32 * p4]));
                } else {
#pragma unroll
                    for (int p4 = 0; p4 < 4; ++p4) {
                        if (cand >= 0) {
                            const float4* src = reinterpret_cast<const float4*>(p.a.init_states + zrow * D + 128 * hh + 32 * p4);
#pragma unroll
                            for (int i = 0; i < 8; ++i) {
                                const float4 f = __ldg(src + i);
                                range_check(f, p.a.fault);
                                v[32 * p4 + 4 * i + 0] = __float_as_uint(f.x); v[32 * p4 + 4 * i + 1] = __float_as_uint(f.y);
                                v[32 * p4 + 4 * i + 2] = __float_as_uint(f.z); v[32 * p4 + 4 * i + 3] = __float_as_uint(f.w);
                            }
                        } else {
#pragma unroll
                            for (int i = 0; i < 32; ++i) v[32 * p4 + i] = 0u;
                        }
                    }
                }
                if (has_u) {
                    mbar_wait_inline(bar(B_UFULL), n_u & 1);
                    ++n_u;
                    tc_fence_after();
                }
                tmem_ld_wait();
                // pass 1: |v|^2, |u|^2, u.v over this thread's 128 columns (u streamed from the GEMM1 accumulators)
                float2 svv = make_float2(0.0f, 0.0f), suu = make_float2(0.0f, 0.0f), suv = make_float2(0.0f, 0.0f);
#pragma unroll
                for (int i = 0; i < 64; ++i) {
                    const float2 x = make_float2(__uint_as_float(v[2 * i]), __uint_as_float(v[2 * i + 1]));
                    svv = __ffma2_rn(x, x, svv);
                }
                if (has_u) {
#pragma unroll
                    for (int p4 = 0; p4 < 4; ++p4) {
                        uint32_t u[32];
                        tmem_ld32(T_D1 + lane_off + (uint32_t)(128 * hh + 32 * p4), u);
                        tmem_ld_wait();
#pragma unroll
                        for (int i = 0; i < 16; ++i) {
                            const float2 uu = make_float2(__uint_as_float(u[2 * i]), __uint_as_float(u[2 * i + 1]));
                            const float2 x = make_float2(__uint_as_float(v[32 * p4 + 2 * i]), __uint_as_float(v[32 * p4 + 2 * i + 1]));
                            suu = __ffma2_rn(uu, uu, suu);
                            suv = __ffma2_rn(uu, x, suv);
                        }
                    }
                }
                float4* red = s_red + (n_b & 1u) * 2 * TM;      // (parity slots as in the LayerNorm: one barrier per exchange)
                ++n_b;
                red[hh * TM + row] = make_float4(svv.x + svv.y, suu.x + suu.y, suv.x + suv.y, 0.0f);
                named_bar_sync(1 + q, 64);
                const float4 other = red[(hh ^ 1) * TM + row];
                const float vv = svv.x + svv.y + other.x, uu2 = suu.x + suu.y + other.y, uv = suv.x + suv.y + other.z;
                const float rn = t > 0 ? rsqrtf(vv + kEps) : 1.0f;        // z' = v / sqrt(|v|^2 + eps); boundary 0 keeps z_0
                const bool live = t < rem;                                 // a step t follows for this row
                const bool done_now = t == rem;                            // z' is this row's terminal latent
                const float c = (has_u && live) ? uv * rn / (uu2 + kEps) : 0.0f;   // (w.z') w = (u.z') u / (|u|^2 + eps)
                float4* lat = nullptr;     // wm_rollout_latents: z after step t - 1 (or only the terminal one: [B, d])
                if (EXT && p.a.latents_out && t > 0 && t - 1 < rem) {
                    if (!p.a.latents_terminal)
                        lat = reinterpret_cast<float4*>(p.a.latents_out + ((size_t)cand * p.a.T_max + st + t - 1) * D);
                    else if (done_now)
                        lat = reinterpret_cast<float4*>(p.a.latents_out + (size_t)cand * D);
                }
                const float2 rn2 = make_float2(rn, rn), mc2 = make_float2(-c, -c);
#pragma unroll
                for (int p4 = 0; p4 < 4; ++p4) {
                    const int col0 = 128 * hh + 32 * p4;
                    uint32_t* vv32 = v + 32 * p4;
                    uint32_t u[32];
                    if (has_u) {
                        tmem_ld32(T_D1 + lane_off + (uint32_t)col0, u);
                        tmem_ld_wait();
                    }
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        float2 x = __fmul2_rn(make_float2(__uint_as_float(vv32[2 * i]), __uint_as_float(vv32[2 * i + 1])), rn2);   // z'
                        if (EXT && lat) reinterpret_cast<float2*>(lat)[(col0 >> 1) + i] = x;
                        if (done_now) { vv32[2 * i] = __float_as_uint(x.x); vv32[2 * i + 1] = __float_as_uint(x.y); }
                        if (has_u) x = __ffma2_rn(make_float2(__uint_as_float(u[2 * i]), __uint_as_float(u[2 * i + 1])), mc2, x);   // z_perp
                        if (!done_now) { vv32[2 * i] = __float_as_uint(x.x); vv32[2 * i + 1] = __float_as_uint(x.y); }
                    }
                    // live rows: z_perp -> fp16 operand; a row that has just finished: its terminal z' (and it is frozen);
                    // rows that finished earlier keep theirs.  The fp32 copy is written for every row (it stays bounded).
                    if (live || done_now) z_to_smem(col0, vv32);
                    tmem_st32(T_Z + lane_off + (uint32_t)col0, reinterpret_cast<const uint32_t(&)[32]>(v[32 * p4]));
                }
                publish(r_zready2, true);
                if (has_u)
                    for (int cc = 0; cc < NC; ++cc) gelu_chunk(cc & 1, T_D1 + 128u * (cc & 1) + 64u * hh);
            }
            } else {
            // ---- z_0 (the task's initial latent; or the banked latent after the first st steps)
#pragma unroll 1
            for (int p4 = 0; p4 < 4; ++p4) {
                const int col0 = 128 * hh + 32 * p4;
                uint32_t v[32];
                if (cand >= 0) {
                    const float4* src = reinterpret_cast<const float4*>(p.a.init_states + zrow * D + col0);
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const float4 f = __ldg(src + i);
                        range_check(f, p.a.fault);
                        v[4 * i + 0] = __float_as_uint(f.x); v[4 * i + 1] = __float_as_uint(f.y);
                        v[4 * i + 2] = __float_as_uint(f.z); v[4 * i + 3] = __float_as_uint(f.w);
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < 32; ++i) v[i] = 0u;
                }
                const float4* b2v = reinterpret_cast<const float4*>(s_b2 + col0);
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const float4 bb = b2v[i];
                    v[4 * i + 0] = __float_as_uint(__uint_as_float(v[4 * i + 0]) + bb.x);
                    v[4 * i + 1] = __float_as_uint(__uint_as_float(v[4 * i + 1]) + bb.y);
                    v[4 * i + 2] = __float_as_uint(__uint_as_float(v[4 * i + 2]) + bb.z);
                    v[4 * i + 3] = __float_as_uint(__uint_as_float(v[4 * i + 3]) + bb.w);
                }
                z_to_smem(col0, v);
                tmem_st32(T_Z + lane_off + (uint32_t)col0, reinterpret_cast<const uint32_t(&)[32]>(v));
                if (p4 == 1) publish_half();
            }
            publish(r_zready2, true);

            for (int t = 0; t < nsteps; ++t) {
                for (int c = 0; c < NC; ++c)
                    gelu_chunk(c & 1, T_D1 + 128u * (c & 1) + 64u * hh);
                // ---- LayerNorm(z + W2 h + b2) = LayerNorm(accumulator), this thread's 128 columns held in registers
                WM_TRACE(50);
                mbar_wait_inline(bar(B_D2FULL), n_d2 & 1);
                WM_TRACE(51);
                ++n_d2;
                tc_fence_after();
                uint32_t v[128];
#pragma unroll
                for (int p4 = 0; p4 < 4; ++p4)
                    tmem_ld32(T_Z + lane_off + (uint32_t)(128 * hh + 32 * p4), reinterpret_cast<uint32_t(&)[32]>(v[32 * p4]));
                tmem_ld_wait();
                WM_TRACE(54);
                float2 s1v = make_float2(0.0f, 0.0f), s2v = make_float2(0.0f, 0.0f);
#pragma unroll
                for (int i = 0; i < 64; ++i) {
                    const float2 x = make_float2(__uint_as_float(v[2 * i]), __uint_as_float(v[2 * i + 1]));
                    s1v = __fadd2_rn(s1v, x);
                    s2v = __ffma2_rn(x, x, s2v);
                }
                const float s1 = s1v.x + s1v.y, s2 = s2v.x + s2v.y;
                // exchanged through the slot of this LayerNorm's parity: the partner reads the previous LayerNorm's value
                // from the other slot, so no second barrier is needed before the next one writes
                float4* red = s_red + (n_d2 & 1u) * 2 * TM;
                red[hh * TM + row] = make_float4(s1, s2, 0.0f, 0.0f);
                WM_TRACE(55);
                named_bar_sync(1 + q, 64);
                const float4 other = red[(hh ^ 1) * TM + row];
                WM_TRACE(52);
                const float mean = (s1 + other.x) * inv_d;
                const float var = fmaxf((s2 + other.y) * inv_d - mean * mean, 0.0f);
                const float rstd = rsqrtf(var + p.ln_eps);
                const bool live = t < rem;     // masked steps leave the state unchanged
                float4* lat = nullptr;     // wm_rollout_latents: z after this step (or only the terminal one: [B, d])
                if (EXT && p.a.latents_out && live) {
                    if (!p.a.latents_terminal)
                        lat = reinterpret_cast<float4*>(p.a.latents_out + ((size_t)cand * p.a.T_max + st + t) * D);
                    else if (st + t == len - 1)
                        lat = reinterpret_cast<float4*>(p.a.latents_out + (size_t)cand * D);
                }
                const float2 rs2 = make_float2(rstd, rstd), mr2 = make_float2(-mean * rstd, -mean * rstd);
#pragma unroll
                for (int p4 = 0; p4 < 4; ++p4) {
                    const int col0 = 128 * hh + 32 * p4;
                    uint32_t* vv = v + 32 * p4;
                    const float4* gv = reinterpret_cast<const float4*>(s_gamma + col0);
                    const float4* bev = reinterpret_cast<const float4*>(s_beta + col0);
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const float4 gg = gv[i], be = bev[i];
                        float2 x0 = make_float2(__uint_as_float(vv[4 * i]), __uint_as_float(vv[4 * i + 1]));
                        float2 x1 = make_float2(__uint_as_float(vv[4 * i + 2]), __uint_as_float(vv[4 * i + 3]));
                        x0 = __ffma2_rn(__ffma2_rn(x0, rs2, mr2), make_float2(gg.x, gg.y), make_float2(be.x, be.y));
                        x1 = __ffma2_rn(__ffma2_rn(x1, rs2, mr2), make_float2(gg.z, gg.w), make_float2(be.z, be.w));
                        vv[4 * i] = __float_as_uint(x0.x); vv[4 * i + 1] = __float_as_uint(x0.y);
                        vv[4 * i + 2] = __float_as_uint(x1.x); vv[4 * i + 3] = __float_as_uint(x1.y);
                    }
                    // frozen rows: the fp16 copy (GEMM1 operand, scorer input) keeps the terminal latent; their
                    // fp32 master is never read again
                    if (live) z_to_smem(col0, vv);
                    if (EXT && lat) {      // the caller's latent is z = u - b2
                        const float4* b2v = reinterpret_cast<const float4*>(s_b2 + col0);
#pragma unroll
                        for (int i = 0; i < 8; ++i) {
                            const float4 bb = b2v[i];
                            lat[(col0 >> 2) + i] = make_float4(__uint_as_float(vv[4 * i]) - bb.x, __uint_as_float(vv[4 * i + 1]) - bb.y,
                                                               __uint_as_float(vv[4 * i + 2]) - bb.z, __uint_as_float(vv[4 * i + 3]) - bb.w);
                        }
                    }
                    tmem_st32(T_Z + lane_off + (uint32_t)col0, reinterpret_cast<const uint32_t(&)[32]>(v[32 * p4]));
                    if (p4 == 1) publish_half();
                }
                publish(r_zready2, true);
                WM_TRACE(53);
            }

            }
            if (!rank_it) continue;
            // ---- scorer layer 1 -> H1 (fp16) in TMEM columns [0,256)
            for (int c = 0; c < 4; ++c)
                gelu_chunk(c & 1, T_Z + 64u * c + 32u * hh);
            // ---- scorer layer 2 + output dot product
            float part = 0.0f;
            for (int c = 0; c < 4; ++c) {
                const int b = c & 1;
                mbar_wait_inline(bar(B_D1FULL + b), n_d1[b] & 1);
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
            s_red[hh * TM + row] = make_float4(part, 0.0f, 0.0f, 0.0f);
            named_bar_sync(1 + q, 64);
            if (hh == 0 && cand >= 0 && (!EXT || p.a.scores_out)) p.a.scores_out[cand] = part + s_red[TM + row].x + __ldg(p.bs2);
            named_bar_sync(1 + q, 64);   // s_red is reused by the next tile's first LayerNorm
        }
    } else {
        // =============================================================== action-feature warps (one row per lane)
        reg_dealloc<64>();
        // Per step a row's action enters GEMM1 as the feature row f_t = [onehot(id) (NT) | log2 p_j (P) | 1] of K-block 4
        // (and 5 when NT + P + 1 > 64): the embedding tables and biases are folded into the weights (tcp_prepare).
        const int aw = warp - ACT_WARP0;
        const int row = 32 * aw + lane;
        uint8_t* a1 = smem + L.a1;
        uint8_t* s_cnt = smem + L.cnt;
        const uint32_t r_aready = mapa(bar(B_AREADY), 0);
        const int P = p.P, NT = p.n_types;
        uint32_t n_w = 0;
        WM_TRACE_DECL(aw == 0 ? p.prof : nullptr, 3)
        // 16-bit feature store: column c of this row in K-blocks 4, 5
        auto put = [&](int c, uint32_t h16) {
            *reinterpret_cast<uint16_t*>(a1 + (4 + (c >> 6)) * KB_BYTES + sw128_off(row, (c & 63) >> 3) + (c & 7) * 2) = (uint16_t)h16;
        };
        auto clear_row = [&](int nkb) {
            for (int ch = 0; ch < 8 * nkb; ++ch)
                *reinterpret_cast<uint4*>(a1 + (4 + (ch >> 3)) * KB_BYTES + sw128_off(row, ch & 7)) = make_uint4(0u, 0u, 0u, 0u);
        };
        for (uint32_t it = 0;; ++it) {
            const uint32_t slot = it & 1;
            mbar_wait(bar(B_SFULL + slot), (it >> 1) & 1);
            const int tile = s_sched[slot * 2 + 0], nsteps = s_sched[slot * 2 + 1];
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(B_SEMPTY + slot));
            if (tile < 0) break;
            int cand, len, seg;
            row_meta(p.a, (int64_t)tile * TMP + TM * (int)rank + row, cand, len, seg, false);
            for (int c = 0; c < NT; ++c) s_cnt[row * NT + c] = 0;
            float slp[MAX_P];   // per parameter slot: running sum of log2 p
#pragma unroll
            for (int j = 0; j < MAX_P; ++j) slp[j] = 0.0f;
            // structured phi: the per-slot running maximum lives in shared memory
            float4* s_mx4 = reinterpret_cast<float4*>(smem + L.mx) + row * (MAX_P / 4);
            if (PHI == WM_PHI_STRUCT) s_mx4[0] = s_mx4[1] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            // one action of this row: type id (clamped), log2 of its parameters, phi statistics
            auto account = [&](int id, const int (&raw)[MAX_P], float (&lp)[MAX_P]) -> int {
                if (id < 0 || id >= NT) {
                    atomicOr(p.a.fault, WM_FAULT_TYPE);
                    id = id < 0 ? 0 : NT - 1;
                }
#pragma unroll
                for (int j = 0; j < MAX_P; ++j) {
                    if (j < P) {
                        int prm = raw[j];
                        if (prm < 1) {
                            atomicOr(p.a.fault, WM_FAULT_PARAM);
                            prm = 1;
                        }
                        lp[j] = log2f((float)prm);
                        slp[j] += lp[j];
                    }
                }
                s_cnt[row * NT + id] += 1;
                if (PHI == WM_PHI_STRUCT) {
                    float4 m0 = s_mx4[0], m1 = s_mx4[1];
                    m0.x = fmaxf(m0.x, lp[0]); m0.y = fmaxf(m0.y, lp[1]); m0.z = fmaxf(m0.z, lp[2]); m0.w = fmaxf(m0.w, lp[3]);
                    m1.x = fmaxf(m1.x, lp[4]); m1.y = fmaxf(m1.y, lp[5]); m1.z = fmaxf(m1.z, lp[6]); m1.w = fmaxf(m1.w, lp[7]);
                    s_mx4[0] = m0; s_mx4[1] = m1;
                }
                return id;
            };
            auto take = [&](int pos, float (&lp)[MAX_P]) -> int {   // the action at position `pos`
                const int id = __ldg(p.a.action_ids + (size_t)cand * p.a.T_max + pos);
                const int32_t* pp = p.a.action_params + ((size_t)cand * p.a.T_max + pos) * P;
                int raw[MAX_P];
#pragma unroll
                for (int j = 0; j < MAX_P; ++j) raw[j] = j < P ? __ldg(pp + j) : 1;
                return account(id, raw, lp);
            };
            // prefix-latent reuse: positions [0, st) only feed phi; scanned four at a time BEFORE the first rollout step, in
            // position order, so the running sums see the positions in the literal call's order (bit-identical scores)
            const int st = EXT ? row_start(p.a, cand, len) : 0;
            int scanned = 0;
            auto scan4 = [&]() {
                int rid[4], raw[4][MAX_P];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int pos = scanned + u < st ? scanned + u : 0;      // (in-bounds dummy for finished lanes)
                    rid[u] = cand >= 0 ? __ldg(p.a.action_ids + (size_t)cand * p.a.T_max + pos) : 0;
#pragma unroll
                    for (int j = 0; j < MAX_P; ++j)
                        raw[u][j] = (cand >= 0 && j < P)
                                        ? __ldg(p.a.action_params + ((size_t)cand * p.a.T_max + pos) * P + j) : 1;
                }
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (scanned + u < st) {
                        float lp[MAX_P];
#pragma unroll
                        for (int j = 0; j < MAX_P; ++j) lp[j] = 0.0f;
                        account(rid[u], raw[u], lp);
                    }
                scanned += 4;
            };
            if (EXT && p.a.start)
                while (__any_sync(0xffffffffu, scanned < st)) scan4();

            int prev_id = -1;      // the one-hot column this row has set
            for (int t = 0; t < nsteps; ++t) {
                // read the step's action, log2 of its parameters, phi statistics — before the wait: the loads' latency hides
                WM_TRACE(70);
                int id = -1;
                float lp[MAX_P];
#pragma unroll
                for (int j = 0; j < MAX_P; ++j) lp[j] = 0.0f;
                if (st + t < len) id = take(st + t, lp);
                // store only once GEMM1 of the previous step (or the previous tile's scorer) no longer reads K-blocks 4, 5
                WM_TRACE(71);
                if (n_w > 0) mbar_wait(bar(B_AFREE), (n_w - 1) & 1);
                WM_TRACE(72);
                ++n_w;
                if (t == 0) {          // the K-blocks still hold the previous tile's phi features
                    clear_row(WIDE ? 1 : 2);
                    put(NT + P, 0x3C00u);                      // the constant-1 column (carries W1a b_p + b1)
                }
                if (id >= 0) {         // a masked row keeps its last features: its result is discarded anyway (frozen row)
                    if (prev_id >= 0 && prev_id != id) put(prev_id, 0u);
                    put(id, 0x3C00u);
                    prev_id = id;
#pragma unroll
                    for (int j = 0; j < MAX_P; ++j)
                        if (j < P) put(NT + j, pack_f16(lp[j], 0.0f));
                }
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive_remote(r_aready);
                WM_TRACE(73);
            }

            // ---- the phi features of the scorer's A operand (K-blocks 4, 5), one row per lane:
            //   WM_PHI_MEAN    phi = mean_t a_t is LINEAR in psi = [count_c / len (NT) | sum_t log2 p_tj / len (P) | 1 (len > 0)];
            //                  the host folds E, W_p and b_p into scorer layer 1's phi weights (tcp_prepare)
            //   WM_PHI_STRUCT  phi = [count_c (NT) | len | sum_j (P) | mean_j (P) | max_j (P)]   (S25)
            // followed by a constant-1 column that carries scorer layer 1's bias
            if (!rank_it) continue;
            if (n_w > 0) mbar_wait(bar(B_AFREE), (n_w - 1) & 1);
            ++n_w;
            {
                auto putf = [&](int c, float v) { put(c, pack_f16(v, 0.0f)); };
                clear_row(WIDE ? 1 : 2);
                const float inv = len > 0 ? 1.0f / (float)len : 0.0f;
                if (PHI == WM_PHI_STRUCT) {
                    for (int c = 0; c < NT; ++c) putf(c, (float)s_cnt[row * NT + c]);
                    putf(NT, (float)len);
                    const float4 m0 = s_mx4[0], m1 = s_mx4[1];
                    const float mxr[8] = {m0.x, m0.y, m0.z, m0.w, m1.x, m1.y, m1.z, m1.w};
#pragma unroll
                    for (int j = 0; j < MAX_P; ++j)
                        if (j < P) {
                            putf(NT + 1 + j, slp[j]);
                            putf(NT + 1 + P + j, slp[j] * inv);
                            putf(NT + 1 + 2 * P + j, mxr[j]);
                        }
                    put(NT + 1 + 3 * P, 0x3C00u);
                } else {
                    for (int c = 0; c < NT; ++c) putf(c, (float)s_cnt[row * NT + c] * inv);
#pragma unroll
                    for (int j = 0; j < MAX_P; ++j)
                        if (j < P) putf(NT + j, slp[j] * inv);
                    putf(NT + P, len > 0 ? 1.0f : 0.0f);
                    put(NT + P + 1, 0x3C00u);
                }
            }
            // hardware features of this row -> the hw operand tile (columns >= H stay zero)
            for (int ch = 0; ch < p.H / 8; ++ch) {
                uint4 o = make_uint4(0u, 0u, 0u, 0u);
                if (cand >= 0 && (!EXT || p.a.hw_feats)) {
                    const float4* src = reinterpret_cast<const float4*>(p.a.hw_feats + (size_t)seg * p.H + 8 * ch);
                    const float4 f0 = __ldg(src), f1 = __ldg(src + 1);
                    o.x = pack_f16(f0.x, f0.y); o.y = pack_f16(f0.z, f0.w);
                    o.z = pack_f16(f1.x, f1.y); o.w = pack_f16(f1.z, f1.w);
                }
                // K-step ch/2, K half ch&1 of the no-swizzle tile (see smem_desc_nosw)
                *reinterpret_cast<uint4*>(smem + L.hwk + (ch >> 1) * HWK_BYTES + (row >> 3) * 256 + (ch & 1) * 128 +
                                          (row & 7) * 16) = o;
            }
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) mbar_arrive_remote(r_aready);
        }
    }

    // ---- teardown: no CTA of the pair may exit (or free TMEM) while the other's MMAs / arrivals can still reach it
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    if (warp == ALLOC_WARP) tmem_dealloc2(tmem_base, 512);
}

}  // namespace tcp

// ------------------------------------------------------------------------------------------------ host side
namespace {

// Append one box slot: for each CTA (rank 0, then rank 1) 64 image rows of 128 B = the SW128 K-major image of
// W[row0 + rstride * r + n][k0 + k], n < 64, k < 64 (k >= kvalid reads as zero): row n at n * 128 B, 16-byte chunk c at
// (c ^ (n & 7)).  N = 128 K-block: rstride = 64 (the CTAs hold the two halves of the 128 weight rows).  N = 256 K-block:
// two slots, rstride = 128, row0 = 0 and 64 (two consecutive boxes of a CTA = its 128 weight rows).
// Returns false when a weight is not finite in fp16 (|w| > 65504): the model then stays on the fp32 kernel.
bool append_slot(std::vector<uint16_t>& blob, const std::vector<float>& W, int ld, int row0, int rstride, int k0, int kvalid) {
    const size_t base = blob.size();
    blob.resize(base + 2 * tcp::HB_BYTES / 2, 0);
    bool ok = true;
    for (int r = 0; r < 2; ++r)
        for (int n = 0; n < 64; ++n)
            for (int k = 0; k < 64; ++k) {
                const float v = k < kvalid ? W[(size_t)(row0 + rstride * r + n) * ld + k0 + k] : 0.0f;
                const size_t off = (size_t)r * tcp::HB_BYTES + (size_t)n * 128 + (size_t)((((k >> 3) ^ (n & 7)) << 4)) +
                                   (size_t)(k & 7) * 2;
                uint16_t hb;
                ok &= f32_to_f16_bits(v, &hb);
                blob[base + off / 2] = hb;
            }
    return ok;
}

}  // namespace

bool tcp_model_ok(const Model& m) {
    // per-type phi (WM_PHI_TYPED, S28): this kernel rolls such a model and hands the terminal latents to the fp32 kernel, which
    // builds phi and runs the scorer (wm_api.cu): no scorer shape to match, as for the forest ranker
    return m.phi_kind <= WM_PHI_TYPED && (m.kind == WM_KIND_MLP_LN || m.kind == WM_KIND_TRANSH) && m.dtype == WM_DTYPE_BF16 && m.embed == WM_EMBED_LINEAR && m.d == tcp::D &&
           m.d_a == tcp::DA && m.hidden >= 256 && m.hidden <= tcp::MAX_HID && m.hidden % 128 == 0 &&
           ((m.n_lin == 3 && m.sdim[1] == tcp::SW && m.sdim[2] == tcp::SW) || m.ranker_kind == WM_RANKER_FOREST || m.phi_kind == WM_PHI_TYPED) &&
           m.H >= 8 && m.H <= tcp::MAX_H && m.H % 8 == 0 && m.n_types <= tcp::MAX_TYPES && m.P <= tcp::MAX_P;
}

int tcp_prepare(wm_ctx* ctx, const std::vector<std::vector<float>>& hv, const std::vector<std::string>& names) {
    Model& m = ctx->m;
    m.tcp_ok = 0;
    if (!tcp_model_ok(m)) return WM_OK;
    auto get = [&](const char* n) -> const std::vector<float>& {
        for (size_t i = 0; i < names.size(); ++i)
            if (names[i] == n) return hv[i];
        static const std::vector<float> empty;
        return empty;
    };
    const std::vector<float>&W1 = get("W1"), &W2 = get("W2"), &b1 = get("b1"), &E = get("E"), &Wp = get("W_p"), &bpv = get("b_p");
    const std::vector<float>& b2h = get("b2");
    // `forest` = the kernel's MLP scorer is never run for this model (zero image): forest ranker, or per-type phi
    const bool forest = m.ranker_kind == WM_RANKER_FOREST || m.phi_kind == WM_PHI_TYPED, transh = m.kind == WM_KIND_TRANSH;
    const int hid = m.hidden, NC = hid / 128, K1 = tcp::D + tcp::DA, NT = m.n_types, P = m.P;
    // ---- A matrix that multiplies the action embedding, folded onto the action features f = [onehot(id) (NT) | log2 p_j (P) | 1]:
    //      M (E[id] + W_p lp + b_p) + bias  =  (M E^T)[:, id] + (M W_p) lp + (M b_p + bias); products summed in double
    const int NF = NT + P + 1, AKB = (NF + 63) / 64;
    auto fold = [&](const double* M, int rows, const double* bias) {     // M [rows][d_a], row-major
        std::vector<float> out((size_t)rows * 64 * AKB, 0.0f);
        for (int n = 0; n < rows; ++n) {
            const double* wr = M + (size_t)n * tcp::DA;
            float* o = &out[(size_t)n * 64 * AKB];
            for (int c = 0; c < NT; ++c) {
                double acc = 0.0;
                for (int k = 0; k < tcp::DA; ++k) acc += wr[k] * E[(size_t)c * tcp::DA + k];
                o[c] = (float)acc;
            }
            for (int j = 0; j < P; ++j) {
                double acc = 0.0;
                for (int k = 0; k < tcp::DA; ++k) acc += wr[k] * Wp[(size_t)k * P + j];
                o[NT + j] = (float)acc;
            }
            double acc = bias ? bias[n] : 0.0;
            for (int k = 0; k < tcp::DA; ++k) acc += wr[k] * bpv[k];
            o[NT + P] = (float)acc;
        }
        return out;
    };
    // GEMM1's a-columns (+ b1 on the constant column).  MLP+LN: the z operand is u = z + b2, so W1z b2 comes off the bias.
    // TransH: W1 [x ; a] with x = z_perp + W_d a  =  W1z z_perp + (W1a + W1z W_d) a: the translation is folded in as well.
    std::vector<double> W1a((size_t)hid * tcp::DA), b1f(hid);
    std::vector<float> W1f, Uf, Df;
    {
        const std::vector<float>* Wd = transh ? &get("W_d") : nullptr;
        for (int n = 0; n < hid; ++n) {
            for (int j = 0; j < tcp::DA; ++j) {
                double acc = W1[(size_t)n * K1 + tcp::D + j];
                if (transh)
                    for (int k = 0; k < tcp::D; ++k) acc += (double)W1[(size_t)n * K1 + k] * (double)(*Wd)[(size_t)k * tcp::DA + j];
                W1a[(size_t)n * tcp::DA + j] = acc;
            }
            double bb = b1[n];
            if (!transh)
                for (int k = 0; k < tcp::D; ++k) bb -= (double)W1[(size_t)n * K1 + k] * b2h[k];
            b1f[n] = bb;
        }
        W1f = fold(W1a.data(), hid, b1f.data());
        if (transh) {     // u = W_w a and the translation W_d a (+ b2: the accumulator then is v = x + W2 h + b2)
            const std::vector<float>& Ww = get("W_w");
            std::vector<double> Mw(Ww.begin(), Ww.end()), Md(Wd->begin(), Wd->end()), b2d(b2h.begin(), b2h.end());
            Uf = fold(Mw.data(), tcp::D, nullptr);
            Df = fold(Md.data(), tcp::D, b2d.data());
        }
    }
    // ---- scorer layer 1's phi columns as the kernel's phi features see them, plus the bias on a constant-1 column:
    //      WM_PHI_STRUCT: the F columns of Ws0 as they are; WM_PHI_MEAN: folded onto psi (see the action warps)
    const int F = m.phi_dim, K0 = tcp::D + F + m.H;   // scorer input [z ; phi ; hw]
    const int NPSI = (m.phi_kind == WM_PHI_STRUCT ? NT + 1 + 3 * P : NT + P + 1) + 1, PKB = (NPSI + 63) / 64;
    std::vector<float> Wphi((size_t)tcp::SW * 64 * PKB, 0.0f);
    if (!forest) {
        const std::vector<float>&Ws0 = get("Ws0"), &bs0 = get("bs0");
        for (int n = 0; n < tcp::SW; ++n) {
            const float* wr = &Ws0[(size_t)n * K0 + tcp::D];
            float* out = &Wphi[(size_t)n * 64 * PKB];
            if (m.phi_kind == WM_PHI_STRUCT) {
                for (int c = 0; c < F; ++c) out[c] = wr[c];
            } else {
                for (int c = 0; c < NT; ++c) {
                    double acc = 0.0;
                    for (int k = 0; k < tcp::DA; ++k) acc += (double)wr[k] * E[(size_t)c * tcp::DA + k];
                    out[c] = (float)acc;
                }
                for (int j = 0; j < P; ++j) {
                    double acc = 0.0;
                    for (int k = 0; k < tcp::DA; ++k) acc += (double)wr[k] * Wp[(size_t)k * P + j];
                    out[NT + j] = (float)acc;
                }
                double acc = 0.0;
                for (int k = 0; k < tcp::DA; ++k) acc += (double)wr[k] * bpv[k];
                out[NT + P] = (float)acc;
            }
            double bias = bs0[n];
            if (!transh)
                for (int k = 0; k < tcp::D; ++k) bias -= (double)Ws0[(size_t)n * K0 + k] * b2h[k];       // z_T arrives as u = z_T + b2
            out[NPSI - 1] = (float)bias;
        }
    }
    const tcp::SmemLayout L = tcp::smem_layout(m.n_types, (m.H + 15) / 16, m.phi_kind == WM_PHI_STRUCT, AKB == 1 && PKB == 1);
    if ((int)L.total > ctx->smem_optin) return WM_OK;
    const size_t n_slots = (size_t)(transh ? tcp::th_step_boxes(NC, AKB) : tcp::step_boxes(NC, AKB)) + tcp::scorer_boxes(PKB);
    std::vector<uint16_t> blob;
    bool ok = true;   // every weight finite in fp16
    blob.reserve(n_slots * tcp::HB_BYTES);
    // the MMA warp's order (tcp::stage_boxes): feature K-blocks of chunks 0 and 1, z K-blocks (0-3) of chunk 0, of chunk 1,
    // GEMM2 chunk 0, then per chunk i >= 2: features, z, GEMM2 chunk i - 1; last GEMM2 chunk NC - 1
    auto g1a = [&](int c) { for (int k = 0; k < AKB; ++k) ok &= append_slot(blob, W1f, 64 * AKB, c * 128, 64, k * 64, 64); };
    auto g1z = [&](int c) { for (int k = 0; k < 4; ++k) ok &= append_slot(blob, W1, K1, c * 128, 64, k * 64, 64); };
    auto g2 = [&](int c) {            // GEMM2 chunk c: the chunk's two hidden K-blocks x all 256 latent columns
        for (int k = 0; k < 2; ++k)
            for (int hrow = 0; hrow < 2; ++hrow) ok &= append_slot(blob, W2, hid, 64 * hrow, 128, c * 128 + k * 64, 64);
    };
    if (transh) {
        // u = W_w' f, then the translation W_d' f: N = 256, two slots per feature K-block (weight rows 0-63 / 128-191, 64-127 / 192-255)
        for (const std::vector<float>* M : {&Uf, &Df})
            for (int k = 0; k < AKB; ++k)
                for (int hrow = 0; hrow < 2; ++hrow) ok &= append_slot(blob, *M, 64 * AKB, 64 * hrow, 128, k * 64, 64);
        g1a(0); g1a(1); g1z(0); g1z(1);
    } else {
        g1a(0); g1a(1);
        // step boundary: z K-blocks 0 and 2 of chunks 0, 1 (stage_za), then K-blocks 1 and 3 (stage_zb)
        for (int half = 0; half < 2; ++half)
            for (int c = 0; c < 2; ++c)
                for (int k = half; k < 4; k += 2) ok &= append_slot(blob, W1, K1, c * 128, 64, k * 64, 64);
    }
    g2(0);
    for (int i = 2; i <= NC; ++i) {
        if (i < NC) { g1a(i); g1z(i); }
        g2(i - 1);
    }
    {
        static const std::vector<float> none;
        const std::vector<float>&Ws0 = forest ? none : get("Ws0"), &Ws1 = forest ? none : get("Ws1");
        const std::vector<float> zeros((size_t)tcp::SW * 64, 0.0f);
        for (int c = 0; c < 4; ++c) {     // scorer layer 1: phi features (PKB), hw, z (4 K-blocks)
            for (int k = 0; k < PKB; ++k) ok &= append_slot(blob, Wphi, 64 * PKB, c * 128, 64, k * 64, 64);
            if (forest) {
                for (int k = 0; k < 5; ++k) ok &= append_slot(blob, zeros, 64, c * 128, 64, 0, 0);
            } else {
                ok &= append_slot(blob, Ws0, K0, c * 128, 64, tcp::D + F, m.H);
                for (int k = 0; k < 4; ++k) ok &= append_slot(blob, Ws0, K0, c * 128, 64, k * 64, 64);
            }
        }
        for (int c = 0; c < 4; ++c)       // scorer layer 2: K = 512 = 8 K-blocks
            for (int kb = 0; kb < 8; ++kb)
                ok &= forest ? append_slot(blob, zeros, 64, c * 128, 64, 0, 0) : append_slot(blob, Ws1, tcp::SW, c * 128, 64, kb * 64, 64);
    }
    if (blob.size() * 2 != n_slots * 2 * tcp::HB_BYTES) {
        set_error("tcp_prepare: internal weight-image size mismatch");
        return WM_ERR_FORMAT;
    }
    if (!ok) return WM_OK;   // a weight beyond the fp16 range: this model stays on the fp32 kernel

    void* d_blob = nullptr;
    WM_CUDA_TRY(cudaMalloc(&d_blob, blob.size() * 2));
    ctx->allocs.push_back(d_blob);
    WM_CUDA_TRY(cudaMemcpy(d_blob, blob.data(), blob.size() * 2, cudaMemcpyHostToDevice));

    // tensor map over the image seen as rows of 64 16-bit values (128 B); one box = 128 rows.  The image is already
    // swizzled, so the map itself uses no swizzle.
    static_assert(sizeof(CUtensorMap) <= sizeof(m.tcp_tmap), "tensor map storage");
    CUtensorMap tm;
    {
        const int rc = encode_tmap_2d(&tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, d_blob, 64, blob.size() * 2 / 128, 128, 64, 64, false, "tcp_prepare");
        if (rc != WM_OK) return rc;
    }
    memcpy(m.tcp_tmap, &tm, sizeof(tm));
    {
        const void* fns[8] = {(const void*)tcp::wm_tcp_kernel<WM_PHI_MEAN, false, tcp::STEP_MLP_LN>, (const void*)tcp::wm_tcp_kernel<WM_PHI_MEAN, true, tcp::STEP_MLP_LN>,
                              (const void*)tcp::wm_tcp_kernel<WM_PHI_STRUCT, false, tcp::STEP_MLP_LN>, (const void*)tcp::wm_tcp_kernel<WM_PHI_STRUCT, true, tcp::STEP_MLP_LN>,
                              (const void*)tcp::wm_tcp_kernel<WM_PHI_MEAN, false, tcp::STEP_TRANSH>, (const void*)tcp::wm_tcp_kernel<WM_PHI_MEAN, true, tcp::STEP_TRANSH>,
                              (const void*)tcp::wm_tcp_kernel<WM_PHI_STRUCT, false, tcp::STEP_TRANSH>, (const void*)tcp::wm_tcp_kernel<WM_PHI_STRUCT, true, tcp::STEP_TRANSH>};
        const int base = (transh ? 4 : 0) + (m.phi_kind == WM_PHI_STRUCT ? 2 : 0);
        for (int e = 0; e < 2; ++e)
            WM_CUDA_TRY(cudaFuncSetAttribute(fns[base + e], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.total));
    }
    m.tcp_ok = 1;
    m.tcp_akb = AKB;
    m.tcp_pkb = PKB;
    return WM_OK;
}

int launch_tcp(wm_ctx* ctx, Workspace* ws, const CallArgs& a, cudaStream_t st) {
    (void)ws;
    const Model& m = ctx->m;
    tcp::Params p;
    p.hid = m.hidden; p.nc = m.hidden / 128; p.n_types = m.n_types; p.P = m.P; p.H = m.H;
    p.hw_ksteps = (m.H + 15) / 16;
    p.ln_eps = m.ln_eps;
    p.akb = m.tcp_akb; p.pkb = m.tcp_pkb;
    p.b2 = m.b2; p.gamma = m.gamma; p.beta = m.beta;
    p.bs1 = m.bs[1]; p.w3 = m.Wst[2]; p.bs2 = m.bs[2];
    if (m.ranker_kind == WM_RANKER_FOREST || m.phi_kind == WM_PHI_TYPED) p.bs1 = p.w3 = p.bs2 = m.zeros;   // (unused scorer, zero image)
    p.a = a;
    p.n_tiles = (int)((a.B + tcp::TMP - 1) / tcp::TMP);
    p.prof = trace::begin(st);
    CUtensorMap tm;
    memcpy(&tm, m.tcp_tmap, sizeof(tm));
    const tcp::SmemLayout L = tcp::smem_layout(m.n_types, p.hw_ksteps, m.phi_kind == WM_PHI_STRUCT, p.akb == 1 && p.pkb == 1);
    const int max_pairs = ctx->n_sms / 2;
    const int pairs = p.n_tiles < max_pairs ? p.n_tiles : max_pairs;
    const bool prefix_call = a.start || a.init_index || a.latents_out;
    const bool ps = m.phi_kind == WM_PHI_STRUCT;
    const dim3 grid(2 * pairs), block(tcp::THREADS);
#define WM_TCP_LAUNCH(PHI_, EXT_, STEP_) tcp::wm_tcp_kernel<PHI_, EXT_, STEP_><<<grid, block, L.total, st>>>(p, tm)
    if (m.kind == WM_KIND_TRANSH) {
        if (ps) { if (prefix_call) WM_TCP_LAUNCH(WM_PHI_STRUCT, true, tcp::STEP_TRANSH); else WM_TCP_LAUNCH(WM_PHI_STRUCT, false, tcp::STEP_TRANSH); }
        else { if (prefix_call) WM_TCP_LAUNCH(WM_PHI_MEAN, true, tcp::STEP_TRANSH); else WM_TCP_LAUNCH(WM_PHI_MEAN, false, tcp::STEP_TRANSH); }
    } else {
        if (ps) { if (prefix_call) WM_TCP_LAUNCH(WM_PHI_STRUCT, true, tcp::STEP_MLP_LN); else WM_TCP_LAUNCH(WM_PHI_STRUCT, false, tcp::STEP_MLP_LN); }
        else { if (prefix_call) WM_TCP_LAUNCH(WM_PHI_MEAN, true, tcp::STEP_MLP_LN); else WM_TCP_LAUNCH(WM_PHI_MEAN, false, tcp::STEP_MLP_LN); }
    }
#undef WM_TCP_LAUNCH
    WM_CUDA_TRY(cudaGetLastError());
    ctx->launches.fetch_add(1);
    trace::dump(p.prof, st);
    return WM_OK;
}

}  // namespace wm

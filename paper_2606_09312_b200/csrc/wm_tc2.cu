// K2 (tcgen05, CTA pair): fused persistent rollout + score kernel for the bf16 residual-MLP + LayerNorm model with
// d = 512, d_a = 256 (BASELINE.json cfg 3), sm_100a only.
//
// PAPER.md:162 Eq.8 / :166 — z_t = F(z_{t-1}, a_t) applied recurrently; :176 — masked steps leave z unchanged;
// :186-188 Eq.12 — y = G([z_T ; phi ; h]).  Parametrisation: BASELINE.json cfg 3.
//
// Why a pair: the fp32 master latent of a 128-candidate tile is 128 x 512 x 4 B = all 256 KB of one SM's tensor
// memory, leaving no room for GEMM1's accumulators.  A cluster of two CTAs (one TPC) therefore owns a tile of 128
// candidates together, 64 rows each, and the leader CTA issues `tcgen05.mma.cta_group::2` with M = 128, N = 256:
//   * each CTA's D tile is 64 rows x 256 columns held as 128 lanes x 128 columns (lane l: row l % 64, columns
//     128 * (l / 64) ...), so the fp32 latent of its 64 rows is 2 x 128 = 256 TMEM columns and IS the accumulator
//     of GEMM2 (the residual add is the MMA's accumulate); the other 256 columns are two GEMM1 accumulators;
//   * each CTA supplies its own 64 rows of the A operand (fp16 [z ; a], K-major 128B-swizzled 64-column K-blocks
//     in shared memory) and HALF of every B tile (128 of the 256 weight rows): the L2 -> SM weight stream per
//     candidate row is the same as for a 128-row single-CTA tile;
//   * the GELU epilogue writes the fp16 hidden chunk to shared memory (GEMM2's A operand; with 64 rows per CTA a
//     TMEM A operand would have to be duplicated across lane halves);
//   * weights stream through a ring of 16 KB half tiles filled by TMA (`cp.async.bulk.tensor ... cta_group::2`, whose
//     complete_tx lands on the LEADER's barrier for both halves) from a pre-tiled, pre-swizzled image laid out in
//     consumption order; MMA completion is multicast to both CTAs' barriers (`tcgen05.commit ... multicast`);
//   * epilogue / action warps of both CTAs arrive on the leader's barriers with cluster-scope release.
// Warp roles per CTA (512 threads): warps 0-7 epilogue (lane quadrant q = warp % 4: rows 32 (q & 1) + lane, N half
// q / 2; e = warp / 4: column half of the 128-column buffer), warps 8-10 and 12 action embedding, warp 11 TMEM
// allocator, warp 13 tile schedule + TMA producer, warp 15 MMA issuer (leader CTA only).
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

namespace tc2 {

using namespace ptx;

constexpr int TMP = 128;           // candidates per pair tile (MMA M)
constexpr int TMR = 64;            // rows per CTA
constexpr int D = 512;             // latent width
constexpr int DA = 256;            // action-embedding width
constexpr int SW = 1024;           // scorer hidden width (both hidden layers)
constexpr int KB_BYTES = 8192;     // one A K-block: [64 rows x 64 cols] fp16, SW128 K-major
constexpr int BT_BYTES = 16384;    // one B half tile: [128 weight rows x 64 cols] fp16, SW128 K-major (= ring stage)
constexpr int NSTAGE = 4;            // ring depth: the stand-alone issue loop reaches 66 % of the pipe with 3 stages, 85 % with 4
constexpr int A1_KB = 10;          // z: 0-7, action / phi features: 8-9 (akb, pkb <= 2)
constexpr int H_KB = 4;            // K-blocks of one hidden chunk buffer (256 columns)
constexpr int HWK_BYTES = 2048;    // hw operand: one [64 x 16] no-swizzle K-major tile per K = 16 step
constexpr int THREADS = 512;
// The MMA issuer is one serial instruction stream (~70 instructions per ring stage) racing the stage's 256 tensor
// cycles, so its scheduler (SMSP 3 = warps 3, 7, 11, 15) carries as little else as possible: the fourth action warp is
// warp 12, and warp 11 is the TMEM allocator, idle after setup.
constexpr int EPI_WARP0 = 0, ACT_WARP0 = 8, ALLOC_WARP = 11, PROD_WARP = 13, MMA_WARP = 15;
__device__ __forceinline__ int action_index(int warp) { return warp == 12 ? 3 : (warp >= 8 && warp <= 10) ? warp - 8 : -1; }
constexpr int MAX_TYPES = 64, MAX_P = 8, MAX_H = 64, MAX_HID = 1024;
constexpr int G2_STAGES = 8;                              // per 256-column hidden chunk: GEMM2; GEMM1 takes akb + 8
// scorer: layer 1 (4 x (pkb phi features, hw, 8 z)), layer 2 (2 rounds x 16 x 2)
__host__ __device__ inline int sc_stages(int pkb) { return 4 * (pkb + 9) + 2 * 32; }

enum {
    B_FULL = 0,                    // [NSTAGE] TMA (both CTAs) -> leader's MMA warp
    B_EMPTY = B_FULL + NSTAGE,     // [NSTAGE] MMA commit (multicast) -> each CTA's producer
    B_D1FULL = B_EMPTY + NSTAGE,   // [2] MMA commit -> epilogue: accumulator buffer b filled
    B_HREADY = B_D1FULL + 2,       // [2] epilogue (both CTAs) -> leader MMA: buffer b read, fp16 hidden written
    B_HFREE = B_HREADY + 2,        // [2] MMA commit -> epilogue: hidden buffer b no longer read
    B_D2FULL = B_HFREE + 2,        // MMA commit -> epilogue: GEMM2 of the step done
    B_ZREADY,                      // epilogue (both CTAs) -> leader MMA: z written
    B_AFREE,                       // MMA commit -> action warps: a-part of A1 no longer read
    B_AREADY,                      // action warps (both CTAs) -> leader MMA: a-part written
    B_SFULL,                       // [2] schedule slot filled (CTA-local)
    B_SEMPTY = B_SFULL + 2,        // [2] schedule slot consumed (CTA-local)
    B_COUNT = B_SEMPTY + 2
};

struct Params {
    int hid, nc, n_types, P, H, hw_ksteps;
    int akb, pkb;               // K-blocks of the folded action features f_t (1 or 2) and of the phi features (1 or 2)
    float ln_eps;
    const float *b2, *gamma, *beta;
    const float *bs1, *w3, *bs2;
    CallArgs a;
    int n_tiles;
    unsigned long long* prof;   // developer trace buffer (wm_trace.cuh), null in a normal build
};

struct SmemLayout {
    uint32_t a1, hbuf, ring, hwk, lp, ids, cnt, b1, red, bars, sched, tmem_slot, total;
};

__host__ __device__ inline SmemLayout smem_layout(int n_types, int hid, int hw_ksteps) {
    SmemLayout L;
    uint32_t o = 0;
    L.a1 = o; o += A1_KB * KB_BYTES;
    L.hbuf = o; o += 2 * H_KB * KB_BYTES;
    L.ring = o; o += NSTAGE * BT_BYTES;
    L.hwk = o; o += (uint32_t)hw_ksteps * HWK_BYTES;
    L.lp = o; L.ids = o;                               // (unused since the action features are folded)
    L.cnt = o; o += TMR * (uint32_t)n_types;          // u8 counts, row-major [64][n_types]
    o = (o + 15) & ~15u;
    L.b1 = o; o += 3 * D * 4;                          // b2, gamma, beta (LayerNorm: on the critical path; b1 is __ldg)
    L.red = o; o += 4 * TMR * 8;                       // [4 column parts][64 rows] float2
    L.bars = o; o += B_COUNT * 8;
    L.sched = o; o += 2 * 8;
    L.tmem_slot = o; o += 16;
    L.total = o;
    return L;
}

// Static tile schedule: pair `pair` of `np` pairs takes, in round `it`, tile it*np + pair on even rounds and
// it*np + (np-1-pair) on odd rounds (tiles are sorted longest first: the serpentine evens out the step totals).
__device__ __forceinline__ int tile_of(int it, int pair, int np, int n_tiles) {
    const int idx = it * np + ((it & 1) ? np - 1 - pair : pair);
    return idx < n_tiles ? idx : -1;
}

// PHI = WM_PHI_MEAN | WM_PHI_STRUCT (what the action warps write into the phi K-blocks at the end of a tile); EXT = the
// prefix-latent-reuse calls (wm_rollout_latents / wm_rollout_score_from: per-candidate start and initial-latent row,
// latents stored), compiled out of the literal path — as in wm_tcp_kernel.
template <int PHI, bool EXT>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(THREADS, 1)
wm_tc2_kernel(const Params p, const __grid_constant__ CUtensorMap tmap) {
    extern __shared__ __align__(1024) uint8_t smem[];
    const SmemLayout L = smem_layout(p.n_types, p.hid, p.hw_ksteps);
    const uint32_t s_base = smem_u32(smem);
    const uint32_t s_a1 = s_base + L.a1, s_h = s_base + L.hbuf, s_ring = s_base + L.ring, s_bars = s_base + L.bars;
    auto bar = [&](int i) -> uint32_t { return s_bars + 8u * (uint32_t)i; };
    volatile int* s_sched = reinterpret_cast<volatile int*>(smem + L.sched);   // [2][2]: tile, nsteps
    float* s_ln = reinterpret_cast<float*>(smem + L.b1);                      // [3][512]: b2, gamma, beta
    float2* s_red = reinterpret_cast<float2*>(smem + L.red);                  // [4][64]

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();          // 0 = leader (issues the MMAs)
    const int pair = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;
    const int NC = p.nc;
    const int AKB = p.akb, PKB = p.pkb;
    const int ROLL_STAGES = NC * (AKB + 8 + G2_STAGES);

    // ---- one-time setup
    if (threadIdx.x == 0) {
        for (int i = 0; i < NSTAGE; ++i) { mbar_init(bar(B_FULL + i), 1); mbar_init(bar(B_EMPTY + i), 1); }
        for (int i = 0; i < 2; ++i) {
            mbar_init(bar(B_D1FULL + i), 1);
            mbar_init(bar(B_HREADY + i), 16);
            mbar_init(bar(B_HFREE + i), 1);
            mbar_init(bar(B_SFULL + i), 1);
            mbar_init(bar(B_SEMPTY + i), 13);
        }
        mbar_init(bar(B_D2FULL), 1);
        mbar_init(bar(B_ZREADY), 16);
        mbar_init(bar(B_AFREE), 1);
        mbar_init(bar(B_AREADY), 8);
        fence_barrier_init();
        fence_proxy_async();
    }
    if (warp == ALLOC_WARP) tmem_alloc2(s_base + L.tmem_slot, 512);
    for (int i = threadIdx.x; i < D; i += THREADS) {
        s_ln[i] = __ldg(p.b2 + i);
        s_ln[D + i] = __ldg(p.gamma + i);
        s_ln[2 * D + i] = __ldg(p.beta + i);
    }
    {
        // the hw operand tile is only ever written in its first columns: clear it once so unread bytes are not NaNs
        uint32_t* hwk = reinterpret_cast<uint32_t*>(smem + L.hwk);
        for (int i = threadIdx.x; i < p.hw_ksteps * HWK_BYTES / 4; i += THREADS) hwk[i] = 0u;
    }
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();      // both CTAs' barriers are initialised before anyone arrives remotely / multicasts
    tc_fence_after();
    const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(smem + L.tmem_slot);
    const uint32_t T_Z = tmem_base;                 // fp32 latent / GEMM2 accumulators: two 128-column N tiles
    const uint32_t T_D1 = tmem_base + 256;          // two 128-column GEMM1 accumulators (256 hidden units each)
    // EXT calls that store latents and rank nothing skip the scorer in every role
    const bool rank_it = !EXT || p.a.scores_out != nullptr;

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
                const int roll_total = nsteps * ROLL_STAGES, total = roll_total + (rank_it ? sc_stages(PKB) : 0);
                int src = 0;
                for (int i = 0; i < total; ++i) {
                    if (i == roll_total) src = ROLL_STAGES;
                    else if (i < roll_total && src == ROLL_STAGES) src = 0;
                    WM_TRACE(30);
                    mbar_wait(bar(B_EMPTY + stage), ph ^ 1);
                    WM_TRACE(31);
                    // the leader's barrier collects both halves of the [256 x 64] tile
                    if (rank == 0) mbar_arrive_expect_tx(bar(B_FULL + stage), 2 * BT_BYTES);
                    tma_load_2sm(s_ring + stage * BT_BYTES, &tmap, 0, 128 * (2 * src + (int)rank), bar(B_FULL + stage));
                    ++src;
                    if (++stage == NSTAGE) { stage = 0; ph ^= 1; }
                }
            }
            __syncwarp();
        }
    } else if (warp == MMA_WARP) {
        // =============================================================== MMA issuer (leader CTA; the peer's warp only
        // follows the schedule so that both CTAs' slot barriers have the same arrival count)
        // Everything this warp computes with is made PROVABLY warp-uniform (a warp reduction's result lives in a uniform
        // register): ptxas then keeps descriptors, ring state and loop counters in the uniform datapath instead of
        // moving them there (R2UR) for every MMA — the issuing warp is one instruction stream, its latency per stage
        // competes with the stage's 256 tensor cycles.
        const uint32_t T_Z = __reduce_max_sync(0xffffffffu, tmem_base);
        const uint32_t T_D1 = T_Z + 256;
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
        // Ring consumer state.  `ready` = the current stage's full barrier is already known complete: it was probed
        // (non-blocking test_wait) before the previous stage's MMAs were issued, so the probe's latency overlaps that
        // issue instead of preceding this one.  b_lo = descriptor low word of the current ring slot.
        const uint32_t ring_lo0 = smem_desc_lo(s_ring);
        uint32_t b_lo = ring_lo0;
        bool ready = false;
        auto acquire_stage = [&]() {       // returns with the current stage's data landed; probes the next stage
            WM_TRACE(1);
            if (!ready) mbar_wait_warp(bar(B_FULL + stage), ph);
            WM_TRACE(2);
            tc_fence_after();
            const uint32_t nst = stage + 1 == NSTAGE ? 0u : stage + 1;
            ready = __all_sync(0xffffffffu, mbar_test_wait(bar(B_FULL + nst), nst == 0 ? ph ^ 1u : ph));
        };
        auto advance = [&]() {
            __syncwarp();
            b_lo += BT_BYTES >> 4;
            if (++stage == NSTAGE) { stage = 0; ph ^= 1; b_lo = ring_lo0; }
        };
        // one ring stage = one [256 x 64] B tile against the [64(+64) x 64] A K-block at a_tile: 4 MMAs of K = 16
        auto stage_ss = [&](uint32_t d_tmem, uint32_t a_tile, bool first) {
            const uint32_t a_lo = smem_desc_lo(a_tile);
            acquire_stage();
            if (elect_one()) {
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    mma_ss2(d_tmem, desc_of(a_lo + 2u * j), desc_of(b_lo + 2u * j), IDESC2, (first && j == 0) ? 0u : 1u);
                mma_commit2(bar(B_EMPTY + stage));
            }
            WM_TRACE(3);
            advance();
        };
        // stage = the hw weight tile: hw_ksteps MMAs whose A operand is the no-swizzle [64 x 16] hw tile
        auto stage_hw = [&](uint32_t d_tmem) {
            acquire_stage();
            if (elect_one()) {
                for (int j = 0; j < p.hw_ksteps; ++j)
                    mma_ss2(d_tmem, smem_desc_nosw(s_hwk + j * HWK_BYTES), desc_of(b_lo + 2u * j), IDESC2, 1u);
                mma_commit2(bar(B_EMPTY + stage));
            }
            advance();
        };
        auto commit = [&](int barrier) {
            if (elect_one()) mma_commit2(bar(barrier));
            __syncwarp();
        };
        // 256-column chunk of W [z ; a (; hw)] into accumulator b: K-blocks a/phi (8-11), [hw], z (0-7)
        auto gemm_a1 = [&](int b, bool first_chunk, bool last_chunk, bool with_hw) {
            wait_h(b);
            const uint32_t d = T_D1 + 128u * b;
            if (first_chunk) { WM_TRACE(20); mbar_wait_warp(bar(B_AREADY), n_a & 1); WM_TRACE(21); ++n_a; tc_fence_after(); }
            const int nk = with_hw ? PKB : AKB;      // scorer layer 1: phi features; rollout: action features
#pragma unroll 1
            for (int k = 0; k < nk; ++k) stage_ss(d, s_a1 + (8 + k) * KB_BYTES, k == 0);
            if (with_hw) stage_hw(d);
            if (last_chunk) commit(B_AFREE);
            if (first_chunk) { WM_TRACE(22); mbar_wait_warp(bar(B_ZREADY), n_z & 1); WM_TRACE(23); ++n_z; tc_fence_after(); }
#pragma unroll 1
            for (int k = 0; k < 8; ++k) stage_ss(d, s_a1 + k * KB_BYTES, false);
            commit(B_D1FULL + b);
            pend[b] = true;
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
                // Step boundary: the a K-blocks of chunk 0 AND chunk 1 depend only on a_{t+1} and both GEMM1 accumulators
                // are free, so both a-parts are issued before the wait for z' (pipe drain + LayerNorm is the serial
                // section of a step); then the z K-blocks of chunks 0 and 1.  (NC >= 2.)
                wait_h(0);
                wait_h(1);
                WM_TRACE(20); mbar_wait_warp(bar(B_AREADY), n_a & 1); WM_TRACE(21); ++n_a; tc_fence_after();
#pragma unroll 1
                for (int b = 0; b < 2; ++b)
#pragma unroll 1
                    for (int k = 0; k < AKB; ++k) stage_ss(T_D1 + 128u * b, s_a1 + (8 + k) * KB_BYTES, k == 0);
                if (NC == 2) commit(B_AFREE);
                WM_TRACE(22); mbar_wait_warp(bar(B_ZREADY), n_z & 1); WM_TRACE(23); ++n_z; tc_fence_after();
#pragma unroll 1
                for (int b = 0; b < 2; ++b) {
#pragma unroll 1
                    for (int k = 0; k < 8; ++k) stage_ss(T_D1 + 128u * b, s_a1 + k * KB_BYTES, false);
                    commit(B_D1FULL + b);
                    pend[b] = true;
                }
                auto gemm2 = [&](int c) {                                        // GEMM2 chunk c: Z += H[b] W2^T
                    const int b = c & 1;
                    wait_h(b);
#pragma unroll 1
                    for (int kb = 0; kb < H_KB; ++kb) {
                        stage_ss(T_Z, s_h + (b * H_KB + kb) * KB_BYTES, false);
                        stage_ss(T_Z + 128u, s_h + (b * H_KB + kb) * KB_BYTES, false);
                    }
                    commit(B_HFREE + b);
                    if (c == NC - 1) commit(B_D2FULL);
                };
                gemm2(0);
#pragma unroll 1
                for (int i = 2; i <= NC; ++i) {
                    if (i < NC) gemm_a1(i & 1, false, i == NC - 1, false);       // GEMM1 chunk i
                    gemm2(i - 1);
                }
            }
            if (!rank_it) {   // nothing to rank: only take the terminal latent's ZREADY so the phase count stays in step
                mbar_wait_warp(bar(B_ZREADY), n_z & 1);
                ++n_z;
                continue;
            }
            // ---- scorer layer 1: four 256-column chunks of gelu(Ws0 [z_T; phi; hw] + bs0).  Chunks 0, 1 land in the
            // hidden buffers; chunks 2, 3 are written over A1's z K-blocks once every layer-1 MMA has completed.
#pragma unroll 1
            for (int c = 0; c < 4; ++c) gemm_a1(c & 1, c == 0, c == 3, true);
            // ---- scorer layer 2, K = 1024 in K-chunks (H[0], H[1], A1 kb 0-3, A1 kb 4-7), N = 1024 in two rounds of
            // two 256-column N tiles: round 0 into the (dead) latent columns, round 1 into the GEMM1 accumulators
#pragma unroll 1
            for (int round = 0; round < 2; ++round) {
                const uint32_t d0 = round == 0 ? T_Z : T_D1;
#pragma unroll 1
                for (int kc = 0; kc < 4; ++kc) {
                    if (round == 0 && kc >= 2) wait_h(kc - 2);     // h1 chunk kc written over A1 (and D1[kc-2] read)
                    const uint32_t a_base = kc < 2 ? s_h + kc * H_KB * KB_BYTES : s_a1 + (kc - 2) * 4 * KB_BYTES;
#pragma unroll 1
                    for (int kb = 0; kb < 4; ++kb) {
                        stage_ss(d0, a_base + kb * KB_BYTES, kc == 0 && kb == 0);
                        stage_ss(d0 + 128u, a_base + kb * KB_BYTES, kc == 0 && kb == 0);
                    }
                    if (round == 1 && kc < 2) commit(B_HFREE + kc);
                }
                if (round == 0) {
                    commit(B_D2FULL);
                } else {
                    commit(B_D1FULL + 0);
                    commit(B_D1FULL + 1);
                    pend[0] = pend[1] = true;
                }
            }
        }
        __syncwarp();
    }
    else if (warp >= EPI_WARP0 && warp < ACT_WARP0) {
        // =============================================================== epilogue warps (GELU / LayerNorm / scorer)
        const int q = warp & 3, e = (warp - EPI_WARP0) >> 2;
        const int rh = q & 1, nh = q >> 1;
        const int row = 32 * rh + lane;                 // row of this CTA's 64
        const int part = 2 * nh + e;                    // this thread's 64-column quarter of every 256-column tile
        const uint32_t lane_off = (uint32_t)(32 * q) << 16;
        uint8_t* a1 = smem + L.a1;
        uint8_t* hb = smem + L.hbuf;
        const uint32_t r_hready0 = mapa(bar(B_HREADY), 0), r_hready1 = mapa(bar(B_HREADY + 1), 0);
        const uint32_t r_zready = mapa(bar(B_ZREADY), 0);
        uint32_t n_d1[2] = {0, 0}, n_d2 = 0, n_hw[2] = {0, 0};
        const float inv_d = 1.0f / (float)D;
        WM_TRACE_DECL(p.prof, 2)
        // write 32 consecutive z columns of this row (N tile j, 32-column half `half` of the thread's quarter):
        // fp32 -> TMEM, fp16 -> A1 K-block 4 j + part (when `to_smem`)
        auto put_z = [&](int j, int half, const uint32_t (&v)[32], bool to_smem) {
            tmem_st32(T_Z + 128u * j + 64u * e + 32u * half + lane_off, v);
            if (to_smem) {
                uint8_t* kb = a1 + (4 * j + part) * KB_BYTES;
#pragma unroll
                for (int ch = 0; ch < 4; ++ch) {
                    uint4 o;
                    o.x = pack_f16(__uint_as_float(v[8 * ch + 0]), __uint_as_float(v[8 * ch + 1]));
                    o.y = pack_f16(__uint_as_float(v[8 * ch + 2]), __uint_as_float(v[8 * ch + 3]));
                    o.z = pack_f16(__uint_as_float(v[8 * ch + 4]), __uint_as_float(v[8 * ch + 5]));
                    o.w = pack_f16(__uint_as_float(v[8 * ch + 6]), __uint_as_float(v[8 * ch + 7]));
                    *reinterpret_cast<uint4*>(kb + sw128_off(row, 4 * half + ch)) = o;
                }
            }
        };
        auto publish = [&](uint32_t leader_bar, bool tmem_written) {
            if (tmem_written) tmem_st_wait();
            fence_proxy_async();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_remote(leader_bar);
        };
        auto wait_d1 = [&](int b) {
            mbar_wait(bar(B_D1FULL + b), n_d1[b] & 1);
            ++n_d1[b];
            tc_fence_after();
        };
        // GELU over this thread's 64 columns of accumulator b (the bias is already in the accumulator: it rides on the
        // constant-1 feature column) -> fp16 row of the K-block at dst (SW128).  Packed fp16x2 arithmetic (gelu2_h2).
        auto gelu_to_smem = [&](int b, uint8_t* dst) {
            uint32_t v0[32], v1[32];
            tmem_ld32(T_D1 + 128u * b + 64u * e + lane_off, v0);
            tmem_ld32(T_D1 + 128u * b + 64u * e + 32u + lane_off, v1);
            tmem_ld_wait();
#pragma unroll
            for (int ch = 0; ch < 4; ++ch)
                *reinterpret_cast<uint4*>(dst + sw128_off(row, ch)) =
                    make_uint4(gelu2_h2(__uint_as_float(v0[8 * ch + 0]), __uint_as_float(v0[8 * ch + 1])),
                               gelu2_h2(__uint_as_float(v0[8 * ch + 2]), __uint_as_float(v0[8 * ch + 3])),
                               gelu2_h2(__uint_as_float(v0[8 * ch + 4]), __uint_as_float(v0[8 * ch + 5])),
                               gelu2_h2(__uint_as_float(v0[8 * ch + 6]), __uint_as_float(v0[8 * ch + 7])));
#pragma unroll
            for (int ch = 0; ch < 4; ++ch)
                *reinterpret_cast<uint4*>(dst + sw128_off(row, 4 + ch)) =
                    make_uint4(gelu2_h2(__uint_as_float(v1[8 * ch + 0]), __uint_as_float(v1[8 * ch + 1])),
                               gelu2_h2(__uint_as_float(v1[8 * ch + 2]), __uint_as_float(v1[8 * ch + 3])),
                               gelu2_h2(__uint_as_float(v1[8 * ch + 4]), __uint_as_float(v1[8 * ch + 5])),
                               gelu2_h2(__uint_as_float(v1[8 * ch + 6]), __uint_as_float(v1[8 * ch + 7])));
            publish(b == 0 ? r_hready0 : r_hready1, false);
        };
        // hidden chunk into hidden buffer b (waits until GEMM2 no longer reads the buffer's previous contents)
        auto gelu_to_h = [&](int b) {
            WM_TRACE(40);
            wait_d1(b);
            WM_TRACE(41);
            mbar_wait(bar(B_HFREE + b), (n_hw[b] & 1) ^ 1);
            ++n_hw[b];
            WM_TRACE(42);
            gelu_to_smem(b, hb + (b * H_KB + part) * KB_BYTES);
            WM_TRACE(43);
        };

        for (uint32_t it = 0;; ++it) {
            const uint32_t slot = it & 1;
            mbar_wait(bar(B_SFULL + slot), (it >> 1) & 1);
            const int tile = s_sched[slot * 2 + 0], nsteps = s_sched[slot * 2 + 1];
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(B_SEMPTY + slot));
            if (tile < 0) break;
            int cand, len, seg;
            row_meta(p.a, (int64_t)tile * TMP + TMR * (int)rank + row, cand, len, seg, false);
            // prefix-latent reuse: the rollout covers positions [st, len) and starts from the row init_index names
            const int st = EXT ? row_start(p.a, cand, len) : 0, rem = len - st;
            const size_t zrow = EXT ? row_init(p.a, cand, seg) : (size_t)seg;

            // ---- z_0 (the task's initial latent; or the banked latent after the first st steps)
#pragma unroll 1
            for (int jh = 0; jh < 4; ++jh) {
                const int j = jh >> 1, half = jh & 1;
                const int col0 = 256 * j + 64 * part + 32 * half;
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
                put_z(j, half, v, true);
            }
            publish(r_zready, true);

            for (int t = 0; t < nsteps; ++t) {
                for (int c = 0; c < NC; ++c) gelu_to_h(c & 1);
                // ---- LayerNorm(z + W2 h + b2): the accumulator already holds z + W2 h
                WM_TRACE(50);
                mbar_wait(bar(B_D2FULL), n_d2 & 1);
                WM_TRACE(51);
                ++n_d2;
                tc_fence_after();
                float2 s1v = make_float2(0.0f, 0.0f), s2v = make_float2(0.0f, 0.0f);
#pragma unroll 1
                for (int jh = 0; jh < 4; ++jh) {
                    const int j = jh >> 1, half = jh & 1;
                    const int col0 = 256 * j + 64 * part + 32 * half;
                    uint32_t v[32];
                    tmem_ld32(T_Z + 128u * j + 64u * e + 32u * half + lane_off, v);
                    tmem_ld_wait();
                    const float4* b2v = reinterpret_cast<const float4*>(s_ln + col0);
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const float4 bb = b2v[i];
                        const float2 x0 = __fadd2_rn(make_float2(__uint_as_float(v[4 * i]), __uint_as_float(v[4 * i + 1])),
                                                     make_float2(bb.x, bb.y));
                        const float2 x1 = __fadd2_rn(make_float2(__uint_as_float(v[4 * i + 2]), __uint_as_float(v[4 * i + 3])),
                                                     make_float2(bb.z, bb.w));
                        s1v = __fadd2_rn(s1v, __fadd2_rn(x0, x1));
                        s2v = __ffma2_rn(x0, x0, s2v);
                        s2v = __ffma2_rn(x1, x1, s2v);
                    }
                }
                s_red[part * TMR + row] = make_float2(s1v.x + s1v.y, s2v.x + s2v.y);
                named_bar_sync(1 + rh, 128);
                float s1 = 0.0f, s2 = 0.0f;
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const float2 o = s_red[k * TMR + row];
                    s1 += o.x; s2 += o.y;
                }
                named_bar_sync(1 + rh, 128);   // all four parts have read s_red before the next LayerNorm rewrites it
                const float mean = s1 * inv_d;
                const float var = fmaxf(s2 * inv_d - mean * mean, 0.0f);
                const float rstd = rsqrtf(var + p.ln_eps);
                const bool live = t < rem;     // masked steps leave the state unchanged
                float4* lat = nullptr;     // wm_rollout_latents: z after this step (or only the terminal one: [B, d])
                if (EXT && p.a.latents_out && live) {
                    if (!p.a.latents_terminal)
                        lat = reinterpret_cast<float4*>(p.a.latents_out + ((size_t)cand * p.a.T_max + st + t) * D);
                    else if (st + t == len - 1)
                        lat = reinterpret_cast<float4*>(p.a.latents_out + (size_t)cand * D);
                }
#pragma unroll 1
                for (int jh = 0; jh < 4; ++jh) {
                    const int j = jh >> 1, half = jh & 1;
                    const int col0 = 256 * j + 64 * part + 32 * half;
                    uint32_t v[32];
                    tmem_ld32(T_Z + 128u * j + 64u * e + 32u * half + lane_off, v);
                    tmem_ld_wait();
                    const float4* b2v = reinterpret_cast<const float4*>(s_ln + col0);
                    const float4* gv = reinterpret_cast<const float4*>(s_ln + D + col0);
                    const float4* bev = reinterpret_cast<const float4*>(s_ln + 2 * D + col0);
                    const float2 rs2 = make_float2(rstd, rstd), mr2 = make_float2(-mean * rstd, -mean * rstd);
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const float4 bb = b2v[i], gg = gv[i], be = bev[i];
                        float2 x0 = __fadd2_rn(make_float2(__uint_as_float(v[4 * i]), __uint_as_float(v[4 * i + 1])),
                                               make_float2(bb.x, bb.y));
                        float2 x1 = __fadd2_rn(make_float2(__uint_as_float(v[4 * i + 2]), __uint_as_float(v[4 * i + 3])),
                                               make_float2(bb.z, bb.w));
                        x0 = __ffma2_rn(__ffma2_rn(x0, rs2, mr2), make_float2(gg.x, gg.y), make_float2(be.x, be.y));
                        x1 = __ffma2_rn(__ffma2_rn(x1, rs2, mr2), make_float2(gg.z, gg.w), make_float2(be.z, be.w));
                        v[4 * i] = __float_as_uint(x0.x); v[4 * i + 1] = __float_as_uint(x0.y);
                        v[4 * i + 2] = __float_as_uint(x1.x); v[4 * i + 3] = __float_as_uint(x1.y);
                    }
                    // frozen rows: the fp16 copy (GEMM1 operand, scorer input) keeps the terminal latent; their
                    // fp32 master is never read again
                    put_z(j, half, v, live);
                    if (EXT && lat) {
#pragma unroll
                        for (int i = 0; i < 8; ++i)
                            lat[(col0 >> 2) + i] = make_float4(__uint_as_float(v[4 * i]), __uint_as_float(v[4 * i + 1]),
                                                               __uint_as_float(v[4 * i + 2]), __uint_as_float(v[4 * i + 3]));
                    }
                }
                publish(r_zready, true);
                WM_TRACE(52);
            }

            if (!rank_it) continue;
            // ---- scorer layer 1 -> h1 (fp16): chunks 0, 1 into the hidden buffers ...
            gelu_to_h(0);
            gelu_to_h(1);
            // ... chunks 2, 3 over A1's z K-blocks, once every layer-1 MMA (the readers of A1) has completed
            wait_d1(0);
            wait_d1(1);
            gelu_to_smem(0, a1 + part * KB_BYTES);
            gelu_to_smem(1, a1 + (4 + part) * KB_BYTES);
            // ---- scorer layer 2 + output dot product: N tiles 0, 1 in the latent columns, 2, 3 in the accumulators
            float acc = 0.0f;
            auto dot32 = [&](uint32_t taddr, int n0) {
                uint32_t v[32];
                tmem_ld32(taddr, v);
                tmem_ld_wait();
#pragma unroll
                for (int i = 0; i < 32; ++i)
                    acc = fmaf(gelu_fast(__uint_as_float(v[i]) + __ldg(p.bs1 + n0 + i)), __ldg(p.w3 + n0 + i), acc);
            };
            mbar_wait(bar(B_D2FULL), n_d2 & 1);
            ++n_d2;
            tc_fence_after();
#pragma unroll 1
            for (int jh = 0; jh < 4; ++jh) {
                const int j = jh >> 1, half = jh & 1;
                dot32(T_Z + 128u * j + 64u * e + 32u * half + lane_off, 256 * j + 64 * part + 32 * half);
            }
#pragma unroll 1
            for (int b = 0; b < 2; ++b) {
                wait_d1(b);
                dot32(T_D1 + 128u * b + 64u * e + lane_off, 512 + 256 * b + 64 * part);
                dot32(T_D1 + 128u * b + 64u * e + 32u + lane_off, 512 + 256 * b + 64 * part + 32);
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_remote(b == 0 ? r_hready0 : r_hready1);
            }
            s_red[part * TMR + row] = make_float2(acc, 0.0f);
            named_bar_sync(1 + rh, 128);
            if (part == 0 && cand >= 0 && (!EXT || p.a.scores_out))
                p.a.scores_out[cand] = (s_red[row].x + s_red[TMR + row].x) + (s_red[2 * TMR + row].x + s_red[3 * TMR + row].x) +
                                       __ldg(p.bs2);
            named_bar_sync(1 + rh, 128);   // s_red is reused by the next tile's first LayerNorm
        }
    }
    else if (action_index(warp) >= 0) {
        // =============================================================== action-feature warps
        // warp aw owns rows [16 aw, 16 aw + 16), one row per lane 0-15 (lanes 16-31 help clearing).  Per step a row's
        // action enters GEMM1 as the feature row f_t = [onehot(id) (NT) | log2 p_j (P) | 1] of K-block 8 (and 9 when
        // NT + P + 1 > 64): the host folds E, W_p, b_p and b1 into GEMM1's a-columns (tc2_prepare), so the embedding
        // a_t = E[id] + W_p log2 p + b_p is never formed.
        const int aw = action_index(warp);
        const int row = 16 * aw + (lane & 15);
        const bool row_lane = lane < 16;
        uint8_t* a1 = smem + L.a1;
        uint8_t* s_cnt = smem + L.cnt;
        const uint32_t r_aready = mapa(bar(B_AREADY), 0);
        const int P = p.P, NT = p.n_types;
        uint32_t n_w = 0;
        // 16-bit feature store: column c of this row in K-blocks 8 ..
        auto put = [&](int c, uint32_t h16) {
            *reinterpret_cast<uint16_t*>(a1 + (8 + (c >> 6)) * KB_BYTES + sw128_off(row, (c & 63) >> 3) + (c & 7) * 2) = (uint16_t)h16;
        };
        // lanes l and l + 16 clear the row's K-blocks 8, 9 (one each)
        auto clear_row = [&]() {
            const int hk = 8 + (lane >> 4);
#pragma unroll
            for (int ch = 0; ch < 8; ++ch)
                *reinterpret_cast<uint4*>(a1 + hk * KB_BYTES + sw128_off(row, ch)) = make_uint4(0u, 0u, 0u, 0u);
        };
        for (uint32_t it = 0;; ++it) {
            const uint32_t slot = it & 1;
            mbar_wait(bar(B_SFULL + slot), (it >> 1) & 1);
            const int tile = s_sched[slot * 2 + 0], nsteps = s_sched[slot * 2 + 1];
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(B_SEMPTY + slot));
            if (tile < 0) break;
            int cand = -1, len = 0, seg = 0;
            if (row_lane) {
                row_meta(p.a, (int64_t)tile * TMP + TMR * (int)rank + row, cand, len, seg, false);
                for (int c = 0; c < NT; ++c) s_cnt[row * NT + c] = 0;
            }
            float slp[MAX_P], smx[MAX_P];    // per parameter slot: running sum and (WM_PHI_STRUCT) maximum of log2 p
#pragma unroll
            for (int j = 0; j < MAX_P; ++j) slp[j] = smx[j] = 0.0f;
            // one action of this row: type id (clamped), log2 of its parameters, phi statistics
            auto take = [&](int pos, float (&lp)[MAX_P]) -> int {
                int id = __ldg(p.a.action_ids + (size_t)cand * p.a.T_max + pos);
                if (id < 0 || id >= NT) {
                    atomicOr(p.a.fault, WM_FAULT_TYPE);
                    id = id < 0 ? 0 : NT - 1;
                }
                const int32_t* pp = p.a.action_params + ((size_t)cand * p.a.T_max + pos) * P;
#pragma unroll
                for (int j = 0; j < MAX_P; ++j) {
                    if (j < P) {
                        int prm = __ldg(pp + j);
                        if (prm < 1) {
                            atomicOr(p.a.fault, WM_FAULT_PARAM);
                            prm = 1;
                        }
                        lp[j] = log2f((float)prm);
                        slp[j] += lp[j];
                        if (PHI == WM_PHI_STRUCT) smx[j] = fmaxf(smx[j], lp[j]);
                    }
                }
                s_cnt[row * NT + id] += 1;
                return id;
            };
            // prefix-latent reuse: positions [0, st) only feed phi; scanned in position order BEFORE the first rollout step
            // (the running sums then see the positions in the literal call's order: bit-identical scores)
            const int st = (EXT && row_lane) ? row_start(p.a, cand, len) : 0;
            if (EXT && p.a.start) {
                for (int pos = 0; pos < st; ++pos) {
                    float lp[MAX_P];
#pragma unroll
                    for (int j = 0; j < MAX_P; ++j) lp[j] = 0.0f;
                    take(pos, lp);
                }
                __syncwarp();
            }
            int prev_id = -1;

            for (int t = 0; t < nsteps; ++t) {
                // read the step's action, log2 of its parameters, phi statistics — before the wait: the loads' latency hides
                int id = -1;
                float lp[MAX_P];
#pragma unroll
                for (int j = 0; j < MAX_P; ++j) lp[j] = 0.0f;
                if (row_lane && st + t < len) id = take(st + t, lp);
                // store only once GEMM1 of the previous step (or the previous tile's scorer) no longer reads K-blocks 8 ..
                if (n_w > 0) mbar_wait(bar(B_AFREE), (n_w - 1) & 1);
                ++n_w;
                if (t == 0) {          // the K-blocks still hold the previous tile's phi features
                    clear_row();
                    __syncwarp();
                    if (row_lane) put(NT + P, 0x3C00u);        // the constant-1 column (carries W1a b_p + b1)
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
            }

            // ---- the phi features (K-blocks 8 ..) of the scorer's A operand, followed by a constant-1 column that carries
            // scorer layer 1's bias:
            //   WM_PHI_MEAN    phi = mean_t a_t is LINEAR in psi = [count_c / len (NT) | sum_t log2 p_tj / len (P) | 1 (len > 0)];
            //                  the host folds E, W_p and b_p into scorer layer 1's phi weights (tc2_prepare)
            //   WM_PHI_STRUCT  phi = [count_c (NT) | len | sum_j (P) | mean_j (P) | max_j (P)]   (S25)
            if (!rank_it) continue;
            if (n_w > 0) mbar_wait(bar(B_AFREE), (n_w - 1) & 1);
            ++n_w;
            clear_row();
            __syncwarp();
            if (row_lane) {
                auto putf = [&](int c, float v) { put(c, pack_f16(v, 0.0f)); };
                const float inv = len > 0 ? 1.0f / (float)len : 0.0f;
                if (PHI == WM_PHI_STRUCT) {
                    for (int c = 0; c < NT; ++c) putf(c, (float)s_cnt[row * NT + c]);
                    putf(NT, (float)len);
#pragma unroll
                    for (int j = 0; j < MAX_P; ++j)
                        if (j < P) {
                            putf(NT + 1 + j, slp[j]);
                            putf(NT + 1 + P + j, slp[j] * inv);
                            putf(NT + 1 + 2 * P + j, smx[j]);
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

}  // namespace tc2

// ------------------------------------------------------------------------------------------------ host side
namespace {

uint16_t f32_to_bf16(float f) {
    uint32_t u;
    memcpy(&u, &f, 4);
    u += 0x7FFFu + ((u >> 16) & 1u);   // round to nearest even (the stored values are already bf16-exact)
    return (uint16_t)(u >> 16);
}

// Append the [256 x 64] pair tile W[n0 + n][k0 + k] (k < kvalid, else 0) as two 16 KB halves (weight rows 0-127 for
// the leader CTA, 128-255 for its peer), each in the SW128 K-major shared-memory image.
// Returns false when a weight is not finite in fp16 (|w| > 65504): the model then stays on the fp32 kernel.
bool append_pair_tile(std::vector<uint16_t>& blob, const std::vector<float>& W, int ld, int n0, int k0, int kvalid) {
    const size_t base = blob.size();
    blob.resize(base + 2 * tc2::BT_BYTES / 2, 0);
    bool ok = true;
    for (int n = 0; n < 256; ++n)
        for (int k = 0; k < 64; ++k) {
            const float v = k < kvalid ? W[(size_t)(n0 + n) * ld + k0 + k] : 0.0f;
            const int nn = n & 127;
            const size_t off = (size_t)(n >> 7) * tc2::BT_BYTES + (size_t)nn * 128 + (size_t)((((k >> 3) ^ (nn & 7)) << 4)) +
                               (size_t)(k & 7) * 2;
            uint16_t hb;
            ok &= f32_to_f16_bits(v, &hb);
            blob[base + off / 2] = hb;
        }
    return ok;
}

}  // namespace

bool tc2_model_ok(const Model& m) {
    return m.kind == WM_KIND_MLP_LN && m.phi_kind <= WM_PHI_STRUCT && m.dtype == WM_DTYPE_BF16 && m.embed == WM_EMBED_LINEAR && m.d == tc2::D &&
           m.d_a == tc2::DA && m.hidden >= 512 && m.hidden <= tc2::MAX_HID && m.hidden % 256 == 0 && m.n_lin == 3 &&
           m.sdim[1] == tc2::SW && m.sdim[2] == tc2::SW && m.H >= 8 && m.H <= tc2::MAX_H && m.H % 8 == 0 &&
           m.n_types <= tc2::MAX_TYPES && m.P <= tc2::MAX_P;
}

int tc2_prepare(wm_ctx* ctx, const std::vector<std::vector<float>>& hv, const std::vector<std::string>& names) {
    Model& m = ctx->m;
    if (!tc2_model_ok(m)) return WM_OK;
    const tc2::SmemLayout L = tc2::smem_layout(m.n_types, m.hidden, (m.H + 15) / 16);
    if ((int)L.total > ctx->smem_optin) return WM_OK;
    auto get = [&](const char* n) -> const std::vector<float>& {
        for (size_t i = 0; i < names.size(); ++i)
            if (names[i] == n) return hv[i];
        static const std::vector<float> empty;
        return empty;
    };
    const std::vector<float>&W1 = get("W1"), &W2 = get("W2"), &Ws0 = get("Ws0"), &Ws1 = get("Ws1"), &E = get("E");
    const std::vector<float>&b1 = get("b1"), &bs0 = get("bs0"), &Wp = get("W_p"), &bpv = get("b_p");
    const int hid = m.hidden, NC = hid / 256, K1 = tc2::D + tc2::DA, K0 = tc2::D + m.phi_dim + m.H, NT = m.n_types, P = m.P;
    // ---- GEMM1's a-columns folded onto the action features f = [onehot(id) (NT) | log2 p_j (P) | 1]:
    //      W1[:, d:] (E[id] + W_p lp + b_p) + b1  =  (W1a E^T)[:, id] + (W1a W_p) lp + (W1a b_p + b1)
    const int NF = NT + P + 1, AKB = (NF + 63) / 64;
    std::vector<float> W1f((size_t)hid * 64 * AKB, 0.0f);
    for (int n = 0; n < hid; ++n) {
        const float* wr = &W1[(size_t)n * K1 + tc2::D];
        float* out = &W1f[(size_t)n * 64 * AKB];
        for (int c = 0; c < NT; ++c) {
            double acc = 0.0;
            for (int k = 0; k < tc2::DA; ++k) acc += (double)wr[k] * E[(size_t)c * tc2::DA + k];
            out[c] = (float)acc;
        }
        for (int j = 0; j < P; ++j) {
            double acc = 0.0;
            for (int k = 0; k < tc2::DA; ++k) acc += (double)wr[k] * Wp[(size_t)k * P + j];
            out[NT + j] = (float)acc;
        }
        double acc = b1[n];
        for (int k = 0; k < tc2::DA; ++k) acc += (double)wr[k] * bpv[k];
        out[NT + P] = (float)acc;
    }
    // ---- scorer layer 1's phi columns folded onto psi = [count_c / len | sum log2 p_j / len | 1 (len > 0)] (see the action
    //      warps): Ws0_phi E^T, Ws0_phi W_p, Ws0_phi b_p, summed in double; then a constant-1 column that carries bs0
    const bool pstruct = m.phi_kind == WM_PHI_STRUCT;
    const int NPSI = (pstruct ? NT + 1 + 3 * P : NT + P + 1) + 1, PKB = (NPSI + 63) / 64;
    std::vector<float> Wphi((size_t)tc2::SW * 64 * PKB, 0.0f);
    for (int n = 0; n < tc2::SW; ++n) {
        const float* wr = &Ws0[(size_t)n * K0 + tc2::D];
        float* out = &Wphi[(size_t)n * 64 * PKB];
        if (pstruct) {           // the structured statistics enter as they are (S25)
            for (int c = 0; c < m.phi_dim; ++c) out[c] = wr[c];
            out[NPSI - 1] = bs0[n];
            continue;
        }
        for (int c = 0; c < NT; ++c) {
            double acc = 0.0;
            for (int k = 0; k < tc2::DA; ++k) acc += (double)wr[k] * E[(size_t)c * tc2::DA + k];
            out[c] = (float)acc;
        }
        for (int j = 0; j < P; ++j) {
            double acc = 0.0;
            for (int k = 0; k < tc2::DA; ++k) acc += (double)wr[k] * Wp[(size_t)k * P + j];
            out[NT + j] = (float)acc;
        }
        double acc = 0.0;
        for (int k = 0; k < tc2::DA; ++k) acc += (double)wr[k] * bpv[k];
        out[NT + P] = (float)acc;
        out[NT + P + 1] = bs0[n];
    }
    const size_t n_tiles = (size_t)NC * (AKB + 8 + tc2::G2_STAGES) + tc2::sc_stages(PKB);
    std::vector<uint16_t> blob;
    bool ok = true;   // every weight finite in fp16
    blob.reserve(n_tiles * tc2::BT_BYTES);
    // the MMA warp's order: feature K-blocks of chunks 0 and 1, z K-blocks (0-7) of chunks 0 and 1, G2(0), then G1(i)
    // (features then z), G2(i-1)
    auto g1a = [&](int c) { for (int k = 0; k < AKB; ++k) ok &= append_pair_tile(blob, W1f, 64 * AKB, c * 256, k * 64, 64); };
    auto g1z = [&](int c) { for (int k = 0; k < 8; ++k) ok &= append_pair_tile(blob, W1, K1, c * 256, k * 64, 64); };
    auto g2 = [&](int c) {            // GEMM2 chunk c: hidden K-blocks x the two 256-column N tiles of d
        for (int kb = 0; kb < 4; ++kb)
            for (int j = 0; j < 2; ++j) ok &= append_pair_tile(blob, W2, hid, j * 256, c * 256 + kb * 64, 64);
    };
    g1a(0); g1a(1); g1z(0); g1z(1);
    g2(0);
    for (int i = 2; i <= NC; ++i) {
        if (i < NC) { g1a(i); g1z(i); }
        g2(i - 1);
    }
    for (int c = 0; c < 4; ++c) {     // scorer layer 1: phi features (PKB), hw (1, zero-padded to 64 columns), z (8)
        for (int k = 0; k < PKB; ++k) ok &= append_pair_tile(blob, Wphi, 64 * PKB, c * 256, k * 64, 64);
        ok &= append_pair_tile(blob, Ws0, K0, c * 256, tc2::D + m.phi_dim, m.H);
        for (int k = 0; k < 8; ++k) ok &= append_pair_tile(blob, Ws0, K0, c * 256, k * 64, 64);
    }
    for (int round = 0; round < 2; ++round)   // scorer layer 2: two rounds of two N tiles over all 16 K-blocks
        for (int kb = 0; kb < 16; ++kb)
            for (int jj = 0; jj < 2; ++jj) ok &= append_pair_tile(blob, Ws1, tc2::SW, (2 * round + jj) * 256, kb * 64, 64);
    if (blob.size() * 2 != n_tiles * 2 * tc2::BT_BYTES) {
        set_error("tc2_prepare: internal weight-image size mismatch");
        return WM_ERR_FORMAT;
    }

    if (!ok) return WM_OK;   // a weight beyond the fp16 range: this model stays on the fp32 kernel

    void* d_blob = nullptr;
    WM_CUDA_TRY(cudaMalloc(&d_blob, blob.size() * 2));
    ctx->allocs.push_back(d_blob);
    WM_CUDA_TRY(cudaMemcpy(d_blob, blob.data(), blob.size() * 2, cudaMemcpyHostToDevice));

    // tensor map over the image seen as rows of 64 bf16 (128 B); one box = 128 rows = one 16 KB half tile.  The
    // image is already swizzled, so the map itself uses no swizzle.
    static_assert(sizeof(CUtensorMap) <= sizeof(m.tc2_tmap), "tensor map storage");
    CUtensorMap tm;
    {
        const int rc = encode_tmap_2d(&tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, d_blob, 64, blob.size() * 2 / 128, 128, 64, 128, false, "tc2_prepare");
        if (rc != WM_OK) return rc;
    }
    memcpy(m.tc2_tmap, &tm, sizeof(tm));
    m.tc_blob = d_blob;
    m.tc_blob_bytes = blob.size() * 2;
    m.tcp_akb = AKB;      // (shared fields: a model has either the d = 256 pair kernel or this one)
    m.tcp_pkb = PKB;
    if (pstruct) {
        WM_CUDA_TRY(cudaFuncSetAttribute(tc2::wm_tc2_kernel<WM_PHI_STRUCT, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.total));
        WM_CUDA_TRY(cudaFuncSetAttribute(tc2::wm_tc2_kernel<WM_PHI_STRUCT, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.total));
    } else {
        WM_CUDA_TRY(cudaFuncSetAttribute(tc2::wm_tc2_kernel<WM_PHI_MEAN, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.total));
        WM_CUDA_TRY(cudaFuncSetAttribute(tc2::wm_tc2_kernel<WM_PHI_MEAN, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.total));
    }
    m.tc_ok = 2;
    return WM_OK;
}

int launch_tc2(wm_ctx* ctx, Workspace* ws, const CallArgs& a, cudaStream_t st) {
    (void)ws;
    const Model& m = ctx->m;
    tc2::Params p;
    p.hid = m.hidden; p.nc = m.hidden / 256; p.n_types = m.n_types; p.P = m.P; p.H = m.H;
    p.hw_ksteps = (m.H + 15) / 16;
    p.ln_eps = m.ln_eps;
    p.akb = m.tcp_akb; p.pkb = m.tcp_pkb;
    p.b2 = m.b2; p.gamma = m.gamma; p.beta = m.beta;
    p.bs1 = m.bs[1]; p.w3 = m.Wst[2]; p.bs2 = m.bs[2];
    p.a = a;
    p.n_tiles = (int)((a.B + tc2::TMP - 1) / tc2::TMP);
    p.prof = trace::begin(st);
    CUtensorMap tm;
    memcpy(&tm, m.tc2_tmap, sizeof(tm));
    const tc2::SmemLayout L = tc2::smem_layout(m.n_types, m.hidden, p.hw_ksteps);
    const int max_pairs = ctx->n_sms / 2;
    const int pairs = p.n_tiles < max_pairs ? p.n_tiles : max_pairs;
    const bool prefix_call = a.start || a.init_index || a.latents_out;
    if (m.phi_kind == WM_PHI_STRUCT) {
        if (prefix_call) tc2::wm_tc2_kernel<WM_PHI_STRUCT, true><<<2 * pairs, tc2::THREADS, L.total, st>>>(p, tm);
        else tc2::wm_tc2_kernel<WM_PHI_STRUCT, false><<<2 * pairs, tc2::THREADS, L.total, st>>>(p, tm);
    } else {
        if (prefix_call) tc2::wm_tc2_kernel<WM_PHI_MEAN, true><<<2 * pairs, tc2::THREADS, L.total, st>>>(p, tm);
        else tc2::wm_tc2_kernel<WM_PHI_MEAN, false><<<2 * pairs, tc2::THREADS, L.total, st>>>(p, tm);
    }
    WM_CUDA_TRY(cudaGetLastError());
    ctx->launches.fetch_add(1);
    trace::dump(p.prof, st);
    return WM_OK;
}

}  // namespace wm

// K2 (tcgen05): fused persistent rollout + score kernel for the bf16 residual-MLP + LayerNorm models with
// d = 256, d_a = 128 (BASELINE.json cfg 2 and cfg 4), sm_100a only.
//
// PAPER.md:162 Eq.8 / :166 — z_t = F(z_{t-1}, a_t) applied recurrently; :176 — masked steps leave z unchanged;
// :186-188 Eq.12 — y = G([z_T ; phi ; h]).  Parametrisation: BASELINE.json cfg 2/4.
//
// One CTA owns a tile of 128 candidates (length-sorted by K1) for ALL of its steps:
//   * the fp32 master latent of the tile lives in TMEM columns [0,256) and IS the accumulator of GEMM2: the
//     residual add is the MMA's accumulate, the epilogue adds b2, applies LayerNorm and writes z' back;
//   * a fp16 copy of [z ; a] lives in shared memory (K-major, 128B-swizzled 64-column K-blocks) as the A operand
//     of GEMM1;
//   * GEMM1 runs in 128-column chunks of the hidden layer into two alternating TMEM accumulators; the GELU
//     epilogue writes the fp16 hidden chunk back INTO TMEM (over its own fp32 columns) and GEMM2 consumes it as a
//     TMEM A operand (tcgen05.mma with A in tensor memory), so the hidden activations never touch shared memory;
//   * weights stream from L2 through a 3-stage ring of 32 KB tile pairs filled by bulk async copies (TMA engine,
//     mbarrier complete_tx); the weight image in global memory is pre-tiled, pre-swizzled and laid out in exactly
//     the order the MMA warp consumes it, so the producer is a linear stream;
//   * the scorer's two hidden layers run on the same machinery (layer-1 output kept in TMEM as layer-2's A
//     operand), the last 512->1 layer is a dot product in the epilogue.
// Warp roles (512 threads): warps 0-7 epilogue (GELU / LayerNorm / scorer; one thread per row and column half),
// warps 8-11 action embedding (a_t for step t+1 while step t runs; phi and hw at the end of the tile), warp 12 TMEM
// allocator, warp 13 tile scheduler + weight producer, warp 15 MMA issuer (one elected lane).
#include <cuda_bf16.h>

#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "wm_internal.h"
#include "wm_ptx.cuh"
#include "wm_trace.cuh"

namespace wm {

namespace tc {

constexpr int TM = 128;            // candidates per tile (MMA M)
constexpr int D = 256;             // latent width
constexpr int DA = 128;            // action-embedding width
constexpr int SW = 512;            // scorer hidden width (both hidden layers)
constexpr int TILE_BYTES = 16384;  // one [128 x 64] 16-bit K-block tile, SW128 K-major
constexpr int STAGE_BYTES = 2 * TILE_BYTES;   // one ring stage = a PAIR of tiles (one barrier wait / commit per 8 MMAs)
constexpr int NSTAGE = 3;
constexpr int A1_KB = 6;           // z: 0-3, a/phi: 4-5
constexpr int HWK_BYTES = 4096;    // hw operand: one [128 x 16] no-swizzle K-major tile per K = 16 step
constexpr int THREADS = 512;
// Warp roles.  The SM's warp arbiter favours higher warp ids, so the latency-critical single-warp roles (MMA
// issuer, weight producer) sit at the top and the throughput roles (epilogue, action) below them.
constexpr int EPI_WARP0 = 0, ACT_WARP0 = 8, ALLOC_WARP = 12, PROD_WARP = 13, MMA_WARP = 15;
constexpr int MAX_TYPES = 64, MAX_P = 8, MAX_H = 64, MAX_HID = 1024;
constexpr int SC_TILES = 4 * 8 + 4 * 8;   // scorer stream: layer 1 (4 chunks x (2 phi, hw + pad, 4 z)), layer 2 (4 x 8)

// barrier indices
enum {
    B_FULL = 0,                 // [NSTAGE] producer -> MMA
    B_EMPTY = B_FULL + NSTAGE,  // [NSTAGE] MMA commit -> producer
    B_D1FULL = B_EMPTY + NSTAGE,   // [2] MMA commit -> epilogue: accumulator buffer b filled
    B_HREADY = B_D1FULL + 2,       // [2] epilogue -> MMA: buffer b consumed (fp16 hidden written)
    B_D2FULL = B_HREADY + 2,       // MMA commit -> epilogue: GEMM2 of the step done
    B_ZREADY,                      // epilogue -> MMA: z (fp16 smem + fp32 TMEM) written
    B_AFREE,                       // MMA commit -> action warps: a-part of A1 no longer read
    B_AREADY,                      // action warps -> MMA: a-part written
    B_SFULL,                       // [2] scheduler -> consumers
    B_SEMPTY = B_SFULL + 2,        // [2] consumers -> scheduler
    B_COUNT = B_SEMPTY + 2
};

struct Params {
    // model
    int hid, nc, n_types, P, H, hw_ksteps;
    float ln_eps;
    const uint8_t* blob;        // weight tiles in consumption order
    const __nv_bfloat16* E;     // [n_types][128]
    const float *WpT, *bp;      // [P][128], [128]
    const float *b1, *b2, *gamma, *beta;
    const float *bs0, *bs1, *w3, *bs2;
    // call
    CallArgs a;
    int n_tiles;
    int* tile_counter;
    unsigned long long* prof;   // developer trace buffer (wm_trace.cuh), null in a normal build
};

struct SmemLayout {
    uint32_t a1, hwk, ring, e_tab, lp, mx, ids, cnt, b1, b2, gamma, beta, red, bars, sched, tmem_slot, total;
};

// phi_struct: the structured action features (WM_PHI_STRUCT) also keep a per-row, per-slot running maximum
__host__ __device__ inline SmemLayout smem_layout(int n_types, int hid, int hw_ksteps, int phi_struct) {
    SmemLayout L;
    uint32_t o = 0;
    L.a1 = o; o += A1_KB * TILE_BYTES;
    L.ring = o; o += NSTAGE * STAGE_BYTES;
    L.hwk = o; o += (uint32_t)hw_ksteps * HWK_BYTES;
    L.e_tab = o; o += (uint32_t)n_types * DA * 2;
    L.lp = o; o += TM * MAX_P * 4;
    L.mx = o; o += phi_struct ? TM * MAX_P * 4 : 0;
    L.ids = o; o += TM * 4;
    L.cnt = o; o += TM * (uint32_t)n_types;           // u8 counts, row-major [128][n_types]
    o = (o + 15) & ~15u;
    L.b1 = o; o += (uint32_t)hid * 4;
    L.b2 = o; o += D * 4;
    L.gamma = o; o += D * 4;
    L.beta = o; o += D * 4;
    L.red = o; o += 4 * TM * 8;                        // [2 (LayerNorm parity)][2 column halves][128 rows] float2
    L.bars = o; o += B_COUNT * 8;
    L.sched = o; o += 2 * 8;
    L.tmem_slot = o; o += 16;
    L.total = o;
    return L;
}

using namespace ptx;

}  // namespace tc

namespace tc {

// PHI = WM_PHI_MEAN: phi = mean action embedding; WM_PHI_STRUCT: the paper's structured statistics (S25),
// which only changes what the action warps write into the phi K-blocks at the end of a tile.
// EXT = true: the prefix-latent-reuse calls (wm_rollout_latents / wm_rollout_score_from: per-candidate start position and
// initial-latent row, latent stored after every step); false compiles all of that out of the literal path.
template <int PHI, bool EXT>
__global__ void __launch_bounds__(THREADS, 1) wm_tc_kernel(const Params p) {
    extern __shared__ __align__(1024) uint8_t smem[];
    const SmemLayout L = smem_layout(p.n_types, p.hid, p.hw_ksteps, PHI);
    const uint32_t s_base = smem_u32(smem);
    const uint32_t s_a1 = s_base + L.a1, s_ring = s_base + L.ring, s_bars = s_base + L.bars;
    auto bar = [&](int i) -> uint32_t { return s_bars + 8u * (uint32_t)i; };
    volatile int* s_sched = reinterpret_cast<volatile int*>(smem + L.sched);   // [2][2]: tile, nsteps
    float* s_b1 = reinterpret_cast<float*>(smem + L.b1);
    float* s_b2 = reinterpret_cast<float*>(smem + L.b2);
    float* s_gamma = reinterpret_cast<float*>(smem + L.gamma);
    float* s_beta = reinterpret_cast<float*>(smem + L.beta);
    float2* s_red = reinterpret_cast<float2*>(smem + L.red);                  // [2][2][128]

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int NC = p.nc;
    const int ROLL_TILES = NC * 10;

    // ---- one-time setup
    if (threadIdx.x == 0) {
        for (int i = 0; i < NSTAGE; ++i) { mbar_init(bar(B_FULL + i), 1); mbar_init(bar(B_EMPTY + i), 1); }
        for (int i = 0; i < 2; ++i) {
            mbar_init(bar(B_D1FULL + i), 1);
            mbar_init(bar(B_HREADY + i), 8);
            mbar_init(bar(B_SFULL + i), 1);
            mbar_init(bar(B_SEMPTY + i), 13);
        }
        mbar_init(bar(B_D2FULL), 1);
        mbar_init(bar(B_ZREADY), 8);
        mbar_init(bar(B_AFREE), 1);
        mbar_init(bar(B_AREADY), 4);
        fence_barrier_init();
        fence_proxy_async();
    }
    if (warp == ALLOC_WARP) tmem_alloc(s_base + L.tmem_slot, 512);
    for (int i = threadIdx.x; i < p.hid; i += THREADS) s_b1[i] = __ldg(p.b1 + i);
    for (int i = threadIdx.x; i < D; i += THREADS) {
        s_b2[i] = __ldg(p.b2 + i);
        s_gamma[i] = __ldg(p.gamma + i);
        s_beta[i] = __ldg(p.beta + i);
    }
    {
        const uint32_t* src = reinterpret_cast<const uint32_t*>(p.E);
        uint32_t* dst = reinterpret_cast<uint32_t*>(smem + L.e_tab);
        for (int i = threadIdx.x; i < p.n_types * DA / 2; i += THREADS) dst[i] = __ldg(src + i);
        // the hw K-block is only ever written in its first columns: clear it once so unread bytes are not NaNs
        uint32_t* hwk = reinterpret_cast<uint32_t*>(smem + L.hwk);
        for (int i = threadIdx.x; i < p.hw_ksteps * HWK_BYTES / 4; i += THREADS) hwk[i] = 0u;
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(smem + L.tmem_slot);
    // EXT calls that store latents and rank nothing (wm_rollout_latents; the rollout half of a forest-ranker model) skip
    // the scorer in every role: no scorer tiles streamed, no scorer MMAs, no phi / hw operand, no score
    const bool rank = !EXT || p.a.scores_out != nullptr;
    const uint32_t T_Z = tmem_base;                 // fp32 latent / GEMM2 accumulator, 256 columns
    const uint32_t T_D1 = tmem_base + 256;          // two 128-column GEMM1 accumulators

    if (warp == PROD_WARP) {
        // =============================================================== scheduler + weight producer
        uint32_t stage = 0, ph = 0;
        for (uint32_t it = 0;; ++it) {
            const uint32_t slot = it & 1;
            int tile = 0;
            if (lane == 0) tile = atomicAdd(p.tile_counter, 1);
            tile = __shfl_sync(0xffffffffu, tile, 0);
            int nsteps = 0;
            if (tile < p.n_tiles) {
                for (int r = lane; r < TM; r += 32) {
                    int cand, len, seg;
                    row_meta(p.a, (int64_t)tile * TM + r, cand, len, seg, true);
                    nsteps = max(nsteps, EXT ? len - row_start(p.a, cand, len) : len);
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) nsteps = max(nsteps, __shfl_xor_sync(0xffffffffu, nsteps, o));
            } else {
                tile = -1;
            }
            if (lane == 0) {
                mbar_wait(bar(B_SEMPTY + slot), ((it >> 1) & 1) ^ 1);
                s_sched[slot * 2 + 0] = tile;
                s_sched[slot * 2 + 1] = nsteps;
                mbar_arrive(bar(B_SFULL + slot));   // release semantics order the two stores before it
            }
            if (tile < 0) break;
            if (lane == 0) {
                // the stream is consumed in pairs of tiles that are adjacent in the image: one 32 KB copy per stage
                const int roll_total = nsteps * ROLL_TILES, total = roll_total + (rank ? SC_TILES : 0);
                for (int i = 0; i < total; i += 2) {
                    const int src_tile = i < roll_total ? i % ROLL_TILES : ROLL_TILES + (i - roll_total);
                    mbar_wait(bar(B_EMPTY + stage), ph ^ 1);
                    mbar_arrive_expect_tx(bar(B_FULL + stage), STAGE_BYTES);
                    bulk_g2s(s_ring + stage * STAGE_BYTES, p.blob + (size_t)src_tile * TILE_BYTES, STAGE_BYTES,
                             bar(B_FULL + stage));
                    if (++stage == NSTAGE) { stage = 0; ph ^= 1; }
                }
            }
            __syncwarp();
        }
    } else if (warp == MMA_WARP) {
        // =============================================================== MMA issuer (converged warp, one elected lane)
        // The MMAs themselves are asynchronous (4 issue in ~70 cycles and queue in the tensor pipe), so the pipe
        // stays busy only while this warp's bookkeeping per 8 MMAs (512 pipe cycles) costs less than 512 cycles:
        // one full-barrier wait and one commit per ring stage (a pair of tiles), rolled loops, nothing else.
        {
            uint32_t stage = 0, ph = 0;
            uint32_t n_z = 0, n_a = 0, n_h[2] = {0, 0};
            bool pend[2] = {false, false};
            const uint32_t s_hwk = s_base + L.hwk;
            WM_TRACE_DECL(p.prof, 0)
            auto wait_h = [&](int b) {
                if (pend[b]) {
                    WM_TRACE(10 + b);
                    mbar_wait(bar(B_HREADY + b), n_h[b] & 1);
                    ++n_h[b];
                    pend[b] = false;
                    tc_fence_after();
                    WM_TRACE(12 + b);
                }
            };
            auto wait_full = [&]() {
                WM_TRACE(1);
                mbar_wait(bar(B_FULL + stage), ph);
                tc_fence_after();
                WM_TRACE(2);
            };
            auto release = [&]() {   // called by the elected lane after the stage's last MMA
                mma_commit(bar(B_EMPTY + stage));
            };
            auto advance = [&]() {
                __syncwarp();
                WM_TRACE(3);
                if (++stage == NSTAGE) { stage = 0; ph ^= 1; }
            };
            // stage = two [128 x 64] B tiles against the A1 K-blocks a_tile0, a_tile1 (8 MMAs of K = 16)
            auto pair_ss = [&](uint32_t d_tmem, uint32_t a_tile0, uint32_t a_tile1, bool first) {
                wait_full();
                const uint64_t a0 = smem_desc(a_tile0), a1d = smem_desc(a_tile1);
                const uint64_t b0 = smem_desc(s_ring + stage * STAGE_BYTES), b1 = b0 + (TILE_BYTES >> 4);
                if (elect_one()) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) mma_ss(d_tmem, a0 + 2u * j, b0 + 2u * j, IDESC, (first && j == 0) ? 0u : 1u);
#pragma unroll
                    for (int j = 0; j < 4; ++j) mma_ss(d_tmem, a1d + 2u * j, b1 + 2u * j, IDESC, 1u);
                    release();
                }
                advance();
            };
            // stage = (hw tile, padding tile): hw_ksteps MMAs whose A operand is the no-swizzle [128 x 16] hw tile
            auto pair_hw = [&](uint32_t d_tmem) {
                wait_full();
                const uint64_t b0 = smem_desc(s_ring + stage * STAGE_BYTES);
                if (elect_one()) {
                    for (int j = 0; j < p.hw_ksteps; ++j)
                        mma_ss(d_tmem, smem_desc_nosw(s_hwk + j * HWK_BYTES), b0 + 2u * j, IDESC, 1u);
                    release();
                }
                advance();
            };
            // stage = two B tiles against TMEM A operands a_tmem0, a_tmem1 into d0, d1
            auto pair_ts = [&](uint32_t d0, uint32_t d1, uint32_t a_tmem0, uint32_t a_tmem1, bool first) {
                wait_full();
                const uint64_t b0 = smem_desc(s_ring + stage * STAGE_BYTES), b1 = b0 + (TILE_BYTES >> 4);
                if (elect_one()) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) mma_ts(d0, a_tmem0 + 8u * j, b0 + 2u * j, IDESC, (first && j == 0) ? 0u : 1u);
#pragma unroll
                    for (int j = 0; j < 4; ++j) mma_ts(d1, a_tmem1 + 8u * j, b1 + 2u * j, IDESC, 1u);
                    release();
                }
                advance();
            };
            // stage = ONE [256 x 64] B tile (the two adjacent [128 x 64] tiles of a stage are exactly that: row n at
            // n * 128 B, same swizzle) against the TMEM A operand a_tmem into the 256-column accumulator d: 4 MMAs with
            // N = 256 instead of 8 with N = 128.  The issuing warp, not the tensor pipe, bounds this kernel, and an
            // N = 256 MMA carries twice the work per issued instruction.
            auto stage_ts256 = [&](uint32_t d, uint32_t a_tmem) {
                wait_full();
                const uint64_t b0 = smem_desc(s_ring + stage * STAGE_BYTES);
                if (elect_one()) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) mma_ts(d, a_tmem + 8u * j, b0 + 2u * j, IDESC_N256, 1u);
                    release();
                }
                advance();
            };
            auto commit = [&](int barrier) {
                if (elect_one()) mma_commit(bar(barrier));
                __syncwarp();
            };
            // GEMM over the A1 K-blocks in the order a/phi (4,5), [hw], z (0..3); waits for the operands of the
            // first chunk of the scorer.  The a-buffer is released right after the last chunk's a K-blocks, not after
            // the whole chunk (the action warps write a_{t+1} / phi into it as soon as it is free).
            auto gemm_a1 = [&](int b, bool first_chunk, bool last_chunk, bool with_hw) {
                wait_h(b);
                const uint32_t d = T_D1 + 128u * b;
                if (first_chunk) { WM_TRACE(20); mbar_wait(bar(B_AREADY), n_a & 1); ++n_a; WM_TRACE(21); }
                pair_ss(d, s_a1 + 4 * TILE_BYTES, s_a1 + 5 * TILE_BYTES, true);
                if (with_hw) pair_hw(d);
                if (last_chunk) commit(B_AFREE);
                if (first_chunk) { WM_TRACE(22); mbar_wait(bar(B_ZREADY), n_z & 1); ++n_z; WM_TRACE(23); }
                pair_ss(d, s_a1, s_a1 + TILE_BYTES, false);
                pair_ss(d, s_a1 + 2 * TILE_BYTES, s_a1 + 3 * TILE_BYTES, false);
                commit(B_D1FULL + b);
                pend[b] = true;
            };
            for (uint32_t it = 0;; ++it) {
                const uint32_t slot = it & 1;
                mbar_wait(bar(B_SFULL + slot), (it >> 1) & 1);
                const int tile = s_sched[slot * 2 + 0], nsteps = s_sched[slot * 2 + 1];
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(B_SEMPTY + slot));
                if (tile < 0) break;
#pragma unroll 1
                for (int t = 0; t < nsteps; ++t) {
                    // Step boundary: the a K-blocks of chunk 0 AND chunk 1 depend only on a_{t+1} and both GEMM1
                    // accumulators are free, so both a-parts are issued before the wait for z' (pipe drain + LayerNorm
                    // is the serial section of a step); then the z K-blocks of chunks 0 and 1.
                    {
                        wait_h(0);
                        wait_h(1);
                        WM_TRACE(20); mbar_wait(bar(B_AREADY), n_a & 1); ++n_a; WM_TRACE(21);
                        pair_ss(T_D1, s_a1 + 4 * TILE_BYTES, s_a1 + 5 * TILE_BYTES, true);
                        pair_ss(T_D1 + 128u, s_a1 + 4 * TILE_BYTES, s_a1 + 5 * TILE_BYTES, true);
                        if (NC == 2) commit(B_AFREE);
                        WM_TRACE(22); mbar_wait(bar(B_ZREADY), n_z & 1); ++n_z; WM_TRACE(23);
                        for (int b = 0; b < 2; ++b) {
                            pair_ss(T_D1 + 128u * b, s_a1, s_a1 + TILE_BYTES, false);
                            pair_ss(T_D1 + 128u * b, s_a1 + 2 * TILE_BYTES, s_a1 + 3 * TILE_BYTES, false);
                            commit(B_D1FULL + b);
                            pend[b] = true;
                        }
                    }
                    auto gemm2 = [&](int c) {                                    // GEMM2 chunk c (A from TMEM)
                        const int b = c & 1;
                        wait_h(b);
                        const uint32_t hbuf = T_D1 + 128u * b;
                        stage_ts256(T_Z, hbuf);            // K-block 0 of the chunk x all 256 latent columns
                        stage_ts256(T_Z, hbuf + 64u);      // K-block 1
                        if (c == NC - 1) commit(B_D2FULL);
                    };
                    gemm2(0);
#pragma unroll 1
                    for (int i = 2; i <= NC; ++i) {
                        if (i < NC) gemm_a1(i & 1, false, i == NC - 1, false);   // GEMM1 chunk i
                        gemm2(i - 1);
                    }
                }
                if (!rank) {   // nothing to rank: only take the terminal latent's ZREADY so the phase count stays in step
                    mbar_wait(bar(B_ZREADY), n_z & 1);
                    ++n_z;
                    continue;
                }
                // ---- scorer layer 1: four 128-column chunks of gelu(Ws0 [z_T; phi; hw] + bs0)
#pragma unroll 1
                for (int c = 0; c < 4; ++c) {
                    gemm_a1(c & 1, c == 0, c == 3, true);
                }
                wait_h(0);
                wait_h(1);   // all of H1 (fp16, TMEM columns [0,256)) written
                // ---- scorer layer 2: A = H1 from TMEM, K = 512
#pragma unroll 1
                for (int c = 0; c < 4; ++c) {
                    const int b = c & 1;
                    wait_h(b);
#pragma unroll 1
                    for (int kb = 0; kb < 8; kb += 2)
                        pair_ts(T_D1 + 128u * b, T_D1 + 128u * b, T_Z + 32u * kb, T_Z + 32u * (kb + 1), kb == 0);
                    commit(B_D1FULL + b);
                    pend[b] = true;
                }
            }
        }
        __syncwarp();
    }
    else if (warp >= EPI_WARP0 && warp < ACT_WARP0) {
        // =============================================================== epilogue warps (GELU / LayerNorm / scorer)
        const int q = warp & 3, hh = (warp - EPI_WARP0) >> 2;
        const int row = 32 * q + lane;
        const uint32_t lane_off = (uint32_t)(32 * q) << 16;
        uint8_t* a1 = smem + L.a1;
        uint32_t n_d1[2] = {0, 0}, n_d2 = 0;
        const float inv_d = 1.0f / (float)D;
        // write 32 consecutive z columns of this row: fp32 -> TMEM, fp16 -> A1 (when `to_smem`)
        auto put_z = [&](int col0, const uint32_t (&v)[32], bool to_smem) {
            tmem_st32(T_Z + lane_off + (uint32_t)col0, v);
            if (to_smem) {
                uint8_t* kb = a1 + (col0 >> 6) * TILE_BYTES;
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
            }
        };
        auto publish = [&](int barrier, bool smem_written) {
            tmem_st_wait();
            if (smem_written) fence_proxy_async();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(barrier));
        };
        // bias + GELU over this thread's 64 columns of accumulator buffer b, fp16 result to TMEM at dst_col
        auto gelu_chunk = [&](int b, const float* bias, bool bias_in_smem, uint32_t dst_col) {
            mbar_wait(bar(B_D1FULL + b), n_d1[b] & 1);
            ++n_d1[b];
            tc_fence_after();
#pragma unroll
            for (int p2 = 0; p2 < 2; ++p2) {
                uint32_t v[32], o[16];
                tmem_ld32(T_D1 + 128u * b + lane_off + 64u * hh + 32u * p2, v);
                tmem_ld_wait();
                const float4* bp_ = reinterpret_cast<const float4*>(bias + 32 * p2);
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const float4 bv = bias_in_smem ? bp_[i] : __ldg(bp_ + i);
                    o[2 * i] = gelu2_f16(make_float2(__uint_as_float(v[4 * i]), __uint_as_float(v[4 * i + 1])),
                                          make_float2(bv.x, bv.y));
                    o[2 * i + 1] = gelu2_f16(make_float2(__uint_as_float(v[4 * i + 2]), __uint_as_float(v[4 * i + 3])),
                                              make_float2(bv.z, bv.w));
                }
                tmem_st16(dst_col + lane_off + 16u * p2, o);
            }
            publish(B_HREADY + b, false);
        };

        for (uint32_t it = 0;; ++it) {
            const uint32_t slot = it & 1;
            mbar_wait(bar(B_SFULL + slot), (it >> 1) & 1);
            const int tile = s_sched[slot * 2 + 0], nsteps = s_sched[slot * 2 + 1];
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(B_SEMPTY + slot));
            if (tile < 0) break;
            int cand, len, seg;
            row_meta(p.a, (int64_t)tile * TM + row, cand, len, seg, false);
            // prefix-latent reuse: the rollout covers positions [st, len) and starts from the row init_index names
            const int st = EXT ? row_start(p.a, cand, len) : 0, rem = len - st;
            const size_t zrow = EXT ? row_init(p.a, cand, seg) : (size_t)seg;

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
                put_z(col0, v, true);
            }
            publish(B_ZREADY, true);

            for (int t = 0; t < nsteps; ++t) {
                for (int c = 0; c < NC; ++c)
                    gelu_chunk(c & 1, s_b1 + c * 128 + 64 * hh, true, T_D1 + 128u * (c & 1) + 64u * hh);
                // ---- LayerNorm(z + W2 h + b2): the accumulator already holds z + W2 h
                mbar_wait(bar(B_D2FULL), n_d2 & 1);
                ++n_d2;
                tc_fence_after();
                float2 s1v = make_float2(0.0f, 0.0f), s2v = make_float2(0.0f, 0.0f);
#pragma unroll 1
                for (int p4 = 0; p4 < 4; ++p4) {
                    const int col0 = 128 * hh + 32 * p4;
                    uint32_t v[32];
                    tmem_ld32(T_Z + lane_off + (uint32_t)col0, v);
                    tmem_ld_wait();
                    const float4* b2v = reinterpret_cast<const float4*>(s_b2 + col0);
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
                const float s1 = s1v.x + s1v.y, s2 = s2v.x + s2v.y;
                // exchanged through the slot of this LayerNorm's parity: the partner reads the previous LayerNorm's value
                // from the other slot, so no second barrier is needed before the next one writes
                float2* red = s_red + (n_d2 & 1u) * 2 * TM;
                red[hh * TM + row] = make_float2(s1, s2);
                named_bar_sync(1 + q, 64);
                const float2 other = red[(hh ^ 1) * TM + row];
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
#pragma unroll 1
                for (int p4 = 0; p4 < 4; ++p4) {
                    const int col0 = 128 * hh + 32 * p4;
                    uint32_t v[32];
                    tmem_ld32(T_Z + lane_off + (uint32_t)col0, v);
                    tmem_ld_wait();
                    const float4* b2v = reinterpret_cast<const float4*>(s_b2 + col0);
                    const float4* gv = reinterpret_cast<const float4*>(s_gamma + col0);
                    const float4* bev = reinterpret_cast<const float4*>(s_beta + col0);
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
                    put_z(col0, v, live);
                    if (lat) {
#pragma unroll
                        for (int i = 0; i < 8; ++i)
                            lat[(col0 >> 2) + i] = make_float4(__uint_as_float(v[4 * i]), __uint_as_float(v[4 * i + 1]),
                                                               __uint_as_float(v[4 * i + 2]), __uint_as_float(v[4 * i + 3]));
                    }
                }
                publish(B_ZREADY, true);
            }

            if (!rank) continue;
            // ---- scorer layer 1 -> H1 (fp16) in TMEM columns [0,256)
            for (int c = 0; c < 4; ++c)
                gelu_chunk(c & 1, p.bs0 + c * 128 + 64 * hh, false, T_Z + 64u * c + 32u * hh);
            // ---- scorer layer 2 + output dot product
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
                if (lane == 0) mbar_arrive(bar(B_HREADY + b));
            }
            s_red[hh * TM + row] = make_float2(part, 0.0f);
            named_bar_sync(1 + q, 64);
            if (hh == 0 && cand >= 0 && (!EXT || p.a.scores_out)) p.a.scores_out[cand] = part + s_red[TM + row].x + __ldg(p.bs2);
            named_bar_sync(1 + q, 64);   // s_red is reused by the next tile's first LayerNorm
        }
    } else if (warp >= ACT_WARP0 && warp < ACT_WARP0 + 4) {
        // =============================================================== action-embedding warps
        const int aw = warp - ACT_WARP0;
        const int row = 32 * aw + lane;       // row-mapped phases
        const int col4 = 4 * lane;            // column-mapped phases: this lane's 4 embedding columns
        uint8_t* a1 = smem + L.a1;
        const uint8_t* s_E = smem + L.e_tab;
        float* s_lp = reinterpret_cast<float*>(smem + L.lp);
        int* s_ids = reinterpret_cast<int*>(smem + L.ids);
        uint8_t* s_cnt = smem + L.cnt;
        const int P = p.P, NT = p.n_types;
        float wp[MAX_P][4], bp4[4];
#pragma unroll
        for (int j = 0; j < MAX_P; ++j)
#pragma unroll
            for (int e = 0; e < 4; ++e) wp[j][e] = j < P ? __ldg(p.WpT + j * DA + col4 + e) : 0.0f;
#pragma unroll
        for (int e = 0; e < 4; ++e) bp4[e] = __ldg(p.bp + col4 + e);
        uint32_t n_w = 0;
        // A1 destination of this lane's 4 columns (8 bytes) in row r: K-block 4 + lane/16
        auto a_dst = [&](int r) -> uint2* {
            return reinterpret_cast<uint2*>(a1 + (4 + (lane >> 4)) * TILE_BYTES + sw128_off(r, (lane & 15) >> 1) +
                                            (lane & 1) * 8);
        };
        for (uint32_t it = 0;; ++it) {
            const uint32_t slot = it & 1;
            mbar_wait(bar(B_SFULL + slot), (it >> 1) & 1);
            const int tile = s_sched[slot * 2 + 0], nsteps = s_sched[slot * 2 + 1];
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(B_SEMPTY + slot));
            if (tile < 0) break;
            int cand, len, seg;
            row_meta(p.a, (int64_t)tile * TM + row, cand, len, seg, false);
            for (int c = 0; c < NT; ++c) s_cnt[row * NT + c] = 0;
            float slp[MAX_P];   // per parameter slot: running sum of log2 p
#pragma unroll
            for (int j = 0; j < MAX_P; ++j) slp[j] = 0.0f;
            // structured phi: the per-slot running maximum lives in shared memory (the registers of this role are full)
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
            // prefix-latent reuse: positions [0, st) were rolled before (their latent is z_0 of this call); they only
            // feed phi.  They are scanned four at a time (all loads issued before the first is used) BEFORE the first rollout
            // step, in position order, so the running sums see the positions in the literal call's order and the scores
            // of the two calls are bit-identical (interleaving the scan with the steps was no faster and was not).
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

            for (int t = 0; t < nsteps; ++t) {
                // phase 1 (one row per lane): read the step's action, log2 of its parameters, phi statistics
                int id = -1;
                float lp[MAX_P];
#pragma unroll
                for (int j = 0; j < MAX_P; ++j) lp[j] = 0.0f;
                if (st + t < len) id = take(st + t, lp);
                s_ids[row] = id;
                *reinterpret_cast<float4*>(s_lp + row * MAX_P) = make_float4(lp[0], lp[1], lp[2], lp[3]);
                *reinterpret_cast<float4*>(s_lp + row * MAX_P + 4) = make_float4(lp[4], lp[5], lp[6], lp[7]);
                __syncwarp();
                // phase 2 (4 columns per lane, loop over the warp's 32 rows): a = E[id] + W_p log2(p) + b_p.  The first
                // PRE rows are computed into registers BEFORE the wait below (the issuer needs a_{t+1} soon after it has
                // released the a-buffer), the rest after it.
                constexpr int PRE = 16;
                uint2 pk[PRE];
                auto a_row = [&](int r) -> uint2 {
                    const int idr = s_ids[r];
                    float a4[4] = {0.0f, 0.0f, 0.0f, 0.0f};
                    if (idr >= 0) {
                        const uint2 e = *reinterpret_cast<const uint2*>(s_E + ((size_t)idr * DA + col4) * 2);
                        a4[0] = __uint_as_float(e.x << 16) + bp4[0];
                        a4[1] = __uint_as_float(e.x & 0xffff0000u) + bp4[1];
                        a4[2] = __uint_as_float(e.y << 16) + bp4[2];
                        a4[3] = __uint_as_float(e.y & 0xffff0000u) + bp4[3];
                        const float4 l0 = *reinterpret_cast<const float4*>(s_lp + r * MAX_P);
                        const float4 l1 = *reinterpret_cast<const float4*>(s_lp + r * MAX_P + 4);
                        const float lr[8] = {l0.x, l0.y, l0.z, l0.w, l1.x, l1.y, l1.z, l1.w};
#pragma unroll
                        for (int j = 0; j < MAX_P; ++j)
#pragma unroll
                            for (int e2 = 0; e2 < 4; ++e2) a4[e2] = fmaf(wp[j][e2], lr[j], a4[e2]);
                    }
                    return make_uint2(pack_f16(a4[0], a4[1]), pack_f16(a4[2], a4[3]));
                };
#pragma unroll
                for (int rr = 0; rr < PRE; ++rr) pk[rr] = a_row(32 * aw + rr);
                // store only once GEMM1 of the previous step no longer reads the a-part of A1
                if (n_w > 0) mbar_wait(bar(B_AFREE), (n_w - 1) & 1);
                ++n_w;
#pragma unroll
                for (int rr = 0; rr < PRE; ++rr) *a_dst(32 * aw + rr) = pk[rr];
#pragma unroll 4
                for (int rr = PRE; rr < 32; ++rr) {
                    const int r = 32 * aw + rr;
                    *a_dst(r) = a_row(r);
                }
                fence_proxy_async();
                __syncwarp();   // also: phase 2 reads of s_ids / s_lp are done before the next phase 1 overwrites
                if (lane == 0) mbar_arrive(bar(B_AREADY));
            }

            // ---- the phi K-blocks of the scorer's A operand, one ROW per lane (uniform control flow; everything a lane
            // needs is its own row's): clear the row's two K-blocks, then one 16-bit store per feature.
            //   WM_PHI_MEAN    phi = mean_t a_t = (sum_c count_c E[c] + W_p sum_t log2 p_t) / len + b_p is LINEAR in
            //                  psi = [count_c / len (NT) | sum_t log2 p_tj / len (P) | 1 (len > 0)], so the host folds
            //                  E, W_p and b_p into scorer layer 1's phi weights (tc_prepare) and the kernel only writes psi
            //   WM_PHI_STRUCT  phi = [count_c (NT) | len | sum_j (P) | mean_j (P) | max_j (P)]   (S25)
            if (!rank) continue;
            if (n_w > 0) mbar_wait(bar(B_AFREE), (n_w - 1) & 1);
            ++n_w;
            {
                auto put = [&](int c, float v) {
                    *reinterpret_cast<uint16_t*>(a1 + (4 + (c >> 6)) * TILE_BYTES + sw128_off(row, (c & 63) >> 3) +
                                                 (c & 7) * 2) = (uint16_t)pack_f16(v, 0.0f);
                };
#pragma unroll
                for (int ch = 0; ch < 16; ++ch)
                    *reinterpret_cast<uint4*>(a1 + (4 + (ch >> 3)) * TILE_BYTES + sw128_off(row, ch & 7)) =
                        make_uint4(0u, 0u, 0u, 0u);
                const float inv = len > 0 ? 1.0f / (float)len : 0.0f;
                if (PHI == WM_PHI_STRUCT) {
                    for (int c = 0; c < NT; ++c) put(c, (float)s_cnt[row * NT + c]);
                    put(NT, (float)len);
                    const float4 m0 = s_mx4[0], m1 = s_mx4[1];
                    const float mxr[8] = {m0.x, m0.y, m0.z, m0.w, m1.x, m1.y, m1.z, m1.w};
#pragma unroll
                    for (int j = 0; j < MAX_P; ++j)
                        if (j < P) {
                            put(NT + 1 + j, slp[j]);
                            put(NT + 1 + P + j, slp[j] * inv);
                            put(NT + 1 + 2 * P + j, mxr[j]);
                        }
                } else {
                    for (int c = 0; c < NT; ++c) put(c, (float)s_cnt[row * NT + c] * inv);
#pragma unroll
                    for (int j = 0; j < MAX_P; ++j)
                        if (j < P) put(NT + j, slp[j] * inv);
                    put(NT + P, len > 0 ? 1.0f : 0.0f);
                }
            }
            // hardware features of this row -> the hw operand tile (columns >= H stay zero)
            for (int ch = 0; ch < p.H / 8; ++ch) {
                uint4 o = make_uint4(0u, 0u, 0u, 0u);
                if (cand >= 0 && (!EXT || p.a.hw_feats)) {   // (wm_rollout_latents passes no hardware features: nothing is ranked)
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
            if (lane == 0) mbar_arrive(bar(B_AREADY));
        }
    }

    // ---- teardown
    tc_fence_before();
    __syncthreads();
    if (warp == ALLOC_WARP) tmem_dealloc(tmem_base, 512);
}

}  // namespace tc

// ------------------------------------------------------------------------------------------------ host side
namespace {

uint16_t f32_to_bf16(float f) {
    uint32_t u;
    memcpy(&u, &f, 4);
    u += 0x7FFFu + ((u >> 16) & 1u);   // round to nearest even (the stored values are already bf16-exact)
    return (uint16_t)(u >> 16);
}

// Append the [128 x 64] tile W[n0 + n][k0 + k] (k < kvalid, else 0) in the SW128 K-major shared-memory image.
// Returns false when a weight is not finite in fp16 (|w| > 65504): the model then stays on the fp32 kernel.
bool append_tile(std::vector<uint16_t>& blob, const std::vector<float>& W, int ld, int n0, int k0, int kvalid) {
    const size_t base = blob.size();
    blob.resize(base + tc::TILE_BYTES / 2, 0);
    bool ok = true;
    for (int n = 0; n < 128; ++n)
        for (int k = 0; k < 64; ++k) {
            const float v = k < kvalid ? W[(size_t)(n0 + n) * ld + k0 + k] : 0.0f;
            const size_t off = (size_t)n * 128 + (size_t)((((k >> 3) ^ (n & 7)) << 4)) + (size_t)(k & 7) * 2;
            uint16_t hb;
            ok &= f32_to_f16_bits(v, &hb);
            blob[base + off / 2] = hb;
        }
    return ok;
}

struct TcState {
    tc::Params p;
};

}  // namespace

static bool tc_model_ok(const Model& m) {
    return m.phi_kind <= WM_PHI_STRUCT && m.kind == WM_KIND_MLP_LN && m.dtype == WM_DTYPE_BF16 && m.embed == WM_EMBED_LINEAR && m.d == tc::D &&
           m.d_a == tc::DA && m.hidden >= 256 && m.hidden <= tc::MAX_HID && m.hidden % 128 == 0 &&
           ((m.n_lin == 3 && m.sdim[1] == tc::SW && m.sdim[2] == tc::SW) || m.ranker_kind == WM_RANKER_FOREST) && m.H >= 8 && m.H <= tc::MAX_H && m.H % 8 == 0 &&
           m.n_types <= tc::MAX_TYPES && m.P <= tc::MAX_P;
}

int tc_prepare(wm_ctx* ctx, const std::vector<std::vector<float>>& hv, const std::vector<std::string>& names) {
    Model& m = ctx->m;
    m.tc_ok = 0;
    if (!tc_model_ok(m)) {   // d = 512 MLP+LN models and the GRU model: the CTA-pair kernels
        const int rc = tc2_prepare(ctx, hv, names);
        if (rc != WM_OK || m.tc_ok) return rc;
        const int rc2 = tcg_prepare(ctx, hv, names);
        if (rc2 != WM_OK || m.tc_ok) return rc2;
        // TransH models (NEXT row f1): the TransH step of the pair kernel (tc_ok 4: no single-CTA form); models with the
        // per-type phi (S28): the pair kernel for the rollout, the fp32 kernel for phi + scorer (wm_rollout_score)
        if (m.kind == WM_KIND_TRANSH || m.phi_kind == WM_PHI_TYPED) {
            const int rc4 = tcp_prepare(ctx, hv, names);
            if (rc4 != WM_OK) return rc4;
            if (m.tcp_ok) m.tc_ok = 4;
            if (m.tcp_ok && m.phi_kind == WM_PHI_TYPED) {      // ... and the tcgen05 ranking MLP over [z_T | phi | h] rows
                const int rc5 = tsc_prepare(ctx, hv, names);
                if (rc5 != WM_OK) return rc5;
            }
        }
        return WM_OK;
    }
    // the pair form (wm_tcp_kernel) of the same model, taken by default when built; then the single-CTA form
    {
        const int rc = tcp_prepare(ctx, hv, names);
        if (rc != WM_OK) return rc;
        if (m.tcp_ok) m.tc_ok = 1;
    }
    const tc::SmemLayout L = tc::smem_layout(m.n_types, m.hidden, (m.H + 15) / 16, m.phi_kind == WM_PHI_STRUCT);
    if ((int)L.total > ctx->smem_optin) return WM_OK;      // (e.g. many action types: the embedding table does not fit)
    auto get = [&](const char* n) -> const std::vector<float>& {
        for (size_t i = 0; i < names.size(); ++i)
            if (names[i] == n) return hv[i];
        static const std::vector<float> empty;
        return empty;
    };
    const std::vector<float>&W1 = get("W1"), &W2 = get("W2"), &Ws0 = get("Ws0"), &Ws1 = get("Ws1"), &E = get("E");
    const int hid = m.hidden, NC = hid / 128, K1 = tc::D + tc::DA;
    const int F = m.phi_dim, K0 = tc::D + F + m.H;   // scorer input [z ; phi (F <= 128 columns) ; hw]
    std::vector<uint16_t> blob;
    bool ok = true;   // every weight finite in fp16
    blob.reserve((size_t)(NC * 10 + tc::SC_TILES) * tc::TILE_BYTES / 2);
    auto g2 = [&](int c) {   // GEMM2 chunk c: K halves of the hidden chunk x N halves of d
        for (int ks = 0; ks < 2; ++ks)
            for (int h = 0; h < 2; ++h) ok &= append_tile(blob, W2, hid, h * 128, c * 128 + ks * 64, 64);
    };
    // same order as the MMA warp: a K-blocks of chunks 0 and 1, z K-blocks of chunks 0 and 1, G2(0), then G1(i), G2(i-1)
    auto g1_part = [&](int c, int k0, int k1) {
        for (int k = k0; k < k1; ++k) ok &= append_tile(blob, W1, K1, c * 128, k * 64, 64);
    };
    g1_part(0, 4, 6); g1_part(1, 4, 6); g1_part(0, 0, 4); g1_part(1, 0, 4);
    g2(0);
    for (int i = 2; i <= NC; ++i) {
        if (i < NC) { g1_part(i, 4, 6); g1_part(i, 0, 4); }   // GEMM1 chunk i: K-blocks a (4, 5), then z (0..3)
        g2(i - 1);
    }
    // phi weights of scorer layer 1 as the kernel's phi K-blocks see them, [SW][128].  WM_PHI_STRUCT: the F columns of
    // Ws0 as they are.  WM_PHI_MEAN: the mean action embedding is linear in psi = [count_c / len | sum log2 p_j / len | 1]
    // (see the action warps), so its weights are Ws0_phi E^T, Ws0_phi W_p and Ws0_phi b_p, summed in double here.
    // Forest models (WM_RANKER_FOREST) run this kernel for the rollout only (terminal latents -> wm_forest_kernel): their
    // scorer image is all zero and its result is never stored.
    const bool forest = m.ranker_kind == WM_RANKER_FOREST;
    std::vector<float> Wphi((size_t)tc::SW * 128, 0.0f);
    if (forest) {
    } else if (m.phi_kind == WM_PHI_STRUCT) {
        for (int n = 0; n < tc::SW; ++n)
            for (int c = 0; c < F; ++c) Wphi[(size_t)n * 128 + c] = Ws0[(size_t)n * K0 + tc::D + c];
    } else {
        const std::vector<float>&Wp = get("W_p"), &bpv = get("b_p");
        for (int n = 0; n < tc::SW; ++n) {
            const float* wr = &Ws0[(size_t)n * K0 + tc::D];
            for (int c = 0; c < m.n_types; ++c) {
                double acc = 0.0;
                for (int k = 0; k < tc::DA; ++k) acc += (double)wr[k] * E[(size_t)c * tc::DA + k];
                Wphi[(size_t)n * 128 + c] = (float)acc;
            }
            for (int j = 0; j < m.P; ++j) {
                double acc = 0.0;
                for (int k = 0; k < tc::DA; ++k) acc += (double)wr[k] * Wp[(size_t)k * m.P + j];
                Wphi[(size_t)n * 128 + m.n_types + j] = (float)acc;
            }
            double acc = 0.0;
            for (int k = 0; k < tc::DA; ++k) acc += (double)wr[k] * bpv[k];
            Wphi[(size_t)n * 128 + m.n_types + m.P] = (float)acc;
        }
    }
    for (int c = 0; c < 4; ++c) {     // scorer layer 1: phi (2), hw + an all-zero padding tile, z (4)
        ok &= append_tile(blob, Wphi, 128, c * 128, 0, 64);
        ok &= append_tile(blob, Wphi, 128, c * 128, 64, 64);
        ok &= append_tile(blob, Ws0, K0, c * 128, tc::D + F, forest ? 0 : m.H);
        ok &= append_tile(blob, Ws0, K0, c * 128, tc::D + F, 0);
        for (int kb = 0; kb < 4; ++kb) ok &= append_tile(blob, Ws0, K0, c * 128, kb * 64, forest ? 0 : 64);
    }
    for (int c = 0; c < 4; ++c)       // scorer layer 2
        for (int kb = 0; kb < 8; ++kb) ok &= append_tile(blob, Ws1, tc::SW, c * 128, kb * 64, forest ? 0 : 64);

    if (!ok) return WM_OK;   // a weight beyond the fp16 range: this model stays on the fp32 kernel

    void* d_blob = nullptr;
    WM_CUDA_TRY(cudaMalloc(&d_blob, blob.size() * 2));
    ctx->allocs.push_back(d_blob);
    WM_CUDA_TRY(cudaMemcpy(d_blob, blob.data(), blob.size() * 2, cudaMemcpyHostToDevice));
    std::vector<uint16_t> e16(E.size());
    for (size_t i = 0; i < E.size(); ++i) e16[i] = f32_to_bf16(E[i]);
    void* d_e = nullptr;
    WM_CUDA_TRY(cudaMalloc(&d_e, e16.size() * 2 + 16));
    ctx->allocs.push_back(d_e);
    WM_CUDA_TRY(cudaMemcpy(d_e, e16.data(), e16.size() * 2, cudaMemcpyHostToDevice));
    m.tc_blob = d_blob;
    m.tc_blob_bytes = blob.size() * 2;
    m.tc_E = d_e;
    if (m.phi_kind == WM_PHI_STRUCT) {
        WM_CUDA_TRY(cudaFuncSetAttribute(tc::wm_tc_kernel<WM_PHI_STRUCT, false>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.total));
        WM_CUDA_TRY(cudaFuncSetAttribute(tc::wm_tc_kernel<WM_PHI_STRUCT, true>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.total));
    } else {
        WM_CUDA_TRY(cudaFuncSetAttribute(tc::wm_tc_kernel<WM_PHI_MEAN, false>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.total));
        WM_CUDA_TRY(cudaFuncSetAttribute(tc::wm_tc_kernel<WM_PHI_MEAN, true>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.total));
    }
    m.tc_ok = 1;
    m.tc1_ok = 1;
    return WM_OK;
}

int tc_supported(const wm_ctx* ctx) { return ctx->m.tc_ok; }

int launch_tc(wm_ctx* ctx, Workspace* ws, const CallArgs& a, cudaStream_t st) {
    const Model& m = ctx->m;
    // per-call conditions the kernel relies on; otherwise the fp32 kernel takes the call
    // (the EXT kernels store latents as float4: a latents_out view that is only 4-byte aligned goes to the fp32 kernel)
    const bool aligned = ((uintptr_t)a.init_states % 16 == 0) && ((uintptr_t)a.hw_feats % 16 == 0) &&
                         ((uintptr_t)a.latents_out % 16 == 0);
    const bool prefix_call = a.start || a.init_index || a.latents_out;   // wm_rollout_latents / wm_rollout_score_from
    const bool use_pair = m.tcp_ok && (ctx->opt_pair || !m.tc1_ok);      // d = 256 models: the pair kernel takes the call
    const bool ext_ok = m.tc_ok >= 1 && m.tc_ok <= 4;                      // every tcgen05 kernel takes the prefix-reuse calls
    if (prefix_call && !ext_ok && ctx->opt_path != 2) return launch_generic(ctx, a, st);
    // per-type phi: the rollout kernels hold no scorer for it (wm_rollout_score / wm_rollout_score_from split the call
    // themselves, wm_api.cu); a call that still wants scores from them (wm_rollout_score_static; a prefix call of a model
    // without the tcgen05 ranking MLP) runs on the fp32 kernel
    if (m.phi_kind == WM_PHI_TYPED && a.scores_out) {
        if (ctx->opt_path == 2) {
            set_error("tcgen05 path: a WM_PHI_TYPED model is scored by wm_rollout_score only");
            return WM_ERR_UNSUPPORTED;
        }
        return launch_generic(ctx, a, st);
    }
    if (!m.tc_ok || a.T_max > 255 || !aligned || (prefix_call && !ext_ok)) {
        if (ctx->opt_path == 2) {
            set_error("tcgen05 path: needs T_max <= 255, 16-byte aligned init_states / hw_feats (and, for "
                      "wm_rollout_latents / wm_rollout_score_from, a 16-byte aligned latents_out)");
            return WM_ERR_UNSUPPORTED;
        }
        return launch_generic(ctx, a, st);
    }
    if (m.tc_ok == 2) return launch_tc2(ctx, ws, a, st);
    if (m.tc_ok == 3) return launch_tcg(ctx, ws, a, st);
    if (use_pair) return launch_tcp(ctx, ws, a, st);
    tc::Params p;
    p.hid = m.hidden; p.nc = m.hidden / 128; p.n_types = m.n_types; p.P = m.P; p.H = m.H;
    p.hw_ksteps = (m.H + 15) / 16;
    p.ln_eps = m.ln_eps;
    p.blob = static_cast<const uint8_t*>(m.tc_blob);
    p.E = static_cast<const __nv_bfloat16*>(m.tc_E);
    p.WpT = m.WpT; p.bp = m.bp; p.b1 = m.b1; p.b2 = m.b2; p.gamma = m.gamma; p.beta = m.beta;
    p.bs0 = m.bs[0]; p.bs1 = m.bs[1]; p.w3 = m.Wst[2]; p.bs2 = m.bs[2];
    if (m.ranker_kind == WM_RANKER_FOREST) p.bs0 = p.bs1 = p.w3 = p.bs2 = m.zeros;   // (unused scorer, zero image)
    p.a = a;
    p.n_tiles = (int)((a.B + tc::TM - 1) / tc::TM);
    p.tile_counter = ws->counters + kTileCtrOff;
    WM_CUDA_TRY(cudaMemsetAsync(p.tile_counter, 0, sizeof(int), st));
    p.prof = trace::begin(st);
    const tc::SmemLayout L = tc::smem_layout(m.n_types, m.hidden, p.hw_ksteps, m.phi_kind == WM_PHI_STRUCT);
    const int grid = p.n_tiles < ctx->n_sms ? p.n_tiles : ctx->n_sms;
    if (m.phi_kind == WM_PHI_STRUCT) {
        if (prefix_call) tc::wm_tc_kernel<WM_PHI_STRUCT, true><<<grid, tc::THREADS, L.total, st>>>(p);
        else tc::wm_tc_kernel<WM_PHI_STRUCT, false><<<grid, tc::THREADS, L.total, st>>>(p);
    } else {
        if (prefix_call) tc::wm_tc_kernel<WM_PHI_MEAN, true><<<grid, tc::THREADS, L.total, st>>>(p);
        else tc::wm_tc_kernel<WM_PHI_MEAN, false><<<grid, tc::THREADS, L.total, st>>>(p);
    }
    WM_CUDA_TRY(cudaGetLastError());
    ctx->launches.fetch_add(1);
    trace::dump(p.prof, st);
    return WM_OK;
}

}  // namespace wm

// K2 (tcgen05, CTA pair, gated): fused persistent rollout + score kernel for the bf16 GRU-style transition with
// d = 384, d_a = 128 and the bucketed action-parameter table (BASELINE.json cfg 5), sm_100a only.
//
// PAPER.md:162 Eq.8 / :166 — z_t = F(z_{t-1}, a_t) applied recurrently; :176 — masked steps leave z unchanged;
// :186-188 Eq.12 — y = G([z_T ; phi ; h]).  Parametrisation (BASELINE.json cfg 5, DESIGN.md §3 S10):
//   g = sigma(W_g [z;a]),  r = sigma(W_r [z;a]),  z' = (1 - g) z + g tanh(W_h [r*z ; a]),  a = sum_j Tbl[slot_j row].
//
// A cluster of two CTAs owns a tile of 128 candidates, 64 rows each; the leader issues tcgen05.mma.cta_group::2 with
// M = 128, N = 192 (d = 2 N tiles).  Per CTA, a D tile is 64 rows x 192 columns held as 128 lanes x 96 columns (lane
// l: row l % 64, columns 96 (l / 64) ...).  Tensor memory (512 columns): the fp32 master latent (2 x 96) and three
// 96-column accumulators X0..X2.  Per step the MMA warp issues six N tiles of K = 512 in the order
//     R_0 -> X2, R_1 -> X1, G_0 -> X0, H_0 -> X2, H_1 -> X1, G_1 -> X0
// (H_j needs all of r*z, i.e. both R epilogues; G_1 reuses G_0's accumulator once blend_0 has read it), while the
// epilogue warps turn R_j into the fp16 operand r*z (shared memory) and (G_j, H_j) into z' (fp32 -> TMEM, fp16 ->
// shared memory: z'_0 goes to the OTHER of two buffers of K-blocks 0-2, because G_1 still reads the old z while z'_0 is
// written; z'_1 overwrites K-blocks 3-5 in place, G_1 having completed before blend_1 starts).  z'_0 and z'_1 are
// published separately, so R_0 of step t+1 runs its first five K-blocks (z'_0 and a_{t+1}) under blend_1 of step t.
// A ring stage is TWO [192 x 64] weight tiles (8 MMAs per wait / commit: the issuing warp, not the tensor pipe, was
// the limiter with one tile per stage).  Everything else — weight ring fed by TMA into both CTAs with completion on
// the leader's barrier, multicast commits, remote arrivals, static serpentine tile schedule, scorer on the same
// machinery — is as in wm_tc2.cu.
// Warp roles per CTA (512 threads): warps 0-7 epilogue (q = warp % 4: rows 32 (q & 1) + lane, N half q / 2; e = warp / 4:
// 48-column half of the 96-column buffer), warps 8-11 action embedding (bucket-table gather), warp 12 TMEM allocator,
// warp 13 tile schedule + TMA producer, warp 15 MMA issuer (leader CTA only).
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

namespace tcg {

using namespace ptx;

constexpr int TMP = 128;           // candidates per pair tile (MMA M)
constexpr int TMR = 64;            // rows per CTA
constexpr int D = 384;             // latent width
constexpr int DA = 128;            // action-embedding width
constexpr int SW = 768;            // scorer hidden width (both hidden layers)
constexpr int NT = 192;            // MMA N (columns per tile)
constexpr int XC = NT / 2;         // TMEM columns per tile and CTA
constexpr int KB_BYTES = 8192;     // one A K-block: [64 rows x 64 cols] fp16, SW128 K-major
constexpr int BT_BYTES = 12288;    // one B half tile: [96 weight rows x 64 cols] fp16, SW128 K-major
constexpr int STG_BYTES = 2 * BT_BYTES;   // a ring stage: two half tiles per CTA
constexpr int NSTAGE = 3;
constexpr int Z_KB = 6, A_KB = 2;  // K-blocks of the z part / the a (phi) part of an operand
constexpr int ZH_KB = Z_KB / 2;    // K-blocks of one 192-column latent tile
constexpr int ZH_BYTES = ZH_KB * KB_BYTES;
constexpr int ZB_BYTES = Z_KB * KB_BYTES;
constexpr int HWK_BYTES = 2048;    // hw operand: one [64 x 16] no-swizzle K-major tile per K = 16 step
constexpr int THREADS = 512;
constexpr int EPI_WARP0 = 0, ACT_WARP0 = 8, ALLOC_WARP = 12, PROD_WARP = 13, MMA_WARP = 15;
constexpr int MAX_P = 8, MAX_H = 64, MAX_BUCKETS = 64;
constexpr int TILE_STAGES = (A_KB + Z_KB) / 2;            // ring stages of one N tile of the rollout
constexpr int ROLL_STAGES = 6 * TILE_STAGES;              // per step
constexpr int SC_STAGES = 4 * (1 + 1 + Z_KB / 2) + 2 * 12; // scorer: layer 1 (4 x (phi pair, hw, 3 z pairs)), layer 2 (2 rounds x 12)
constexpr uint32_t IDESC_G = idesc_pair(NT);
constexpr int NXB = 5;             // accumulators: X0, X1, X2 and, in the scorer, the two (dead) latent tiles

enum {
    B_FULL = 0,                    // [NSTAGE] TMA (both CTAs) -> leader's MMA warp
    B_EMPTY = B_FULL + NSTAGE,     // [NSTAGE] MMA commit (multicast) -> each CTA's producer
    B_XFULL = B_EMPTY + NSTAGE,    // [NXB] MMA commit -> epilogue: accumulator b filled
    B_XFREE = B_XFULL + NXB,       // [NXB] epilogue (both CTAs) -> leader MMA: accumulator b read, its output written
    B_ZREADY = B_XFREE + NXB,      // [2] epilogue (both CTAs) -> leader MMA: z' tile 0 / tile 1 written
    B_AFREE = B_ZREADY + 2,                       // MMA commit -> action warps: a-part no longer read
    B_AREADY,                      // action warps (both CTAs) -> leader MMA: a-part written
    B_SFULL,                       // [2] schedule slot filled (CTA-local)
    B_SEMPTY = B_SFULL + 2,        // [2] schedule slot consumed (CTA-local)
    B_COUNT = B_SEMPTY + 2
};

struct Params {
    int n_types, P, n_buckets, H, hw_ksteps;
    const __nv_bfloat16* Tbl;   // [n_types * P * n_buckets][128]
    const float *bs0, *bs1, *w3, *bs2;
    CallArgs a;
    int n_tiles;
    unsigned long long* prof;   // developer trace buffer (wm_trace.cuh), null in a normal build
};

struct SmemLayout {
    uint32_t zbuf, abuf, rz, ring, hwk, idx, lens, red, bars, sched, tmem_slot, total;
};

__host__ __device__ inline SmemLayout smem_layout(int hw_ksteps) {
    SmemLayout L;
    uint32_t o = 0;
    L.zbuf = o; o += 3 * ZH_BYTES;                     // fp16 z operand: K-blocks 0-2 twice (double-buffered), then 3-5
    L.abuf = o; o += A_KB * KB_BYTES;                  // fp16 a_t / phi
    L.rz = o; o += ZB_BYTES;                           // fp16 r*z
    L.ring = o; o += NSTAGE * STG_BYTES;
    L.hwk = o; o += (uint32_t)hw_ksteps * HWK_BYTES;
    L.idx = o; o += TMR * MAX_P * 4;                   // table row of every parameter slot of the step
    L.lens = o; o += TMR * 4;
    L.red = o; o += 4 * TMR * 4;                       // [4 column parts][64 rows] float
    L.bars = o; o += B_COUNT * 8;
    L.sched = o; o += 2 * 8;
    L.tmem_slot = o; o += 16;
    L.total = o;
    return L;
}

__device__ __forceinline__ int tile_of(int it, int pair, int np, int n_tiles) {
    const int idx = it * np + ((it & 1) ? np - 1 - pair : pair);
    return idx < n_tiles ? idx : -1;
}

// EXT = the prefix-latent reuse calls (S26; as in wm_tcp_kernel / wm_tc2_kernel): a per-candidate first position
// `start` (the rollout covers [start, len), phi still sees [0, len)), the initial latent from a bank row, z' stored to
// latents_out, and no scorer when scores_out is null.  Compiled out of the literal instance.
template <bool EXT>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(THREADS, 1)
wm_tcg_kernel(const Params p, const __grid_constant__ CUtensorMap tmap) {
    extern __shared__ __align__(1024) uint8_t smem[];
    const SmemLayout L = smem_layout(p.hw_ksteps);
    const uint32_t s_base = smem_u32(smem);
    const uint32_t s_z = s_base + L.zbuf, s_a = s_base + L.abuf, s_rz = s_base + L.rz, s_ring = s_base + L.ring;
    const uint32_t s_bars = s_base + L.bars;
    auto bar = [&](int i) -> uint32_t { return s_bars + 8u * (uint32_t)i; };
    volatile int* s_sched = reinterpret_cast<volatile int*>(smem + L.sched);   // [2][2]: tile, nsteps
    float* s_red = reinterpret_cast<float*>(smem + L.red);                     // [4][64]

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();          // 0 = leader (issues the MMAs)
    const int pair = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;
    const bool rank_it = !EXT || p.a.scores_out != nullptr;   // EXT calls that only store latents skip the scorer in every role

    // ---- one-time setup
    if (threadIdx.x == 0) {
        for (int i = 0; i < NSTAGE; ++i) { mbar_init(bar(B_FULL + i), 1); mbar_init(bar(B_EMPTY + i), 1); }
        for (int i = 0; i < NXB; ++i) { mbar_init(bar(B_XFULL + i), 1); mbar_init(bar(B_XFREE + i), 16); }
        for (int i = 0; i < 2; ++i) { mbar_init(bar(B_SFULL + i), 1); mbar_init(bar(B_SEMPTY + i), 13); }
        mbar_init(bar(B_ZREADY), 16);
        mbar_init(bar(B_ZREADY + 1), 16);
        mbar_init(bar(B_AFREE), 1);
        mbar_init(bar(B_AREADY), 8);
        fence_barrier_init();
        fence_proxy_async();
    }
    if (warp == ALLOC_WARP) tmem_alloc2(s_base + L.tmem_slot, 512);
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
    const uint32_t T_Z = tmem_base;                 // fp32 latent: two 96-column tiles
    const uint32_t T_X = tmem_base + 2 * XC;        // accumulators X0, X1, X2
    // TMEM column base of accumulator b (3, 4 = the latent tiles, free once the rollout of a tile is over)
    auto xcol = [&](int b) -> uint32_t { return b < 3 ? T_X + (uint32_t)(XC * b) : T_Z + (uint32_t)(XC * (b - 3)); };

    // Register hand-over (setmaxnreg works per warpgroup of four warps): the two epilogue warpgroups give up 16
    // registers per thread, the action warpgroup (8-11) takes them: it holds a whole step's 16 embedded rows per warp in
    // registers while the a-buffer is still being read, so that only the stores stand between the buffer's release and
    // the next step's first a K-block.
    if (warp == PROD_WARP) {
        // =============================================================== tile schedule + TMA producer
        uint32_t stage = 0, ph = 0;
        for (uint32_t it = 0;; ++it) {
            const uint32_t slot = it & 1;
            const int tile = tile_of((int)it, pair, n_pairs, p.n_tiles);
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
                const int roll_total = nsteps * ROLL_STAGES, total = roll_total + (rank_it ? SC_STAGES : 0);
                int src = 0;
                for (int i = 0; i < total; ++i) {
                    if (i == roll_total) src = ROLL_STAGES;
                    else if (i < roll_total && src == ROLL_STAGES) src = 0;
                    mbar_wait(bar(B_EMPTY + stage), ph ^ 1);
                    // the leader's barrier collects both CTAs' halves of the stage's two [192 x 64] tiles
                    if (rank == 0) mbar_arrive_expect_tx(bar(B_FULL + stage), 2 * STG_BYTES);
                    tma_load_2sm(s_ring + stage * STG_BYTES, &tmap, 0, 2 * XC * (2 * src + (int)rank), bar(B_FULL + stage));
                    ++src;
                    if (++stage == NSTAGE) { stage = 0; ph ^= 1; }
                }
            }
            __syncwarp();
        }
    } else if (warp == MMA_WARP) {
        // =============================================================== MMA issuer (leader CTA; the peer's warp only
        // follows the schedule so that both CTAs' slot barriers have the same arrival count)
        uint32_t stage = 0, ph = 0;
        uint32_t n_z = 0, n_a = 0;
        uint32_t pend = 0, xpar = 0;     // per accumulator: a commit is outstanding / parity of its XFREE barrier
        const uint32_t s_hwk = s_base + L.hwk;
        WM_TRACE_DECL(p.prof, 0)
        auto wait_x = [&](int b) {       // accumulator b read by the epilogue (and that epilogue's output written)
            if ((pend >> b) & 1u) {
                WM_TRACE(10 + b);
                mbar_wait(bar(B_XFREE + b), (xpar >> b) & 1u);
                WM_TRACE(15);
                xpar ^= 1u << b;
                pend &= ~(1u << b);
                tc_fence_after();
            }
        };
        auto wait_full = [&]() {
            WM_TRACE(1);
            mbar_wait(bar(B_FULL + stage), ph);
            WM_TRACE(2);
            tc_fence_after();
        };
        auto advance = [&]() {
            __syncwarp();
            WM_TRACE(3);
            if (++stage == NSTAGE) { stage = 0; ph ^= 1; }
        };
        // A ring stage holds two [192 x 64] B tiles; each goes against one [64(+64) x 64] A K-block: 4 MMAs of K = 16.
        // tile_mma is called by the elected lane only.
        auto tile_mma = [&](uint32_t d_tmem, uint32_t a_tile, int i, bool first) {
            const uint64_t a0 = smem_desc(a_tile), b0 = smem_desc(s_ring + stage * STG_BYTES + i * BT_BYTES);
#pragma unroll
            for (int j = 0; j < 4; ++j) mma_ss2(d_tmem, a0 + 2u * j, b0 + 2u * j, IDESC_G, (first && j == 0) ? 0u : 1u);
        };
        auto stage_end = [&]() {
            if (elect_one()) mma_commit2(bar(B_EMPTY + stage));
            advance();
        };
        // both tiles of the stage in one go: (accumulator, A K-block) x 2
        auto stage2 = [&](uint32_t d0, uint32_t a_tile0, bool first0, uint32_t d1, uint32_t a_tile1, bool first1) {
            wait_full();
            if (elect_one()) {
                tile_mma(d0, a_tile0, 0, first0);
                tile_mma(d1, a_tile1, 1, first1);
                mma_commit2(bar(B_EMPTY + stage));
            }
            advance();
        };
        auto half = [&](uint32_t d, uint32_t a_tile, int i, bool first) {     // one tile of an open stage
            if (elect_one()) tile_mma(d, a_tile, i, first);
            __syncwarp();
        };
        auto stage_hw = [&](uint32_t d_tmem) {       // the stage's second tile is padding
            wait_full();
            const uint64_t b0 = smem_desc(s_ring + stage * STG_BYTES);
            if (elect_one()) {
                for (int j = 0; j < p.hw_ksteps; ++j)
                    mma_ss2(d_tmem, smem_desc_nosw(s_hwk + j * HWK_BYTES), b0 + 2u * j, IDESC_G, 1u);
                mma_commit2(bar(B_EMPTY + stage));
            }
            advance();
        };
        auto commit = [&](int barrier) {
            if (elect_one()) mma_commit2(bar(barrier));
            __syncwarp();
        };
        auto finish = [&](int b) {
            commit(B_XFULL + b);
            pend |= 1u << b;
        };
        // the a (or phi) K-block pair; `first` starts the accumulation
        auto seg_a = [&](int b, bool first) { stage2(xcol(b), s_a, first, xcol(b), s_a + KB_BYTES, false); };
        // six z-like K-blocks as three stages: K-blocks 0-2 at lo, 3-5 at hi
        auto seg_z = [&](int b, uint32_t lo, uint32_t hi, bool first) {
            stage2(xcol(b), lo, first, xcol(b), lo + KB_BYTES, false);
            stage2(xcol(b), lo + 2 * KB_BYTES, false, xcol(b), hi, false);
            stage2(xcol(b), hi + KB_BYTES, false, xcol(b), hi + 2 * KB_BYTES, false);
        };
        auto wait_a = [&]() { WM_TRACE(20); mbar_wait(bar(B_AREADY), n_a & 1); WM_TRACE(21); ++n_a; tc_fence_after(); };
        auto wait_z = [&](int j) {
            WM_TRACE(22 + 2 * j);
            mbar_wait(bar(B_ZREADY + j), (n_z >> j) & 1);
            WM_TRACE(23 + 2 * j);
            n_z ^= 1u << j;
            tc_fence_after();
        };
        const uint32_t s_zhi = s_z + 2 * ZH_BYTES, s_rzhi = s_rz + ZH_BYTES;
        for (uint32_t it = 0;; ++it) {
            const uint32_t slot = it & 1;
            mbar_wait(bar(B_SFULL + slot), (it >> 1) & 1);
            const int tile = s_sched[slot * 2 + 0], nsteps = s_sched[slot * 2 + 1];
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(B_SEMPTY + slot));
            if (tile < 0) break;
            if (rank != 0) continue;
#pragma unroll 1
            for (int t = 0; t < nsteps; ++t) {
                WM_TRACE(30);
                const uint32_t zlo = s_z + (uint32_t)(t & 1) * ZH_BYTES;    // fp16 z_t, K-blocks 0-2 (3-5 are at s_zhi)
                // R_0 -> X2 starts on z'_0 (tile 0 of the previous blend) and a_t while blend_1 of step t-1 is still
                // running: K-blocks z0 z1 | z2 a0 | a1 z3 | z4 z5
                wait_x(2); wait_z(0);
                stage2(xcol(2), zlo, true, xcol(2), zlo + KB_BYTES, false);
                wait_full(); half(xcol(2), zlo + 2 * KB_BYTES, 0, false); wait_a(); half(xcol(2), s_a, 1, false); stage_end();
                wait_full(); half(xcol(2), s_a + KB_BYTES, 0, false); wait_z(1); half(xcol(2), s_zhi, 1, false); stage_end();
                stage2(xcol(2), s_zhi + KB_BYTES, false, xcol(2), s_zhi + 2 * KB_BYTES, false);
                finish(2);
                wait_x(1); seg_z(1, zlo, s_zhi, true); seg_a(1, false); finish(1);               // R_1 -> X1
                wait_x(0); seg_z(0, zlo, s_zhi, true); seg_a(0, false); finish(0);               // G_0 -> X0
                wait_x(2); wait_x(1);                                       // r*z complete, X2 / X1 read
                seg_a(2, true); seg_z(2, s_rz, s_rzhi, false); finish(2);   // H_0 -> X2
                seg_a(1, true); seg_z(1, s_rz, s_rzhi, false); finish(1);   // H_1 -> X1
                wait_x(0);                                                  // blend_0 has read G_0
                seg_a(0, true); commit(B_AFREE); seg_z(0, zlo, s_zhi, false); finish(0);   // G_1 -> X0 (still the OLD z)
            }
            if (!rank_it) {     // no scorer: take the last z' phases so that the barrier parities stay in step
                wait_z(0);
                wait_z(1);
                continue;
            }
            // ---- scorer layer 1: four 192-column tiles of gelu(Ws0 [z_T; phi; hw] + bs0) into X2, X1, X0 and latent
            // tile 0; their fp16 outputs h1 go to the spare z K-blocks (tile 0), the r*z buffer (tiles 1, 2) and, once
            // every layer-1 MMA has completed, over z_T's K-blocks 3-5 (tile 3)
            const uint32_t zlo = s_z + (uint32_t)(nsteps & 1) * ZH_BYTES;   // z_T, K-blocks 0-2
            const uint32_t h1_0 = s_z + (uint32_t)((nsteps & 1) ^ 1) * ZH_BYTES;
            const int l1buf[4] = {2, 1, 0, 3};
#pragma unroll
            for (int n = 0; n < 4; ++n) {
                const int b = l1buf[n];
                wait_x(b);
                if (n == 0) wait_a();
                seg_a(b, true);
                stage_hw(xcol(b));
                if (n == 3) commit(B_AFREE);
                if (n == 0) { wait_z(0); wait_z(1); }
                seg_z(b, zlo, s_zhi, false);
                finish(b);
            }
            // ---- scorer layer 2, K = 768 as the four h1 tiles (3 K-blocks each), N = 768 in two rounds of two
            // 192-column tiles (a stage = one K-block of both): round 0 into latent tile 1 and X2, round 1 into X1 and X0
#pragma unroll
            for (int round = 0; round < 2; ++round) {
                const int b0 = round == 0 ? 4 : 1, b1 = round == 0 ? 2 : 0;
                if (round == 0) wait_x(4);
#pragma unroll 1
                for (int kc = 0; kc < 4; ++kc) {
                    if (round == 0) wait_x(kc == 0 ? 2 : kc == 1 ? 1 : kc == 2 ? 0 : 3);   // h1 tile kc written
                    const uint32_t a_base = kc == 0 ? h1_0 : kc == 1 ? s_rz : kc == 2 ? s_rzhi : s_zhi;
#pragma unroll 1
                    for (int kb = 0; kb < 3; ++kb)
                        stage2(xcol(b0), a_base + kb * KB_BYTES, kc == 0 && kb == 0, xcol(b1), a_base + kb * KB_BYTES,
                               kc == 0 && kb == 0);
                }
                commit(B_XFULL + b0);
                commit(B_XFULL + b1);
                pend |= (1u << b0) | (1u << b1);
            }
        }
        __syncwarp();
    }
    else if (warp >= EPI_WARP0 && warp < ACT_WARP0) {
        // =============================================================== epilogue warps (gates / blend / scorer)
        reg_dealloc<112>();
        const int q = warp & 3, e = (warp - EPI_WARP0) >> 2;
        const int rh = q & 1, nh = q >> 1;
        const int row = 32 * rh + lane;                 // row of this CTA's 64
        const int part = 2 * nh + e;                    // this thread's 48-column quarter of every 192-column tile
        const int cb = 48 * part;                       // first column of the quarter inside a tile
        const uint32_t lane_off = (uint32_t)(32 * q) << 16;
        const uint32_t tcol = 48u * e + lane_off;       // TMEM offset of the quarter inside a 96-column buffer
        uint8_t* zb = smem + L.zbuf;
        uint8_t* rzb = smem + L.rz;
        const uint32_t r_xfree0 = mapa(bar(B_XFREE), 0);      // leader's XFREE[b] = r_xfree0 + 8 b
        auto r_xfree = [&](int b) -> uint32_t { return r_xfree0 + 8u * (uint32_t)b; };
        const uint32_t r_zready = mapa(bar(B_ZREADY), 0);      // tile 0; tile 1 at + 8
        uint8_t* zhi = zb + 2 * ZH_BYTES;                      // fp16 z K-blocks 3-5 (latent tile 1)
        uint32_t fpar = 0;                              // parity of every XFULL barrier
        auto wait_full = [&](int b) {
            mbar_wait(bar(B_XFULL + b), (fpar >> b) & 1u);
            fpar ^= 1u << b;
            tc_fence_after();
        };
        // 16 fp16 values of this row at column m0 (multiple of 16) of a 192-wide operand region (3 K-blocks)
        auto put16 = [&](uint8_t* buf, int m0, const uint32_t (&o)[8]) {
            uint8_t* kb = buf + (m0 >> 6) * KB_BYTES;
            const int ch = (m0 & 63) >> 3;
            *reinterpret_cast<uint4*>(kb + sw128_off(row, ch)) = make_uint4(o[0], o[1], o[2], o[3]);
            *reinterpret_cast<uint4*>(kb + sw128_off(row, ch + 1)) = make_uint4(o[4], o[5], o[6], o[7]);
        };
        // arrive on up to two leader barriers after this warp's TMEM / shared-memory writes are visible
        auto publish = [&](uint32_t bar_a, uint32_t bar_b, uint32_t bar_c, bool tmem_written) {
            if (tmem_written) tmem_st_wait();
            fence_proxy_async();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) {
                mbar_arrive_remote(bar_a);
                if (bar_b) mbar_arrive_remote(bar_b);
                if (bar_c) mbar_arrive_remote(bar_c);
            }
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

            // ---- z_0 (the task's initial latent, or the banked latent after the first st steps) -> fp32
            // TMEM + fp16 buffer 0
#pragma unroll 1
            for (int js = 0; js < 6; ++js) {
                const int j = js / 3, s = js % 3;
                const int m0 = NT * j + cb + 16 * s;
                uint32_t v[16], o[8];
                if (cand >= 0) {
                    const float4* src = reinterpret_cast<const float4*>(p.a.init_states + zrow * D + m0);
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const float4 f = __ldg(src + i);
                        range_check(f, p.a.fault);
                        v[4 * i + 0] = __float_as_uint(f.x); v[4 * i + 1] = __float_as_uint(f.y);
                        v[4 * i + 2] = __float_as_uint(f.z); v[4 * i + 3] = __float_as_uint(f.w);
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < 16; ++i) v[i] = 0u;
                }
#pragma unroll
                for (int i = 0; i < 8; ++i) o[i] = pack_f16(__uint_as_float(v[2 * i]), __uint_as_float(v[2 * i + 1]));
                tmem_st16(T_Z + (uint32_t)(XC * j) + tcol + 16u * s, v);
                put16(j == 0 ? zb : zhi, cb + 16 * s, o);
            }
            publish(r_zready, r_zready + 8u, 0u, true);

            for (int t = 0; t < nsteps; ++t) {
                uint8_t* znext = zb + ((t & 1) ^ 1) * ZH_BYTES;     // z'_0 (K-blocks 0-2); z'_1 overwrites zhi
                const bool live = t < rem;     // masked steps leave the state unchanged
                float* lat = nullptr;          // wm_rollout_latents: z after this step (or only the terminal one: [B, d])
                if (EXT && p.a.latents_out && live) {
                    if (!p.a.latents_terminal) lat = p.a.latents_out + ((size_t)cand * p.a.T_max + st + t) * D;
                    else if (st + t == len - 1) lat = p.a.latents_out + (size_t)cand * D;
                }
                // ---- r = sigma(R_j), fp16 r*z -> the r*z operand buffer (R_0 in X2, R_1 in X1)
#pragma unroll 1
                for (int j = 0; j < 2; ++j) {
                    const int xb = j == 0 ? 2 : 1;
                    wait_full(xb);
#pragma unroll 1
                    for (int s = 0; s < 3; ++s) {
                        uint32_t x[16], z[16], o[8];
                        tmem_ld16(xcol(xb) + tcol + 16u * s, x);
                        tmem_ld16(T_Z + (uint32_t)(XC * j) + tcol + 16u * s, z);
                        tmem_ld_wait();
#pragma unroll
                        for (int i = 0; i < 8; ++i)
                            o[i] = pack_f16(sigmoid_fast(__uint_as_float(x[2 * i])) * __uint_as_float(z[2 * i]),
                                            sigmoid_fast(__uint_as_float(x[2 * i + 1])) * __uint_as_float(z[2 * i + 1]));
                        put16(rzb + j * ZH_BYTES, cb + 16 * s, o);
                    }
                    publish(r_xfree(xb), 0u, 0u, false);
                }
                // ---- z'_j = z + g (tanh(H_j) - z) = (1 - g) z + g h,  g = sigma(G_j)  (G_j in X0; H_0 in X2, H_1 in X1).
                // The blend is bound by the special-function unit (sigma and tanh: 2 of 16 per clock and SM for each of
                // 12,288 elements of a tile) and blend_1 is the serial section of a step (G_1 is the last tile), so
                // tanh(H_1) - z is applied IN PLACE to X1 as soon as H_1 completes, while G_1 is still running:
                // blend_1 then needs one special function and one FMA per element.
                auto blend = [&](int j, int xh, bool h_is_delta) {
#pragma unroll 1
                    for (int s = 0; s < 3; ++s) {
                        uint32_t g[16], h[16], z[16], o[8];
                        tmem_ld16(xcol(0) + tcol + 16u * s, g);
                        tmem_ld16(xcol(xh) + tcol + 16u * s, h);
                        tmem_ld16(T_Z + (uint32_t)(XC * j) + tcol + 16u * s, z);
                        tmem_ld_wait();
#pragma unroll
                        for (int i = 0; i < 16; ++i) {
                            const float zf = __uint_as_float(z[i]);
                            const float gf = sigmoid_fast(__uint_as_float(g[i]));
                            const float df = h_is_delta ? __uint_as_float(h[i]) : tanh_fast(__uint_as_float(h[i])) - zf;
                            z[i] = __float_as_uint(live ? fmaf(gf, df, zf) : zf);
                        }
#pragma unroll
                        for (int i = 0; i < 8; ++i) o[i] = pack_f16(__uint_as_float(z[2 * i]), __uint_as_float(z[2 * i + 1]));
                        tmem_st16(T_Z + (uint32_t)(XC * j) + tcol + 16u * s, z);
                        put16(j == 0 ? znext : zhi, cb + 16 * s, o);
                        if (EXT && lat) {
                            float4* dst = reinterpret_cast<float4*>(lat + NT * j + cb + 16 * s);
#pragma unroll
                            for (int i = 0; i < 4; ++i)
                                dst[i] = make_float4(__uint_as_float(z[4 * i]), __uint_as_float(z[4 * i + 1]),
                                                     __uint_as_float(z[4 * i + 2]), __uint_as_float(z[4 * i + 3]));
                        }
                    }
                    // tile j of z' is written: X0 and the H accumulator are free, R_0 of the next step may read z'_j
                    publish(r_xfree(0), r_xfree(xh), r_zready + 8u * (uint32_t)j, true);
                };
                wait_full(0);      // G_0
                wait_full(2);      // H_0
                blend(0, 2, false);
                wait_full(1);      // H_1: X1 <- tanh(H_1) - z (tile 1), off the critical path
#pragma unroll 1
                for (int s = 0; s < 3; ++s) {
                    uint32_t h[16], z[16];
                    tmem_ld16(xcol(1) + tcol + 16u * s, h);
                    tmem_ld16(T_Z + (uint32_t)XC + tcol + 16u * s, z);
                    tmem_ld_wait();
#pragma unroll
                    for (int i = 0; i < 16; ++i)
                        h[i] = __float_as_uint(tanh_fast(__uint_as_float(h[i])) - __uint_as_float(z[i]));
                    tmem_st16(xcol(1) + tcol + 16u * s, h);
                }
                tmem_st_wait();
                wait_full(0);      // G_1
                blend(1, 1, true);
            }

            if (!rank_it) continue;
            // ---- scorer layer 1 -> h1 (fp16): tile 0 into the spare z K-blocks, tiles 1, 2 into the r*z buffer, tile 3
            // over z_T's K-blocks 3-5 (its accumulator is the last of layer 1: every MMA that reads z_T has completed)
            uint8_t* h1_0 = zb + ((nsteps & 1) ^ 1) * ZH_BYTES;
#pragma unroll 1
            for (int n = 0; n < 4; ++n) {
                const int xb = n == 0 ? 2 : n == 1 ? 1 : n == 2 ? 0 : 3;
                wait_full(xb);
#pragma unroll 1
                for (int s = 0; s < 3; ++s) {
                    uint32_t x[16], o[8];
                    tmem_ld16(xcol(xb) + tcol + 16u * s, x);
                    tmem_ld_wait();
                    const int m0 = NT * n + cb + 16 * s;
                    const float4* bp_ = reinterpret_cast<const float4*>(p.bs0 + m0);
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const float4 bv = __ldg(bp_ + i);
                        o[2 * i] = gelu2_f16(make_float2(__uint_as_float(x[4 * i]), __uint_as_float(x[4 * i + 1])),
                                             make_float2(bv.x, bv.y));
                        o[2 * i + 1] = gelu2_f16(make_float2(__uint_as_float(x[4 * i + 2]), __uint_as_float(x[4 * i + 3])),
                                                 make_float2(bv.z, bv.w));
                    }
                    put16(n == 0 ? h1_0 : n == 1 ? rzb : n == 2 ? rzb + ZH_BYTES : zhi, cb + 16 * s, o);
                }
                publish(r_xfree(xb), 0u, 0u, false);
            }
            // ---- scorer layer 2 + output dot product: N tiles 0..3 arrive in latent tile 1, X2, X1, X0
            float acc = 0.0f;
#pragma unroll 1
            for (int n = 0; n < 4; ++n) {
                const int xb = n == 0 ? 4 : n == 1 ? 2 : n == 2 ? 1 : 0;
                wait_full(xb);
#pragma unroll 1
                for (int s = 0; s < 3; ++s) {
                    uint32_t x[16];
                    tmem_ld16(xcol(xb) + tcol + 16u * s, x);
                    tmem_ld_wait();
                    const int n0 = NT * n + cb + 16 * s;
#pragma unroll
                    for (int i = 0; i < 16; ++i)
                        acc = fmaf(gelu_fast(__uint_as_float(x[i]) + __ldg(p.bs1 + n0 + i)), __ldg(p.w3 + n0 + i), acc);
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_remote(r_xfree(xb));
            }
            s_red[part * TMR + row] = acc;
            named_bar_sync(1 + rh, 128);
            if (part == 0 && cand >= 0)
                p.a.scores_out[cand] = (s_red[row] + s_red[TMR + row]) + (s_red[2 * TMR + row] + s_red[3 * TMR + row]) +
                                       __ldg(p.bs2);
            named_bar_sync(1 + rh, 128);   // s_red is reused by the next tile
        }
    }
    else if (warp >= ACT_WARP0 && warp < ACT_WARP0 + 4) {
        // =============================================================== action-embedding warps
        // warp aw owns rows [16 aw, 16 aw + 16).  Phase 1 is row-mapped (lanes 0-15: table row of every parameter
        // slot), phase 2 column-mapped (lane = 4 embedding columns: gather P table rows per candidate row and add).
        reg_alloc<160>();
        const int aw = warp - ACT_WARP0;
        const int row = 16 * aw + (lane & 15);
        const bool row_lane = lane < 16;
        const int col4 = 4 * lane;
        uint8_t* ab = smem + L.abuf;
        int* s_idx = reinterpret_cast<int*>(smem + L.idx);
        int* s_lens = reinterpret_cast<int*>(smem + L.lens);
        const uint32_t r_aready = mapa(bar(B_AREADY), 0);
        const int P = p.P, NB = p.n_buckets;
        uint32_t n_w = 0;
        auto a_dst = [&](int r) -> uint2* {
            return reinterpret_cast<uint2*>(ab + (lane >> 4) * KB_BYTES + sw128_off(r, (lane & 15) >> 1) + (lane & 1) * 8);
        };
        for (uint32_t it = 0;; ++it) {
            const uint32_t slot = it & 1;
            mbar_wait_inline(bar(B_SFULL + slot), (it >> 1) & 1);
            const int tile = s_sched[slot * 2 + 0], nsteps = s_sched[slot * 2 + 1];
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(B_SEMPTY + slot));
            if (tile < 0) break;
            int cand = -1, len = 0, seg = 0;
            if (row_lane) row_meta(p.a, (int64_t)tile * TMP + TMR * (int)rank + row, cand, len, seg, false);
            float phi[16][4];
#pragma unroll
            for (int rr = 0; rr < 16; ++rr) phi[rr][0] = phi[rr][1] = phi[rr][2] = phi[rr][3] = 0.0f;
            // the action at position `pos` of this lane's row, fetched one step ahead (the arrays stream from HBM)
            int id_n = 0, prm_n[MAX_P];
            auto fetch = [&](int pos) {
                if (row_lane && pos < len) {
                    id_n = __ldg(p.a.action_ids + (size_t)cand * p.a.T_max + pos);
                    const int32_t* pp = p.a.action_params + ((size_t)cand * p.a.T_max + pos) * P;
#pragma unroll
                    for (int j = 0; j < MAX_P; ++j)
                        if (j < P) prm_n[j] = __ldg(pp + j);
                }
            };
            // phase 1 (row-mapped): table row of every parameter slot of the fetched action: (id P + j) n_b + bucket(p_j);
            // -1 in slot 0 marks a row with no action at this position
            auto index_rows = [&](bool valid) {
                if (row_lane) {
                    int ix[MAX_P];
#pragma unroll
                    for (int j = 0; j < MAX_P; ++j) ix[j] = 0;
                    if (valid) {
                        int id = id_n;
                        if (id < 0 || id >= p.n_types) {
                            atomicOr(p.a.fault, WM_FAULT_TYPE);
                            id = id < 0 ? 0 : p.n_types - 1;
                        }
#pragma unroll
                        for (int j = 0; j < MAX_P; ++j) {
                            if (j < P) {
                                int prm = prm_n[j];
                                if (prm < 1) {
                                    atomicOr(p.a.fault, WM_FAULT_PARAM);
                                    prm = 1;
                                }
                                // bucket(p) = min(n_b - 1, floor(4 log2 p)) = bit_length(p^4) - 1, exact in 64-bit
                                // integers for p < 2^16 (beyond that the bucket is saturated for n_b <= 64)
                                unsigned long long q4 = (unsigned long long)min(prm, 65535);
                                q4 = q4 * q4;
                                q4 = q4 * q4;
                                const int bk = min(63 - __clzll((long long)q4), NB - 1);
                                ix[j] = (id * P + j) * NB + bk;
                            }
                        }
                    } else {
                        ix[0] = -1;
                    }
                    *reinterpret_cast<int4*>(s_idx + row * MAX_P) = make_int4(ix[0], ix[1], ix[2], ix[3]);
                    *reinterpret_cast<int4*>(s_idx + row * MAX_P + 4) = make_int4(ix[4], ix[5], ix[6], ix[7]);
                }
                __syncwarp();
            };
            // phase 2 (column-mapped, lane = 4 embedding columns): the warp's 16 rows are gathered from the table (L2) and
            // summed in registers, two rows' loads in flight at a time; phi accumulates, pk takes the fp16 operand
            auto gather = [&](uint2 (&pk)[16]) {
#pragma unroll
                for (int g = 0; g < 8; ++g) {
                    uint2 v[2][MAX_P];
                    bool on[2];
#pragma unroll
                    for (int q = 0; q < 2; ++q) {
                        const int r = 16 * aw + 2 * g + q;
                        const int4 i0 = *reinterpret_cast<const int4*>(s_idx + r * MAX_P);
                        const int4 i1 = *reinterpret_cast<const int4*>(s_idx + r * MAX_P + 4);
                        on[q] = i0.x >= 0;
                        const int ix[8] = {i0.x, i0.y, i0.z, i0.w, i1.x, i1.y, i1.z, i1.w};
#pragma unroll
                        for (int j = 0; j < MAX_P; ++j)
                            if (j < P && on[q]) v[q][j] = __ldg(reinterpret_cast<const uint2*>(p.Tbl + (size_t)ix[j] * DA + col4));
                    }
#pragma unroll
                    for (int q = 0; q < 2; ++q) {
                        float a4[4] = {0.0f, 0.0f, 0.0f, 0.0f};
                        if (on[q]) {
#pragma unroll
                            for (int j = 0; j < MAX_P; ++j) {
                                if (j < P) {
                                    a4[0] += __uint_as_float(v[q][j].x << 16);
                                    a4[1] += __uint_as_float(v[q][j].x & 0xffff0000u);
                                    a4[2] += __uint_as_float(v[q][j].y << 16);
                                    a4[3] += __uint_as_float(v[q][j].y & 0xffff0000u);
                                }
                            }
#pragma unroll
                            for (int c = 0; c < 4; ++c) phi[2 * g + q][c] += a4[c];
                        }
                        pk[2 * g + q] = make_uint2(pack_f16(a4[0], a4[1]), pack_f16(a4[2], a4[3]));
                    }
                }
            };
            // prefix-latent reuse: positions [0, st) only feed phi; scanned in position order BEFORE the first rollout step
            // (the running sums then see the positions in the literal call's order: bit-identical phi)
            const int st = (EXT && row_lane) ? row_start(p.a, cand, len) : 0;
            if (EXT && p.a.start) {
                int st_max = st;
#pragma unroll
                for (int o = 8; o > 0; o >>= 1) st_max = max(st_max, __shfl_xor_sync(0xffffffffu, st_max, o));
                st_max = __shfl_sync(0xffffffffu, st_max, 0);
                for (int pos = 0; pos < st_max; ++pos) {
                    uint2 pk[16];
                    fetch(pos);
                    index_rows(pos < st);
                    gather(pk);
                    __syncwarp();   // phase 2 reads of s_idx are done before the next phase 1 overwrites
                }
            }
            fetch(st);

            for (int t = 0; t < nsteps; ++t) {
                index_rows(st + t < len);
                fetch(st + t + 1);
                // all 16 rows are gathered BEFORE the a-buffer is free: only the stores stand between its release and the
                // next step's a K-blocks
                uint2 pk[16];
                gather(pk);
                if (n_w > 0) mbar_wait_inline(bar(B_AFREE), (n_w - 1) & 1);
                ++n_w;
#pragma unroll
                for (int rr = 0; rr < 16; ++rr) *a_dst(16 * aw + rr) = pk[rr];
                fence_proxy_async();
                __syncwarp();   // also: phase 2 reads of s_idx are done before the next phase 1 overwrites
                if (lane == 0) mbar_arrive_remote(r_aready);
            }
            if (!rank_it) continue;

            // ---- phi = mean_t a_t (0 when len = 0)
            if (row_lane) s_lens[row] = len;
            __syncwarp();
            if (n_w > 0) mbar_wait_inline(bar(B_AFREE), (n_w - 1) & 1);
            ++n_w;
#pragma unroll
            for (int rr = 0; rr < 16; ++rr) {
                const int lr_ = s_lens[16 * aw + rr];
                const float inv = lr_ > 0 ? 1.0f / (float)lr_ : 0.0f;
                *a_dst(16 * aw + rr) = make_uint2(pack_f16(phi[rr][0] * inv, phi[rr][1] * inv),
                                                  pack_f16(phi[rr][2] * inv, phi[rr][3] * inv));
            }
            // hardware features of this row -> the hw operand tile (columns >= H stay zero)
            if (row_lane) {
                for (int ch = 0; ch < p.H / 8; ++ch) {
                    uint4 o = make_uint4(0u, 0u, 0u, 0u);
                    if (cand >= 0) {
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

}  // namespace tcg

// ------------------------------------------------------------------------------------------------ host side
namespace {

uint16_t f32_to_bf16(float f) {
    uint32_t u;
    memcpy(&u, &f, 4);
    u += 0x7FFFu + ((u >> 16) & 1u);   // round to nearest even (the stored values are already bf16-exact)
    return (uint16_t)(u >> 16);
}

// One [192 x 64] weight tile W[n0 + n][k0 + k] (k < kvalid, else 0); W == nullptr is padding.
struct Box {
    const std::vector<float>* W;
    int ld, n0, k0, kvalid;
};

// Append one ring stage = two tiles.  Image of a stage: the leader CTA's 24 KB (weight rows 0-95 of tile A, then of tile
// B), then its peer's (rows 96-191 of A, of B); every 12 KB half tile in the SW128 K-major shared-memory image, fp16.
// Returns false when a weight is not finite in fp16 (|w| > 65504): the model then stays on the fp32 kernel.
bool append_stage(std::vector<uint16_t>& blob, const Box& A, const Box& B) {
    const size_t base = blob.size();
    blob.resize(base + 2 * tcg::STG_BYTES / 2, 0);
    bool ok = true;
    const Box* bx[2] = {&A, &B};
    for (int i = 0; i < 2; ++i) {
        if (!bx[i]->W) continue;
        const std::vector<float>& W = *bx[i]->W;
        for (int n = 0; n < tcg::NT; ++n)
            for (int k = 0; k < 64; ++k) {
                const float v = k < bx[i]->kvalid ? W[(size_t)(bx[i]->n0 + n) * bx[i]->ld + bx[i]->k0 + k] : 0.0f;
                const int nn = n % tcg::XC;
                const size_t off = (size_t)(n / tcg::XC) * tcg::STG_BYTES + (size_t)i * tcg::BT_BYTES + (size_t)nn * 128 +
                                   (size_t)((((k >> 3) ^ (nn & 7)) << 4)) + (size_t)(k & 7) * 2;
                uint16_t hb;
                ok &= f32_to_f16_bits(v, &hb);
                blob[base + off / 2] = hb;
            }
    }
    return ok;
}

}  // namespace

bool tcg_model_ok(const Model& m) {
    return m.kind == WM_KIND_GRU && m.phi_kind == WM_PHI_MEAN && m.dtype == WM_DTYPE_BF16 && m.embed == WM_EMBED_BUCKET && m.d == tcg::D &&
           m.d_a == tcg::DA && m.n_lin == 3 && m.sdim[1] == tcg::SW && m.sdim[2] == tcg::SW && m.H >= 8 &&
           m.H <= tcg::MAX_H && m.H % 8 == 0 && m.P >= 1 && m.P <= tcg::MAX_P && m.n_buckets >= 1 &&
           m.n_buckets <= tcg::MAX_BUCKETS;
}

int tcg_prepare(wm_ctx* ctx, const std::vector<std::vector<float>>& hv, const std::vector<std::string>& names) {
    Model& m = ctx->m;
    if (!tcg_model_ok(m)) return WM_OK;
    const tcg::SmemLayout L = tcg::smem_layout((m.H + 15) / 16);
    if ((int)L.total > ctx->smem_optin) return WM_OK;
    auto get = [&](const char* n) -> const std::vector<float>& {
        for (size_t i = 0; i < names.size(); ++i)
            if (names[i] == n) return hv[i];
        static const std::vector<float> empty;
        return empty;
    };
    const std::vector<float>&Wg = get("W_g"), &Wr = get("W_r"), &Wh = get("W_h"), &Ws0 = get("Ws0"), &Ws1 = get("Ws1");
    const std::vector<float>& Tbl = get("Tbl");
    const int K1 = tcg::D + tcg::DA, K0 = K1 + m.H;
    const size_t n_stages = (size_t)tcg::ROLL_STAGES + tcg::SC_STAGES;
    std::vector<uint16_t> blob;
    bool ok = true;   // every weight finite in fp16
    blob.reserve(n_stages * tcg::STG_BYTES);
    // K-block k of the rollout operand [z ; a]: 0-5 = z (or r*z), 6, 7 = a
    auto rb = [&](const std::vector<float>& W, int j, int k) { return Box{&W, K1, j * tcg::NT, k * 64, 64}; };
    auto st = [&](const Box& A, const Box& B) { ok &= append_stage(blob, A, B); };
    // the MMA warp's order (wm_tcg_kernel): R_0 interleaves a between z'_0 and z'_1; R_1, G_0 take z first; H_0, H_1,
    // G_1 take a first
    st(rb(Wr, 0, 0), rb(Wr, 0, 1)); st(rb(Wr, 0, 2), rb(Wr, 0, 6)); st(rb(Wr, 0, 7), rb(Wr, 0, 3)); st(rb(Wr, 0, 4), rb(Wr, 0, 5));
    auto roll_tile = [&](const std::vector<float>& W, int j, bool a_first) {
        if (a_first) st(rb(W, j, 6), rb(W, j, 7));
        for (int k = 0; k < tcg::Z_KB; k += 2) st(rb(W, j, k), rb(W, j, k + 1));
        if (!a_first) st(rb(W, j, 6), rb(W, j, 7));
    };
    roll_tile(Wr, 1, false); roll_tile(Wg, 0, false);
    roll_tile(Wh, 0, true); roll_tile(Wh, 1, true); roll_tile(Wg, 1, true);
    const Box pad{nullptr, 0, 0, 0, 0};
    for (int n = 0; n < 4; ++n) {     // scorer layer 1: phi pair, hw (zero-padded to 64 columns) + padding, three z pairs
        auto sb = [&](int k0, int kvalid) { return Box{&Ws0, K0, n * tcg::NT, k0, kvalid}; };
        st(sb(tcg::D, 64), sb(tcg::D + 64, 64));
        st(sb(K1, m.H), pad);
        for (int k = 0; k < tcg::Z_KB; k += 2) st(sb(k * 64, 64), sb((k + 1) * 64, 64));
    }
    for (int round = 0; round < 2; ++round)   // scorer layer 2: two rounds of two N tiles over all 12 K-blocks
        for (int kb = 0; kb < 12; ++kb)
            st(Box{&Ws1, tcg::SW, (2 * round) * tcg::NT, kb * 64, 64}, Box{&Ws1, tcg::SW, (2 * round + 1) * tcg::NT, kb * 64, 64});
    if (blob.size() * 2 != n_stages * 2 * tcg::STG_BYTES) {
        set_error("tcg_prepare: internal weight-image size mismatch");
        return WM_ERR_FORMAT;
    }
    if (!ok) return WM_OK;   // a weight beyond the fp16 range: this model stays on the fp32 kernel

    void* d_blob = nullptr;
    WM_CUDA_TRY(cudaMalloc(&d_blob, blob.size() * 2));
    ctx->allocs.push_back(d_blob);
    WM_CUDA_TRY(cudaMemcpy(d_blob, blob.data(), blob.size() * 2, cudaMemcpyHostToDevice));
    std::vector<uint16_t> t16(Tbl.size());
    for (size_t i = 0; i < Tbl.size(); ++i) t16[i] = f32_to_bf16(Tbl[i]);
    void* d_t = nullptr;
    WM_CUDA_TRY(cudaMalloc(&d_t, t16.size() * 2 + 16));
    ctx->allocs.push_back(d_t);
    WM_CUDA_TRY(cudaMemcpy(d_t, t16.data(), t16.size() * 2, cudaMemcpyHostToDevice));

    // tensor map over the image seen as rows of 64 fp16 (128 B); one box = 192 rows = one CTA's 24 KB of a stage.  The
    // image is already swizzled, so the map itself uses no swizzle.
    static_assert(sizeof(CUtensorMap) <= sizeof(m.tc2_tmap), "tensor map storage");
    CUtensorMap tm;
    {
        const int rc = encode_tmap_2d(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, d_blob, 64, blob.size() * 2 / 128, 128, 64, (uint32_t)(2 * tcg::XC), false, "tcg_prepare");
        if (rc != WM_OK) return rc;
    }
    memcpy(m.tc2_tmap, &tm, sizeof(tm));
    m.tc_blob = d_blob;
    m.tc_blob_bytes = blob.size() * 2;
    m.tc_E = d_t;
    WM_CUDA_TRY(cudaFuncSetAttribute(tcg::wm_tcg_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.total));
    WM_CUDA_TRY(cudaFuncSetAttribute(tcg::wm_tcg_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.total));
    m.tc_ok = 3;
    return WM_OK;
}

int launch_tcg(wm_ctx* ctx, Workspace* ws, const CallArgs& a, cudaStream_t st) {
    (void)ws;
    const Model& m = ctx->m;
    tcg::Params p;
    p.n_types = m.n_types; p.P = m.P; p.n_buckets = m.n_buckets; p.H = m.H;
    p.hw_ksteps = (m.H + 15) / 16;
    p.Tbl = static_cast<const __nv_bfloat16*>(m.tc_E);
    p.bs0 = m.bs[0]; p.bs1 = m.bs[1]; p.w3 = m.Wst[2]; p.bs2 = m.bs[2];
    p.a = a;
    p.n_tiles = (int)((a.B + tcg::TMP - 1) / tcg::TMP);
    p.prof = trace::begin(st);
    CUtensorMap tm;
    memcpy(&tm, m.tc2_tmap, sizeof(tm));
    const tcg::SmemLayout L = tcg::smem_layout(p.hw_ksteps);
    const int max_pairs = ctx->n_sms / 2;
    const int pairs = p.n_tiles < max_pairs ? p.n_tiles : max_pairs;
    if (a.start || a.init_index || a.latents_out) tcg::wm_tcg_kernel<true><<<2 * pairs, tcg::THREADS, L.total, st>>>(p, tm);
    else tcg::wm_tcg_kernel<false><<<2 * pairs, tcg::THREADS, L.total, st>>>(p, tm);
    WM_CUDA_TRY(cudaGetLastError());
    ctx->launches.fetch_add(1);
    trace::dump(p.prof, st);
    return WM_OK;
}

}  // namespace wm

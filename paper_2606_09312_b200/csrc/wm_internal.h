// Internal declarations shared by the library's translation units (not part of the ABI).
#pragma once

#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>
#include <stdint.h>

#include <atomic>
#include <mutex>
#include <string>
#include <vector>

#include "wm.h"

namespace wm {

constexpr int kMaxScorerLinears = 7;

// ---------------------------------------------------------------------------------------------------------
// Model description + device weights in every layout a kernel wants.
struct Model {
    int kind = 0, dtype = 0, embed = 0;
    int d = 0, d_a = 0, hidden = 0, n_types = 0, P = 0, n_buckets = 0, H = 0;
    int n_lin = 0;                       // linears of G
    int sdim[kMaxScorerLinears + 1] = {};  // sdim[0] = d+phi_dim+H, ..., sdim[n_lin] = 1
    float ln_eps = 1e-5f;
    int ranker_kind = 0, n_trees = 0, tree_depth = 0;   // WM_RANKER_*; forest geometry
    int2* Tnode = nullptr;               // forest: [n_trees][2^depth - 1] {feature index, threshold bits}: one 8-byte
                                         //         load per level of a walk
    float* Tv = nullptr;                 //         [n_trees][2^depth] leaf value
    float Tb = 0.0f;                     //         base score
    float* zeros = nullptr;              // 1024 zero floats (dummy scorer vectors of the tcgen05 kernel for forest models)
    int phi_kind = 0;                    // WM_PHI_*
    int phi_dim = 0;                     // d_a (mean embedding) or n_types + 1 + 3P (structured), <= d_a

    // fp32 CUDA-core path: matrices stored TRANSPOSED ([in][out]) so that consecutive threads (one output unit
    // each) read consecutive addresses; vectors as in the file.
    float* E = nullptr;        // [n_types][d_a]
    float* WpT = nullptr;      // [P][d_a]
    float* bp = nullptr;       // [d_a]
    float* Tbl = nullptr;      // [n_types*P*n_buckets][d_a]
    float* W1t = nullptr;      // [d+d_a][hidden]
    float* b1 = nullptr;
    float* W2t = nullptr;      // [hidden][d]
    float* b2 = nullptr;
    float* gamma = nullptr;
    float* beta = nullptr;
    float* Wwt = nullptr;      // [d_a][d]  TransH: hyperplane normal W_w, translation W_d (transposed)
    float* Wdt = nullptr;
    float* Wgt = nullptr;      // [d+d_a][d]
    float* Wrt = nullptr;
    float* Wht = nullptr;
    float* Wst[kMaxScorerLinears] = {};   // [in_i][out_i]
    float* bs[kMaxScorerLinears] = {};

    // tcgen05 path (bf16 MLP_LN models): weight images pre-tiled into the shared-memory layout the MMA
    // descriptors expect, see wm_tc.cu.  nullptr when the path does not apply.
    void* tc_blob = nullptr;
    size_t tc_blob_bytes = 0;
    void* tc_E = nullptr;      // bf16 [n_types][d_a]
    int tc_ok = 0;             // 0 = no tcgen05 path, 1 = wm_tc_kernel (one CTA per tile), 2 = wm_tc2_kernel (CTA pair), 3 = wm_tcg_kernel (CTA pair, GRU), 4 = TransH model on wm_tcp_kernel (no single-CTA form)
    alignas(64) unsigned char tc2_tmap[128] = {};   // CUtensorMap over tc_blob (pair kernel)
    int tc1_ok = 0;            // the single-CTA form wm_tc_kernel is built (tc_ok == 1 means: at least one of the two forms is)
    int tcp_akb = 1, tcp_pkb = 1;   // wm_tcp_kernel: K-blocks of the folded action features / phi features
    int tcp_ok = 0;            // 1 = wm_tcp_kernel (the CTA-pair, M = 256 form of wm_tc_kernel) is built for this model too
    alignas(64) unsigned char tcp_tmap[128] = {};   // CUtensorMap over wm_tcp_kernel's own weight image
    int tsc_ok = 0;            // 1 = wm_tsc_kernel (tcgen05 ranking MLP over a precomputed input row: WM_PHI_TYPED models)
    int tsc_nkb = 0;           // K-blocks of its input row [z_T | phi | 1 | h]
    void* tsc_blob = nullptr;  // its weight image
    alignas(64) unsigned char tsc_tmap[128] = {};   // CUtensorMap over tsc_blob
};

// NVTX range around an ABI call (header-only NVTX 3: a no-op unless a profiler injects itself)
namespace nvtx {
struct Range {
    explicit Range(const char* name) { nvtxRangePushA(name); }
    ~Range() { nvtxRangePop(); }
    Range(const Range&) = delete;
    Range& operator=(const Range&) = delete;
};
}  // namespace nvtx

// Per-stream slice of the workspace (perm, histogram/cursors, tile counter).
struct Workspace {
    std::mutex mu;                 // held while one call enqueues its kernels on this slice (wm_api.cu run_rollout)
    cudaStream_t stream = nullptr;
    int32_t* perm = nullptr;
    int64_t perm_cap = 0;
    int32_t* counters = nullptr;   // [kCounterInts] hist[WM_MAX_T+1], cursor[WM_MAX_T+1], tile counter, ...
    // staging for wm_score_topk_host
    void* stage = nullptr;
    size_t stage_cap = 0;
    // terminal latents [B, d] handed from K2 to the forest kernel (WM_RANKER_FOREST)
    float* zt = nullptr;
    size_t zt_cap = 0;
    // fp16 input rows of the tcgen05 ranking MLP (wm_tsc.cu; WM_PHI_TYPED models)
    void* xbuf = nullptr;
    size_t xbuf_cap = 0;
    // WM_OPT_TIMING
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    bool timed = false;
};

constexpr int kHistOff = 0;
constexpr int kCursorOff = WM_MAX_T + 1;
constexpr int kTileCtrOff = 2 * (WM_MAX_T + 1);
constexpr int kCounterInts = 2 * (WM_MAX_T + 1) + 8;

}  // namespace wm

struct wm_ctx {
    wm::Model m;
    int device = 0;
    int n_sms = 148;
    int smem_optin = 0;
    int opt_path = 0;     // WM_OPT_PATH
    int opt_sort = 1;     // WM_OPT_SORT
    int opt_timing = 0;   // WM_OPT_TIMING
    int opt_pair = 1;     // WM_OPT_PAIR
    uint32_t* fault = nullptr;   // device fault word
    std::mutex mu;
    std::vector<wm::Workspace*> pool;
    std::vector<void*> allocs;   // every device allocation owned by the ctx (weights)
    std::atomic<int64_t> launches{0};
    std::string path_reason;     // wm_path_reason(): why the model is on the fp32 kernel ("" on a tcgen05 kernel)
    // wm_score_topk_host pipelines a call by chunks of whole subgraphs: a copy stream, two compute streams, events and
    // a pinned staging buffer for the per-chunk (rebased) offsets; created on first use
    std::mutex host_mu;
    cudaStream_t hs_copy = nullptr, hs_k[2] = {nullptr, nullptr};
    cudaEvent_t hev_start = nullptr, hev_done[2] = {nullptr, nullptr}, hev_copy[8] = {};
    int32_t* h_off = nullptr;
    size_t h_off_cap = 0;
};

namespace wm {

void set_error(const char* fmt, ...);
#define WM_CUDA_TRY(expr)                                                                       \
    do {                                                                                        \
        cudaError_t e__ = (expr);                                                               \
        if (e__ != cudaSuccess) {                                                               \
            ::wm::set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
            return WM_ERR_CUDA;                                                                 \
        }                                                                                       \
    } while (0)

// Arguments of one wm_rollout_score call, after validation.
struct CallArgs {
    const float* init_states;
    const int32_t* action_ids;
    const int32_t* action_params;
    const int32_t* lengths;
    const float* hw_feats;
    float* scores_out;
    const int32_t* offsets;   // may be null (per-candidate mode)
    const int32_t* perm;      // may be null (identity)
    int64_t B;
    int S, T_max;
    uint32_t* fault;
    // prefix-latent reuse (NEXT row f3; wm_rollout_latents / wm_rollout_score_from), all null for wm_rollout_score:
    const int32_t* start;       // [B] steps [0, start) only feed phi, the rollout runs over [start, len)
    const int32_t* init_index;  // [B] row of init_states that holds candidate b's initial latent
    int64_t n_init;             // rows of init_states when init_index is used (indices are clamped to it)
    float* latents_out;         // [B, T_max, d] z after step t+1 at [b][t] for start <= t < len; scores_out may be null
    bool latents_terminal;      // latents_out is [B, d]: only the latent after the LAST step (t = len - 1) is stored
    const float* cand_latents;  // [B, d] (fp32 kernel only): a candidate with len > 0 starts from its own row of this array
                                // instead of its init_states row (the second pass of a WM_PHI_TYPED model, wm_api.cu)
};

// Quarter-octave bucket floor(4 log2 p) of a parameter p >= 1, exact for every int32 p (S10): with
// e = floor(log2 p) and q = p << (31 - e) in [2^31, 2^32), q^2 is exact in 64 bits and p^4 >= 2^(4e + j)  <=>
// (q^2)^2 >= 2^(124 + j)  <=>  hi64((q^2)^2) >= 2^(60 + j).  The caller clamps to n_buckets - 1.
__host__ __device__ inline int quarter_octave_bucket(int p) {
    const unsigned up = (unsigned)p;
#ifdef __CUDA_ARCH__
    const int e = 31 - __clz((int)up);
    const unsigned long long q = (unsigned long long)(up << (31 - e));
    const unsigned long long q2 = q * q;
    const unsigned long long hi = __umul64hi(q2, q2);
#else
    int e = 31;
    while (!((up >> e) & 1u)) --e;
    const unsigned long long q = (unsigned long long)(up << (31 - e));
    const unsigned long long q2 = q * q;
    const unsigned long long hi = (unsigned long long)(((unsigned __int128)q2 * q2) >> 64);
#endif
    return 4 * e + (hi >= (1ull << 61)) + (hi >= (1ull << 62)) + (hi >= (1ull << 63));
}

// rollout steps of a candidate: its clamped length minus its clamped start (the single place that defines it)
__host__ __device__ inline int clamp_start(int start, int len) { return start < 0 ? 0 : (start > len ? len : start); }

// K1 (wm_bucket.cu): perm = candidates sorted by clamped length, descending.  2 launches + 1 memset.
int launch_length_bucketing(wm_ctx* ctx, Workspace* ws, const int32_t* lengths, const int32_t* start, int64_t B,
                            int T_max, cudaStream_t st);

// K2-fp32 (wm_generic.cu): every model kind, fp32 CUDA cores.
int launch_generic(wm_ctx* ctx, const CallArgs& a, cudaStream_t st);
int generic_supported(const wm_ctx* ctx);

// K2 tcgen05 (wm_tc.cu): bf16 MLP_LN models with d = 256.
int tc_prepare(wm_ctx* ctx, const std::vector<std::vector<float>>& host_tensors_by_name_order,
               const std::vector<std::string>& names);
int tc_supported(const wm_ctx* ctx);
int launch_tc(wm_ctx* ctx, Workspace* ws, const CallArgs& a, cudaStream_t st);

// K2 tcgen05, CTA pair (wm_tc2.cu): bf16 MLP_LN models with d = 512.  Reached through tc_prepare / launch_tc.
int tc2_prepare(wm_ctx* ctx, const std::vector<std::vector<float>>& host_tensors_by_name_order,
                const std::vector<std::string>& names);
int launch_tc2(wm_ctx* ctx, Workspace* ws, const CallArgs& a, cudaStream_t st);

// K2 tcgen05, CTA pair with M = 256 (wm_tcp.cu): the pair form of wm_tc_kernel, same models.  Prepared after tc_prepare
// succeeds; launch_tc dispatches to it unless WM_OPT_PAIR = 0.
int tcp_prepare(wm_ctx* ctx, const std::vector<std::vector<float>>& host_tensors_by_name_order,
                const std::vector<std::string>& names);
int launch_tcp(wm_ctx* ctx, Workspace* ws, const CallArgs& a, cudaStream_t st);

// K2 tcgen05, CTA pair, gated (wm_tcg.cu): bf16 GRU models with d = 384 and the bucket table.  Same entry route.
int tcg_prepare(wm_ctx* ctx, const std::vector<std::vector<float>>& host_tensors_by_name_order,
                const std::vector<std::string>& names);
int launch_tcg(wm_ctx* ctx, Workspace* ws, const CallArgs& a, cudaStream_t st);

// K4 (wm_forest.cu): tree-ensemble ranker over [z_T ; structured phi ; h] (NEXT row f4)
int launch_forest(wm_ctx* ctx, const float* zT, const CallArgs& a, float* scores_out, cudaStream_t st);

// wm_tsc.cu: the ranking MLP on tcgen05 for WM_PHI_TYPED models the pair kernel can roll (d = 256, scorer 512 / 512).
// tsc_prepare builds the weight image at load time (m.tsc_ok); launch_tsc turns the terminal latents zT [B, d] and the
// action arrays into the fp16 input rows X (caller-provided, tsc_x_bytes(B) bytes) and ranks them: two launches.
int tsc_prepare(wm_ctx* ctx, const std::vector<std::vector<float>>& host_tensors_by_name_order,
                const std::vector<std::string>& names);
size_t tsc_x_bytes(const wm_ctx* ctx, int64_t B);
int launch_tsc(wm_ctx* ctx, const float* zT, void* X, const CallArgs& a, float* scores_out, cudaStream_t st);

// K3 (wm_topk.cu)
int64_t topk_launches();
int launch_topk(const float* scores, const int32_t* offsets, int S, int k, int32_t* idx_out, cudaStream_t st);

}  // namespace wm

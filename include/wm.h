/* wm.h — C ABI of the batched candidate evaluator (B200 / sm_100a).
 *
 * What the library computes (arxiv/paper_2606_09312, citations are PAPER.md:<line>):
 *
 *   z_0 = init_states[s]                       the task's initial latent program state
 *   z_t = F(z_{t-1}, a_t),  t = 1..len         action-conditioned transition, applied
 *                                              recurrently                               PAPER.md:68-71 Eq.1, :162 Eq.8, :166
 *   steps t > len leave z unchanged            rollout mask m_t                          PAPER.md:176 Eq.11
 *   phi = mean_t a_t (0 when len = 0)          action features
 *         or (WM_PHI_STRUCT) the paper's structured statistics: per-type action counts, sequence length and, per
 *         parameter slot, the sum / mean / max over the steps of log2 p   (S25)
 *   y   = G([z_T ; phi ; h])                   ranking score                             PAPER.md:122 Eq.3, :188 Eq.12
 *   top-k per subgraph, (score desc, idx asc)  candidates prioritised for measurement
 *
 * F, G and the action embedding take the parametrisations BASELINE.json's configs bind:
 *   embedding  a = E[id] + W_p log2(p) + b_p            (EMBED_LINEAR)
 *              a = sum_j Tbl[(id*P + j)*n_b + bucket(p_j)], bucket(p)=min(n_b-1, floor(4 log2 p)) (EMBED_BUCKET)
 *   F (MLP)    z' = z + W2 gelu(W1 [z;a] + b1) + b2     (KIND_MLP; KIND_MLP_LN adds LayerNorm(z'), eps in header)
 *   F (GRU)    g = s(W_g[z;a]); r = s(W_r[z;a]); z' = (1-g) z + g tanh(W_h [r*z ; a])   (KIND_GRU)
 *   G          MLP, hidden linears followed by exact (erf) GELU, last linear plain.
 *
 * Conventions
 *   - Every array argument of wm_rollout_score / wm_topk is a DEVICE pointer owned by the caller (any
 *     allocator; the tests use torch).  The library never frees or retains them.  wm_score_topk_host takes
 *     HOST pointers (pinned or pageable) and does the copies itself.
 *   - Calls enqueue work on `cuda_stream` (a cudaStream_t cast to void*; NULL = the legacy default stream) and
 *     return without synchronising, except wm_load_weights, wm_check, wm_free and wm_score_topk_host.
 *   - Return value: WM_OK (0) or a negative WM_ERR_* code; wm_last_error() then returns a thread-local,
 *     NUL-terminated message.  No exceptions, no aborts.
 *   - Data-dependent faults (len outside [0,T_max]; type id outside [0,n_types) or a parameter < 1 at a valid
 *     position t < len) cannot be seen by the host without a sync: kernels clamp the value so every access
 *     stays in bounds and OR a bit into a device flag word that wm_check() reads.  Padding positions
 *     (t >= len) may hold anything and are never read.
 *   - One ctx may be used from several streams concurrently: each call takes a private slice of the
 *     workspace (a small pool keyed by stream).
 */
#ifndef WM_H_
#define WM_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define WM_OK               0
#define WM_ERR_ARG         -1   /* null pointer, negative size, k <= 0, k > WM_MAX_K, T_max > WM_MAX_T        */
#define WM_ERR_IO          -2   /* weight file cannot be opened / read                                        */
#define WM_ERR_FORMAT      -3   /* bad magic, version, header field or file size                              */
#define WM_ERR_CUDA        -4   /* a CUDA runtime call failed (message carries cudaGetErrorString)            */
#define WM_ERR_UNSUPPORTED -5   /* header describes a model no kernel in this build handles                   */

#define WM_MAX_T   256          /* largest T_max accepted                                                     */
#define WM_MAX_K   1024         /* largest k accepted by wm_topk                                              */

/* bits of the device fault word returned by wm_check() */
#define WM_FAULT_LEN    1u      /* a length was outside [0, T_max] (clamped)                                  */
#define WM_FAULT_TYPE   2u      /* an action type id at a valid position was outside [0, n_types) (clamped)   */
#define WM_FAULT_PARAM  4u      /* an action parameter at a valid position was < 1 (treated as 1)             */
#define WM_FAULT_INDEX  8u      /* wm_rollout_score_from: a bank_index was outside [0, n_bank) (clamped)      */
#define WM_FAULT_RANGE  16u     /* tcgen05 kernels: an initial latent (init_states / bank row) had |value| > 65504, */
                                /* the largest fp16 MMA operand; it was clamped (the fp32 kernel has no such limit) */

/* values of wm_info.kind / dtype / embed (the weight-file header fields) */
#define WM_KIND_MLP     0
#define WM_KIND_MLP_LN  1
#define WM_KIND_GRU     2
#define WM_KIND_TRANSH  3      /* the paper's TransH-style transition (S24): project z onto the */
                               /* action's hyperplane, translate, residual MLP with the action embedding, L2-normalise  */
#define WM_DTYPE_FP32   0
#define WM_DTYPE_BF16   1
#define WM_EMBED_LINEAR 0
#define WM_EMBED_BUCKET 1
#define WM_PHI_MEAN     0      /* phi = mean over the valid steps of the action embedding (BASELINE.json cfg 1)       */
#define WM_PHI_STRUCT   1      /* phi = [c_0..c_{n_types-1} | len | s_0..s_{P-1} | m_0..m_{P-1} | x_0..x_{P-1}]:      */
                               /* c_k = number of steps of type k, s_j / m_j / x_j = sum / mean / max over the valid   */
                               /* steps of log2 p_tj, all 0 for an empty sequence (S25).       */
                               /* n_types + 1 + 3P values; this build needs n_types + 1 + 3P <= d_a                    */
#define WM_PHI_TYPED    2      /* phi = [c_k (n_types) | len | per type k: s_kj (P) | m_kj (P) | x_kj (P)]: the numeric  */
                               /* statistics kept PER ACTION TYPE, over the steps of that type, 0 for a type that does   */
                               /* not occur ("action-specific numeric attributes"; S28).         */
                               /* n_types (1 + 3P) + 1 values, no relation to d_a.  wm_rollout_score of a model the pair   */
                               /* kernel can roll (d = 256, scorer 512 / 512) is rollout + input rows + a tcgen05 ranking   */
                               /* MLP (three launches); other shapes run on the fp32 kernel                                */

/* wm_set_option keys */
#define WM_RANKER_MLP    0     /* G = the configs' MLP                                                              */
#define WM_RANKER_FOREST 1     /* G = an ensemble of complete binary regression trees over [z_T ; phi ; h] (*/
                               /* the paper's G is an XGBoost model; S27): heap order, at node i go to child    */
                               /* 2i+1 when x[f_i] < t_i (fp32 comparison), else 2i+2; score = base + sum of leaf values. */
                               /* Needs WM_PHI_STRUCT and P <= 8 in this build                                           */

#define WM_OPT_PATH      1      /* 0 = auto (default), 1 = force the fp32 CUDA-core kernel, 2 = force tcgen05  */
#define WM_OPT_SORT      2      /* 1 = bucket candidates by length before tiling (default), 0 = input order    */
#define WM_OPT_TIMING    3      /* 1 = record CUDA events around the rollout+score kernel (K2) of every call,   */
                                /*     read back with wm_last_kernel_ms; 0 = off (default)                      */

#define WM_OPT_PAIR      4      /* d = 256 MLP+LayerNorm models: 1 = the CTA-pair form wm_tcp_kernel (256-candidate tiles,  */
                                /*     tcgen05.mma.cta_group::2, default), 0 = wm_tc_kernel (one CTA per 128-candidate tile) */

typedef struct wm_ctx wm_ctx;   /* opaque: device weights (all layouts the kernels need) + workspace pool      */

typedef struct wm_info {        /* model hyper-parameters, as read from the weight-file header                 */
    int32_t kind, dtype, embed;
    int32_t d, d_a, hidden, n_types, P, n_buckets, H;
    int32_t n_scorer_layers;    /* number of linears of G                                                      */
    int32_t scorer_widths[6];   /* hidden widths of G (n_scorer_layers-1 used)                                 */
    float   ln_eps;
    int32_t path;               /* kernel the auto policy picks for this model: 1 = fp32 CUDA-core, 2 = tcgen05 */
    int32_t tc_variant;         /* tcgen05 kernel built for this model: 0 = none, 1 = wm_tc_kernel (one CTA per  */
                                /* 128-candidate tile, d = 256), 2 = wm_tc2_kernel (CTA pair per tile, d = 512),  */
                                /* 3 = wm_tcg_kernel (CTA pair per tile, GRU transition, d = 384),             */
                                /* 5 = wm_tcp_kernel (CTA pair per 256-candidate tile, d = 256: MLP+LayerNorm   */
                                /* and TransH steps; the default form of variant 1, WM_OPT_PAIR)               */
    int32_t phi_kind;           /* WM_PHI_*: which action features G reads                                     */
    int32_t ranker_kind;        /* WM_RANKER_*                                                                 */
    int32_t n_trees, tree_depth;   /* WM_RANKER_FOREST only                                                    */
} wm_info;

/* Read a WMW1 weight file (format below), convert to the kernels' layouts and copy to `device`.
 *   path     host path, NUL-terminated.
 *   device   CUDA device ordinal.
 *   ctx_out  receives the context (caller frees with wm_free).
 * File format (little-endian): "WMW1", then uint32 version, kind, dtype, embed, d, d_a, hidden, n_types, P,
 * n_buckets, H, n_scorer_layers, uint32 scorer_widths[6], float ln_eps (80 bytes in all); version 2 files carry one
 * more uint32, phi_kind (version 1 means WM_PHI_MEAN); version 3 files three more, ranker_kind, n_trees, tree_depth (and
 * n_scorer_layers = 0 for a forest); then fp32 tensors, row-major, in this order:
 *   EMBED_LINEAR: E[n_types,d_a], W_p[d_a,P], b_p[d_a]        EMBED_BUCKET: Tbl[n_types*P*n_buckets, d_a]
 *   MLP / MLP_LN: W1[hidden,d+d_a], b1[hidden], W2[d,hidden], b2[d] (, gamma[d], beta[d])
 *   GRU:          W_g[d,d+d_a], W_r[d,d+d_a], W_h[d,d+d_a]
 *   TRANSH:       W_w[d,d_a], W_d[d,d_a], then W1, b1, W2, b2 as for MLP
 *   G:            for each linear i: Ws_i[out_i,in_i], bs_i[out_i];  in_0 = d+dim(phi)+H, out_last = 1
 *   G (forest):   Tf[n_trees, 2^depth-1] feature indices (stored as fp32), Tt[n_trees, 2^depth-1] thresholds,
 *                 Tv[n_trees, 2^depth] leaf values, Tb[1] base score
 * With dtype = bf16 every stored value is already bf16-representable (BASELINE.json cfg 2-5: "bf16 weights with
 * fp32 accumulate"); the tcgen05 kernels encode them as fp16 operands — exact for 2^-14 <= |w| <= 65504 (smaller magnitudes
 * land on the fp16 subnormal grid, absolute change <= 3e-8; a larger one sends the model to the fp32 kernel) — with
 * activations rounded to fp16, accumulate
 * in fp32 and keep the latent in fp32 (S14).
 * Errors: WM_ERR_ARG, WM_ERR_IO, WM_ERR_FORMAT, WM_ERR_UNSUPPORTED, WM_ERR_CUDA.  Synchronous. */
int wm_load_weights(const char* path, int device, wm_ctx** ctx_out);

/* Free a context (device weights, workspace).  Synchronises the device.  NULL is a no-op. */
void wm_free(wm_ctx* ctx);

/* Copy the model description out of a context. */
int wm_get_info(const wm_ctx* ctx, wm_info* info_out);

/* Why this model runs where it runs.  "" when a tcgen05 kernel takes it (wm_info.path = 2); otherwise one sentence that
 * names the first property that keeps it on the fp32 CUDA-core kernel (wm_info.path = 1, typically 50-80 x slower on the
 * bf16 configurations of BASELINE.json: a latent width no tcgen05 kernel is built for, a scorer of another shape, a weight
 * beyond the fp16 range, ...), so that a caller one notch off a supported shape is told instead of silently slowed down.
 * The string is owned by the context.  NULL ctx: "". */
const char* wm_path_reason(const wm_ctx* ctx);

/* Set a WM_OPT_* option; returns WM_ERR_ARG for an unknown key or value, WM_ERR_UNSUPPORTED when the forced
 * path cannot run this model. */
int wm_set_option(wm_ctx* ctx, int32_t key, int32_t value);

/* Roll every candidate's action sequence through F from its subgraph's initial latent, then score it with G
 * (Eq.1/8/12).  Steps a0-a6 of DESIGN.md §1.
 *   init_states       [S, d]  fp32 row-major, one z_0 per subgraph        ([B, d] when subgraph_offsets == NULL)
 *   action_ids        [B, T_max] int32, entries at t >= lengths[b] ignored
 *   action_params     [B, T_max, P] int32, >= 1 at valid positions
 *   lengths           [B] int32, 0 <= len <= T_max
 *   hw_feats          [S, H]  fp32, one h per subgraph                    ([B, H] when subgraph_offsets == NULL)
 *   scores_out        [B] fp32, written in the original candidate order
 *   subgraph_offsets  [S+1] int32 CSR, offsets[0] = 0, offsets[S] = B, non-decreasing (empty segments allowed);
 *                     NULL selects per-candidate mode and S is ignored
 *   B, S, T_max       sizes; B = 0 is a no-op.  P, d, H come from the weight file.
 *   cuda_stream       stream to enqueue on
 * WM_RANKER_FOREST models: the rollout stores the terminal latents in a ctx-owned [B, d] buffer and a second kernel
 * ranks [z_T ; phi ; h] with the tree ensemble (two launches instead of one; same arguments, same output).
 * Errors: WM_ERR_ARG (null pointer with B > 0, B < 0, S < 0, T_max < 0 or > WM_MAX_T), WM_ERR_CUDA. */
int wm_rollout_score(wm_ctx* ctx,
                     const float* init_states, const int32_t* action_ids, const int32_t* action_params,
                     const int32_t* lengths, const float* hw_feats, float* scores_out,
                     const int32_t* subgraph_offsets, int64_t B, int32_t S, int32_t T_max, void* cuda_stream);

/* wm_rollout_score for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc).  Same arguments, same scores_out (PAPER.md:215 / :162 Eq.8 / :188 Eq.12, as above).  The
 * call's scratch — the length-sorted permutation of K1 (a0), its histogram / cursor counters and the tile counter of
 * the single-CTA tcgen05 kernel — lives in ONE file-scope device array of the library, sized for WM_STATIC_MAX_B
 * candidates (1 MB + 2 KB; every GPU that loads the library holds it until the process exits) instead of the
 * per-stream workspace wm_rollout_score grows with cudaMalloc.  The entry calls no cudaMalloc / cudaFree / event or
 * stream creation (the first launch of a kernel in a process may still load its module: call once before capturing).
 * Every call on a device shares the array, in every context and on every stream: the counters are cleared at the
 * start of each call (on the stream), the permutation is rewritten; two calls whose kernels can OVERLAP on the GPU
 * (different streams without an event between them) race on it — serialise them on one stream.  Host threads are
 * serialised by the library while they enqueue.
 * Errors: those of wm_rollout_score; WM_ERR_ARG when B > WM_STATIC_MAX_B (the message names the limit);
 * WM_ERR_UNSUPPORTED for WM_RANKER_FOREST models (they need a [B, d] latent buffer) and while WM_OPT_TIMING is on
 * (it creates events).  A WM_PHI_TYPED model runs this entry on the fp32 kernel (wm_rollout_score's split of such a call
 * needs two buffers of the batch's size). */
#define WM_STATIC_MAX_B 262144
int wm_rollout_score_static(wm_ctx* ctx,
                            const float* init_states, const int32_t* action_ids, const int32_t* action_params,
                            const int32_t* lengths, const float* hw_feats, float* scores_out,
                            const int32_t* subgraph_offsets, int64_t B, int32_t S, int32_t T_max, void* cuda_stream);

/* Prefix-latent reuse (SURVEY.md §8(b) extension and NEXT row f3; the online loop of PAPER.md:215 scores, round after
 * round, candidates that share long action prefixes with survivors of earlier rounds).  Two calls:
 *
 * wm_rollout_latents rolls every candidate like wm_rollout_score but stores the latent after every step instead of
 * ranking:  latents_out[b][t][:] = z_{t+1} of candidate b for 0 <= t < lengths[b]  ([B, T_max, d] fp32, device; entries
 * with t >= lengths[b] are not written).  init_states / subgraph_offsets as in wm_rollout_score.
 *
 * wm_rollout_score_from scores candidates whose first start[b] steps were rolled before:
 *   bank              [n_bank, d] fp32: latents (rows of a latents_out array, or any other store)
 *   bank_index        [B] int32: the row of `bank` that holds candidate b's latent after its first start[b] steps
 *                     (the task's initial latent when start[b] = 0); a value outside [0, n_bank) is clamped and
 *                     raises WM_FAULT_INDEX in the fault word wm_check() reads
 *   start             [B] int32, clamped to [0, lengths[b]]: steps [0, start) are not rolled, they only feed phi
 *   action_ids, action_params, lengths, hw_feats, scores_out, subgraph_offsets (non-NULL), B, S, T_max: as in
 *                     wm_rollout_score, the action arrays holding each candidate's WHOLE sequence
 * The score equals wm_rollout_score's for the same candidate (to the rounding of the stored fp32 latent: the
 * tcgen05 kernels keep the latent in fp32 between steps, so a bank written by wm_rollout_latents reproduces them).
 * Candidates are bucketed by their remaining steps lengths[b] - start[b].
 * Errors: as wm_rollout_score; WM_ERR_ARG also for a null bank / bank_index / start / latents_out or n_bank < 1;
 * WM_ERR_UNSUPPORTED for wm_rollout_score_from on a WM_RANKER_FOREST model.  Every tcgen05 kernel takes both calls (its EXT
 * instance); a call whose latents_out is not 16-byte aligned runs on the fp32 kernel (WM_ERR_UNSUPPORTED when the tcgen05
 * path is forced with WM_OPT_PATH = 2). */
int wm_rollout_latents(wm_ctx* ctx,
                       const float* init_states, const int32_t* action_ids, const int32_t* action_params,
                       const int32_t* lengths, const int32_t* subgraph_offsets, float* latents_out,
                       int64_t B, int32_t S, int32_t T_max, void* cuda_stream);
int wm_rollout_score_from(wm_ctx* ctx,
                          const float* bank, const int32_t* bank_index, const int32_t* start,
                          const int32_t* action_ids, const int32_t* action_params, const int32_t* lengths,
                          const float* hw_feats, float* scores_out, const int32_t* subgraph_offsets,
                          int64_t B, int32_t S, int32_t T_max, int64_t n_bank, void* cuda_stream);

/* Per subgraph segment [offsets[s], offsets[s+1]) select the k largest scores, ordered by
 * (score descending, index ascending).  -0.0 == +0.0; NaN ranks below every number (ties by index).
 *   scores            [offsets[S]] fp32
 *   subgraph_offsets  [S+1] int32 CSR (device)
 *   idx_out           [S, k] int32: GLOBAL candidate indices; rows of segments with fewer than k candidates
 *                     are padded with -1
 * Needs no context.  Errors: WM_ERR_ARG (null pointer with S > 0, S < 0, k <= 0, k > WM_MAX_K), WM_ERR_CUDA. */
int wm_topk(const float* scores, const int32_t* subgraph_offsets, int32_t S, int32_t k, int32_t* idx_out,
            void* cuda_stream);

/* Synchronise `cuda_stream` and return the OR of the WM_FAULT_* bits raised since the last wm_check on this
 * ctx (>= 0), or a negative error code.  Resets the word. */
int wm_check(wm_ctx* ctx, void* cuda_stream);

/* End-to-end convenience entry: same computation as wm_rollout_score followed by wm_topk, with HOST buffers.
 * Copies the inputs host->device into ctx-owned staging, runs both steps on `cuda_stream`, copies scores
 * ([B] fp32, may be NULL to skip) and idx ([S,k] int32) back, and synchronises the stream before returning.
 * subgraph_offsets must be non-NULL (top-k needs segments) and, like every input here, a HOST array (it is read on
 * the host to plan the copies).  From 65,536 candidates on, the call is pipelined internally over chunks of whole
 * subgraphs (copies on a ctx-owned stream overlap the kernels of the previous chunk; everything is ordered after the
 * work already queued on `cuda_stream` and complete when the call returns); results are bit-identical to the
 * unpipelined sequence.  Concurrent calls on one ctx are serialised.  Used by bench.py's e2e leg. */
int wm_score_topk_host(wm_ctx* ctx,
                       const float* init_states, const int32_t* action_ids, const int32_t* action_params,
                       const int32_t* lengths, const float* hw_feats, const int32_t* subgraph_offsets,
                       int64_t B, int32_t S, int32_t T_max, int32_t k,
                       float* scores_out, int32_t* idx_out, void* cuda_stream);

/* The same call for callers that keep the action arrays compact — type ids as uint8 (n_types <= 256, else
 * WM_ERR_UNSUPPORTED), parameters as uint16 (values 1..65535; BASELINE.json's configs draw them from 1..1024) — which is
 * 13 instead of 28 bytes per action on the host-to-device link (the call is PCIe-bound at evolution-round sizes): the arrays
 * are copied as they are and widened to int32 on the device (one extra small kernel).  Padding positions may hold anything.
 * Same results, bit for bit, as wm_score_topk_host on the widened arrays; same errors. */
int wm_score_topk_host_compact(wm_ctx* ctx,
                               const float* init_states, const uint8_t* action_ids, const uint16_t* action_params,
                               const int32_t* lengths, const float* hw_feats, const int32_t* subgraph_offsets,
                               int64_t B, int32_t S, int32_t T_max, int32_t k,
                               float* scores_out, int32_t* idx_out, void* cuda_stream);

/* The same with the VALID steps only (candidates of one search round have very different lengths; at cfg 2 the
 * padded arrays are 37 % padding).  step_offsets [B + 1] int32 (host): candidate b's steps are rows
 * [step_offsets[b], step_offsets[b + 1]) of step_ids [N] uint8 and step_params [N, P] uint16, N = step_offsets[B],
 * step_offsets[0] = 0; its length is the difference (a length above T_max raises WM_FAULT_LEN and is clamped).  The packed
 * arrays are staged as they are and expanded on the device.  Results are bit-identical to wm_score_topk_host on the padded
 * form of the same candidates.  Errors: as wm_score_topk_host_compact; WM_ERR_ARG for inconsistent step_offsets. */
int wm_score_topk_host_ragged(wm_ctx* ctx,
                              const float* init_states, const uint8_t* step_ids, const uint16_t* step_params,
                              const int32_t* step_offsets, const float* hw_feats, const int32_t* subgraph_offsets,
                              int64_t B, int32_t S, int32_t T_max, int32_t k,
                              float* scores_out, int32_t* idx_out, void* cuda_stream);

/* With WM_OPT_TIMING = 1: synchronise `cuda_stream` and return, in *ms_out, the device time of the rollout+score
 * kernel (K2 alone: bucketing and top-k excluded) of the most recent wm_rollout_score call made on that stream.
 * bench.py's roofline leg uses it.  Errors: WM_ERR_ARG (null, timing off, or no call yet), WM_ERR_CUDA. */
int wm_last_kernel_ms(wm_ctx* ctx, void* cuda_stream, float* ms_out);

/* Number of kernels the library launched on behalf of this ctx since it was created (bench.py's
 * gpu_launches); wm_topk's launches are counted in a process-wide counter returned when ctx == NULL. */
int64_t wm_launch_count(const wm_ctx* ctx);

/* Launch one empty kernel (1 block, 32 threads, no work) on `cuda_stream`: the launch-latency yardstick of bench.py's
 * cfg 1 line (cfg 1 is 12 MFLOP and 10 KB, bound by launch latency; its time is reported as a ratio
 * to this).  Needs no context.  Errors: WM_ERR_CUDA. */
int wm_launch_empty(void* cuda_stream);

/* Message for the last nonzero status returned on this thread ("" if none). */
const char* wm_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* WM_H_ */

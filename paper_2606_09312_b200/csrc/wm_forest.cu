// K4: tree-ensemble ranker (NEXT row f4).  PAPER.md:190 — "G is implemented as an XGBoost ranking model" over
// [z_T ; phi(a_1:T) ; h] (Eq.12); reading S27 of DESIGN.md §3 fixes synthetic COMPLETE binary trees in heap order:
// at node i go to child 2i+1 when x[f_i] < t_i (fp32), else 2i+2; score = base + sum over trees of the leaf value.
//
// One warp per candidate.  The warp builds the candidate's feature vector in shared memory — the terminal latent K2
// left in HBM (the task's z_0 for an empty sequence), the structured phi (S25) straight from the action arrays (lanes
// stride over the steps; exact counts through shared-memory atomics, per-slot sum / max through fixed-order warp
// reductions, so the features and therefore every branch decision are deterministic), the subgraph's hardware
// features — then lane l walks trees l, l + 32, ... and a fixed-order warp reduction adds the leaves.
// Gather / latency-bound: per candidate d + H floats and len * (1 + P) int32 of input, n_trees * depth dependent
// 12-byte node reads that stay in L1/L2 (the forest is n_trees * (3 * 2^depth - 2) * 4 bytes: 97 KB for 128 x depth 6).
#include "wm_internal.h"

namespace wm {

namespace {

constexpr int kForestWarps = 8;
constexpr int kMaxP = 8;

struct ForestParams {
    const float* zT;            // [B, d] terminal latents (rows of candidates with len = 0 are not read)
    const float* init_states;   // [S, d] ([B, d] without offsets)
    const int32_t *ids, *params, *lengths, *offsets;
    const float* hw;
    float* scores;
    int64_t B;
    int S, T_max, d, n_types, P, H, n_in, n_trees, nodes, depth;
    const int2* Tnode;          // {feature index, threshold bits} per internal node
    const float* Tv;
    float Tb;
};

__device__ __forceinline__ int seg_of(const int32_t* __restrict__ off, int S, int cand) {
    int lo = 0, hi = S;   // largest s with off[s] <= cand
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (__ldg(off + mid) <= cand) lo = mid; else hi = mid;
    }
    return lo;
}

__global__ void __launch_bounds__(kForestWarps * 32) wm_forest_kernel(const ForestParams p) {
    extern __shared__ float s_x[];                       // [kForestWarps][n_in]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float* x = s_x + (size_t)warp * p.n_in;
    const int d = p.d, NT = p.n_types, P = p.P;
    float* phi = x + d;
    for (int64_t c = (int64_t)blockIdx.x * kForestWarps + warp; c < p.B; c += (int64_t)gridDim.x * kForestWarps) {
        int len = __ldg(p.lengths + c);
        len = len < 0 ? 0 : (len > p.T_max ? p.T_max : len);           // (K2 has reported the fault)
        const int seg = p.offsets ? seg_of(p.offsets, p.S, (int)c) : (int)c;
        // z_T, or the task's initial latent when no step was taken
        const float* z = len > 0 ? p.zT + (size_t)c * d : p.init_states + (size_t)seg * d;
        for (int j = lane; j < d; j += 32) x[j] = __ldg(z + j);
        for (int j = lane; j < NT; j += 32) phi[j] = 0.0f;
        for (int j = lane; j < p.H; j += 32) x[d + NT + 1 + 3 * P + j] = __ldg(p.hw + (size_t)seg * p.H + j);
        __syncwarp();
        // structured phi (S25): counts | len | per slot: sum, mean, max of log2 p
        float sum[kMaxP], mx[kMaxP];
#pragma unroll
        for (int j = 0; j < kMaxP; ++j) sum[j] = mx[j] = 0.0f;
        for (int t = lane; t < len; t += 32) {
            int id = __ldg(p.ids + (size_t)c * p.T_max + t);
            id = id < 0 ? 0 : (id >= NT ? NT - 1 : id);
            atomicAdd(phi + id, 1.0f);                                  // small integers: exact in any order
            const int32_t* pp = p.params + ((size_t)c * p.T_max + t) * P;
#pragma unroll
            for (int j = 0; j < kMaxP; ++j)
                if (j < P) {
                    const int prm = __ldg(pp + j);
                    // MUFU.LG2 (2 ulp): the features feed comparisons whose margins the parity test accounts for
                    const float l2 = __log2f((float)(prm < 1 ? 1 : prm));
                    sum[j] += l2;
                    mx[j] = fmaxf(mx[j], l2);
                }
        }
#pragma unroll
        for (int j = 0; j < kMaxP; ++j)
            if (j < P) {      // (warp-uniform)
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) sum[j] += __shfl_xor_sync(0xffffffffu, sum[j], o);
                // log2 p >= 0: the float order is the order of the bit patterns, one redux instruction
                mx[j] = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(mx[j])));
            }
        if (lane == 0) {
            const float inv = len > 0 ? 1.0f / (float)len : 0.0f;
            phi[NT] = (float)len;
#pragma unroll
            for (int j = 0; j < kMaxP; ++j)
                if (j < P) {
                    phi[NT + 1 + j] = sum[j];
                    phi[NT + 1 + P + j] = sum[j] * inv;
                    phi[NT + 1 + 2 * P + j] = mx[j];
                }
        }
        __syncwarp();
        // the trees
        // the trees: a walk is `depth` dependent (node load, feature read) pairs, so a lane walks four trees at once
        float acc = 0.0f;
        for (int t0 = lane; t0 < p.n_trees; t0 += 128) {
            int node[4] = {0, 0, 0, 0};
            for (int l = 0; l < p.depth; ++l) {
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int t = t0 + 32 * u < p.n_trees ? t0 + 32 * u : t0;      // (in-bounds dummy past the last tree)
                    const int2 nd = __ldg(p.Tnode + (size_t)t * p.nodes + node[u]);
                    node[u] = 2 * node[u] + (x[nd.x] < __int_as_float(nd.y) ? 1 : 2);
                }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (t0 + 32 * u < p.n_trees)
                    acc += __ldg(p.Tv + (size_t)(t0 + 32 * u) * (p.nodes + 1) + (node[u] - p.nodes));
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (lane == 0) p.scores[c] = p.Tb + acc;
        __syncwarp();   // x is rewritten for the warp's next candidate
    }
}

}  // namespace

int launch_forest(wm_ctx* ctx, const float* zT, const CallArgs& a, float* scores_out, cudaStream_t st) {
    const Model& m = ctx->m;
    ForestParams p;
    p.zT = zT; p.init_states = a.init_states; p.ids = a.action_ids; p.params = a.action_params; p.lengths = a.lengths;
    p.offsets = a.offsets; p.hw = a.hw_feats; p.scores = scores_out;
    p.B = a.B; p.S = a.S; p.T_max = a.T_max; p.d = m.d; p.n_types = m.n_types; p.P = m.P; p.H = m.H;
    p.n_in = m.sdim[0]; p.n_trees = m.n_trees; p.depth = m.tree_depth; p.nodes = (1 << m.tree_depth) - 1;
    p.Tnode = m.Tnode; p.Tv = m.Tv; p.Tb = m.Tb;
    const size_t smem = (size_t)kForestWarps * p.n_in * sizeof(float);
    if (smem > (size_t)ctx->smem_optin) {
        set_error("forest ranker: feature vector too wide for shared memory");
        return WM_ERR_UNSUPPORTED;
    }
    if (smem > 48 * 1024)
        WM_CUDA_TRY(cudaFuncSetAttribute(wm_forest_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int64_t blocks = (a.B + kForestWarps - 1) / kForestWarps;
    const int grid = (int)(blocks < (int64_t)ctx->n_sms * 16 ? blocks : (int64_t)ctx->n_sms * 16);
    wm_forest_kernel<<<grid, kForestWarps * 32, smem, st>>>(p);
    WM_CUDA_TRY(cudaGetLastError());
    ctx->launches.fetch_add(1);
    return WM_OK;
}

}  // namespace wm

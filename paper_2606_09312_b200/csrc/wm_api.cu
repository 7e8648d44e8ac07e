// The C ABI (include/wm.h): weight loading, context/workspace management, argument validation and dispatch.
// No arithmetic of the method lives here; see wm_bucket.cu (a0), wm_generic.cu / wm_tc.cu (a1-a6), wm_topk.cu (a7).
#include <cstdarg>
#include <cstdio>
#include <algorithm>
#include <cstring>
#include <new>

#include "wm_internal.h"

namespace wm {

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

namespace {

struct Header {
    uint32_t version, kind, dtype, embed, d, d_a, hidden, n_types, P, n_buckets, H, n_lin;
    uint32_t widths[6];
    float ln_eps;
};
static_assert(sizeof(Header) == 76, "WMW1 header is 4 + 76 bytes");

struct HostTensor {
    std::string name;
    uint64_t rows = 0, cols = 0;   // vectors: rows = n, cols = 1 (64-bit: header fields multiply past 2^32)
    std::vector<float> v;
};

int upload(wm_ctx* ctx, const std::vector<float>& h, float** out) {
    void* p = nullptr;
    WM_CUDA_TRY(cudaMalloc(&p, h.size() * sizeof(float) + 16));
    ctx->allocs.push_back(p);
    WM_CUDA_TRY(cudaMemcpy(p, h.data(), h.size() * sizeof(float), cudaMemcpyHostToDevice));
    *out = static_cast<float*>(p);
    return WM_OK;
}

std::vector<float> transposed(const HostTensor& t) {
    std::vector<float> o(t.v.size());
    for (uint64_t r = 0; r < t.rows; ++r)
        for (uint64_t c = 0; c < t.cols; ++c) o[(size_t)(c * t.rows + r)] = t.v[(size_t)(r * t.cols + c)];
    return o;
}

Workspace* acquire_ws(wm_ctx* ctx, cudaStream_t st) {
    std::lock_guard<std::mutex> lk(ctx->mu);
    for (Workspace* w : ctx->pool)
        if (w->stream == st) return w;
    Workspace* w = new Workspace();
    w->stream = st;
    if (cudaMalloc(&w->counters, sizeof(int32_t) * kCounterInts) != cudaSuccess) {
        delete w;
        return nullptr;
    }
    ctx->pool.push_back(w);
    return w;
}

int ensure_perm(Workspace* ws, int64_t B, cudaStream_t st) {
    if (ws->perm_cap >= B) return WM_OK;
    // growing frees the old buffer: work already queued on this stream may still read it
    if (ws->perm) {
        WM_CUDA_TRY(cudaStreamSynchronize(st));
        WM_CUDA_TRY(cudaFree(ws->perm));
        ws->perm = nullptr;
        ws->perm_cap = 0;
    }
    const int64_t cap = B + B / 4 + 1024;
    WM_CUDA_TRY(cudaMalloc(&ws->perm, sizeof(int32_t) * cap));
    ws->perm_cap = cap;
    return WM_OK;
}

int pick_path(const wm_ctx* ctx) {
    if (ctx->opt_path == 1) return 1;
    if (ctx->opt_path == 2) return 2;
    return tc_supported(ctx) ? 2 : 1;
}

}  // namespace
}  // namespace wm

using namespace wm;

__global__ void wm_empty_kernel() {}

#pragma GCC visibility push(default)
extern "C" {

const char* wm_last_error(void) { return g_err; }

static int load_weights_impl(const char* path, int device, wm_ctx** ctx_out) {
    if (!path || !ctx_out) {
        set_error("wm_load_weights: null argument");
        return WM_ERR_ARG;
    }
    *ctx_out = nullptr;
    FILE* f = fopen(path, "rb");
    if (!f) {
        set_error("wm_load_weights: cannot open '%s'", path);
        return WM_ERR_IO;
    }
    char magic[4];
    Header h;
    if (fread(magic, 1, 4, f) != 4 || fread(&h, sizeof(h), 1, f) != 1) {
        fclose(f);
        set_error("wm_load_weights: file shorter than the header");
        return WM_ERR_FORMAT;
    }
    if (memcmp(magic, "WMW1", 4) != 0 || h.version < 1 || h.version > 3) {
        fclose(f);
        set_error("wm_load_weights: bad magic or version");
        return WM_ERR_FORMAT;
    }
    uint32_t phi_kind = WM_PHI_MEAN;   // version 2 = the version-1 header followed by uint32 phi_kind
    if (h.version >= 2 && (fread(&phi_kind, 4, 1, f) != 1 || phi_kind > WM_PHI_TYPED)) {
        fclose(f);
        set_error("wm_load_weights: bad phi_kind");
        return WM_ERR_FORMAT;
    }
    uint32_t forest[3] = {WM_RANKER_MLP, 0, 0};   // version 3 = version 2 + uint32 ranker_kind, n_trees, tree_depth
    if (h.version == 3 && (fread(forest, 4, 3, f) != 3 || forest[0] > WM_RANKER_FOREST ||
                           (forest[0] == WM_RANKER_FOREST &&
                            (forest[1] < 1 || forest[1] > 65536 || forest[2] < 1 || forest[2] > 12 || h.n_lin != 0)))) {
        fclose(f);
        set_error("wm_load_weights: bad ranker fields (kind, n_trees 1..65536, tree_depth 1..12, n_scorer_layers 0)");
        return WM_ERR_FORMAT;
    }
    const bool is_forest = forest[0] == WM_RANKER_FOREST;
    if (is_forest && (phi_kind != WM_PHI_STRUCT || h.P > 8)) {
        fclose(f);
        set_error("wm_load_weights: the forest ranker needs the structured phi and P <= 8 in this build");
        return WM_ERR_UNSUPPORTED;
    }
    const bool mlp = h.kind == WM_KIND_MLP || h.kind == WM_KIND_MLP_LN || h.kind == WM_KIND_TRANSH;
    if (h.kind > 3 || h.dtype > 1 || h.embed > 1 || h.d == 0 || h.d_a == 0 || h.n_types == 0 || h.P == 0 ||
        h.d > 65536 || h.d_a > 65536 || h.hidden > 65536 || h.P > 64 || h.H > 65536 || h.n_types > (1u << 20) ||
        h.n_lin > 7 || (mlp && h.hidden == 0) || (h.embed == WM_EMBED_BUCKET && h.n_buckets == 0) ||
        h.n_buckets > 4096 || !(h.ln_eps >= 0.0f)) {
        fclose(f);
        set_error("wm_load_weights: header field out of range");
        return WM_ERR_FORMAT;
    }
    for (uint32_t i = 0; i + 1 < h.n_lin; ++i)
        if (h.widths[i] == 0 || h.widths[i] > 65536) {
            fclose(f);
            set_error("wm_load_weights: scorer width out of range");
            return WM_ERR_FORMAT;
        }

    // tensor list in file order
    std::vector<HostTensor> ts;
    uint64_t payload_floats = 0;   // sum of all tensor sizes, in 64-bit: checked against the file size before any allocation
    auto add = [&](const char* name, uint64_t rows, uint64_t cols) {
        HostTensor t;
        t.name = name;
        t.rows = rows;
        t.cols = cols;
        payload_floats += rows * cols;   // every factor <= 2^20 and at most three of them: no 64-bit overflow
        ts.push_back(t);
    };
    const int d = h.d, da = h.d_a, hid = h.hidden;
    // width of phi: the mean action embedding, or counts | len | per-slot sum, mean, max of log2 params (S25)
    const uint64_t phi_dim64 = phi_kind == WM_PHI_MEAN ? (uint64_t)da
                               : phi_kind == WM_PHI_STRUCT ? (uint64_t)h.n_types + 1 + 3 * (uint64_t)h.P
                                                           : (uint64_t)h.n_types * (1 + 3 * (uint64_t)h.P) + 1;
    if (phi_dim64 > (1u << 20)) {
        fclose(f);
        set_error("wm_load_weights: header field out of range (phi width)");
        return WM_ERR_FORMAT;
    }
    const int phi_dim = (int)phi_dim64;
    if (phi_kind == WM_PHI_STRUCT && phi_dim > da) {   // the kernels keep the pooled phi in the rows / K-blocks of the action embedding
        fclose(f);
        set_error("wm_load_weights: structured phi needs n_types + 1 + 3 P <= d_a in this build");
        return WM_ERR_UNSUPPORTED;
    }
    if (h.embed == WM_EMBED_LINEAR) {
        add("E", h.n_types, da); add("W_p", da, h.P); add("b_p", da, 1);
    } else {
        add("Tbl", (uint64_t)h.n_types * h.P * h.n_buckets, da);
    }
    if (h.kind == WM_KIND_TRANSH) { add("W_w", d, da); add("W_d", d, da); }
    if (mlp) {
        add("W1", hid, d + da); add("b1", hid, 1); add("W2", d, hid); add("b2", d, 1);
        if (h.kind == WM_KIND_MLP_LN) { add("gamma", d, 1); add("beta", d, 1); }
    } else {
        add("W_g", d, d + da); add("W_r", d, d + da); add("W_h", d, d + da);
    }
    int sdim[kMaxScorerLinears + 1] = {};
    sdim[0] = d + phi_dim + h.H;
    for (uint32_t i = 0; i + 1 < h.n_lin; ++i) sdim[i + 1] = h.widths[i];
    if (h.n_lin >= 1) sdim[h.n_lin] = 1;   // (a forest model has no linears: sdim[0] stays the feature count)
    for (uint32_t i = 0; i < h.n_lin; ++i) {
        char nm[16];
        snprintf(nm, sizeof(nm), "Ws%u", i); add(nm, sdim[i + 1], sdim[i]);
        snprintf(nm, sizeof(nm), "bs%u", i); add(nm, sdim[i + 1], 1);
    }
    if (is_forest) {
        const int nodes = (1 << forest[2]) - 1;
        add("Tf", forest[1], nodes); add("Tt", forest[1], nodes); add("Tv", forest[1], nodes + 1); add("Tb", 1, 1);
    } else if (h.n_lin < 1) {
        fclose(f);
        set_error("wm_load_weights: header field out of range");
        return WM_ERR_FORMAT;
    }
    {   // the file must hold exactly the tensors the header announces: nothing is allocated for a header that lies
        const long pos = ftell(f);
        if (pos < 0 || fseek(f, 0, SEEK_END) != 0) {
            fclose(f);
            set_error("wm_load_weights: cannot seek in '%s'", path);
            return WM_ERR_IO;
        }
        const long end = ftell(f);
        if (end < 0 || fseek(f, pos, SEEK_SET) != 0) {
            fclose(f);
            set_error("wm_load_weights: cannot seek in '%s'", path);
            return WM_ERR_IO;
        }
        const uint64_t have = (uint64_t)(end - pos);
        if (have != payload_floats * 4) {
            fclose(f);
            set_error(have < payload_floats * 4 ? "wm_load_weights: file truncated (%llu tensor bytes, header needs %llu)"
                                                : "wm_load_weights: trailing bytes after the last tensor (%llu tensor bytes, header needs %llu)",
                      (unsigned long long)have, (unsigned long long)(payload_floats * 4));
            return WM_ERR_FORMAT;
        }
    }
    for (HostTensor& t : ts) {
        t.v.resize((size_t)(t.rows * t.cols));
        if (fread(t.v.data(), sizeof(float), t.v.size(), f) != t.v.size()) {
            fclose(f);
            set_error("wm_load_weights: file truncated in tensor %s", t.name.c_str());
            return WM_ERR_FORMAT;
        }
    }
    char extra;
    const bool trailing = fread(&extra, 1, 1, f) == 1;
    fclose(f);
    if (trailing) {
        set_error("wm_load_weights: trailing bytes after the last tensor");
        return WM_ERR_FORMAT;
    }

    WM_CUDA_TRY(cudaSetDevice(device));
    wm_ctx* ctx = new wm_ctx();
    ctx->device = device;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) {
        delete ctx;
        set_error("wm_load_weights: cudaGetDeviceProperties failed");
        return WM_ERR_CUDA;
    }
    ctx->n_sms = prop.multiProcessorCount;
    ctx->smem_optin = (int)prop.sharedMemPerBlockOptin;
    Model& m = ctx->m;
    m.kind = h.kind; m.dtype = h.dtype; m.embed = h.embed; m.d = d; m.d_a = da; m.hidden = hid;
    m.n_types = h.n_types; m.P = h.P; m.n_buckets = h.n_buckets; m.H = h.H; m.n_lin = h.n_lin;
    for (int i = 0; i <= kMaxScorerLinears; ++i) m.sdim[i] = sdim[i];
    m.ln_eps = h.ln_eps;
    m.phi_kind = (int)phi_kind;
    m.phi_dim = phi_dim;
    m.ranker_kind = (int)forest[0]; m.n_trees = (int)forest[1]; m.tree_depth = (int)forest[2];

    int rc = WM_OK;
    auto find = [&](const std::string& n) -> const HostTensor* {
        for (const HostTensor& t : ts)
            if (t.name == n) return &t;
        return nullptr;
    };
    auto up = [&](const char* n, float** dst, bool transpose) {
        const HostTensor* t = find(n);
        if (!t || rc != WM_OK) return;
        rc = transpose ? upload(ctx, transposed(*t), dst) : upload(ctx, t->v, dst);
    };
    up("E", &m.E, false); up("W_p", &m.WpT, true); up("b_p", &m.bp, false); up("Tbl", &m.Tbl, false);
    up("W1", &m.W1t, true); up("b1", &m.b1, false); up("W2", &m.W2t, true); up("b2", &m.b2, false);
    up("gamma", &m.gamma, false); up("beta", &m.beta, false);
    up("W_w", &m.Wwt, true); up("W_d", &m.Wdt, true);
    up("W_g", &m.Wgt, true); up("W_r", &m.Wrt, true); up("W_h", &m.Wht, true);
    for (int i = 0; i < m.n_lin; ++i) {
        char nm[16];
        snprintf(nm, sizeof(nm), "Ws%d", i); up(nm, &m.Wst[i], true);
        snprintf(nm, sizeof(nm), "bs%d", i); up(nm, &m.bs[i], false);
    }
    if (rc == WM_OK && is_forest) {
        // forest tensors: feature indices as int32 (validated against the feature count), thresholds, leaves, base
        const HostTensor *tf = find("Tf"), *tt = find("Tt");
        std::vector<int2> nodes(tf->v.size());
        for (size_t i = 0; i < nodes.size(); ++i) {
            const float v = tf->v[i];
            if (!(v >= 0.0f) || v >= (float)sdim[0] || v != (float)(int)v) {
                set_error("wm_load_weights: forest feature index out of range");
                rc = WM_ERR_FORMAT;
                break;
            }
            nodes[i].x = (int)v;
            memcpy(&nodes[i].y, &tt->v[i], 4);
        }
        void* p = nullptr;
        if (rc == WM_OK) {
            if (cudaMalloc(&p, nodes.size() * sizeof(int2) + 16) != cudaSuccess ||
                cudaMemcpy(p, nodes.data(), nodes.size() * sizeof(int2), cudaMemcpyHostToDevice) != cudaSuccess) {
                set_error("wm_load_weights: cannot upload the forest");
                rc = WM_ERR_CUDA;
            } else {
                ctx->allocs.push_back(p);
                m.Tnode = static_cast<int2*>(p);
            }
        }
        up("Tv", &m.Tv, false);
        m.Tb = find("Tb")->v[0];
        if (rc == WM_OK) rc = upload(ctx, std::vector<float>(1024, 0.0f), &m.zeros);
    }
    if (rc == WM_OK) {
        void* p = nullptr;
        if (cudaMalloc(&p, 16) != cudaSuccess || cudaMemset(p, 0, 16) != cudaSuccess) {
            set_error("wm_load_weights: cannot allocate the fault word");
            rc = WM_ERR_CUDA;
        } else {
            ctx->allocs.push_back(p);
            ctx->fault = static_cast<uint32_t*>(p);
        }
    }
    if (rc == WM_OK) {
        std::vector<std::vector<float>> hv;
        std::vector<std::string> names;
        for (HostTensor& t : ts) {
            names.push_back(t.name);
            hv.push_back(std::move(t.v));
        }
        rc = tc_prepare(ctx, hv, names);
    }
    if (rc == WM_OK && !tc_supported(ctx)) {
        // wm_path_reason: the first property that keeps the model off the tcgen05 kernels
        const Model& m = ctx->m;
        char buf[400];
        const bool mlp_ln = m.kind == WM_KIND_MLP_LN, transh = m.kind == WM_KIND_TRANSH, gru = m.kind == WM_KIND_GRU;
        if (m.dtype != WM_DTYPE_BF16)
            snprintf(buf, sizeof buf, "fp32 weights: the tcgen05 kernels take bf16-valued weights (an fp32 model needs fp32 products for its 1e-4 tolerance)");
        else if (m.kind == WM_KIND_MLP)
            snprintf(buf, sizeof buf, "residual MLP without LayerNorm: the tcgen05 kernels are built for MLP+LayerNorm, TransH and GRU transitions");
        else if ((mlp_ln && m.d != 256 && m.d != 512) || (transh && m.d != 256) || (gru && m.d != 384))
            snprintf(buf, sizeof buf, "latent width d = %d: the tcgen05 kernels are built for d = 256 (MLP+LayerNorm, TransH), 512 (MLP+LayerNorm) and 384 (GRU)", m.d);
        else if ((m.d == 256 && m.d_a != 128) || (m.d == 512 && m.d_a != 256) || (m.d == 384 && m.d_a != 128))
            snprintf(buf, sizeof buf, "action-embedding width d_a = %d: the d = %d tcgen05 kernel is built for d_a = %d", m.d_a, m.d, m.d == 512 ? 256 : 128);
        else if ((gru && m.embed != WM_EMBED_BUCKET) || (!gru && m.embed != WM_EMBED_LINEAR))
            snprintf(buf, sizeof buf, "action embedding kind %d: the GRU kernel takes the bucketed table, the others the linear embedding", m.embed);
        else if (m.ranker_kind == WM_RANKER_MLP && m.phi_kind != WM_PHI_TYPED &&
                 (m.n_lin != 3 || m.sdim[1] != m.sdim[2] || m.sdim[1] != (m.d == 256 ? 512 : m.d == 512 ? 1024 : 768)))
            snprintf(buf, sizeof buf, "scorer shape: the d = %d tcgen05 kernel is built for two hidden layers of %d units", m.d, m.d == 256 ? 512 : m.d == 512 ? 1024 : 768);
        else if (m.H < 8 || m.H > 64 || m.H % 8 != 0)
            snprintf(buf, sizeof buf, "hardware-feature width H = %d: the tcgen05 kernels take 8 <= H <= 64, a multiple of 8", m.H);
        else if (!gru && (m.hidden % (m.d == 512 ? 256 : 128) != 0 || m.hidden < (m.d == 512 ? 512 : 256) || m.hidden > 1024))
            snprintf(buf, sizeof buf, "hidden width %d: the d = %d tcgen05 kernel takes a multiple of %d up to 1024", m.hidden, m.d, m.d == 512 ? 256 : 128);
        else if (m.phi_kind != WM_PHI_MEAN && (gru || (m.phi_kind == WM_PHI_TYPED && m.d != 256)))
            snprintf(buf, sizeof buf, "phi kind %d with this transition: structured phi runs on the d = 256 / 512 kernels, per-type phi on the d = 256 one", m.phi_kind);
        else
            snprintf(buf, sizeof buf, "outside the tcgen05 kernels' limits (action types, parameter slots, buckets, shared memory) or a weight beyond the fp16 range (|w| > 65504)");
        ctx->path_reason = buf;
    }
    if (rc == WM_OK && !generic_supported(ctx) && !tc_supported(ctx)) {
        set_error("wm_load_weights: no kernel in this build handles this model (too wide for shared memory)");
        rc = WM_ERR_UNSUPPORTED;
    }
    if (rc != WM_OK) {
        wm_free(ctx);
        return rc;
    }
    *ctx_out = ctx;
    return WM_OK;
}

void wm_free(wm_ctx* ctx) {
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    cudaDeviceSynchronize();
    for (Workspace* w : ctx->pool) {
        if (w->perm) cudaFree(w->perm);
        if (w->counters) cudaFree(w->counters);
        if (w->stage) cudaFree(w->stage);
        if (w->zt) cudaFree(w->zt);
        if (w->xbuf) cudaFree(w->xbuf);
        if (w->ev0) cudaEventDestroy(w->ev0);
        if (w->ev1) cudaEventDestroy(w->ev1);
        delete w;
    }
    for (void* p : ctx->allocs) cudaFree(p);
    if (ctx->hs_copy) cudaStreamDestroy(ctx->hs_copy);
    for (int i = 0; i < 2; ++i) {
        if (ctx->hs_k[i]) cudaStreamDestroy(ctx->hs_k[i]);
        if (ctx->hev_done[i]) cudaEventDestroy(ctx->hev_done[i]);
    }
    if (ctx->hev_start) cudaEventDestroy(ctx->hev_start);
    for (int i = 0; i < 8; ++i)
        if (ctx->hev_copy[i]) cudaEventDestroy(ctx->hev_copy[i]);
    if (ctx->h_off) cudaFreeHost(ctx->h_off);
    delete ctx;
}

int wm_load_weights(const char* path, int device, wm_ctx** ctx_out) {
    // "No exceptions, no aborts" (include/wm.h): an allocation failure on the host is an error code, not a terminate
    try {
        nvtx::Range r("wm_load_weights");
        return load_weights_impl(path, device, ctx_out);
    } catch (const std::bad_alloc&) {
        if (ctx_out) *ctx_out = nullptr;
        set_error("wm_load_weights: out of host memory");
        return WM_ERR_IO;
    } catch (...) {
        if (ctx_out) *ctx_out = nullptr;
        set_error("wm_load_weights: unexpected host exception");
        return WM_ERR_IO;
    }
}

const char* wm_path_reason(const wm_ctx* ctx) { return ctx ? ctx->path_reason.c_str() : ""; }

int wm_get_info(const wm_ctx* ctx, wm_info* o) {
    if (!ctx || !o) {
        set_error("wm_get_info: null argument");
        return WM_ERR_ARG;
    }
    const Model& m = ctx->m;
    o->kind = m.kind; o->dtype = m.dtype; o->embed = m.embed; o->d = m.d; o->d_a = m.d_a; o->hidden = m.hidden;
    o->n_types = m.n_types; o->P = m.P; o->n_buckets = m.n_buckets; o->H = m.H; o->n_scorer_layers = m.n_lin;
    for (int i = 0; i < 6; ++i) o->scorer_widths[i] = (i + 1 < m.n_lin) ? m.sdim[i + 1] : 0;
    o->ln_eps = m.ln_eps;
    o->path = tc_supported(ctx) ? 2 : 1;
    o->tc_variant = (tc_supported(ctx) == 1 || tc_supported(ctx) == 4) && m.tcp_ok && (ctx->opt_pair || !m.tc1_ok) ? 5 : tc_supported(ctx);
    o->phi_kind = m.phi_kind;
    o->ranker_kind = m.ranker_kind; o->n_trees = m.n_trees; o->tree_depth = m.tree_depth;
    return WM_OK;
}

int wm_set_option(wm_ctx* ctx, int32_t key, int32_t value) {
    if (!ctx) {
        set_error("wm_set_option: null ctx");
        return WM_ERR_ARG;
    }
    if (key == WM_OPT_PATH) {
        if (value < 0 || value > 2) {
            set_error("wm_set_option: WM_OPT_PATH takes 0, 1 or 2");
            return WM_ERR_ARG;
        }
        if (value == 2 && !tc_supported(ctx)) {
            set_error("wm_set_option: the tcgen05 path does not handle this model");
            return WM_ERR_UNSUPPORTED;
        }
        if (value == 1 && !generic_supported(ctx)) {
            set_error("wm_set_option: the fp32 path does not handle this model");
            return WM_ERR_UNSUPPORTED;
        }
        ctx->opt_path = value;
        return WM_OK;
    }
    if (key == WM_OPT_SORT) {
        if (value < 0 || value > 1) {
            set_error("wm_set_option: WM_OPT_SORT takes 0 or 1");
            return WM_ERR_ARG;
        }
        ctx->opt_sort = value;
        return WM_OK;
    }
    if (key == WM_OPT_TIMING) {
        if (value < 0 || value > 1) {
            set_error("wm_set_option: WM_OPT_TIMING takes 0 or 1");
            return WM_ERR_ARG;
        }
        ctx->opt_timing = value;
        return WM_OK;
    }
    if (key == WM_OPT_PAIR) {
        if (value < 0 || value > 1) {
            set_error("wm_set_option: WM_OPT_PAIR takes 0 or 1");
            return WM_ERR_ARG;
        }
        if (value == 0 && ctx->m.tcp_ok && !ctx->m.tc1_ok) {
            set_error("wm_set_option: this model has no single-CTA tcgen05 form (its embedding table does not fit shared memory)");
            return WM_ERR_UNSUPPORTED;
        }
        ctx->opt_pair = value;
        return WM_OK;
    }
    set_error("wm_set_option: unknown key %d", key);
    return WM_ERR_ARG;
}

// Common tail of the three rollout entries: bucketing by rollout steps, timing events, dispatch.  The caller holds
// ws->mu: one call's enqueue sequence (memset, histogram, scatter, K2 [, K4]) shares the slice's perm / counters / zt, so
// two host threads that use the same stream must not interleave theirs (in stream order the sequences then run one
// after the other and the second reuses the buffers only after the first has finished with them).
static int run_rollout_locked(wm_ctx* ctx, Workspace* ws, CallArgs a, cudaStream_t st) {
    a.perm = nullptr;
    a.fault = ctx->fault;
    // (a batch that fits one tile of any kernel gains nothing from the sort and pays three launches for it)
    if (ctx->opt_sort && a.B > 256) {
        int rc = ensure_perm(ws, a.B, st);
        if (rc != WM_OK) return rc;
        rc = launch_length_bucketing(ctx, ws, a.lengths, a.start, a.B, a.T_max, st);
        if (rc != WM_OK) return rc;
        a.perm = ws->perm;
    }
    if (ctx->opt_timing) {
        if (!ws->ev0) {
            WM_CUDA_TRY(cudaEventCreate(&ws->ev0));
            WM_CUDA_TRY(cudaEventCreate(&ws->ev1));
        }
        WM_CUDA_TRY(cudaEventRecord(ws->ev0, st));
    }
    const int rc = pick_path(ctx) == 2 ? launch_tc(ctx, ws, a, st) : launch_generic(ctx, a, st);
    if (ctx->opt_timing && rc == WM_OK) {
        WM_CUDA_TRY(cudaEventRecord(ws->ev1, st));
        ws->timed = true;
    }
    return rc;
}

static int run_rollout(wm_ctx* ctx, const CallArgs& a, cudaStream_t st, const char* who) {
    WM_CUDA_TRY(cudaSetDevice(ctx->device));
    Workspace* ws = acquire_ws(ctx, st);
    if (!ws) {
        set_error("%s: cannot allocate workspace", who);
        return WM_ERR_CUDA;
    }
    std::lock_guard<std::mutex> lk(ws->mu);
    nvtx::Range r(who);
    return run_rollout_locked(ctx, ws, a, st);
}

static bool sizes_ok(const char* who, int64_t B, int32_t S, int32_t T_max) {
    if (B < 0 || B > 0x7fffffffLL || S < 0 || T_max < 0 || T_max > WM_MAX_T) {
        set_error("%s: size out of range (B=%lld S=%d T_max=%d)", who, (long long)B, S, T_max);
        return false;
    }
    return true;
}

// Per-type phi (S28) on a model the pair kernel can roll: 609 running statistics per row do not fit beside a 256-row tile,
// so the call is split.  K2 (tcgen05, EXT instance) rolls the candidates — from z_0, or from a bank row and a start
// position for wm_rollout_score_from — and stores the terminal latents [B, d]; then either the tcgen05 ranking MLP
// (wm_typed_x_kernel writes the fp16 rows [z_T | phi | 1 | h], wm_tsc_kernel ranks them) or, where that kernel is not
// built for the model, the fp32 kernel with the latents as per-candidate initial latents and start = len (it walks every
// position for phi only).  A prefix call takes the split only with the tcgen05 ranking MLP (the fp32 kernel runs such a
// call whole).
static bool typed_split_applies(const wm_ctx* ctx, const CallArgs& a, bool prefix_call) {
    return ctx->m.phi_kind == WM_PHI_TYPED && ctx->m.ranker_kind == WM_RANKER_MLP && pick_path(ctx) == 2 &&
           a.B <= 0x7fffffffLL / ctx->m.d && (uintptr_t)a.init_states % 16 == 0 && a.T_max > 0 && a.T_max <= 255 &&
           (!prefix_call || ctx->m.tsc_ok);
}

static int typed_split_score(wm_ctx* ctx, const CallArgs& a, cudaStream_t st, const char* who) {
    WM_CUDA_TRY(cudaSetDevice(ctx->device));
    Workspace* ws = acquire_ws(ctx, st);
    if (!ws) {
        set_error("%s: cannot allocate workspace", who);
        return WM_ERR_CUDA;
    }
    std::lock_guard<std::mutex> lk(ws->mu);
    nvtx::Range nr(who);
    const size_t need = (size_t)a.B * ctx->m.d;
    if (ws->zt_cap < need) {
        if (ws->zt) {
            WM_CUDA_TRY(cudaStreamSynchronize(st));
            WM_CUDA_TRY(cudaFree(ws->zt));
            ws->zt = nullptr;
            ws->zt_cap = 0;
        }
        WM_CUDA_TRY(cudaMalloc(&ws->zt, (need + need / 4 + 1024) * sizeof(float)));
        ws->zt_cap = need + need / 4 + 1024;
    }
    CallArgs r = a;
    r.scores_out = nullptr; r.latents_out = ws->zt; r.latents_terminal = true;
    int rc = run_rollout_locked(ctx, ws, r, st);
    if (rc != WM_OK) return rc;
    if (ctx->m.tsc_ok) {
        const size_t xneed = tsc_x_bytes(ctx, a.B);
        if (ws->xbuf_cap < xneed) {
            if (ws->xbuf) {
                WM_CUDA_TRY(cudaStreamSynchronize(st));
                WM_CUDA_TRY(cudaFree(ws->xbuf));
                ws->xbuf = nullptr;
                ws->xbuf_cap = 0;
            }
            WM_CUDA_TRY(cudaMalloc(&ws->xbuf, xneed + xneed / 4 + 4096));
            ws->xbuf_cap = xneed + xneed / 4 + 4096;
        }
        CallArgs xa = a;
        xa.fault = ctx->fault;
        rc = launch_tsc(ctx, ws->zt, ws->xbuf, xa, a.scores_out, st);
    } else {
        CallArgs sc = a;
        sc.fault = ctx->fault;
        sc.perm = (ctx->opt_sort && a.B > 256) ? ws->perm : nullptr;   // K1's order by length serves both passes
        sc.cand_latents = ws->zt;     // (rows of length 0 stored no latent: they keep init_states, their z_T = z_0)
        sc.start = a.lengths;
        rc = launch_generic(ctx, sc, st);
    }
    if (rc == WM_OK && ctx->opt_timing && ws->ev1) WM_CUDA_TRY(cudaEventRecord(ws->ev1, st));
    return rc;
}

int wm_rollout_score(wm_ctx* ctx, const float* init_states, const int32_t* action_ids, const int32_t* action_params,
                     const int32_t* lengths, const float* hw_feats, float* scores_out,
                     const int32_t* subgraph_offsets, int64_t B, int32_t S, int32_t T_max, void* cuda_stream) {
    if (!ctx) {
        set_error("wm_rollout_score: null ctx");
        return WM_ERR_ARG;
    }
    if (!sizes_ok("wm_rollout_score", B, S, T_max)) return WM_ERR_ARG;
    if (B == 0) return WM_OK;
    if (!init_states || !lengths || !scores_out || (ctx->m.H > 0 && !hw_feats) ||
        (T_max > 0 && (!action_ids || !action_params)) || (subgraph_offsets && S < 1)) {
        set_error("wm_rollout_score: null pointer (or S < 1 with offsets) for a non-empty batch");
        return WM_ERR_ARG;
    }
    CallArgs a = {};
    a.init_states = init_states; a.action_ids = action_ids; a.action_params = action_params; a.lengths = lengths;
    a.hw_feats = hw_feats; a.scores_out = scores_out; a.offsets = subgraph_offsets;
    a.B = B; a.S = S; a.T_max = T_max;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (ctx->m.ranker_kind == WM_RANKER_FOREST) {
        // tree-ensemble ranker: K2 rolls the candidates and hands the terminal latents [B, d] to K4, which builds
        // [z_T ; structured phi ; h] per candidate and walks the trees
        WM_CUDA_TRY(cudaSetDevice(ctx->device));
        Workspace* ws = acquire_ws(ctx, st);
        if (!ws) {
            set_error("wm_rollout_score: cannot allocate workspace");
            return WM_ERR_CUDA;
        }
        std::lock_guard<std::mutex> lk(ws->mu);
        nvtx::Range nr("wm_rollout_score");
        const size_t need = (size_t)B * ctx->m.d;
        if (ws->zt_cap < need) {
            if (ws->zt) {
                WM_CUDA_TRY(cudaStreamSynchronize(st));
                WM_CUDA_TRY(cudaFree(ws->zt));
                ws->zt = nullptr;
                ws->zt_cap = 0;
            }
            WM_CUDA_TRY(cudaMalloc(&ws->zt, (need + need / 4 + 1024) * sizeof(float)));
            ws->zt_cap = need + need / 4 + 1024;
        }
        CallArgs r = a;
        r.scores_out = nullptr; r.latents_out = ws->zt; r.latents_terminal = true;
        const int rc = run_rollout_locked(ctx, ws, r, st);
        return rc != WM_OK ? rc : launch_forest(ctx, ws->zt, a, scores_out, st);
    }
    if (typed_split_applies(ctx, a, false)) return typed_split_score(ctx, a, st, "wm_rollout_score");
    return run_rollout(ctx, a, st, "wm_rollout_score");
}

// ---- wm_rollout_score_static: the allocation-free entry (include/wm.h).  Its scratch is this file-scope device array:
// [kCounterInts] counters (histogram, cursors, tile counter) followed by the permutation of up to WM_STATIC_MAX_B
// candidates.  In host code the NAME of a __device__ array is a host-side stand-in, not a device address: the address the
// kernels get comes from cudaGetSymbolAddress, once per device, with that device current.
constexpr int kStaticPermOff = (kCounterInts + 63) / 64 * 64;   // keeps the permutation 256-byte aligned
static __device__ __align__(256) int32_t g_static_scratch[kStaticPermOff + WM_STATIC_MAX_B];
static std::mutex g_static_mu;                 // one call at a time enqueues on the shared scratch
static int32_t* g_static_ptr[64] = {};         // per device: the array's device address

int wm_rollout_score_static(wm_ctx* ctx, const float* init_states, const int32_t* action_ids,
                            const int32_t* action_params, const int32_t* lengths, const float* hw_feats,
                            float* scores_out, const int32_t* subgraph_offsets, int64_t B, int32_t S, int32_t T_max,
                            void* cuda_stream) {
    if (!ctx) {
        set_error("wm_rollout_score_static: null ctx");
        return WM_ERR_ARG;
    }
    if (!sizes_ok("wm_rollout_score_static", B, S, T_max)) return WM_ERR_ARG;
    if (B > WM_STATIC_MAX_B) {
        set_error("wm_rollout_score_static: B = %lld exceeds the static scratch (WM_STATIC_MAX_B = %d candidates); "
                  "use wm_rollout_score",
                  (long long)B, (int)WM_STATIC_MAX_B);
        return WM_ERR_ARG;
    }
    if (ctx->m.ranker_kind == WM_RANKER_FOREST || ctx->opt_timing) {
        set_error("wm_rollout_score_static: not available for WM_RANKER_FOREST models or with WM_OPT_TIMING on");
        return WM_ERR_UNSUPPORTED;
    }
    if (B == 0) return WM_OK;
    if (!init_states || !lengths || !scores_out || (ctx->m.H > 0 && !hw_feats) ||
        (T_max > 0 && (!action_ids || !action_params)) || (subgraph_offsets && S < 1)) {
        set_error("wm_rollout_score_static: null pointer (or S < 1 with offsets) for a non-empty batch");
        return WM_ERR_ARG;
    }
    if (ctx->device < 0 || ctx->device >= 64) {
        set_error("wm_rollout_score_static: device ordinal %d out of range", ctx->device);
        return WM_ERR_ARG;
    }
    WM_CUDA_TRY(cudaSetDevice(ctx->device));
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_ptr[ctx->device]) {
        int32_t* ptr = nullptr;
        WM_CUDA_TRY(cudaGetSymbolAddress((void**)&ptr, g_static_scratch));
        g_static_ptr[ctx->device] = ptr;
    }
    nvtx::Range nr("wm_rollout_score_static");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    Workspace ws;                    // a view of the static array: nothing in it is owned, grown or freed
    ws.stream = st;
    ws.counters = g_static_ptr[ctx->device];
    ws.perm = g_static_ptr[ctx->device] + kStaticPermOff;
    ws.perm_cap = WM_STATIC_MAX_B;
    CallArgs a = {};
    a.init_states = init_states; a.action_ids = action_ids; a.action_params = action_params; a.lengths = lengths;
    a.hw_feats = hw_feats; a.scores_out = scores_out; a.offsets = subgraph_offsets;
    a.B = B; a.S = S; a.T_max = T_max;
    a.fault = ctx->fault;
    // the steps of run_rollout_locked without its growing / event-creating branches: K1 clears the counters it starts
    // from (cudaMemsetAsync on the stream) and rewrites the permutation; the single-CTA kernel clears its tile counter
    if (ctx->opt_sort && B > 256) {
        const int rc = launch_length_bucketing(ctx, &ws, a.lengths, nullptr, a.B, a.T_max, st);
        if (rc != WM_OK) return rc;
        a.perm = ws.perm;
    }
    return pick_path(ctx) == 2 ? launch_tc(ctx, &ws, a, st) : launch_generic(ctx, a, st);
}

int wm_rollout_latents(wm_ctx* ctx, const float* init_states, const int32_t* action_ids, const int32_t* action_params,
                       const int32_t* lengths, const int32_t* subgraph_offsets, float* latents_out, int64_t B,
                       int32_t S, int32_t T_max, void* cuda_stream) {
    if (!ctx) {
        set_error("wm_rollout_latents: null ctx");
        return WM_ERR_ARG;
    }
    if (!sizes_ok("wm_rollout_latents", B, S, T_max)) return WM_ERR_ARG;
    if (B == 0 || T_max == 0) return WM_OK;
    if (!init_states || !lengths || !latents_out || !action_ids || !action_params || (subgraph_offsets && S < 1)) {
        set_error("wm_rollout_latents: null pointer (or S < 1 with offsets) for a non-empty batch");
        return WM_ERR_ARG;
    }
    CallArgs a = {};
    a.init_states = init_states; a.action_ids = action_ids; a.action_params = action_params; a.lengths = lengths;
    a.offsets = subgraph_offsets; a.latents_out = latents_out;
    a.B = B; a.S = S; a.T_max = T_max;
    return run_rollout(ctx, a, static_cast<cudaStream_t>(cuda_stream), "wm_rollout_latents");
}

int wm_rollout_score_from(wm_ctx* ctx, const float* bank, const int32_t* bank_index, const int32_t* start,
                          const int32_t* action_ids, const int32_t* action_params, const int32_t* lengths,
                          const float* hw_feats, float* scores_out, const int32_t* subgraph_offsets, int64_t B,
                          int32_t S, int32_t T_max, int64_t n_bank, void* cuda_stream) {
    if (!ctx) {
        set_error("wm_rollout_score_from: null ctx");
        return WM_ERR_ARG;
    }
    if (!sizes_ok("wm_rollout_score_from", B, S, T_max)) return WM_ERR_ARG;
    if (B == 0) return WM_OK;
    if (ctx->m.ranker_kind == WM_RANKER_FOREST) {
        set_error("wm_rollout_score_from: not built for the forest ranker");
        return WM_ERR_UNSUPPORTED;
    }
    if (!bank || !bank_index || !start || n_bank < 1 || !lengths || !scores_out || (ctx->m.H > 0 && !hw_feats) ||
        (T_max > 0 && (!action_ids || !action_params)) || !subgraph_offsets || S < 1) {
        set_error("wm_rollout_score_from: null pointer, n_bank < 1 or S < 1 for a non-empty batch");
        return WM_ERR_ARG;
    }
    CallArgs a = {};
    a.init_states = bank; a.init_index = bank_index; a.n_init = n_bank; a.start = start;
    a.action_ids = action_ids; a.action_params = action_params; a.lengths = lengths;
    a.hw_feats = hw_feats; a.scores_out = scores_out; a.offsets = subgraph_offsets;
    a.B = B; a.S = S; a.T_max = T_max;
    if (typed_split_applies(ctx, a, true))
        return typed_split_score(ctx, a, static_cast<cudaStream_t>(cuda_stream), "wm_rollout_score_from");
    return run_rollout(ctx, a, static_cast<cudaStream_t>(cuda_stream), "wm_rollout_score_from");
}

int wm_last_kernel_ms(wm_ctx* ctx, void* cuda_stream, float* ms_out) {
    if (!ctx || !ms_out) {
        set_error("wm_last_kernel_ms: null argument");
        return WM_ERR_ARG;
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    Workspace* ws = nullptr;
    {
        std::lock_guard<std::mutex> lk(ctx->mu);
        for (Workspace* w : ctx->pool)
            if (w->stream == st) ws = w;
    }
    if (!ws || !ws->timed) {
        set_error("wm_last_kernel_ms: no timed call on this stream (set WM_OPT_TIMING first)");
        return WM_ERR_ARG;
    }
    WM_CUDA_TRY(cudaEventSynchronize(ws->ev1));
    WM_CUDA_TRY(cudaEventElapsedTime(ms_out, ws->ev0, ws->ev1));
    return WM_OK;
}

int wm_topk(const float* scores, const int32_t* subgraph_offsets, int32_t S, int32_t k, int32_t* idx_out,
            void* cuda_stream) {
    if (S < 0 || k <= 0 || k > WM_MAX_K) {
        set_error("wm_topk: size out of range (S=%d k=%d)", S, k);
        return WM_ERR_ARG;
    }
    if (S == 0) return WM_OK;
    if (!scores || !subgraph_offsets || !idx_out) {
        set_error("wm_topk: null pointer");
        return WM_ERR_ARG;
    }
    nvtx::Range r("wm_topk");
    return launch_topk(scores, subgraph_offsets, S, k, idx_out, static_cast<cudaStream_t>(cuda_stream));
}

int wm_check(wm_ctx* ctx, void* cuda_stream) {
    if (!ctx) {
        set_error("wm_check: null ctx");
        return WM_ERR_ARG;
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    WM_CUDA_TRY(cudaSetDevice(ctx->device));
    uint32_t word = 0;
    WM_CUDA_TRY(cudaMemcpyAsync(&word, ctx->fault, sizeof(word), cudaMemcpyDeviceToHost, st));
    WM_CUDA_TRY(cudaMemsetAsync(ctx->fault, 0, sizeof(word), st));
    WM_CUDA_TRY(cudaStreamSynchronize(st));
    return (int)(word & 0x7fffffffu);
}

// wm_score_topk_host splits a call into chunks of whole subgraphs of at least this many candidates (WM_HOST_CHUNK_MIN
// in the environment overrides it: the tests use a small value to exercise the chunked path on small batches)
static int64_t host_chunk_min() {
    static const int64_t v = [] {
        const char* e = getenv("WM_HOST_CHUNK_MIN");
        const long long x = e ? atoll(e) : 0;
        return (int64_t)(x > 0 ? x : 16384);
    }();
    return v;
}
#define kHostChunkMin host_chunk_min()

// widen the compact host encodings (uint8 type ids, uint16 parameters) to the int32 arrays the kernels read
__global__ void wm_widen_kernel(const uint8_t* __restrict__ ids8, const uint16_t* __restrict__ par16, int32_t* __restrict__ ids,
                                int32_t* __restrict__ par, int64_t n_ids, int64_t n_par) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_par; i += stride) par[i] = par16[i];
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_ids; i += stride) ids[i] = ids8[i];
}

// Ragged entry: the VALID steps only, packed candidate after candidate (ids8 [N], par16 [N, P], so [B + 1] = first step of
// every candidate, all indexed from the call's first step) -> the padded int32 arrays the kernels read and the lengths.
// Positions past a candidate's length are left as they are: no kernel reads them.  A length outside [0, T_max] is stored as
// it is (K2 clamps it and raises WM_FAULT_LEN) and clamped here.
__global__ void wm_expand_kernel(const uint8_t* __restrict__ ids8, const uint16_t* __restrict__ par16,
                                 const int32_t* __restrict__ so, int32_t* __restrict__ ids, int32_t* __restrict__ par,
                                 int32_t* __restrict__ lens, int64_t c0, int64_t Bc, int T_max, int P) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x, n = Bc * T_max;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += stride) {
        const int64_t b = c0 + e / T_max;
        const int t = (int)(e % T_max);
        const int first = so[b], len = so[b + 1] - first;
        if (t == 0) lens[b] = len;
        if (t < len) {
            const int64_t src = (int64_t)first + t, dst = b * T_max + t;
            ids[dst] = ids8[src];
            for (int j = 0; j < P; ++j) par[dst * P + j] = par16[src * P + j];
        }
    }
}

// Shared body of wm_score_topk_host (int32 arrays: ib = pb = 4), wm_score_topk_host_compact (ib = 1, pb = 2: the arrays
// are staged as they come and widened on the device by wm_widen_kernel) and wm_score_topk_host_ragged (ib = 1, pb = 2,
// step_offsets non-null: valid steps only, expanded on the device by wm_expand_kernel).
static int score_topk_host_impl(wm_ctx* ctx, const float* init_states, const void* action_ids, const void* action_params,
                                int ib, int pb, const int32_t* lengths, const int32_t* step_offsets, const float* hw_feats,
                                const int32_t* subgraph_offsets, int64_t B, int32_t S, int32_t T_max, int32_t k,
                                float* scores_out, int32_t* idx_out, void* cuda_stream) {
    const bool compact = ib != 4, ragged = step_offsets != nullptr;
    if (!ctx) {
        set_error("wm_score_topk_host: null ctx");
        return WM_ERR_ARG;
    }
    if (B < 0 || B > 0x7fffffffLL || S < 1 || T_max < 0 || T_max > WM_MAX_T || k <= 0 || k > WM_MAX_K ||
        !subgraph_offsets || !idx_out || !init_states || (!lengths && !ragged) || (ctx->m.H > 0 && !hw_feats) ||
        (B > 0 && T_max > 0 && (!action_ids || !action_params))) {
        set_error("wm_score_topk_host: bad argument");
        return WM_ERR_ARG;
    }
    const int64_t n_steps = ragged ? (B > 0 ? (int64_t)step_offsets[B] - step_offsets[0] : 0) : 0;
    if (ragged && B > 0 && (step_offsets[0] != 0 || n_steps < 0 || n_steps > B * (int64_t)T_max)) {
        set_error("wm_score_topk_host_ragged: step_offsets must start at 0 and end at the number of valid steps (<= B * T_max)");
        return WM_ERR_ARG;
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    WM_CUDA_TRY(cudaSetDevice(ctx->device));
    // host-entry calls on one ctx are serialised (include/wm.h): the staging buffer, the helper streams and their events
    // are shared by every call
    std::lock_guard<std::mutex> host_lock(ctx->host_mu);
    nvtx::Range nr("wm_score_topk_host");
    Workspace* ws = acquire_ws(ctx, st);
    if (!ws) {
        set_error("wm_score_topk_host: cannot allocate workspace");
        return WM_ERR_CUDA;
    }
    const Model& m = ctx->m;
    auto up16 = [](size_t x) { return (x + 255) & ~(size_t)255; };
    const size_t b_z0 = up16((size_t)S * m.d * 4), b_hw = up16((size_t)S * m.H * 4);
    const size_t b_ids = up16((size_t)B * T_max * 4), b_par = up16((size_t)B * T_max * m.P * 4);
    const size_t b_len = up16((size_t)B * 4), b_off = up16((size_t)(S + 1) * 4);
    const size_t b_sc = up16((size_t)B * 4), b_idx = up16((size_t)S * k * 4);
    // Chunk plan: up to 4 chunks of whole subgraphs with about equal candidate counts.  The copy of chunk i+1 then
    // overlaps the kernels of chunk i (PCIe and the rollout kernel are about equally long on the bf16 configs), and
    // consecutive chunks' kernels run on alternating streams so that a chunk too small to fill the GPU does not idle it.
    // (at least kHostChunkMin candidates per chunk: below that the extra launches cost more than the overlap gains)
    // (measured: cfg 3, 65,536 candidates, +33 %; cfg 2, 32,768 candidates / 1 ms per call, -10 % with 2 or 4 chunks)
    int nch = B >= 4 * kHostChunkMin ? 4 : 1;
    nch = nch > S ? S : nch;
    int cs[5] = {0, 0, 0, 0, 0};
    if (nch > 1) {
        int c = 1;
        for (int s = 1; s < S && c < nch; ++s)
            if ((int64_t)subgraph_offsets[s] * nch >= (int64_t)B * c) cs[c++] = s;
        nch = c;
        cs[nch] = S;
    }
    const size_t b_reb = up16((size_t)(S + 5) * 4);
    const size_t n_raw = ragged ? (size_t)n_steps : (size_t)B * T_max;      // staged 8- / 16-bit elements (per slot)
    const size_t b_ids8 = compact ? up16(n_raw * ib) : 0, b_par16 = compact ? up16(n_raw * m.P * pb) : 0;
    const size_t b_so = ragged ? up16((size_t)(B + 1) * 4) : 0;
    const size_t need = b_z0 + b_hw + b_ids + b_par + b_len + b_off + b_sc + b_idx + b_reb + b_ids8 + b_par16 + b_so;
    if (ws->stage_cap < need) {
        if (ws->stage) {
            WM_CUDA_TRY(cudaStreamSynchronize(st));
            WM_CUDA_TRY(cudaFree(ws->stage));
            ws->stage = nullptr;
            ws->stage_cap = 0;
        }
        WM_CUDA_TRY(cudaMalloc(&ws->stage, need));
        ws->stage_cap = need;
    }
    char* p = static_cast<char*>(ws->stage);
    float* dz0 = (float*)p; p += b_z0;
    float* dhw = (float*)p; p += b_hw;
    int32_t* dids = (int32_t*)p; p += b_ids;
    int32_t* dpar = (int32_t*)p; p += b_par;
    int32_t* dlen = (int32_t*)p; p += b_len;
    int32_t* doff = (int32_t*)p; p += b_off;
    float* dsc = (float*)p; p += b_sc;
    int32_t* didx = (int32_t*)p; p += b_idx;
    int32_t* dreb = (int32_t*)p; p += b_reb;
    uint8_t* dids8 = (uint8_t*)p; p += b_ids8;
    uint16_t* dpar16 = (uint16_t*)p; p += b_par16;
    int32_t* dso = (int32_t*)p;
    const auto H2D = cudaMemcpyHostToDevice;
    const char* h_ids = static_cast<const char*>(action_ids);
    const char* h_par = static_cast<const char*>(action_params);
    // copy candidates [c0, c0 + Bc) of the action arrays on stream `cs`; compact: stage raw, widen on stream `ks`
    // (the caller orders `ks` after the copy)
    auto copy_actions = [&](int64_t c0, int64_t Bc, cudaStream_t cs) -> int {
        if (Bc <= 0 || T_max <= 0) return WM_OK;
        const size_t ni = (size_t)Bc * T_max, np_ = ni * m.P;
        if (ragged) {      // the candidates' valid steps are one contiguous run of the packed arrays
            const size_t n0 = (size_t)step_offsets[c0], n1 = (size_t)step_offsets[c0 + Bc];
            WM_CUDA_TRY(cudaMemcpyAsync(dso + c0, step_offsets + c0, (size_t)(Bc + 1) * 4, H2D, cs));
            if (n1 > n0) {
                WM_CUDA_TRY(cudaMemcpyAsync(dids8 + n0, h_ids + n0, n1 - n0, H2D, cs));
                WM_CUDA_TRY(cudaMemcpyAsync(dpar16 + n0 * m.P, h_par + n0 * m.P * 2, (n1 - n0) * m.P * 2, H2D, cs));
            }
        } else if (!compact) {
            WM_CUDA_TRY(cudaMemcpyAsync(dids + c0 * T_max, h_ids + (size_t)c0 * T_max * 4, ni * 4, H2D, cs));
            WM_CUDA_TRY(cudaMemcpyAsync(dpar + c0 * T_max * m.P, h_par + (size_t)c0 * T_max * m.P * 4, np_ * 4, H2D, cs));
        } else {
            WM_CUDA_TRY(cudaMemcpyAsync(dids8 + c0 * T_max, h_ids + (size_t)c0 * T_max, ni, H2D, cs));
            WM_CUDA_TRY(cudaMemcpyAsync(dpar16 + c0 * T_max * m.P, h_par + (size_t)c0 * T_max * m.P * 2, np_ * 2, H2D, cs));
        }
        return WM_OK;
    };
    auto widen = [&](int64_t c0, int64_t Bc, cudaStream_t ks) -> int {
        if (ragged && Bc > 0 && T_max <= 0) WM_CUDA_TRY(cudaMemsetAsync(dlen + c0, 0, (size_t)Bc * 4, ks));   // (no step can exist)
        if (!compact || Bc <= 0 || T_max <= 0) return WM_OK;
        const int64_t ni = Bc * T_max, np_ = ni * m.P;
        const int grid = (int)std::min<int64_t>((np_ + 255) / 256, (int64_t)ctx->n_sms * 8);
        if (ragged) {
            wm_expand_kernel<<<grid, 256, 0, ks>>>(dids8, dpar16, dso, dids, dpar, dlen, c0, Bc, T_max, m.P);
            WM_CUDA_TRY(cudaGetLastError());
            ctx->launches.fetch_add(1);
            return WM_OK;
        }
        wm_widen_kernel<<<grid, 256, 0, ks>>>(dids8 + c0 * T_max, dpar16 + c0 * T_max * m.P, dids + c0 * T_max,
                                              dpar + c0 * T_max * m.P, ni, np_);
        WM_CUDA_TRY(cudaGetLastError());
        ctx->launches.fetch_add(1);
        return WM_OK;
    };
    if (nch > 1) {
        if (!ctx->hs_copy) {
            WM_CUDA_TRY(cudaStreamCreateWithFlags(&ctx->hs_copy, cudaStreamNonBlocking));
            for (int i = 0; i < 2; ++i) {
                WM_CUDA_TRY(cudaStreamCreateWithFlags(&ctx->hs_k[i], cudaStreamNonBlocking));
                WM_CUDA_TRY(cudaEventCreateWithFlags(&ctx->hev_done[i], cudaEventDisableTiming));
            }
            WM_CUDA_TRY(cudaEventCreateWithFlags(&ctx->hev_start, cudaEventDisableTiming));
            for (int i = 0; i < 8; ++i) WM_CUDA_TRY(cudaEventCreateWithFlags(&ctx->hev_copy[i], cudaEventDisableTiming));
        }
        if (ctx->h_off_cap < (size_t)(S + 5)) {
            if (ctx->h_off) WM_CUDA_TRY(cudaFreeHost(ctx->h_off));
            ctx->h_off = nullptr;
            WM_CUDA_TRY(cudaMallocHost(&ctx->h_off, (size_t)(S + 5 + 1024) * 4));
            ctx->h_off_cap = (size_t)(S + 5 + 1024);
        }
        // per-chunk offsets rebased to the chunk's first candidate (the rollout kernel indexes candidates from 0)
        int reb_at[4];
        {
            int o = 0;
            for (int c = 0; c < nch; ++c) {
                reb_at[c] = o;
                for (int s = cs[c]; s <= cs[c + 1]; ++s) ctx->h_off[o++] = subgraph_offsets[s] - subgraph_offsets[cs[c]];
            }
        }
        cudaStream_t cp = ctx->hs_copy;
        WM_CUDA_TRY(cudaEventRecord(ctx->hev_start, st));     // everything below is ordered after prior work on `st`
        WM_CUDA_TRY(cudaStreamWaitEvent(cp, ctx->hev_start, 0));
        for (int i = 0; i < 2; ++i) WM_CUDA_TRY(cudaStreamWaitEvent(ctx->hs_k[i], ctx->hev_start, 0));
        WM_CUDA_TRY(cudaMemcpyAsync(dz0, init_states, (size_t)S * m.d * 4, H2D, cp));
        if (m.H) WM_CUDA_TRY(cudaMemcpyAsync(dhw, hw_feats, (size_t)S * m.H * 4, H2D, cp));
        WM_CUDA_TRY(cudaMemcpyAsync(doff, subgraph_offsets, (size_t)(S + 1) * 4, H2D, cp));
        WM_CUDA_TRY(cudaMemcpyAsync(dreb, ctx->h_off, (size_t)(S + nch) * 4, H2D, cp));
        // one chunk: its copies on the copy stream, its kernels on one of the two compute streams
        auto chunk = [&](int c) -> int {
            const int s0 = cs[c], Sc = cs[c + 1] - cs[c];
            const int64_t c0 = subgraph_offsets[s0], Bc = (int64_t)subgraph_offsets[cs[c + 1]] - c0;
            if (Bc > 0) {
                if (!ragged) WM_CUDA_TRY(cudaMemcpyAsync(dlen + c0, lengths + c0, (size_t)Bc * 4, H2D, cp));
                const int rc0 = copy_actions(c0, Bc, cp);
                if (rc0 != WM_OK) return rc0;
            }
            WM_CUDA_TRY(cudaEventRecord(ctx->hev_copy[c], cp));
            cudaStream_t ks = ctx->hs_k[c & 1];
            WM_CUDA_TRY(cudaStreamWaitEvent(ks, ctx->hev_copy[c], 0));
            {
                const int rc0 = widen(c0, Bc, ks);
                if (rc0 != WM_OK) return rc0;
            }
            if (Bc > 0) {
                const int rc = wm_rollout_score(ctx, dz0 + (size_t)s0 * m.d, dids + c0 * T_max, dpar + c0 * T_max * m.P,
                                                dlen + c0, dhw + (size_t)s0 * m.H, dsc + c0, dreb + reb_at[c], Bc, Sc, T_max, ks);
                if (rc != WM_OK) return rc;
            }
            // global offsets + the global score array: the indices come out global
            return wm_topk(dsc, doff + s0, Sc, k, didx + (size_t)s0 * k, ks);
        };
        int crc = WM_OK;
        for (int c = 0; c < nch && crc == WM_OK; ++c) crc = chunk(c);
        // join the helper streams back into `st` on every path: after an error the caller's stream must still be ordered
        // after whatever was already enqueued on them (they read the staging buffer a later call may free or refill)
        for (int i = 0; i < 2; ++i) {
            if (cudaEventRecord(ctx->hev_done[i], ctx->hs_k[i]) == cudaSuccess) cudaStreamWaitEvent(st, ctx->hev_done[i], 0);
        }
        if (cudaEventRecord(ctx->hev_copy[7], cp) == cudaSuccess) cudaStreamWaitEvent(st, ctx->hev_copy[7], 0);
        if (crc != WM_OK) {
            cudaStreamSynchronize(st);
            return crc;
        }
        if (scores_out && B) WM_CUDA_TRY(cudaMemcpyAsync(scores_out, dsc, (size_t)B * 4, cudaMemcpyDeviceToHost, st));
        WM_CUDA_TRY(cudaMemcpyAsync(idx_out, didx, (size_t)S * k * 4, cudaMemcpyDeviceToHost, st));
        WM_CUDA_TRY(cudaStreamSynchronize(st));
        return WM_OK;
    }
    WM_CUDA_TRY(cudaMemcpyAsync(dz0, init_states, (size_t)S * m.d * 4, H2D, st));
    if (m.H) WM_CUDA_TRY(cudaMemcpyAsync(dhw, hw_feats, (size_t)S * m.H * 4, H2D, st));
    {
        int rc0 = copy_actions(0, B, st);
        if (rc0 == WM_OK) rc0 = widen(0, B, st);
        if (rc0 != WM_OK) return rc0;
    }
    if (B && !ragged) WM_CUDA_TRY(cudaMemcpyAsync(dlen, lengths, (size_t)B * 4, H2D, st));
    WM_CUDA_TRY(cudaMemcpyAsync(doff, subgraph_offsets, (size_t)(S + 1) * 4, H2D, st));
    int rc = wm_rollout_score(ctx, dz0, dids, dpar, dlen, dhw, dsc, doff, B, S, T_max, cuda_stream);
    if (rc != WM_OK) return rc;
    rc = wm_topk(dsc, doff, S, k, didx, cuda_stream);
    if (rc != WM_OK) return rc;
    if (scores_out && B) WM_CUDA_TRY(cudaMemcpyAsync(scores_out, dsc, (size_t)B * 4, cudaMemcpyDeviceToHost, st));
    WM_CUDA_TRY(cudaMemcpyAsync(idx_out, didx, (size_t)S * k * 4, cudaMemcpyDeviceToHost, st));
    WM_CUDA_TRY(cudaStreamSynchronize(st));
    return WM_OK;
}

int wm_launch_empty(void* cuda_stream) {
    wm_empty_kernel<<<1, 32, 0, static_cast<cudaStream_t>(cuda_stream)>>>();
    WM_CUDA_TRY(cudaGetLastError());
    return WM_OK;
}

int wm_score_topk_host(wm_ctx* ctx, const float* init_states, const int32_t* action_ids,
                       const int32_t* action_params, const int32_t* lengths, const float* hw_feats,
                       const int32_t* subgraph_offsets, int64_t B, int32_t S, int32_t T_max, int32_t k,
                       float* scores_out, int32_t* idx_out, void* cuda_stream) {
    return score_topk_host_impl(ctx, init_states, action_ids, action_params, 4, 4, lengths, nullptr, hw_feats, subgraph_offsets, B, S,
                                T_max, k, scores_out, idx_out, cuda_stream);
}

int wm_score_topk_host_compact(wm_ctx* ctx, const float* init_states, const uint8_t* action_ids,
                               const uint16_t* action_params, const int32_t* lengths, const float* hw_feats,
                               const int32_t* subgraph_offsets, int64_t B, int32_t S, int32_t T_max, int32_t k,
                               float* scores_out, int32_t* idx_out, void* cuda_stream) {
    if (ctx && ctx->m.n_types > 256) {
        set_error("wm_score_topk_host_compact: uint8 type ids need n_types <= 256");
        return WM_ERR_UNSUPPORTED;
    }
    return score_topk_host_impl(ctx, init_states, action_ids, action_params, 1, 2, lengths, nullptr, hw_feats, subgraph_offsets, B, S,
                                T_max, k, scores_out, idx_out, cuda_stream);
}

int wm_score_topk_host_ragged(wm_ctx* ctx, const float* init_states, const uint8_t* step_ids, const uint16_t* step_params,
                              const int32_t* step_offsets, const float* hw_feats, const int32_t* subgraph_offsets, int64_t B,
                              int32_t S, int32_t T_max, int32_t k, float* scores_out, int32_t* idx_out, void* cuda_stream) {
    if (ctx && ctx->m.n_types > 256) {
        set_error("wm_score_topk_host_ragged: uint8 type ids need n_types <= 256");
        return WM_ERR_UNSUPPORTED;
    }
    if (!step_offsets) {
        set_error("wm_score_topk_host_ragged: null step_offsets");
        return WM_ERR_ARG;
    }
    return score_topk_host_impl(ctx, init_states, step_ids, step_params, 1, 2, nullptr, step_offsets, hw_feats, subgraph_offsets,
                                B, S, T_max, k, scores_out, idx_out, cuda_stream);
}

int64_t wm_launch_count(const wm_ctx* ctx) {
    if (!ctx) return topk_launches();
    return ctx->launches.load();
}

}  // extern "C"
#pragma GCC visibility pop

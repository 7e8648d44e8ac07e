"""Float64 CPU oracle for the batched candidate evaluator.  TEST INFRASTRUCTURE ONLY.

What it computes is the plain definition (no approximation in the method, so no algorithm to follow):

    z_0 = init_states[s]                                   PAPER.md:215 ("initial tensor-program state of the task")
    z_t = F(z_{t-1}, a_t),  t = 1..len                     PAPER.md:68-71 Eq.1, :162 Eq.8, :166 (recurrent rollout)
    steps with t > len leave z unchanged                   PAPER.md:176 Eq.11 (rollout mask m_t)
    phi = mean_t a_t (0 if len = 0)                        PAPER.md:186 (action features; BASELINE.json cfg 1 form)
      or, phi_kind = PHI_STRUCT, the paper's structured statistics (phi_struct below; S25)
    y   = G([z_T ; phi ; h])                               PAPER.md:122 Eq.3, :188 Eq.12
    top-k per subgraph by (score desc, index asc)

with the network shapes BASELINE.json's configs bind (F = residual MLP [+LayerNorm] or GRU-style gate,
G = MLP, embedding = table + Linear(log2 params) or bucketed table); readings S1..S23 in DESIGN.md §3.

Everything is numpy float64; weights arrive as the dict gen.make_weights() returns (or read_weight_file()).
Two implementations: `rollout_score_vec` (loop over t, matmul over one subgraph's candidates, np.where
mask) and `rollout_score_scalar` (pure per-candidate python loops, math.erf) — the second pins the first.

Pins (tests/test_oracle_pins.py): P1..P13 of SURVEY.md §8(c) — hand-expanded 2x3 MLP step and GRU step
(values in tests/golden/), closed forms, torch float64 library cross-checks, scalar-vs-vector brute
force, top-k vs full sort; P14/P15 the TransH step, P16/P17 the structured phi (hand-worked sequence in
tests/golden/p16_phi_struct.txt, closed forms, a scorer that reads single features), P18 prefix-latent reuse against
the literal path, P19/P20 the tree-ensemble ranker (hand-worked forest in tests/golden/p19_forest.txt, stumps in closed
form, scikit-learn's DecisionTreeRegressor as the library cross-check).  The paper prints no worked numeric example of this path, so the composition
at full size rests on those pins: beyond them, parity unpinned.
"""
from __future__ import annotations

import math
import struct
from typing import Dict, Optional, Tuple

import numpy as np
from scipy.special import erf as _erf

KIND_MLP, KIND_MLP_LN, KIND_GRU, KIND_TRANSH = 0, 1, 2, 3
EMBED_LINEAR, EMBED_BUCKET = 0, 1
PHI_MEAN, PHI_STRUCT, PHI_TYPED = 0, 1, 2
F64 = np.float64


# ----------------------------------------------------------------------------- pieces

def gelu(x: np.ndarray) -> np.ndarray:
    """Exact GELU x*Phi(x) (S5)."""
    x = np.asarray(x, dtype=F64)
    return 0.5 * x * (1.0 + _erf(x / math.sqrt(2.0)))


def layer_norm(v: np.ndarray, gamma: np.ndarray, beta: np.ndarray, eps: float) -> np.ndarray:
    """LayerNorm over the last axis, population variance (S6; PAPER.md:164 'finally normalized')."""
    v = np.asarray(v, dtype=F64)
    mean = v.mean(axis=-1, keepdims=True)
    var = ((v - mean) ** 2).mean(axis=-1, keepdims=True)
    return gamma * (v - mean) / np.sqrt(var + eps) + beta


def embed_linear(ids: np.ndarray, params: np.ndarray, E, W_p, b_p) -> np.ndarray:
    """a = E[id] + W_p @ log2(p) + b_p   (configs 1-4; north_star 'token-id gather plus projection')."""
    lp = np.log2(np.asarray(params, dtype=F64))
    return np.asarray(E, F64)[ids] + lp @ np.asarray(W_p, F64).T + np.asarray(b_p, F64)


def bucket_index(p: int, n_buckets: int) -> int:
    """Quarter-octave bucket min(n_b-1, floor(4*log2 p)) in exact integer arithmetic (S10)."""
    return min(n_buckets - 1, (int(p) ** 4).bit_length() - 1)


def embed_bucket(ids: np.ndarray, params: np.ndarray, Tbl, P: int, n_buckets: int) -> np.ndarray:
    """a = sum_j Tbl[(id*P + j)*n_b + bucket(p_j)]   (config 5, S10)."""
    ids = np.asarray(ids)
    params = np.asarray(params)
    Tbl = np.asarray(Tbl, F64)
    flat_p = params.reshape(-1, P)
    flat_id = ids.reshape(-1)
    out = np.zeros((flat_id.shape[0], Tbl.shape[1]), dtype=F64)
    bk = np.array([[bucket_index(int(p), n_buckets) for p in row] for row in flat_p], dtype=np.int64) \
        if flat_p.size < 4096 else _bucket_vec(flat_p, n_buckets)
    for j in range(P):
        out += Tbl[(flat_id.astype(np.int64) * P + j) * n_buckets + bk[:, j]]
    return out.reshape(ids.shape + (Tbl.shape[1],))


def _bucket_vec(p: np.ndarray, n_buckets: int) -> np.ndarray:
    """Vectorised bucket_index, exact for every int32 p >= 1: bit_length(p^4) - 1 = #{b >= 1 : p^4 >= 2^b}, and
    p^4 >= 2^b  <=>  p^2 >= ceil(sqrt(2^b)) (p^2 < 2^62 is exact in int64; the thresholds come from math.isqrt)."""
    p2 = p.astype(np.int64) ** 2
    bl = np.zeros(p2.shape, dtype=np.int64)
    for b in range(1, 124):
        r = math.isqrt(1 << b)
        thr = r if r * r == (1 << b) else r + 1
        bl += (p2 >= np.int64(thr)).astype(np.int64)
    return np.minimum(n_buckets - 1, bl)


def step_mlp(z, a, W1, b1, W2, b2, gamma=None, beta=None, eps: float = 1e-5) -> np.ndarray:
    """z' = z + W2 gelu(W1 [z;a] + b1) + b2, then LayerNorm if gamma is given (cfg 1 / cfg 2-4)."""
    x = np.concatenate([z, a], axis=-1)
    u = x @ np.asarray(W1, F64).T + np.asarray(b1, F64)
    v = z + gelu(u) @ np.asarray(W2, F64).T + np.asarray(b2, F64)
    if gamma is None:
        return v
    return layer_norm(v, np.asarray(gamma, F64), np.asarray(beta, F64), eps)


def _sigmoid(x):
    return 1.0 / (1.0 + np.exp(-x))


def step_gru(z, a, W_g, W_r, W_h) -> np.ndarray:
    """g=s(W_g[z;a]); r=s(W_r[z;a]); z'=(1-g) z + g tanh(W_h [r*z; a])   (cfg 5)."""
    x = np.concatenate([z, a], axis=-1)
    g = _sigmoid(x @ np.asarray(W_g, F64).T)
    r = _sigmoid(x @ np.asarray(W_r, F64).T)
    h = np.tanh(np.concatenate([r * z, a], axis=-1) @ np.asarray(W_h, F64).T)
    return (1.0 - g) * z + g * h


TRANSH_EPS = 1e-12   # added under both square roots of step_transh (DESIGN.md §3 S24)


def step_transh(z, a, W_w, W_d, W1, b1, W2, b2, eps: float = TRANSH_EPS) -> np.ndarray:
    """The paper's TransH-based predictor (ref [41]; NEXT row f1, reading S24), in its three stated stages:
      1. "the current state is first transformed in an action-conditioned geometric space": the action defines a
         hyperplane with unit normal w = W_w a / sqrt(|W_w a|^2 + eps); the state is projected onto it,
         z_perp = z - (w.z) w, and translated inside it by d = W_d a (TransH: h_perp + d_r);
      2. "then combined with the action embedding through a residual multilayer transformation":
         v = x + W2 gelu(W1 [x ; a] + b1) + b2 with x = z_perp + d;
      3. "and finally normalized": z' = v / sqrt(|v|^2 + eps)  (the losses live in the normalized
         state-representation space)."""
    W_w, W_d = np.asarray(W_w, F64), np.asarray(W_d, F64)
    u = a @ W_w.T
    w = u / np.sqrt(np.sum(u * u, axis=-1, keepdims=True) + eps)
    z_perp = z - np.sum(w * z, axis=-1, keepdims=True) * w
    x = z_perp + a @ W_d.T
    h = gelu(np.concatenate([x, a], axis=-1) @ np.asarray(W1, F64).T + np.asarray(b1, F64))
    v = x + h @ np.asarray(W2, F64).T + np.asarray(b2, F64)
    return v / np.sqrt(np.sum(v * v, axis=-1, keepdims=True) + eps)


def phi_struct(ids, params, n_types: int) -> np.ndarray:
    """Structured action features of ONE action sequence, given by its valid steps only (ids [len], params [len,P]).

    PAPER.md:186: phi(a_1:T) is "a structured action feature vector derived from the scheduling actions, including
    statistics such as action counts, sequence length, and action-specific numeric attributes" — the paper lists the
    ingredients, not a layout; reading S25 fixes it as, in this order,
        c_k   = #{t : id_t = k},             k = 0..n_types-1     (action counts)
        len                                                       (sequence length)
        s_j   = sum_t log2 p_tj,             j = 0..P-1           (numeric attributes: total per parameter slot)
        m_j   = s_j / len                                         (mean; 0 for an empty sequence)
        x_j   = max_t log2 p_tj                                   (largest; 0 for an empty sequence)
    Returns float64 [n_types + 1 + 3P]."""
    ids = np.asarray(ids).astype(np.int64).reshape(-1)
    par = np.asarray(params)
    n, P = ids.shape[0], par.shape[-1]
    counts = np.array([np.count_nonzero(ids == k) for k in range(n_types)], dtype=F64)
    if n == 0:
        s = m = x = np.zeros(P, dtype=F64)
    else:
        lp = np.log2(par.reshape(n, P).astype(F64))
        s, m, x = lp.sum(axis=0), lp.sum(axis=0) / n, lp.max(axis=0)
    return np.concatenate([counts, [float(n)], s, m, x])


def phi_struct_typed(ids, params, n_types: int) -> np.ndarray:
    """Structured action features with ACTION-SPECIFIC numeric attributes (phi_kind = PHI_TYPED; S28).

    PAPER.md:186 lists "action counts, sequence length, and action-specific numeric attributes": slot j of one action type
    is a different attribute from slot j of another (a split factor, an unroll depth, a thread extent ...), so the numeric
    statistics are kept PER ACTION TYPE instead of pooled per slot as in phi_struct (S25).  Layout, in this order:
        c_k                                    k = 0..n_types-1     (action counts)
        len                                                         (sequence length)
        for every type k = 0..n_types-1:
            s_kj = sum over steps of type k of log2 p_tj,   j = 0..P-1
            m_kj = s_kj / c_k                               (0 when the type does not occur)
            x_kj = max over steps of type k of log2 p_tj    (0 when the type does not occur)
    Returns float64 [n_types + 1 + 3 n_types P]."""
    ids = np.asarray(ids).astype(np.int64).reshape(-1)
    par = np.asarray(params)
    n, P = ids.shape[0], par.shape[-1]
    lp = np.log2(par.reshape(n, P).astype(F64)) if n else np.zeros((0, P), dtype=F64)
    counts = np.zeros(n_types, dtype=F64)
    blocks = []
    for k in range(n_types):
        rows = lp[ids == k]
        counts[k] = rows.shape[0]
        if rows.shape[0] == 0:
            blocks.append(np.zeros(3 * P, dtype=F64))
        else:
            blocks.append(np.concatenate([rows.sum(axis=0), rows.sum(axis=0) / rows.shape[0], rows.max(axis=0)]))
    return np.concatenate([counts, [float(n)]] + blocks)


def _phi_features(phi_kind: int, ids, params, n_types: int) -> np.ndarray:
    return phi_struct_typed(ids, params, n_types) if phi_kind == PHI_TYPED else phi_struct(ids, params, n_types)


def forest_score(x, Tf, Tt, Tv, Tb, return_margin: bool = False):
    """Tree-ensemble ranker (NEXT row f4).  PAPER.md:190: "G is implemented as an XGBoost ranking model" — an additive
    ensemble of regression trees over the concatenated features (Eq.12); the paper prints no tree, so reading S27
     fixes synthetic COMPLETE binary trees in heap order: at node i (root 0) go to child 2i+1 when
    x[f_i] < t_i, else to child 2i+2; after `depth` levels the node index minus (2^depth - 1) is the leaf;
    y = Tb + sum over trees of the leaf value.  The comparison is taken in float32 on both sides (x and t rounded to
    float32: a decision, so the kernel's precision), the sum in float64.
    x [n, n_in]; Tf, Tt [n_trees, 2^depth - 1]; Tv [n_trees, 2^depth]; Tb [1].  One candidate, one tree, one level at a
    time.  With return_margin also the smallest |x[f] - t| met on any path of the candidate (how close it came to
    taking another branch)."""
    x32 = np.asarray(x, dtype=np.float32)
    Tf = np.asarray(Tf).astype(np.int64); Tt = np.asarray(Tt, dtype=np.float32); Tv = np.asarray(Tv, dtype=F64)
    n_trees, nodes = Tf.shape
    depth = int(round(math.log2(nodes + 1)))
    assert 2 ** depth - 1 == nodes and Tv.shape == (n_trees, nodes + 1)
    y = np.full(x32.shape[0], float(np.asarray(Tb, F64).reshape(-1)[0]), dtype=F64)
    margin = np.full(x32.shape[0], np.inf, dtype=F64)
    for c in range(x32.shape[0]):
        for t in range(n_trees):
            node = 0
            for _ in range(depth):
                v, thr = x32[c, Tf[t, node]], Tt[t, node]
                margin[c] = min(margin[c], abs(float(v) - float(thr)))
                node = 2 * node + (1 if v < thr else 2)
            y[c] += Tv[t, node - nodes]
    return (y, margin) if return_margin else y


def _rank(x: np.ndarray, w: Dict[str, np.ndarray], n_layers: int) -> np.ndarray:
    """G on the concatenated features: the forest when the model carries one, else the MLP."""
    if "Tf" in w:
        return forest_score(x, w["Tf"], w["Tt"], w["Tv"], w["Tb"])
    return scorer(x, w, n_layers)


def scorer(x: np.ndarray, w: Dict[str, np.ndarray], n_layers: int) -> np.ndarray:
    """G as an MLP: hidden linears followed by GELU, last linear plain (S8). Returns [...]."""
    for i in range(n_layers):
        x = x @ np.asarray(w[f"Ws{i}"], F64).T + np.asarray(w[f"bs{i}"], F64)
        if i + 1 < n_layers:
            x = gelu(x)
    return x[..., 0]


def _n_scorer_layers(w) -> int:
    n = 0
    while f"Ws{n}" in w:
        n += 1
    return n


def _kind(w) -> int:
    if "W_g" in w:
        return KIND_GRU
    if "W_w" in w:
        return KIND_TRANSH
    return KIND_MLP_LN if "gamma" in w else KIND_MLP


def _embed(w, ids, params, P, n_buckets):
    if "Tbl" in w:
        return embed_bucket(ids, params, w["Tbl"], P, n_buckets)
    return embed_linear(ids, params, w["E"], w["W_p"], w["b_p"])


def _step(w, z, a, eps):
    k = _kind(w)
    if k == KIND_GRU:
        return step_gru(z, a, w["W_g"], w["W_r"], w["W_h"])
    if k == KIND_TRANSH:
        return step_transh(z, a, w["W_w"], w["W_d"], w["W1"], w["b1"], w["W2"], w["b2"])
    if k == KIND_MLP_LN:
        return step_mlp(z, a, w["W1"], w["b1"], w["W2"], w["b2"], w["gamma"], w["beta"], eps)
    return step_mlp(z, a, w["W1"], w["b1"], w["W2"], w["b2"])


# ----------------------------------------------------------------------------- the path

def rollout_score_vec(w: Dict[str, np.ndarray], init_states, action_ids, action_params, lengths, hw_feats,
                      subgraph_offsets: Optional[np.ndarray], n_buckets: int = 0, ln_eps: float = 1e-5,
                      return_latent: bool = False, phi_kind: int = PHI_MEAN):
    """Scores [B] float64.  subgraph_offsets None => per-candidate init_states [B,d] / hw_feats [B,H] (S1/S2).
    phi_kind = PHI_STRUCT replaces the mean action embedding by phi_struct of the candidate's valid steps."""
    ids = np.asarray(action_ids)
    par = np.asarray(action_params)
    lens = np.asarray(lengths).astype(np.int64)
    B, T = ids.shape
    P = par.shape[2]
    z0 = np.asarray(init_states, F64)
    hw = np.asarray(hw_feats, F64)
    nl = _n_scorer_layers(w)
    if subgraph_offsets is None:
        segs = [(i, i + 1, i) for i in range(B)] if B else []
        # one block over all candidates is the same computation; keep per-candidate rows together
        segs = [(0, B, None)] if B else []
    else:
        off = np.asarray(subgraph_offsets).astype(np.int64)
        segs = [(int(off[s]), int(off[s + 1]), s) for s in range(len(off) - 1)]
    scores = np.zeros(B, dtype=F64)
    lat = np.zeros((B, z0.shape[1]), dtype=F64) if return_latent else None
    da = (w["Tbl"] if "Tbl" in w else w["E"]).shape[1]
    for lo, hi, s in segs:
        n = hi - lo
        if n <= 0:
            continue
        z = z0[lo:hi].copy() if s is None else np.repeat(z0[s][None, :], n, axis=0)
        h = hw[lo:hi] if s is None else np.repeat(hw[s][None, :], n, axis=0)
        ln = lens[lo:hi]
        asum = np.zeros((n, da), dtype=F64)
        for t in range(int(ln.max()) if n else 0):
            act = ln > t                               # rollout mask m_t
            idx = np.nonzero(act)[0]
            if idx.size == 0:
                break
            a = _embed(w, ids[lo:hi][idx, t], par[lo:hi][idx, t, :], P, n_buckets)
            asum[idx] += a
            z[idx] = _step(w, z[idx], a, ln_eps)       # masked rows keep z unchanged
        phi = np.where(ln[:, None] > 0, asum / np.maximum(ln, 1)[:, None], 0.0)
        if phi_kind != PHI_MEAN:
            n_types = w["E"].shape[0] if "E" in w else w["Tbl"].shape[0] // (P * n_buckets)
            phi = np.stack([_phi_features(phi_kind, ids[lo + i, :ln[i]], par[lo + i, :ln[i], :], n_types) for i in range(n)]) \
                if n else np.zeros((0, 0))
        scores[lo:hi] = _rank(np.concatenate([z, phi, h], axis=-1), w, nl)
        if return_latent:
            lat[lo:hi] = z
    return (scores, lat) if return_latent else scores


def rollout_latents(w, init_states, action_ids, action_params, lengths, subgraph_offsets: Optional[np.ndarray],
                    n_buckets: int = 0, ln_eps: float = 1e-5) -> np.ndarray:
    """Latent after every step (prefix-latent reuse, NEXT row f3; Eq.1/8 applied recurrently):
    out[b][t] = z_{t+1} of candidate b for t < len[b], NaN elsewhere.  float64 [B, T_max, d]; one candidate at a
    time, one step at a time."""
    ids = np.asarray(action_ids); par = np.asarray(action_params)
    lens = np.asarray(lengths).astype(np.int64)
    z0 = np.asarray(init_states, F64)
    B, T = ids.shape
    P = par.shape[2]
    out = np.full((B, T, z0.shape[1]), np.nan, dtype=F64)
    seg = np.arange(B)
    if subgraph_offsets is not None:
        off = np.asarray(subgraph_offsets).astype(np.int64)
        seg = np.searchsorted(off, np.arange(B), side="right") - 1
    for b in range(B):
        z = z0[seg[b]][None, :].copy()
        for t in range(int(lens[b])):
            a = _embed(w, ids[b:b + 1, t], par[b:b + 1, t, :], P, n_buckets)
            z = _step(w, z, a, ln_eps)
            out[b, t] = z[0]
    return out


def rollout_score_from(w, bank, bank_index, start, action_ids, action_params, lengths, hw_feats, subgraph_offsets,
                       n_buckets: int = 0, ln_eps: float = 1e-5, phi_kind: int = PHI_MEAN) -> np.ndarray:
    """Scores of candidates whose first start[b] steps were rolled before: z starts at bank[bank_index[b]], steps
    start[b] .. len[b]-1 are applied, phi is taken over the WHOLE sequence, y = G([z_T ; phi ; h_s]).  Plain
    definition, one candidate at a time (the online loop re-scores mutated survivors)."""
    ids = np.asarray(action_ids); par = np.asarray(action_params)
    lens = np.asarray(lengths).astype(np.int64)
    bank = np.asarray(bank, F64); hw = np.asarray(hw_feats, F64)
    off = np.asarray(subgraph_offsets).astype(np.int64)
    B = ids.shape[0]
    P = par.shape[2]
    nl = _n_scorer_layers(w)
    n_types = w["E"].shape[0] if "E" in w else w["Tbl"].shape[0] // (P * n_buckets)
    seg = np.searchsorted(off, np.arange(B), side="right") - 1
    out = np.zeros(B, dtype=F64)
    for b in range(B):
        n = int(lens[b])
        st = min(max(int(start[b]), 0), n)
        z = bank[int(bank_index[b])][None, :].copy()
        for t in range(st, n):
            z = _step(w, z, _embed(w, ids[b:b + 1, t], par[b:b + 1, t, :], P, n_buckets), ln_eps)
        if phi_kind != PHI_MEAN:
            phi = _phi_features(phi_kind, ids[b, :n], par[b, :n, :], n_types)
        elif n > 0:
            phi = _embed(w, ids[b, :n], par[b, :n, :], P, n_buckets).sum(axis=0) / n
        else:
            phi = np.zeros((w["Tbl"] if "Tbl" in w else w["E"]).shape[1], dtype=F64)
        out[b] = _rank(np.concatenate([z[0], phi, hw[seg[b]]])[None, :], w, nl)[0]
    return out


def rollout_score_scalar(w, init_states, action_ids, action_params, lengths, hw_feats, subgraph_offsets,
                         n_buckets: int = 0, ln_eps: float = 1e-5, phi_kind: int = PHI_MEAN) -> np.ndarray:
    """Pure-python per-candidate loops (tiny inputs only); independent of the vector code above."""
    W = {k: np.asarray(v, F64).tolist() for k, v in w.items()}
    ids = np.asarray(action_ids).tolist()
    par = np.asarray(action_params).tolist()
    lens = [int(x) for x in np.asarray(lengths)]
    z0 = np.asarray(init_states, F64).tolist()
    hw = np.asarray(hw_feats, F64).tolist()
    B = len(lens)
    seg_of = list(range(B))
    if subgraph_offsets is not None:
        off = [int(x) for x in subgraph_offsets]
        for s in range(len(off) - 1):
            for b in range(off[s], off[s + 1]):
                seg_of[b] = s
    kind = _kind(w)
    P = len(par[0][0]) if B and len(par[0]) else 0

    def mv(M, x):
        return [sum(mij * xj for mij, xj in zip(row, x)) for row in M]

    def gelu1(x):
        return 0.5 * x * (1.0 + math.erf(x / math.sqrt(2.0)))

    def sig(x):
        return 1.0 / (1.0 + math.exp(-x))

    out = []
    for b in range(B):
        s = seg_of[b]
        z = list(z0[s])
        d = len(z)
        da = len(W["Tbl"][0]) if "Tbl" in W else len(W["E"][0])
        asum = [0.0] * da
        for t in range(lens[b]):
            if "Tbl" in W:
                a = [0.0] * da
                for j in range(P):
                    row = W["Tbl"][(ids[b][t] * P + j) * n_buckets + bucket_index(par[b][t][j], n_buckets)]
                    a = [x + y for x, y in zip(a, row)]
            else:
                lp = [math.log2(p) for p in par[b][t]]
                a = [e + q + c for e, q, c in zip(W["E"][ids[b][t]], mv(W["W_p"], lp), W["b_p"])]
            asum = [x + y for x, y in zip(asum, a)]
            if kind == KIND_GRU:
                x = z + a
                g = [sig(u) for u in mv(W["W_g"], x)]
                r = [sig(u) for u in mv(W["W_r"], x)]
                hcand = [math.tanh(u) for u in mv(W["W_h"], [ri * zi for ri, zi in zip(r, z)] + a)]
                z = [(1.0 - gi) * zi + gi * hi for gi, zi, hi in zip(g, z, hcand)]
            elif kind == KIND_TRANSH:
                # PAPER.md:164 in its three stages (see step_transh): project onto the action's hyperplane and
                # translate, residual MLP with the action embedding, L2-normalise
                uw = mv(W["W_w"], a)
                nw = math.sqrt(sum(x * x for x in uw) + TRANSH_EPS)
                wn = [x / nw for x in uw]
                dot = sum(wi * zi for wi, zi in zip(wn, z))
                xs = [zi - dot * wi + di for zi, wi, di in zip(z, wn, mv(W["W_d"], a))]
                hdn = [gelu1(ui + bi) for ui, bi in zip(mv(W["W1"], xs + a), W["b1"])]
                v = [xi + wi + bi for xi, wi, bi in zip(xs, mv(W["W2"], hdn), W["b2"])]
                nv = math.sqrt(sum(x * x for x in v) + TRANSH_EPS)
                z = [x / nv for x in v]
            else:
                u = [ui + bi for ui, bi in zip(mv(W["W1"], z + a), W["b1"])]
                hdn = [gelu1(ui) for ui in u]
                v = [zi + wi + bi for zi, wi, bi in zip(z, mv(W["W2"], hdn), W["b2"])]
                if kind == KIND_MLP_LN:
                    m = sum(v) / d
                    var = sum((vi - m) ** 2 for vi in v) / d
                    z = [g_ * (vi - m) / math.sqrt(var + ln_eps) + b_
                         for g_, vi, b_ in zip(W["gamma"], v, W["beta"])]
                else:
                    z = v
        phi = [x / lens[b] for x in asum] if lens[b] > 0 else [0.0] * da
        if phi_kind == PHI_STRUCT:   # S25, by counting loops (independent of phi_struct above)
            n_types = len(W["E"]) if "E" in W else len(W["Tbl"]) // (P * n_buckets)
            cnt = [0.0] * n_types
            tot = [0.0] * P
            big = [0.0] * P
            for t in range(lens[b]):
                cnt[ids[b][t]] += 1.0
                for j in range(P):
                    l2 = math.log2(par[b][t][j])
                    tot[j] += l2
                    big[j] = l2 if t == 0 else max(big[j], l2)
            phi = cnt + [float(lens[b])] + tot + [v / lens[b] if lens[b] > 0 else 0.0 for v in tot] + big
        elif phi_kind == PHI_TYPED:  # S28, by counting loops (independent of phi_struct_typed above)
            n_types = len(W["E"]) if "E" in W else len(W["Tbl"]) // (P * n_buckets)
            cnt = [0.0] * n_types
            tot = [[0.0] * P for _ in range(n_types)]
            big = [[0.0] * P for _ in range(n_types)]
            for t in range(lens[b]):
                k = ids[b][t]
                for j in range(P):
                    l2 = math.log2(par[b][t][j])
                    tot[k][j] += l2
                    big[k][j] = l2 if cnt[k] == 0.0 else max(big[k][j], l2)
                cnt[k] += 1.0
            phi = cnt + [float(lens[b])]
            for k in range(n_types):
                phi += tot[k] + [v / cnt[k] if cnt[k] > 0 else 0.0 for v in tot[k]] + big[k]
        x = z + phi + list(hw[s])
        if "Tf" in W:      # tree ensemble (S27), comparisons in float32
            nodes = len(W["Tf"][0])
            tot = W["Tb"][0]
            for tf, tt, tv in zip(W["Tf"], W["Tt"], W["Tv"]):
                node = 0
                while node < nodes:
                    node = 2 * node + (1 if np.float32(x[int(tf[node])]) < np.float32(tt[node]) else 2)
                tot += tv[node - nodes]
            out.append(tot)
            continue
        nl = _n_scorer_layers(w)
        for i in range(nl):
            x = [ui + bi for ui, bi in zip(mv(W[f"Ws{i}"], x), W[f"bs{i}"])]
            if i + 1 < nl:
                x = [gelu1(ui) for ui in x]
        out.append(x[0])
    return np.array(out, dtype=F64)


def topk_segments(scores, subgraph_offsets, k: int) -> np.ndarray:
    """idx_out [S,k] int32: per segment the first min(k,n_s) candidates of the order (score desc, index asc),
    global indices, -1 fill (S16).  -0.0 == +0.0; NaN ranks below every number (ties by index)."""
    sc = np.asarray(scores)
    off = [int(x) for x in subgraph_offsets]
    S = len(off) - 1
    out = np.full((S, k), -1, dtype=np.int32)
    for s in range(S):
        items = []
        for i in range(off[s], off[s + 1]):
            v = float(sc[i])
            key = (1, 0.0) if math.isnan(v) else (0, -(v + 0.0))
            items.append((key, i))
        items.sort()
        for j, (_, i) in enumerate(items[:k]):
            out[s, j] = i
    return out


# ----------------------------------------------------------------------------- metrics (S15)

def score_error(y_gpu, y_ref, subgraph_offsets) -> float:
    """max_b |y - yref| / max(|yref|, RMS_s(yref))  (S15: relative error with a per-subgraph RMS floor)."""
    y_gpu = np.asarray(y_gpu, F64)
    y_ref = np.asarray(y_ref, F64)
    if y_ref.size == 0:
        return 0.0
    floor = np.zeros_like(y_ref)
    if subgraph_offsets is None:
        floor[:] = math.sqrt(float(np.mean(y_ref ** 2)))
    else:
        off = [int(x) for x in subgraph_offsets]
        for s in range(len(off) - 1):
            seg = y_ref[off[s]:off[s + 1]]
            if seg.size:
                floor[off[s]:off[s + 1]] = math.sqrt(float(np.mean(seg ** 2)))
    den = np.maximum(np.abs(y_ref), floor)
    den = np.where(den == 0.0, 1.0, den)
    return float(np.max(np.abs(y_gpu - y_ref) / den))


def topk_overlap(idx_a, idx_b) -> Tuple[float, float]:
    """(mean, min) over segments of |A ∩ B| / |B valid|  (S15)."""
    vals = []
    for ra, rb in zip(np.asarray(idx_a), np.asarray(idx_b)):
        sb = set(int(x) for x in rb if x >= 0)
        if not sb:
            continue
        sa = set(int(x) for x in ra if x >= 0)
        vals.append(len(sa & sb) / len(sb))
    if not vals:
        return 1.0, 1.0
    return float(np.mean(vals)), float(np.min(vals))


# ----------------------------------------------------------------------------- weight file (own reader)

def read_weight_file(path: str):
    """Independent reader of the WMW1 format (include/wm.h). Returns (header dict, weights dict)."""
    with open(path, "rb") as f:
        raw = f.read()
    if raw[:4] != b"WMW1":
        raise ValueError("bad magic")
    vals = struct.unpack_from("<12I6If", raw, 4)
    (version, kind, dtype, embed, d, d_a, hidden, n_types, P, n_buckets, H, n_lin) = vals[:12]
    widths = [x for x in vals[12:18]][: max(n_lin - 1, 0)]
    eps = vals[18]
    hdr = dict(version=version, kind=kind, dtype=dtype, embed=embed, d=d, d_a=d_a, hidden=hidden,
               n_types=n_types, P=P, n_buckets=n_buckets, H=H, n_scorer_layers=n_lin,
               scorer_widths=widths, ln_eps=eps)
    pos = 4 + struct.calcsize("<12I6If")
    hdr["phi_kind"] = PHI_MEAN
    if version >= 2:      # version 2 = version 1 + uint32 phi_kind
        hdr["phi_kind"] = struct.unpack_from("<I", raw, pos)[0]
        pos += 4
    hdr.update(ranker_kind=0, n_trees=0, tree_depth=0)
    if version == 3:      # version 3 = version 2 + uint32 ranker_kind, n_trees, tree_depth
        hdr["ranker_kind"], hdr["n_trees"], hdr["tree_depth"] = struct.unpack_from("<3I", raw, pos)
        pos += 12
    phi_dim = {PHI_MEAN: d_a, PHI_STRUCT: n_types + 1 + 3 * P, PHI_TYPED: n_types + 1 + 3 * n_types * P}[hdr["phi_kind"]]
    w = {}

    def take(name, *shape):
        nonlocal pos
        n = int(np.prod(shape))
        w[name] = np.frombuffer(raw, dtype="<f4", count=n, offset=pos).reshape(shape).copy()
        pos += 4 * n

    if embed == EMBED_LINEAR:
        take("E", n_types, d_a); take("W_p", d_a, P); take("b_p", d_a)
    else:
        take("Tbl", n_types * P * n_buckets, d_a)
    if kind in (KIND_MLP, KIND_MLP_LN):
        take("W1", hidden, d + d_a); take("b1", hidden); take("W2", d, hidden); take("b2", d)
        if kind == KIND_MLP_LN:
            take("gamma", d); take("beta", d)
    elif kind == KIND_TRANSH:
        take("W_w", d, d_a); take("W_d", d, d_a)
        take("W1", hidden, d + d_a); take("b1", hidden); take("W2", d, hidden); take("b2", d)
    else:
        take("W_g", d, d + d_a); take("W_r", d, d + d_a); take("W_h", d, d + d_a)
    if hdr["ranker_kind"] == 1:
        nodes = 2 ** hdr["tree_depth"] - 1
        take("Tf", hdr["n_trees"], nodes); take("Tt", hdr["n_trees"], nodes); take("Tv", hdr["n_trees"], nodes + 1)
        take("Tb", 1)
    dims = [d + phi_dim + H] + widths + [1]
    for i in range(n_lin):
        take(f"Ws{i}", dims[i + 1], dims[i]); take(f"bs{i}", dims[i + 1])
    if pos != len(raw):
        raise ValueError("trailing bytes in weight file")
    return hdr, w

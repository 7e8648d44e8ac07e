"""Pins for the float64 oracle (P14-P18 for the NEXT rows f1-f3).  CPU only.

Each pin checks the oracle against something other than itself: hand-expanded fixtures under
tests/golden/, closed forms, torch float64 library routines, brute force (scalar loops) and the
invariants BASELINE.json's north_star lists.
"""
import math

import numpy as np
import pytest
import torch

import gen
import oracle
from gen.configs import (WMConfig, KIND_MLP, KIND_MLP_LN, KIND_GRU, KIND_TRANSH, DTYPE_FP32, EMBED_LINEAR,
                         EMBED_BUCKET, PHI_MEAN, PHI_STRUCT)


def tiny_cfg(kind=KIND_MLP_LN, embed=EMBED_LINEAR, S=3, n=7, T=5, d=6, da=4, hid=8, H=3, widths=(5, 4),
             number=9, len_lo=0, phi_kind=PHI_MEAN):
    return WMConfig("tiny", number, kind, DTYPE_FP32, embed, S=S, per_subgraph=n, T_max=T,
                    len_dist="uniform", len_lo=len_lo, len_hi=T, n_types=5, P=3,
                    param_dist="loguniform", param_hi=1024, n_buckets=40 if embed == EMBED_BUCKET else 0,
                    d=d, d_a=da, hidden=0 if kind == KIND_GRU else hid, H=H, scorer_widths=widths, k=3,
                    phi_kind=phi_kind)


def run_vec(cfg, w, b, **kw):
    return oracle.rollout_score_vec(w, b.init_states, b.action_ids, b.action_params, b.lengths, b.hw_feats,
                                    b.subgraph_offsets, n_buckets=cfg.n_buckets, ln_eps=cfg.ln_eps,
                                    phi_kind=cfg.phi_kind, **kw)


ALL_KINDS = [(KIND_MLP, EMBED_LINEAR), (KIND_MLP_LN, EMBED_LINEAR), (KIND_GRU, EMBED_BUCKET),
             (KIND_GRU, EMBED_LINEAR), (KIND_MLP_LN, EMBED_BUCKET), (KIND_TRANSH, EMBED_LINEAR)]


# ---- P4 / P5 / P6 / P11: hand-expanded fixtures ---------------------------------------------------

def test_p4_mlp_step_hand_expanded(golden):
    g = golden("p4_mlp_step.txt")
    z = np.array([[1.0, 2.0]]); a = np.array([[3.0]])
    W1 = [[1, 0, -1], [2, 1, 0]]; b1 = [0.5, -1.0]; W2 = [[1, 1], [0, 2]]; b2 = [0.25, -0.5]
    np.testing.assert_allclose(oracle.gelu(np.array(g["u"])), g["gelu"], rtol=0, atol=1e-15)
    np.testing.assert_allclose(oracle.step_mlp(z, a, W1, b1, W2, b2)[0], g["z_next"], rtol=0, atol=1e-14)
    out = oracle.step_mlp(z, a, W1, b1, W2, b2, gamma=np.ones(2), beta=np.zeros(2), eps=1e-5)[0]
    np.testing.assert_allclose(out, g["z_next_ln"], rtol=0, atol=1e-13)
    # a transposed W1 or a dropped bias must fail: sanity that the fixture discriminates
    bad = oracle.step_mlp(z, a, W1, [0.0, 0.0], W2, b2)[0]
    assert np.abs(bad - np.array(g["z_next"])).max() > 1e-2


def test_p5_layernorm_closed_form(golden):
    g = golden("p5_layernorm.txt")
    x = np.array([1.0, 2.0, 3.0, 4.0])
    np.testing.assert_allclose(oracle.layer_norm(x, 1.0, 0.0, 0.0), g["eps0"], rtol=0, atol=1e-15)
    np.testing.assert_allclose(oracle.layer_norm(x, 1.0, 0.0, 1e-5), g["eps1e-5"], rtol=0, atol=1e-15)


def test_p6_gru_step_hand_expanded(golden):
    g = golden("p6_gru_step.txt")
    z = np.array([[1.0, -2.0]]); a = np.array([[0.5]])
    W_g = [[1, 0, 2], [0, 1, -2]]; W_r = [[0, 1, 0], [1, 0, 0]]; W_h = [[1, 1, 1], [1, -1, 2]]
    np.testing.assert_allclose(oracle.step_gru(z, a, W_g, W_r, W_h)[0], g["z_next"], rtol=0, atol=1e-14)


def test_p14_transh_step_hand_expanded(golden):
    g = golden("p14_transh_step.txt")
    z = np.array([[3.0, 4.0]]); a = np.array([[2.0]])
    Ww = [[1.0], [0.0]]; Wd = [[0.5], [-1.0]]
    W1 = [[1, 0, -1.25], [2, 1, -0.5]]; b1 = [0.0, 0.0]; W2 = [[1, 1], [0, 2]]; b2 = [0.25, -0.5]
    out = oracle.step_transh(z, a, Ww, Wd, W1, b1, W2, b2)[0]
    np.testing.assert_allclose(out, g["z_next"], rtol=0, atol=1e-14)
    # the fixture discriminates: no projection, no translation, a transposed W2 or no normalisation must each fail
    assert np.abs(oracle.step_transh(z, a, [[0.0], [1.0]], Wd, W1, b1, W2, b2)[0] - g["z_next"]).max() > 1e-2
    assert np.abs(oracle.step_transh(z, a, Ww, [[0.0], [0.0]], W1, b1, W2, b2)[0] - g["z_next"]).max() > 1e-2
    assert np.abs(oracle.step_transh(z, a, Ww, Wd, W1, b1, np.array(W2).T, b2)[0] - g["z_next"]).max() > 1e-2
    assert abs(np.linalg.norm(g["v"]) - 1.0) > 1.0


def test_p15_transh_closed_forms():
    rng = np.random.default_rng(15)
    d, da, hid, n = 7, 3, 5, 6
    z = rng.standard_normal((n, d)); a = rng.standard_normal((n, da))
    Ww = rng.standard_normal((d, da)); Wd = rng.standard_normal((d, da))
    W1 = rng.standard_normal((hid, d + da)); b1 = rng.standard_normal(hid)
    W2 = rng.standard_normal((d, hid)); b2 = rng.standard_normal(d)
    Z0 = np.zeros_like
    # (a) the result is always a unit vector ("finally normalized")
    np.testing.assert_allclose(np.linalg.norm(oracle.step_transh(z, a, Ww, Wd, W1, b1, W2, b2), axis=1), 1.0, atol=1e-12)
    # (b) no translation, no MLP: z' is the normalised projection onto the hyperplane, orthogonal to its normal
    zp = oracle.step_transh(z, a, Ww, Z0(Wd), W1, b1, Z0(W2), Z0(b2))
    np.testing.assert_allclose(np.sum(zp * (a @ Ww.T), axis=1), 0.0, atol=1e-12)
    # ... and equals (I - w w^T) z / |.| computed with a projection matrix (library linear algebra)
    for i in range(n):
        w = Ww @ a[i]; w = w / np.linalg.norm(w)
        ref = (np.eye(d) - np.outer(w, w)) @ z[i]
        np.testing.assert_allclose(zp[i], ref / np.linalg.norm(ref), atol=1e-11)
    # (c) the projection is idempotent: the same action again leaves the (unit, in-plane) state unchanged
    np.testing.assert_allclose(oracle.step_transh(zp, a, Ww, Z0(Wd), W1, b1, Z0(W2), Z0(b2)), zp, atol=1e-11)
    # (d) TransH proper: without the MLP, v = z_perp + d_r (Wang et al.: h_perp + d_r), up to the final normalisation
    v = oracle.step_transh(z, a, Ww, Wd, W1, b1, Z0(W2), Z0(b2))
    for i in range(n):
        w = Ww @ a[i]; w = w / np.linalg.norm(w)
        ref = z[i] - (w @ z[i]) * w + Wd @ a[i]
        np.testing.assert_allclose(v[i], ref / np.linalg.norm(ref), atol=1e-11)
    # (e) a state already orthogonal to the normal is only normalised
    zo = z - np.sum(z * (a @ Ww.T), axis=1, keepdims=True) * (a @ Ww.T) / np.sum((a @ Ww.T) ** 2, axis=1, keepdims=True)
    np.testing.assert_allclose(oracle.step_transh(zo, a, Ww, Z0(Wd), W1, b1, Z0(W2), Z0(b2)),
                               zo / np.linalg.norm(zo, axis=1, keepdims=True), atol=1e-11)
    # (f) library cross-check of the full step with torch float64 (gelu, normalize)
    zt, at = torch.from_numpy(z), torch.from_numpy(a)
    u = at @ torch.from_numpy(Ww).T
    wt = torch.nn.functional.normalize(u, dim=1, eps=0.0)
    xt = zt - (wt * zt).sum(1, keepdim=True) * wt + at @ torch.from_numpy(Wd).T
    ht = torch.nn.functional.gelu(torch.cat([xt, at], 1) @ torch.from_numpy(W1).T + torch.from_numpy(b1))
    vt = xt + ht @ torch.from_numpy(W2).T + torch.from_numpy(b2)
    np.testing.assert_allclose(oracle.step_transh(z, a, Ww, Wd, W1, b1, W2, b2),
                               torch.nn.functional.normalize(vt, dim=1, eps=0.0).numpy(), atol=1e-11)


# ---- P16 / P17: structured action features (NEXT row f2, S25) -----------------------

def test_p16_phi_struct_hand_worked(golden):
    g = golden("p16_phi_struct.txt")
    ids = [2, 0, 2]; par = [[1, 8], [4, 2], [16, 8]]
    np.testing.assert_allclose(oracle.phi_struct(ids, par, 4), g["phi"], rtol=0, atol=1e-15)
    np.testing.assert_allclose(oracle.phi_struct(ids[:1], par[:1], 4), g["phi_prefix1"], rtol=0, atol=0)
    np.testing.assert_allclose(oracle.phi_struct([], np.zeros((0, 2), dtype=np.int32), 4), g["phi_empty"], rtol=0, atol=0)
    # the fixture discriminates: swapping the parameter slots or the type ids must change the vector
    assert np.abs(oracle.phi_struct(ids, [q[::-1] for q in par], 4) - np.array(g["phi"])).max() >= 1.0
    assert np.abs(oracle.phi_struct([0, 2, 0], par, 4) - np.array(g["phi"])).max() >= 1.0


def test_p22_phi_typed_hand_worked(golden):
    """NEXT row f2 as SURVEY.md words it: per-TYPE numeric statistics (S28)."""
    g = golden("p22_phi_typed.txt")
    ids = [1, 0, 1]; par = [[2, 8], [4, 1], [16, 2]]
    np.testing.assert_allclose(oracle.phi_struct_typed(ids, par, 3), g["phi"], rtol=0, atol=0)
    np.testing.assert_allclose(oracle.phi_struct_typed(ids[:1], par[:1], 3), g["phi_prefix1"], rtol=0, atol=0)
    np.testing.assert_allclose(oracle.phi_struct_typed([], np.zeros((0, 2), dtype=np.int32), 3), g["phi_empty"], rtol=0, atol=0)
    # the fixture discriminates: swapped parameter slots, swapped type ids, a statistic pooled over types
    assert np.abs(oracle.phi_struct_typed(ids, [q[::-1] for q in par], 3) - np.array(g["phi"])).max() >= 1.0
    assert np.abs(oracle.phi_struct_typed([0, 1, 0], par, 3) - np.array(g["phi"])).max() >= 1.0
    assert len(g["phi"]) == 3 + 1 + 3 * 3 * 2


def test_p23_phi_typed_closed_forms_and_placement():
    """Closed forms that tie phi_struct_typed to the (pinned) pooled phi_struct and to plain numpy, and its placement in
    the ranker's input [z_T ; phi ; h] through the scalar and vector rollouts."""
    rng = np.random.default_rng(23)
    NT, P, n = 5, 3, 17
    ids = rng.integers(0, NT, n); par = rng.integers(1, 200, (n, P))
    t = oracle.phi_struct_typed(ids, par, NT)
    s = oracle.phi_struct(ids, par, NT)
    lp = np.log2(par.astype(np.float64))
    blocks = t[NT + 1:].reshape(NT, 3, P)
    np.testing.assert_array_equal(t[:NT + 1], s[:NT + 1])                                 # counts and length are the same
    np.testing.assert_allclose(blocks[:, 0].sum(axis=0), s[NT + 1:NT + 1 + P], rtol=1e-14)   # per-type sums add up to the pooled sums
    np.testing.assert_allclose((t[:NT, None] * blocks[:, 1]).sum(axis=0), s[NT + 1:NT + 1 + P], rtol=1e-14)   # sum_k c_k m_k = pooled sum
    np.testing.assert_array_equal(blocks[:, 2].max(axis=0), s[NT + 1 + 2 * P:])             # max over types of per-type maxima
    for k in range(NT):                                                                     # each block against numpy on the type's rows
        rows = lp[ids == k]
        want = np.concatenate([rows.sum(0), rows.mean(0), rows.max(0)]) if len(rows) else np.zeros(3 * P)
        np.testing.assert_allclose(blocks[k].reshape(-1), want, rtol=1e-14, atol=0)
    # a sequence of ONE type: that type's block is the pooled statistics, every other block is zero
    one = np.full(n, 3)
    t1 = oracle.phi_struct_typed(one, par, NT); s1 = oracle.phi_struct(one, par, NT)
    np.testing.assert_allclose(t1[NT + 1:].reshape(NT, 3 * P)[3], s1[NT + 1:], rtol=1e-14)
    assert np.count_nonzero(np.delete(t1[NT + 1:].reshape(NT, 3 * P), 3, axis=0)) == 0
    # order of the steps does not matter; concatenating sequences adds counts and sums
    perm = rng.permutation(n)
    np.testing.assert_allclose(oracle.phi_struct_typed(ids[perm], par[perm], NT), t, rtol=1e-14)
    a, b = oracle.phi_struct_typed(ids[:7], par[:7], NT), oracle.phi_struct_typed(ids[7:], par[7:], NT)
    np.testing.assert_allclose(a[:NT + 1] + b[:NT + 1], t[:NT + 1])
    np.testing.assert_allclose(a[NT + 1:].reshape(NT, 3, P)[:, 0] + b[NT + 1:].reshape(NT, 3, P)[:, 0], blocks[:, 0], rtol=1e-14)
    # placement: a one-linear ranker with a unit weight on one input reads exactly that feature, vector == scalar rollout
    cfg = WMConfig(**{**gen.get_config(13).__dict__, "d": 6, "d_a": 4, "hidden": 8, "scorer_widths": (), "S": 2,
                      "per_subgraph": 5, "n_types": 3, "P": 2})
    w = gen.make_weights(cfg); bt = gen.make_inputs(cfg)
    F = cfg.phi_dim
    assert F == 3 + 1 + 18 and w["Ws0"].shape == (1, cfg.d + F + cfg.H)
    for col in (0, 2, 3, 4, 9, 10, F - 1):
        w1 = dict(w); w1["Ws0"] = np.zeros_like(w["Ws0"]); w1["Ws0"][0, cfg.d + col] = 1.0; w1["bs0"] = np.zeros_like(w["bs0"])
        kw = dict(phi_kind=cfg.phi_kind)
        yv = oracle.rollout_score_vec(w1, bt.init_states, bt.action_ids, bt.action_params, bt.lengths, bt.hw_feats, bt.subgraph_offsets, **kw)
        ys = oracle.rollout_score_scalar(w1, bt.init_states, bt.action_ids, bt.action_params, bt.lengths, bt.hw_feats, bt.subgraph_offsets, **kw)
        want = [oracle.phi_struct_typed(bt.action_ids[i, :bt.lengths[i]], bt.action_params[i, :bt.lengths[i]], 3)[col] for i in range(bt.B)]
        np.testing.assert_allclose(yv, want, rtol=1e-14, atol=0)
        np.testing.assert_allclose(ys, want, rtol=1e-13, atol=1e-13)


def test_p17_phi_struct_closed_forms_and_placement():
    rng = np.random.default_rng(17)
    nt, P, n = 7, 3, 11
    ids = rng.integers(0, nt, n); par = rng.integers(1, 1025, (n, P))
    f = oracle.phi_struct(ids, par, nt)
    c, ln, s, m, x = f[:nt], f[nt], f[nt + 1:nt + 1 + P], f[nt + 1 + P:nt + 1 + 2 * P], f[nt + 1 + 2 * P:]
    assert f.shape == (nt + 1 + 3 * P,) and ln == n and c.sum() == n
    np.testing.assert_array_equal(c, np.bincount(ids, minlength=nt))
    # sum of log2 = log2 of the product (exact integers in python), mean = sum / len, max = log2 of the largest
    for j in range(P):
        prod = 1
        for v in par[:, j]:
            prod *= int(v)
        assert abs(s[j] - math.log2(prod)) < 1e-11
        assert abs(m[j] - math.log2(prod) / n) < 1e-12
        assert x[j] == math.log2(int(par[:, j].max()))
    # order of the steps does not matter; concatenation adds counts, lengths and sums and takes the larger maximum
    perm = rng.permutation(n)
    np.testing.assert_allclose(oracle.phi_struct(ids[perm], par[perm], nt), f, rtol=0, atol=1e-12)
    fa, fb = oracle.phi_struct(ids[:4], par[:4], nt), oracle.phi_struct(ids[4:], par[4:], nt)
    np.testing.assert_allclose(fa[:nt + 1 + P] + fb[:nt + 1 + P], f[:nt + 1 + P], rtol=0, atol=1e-12)
    np.testing.assert_array_equal(np.maximum(fa[nt + 1 + 2 * P:], fb[nt + 1 + 2 * P:]), x)
    # constant parameters 2^q: sum = q len, mean = max = q; all-ones parameters: every numeric attribute 0
    fq = oracle.phi_struct(ids, np.full((n, P), 32), nt)
    np.testing.assert_array_equal(fq[nt + 1:], [5.0 * n] * P + [5.0] * P + [5.0] * P)
    assert not oracle.phi_struct(ids, np.ones((n, P), dtype=int), nt)[nt + 1:].any()
    # placement in the ranker input [z_T ; phi ; h] (Eq.12): a one-linear scorer whose weight row is a unit vector
    # returns exactly that feature of each candidate
    cfg = tiny_cfg(KIND_MLP, EMBED_LINEAR, widths=(), phi_kind=PHI_STRUCT)
    w = gen.make_weights(cfg); b = gen.make_inputs(cfg)
    F = cfg.phi_dim
    assert w["Ws0"].shape == (1, cfg.d + F + cfg.H)
    for col in (0, 2, cfg.n_types, cfg.n_types + 1, F - 1):
        w1 = dict(w); w1["Ws0"] = np.zeros_like(w["Ws0"]); w1["Ws0"][0, cfg.d + col] = 1.0
        w1["bs0"] = np.zeros_like(w["bs0"])
        want = [oracle.phi_struct(b.action_ids[i, :b.lengths[i]], b.action_params[i, :b.lengths[i]], cfg.n_types)[col]
                for i in range(b.B)]
        np.testing.assert_allclose(run_vec(cfg, w1, b), want, rtol=0, atol=1e-13)
    w1 = dict(w); w1["Ws0"] = np.zeros_like(w["Ws0"]); w1["Ws0"][0, cfg.d + F] = 1.0; w1["bs0"] = np.zeros_like(w["bs0"])
    seg = np.repeat(np.arange(cfg.S), cfg.per_subgraph)
    np.testing.assert_allclose(run_vec(cfg, w1, b), b.hw_feats[seg, 0].astype(np.float64), rtol=0, atol=0)


@pytest.mark.parametrize("kind,embed", [(KIND_MLP, EMBED_LINEAR), (KIND_GRU, EMBED_BUCKET)])
def test_p9_scalar_vs_vector_struct_phi(kind, embed):
    cfg = tiny_cfg(kind, embed, phi_kind=PHI_STRUCT)
    w = gen.make_weights(cfg); b = gen.make_inputs(cfg)
    ys = oracle.rollout_score_scalar(w, b.init_states, b.action_ids, b.action_params, b.lengths, b.hw_feats,
                                     b.subgraph_offsets, n_buckets=cfg.n_buckets, ln_eps=cfg.ln_eps,
                                     phi_kind=PHI_STRUCT)
    np.testing.assert_allclose(run_vec(cfg, w, b), ys, rtol=0, atol=1e-12)
    # zero-length candidates see phi = 0: their score is G([z_0 ; 0 ; h])
    z = np.where(b.lengths == 0)[0]
    assert z.size > 0
    seg = np.repeat(np.arange(cfg.S), cfg.per_subgraph)
    x0 = np.concatenate([b.init_states[seg[z]], np.zeros((z.size, cfg.phi_dim)), b.hw_feats[seg[z]]], axis=1)
    np.testing.assert_allclose(run_vec(cfg, w, b)[z], oracle.scorer(x0, w, len(cfg.scorer_widths) + 1), rtol=0,
                               atol=1e-12)


def test_p11_bucket_function(golden):
    g = golden("p11_buckets.txt")
    for p, bk in g.items():
        assert oracle.bucket_index(int(p), 40) == int(bk[0])
    # integer formula equals floor(4*log2 p) wherever floating point is unambiguous, for all p in 1..1024
    for p in range(1, 1025):
        x = 4 * math.log2(p)
        if abs(x - round(x)) > 1e-9:
            assert oracle.bucket_index(p, 40) == min(39, math.floor(x))
        else:
            assert oracle.bucket_index(p, 40) == min(39, round(x))
    ps = np.arange(1, 1025).reshape(-1, 1)
    vec = oracle.wm_oracle._bucket_vec(ps, 40)[:, 0]
    assert all(int(vec[i]) == oracle.bucket_index(i + 1, 40) for i in range(1024))
    # the whole int32 range and more buckets than 64 (a loader-accepted n_buckets goes up to 4096): the quarter-octave
    # boundaries are the integers ceil(2^(b/4)); one below, at and one above each of them, plus random parameters
    edges = []
    for b in range(0, 124):
        r = math.isqrt(math.isqrt(1 << b))           # floor(2^(b/4))
        edges += [v for v in (r - 1, r, r + 1, r + 2) if 1 <= v <= 2**31 - 1]
    rng = np.random.default_rng(11)
    big = np.concatenate([np.array(edges, dtype=np.int64), rng.integers(1, 2**31, size=4000), [2**16 - 1, 2**16, 2**31 - 1]])
    vec = oracle.wm_oracle._bucket_vec(big.reshape(-1, 1), 4096)[:, 0]
    for v, got in zip(big, vec):
        want = (int(v) ** 4).bit_length() - 1
        assert int(got) == want == oracle.bucket_index(int(v), 4096), v
        assert 2 ** want <= int(v) ** 4 < 2 ** (want + 1)           # i.e. want = floor(4 log2 v), no floating point
    assert oracle.bucket_index(2**16, 4096) == 64 and oracle.bucket_index(2**31 - 1, 4096) == 123


# ---- P1 / P2 / P3 / P13: invariants -----------------------------------------------------------------

@pytest.mark.parametrize("kind,embed", ALL_KINDS)
def test_p1_zero_length_returns_initial_state(kind, embed):
    cfg = tiny_cfg(kind, embed)
    w = gen.make_weights(cfg); b = gen.make_inputs(cfg)
    b.lengths[:] = 0
    y, lat = run_vec(cfg, w, b, return_latent=True)
    seg = np.repeat(np.arange(cfg.S), cfg.per_subgraph)
    np.testing.assert_array_equal(lat, b.init_states[seg].astype(np.float64))
    x = np.concatenate([b.init_states[seg], np.zeros((cfg.B, cfg.d_a)), b.hw_feats[seg]], -1).astype(np.float64)
    np.testing.assert_allclose(y, oracle.scorer(x, w, len(cfg.scorer_widths) + 1), rtol=0, atol=0)


@pytest.mark.parametrize("kind,embed", ALL_KINDS)
def test_p2_padding_invariance(kind, embed):
    cfg = tiny_cfg(kind, embed)
    w = gen.make_weights(cfg); b = gen.make_inputs(cfg, sentinel_padding=True)
    y1 = run_vec(cfg, w, b)
    b2 = gen.make_inputs(cfg, sentinel_padding=False)       # padding holds ordinary random draws instead
    assert (b2.action_ids != b.action_ids).any()
    y2 = run_vec(cfg, w, b2)
    np.testing.assert_array_equal(y1, y2)                  # bit-identical


@pytest.mark.parametrize("kind,embed", ALL_KINDS)
def test_p3_permutation_equivariance_and_subgraph_move(kind, embed):
    cfg = tiny_cfg(kind, embed)
    w = gen.make_weights(cfg); b = gen.make_inputs(cfg)
    y = run_vec(cfg, w, b)
    rng = np.random.default_rng(5)
    n = cfg.per_subgraph
    perm = np.concatenate([s * n + rng.permutation(n) for s in range(cfg.S)])
    yp = oracle.rollout_score_vec(w, b.init_states, b.action_ids[perm], b.action_params[perm], b.lengths[perm],
                                  b.hw_feats, b.subgraph_offsets, n_buckets=cfg.n_buckets)
    np.testing.assert_allclose(yp, y[perm], rtol=0, atol=1e-13)
    # two subgraphs with equal z0/hw: a candidate scores the same in either
    z0 = b.init_states.copy(); hw = b.hw_feats.copy()
    z0[1] = z0[0]; hw[1] = hw[0]
    ids = b.action_ids.copy(); par = b.action_params.copy(); ln = b.lengths.copy()
    ids[n] = ids[0]; par[n] = par[0]; ln[n] = ln[0]
    ym = oracle.rollout_score_vec(w, z0, ids, par, ln, hw, b.subgraph_offsets, n_buckets=cfg.n_buckets)
    assert abs(ym[n] - ym[0]) < 1e-13


@pytest.mark.parametrize("kind,embed", ALL_KINDS)
def test_p13_batch_independence_and_per_candidate_mode(kind, embed):
    cfg = tiny_cfg(kind, embed)
    w = gen.make_weights(cfg); b = gen.make_inputs(cfg)
    y = run_vec(cfg, w, b)
    seg = np.repeat(np.arange(cfg.S), cfg.per_subgraph)
    for i in (0, 5, cfg.B - 1):
        yi = oracle.rollout_score_vec(w, b.init_states[seg[i]][None], b.action_ids[i:i + 1],
                                      b.action_params[i:i + 1], b.lengths[i:i + 1], b.hw_feats[seg[i]][None],
                                      np.array([0, 1]), n_buckets=cfg.n_buckets)
        assert abs(yi[0] - y[i]) < 1e-13
    ypc = oracle.rollout_score_vec(w, b.init_states[seg], b.action_ids, b.action_params, b.lengths,
                                   b.hw_feats[seg], None, n_buckets=cfg.n_buckets)
    np.testing.assert_allclose(ypc, y, rtol=0, atol=1e-13)


# ---- P7: closed forms ---------------------------------------------------------------------------------

def test_p7_closed_forms():
    cfg = tiny_cfg(KIND_MLP, len_lo=1)
    b = gen.make_inputs(cfg)
    seg = np.repeat(np.arange(cfg.S), cfg.per_subgraph)
    z0 = b.init_states[seg].astype(np.float64)
    # (a) W1 = 0, no LN: z_T = z_0 + T (W2 gelu(b1) + b2)
    w = gen.make_weights(cfg); w["W1"] = np.zeros_like(w["W1"])
    _, lat = run_vec(cfg, w, b, return_latent=True)
    inc = w["W2"].astype(np.float64) @ oracle.gelu(w["b1"].astype(np.float64)) + w["b2"]
    np.testing.assert_allclose(lat, z0 + b.lengths[:, None] * inc[None, :], rtol=0, atol=1e-12)
    # (b) W2 = 0, b2 = 0, no LN: z_T = z_0
    w = gen.make_weights(cfg); w["W2"] = np.zeros_like(w["W2"]); w["b2"] = np.zeros_like(w["b2"])
    _, lat = run_vec(cfg, w, b, return_latent=True)
    np.testing.assert_array_equal(lat, z0)
    # (c) same with LN, gamma=1, beta=0, eps=0: z_T = LN(z_0) for any T >= 1 (idempotent)
    cfg2 = tiny_cfg(KIND_MLP_LN, len_lo=1)
    w = gen.make_weights(cfg2); w["W2"] = np.zeros_like(w["W2"]); w["b2"] = np.zeros_like(w["b2"])
    w["gamma"] = np.ones_like(w["gamma"]); w["beta"] = np.zeros_like(w["beta"])
    b2 = gen.make_inputs(cfg2)
    lat = oracle.rollout_score_vec(w, b2.init_states, b2.action_ids, b2.action_params, b2.lengths, b2.hw_feats,
                                   b2.subgraph_offsets, ln_eps=0.0, return_latent=True)[1]
    z0b = b2.init_states[seg].astype(np.float64)
    ref = (z0b - z0b.mean(-1, keepdims=True)) / z0b.std(-1, keepdims=True)
    np.testing.assert_allclose(lat, ref, rtol=0, atol=1e-12)
    # (d) GRU, all weights 0: g = 1/2, h = 0 => z_T = z_0 / 2^T
    cfg3 = tiny_cfg(KIND_GRU, EMBED_BUCKET, len_lo=1)
    w = gen.make_weights(cfg3)
    for nme in ("W_g", "W_r", "W_h"):
        w[nme] = np.zeros_like(w[nme])
    b3 = gen.make_inputs(cfg3)
    _, lat = run_vec(cfg3, w, b3, return_latent=True)
    z0c = b3.init_states[seg].astype(np.float64)
    np.testing.assert_allclose(lat, z0c / (2.0 ** b3.lengths)[:, None], rtol=0, atol=1e-15)
    # (e) GRU, W_h = 0: one step is (1-g) z
    w = gen.make_weights(cfg3); w["W_h"] = np.zeros_like(w["W_h"])
    z = np.array([[0.3, -1.2, 0.5, 2.0, -0.1, 0.7]]); a = np.array([[1.0, -1.0, 0.5, 0.25]])
    g = 1 / (1 + np.exp(-(np.concatenate([z, a], -1) @ w["W_g"].astype(np.float64).T)))
    np.testing.assert_allclose(oracle.step_gru(z, a, w["W_g"], w["W_r"], w["W_h"]), (1 - g) * z, atol=1e-15)


# ---- P8: library cross-checks (torch float64 CPU) ---------------------------------------------------------

def test_p8_library_cross_checks():
    rng = np.random.default_rng(0)
    x = rng.standard_normal((37, 19)) * 3
    t = torch.from_numpy(x)
    np.testing.assert_allclose(oracle.gelu(x), torch.nn.functional.gelu(t, approximate="none").numpy(),
                               rtol=0, atol=1e-14)
    gam = rng.standard_normal(19); bet = rng.standard_normal(19)
    ref = torch.nn.functional.layer_norm(t, (19,), torch.from_numpy(gam), torch.from_numpy(bet), 1e-5).numpy()
    np.testing.assert_allclose(oracle.layer_norm(x, gam, bet, 1e-5), ref, rtol=0, atol=1e-13)
    # whole MLP+LN step and GRU step against torch linear algebra
    d, da, hid = 19, 7, 23
    z = rng.standard_normal((11, d)); a = rng.standard_normal((11, da))
    W1 = rng.standard_normal((hid, d + da)); b1 = rng.standard_normal(hid)
    W2 = rng.standard_normal((d, hid)); b2 = rng.standard_normal(d)
    tz, ta = torch.from_numpy(z), torch.from_numpy(a)
    F = torch.nn.functional
    tv = tz + F.linear(F.gelu(F.linear(torch.cat([tz, ta], -1), torch.from_numpy(W1), torch.from_numpy(b1))),
                       torch.from_numpy(W2), torch.from_numpy(b2))
    np.testing.assert_allclose(oracle.step_mlp(z, a, W1, b1, W2, b2), tv.numpy(), rtol=0, atol=1e-12)
    tln = F.layer_norm(tv, (d,), torch.from_numpy(gam), torch.from_numpy(bet), 1e-5)
    np.testing.assert_allclose(oracle.step_mlp(z, a, W1, b1, W2, b2, gam, bet, 1e-5), tln.numpy(), atol=1e-12)
    Wg, Wr, Wh = (rng.standard_normal((d, d + da)) for _ in range(3))
    x_ = torch.cat([tz, ta], -1)
    g = torch.sigmoid(F.linear(x_, torch.from_numpy(Wg))); r = torch.sigmoid(F.linear(x_, torch.from_numpy(Wr)))
    h = torch.tanh(F.linear(torch.cat([r * tz, ta], -1), torch.from_numpy(Wh)))
    np.testing.assert_allclose(oracle.step_gru(z, a, Wg, Wr, Wh), ((1 - g) * tz + g * h).numpy(), atol=1e-13)
    # embedding against torch.nn.functional.embedding + linear
    E = rng.standard_normal((5, da)); Wp = rng.standard_normal((da, 3)); bp = rng.standard_normal(da)
    ids = rng.integers(0, 5, 11); par = rng.integers(1, 1025, (11, 3))
    ref = F.embedding(torch.from_numpy(ids), torch.from_numpy(E)) + \
        F.linear(torch.log2(torch.from_numpy(par).double()), torch.from_numpy(Wp), torch.from_numpy(bp))
    np.testing.assert_allclose(oracle.embed_linear(ids, par, E, Wp, bp), ref.numpy(), atol=1e-13)
    # bucketed embedding against an embedding_bag-style torch gather
    Tbl = rng.standard_normal((5 * 3 * 40, da))
    bk = torch.clamp(torch.floor(4 * torch.log2(torch.from_numpy(par).double()) + 1e-9), max=39).long()
    idx = (torch.from_numpy(ids)[:, None] * 3 + torch.arange(3)[None]) * 40 + bk
    ref = F.embedding(idx, torch.from_numpy(Tbl)).sum(1)
    np.testing.assert_allclose(oracle.embed_bucket(ids, par, Tbl, 3, 40), ref.numpy(), atol=1e-13)


# ---- P9: brute force --------------------------------------------------------------------------------------

@pytest.mark.parametrize("kind,embed", ALL_KINDS)
def test_p9_scalar_vs_vector(kind, embed):
    cfg = tiny_cfg(kind, embed)
    w = gen.make_weights(cfg); b = gen.make_inputs(cfg)
    yv = run_vec(cfg, w, b)
    ys = oracle.rollout_score_scalar(w, b.init_states, b.action_ids, b.action_params, b.lengths, b.hw_feats,
                                     b.subgraph_offsets, n_buckets=cfg.n_buckets, ln_eps=cfg.ln_eps)
    np.testing.assert_allclose(yv, ys, rtol=0, atol=1e-12)


def test_p9_cfg1_scalar_vs_vector():
    cfg = gen.get_config(1)
    w = gen.make_weights(cfg); b = gen.make_inputs(cfg)
    yv = run_vec(cfg, w, b)
    ys = oracle.rollout_score_scalar(w, b.init_states, b.action_ids, b.action_params, b.lengths, b.hw_feats,
                                     b.subgraph_offsets)
    np.testing.assert_allclose(yv, ys, rtol=0, atol=1e-11)


# ---- P10: top-k -------------------------------------------------------------------------------------------

def test_p10_topk_matches_full_sort():
    rng = np.random.default_rng(3)
    sc = rng.integers(-3, 4, 50).astype(np.float32)           # many duplicates
    sc[7] = -0.0; sc[9] = 0.0; sc[11] = np.nan; sc[40] = np.nan; sc[13] = np.inf; sc[14] = -np.inf
    off = np.array([0, 0, 20, 23, 50], dtype=np.int32)         # empty, normal, n_s < k, normal
    k = 5
    out = oracle.topk_segments(sc, off, k)
    assert out.shape == (4, 5)
    assert (out[0] == -1).all()
    t = torch.from_numpy(sc.astype(np.float64))
    t = torch.where(torch.isnan(t), torch.full_like(t, -float("inf")), t)   # NaN lowest (after -inf by index)
    for s in range(1, 4):
        lo, hi = off[s], off[s + 1]
        seg = t[lo:hi]
        order = torch.sort(-seg, stable=True).indices.numpy() + lo           # stable => index asc on ties
        # -inf vs NaN: NaN must come after real -inf
        order = sorted(order, key=lambda i: (1 if math.isnan(sc[i]) else 0, -(t[i].item()), i))
        exp = list(order[:k]) + [-1] * max(0, k - (hi - lo))
        assert list(out[s]) == exp[:k]
    assert list(oracle.topk_segments(np.array([0.0, -0.0, 0.0], np.float32), [0, 3], 3)[0]) == [0, 1, 2]
    assert list(oracle.topk_segments(np.array([1.0, 1.0, 1.0, 1.0], np.float32), [0, 4], 2)[0]) == [0, 1]
    # against torch.topk where scores are distinct
    x = rng.standard_normal(200).astype(np.float32)
    ref = torch.topk(torch.from_numpy(x), 17).indices.numpy()
    assert list(oracle.topk_segments(x, [0, 200], 17)[0]) == list(ref)


# ---- P12: shared-prefix reuse equals from-scratch ---------------------------------------------------------------

def test_p12_prefix_reuse_equals_scratch():
    cfg = gen.get_config(4).scaled(S=1, per_subgraph=64)
    cfg = WMConfig(**{**cfg.__dict__, "d": 8, "d_a": 4, "hidden": 12, "H": 3, "scorer_widths": (6, 5)})
    w = gen.make_weights(cfg); b = gen.make_inputs(cfg)
    y = run_vec(cfg, w, b)
    # children 0..63 share parent 0's prefix up to their cut; roll the common prefix (min cut = 16) once
    c = 16
    assert (b.action_ids[:, :c] == b.action_ids[0, :c]).all()
    _, zc = oracle.rollout_score_vec(w, b.init_states, b.action_ids[:1, :c], b.action_params[:1, :c],
                                     np.array([c]), b.hw_feats, np.array([0, 1]), return_latent=True)
    # continue every child from the shared latent in per-candidate mode; phi needs the whole sequence, so
    # compare terminal latents (the quantity prefix reuse shares)
    _, lat_full = run_vec(cfg, w, b, return_latent=True)
    _, lat_sfx = oracle.rollout_score_vec(w, np.repeat(zc, 64, 0), b.action_ids[:, c:], b.action_params[:, c:],
                                          b.lengths - c, np.repeat(b.hw_feats, 64, 0), None, return_latent=True)
    np.testing.assert_allclose(lat_sfx, lat_full, rtol=0, atol=1e-12)
    assert np.isfinite(y).all()


@pytest.mark.parametrize("kind,embed,phi", [(KIND_MLP_LN, EMBED_LINEAR, PHI_MEAN), (KIND_GRU, EMBED_BUCKET, PHI_MEAN),
                                            (KIND_TRANSH, EMBED_LINEAR, PHI_MEAN), (KIND_MLP, EMBED_LINEAR, PHI_STRUCT)])
def test_p18_latents_and_score_from(kind, embed, phi):
    """NEXT row f3 (prefix-latent reuse).  rollout_latents / rollout_score_from are pinned to the already pinned literal
    path: (a) the latent after step t+1 is the terminal latent of the sequence cut to t+1 steps; (b) scoring from a
    banked latent at ANY cut (0 and len included) equals scoring from scratch; (c) start = len is the closed form
    G([bank row ; phi ; h]); (d) phi covers the whole sequence, not the suffix."""
    cfg = tiny_cfg(kind, embed, phi_kind=phi)
    w = gen.make_weights(cfg); b = gen.make_inputs(cfg)
    kw = dict(n_buckets=cfg.n_buckets, ln_eps=cfg.ln_eps)
    lat = oracle.rollout_latents(w, b.init_states, b.action_ids, b.action_params, b.lengths, b.subgraph_offsets, **kw)
    assert lat.shape == (b.B, cfg.T_max, cfg.d)
    valid = np.arange(cfg.T_max)[None, :] < b.lengths[:, None]
    assert np.isnan(lat[~valid]).all() and np.isfinite(lat[valid]).all()
    for t in range(cfg.T_max):                     # (a)
        cut = np.minimum(b.lengths, t + 1)
        _, zt = oracle.rollout_score_vec(w, b.init_states, b.action_ids, b.action_params, cut, b.hw_feats,
                                         b.subgraph_offsets, return_latent=True, phi_kind=phi, **kw)
        rows = b.lengths > t
        np.testing.assert_allclose(lat[rows, t], zt[rows], rtol=0, atol=1e-12)
    y = run_vec(cfg, w, b)
    seg = np.repeat(np.arange(cfg.S), cfg.per_subgraph)
    # bank = [z_0 of every subgraph ; every stored latent], bank_index by (candidate, cut)
    bank = np.concatenate([b.init_states.astype(np.float64), np.nan_to_num(lat).reshape(-1, cfg.d)])
    rng = np.random.default_rng(18)
    for starts in (np.zeros(b.B, dtype=np.int64), b.lengths.astype(np.int64),
                   rng.integers(0, cfg.T_max + 1, b.B), np.full(b.B, 99), np.full(b.B, -3)):
        st = np.clip(starts, 0, b.lengths)
        index = np.where(st == 0, seg, cfg.S + np.arange(b.B) * cfg.T_max + st - 1)
        yf = oracle.rollout_score_from(w, bank, index, starts, b.action_ids, b.action_params, b.lengths, b.hw_feats,
                                       b.subgraph_offsets, phi_kind=phi, **kw)
        np.testing.assert_allclose(yf, y, rtol=0, atol=1e-11)          # (b)
    # (c) nothing left to roll: the score is the ranker on the banked latent
    rb = rng.standard_normal((b.B, cfg.d))
    yc = oracle.rollout_score_from(w, rb, np.arange(b.B), b.lengths, b.action_ids, b.action_params, b.lengths,
                                   b.hw_feats, b.subgraph_offsets, phi_kind=phi, **kw)
    nl = len(cfg.scorer_widths) + 1
    if phi == PHI_STRUCT:
        ph = np.stack([oracle.phi_struct(b.action_ids[i, :b.lengths[i]], b.action_params[i, :b.lengths[i]], cfg.n_types)
                       for i in range(b.B)])
    else:
        ph = np.zeros((b.B, cfg.d_a))               # mean action embedding, from the (pinned) embedding functions
        for i in range(b.B):
            n = int(b.lengths[i])
            if n:
                emb = (oracle.embed_bucket(b.action_ids[i, :n], b.action_params[i, :n], w["Tbl"], cfg.P, cfg.n_buckets)
                       if embed == EMBED_BUCKET else
                       oracle.embed_linear(b.action_ids[i, :n], b.action_params[i, :n], w["E"], w["W_p"], w["b_p"]))
                ph[i] = emb.mean(axis=0)
    np.testing.assert_allclose(yc, oracle.scorer(np.concatenate([rb, ph, b.hw_feats[seg]], axis=1), w, nl),
                               rtol=0, atol=1e-12)
    # (d) scoring the suffix alone (phi over the suffix only) is a different number for cut > 0
    i = int(np.argmax(b.lengths))
    c = int(b.lengths[i]) // 2
    sub = oracle.rollout_score_vec(w, lat[i:i + 1, c - 1], b.action_ids[i:i + 1, c:], b.action_params[i:i + 1, c:],
                                   b.lengths[i:i + 1] - c, b.hw_feats[seg[i]][None], None, phi_kind=phi, **kw)
    assert abs(sub[0] - y[i]) > 1e-6


# ---- P19 / P20: tree-ensemble ranker (NEXT row f4, S27) ---------------------------------

def test_p19_forest_hand_worked(golden):
    g = golden("p19_forest.txt")
    Tf = [[0, 2, 1], [1, 2, 0]]; Tt = [[1.0, 2.0, 0.0], [-1.0, 0.0, 0.5]]
    Tv = [[10, 20, 30, 40], [1, 2, 3, 4]]
    x = [[0.5, -1.0, 3.0], [2.0, -3.0, 1.0]]
    y, m = oracle.forest_score(x, Tf, Tt, Tv, [0.25], return_margin=True)
    np.testing.assert_array_equal(y, g["y"])
    np.testing.assert_array_equal(m, g["margin"])
    # the fixture discriminates: "<=" instead of "<" (x_a sits on two thresholds), swapped children, or a leaf offset
    # of 2^depth instead of 2^depth - 1 would each change y
    assert oracle.forest_score(np.array(x) - 1e-3, Tf, Tt, Tv, [0.25])[0] != g["y"][0]


def test_p20_forest_closed_forms_and_library():
    rng = np.random.default_rng(20)
    n, nin, nt = 40, 9, 17
    x = rng.standard_normal((n, nin))
    # (a) stumps (depth 1): y = base + sum_t (x[f_t] < thr_t ? left_t : right_t), written with numpy comparisons
    f = rng.integers(0, nin, nt); thr = rng.standard_normal(nt).astype(np.float32); lv = rng.standard_normal((nt, 2))
    want = 0.5 + np.where(x.astype(np.float32)[:, f] < thr[None, :], lv[None, :, 0], lv[None, :, 1]).sum(axis=1)
    np.testing.assert_allclose(oracle.forest_score(x, f[:, None], thr[:, None], lv, [0.5]), want, rtol=0, atol=1e-12)
    # (b) a tree whose thresholds are all +inf always goes left: leaf 0; all -inf: the last leaf
    D = 3; nodes = 2 ** D - 1
    Tv = rng.standard_normal((1, nodes + 1))
    inf = np.full((1, nodes), np.inf, dtype=np.float32)
    assert (oracle.forest_score(x, np.zeros((1, nodes)), inf, Tv, [0.0]) == Tv[0, 0]).all()
    assert (oracle.forest_score(x, np.zeros((1, nodes)), -inf, Tv, [0.0]) == Tv[0, -1]).all()
    # (c) moving every feature by less than the reported margin changes no decision
    Tf = rng.integers(0, nin, (nt, nodes)); Tt = rng.standard_normal((nt, nodes)).astype(np.float32)
    Tvv = rng.standard_normal((nt, nodes + 1))
    y, m = oracle.forest_score(x, Tf, Tt, Tvv, [0.0], return_margin=True)
    assert (m > 0).all()
    np.testing.assert_array_equal(oracle.forest_score(x + 0.4 * m[:, None] * rng.choice([-1.0, 1.0], x.shape), Tf, Tt, Tvv, [0.0]), y)
    # (d) library cross-check: scikit-learn regression trees converted to the complete heap layout predict the same.
    # Data on a grid of eighths: sklearn splits at midpoints (odd sixteenths: exact in float32, never hit by an x), so
    # its "x <= t" and this ranker's "x < t" agree.
    from sklearn.tree import DecisionTreeRegressor
    xg = rng.integers(-16, 17, (300, 5)) / 8.0
    total = np.zeros(300)
    trees = []
    for t in range(3):
        yt = rng.standard_normal(300)
        sk = DecisionTreeRegressor(max_depth=D, random_state=t).fit(xg, yt)
        tr = sk.tree_
        hf = np.zeros(nodes); ht = np.full(nodes, np.inf, dtype=np.float32); hv = np.zeros(nodes + 1)

        def fill(sk_node, heap, depth):
            if depth == D:
                hv[heap - nodes] = tr.value[sk_node][0][0]
                return
            if tr.children_left[sk_node] == -1:       # an early leaf: always-left dummy splits below it, same value
                fill(sk_node, 2 * heap + 1, depth + 1)
                fill(sk_node, 2 * heap + 2, depth + 1)
                return
            hf[heap] = tr.feature[sk_node]; ht[heap] = tr.threshold[sk_node]
            assert float(ht[heap]) == tr.threshold[sk_node]
            fill(tr.children_left[sk_node], 2 * heap + 1, depth + 1)
            fill(tr.children_right[sk_node], 2 * heap + 2, depth + 1)

        fill(0, 0, 0)
        trees.append((hf, ht, hv))
        total += sk.predict(xg)
    got = oracle.forest_score(xg, np.stack([a for a, _, _ in trees]), np.stack([b for _, b, _ in trees]),
                              np.stack([c for _, _, c in trees]), [0.0])
    np.testing.assert_allclose(got, total, rtol=0, atol=1e-12)


@pytest.mark.parametrize("n", [10])
def test_p9_scalar_vs_vector_forest(n):
    cfg = gen.get_config(n)
    w = gen.make_weights(cfg); b = gen.make_inputs(cfg)
    yv = run_vec(cfg, w, b)
    ys = oracle.rollout_score_scalar(w, b.init_states, b.action_ids, b.action_params, b.lengths, b.hw_feats,
                                     b.subgraph_offsets, phi_kind=cfg.phi_kind)
    np.testing.assert_allclose(yv, ys, rtol=0, atol=1e-12)
    assert np.unique(np.round(yv, 9)).size > 30        # the forest separates the candidates


# ---- P21: the parity metrics themselves (S15) — every GPU parity assertion passes through these two ------------------

def test_p21_score_error_hand_values():
    """score_error = max_b |y - yref| / max(|yref|, RMS_s(yref)), RMS over the candidate's own subgraph (S15)."""
    # two subgraphs; RMS_0 = sqrt((9 + 16) / 2) = sqrt(12.5) = 3.5355..., RMS_1 = sqrt((0.01 + 0.01 + 100) / 3) = 5.7741...
    ref = np.array([3.0, -4.0, 0.1, -0.1, 10.0])
    off = [0, 2, 5]
    # candidate 0: |ref| = 3 < RMS_0  -> floor used:   0.5 / sqrt(12.5)
    # candidate 1: |ref| = 4 > RMS_0  -> |ref| used:   1.0 / 4 = 0.25
    # candidate 2: tiny score, floor:                  1.0 / sqrt(100.02 / 3)
    # candidate 4: |ref| = 10 > RMS_1:                 0.5 / 10
    y = ref + np.array([0.5, -1.0, 1.0, 0.0, -0.5])
    want = [0.5 / math.sqrt(12.5), 0.25, 1.0 / math.sqrt(100.02 / 3.0), 0.0, 0.05]
    assert oracle.score_error(y, ref, off) == pytest.approx(max(want), rel=1e-14)
    assert max(want) == pytest.approx(0.25, rel=1e-14)
    # one error at a time isolates every branch (a wrong floor, denominator or segment shows in exactly one of them)
    for i, wv in enumerate(want):
        yi = ref.copy(); yi[i] = y[i]
        assert oracle.score_error(yi, ref, off) == pytest.approx(wv, rel=1e-14), i
    # the floor is the candidate's OWN subgraph: moving the boundary changes candidate 2's denominator
    y2 = ref.copy(); y2[2] += 1.0
    assert oracle.score_error(y2, ref, [0, 3, 5]) == pytest.approx(1.0 / math.sqrt((9 + 16 + 0.01) / 3.0), rel=1e-14)
    # None offsets: one floor over the whole batch, RMS = sqrt((9 + 16 + 0.01 + 0.01 + 100) / 5)
    assert oracle.score_error(y2, ref, None) == pytest.approx(1.0 / math.sqrt(125.02 / 5.0), rel=1e-14)
    # the sign of the difference does not matter; the metric is not symmetric in (y, ref)
    assert oracle.score_error(2 * ref - y, ref, off) == pytest.approx(oracle.score_error(y, ref, off), rel=1e-14)
    assert oracle.score_error(ref, y, off) != pytest.approx(oracle.score_error(y, ref, off), rel=1e-6)
    # zero reference everywhere: the guard makes it an absolute error; identical vectors: 0; empty: 0
    assert oracle.score_error([0.0, 0.25], [0.0, 0.0], [0, 2]) == 0.25
    assert oracle.score_error(ref, ref, off) == 0.0
    assert oracle.score_error([], [], [0]) == 0.0
    # empty segments are skipped; a one-candidate segment is a pure relative error (RMS = |ref|)
    assert oracle.score_error([2.2, 5.0], [2.0, 4.0], [0, 0, 1, 1, 2]) == pytest.approx(0.25, rel=1e-14)
    # scale invariance: a relative metric
    assert oracle.score_error(7.0 * y, 7.0 * ref, off) == pytest.approx(oracle.score_error(y, ref, off), rel=1e-13)
    # NaN / inf in y must not pass as "small"
    bad = ref.copy(); bad[1] = np.nan
    assert not (oracle.score_error(bad, ref, off) <= 1e9)
    bad[1] = np.inf
    assert oracle.score_error(bad, ref, off) == np.inf


def test_p21_topk_overlap_hand_values():
    """topk_overlap = (mean, min) over segments of |A and B| / |valid entries of B| (S15), -1 = padding."""
    a = np.array([[0, 1, 2, 3], [10, 11, -1, -1], [20, 21, 22, 23], [-1, -1, -1, -1]])
    b = np.array([[3, 2, 9, 8], [11, 10, -1, -1], [24, 25, 26, 27], [-1, -1, -1, -1]])
    # segment 0: {2,3} of 4 -> 0.5; segment 1: order does not matter, 2 of 2 valid -> 1.0; segment 2: 0 of 4 -> 0;
    # segment 3: no valid reference entry -> skipped (not counted as 1.0 or 0.0)
    mean, mn = oracle.topk_overlap(a, b)
    assert mean == pytest.approx((0.5 + 1.0 + 0.0) / 3.0, rel=1e-15) and mn == 0.0
    assert oracle.topk_overlap(b, b) == (1.0, 1.0)
    # the denominator is the REFERENCE's valid count: a shorter GPU row cannot score 1.0, a padded reference row can
    assert oracle.topk_overlap([[5, -1, -1]], [[5, 6, 7]]) == (pytest.approx(1.0 / 3.0), pytest.approx(1.0 / 3.0))
    assert oracle.topk_overlap([[5, 6, 7]], [[5, -1, -1]]) == (1.0, 1.0)
    # -1 padding never matches -1 padding
    assert oracle.topk_overlap([[-1, -1]], [[4, -1]]) == (0.0, 0.0)
    # nothing to compare at all
    assert oracle.topk_overlap(np.zeros((0, 4), int), np.zeros((0, 4), int)) == (1.0, 1.0)
    # against a brute-force count on random index sets
    rng = np.random.default_rng(3)
    A = np.stack([rng.permutation(50)[:8] for _ in range(6)])
    B = np.stack([rng.permutation(50)[:8] for _ in range(6)])
    per = [sum(int(x in set(B[s])) for x in A[s]) / 8.0 for s in range(6)]
    mean, mn = oracle.topk_overlap(A, B)
    assert mean == pytest.approx(np.mean(per), rel=1e-15) and mn == pytest.approx(min(per), rel=1e-15)


# ---- generator / file format ----------------------------------------------------------------------------------

def test_weight_file_roundtrip(tmp_path):
    for n in (1, 2, 5, 6, 8, 9, 10, 13):
        cfg = gen.get_config(n)
        if n not in (1, 8, 10, 13):
            cfg = WMConfig(**{**cfg.__dict__, "d": 16, "d_a": 8, "hidden": 0 if n == 5 else 24,
                              "scorer_widths": (12, 10)})
        w = gen.make_weights(cfg)
        p = str(tmp_path / f"w{n}.bin")
        gen.write_weight_file(p, cfg, w)
        hdr, w2 = oracle.read_weight_file(p)
        assert hdr["d"] == cfg.d and hdr["kind"] == cfg.kind and hdr["P"] == cfg.P
        assert hdr["phi_kind"] == cfg.phi_kind
        assert hdr["version"] == (3 if cfg.ranker_kind else (1 if cfg.phi_kind == PHI_MEAN else 2))
        assert hdr["ranker_kind"] == cfg.ranker_kind and hdr["n_trees"] == cfg.n_trees
        if cfg.ranker_kind == 0:
            assert w2["Ws0"].shape[1] == cfg.d + cfg.phi_dim + cfg.H
        assert list(w2.keys()) == gen.tensor_order(cfg)
        for kname in w:
            np.testing.assert_array_equal(w[kname], w2[kname])
        if cfg.dtype != DTYPE_FP32:   # bf16 configs: stored values are bf16-representable
            for v in w.values():
                assert (v.view(np.uint32) & 0xFFFF == 0).all()


def test_generator_recipe():
    c2 = gen.get_config(2); b = gen.make_inputs(c2)
    assert b.lengths.min() == 8 and b.lengths.max() == 32 and b.action_ids.shape == (32768, 32)
    valid = np.arange(32)[None, :] < b.lengths[:, None]
    assert b.action_ids[valid].min() == 0 and b.action_ids[valid].max() == 31
    assert b.action_params[valid].min() == 1 and b.action_params[valid].max() <= 1024
    assert set(np.unique(b.action_ids[~valid])) <= {-2**31, 2**31 - 1}
    c3 = gen.get_config(3).scaled(S=8); b3 = gen.make_inputs(c3)
    assert b3.lengths.min() >= 4 and b3.lengths.max() <= 48 and abs(b3.lengths.mean() - 17.14) < 0.6
    c4 = gen.get_config(4).scaled(S=1, per_subgraph=128); b4 = gen.make_inputs(c4)
    assert (b4.lengths == 32).all()
    assert (b4.action_ids[:64, :16] == b4.action_ids[0, :16]).all()          # 64 children share >= 16 steps
    assert (b4.action_ids[64:128, :16] == b4.action_ids[64, :16]).all()
    assert (b4.action_ids[0, :16] != b4.action_ids[64, :16]).any()
    b_again = gen.make_inputs(c2)
    np.testing.assert_array_equal(b.action_params, b_again.action_params)       # seeded

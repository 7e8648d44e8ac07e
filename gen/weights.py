"""Seeded weights and the WMW1 weight-file writer (format: include/wm.h).

Draw order (one Generator(PCG64(weight_seed))):
  embedding (E, W_p, b_p | Tbl), transition (W1, b1, W2, b2[, gamma, beta] | W_g, W_r, W_h),
  scorer layers first to last (W, b each).
Matrices ~ N(0, 1/fan_in) (variance), tables ~ N(0,1), biases ~ N(0, 1/fan_in) of their layer,
gamma = 1 + 0.1 N(0,1), beta = 0.1 N(0,1).  bf16 configs: every tensor is rounded to the nearest-even
bf16 value and stored as fp32 (S14), so every consumer sees identical weights.
Structured-phi configs (f2): the phi columns of Ws0 are scaled, before the bf16 rounding, by the inverse of the
feature's range (counts and length 1/T_max, sums 1/(10 T_max), means and maxima 1/10; log2 of a parameter <= 1024 is
<= 10), as a trained ranker's first layer would be for raw count features, so that the latent still matters to the
score.  Version-2 header: the version-1 fields followed by uint32 phi_kind.
"""
from __future__ import annotations

import struct
from typing import Dict, List

import numpy as np

from .configs import (WMConfig, KIND_MLP, KIND_MLP_LN, KIND_GRU, KIND_TRANSH, DTYPE_BF16, EMBED_LINEAR, EMBED_BUCKET,
                      PHI_STRUCT, PHI_TYPED, RANKER_FOREST)

MAGIC = b"WMW1"
VERSION = 1
MAX_SCORER_HIDDEN = 6


def round_to_bf16(x: np.ndarray) -> np.ndarray:
    """Round fp32 values to the nearest-even bf16 value, returned as fp32."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32).astype(np.uint64)
    u = (u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32).reshape(x.shape)


def tensor_order(cfg: WMConfig) -> List[str]:
    """Names of the tensors in file order."""
    names: List[str] = []
    if cfg.embed == EMBED_LINEAR:
        names += ["E", "W_p", "b_p"]
    else:
        names += ["Tbl"]
    if cfg.kind in (KIND_MLP, KIND_MLP_LN):
        names += ["W1", "b1", "W2", "b2"]
        if cfg.kind == KIND_MLP_LN:
            names += ["gamma", "beta"]
    elif cfg.kind == KIND_TRANSH:      # hyperplane normal, translation, then the residual MLP
        names += ["W_w", "W_d", "W1", "b1", "W2", "b2"]
    else:
        names += ["W_g", "W_r", "W_h"]
    if cfg.ranker_kind == RANKER_FOREST:   # feature index, threshold per internal node; value per leaf; base score
        return names + ["Tf", "Tt", "Tv", "Tb"]
    for i in range(len(cfg.scorer_widths) + 1):
        names += [f"Ws{i}", f"bs{i}"]
    return names


def tensor_shapes(cfg: WMConfig) -> Dict[str, tuple]:
    d, da, hid = cfg.d, cfg.d_a, cfg.hidden
    sh: Dict[str, tuple] = {}
    if cfg.embed == EMBED_LINEAR:
        sh["E"] = (cfg.n_types, da)
        sh["W_p"] = (da, cfg.P)
        sh["b_p"] = (da,)
    else:
        sh["Tbl"] = (cfg.n_types * cfg.P * cfg.n_buckets, da)
    if cfg.kind == KIND_TRANSH:
        sh["W_w"] = (d, da)
        sh["W_d"] = (d, da)
    if cfg.kind in (KIND_MLP, KIND_MLP_LN, KIND_TRANSH):
        sh["W1"] = (hid, d + da)
        sh["b1"] = (hid,)
        sh["W2"] = (d, hid)
        sh["b2"] = (d,)
        if cfg.kind == KIND_MLP_LN:
            sh["gamma"] = (d,)
            sh["beta"] = (d,)
    else:
        for n in ("W_g", "W_r", "W_h"):
            sh[n] = (d, d + da)
    if cfg.ranker_kind == RANKER_FOREST:
        nodes = 2 ** cfg.tree_depth - 1
        sh["Tf"] = (cfg.n_trees, nodes)
        sh["Tt"] = (cfg.n_trees, nodes)
        sh["Tv"] = (cfg.n_trees, nodes + 1)
        sh["Tb"] = (1,)
        return sh
    dims = (cfg.scorer_in,) + tuple(cfg.scorer_widths) + (1,)
    for i, (a, b) in enumerate(zip(dims[:-1], dims[1:])):
        sh[f"Ws{i}"] = (b, a)
        sh[f"bs{i}"] = (b,)
    return sh


def make_weights(cfg: WMConfig) -> Dict[str, np.ndarray]:
    rng = np.random.Generator(np.random.PCG64(cfg.weight_seed))
    shapes = tensor_shapes(cfg)
    w: Dict[str, np.ndarray] = {}
    for name in tensor_order(cfg):
        shp = shapes[name]
        if name in ("Tf", "Tt", "Tv", "Tb"):     # the synthetic forest is drawn in one go, after everything else
            continue
        if name in ("E", "Tbl"):
            t = rng.standard_normal(shp)
        elif name == "gamma":
            t = 1.0 + 0.1 * rng.standard_normal(shp)
        elif name == "beta":
            t = 0.1 * rng.standard_normal(shp)
        elif len(shp) == 2:
            t = rng.standard_normal(shp) / np.sqrt(shp[1])
        else:  # bias of the layer drawn just before it
            fan_in = shapes[_matrix_of(name)][1]
            t = rng.standard_normal(shp) / np.sqrt(fan_in)
        if name == "Ws0" and cfg.phi_kind in (PHI_STRUCT, PHI_TYPED):
            t = t * phi_column_scale(cfg)[None, :]
        t = t.astype(np.float32)
        if cfg.dtype == DTYPE_BF16:
            t = round_to_bf16(t)
        w[name] = t
    if cfg.ranker_kind == RANKER_FOREST:
        w.update(_draw_forest(rng, cfg))
    return w


def _draw_forest(rng: np.random.Generator, cfg: WMConfig) -> Dict[str, np.ndarray]:
    """Synthetic complete binary trees over x = [z_T ; structured phi ; h] (stand-ins for a trained XGBoost ranker, which
    is not available here): a uniformly drawn feature per internal node, a threshold drawn over that feature's typical
    range (latent and hardware features ~ N(0, 0.7); counts, length, sums, means and maxima over their ranges), leaf
    values ~ N(0, 1/n_trees).  Feature indices are stored as fp32 (exact), everything fp32 whatever cfg.dtype says:
    thresholds are compared in fp32 on both sides."""
    nodes = 2 ** cfg.tree_depth - 1
    nin = cfg.scorer_in
    feat = rng.integers(0, nin, size=(cfg.n_trees, nodes))
    lo = np.zeros(nin); hi = np.zeros(nin); gauss = np.zeros(nin, dtype=bool)
    d, nt, P, T = cfg.d, cfg.n_types, cfg.P, float(cfg.T_max)
    gauss[:d] = True; gauss[d + cfg.phi_dim:] = True
    o = d
    hi[o:o + nt] = 3.0 * T / nt + 1.0                       # per-type counts
    lo[o + nt], hi[o + nt] = cfg.len_lo, cfg.len_hi          # length
    top = np.log2(cfg.param_hi)
    hi[o + nt + 1:o + nt + 1 + P] = top * T / 2              # sums of log2 params
    hi[o + nt + 1 + P:o + nt + 1 + 3 * P] = top              # means, maxima
    u = rng.random((cfg.n_trees, nodes)); g = rng.standard_normal((cfg.n_trees, nodes)) * 0.7
    thr = np.where(gauss[feat], g, lo[feat] + u * (hi[feat] - lo[feat]))
    leaf = rng.standard_normal((cfg.n_trees, nodes + 1)) / np.sqrt(cfg.n_trees)
    return {"Tf": feat.astype(np.float32), "Tt": thr.astype(np.float32), "Tv": leaf.astype(np.float32),
            "Tb": rng.standard_normal(1).astype(np.float32)}


def phi_column_scale(cfg: WMConfig) -> np.ndarray:
    """Per-input-column factor of Ws0 for structured-phi configs (1 for the z and hw columns)."""
    sc = np.ones(cfg.scorer_in)
    o, nt, P, T = cfg.d, cfg.n_types, cfg.P, float(cfg.T_max)
    sc[o:o + nt + 1] = 1.0 / T                              # per-type counts, length
    if cfg.phi_kind == PHI_TYPED:                           # per type: sums | means | maxima (a type occurs ~T/nt times)
        for k in range(nt):
            b = o + nt + 1 + 3 * P * k
            sc[b:b + P] = 1.0 / (10.0 * max(T / nt, 1.0))
            sc[b + P:b + 3 * P] = 0.1
        return sc
    sc[o + nt + 1:o + nt + 1 + P] = 1.0 / (10.0 * T)        # sums of log2 params
    sc[o + nt + 1 + P:o + nt + 1 + 3 * P] = 0.1             # means, maxima
    return sc


def _matrix_of(bias: str) -> str:
    return {"b_p": "W_p", "b1": "W1", "b2": "W2"}.get(bias, "Ws" + bias[2:])


def header_bytes(cfg: WMConfig) -> bytes:
    widths = list(cfg.scorer_widths) + [0] * (MAX_SCORER_HIDDEN - len(cfg.scorer_widths))
    # version 2 = version 1 + a trailing uint32 phi_kind; version 3 = version 2 + uint32 ranker_kind, n_trees, tree_depth
    forest = cfg.ranker_kind == RANKER_FOREST
    version = 3 if forest else (VERSION if cfg.phi_kind == 0 else 2)
    hdr = MAGIC + struct.pack(
        "<12I%dIf" % MAX_SCORER_HIDDEN,
        version, cfg.kind, cfg.dtype, cfg.embed, cfg.d, cfg.d_a, cfg.hidden, cfg.n_types, cfg.P,
        cfg.n_buckets, cfg.H, 0 if forest else len(cfg.scorer_widths) + 1, *widths, cfg.ln_eps)
    if version >= 2:
        hdr += struct.pack("<I", cfg.phi_kind)
    if version >= 3:
        hdr += struct.pack("<3I", cfg.ranker_kind, cfg.n_trees, cfg.tree_depth)
    return hdr


def write_weight_file(path: str, cfg: WMConfig, weights: Dict[str, np.ndarray]) -> None:
    shapes = tensor_shapes(cfg)
    with open(path, "wb") as f:
        f.write(header_bytes(cfg))
        for name in tensor_order(cfg):
            t = np.ascontiguousarray(weights[name], dtype="<f4")
            assert t.shape == shapes[name], (name, t.shape, shapes[name])
            f.write(t.tobytes())

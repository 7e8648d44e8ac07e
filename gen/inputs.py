"""Seeded synthetic candidate batches (stand-ins for AutoScheduler candidate populations,
PAPER.md:213-217; recipe SURVEY.md §8(d), S9/S11/S12).

Draw order (one Generator(PCG64(1000 + cfg.number))): z0, hw, lengths, action_ids, action_params;
cfg 4: parents (ids, params), then per child cut, then redrawn suffixes.  Padding positions (t >= len)
are overwritten with sentinel garbage (INT32_MIN / INT32_MAX alternating) so any consumer that touches
them is caught.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from .configs import WMConfig

INT32_MIN = np.int32(-2**31)
INT32_MAX = np.int32(2**31 - 1)


@dataclass
class Batch:
    init_states: np.ndarray        # [S, d] fp32
    hw_feats: np.ndarray           # [S, H] fp32
    action_ids: np.ndarray         # [B, T_max] int32
    action_params: np.ndarray      # [B, T_max, P] int32
    lengths: np.ndarray            # [B] int32
    subgraph_offsets: np.ndarray   # [S+1] int32
    T_max: int
    # shared-prefix structure (cfg 4 only, else None): candidate b copies positions [0, cut[b]) from parent parent_of[b]
    parent_of: np.ndarray = None   # [B] int64
    cut: np.ndarray = None         # [B] int64

    @property
    def B(self) -> int:
        return int(self.lengths.shape[0])

    @property
    def S(self) -> int:
        return int(self.subgraph_offsets.shape[0] - 1)


def _draw_params(rng: np.random.Generator, cfg: WMConfig, shape) -> np.ndarray:
    if cfg.param_dist == "uniform":
        return rng.integers(1, cfg.param_hi + 1, size=shape, dtype=np.int64).astype(np.int32)
    u = rng.random(size=shape, dtype=np.float32) * np.float32(np.log2(cfg.param_hi + 1.0))
    p = np.floor(np.exp2(u.astype(np.float64)))
    return np.clip(p, 1, cfg.param_hi).astype(np.int32)


def _draw_lengths(rng: np.random.Generator, cfg: WMConfig, B: int) -> np.ndarray:
    if cfg.len_dist == "uniform":
        return rng.integers(cfg.len_lo, cfg.len_hi + 1, size=B).astype(np.int32)
    if cfg.len_dist == "const":
        return np.full(B, cfg.len_hi, dtype=np.int32)
    support = np.arange(cfg.len_lo, cfg.len_hi + 1)
    prob = 1.0 / support
    prob /= prob.sum()
    return rng.choice(support, size=B, p=prob).astype(np.int32)


def make_inputs(cfg: WMConfig, sentinel_padding: bool = True) -> Batch:
    rng = np.random.Generator(np.random.PCG64(cfg.input_seed))
    S, n, B, T, P = cfg.S, cfg.per_subgraph, cfg.B, cfg.T_max, cfg.P
    z0 = rng.standard_normal((S, cfg.d)).astype(np.float32)
    hw = rng.standard_normal((S, cfg.H)).astype(np.float32)
    lengths = _draw_lengths(rng, cfg, B)
    parent_of = cut = None
    if cfg.prefix_children == 0:
        ids = rng.integers(0, cfg.n_types, size=(B, T)).astype(np.int32)
        params = _draw_params(rng, cfg, (B, T, P))
    else:
        C = cfg.prefix_children
        assert n % C == 0
        n_par = S * (n // C)
        par_ids = rng.integers(0, cfg.n_types, size=(n_par, T)).astype(np.int32)
        par_params = _draw_params(rng, cfg, (n_par, T, P))
        cut = rng.integers(cfg.prefix_cut_lo, cfg.prefix_cut_hi + 1, size=B)
        ids = rng.integers(0, cfg.n_types, size=(B, T)).astype(np.int32)
        params = _draw_params(rng, cfg, (B, T, P))
        parent_of = np.arange(B) // C
        keep = np.arange(T)[None, :] < cut[:, None]
        ids = np.where(keep, par_ids[parent_of], ids)
        params = np.where(keep[:, :, None], par_params[parent_of], params)
    if sentinel_padding:
        pad = np.arange(T)[None, :] >= lengths[:, None]
        sent = np.where((np.arange(T) % 2) == 0, INT32_MIN, INT32_MAX).astype(np.int32)
        ids = np.where(pad, sent[None, :], ids)
        params = np.where(pad[:, :, None], sent[None, :, None], params)
    offsets = (np.arange(S + 1, dtype=np.int64) * n).astype(np.int32)
    return Batch(z0, hw, np.ascontiguousarray(ids, dtype=np.int32),
                 np.ascontiguousarray(params, dtype=np.int32), lengths, offsets, T, parent_of, cut)

"""Test/bench plumbing: weight files in a temp dir, Batch -> device tensors, one call through the C ABI.

Holds no arithmetic of the method: it only moves the seeded inputs of `gen/` to the GPU and calls the binding.
"""
from __future__ import annotations

import os
import tempfile

import numpy as np

import gen

_TMP = None
_SEQ = 0


def weight_file(cfg, weights=None) -> str:
    """Write (once per process and config name) the WMW1 file for cfg; returns its path."""
    global _TMP
    if _TMP is None:
        _TMP = tempfile.mkdtemp(prefix="wmw_")
    if weights is not None:      # caller-supplied weights: always a fresh file (object ids are reused after a free)
        global _SEQ
        _SEQ += 1
        path = os.path.join(_TMP, f"{cfg.name}_custom{_SEQ}.wmw")
        gen.write_weight_file(path, cfg, weights)
        return path
    path = os.path.join(_TMP, f"{cfg.name}_{cfg.d}_{cfg.d_a}_{cfg.hidden}_{len(cfg.scorer_widths)}.wmw")
    if not os.path.exists(path):
        gen.write_weight_file(path, cfg, gen.make_weights(cfg))
    return path


def to_device(batch, per_candidate=False, device="cuda:0"):
    import torch
    dev = torch.device(device)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    d = dict(init_states=t(batch.init_states), hw_feats=t(batch.hw_feats), action_ids=t(batch.action_ids),
             action_params=t(batch.action_params), lengths=t(batch.lengths),
             subgraph_offsets=None if per_candidate else t(batch.subgraph_offsets))
    return d


def gpu_scores(ctx, batch, per_candidate=False, stream=None):
    """Scores [B] float32 (numpy) from wm_rollout_score; raises if the library reports a data fault."""
    import torch
    import paper_2606_09312_b200 as wm
    dv = to_device(batch, per_candidate)
    out = torch.full((batch.B,), float("nan"), dtype=torch.float32, device="cuda:0")
    wm.wm_rollout_score(ctx, dv["init_states"], dv["action_ids"], dv["action_params"], dv["lengths"],
                        dv["hw_feats"], out, dv["subgraph_offsets"], stream=stream)
    fault = wm.wm_check(ctx, stream)
    assert fault == 0, f"device fault word {fault}"
    return out.cpu().numpy()


def gpu_topk(scores, offsets, k):
    import torch
    import paper_2606_09312_b200 as wm
    sc = torch.from_numpy(np.ascontiguousarray(scores, dtype=np.float32)).cuda()
    off = torch.from_numpy(np.ascontiguousarray(offsets, dtype=np.int32)).cuda()
    S = off.numel() - 1
    idx = torch.full((max(S, 0), k), -7, dtype=torch.int32, device="cuda:0")
    wm.wm_topk(sc, off, k, idx)
    torch.cuda.synchronize()
    return idx.cpu().numpy()


def oracle_scores(cfg, weights, batch, per_candidate=False):
    import oracle
    return oracle.rollout_score_vec(weights, batch.init_states, batch.action_ids, batch.action_params,
                                    batch.lengths, batch.hw_feats,
                                    None if per_candidate else batch.subgraph_offsets,
                                    n_buckets=cfg.n_buckets, ln_eps=cfg.ln_eps, phi_kind=cfg.phi_kind)

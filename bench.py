#!/usr/bin/env python
"""bench.py — candidates scored/sec of the batched evaluator (BASELINE.json `metric`) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2]

A "step" is one pass of the whole hot path (length bucketing, rollout + score, top-k: DESIGN.md §1 rows a0-a7)
over one seeded synthetic batch of the workload config (default: BASELINE.json configs[1] = cfg 2, the
"evolution-round batch": 16 subgraphs x 2048 candidates, lengths U{8..32}).  With N > 1 (torchrun, one rank per
GPU) every rank scores its own full batch (different input seed, same weights): candidates are independent and
top-k is per subgraph, so there is no data-path collective ("scaling": "weak").

`value`   : candidates/s, inputs resident in HBM, CUDA-event time per step, max over ranks, L2 flushed between steps.
`e2e`     : the same metric through the C-ABI entry that takes HOST (pinned) buffers: H2D of the step's inputs and
            D2H of scores + top-k indices inside the timed region.
`roofline`: rollout+score kernel (K2) alone: literal FLOPs of the batch / its CUDA-event time (WM_OPT_TIMING).
`cpu_baseline`: the float64 numpy oracle, as it stands, on a bounded sample of the same workload on the host cores.
--impl reference times that oracle (the only "reference" there is: the paper ships no code).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import numpy as np

import gen

METRIC = "candidates_scored_per_sec"
UNIT = "candidates/s"


def _kernel_name(info) -> str:
    """The rollout+score kernel (K2) the library runs for this model, by its CUDA name."""
    if info.path == 2:
        return {1: "wm_tc_kernel", 2: "wm_tc2_kernel", 3: "wm_tcg_kernel", 4: "wm_tct_kernel"}[info.tc_variant]
    return "wm_generic_kernel"


# dram__bytes_read.sum + dram__bytes_write.sum of one launch of the dominant kernel, from the committed
# `ncu --set full` captures (profiles/*.md); keyed by (config number, kernel).  None where no capture exists yet.
NCU_TRAFFIC = {
    (2, "wm_tc_kernel"): (23_906_304 + 2_048, "profiles/r1_tc_v8.md"),
    (3, "wm_tc2_kernel"): (56_585_216 + 761_856, "profiles/r1_tc2_v4.md"),
    (5, "wm_tcg_kernel"): (3_450_484_000 + 61_085_952, "profiles/r1_tcg_v1.md"),
    (7, "wm_tct_kernel"): (24_100_608 + 2_048, "profiles/r1_tct_v1.md"),
}


def _dtype_name(cfg, info) -> str:
    """Arithmetic type of the path.  The tcgen05 kernels run kind::f16 MMAs on fp16 encodings of the bf16-valued
    weights with fp16 activations and fp32 accumulate / latent (S14); the fp32 kernel is plain fp32."""
    if cfg.dtype == gen.configs.DTYPE_FP32 or info.path != 2:
        return "f32"
    return "f16"


def workload_name(cfg) -> str:
    return f"cfg{cfg.number}:{cfg.name} S={cfg.S} B={cfg.B} T_max={cfg.T_max} d={cfg.d} hidden={cfg.hidden} k={cfg.k}"


def literal_flops(cfg, lengths) -> float:
    """Literal FLOPs of one batch: sum(len) transition steps + B scorer passes."""
    return float(int(lengths.sum())) * cfg.flops_per_step() + float(len(lengths)) * cfg.flops_scorer()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        j = json.load(open(p))
        return dict(bf16=j["bf16_tflops"], bf16_sustained=j.get("bf16_tflops_sustained", j["bf16_tflops"]),
                    hbm=j["hbm_gbs"], sm_max_mhz=float(j.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(bf16=1590.0, bf16_sustained=1400.0, hbm=6650.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        # "under load" = the upper half of the samples (the sampler also sees the idle gaps between steps)
        sm.sort()
        load = sm[len(sm) // 2:] if sm else []
        return {"sm_mhz": float(np.median(load)) if load else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def cpu_baseline(cfg, n_subgraphs: int):
    """Time the oracle (as it stands) on the first n_subgraphs subgraphs of the workload."""
    from wm_harness import oracle_scores
    import oracle
    sub = cfg.scaled(S=min(n_subgraphs, cfg.S))
    w = gen.make_weights(sub)
    b = gen.make_inputs(sub)
    t0 = time.perf_counter()
    y = oracle_scores(sub, w, b)
    oracle.topk_segments(y, b.subgraph_offsets, sub.k)
    dt = time.perf_counter() - t0
    return {"value": b.B / dt, "unit": UNIT, "cores": len(os.sched_getaffinity(0)), "kind": "oracle",
            "sample": f"first {sub.S} of {cfg.S} subgraphs ({b.B} candidates, {int(b.lengths.sum())} rollout "
                      f"steps) of {workload_name(cfg)}, float64 numpy, {dt:.1f} s",
            "rollout_steps_per_sec": float(b.lengths.sum()) / dt, "seconds": dt}


def run_reference(args, cfg):
    """--impl reference: the oracle on the host cores, each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n_sub = 1 if cfg.number != 1 else cfg.S
    for _ in range(args.warmup):
        cpu_baseline(cfg, n_sub)
    vals = [cpu_baseline(cfg, n_sub) for _ in range(args.steps)]
    secs = float(np.mean([v["seconds"] for v in vals]))
    cands = cfg.scaled(S=min(n_sub, cfg.S)).B
    value = cands / secs
    cb = dict(vals[-1]); cb["value"] = value
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": secs * 1e3, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": workload_name(cfg), "sample": cb["sample"]},
           "cpu_baseline": cb,
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


def reduce_max(value: float, dist_mod=None, device=None) -> float:
    """MAX over ranks of a host float (the step time); identity when not distributed."""
    if dist_mod is None or not dist_mod.is_initialized():
        return value
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device or "cpu")
    dist_mod.all_reduce(t, op=dist_mod.ReduceOp.MAX)
    return float(t.item())


def reduce_sum(value: float, dist_mod=None, device=None) -> float:
    if dist_mod is None or not dist_mod.is_initialized():
        return value
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device or "cpu")
    dist_mod.all_reduce(t, op=dist_mod.ReduceOp.SUM)
    return float(t.item())


def rank_config(cfg, rank: int):
    """Rank r's batch: same model and shapes, its own input seed (weak scaling; no exchange between ranks)."""
    from dataclasses import replace
    return cfg if rank == 0 else replace(cfg, number=cfg.number + 1000 * rank)


def run_ours(args, cfg):
    import torch
    import paper_2606_09312_b200 as wm
    from wm_harness import weight_file, to_device

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    assert torch.cuda.is_available(), "bench.py needs a GPU (there is no CPU fallback)"
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dev = torch.device("cuda", local_rank)

    ctx = wm.wm_load_weights(weight_file(cfg), local_rank)
    info = wm.wm_get_info(ctx)
    rcfg = rank_config(cfg, rank)
    batch = gen.make_inputs(rcfg)
    dv = to_device(batch, device=dev)
    B, S, k = batch.B, batch.S, cfg.k
    scores = torch.empty(B, dtype=torch.float32, device=dev)
    idx = torch.empty((S, k), dtype=torch.int32, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    def step():
        wm.wm_rollout_score(ctx, dv["init_states"], dv["action_ids"], dv["action_params"], dv["lengths"],
                            dv["hw_feats"], scores, dv["subgraph_offsets"])
        wm.wm_topk(scores, dv["subgraph_offsets"], k, idx)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        flush.zero_()
        step()
    assert wm.wm_check(ctx) == 0
    launches0 = wm.wm_launch_count(ctx) + wm.wm_launch_count(None)

    # ---- device-resident timing: K steps, each bracketed by events, L2 flushed (untimed) in between
    sampler = ClockSampler(local_rank)
    barrier()
    sampler.start()
    evs = []
    for _ in range(args.steps):
        flush.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        step()
        e1.record()
        evs.append((e0, e1))
    barrier()
    clocks = sampler.stop()
    launches = wm.wm_launch_count(ctx) + wm.wm_launch_count(None) - launches0
    ms = [a.elapsed_time(b) for a, b in evs]
    total_ms = reduce_max(float(np.sum(ms)), dist, dev)
    ms_per_step = total_ms / args.steps
    cands_all = reduce_sum(float(B), dist, dev)
    steps_all = reduce_sum(float(batch.lengths.sum()), dist, dev)
    value = cands_all / (ms_per_step * 1e-3)

    # ---- roofline leg: K2 alone, literal FLOPs / CUDA-event time on its stream
    wm.wm_set_option(ctx, wm.WM_OPT_TIMING, 1)
    kms = []
    for _ in range(args.steps):
        flush.zero_()
        wm.wm_rollout_score(ctx, dv["init_states"], dv["action_ids"], dv["action_params"], dv["lengths"],
                            dv["hw_feats"], scores, dv["subgraph_offsets"])
        kms.append(wm.wm_last_kernel_ms(ctx))
    wm.wm_set_option(ctx, wm.WM_OPT_TIMING, 0)
    k_ms = float(np.mean(kms))
    flops = literal_flops(cfg, batch.lengths)
    pk = peaks()
    achieved = flops / (k_ms * 1e-3) / 1e12
    bytes_in = sum(int(np.asarray(a).nbytes) for a in (batch.action_ids, batch.action_params, batch.lengths)) + 4 * B
    if cfg.dtype == gen.configs.DTYPE_FP32:
        # cfg 1: 12 MFLOP / 10 KB, launch-latency-bound; report the achieved HBM GB/s as north_star asks
        roof = {"bound": "hbm", "achieved": bytes_in / (k_ms * 1e-3) / 1e9, "peak": pk["hbm"], "unit": "GB/s",
                "traffic": None, "note": "latency-bound tiny config; neither roofline applies"}
    else:
        tr = NCU_TRAFFIC.get((cfg.number, _kernel_name(info)))
        if info.path == 2:
            roof = {"bound": "tensor", "achieved": achieved, "peak": pk["bf16"], "unit": "TFLOP/s",
                    "traffic": tr[0] if tr else None, "traffic_source": tr[1] if tr else None}
        else:
            # the fp32 CUDA-core kernel is bound by plain FFMA issue: 148 SMs x 128 lanes x 2 FLOP x SM clock
            # (K2-fp32), not by the tensor pipe
            alu_peak = 148 * 128 * 2 * (pk.get("sm_max_mhz", 1965.0) * 1e6) / 1e12
            roof = {"bound": "alu", "achieved": achieved, "peak": alu_peak, "unit": "TFLOP/s", "traffic": None,
                    "traffic_source": None, "note": "fp32 FFMA peak derived from unit counts and the SM clock"}
    roof["frac"] = roof["achieved"] / roof["peak"]
    roof.update({"kernel": _kernel_name(info), "kernel_ms": k_ms,
                 "peak_source": pk["source"] + " (burst: kernel timed alone)",
                 "algorithmic_flops_per_launch": flops, "share_of_step": k_ms / float(np.mean(ms))})

    # ---- prefix-latent reuse leg (NEXT row f3; configs with a shared-prefix structure, i.e. cfg 4): the representative of
    # every family (the child with the longest copied prefix) is rolled once over that prefix with the latent stored
    # after every step, then every child is scored from its cut.  Same scores, a third of the rollout steps.
    prefix = None
    if batch.cut is not None and args.prefix_reuse:
        C = cfg.prefix_children
        cut = batch.cut.reshape(-1, C)
        rep = (np.arange(cut.shape[0]) * C + cut.argmax(axis=1)).astype(np.int64)       # one representative per family
        rep_len = torch.from_numpy(cut.max(axis=1).astype(np.int32)).to(dev)
        rep_ids = dv["action_ids"][torch.from_numpy(rep).to(dev)].contiguous()
        rep_par = dv["action_params"][torch.from_numpy(rep).to(dev)].contiguous()
        fam_off = torch.from_numpy((np.asarray(batch.subgraph_offsets, dtype=np.int64) // C).astype(np.int32)).to(dev)
        T = batch.T_max
        bank = torch.empty((rep.size, T, cfg.d), dtype=torch.float32, device=dev)
        start = torch.from_numpy(batch.cut.astype(np.int32)).to(dev)
        index = torch.from_numpy(((np.arange(B) // C) * T + batch.cut - 1).astype(np.int32)).to(dev)
        scores2 = torch.empty_like(scores)
        idx2 = torch.empty_like(idx)

        def prefix_step():
            wm.wm_rollout_latents(ctx, dv["init_states"], rep_ids, rep_par, rep_len, bank, fam_off)
            wm.wm_rollout_score_from(ctx, bank.view(-1, cfg.d), index, start, dv["action_ids"], dv["action_params"],
                                     dv["lengths"], dv["hw_feats"], scores2, dv["subgraph_offsets"])
            wm.wm_topk(scores2, dv["subgraph_offsets"], k, idx2)

        for _ in range(3):
            flush.zero_()
            prefix_step()
        assert wm.wm_check(ctx) == 0
        pms = []
        for _ in range(args.steps):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            prefix_step()
            e1.record()
            torch.cuda.synchronize()
            pms.append(e0.elapsed_time(e1))
        p_ms = float(np.mean(pms))
        executed = int(cut.max(axis=1).sum() + (batch.lengths - batch.cut).sum())
        prefix = {"value": B / (p_ms * 1e-3), "unit": UNIT, "ms_per_step": p_ms,
                  "executed_rollout_steps": executed, "literal_rollout_steps": int(batch.lengths.sum()),
                  "bank_bytes": int(bank.numel() * 4),
                  "max_abs_score_diff_vs_literal": float((scores2 - scores).abs().max().item()),
                  "topk_identical_to_literal": bool(torch.equal(idx2, idx)),
                  "calls": "wm_rollout_latents (family representatives) + wm_rollout_score_from (children) + wm_topk"}
        del bank

    # ---- e2e leg: host (pinned) buffers through wm_score_topk_host
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    hb = dict(z0=pin(batch.init_states), ids=pin(batch.action_ids), par=pin(batch.action_params),
              ln=pin(batch.lengths), hw=pin(batch.hw_feats), off=pin(batch.subgraph_offsets))
    h_scores = torch.empty(B, dtype=torch.float32).pin_memory()
    h_idx = torch.empty((S, k), dtype=torch.int32).pin_memory()

    def e2e_step():
        wm.wm_score_topk_host(ctx, hb["z0"], hb["ids"], hb["par"], hb["ln"], hb["hw"], hb["off"], k, h_scores, h_idx)

    for _ in range(3):
        e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        e2e_step()          # synchronous: returns after the D2H copies
    torch.cuda.synchronize()
    e2e_s = reduce_max((time.perf_counter() - t0) / args.steps, dist, dev)
    h2d = sum(int(t.numel() * t.element_size()) for t in hb.values())
    d2h = int(h_scores.numel() * 4 + h_idx.numel() * 4)
    np.testing.assert_array_equal(h_idx.numpy(), idx.cpu().numpy())   # same answer through both entries

    wm.wm_free(ctx)
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": _dtype_name(cfg, info),
           "data": "synthetic",
           "config": {"workload": workload_name(cfg), "per_gpu_batch": B, "l2": "flushed between steps (256 MB write)",
                      "path": _kernel_name(info),
                      "operands": ("fp32" if _dtype_name(cfg, info) == "f32" else
                                   "bf16-valued weights encoded as fp16 (exact), fp16 activations, fp32 accumulate + latent"),
                      "parallelism": f"dp{world} (independent batches, no collective)"},
           "rollout_steps_per_sec": steps_all / (ms_per_step * 1e-3),
           "clocks": clocks, "gpu_launches": int(launches),
           "e2e": {"value": cands_all / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                   "ms_per_step": e2e_s * 1e3},
           "roofline": roof}
    if prefix is not None:
        out["prefix_reuse"] = prefix
    if world == 1:
        out["cpu_baseline"] = cpu_baseline(cfg, 4 if cfg.number != 1 else cfg.S)
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--prefix-reuse", action="store_true",
                    help="config 4: also time the prefix-latent-reuse calls (extra 'prefix_reuse' object in the JSON line)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number (1-5); 2 = configs[1]; 6, 7 = NEXT row f1 (TransH transition); 8, 9 = NEXT row f2 (structured phi); 10, 11 = NEXT row f4 (forest ranker); 12 = TransH + structured phi + forest")
    args = ap.parse_args()
    cfg = gen.get_config(args.config)
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()

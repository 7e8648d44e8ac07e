#!/usr/bin/env python
"""bench.py — candidates scored/sec of the batched evaluator (BASELINE.json `metric`) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2]
                    [--scaling weak|strong] [--no-per-config] [--no-sustained] [--prefix-reuse]

A "step" is one pass of the whole hot path (length bucketing, rollout + score, top-k: DESIGN.md §1 rows a0-a7)
over one seeded synthetic batch of the workload config (default: BASELINE.json configs[1] = cfg 2, the
"evolution-round batch": 16 subgraphs x 2048 candidates, lengths U{8..32}).

`value`      : candidates/s, inputs resident in HBM, CUDA-event time per step, max over ranks, L2 flushed between steps.
`e2e`        : the same metric through the C-ABI entry that takes HOST (pinned) buffers: H2D of the step's inputs and
               D2H of scores + top-k indices inside the timed region.  The entry is wm_score_topk_host_ragged (the valid
               steps only, uint8 / uint16); `e2e_compact` (padded uint8 / uint16) and `e2e_int32` (padded int32) beside it.
`roofline`   : rollout+score kernel (K2) alone: literal FLOPs of the batch / its CUDA-event time (WM_OPT_TIMING).
`sustained`  : (N = 1) the headline config's wm_rollout_score launched back to back for >= 2 s with no flush in between —
               the online loop of PAPER.md:215 calls the evaluator round after round — with the clocks seen, against the
               measured SUSTAINED bf16 peak.
`per_config` : (N = 1, default config only) the other BASELINE.json configs (1, 3, 4, 5) through the same legs: ms per
               step, K2 ms, TFLOP/s, fraction of the burst and of the sustained peak, clocks; cfg 1 also as a ratio to an
               empty-kernel launch.
`cpu_baseline`: the float64 numpy oracle, as it stands, on a bounded sample of the same workload on the host cores.
--impl reference times that oracle (the only "reference" there is: the paper ships no code).

N > 1: one rank per GPU (torchrun; `python bench.py --gpus N` without torchrun re-executes itself under it).  Candidates
are independent and top-k is per subgraph, so there is no data-path collective.  --scaling weak (default): every rank
scores its own full batch (different input seed, same weights).  --scaling strong: ONE batch is
partitioned by whole-subgraph ranges, each rank scores and ranks its subgraphs, the [S_local, k] index blocks are
all-gathered.
"""
from __future__ import annotations

import argparse
import glob
import json
import os
import re
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
KERNELS = {1: "wm_tc_kernel", 2: "wm_tc2_kernel", 3: "wm_tcg_kernel", 5: "wm_tcp_kernel"}


def _kernel_name(info) -> str:
    """The rollout+score kernel (K2) the library runs for this model, by its CUDA name."""
    if info.path == 2 and info.phi_kind == 2:
        # per-type phi: the pair kernel rolls, wm_typed_x_kernel writes the scorer's input rows, wm_tsc_kernel ranks
        return "wm_tcp_kernel + wm_tsc_kernel"
    if info.path != 2 and info.kind in (0, 1) and info.embed == 0 and info.phi_kind == 0 and info.dtype == 0 and info.d <= 256:
        return "wm_small_kernel (<= 592 candidates) / wm_generic_kernel"     # csrc/wm_generic.cu: small_call_ok
    return KERNELS.get(info.tc_variant, "wm_tc_kernel") if info.path == 2 else "wm_generic_kernel"


def ncu_traffic(config: int, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of `kernel` on `config`, from the NEWEST committed
    `ncu --set full` summary under profiles/ that carries a line
        <!-- traffic: config=<n> kernel=<name> dram_bytes_per_launch=<bytes> -->
    (files sort by round and version: r2_* after r1_*).  (bytes, file) or (None, None) when no capture names the pair."""
    best = (None, None)
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "*.md"))):
        try:
            text = open(path).read()
        except OSError:
            continue
        for m in re.finditer(r"<!--\s*traffic:\s*config=(\d+)\s+kernel=(\w+)\s+dram_bytes_per_launch=(\d+)\s*-->", text):
            if int(m.group(1)) == config and m.group(2) == kernel:
                best = (int(m.group(3)), os.path.relpath(path, ROOT))
    return best


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
    return dict(bf16=1590.0, bf16_sustained=1400.0, hbm=6650.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler:
    """SM clock, power and throttle reasons DURING a timed region (B200_PROFILING.md's clocks line).  Polls NVML from a
    thread every ~2 ms (the timed region of the default run is ~20 ms: nvidia-smi's 100 ms loop saw two samples of it);
    falls back to the `nvidia-smi -lms` loop when pynvml cannot be initialised."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int, period_s: float = 0.002):
        self.index, self.period = index, period_s
        self.sm, self.power, self.reasons, self.mx = [], [], set(), None
        self.proc = self.thread = None
        self.stop_flag = False
        self.nvml = None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            # NVML enumerates all GPUs of the host; CUDA_VISIBLE_DEVICES may renumber them
            vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
            phys = self.index
            if vis and all(t.strip().isdigit() for t in vis.split(",")):
                phys = int(vis.split(",")[self.index])
            h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.mx = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            self.nvml = (pynvml, h)
            self.thread = threading.Thread(target=self._poll, daemon=True)
            self.thread.start()
            return self
        except Exception:     # noqa: BLE001 - any NVML problem: use the CLI loop instead
            self.nvml = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "20"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read_cli, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None
        return self

    def _poll(self):
        pynvml, h = self.nvml
        bits = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20}
        get_reasons = getattr(pynvml, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
            getattr(pynvml, "nvmlDeviceGetCurrentClocksThrottleReasons")
        # two pollers: NVML's power and reasons queries take several ms each, the clock query about one; a single loop over
        # all three saw ONE sample of a 10 ms timed region
        def slow():
            while not self.stop_flag:
                try:
                    self.power.append(pynvml.nvmlDeviceGetPowerUsage(h) / 1000.0)
                    r = int(get_reasons(h))
                    for name, bit in bits.items():
                        if r & bit:
                            self.reasons.add(name)
                except Exception:     # noqa: BLE001
                    pass
                time.sleep(self.period)
        self.thread2 = threading.Thread(target=slow, daemon=True)
        self.thread2.start()
        while not self.stop_flag:
            try:
                self.sm.append(float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)))
            except Exception:     # noqa: BLE001
                pass
            time.sleep(self.period / 4)

    def _read_cli(self):
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.proc.stdout:
            r = [x.strip() for x in line.split(",")]
            try:
                self.sm.append(float(r[0]))
                self.mx = float(r[1])
                self.power.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    self.reasons.add(n)

    def stop(self):
        if self.nvml is None and self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["clock sampling unavailable"], "samples": 0}
        if self.proc is not None:
            time.sleep(0.05)
            self.proc.terminate()
        self.stop_flag = True
        if self.thread is not None:
            self.thread.join(1.0)
        if getattr(self, "thread2", None) is not None:
            self.thread2.join(1.0)
        sm = sorted(self.sm)
        # "under load" = the upper half of the samples (the sampler also sees the idle gaps between steps)
        load = sm[len(sm) // 2:] if sm else []
        return {"sm_mhz": float(np.median(load)) if load else None, "sm_min_mhz": sm[0] if sm else None,
                "sm_max_mhz": self.mx, "power_w_max": max(self.power) if self.power else None,
                "reasons": sorted(self.reasons), "samples": len(sm),
                "source": "nvml poll (clock 0.5 ms, power / reasons 2 ms between queries)" if self.nvml else "nvidia-smi -lms 20"}


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
    """Rank r's batch under WEAK scaling: same model and shapes, its own input seed (no exchange between ranks)."""
    from dataclasses import replace
    return cfg if rank == 0 else replace(cfg, number=cfg.number + 1000 * rank)


def subgraph_range(S: int, world: int, rank: int):
    """STRONG scaling: rank r owns the whole subgraphs [s0, s1) of the one batch — contiguous,
    near-equal counts, every subgraph owned exactly once."""
    return (S * rank) // world, (S * (rank + 1)) // world


def slice_batch(batch, s0: int, s1: int):
    """The sub-batch of subgraphs [s0, s1): candidates and offsets rebased to the slice (views, no arithmetic)."""
    off = np.asarray(batch.subgraph_offsets, dtype=np.int64)
    c0, c1 = int(off[s0]), int(off[s1])
    return gen.Batch(batch.init_states[s0:s1], batch.hw_feats[s0:s1], batch.action_ids[c0:c1], batch.action_params[c0:c1],
                     batch.lengths[c0:c1], (off[s0:s1 + 1] - c0).astype(np.int32), batch.T_max,
                     None if batch.parent_of is None else batch.parent_of[c0:c1],
                     None if batch.cut is None else batch.cut[c0:c1]), c0


def gather_topk(idx_local, c0: int, S: int, k: int, world: int, dist_mod, device):
    """All-gather of the per-rank [S_local, k] index blocks into the batch's [S, k] (global candidate indices: the
    slice's base is added to every valid entry).  The only exchange of the strong-scaling mode, after the timed kernels."""
    import torch
    glob_idx = torch.where(idx_local >= 0, idx_local + int(c0), idx_local)
    if dist_mod is None or not dist_mod.is_initialized():
        return glob_idx
    rows = max(subgraph_range(S, world, r)[1] - subgraph_range(S, world, r)[0] for r in range(world))
    pad = torch.full((rows, k), -1, dtype=torch.int32, device=device)
    pad[:glob_idx.shape[0]] = glob_idx
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist_mod.all_gather(parts, pad)
    out = [parts[r][:subgraph_range(S, world, r)[1] - subgraph_range(S, world, r)[0]] for r in range(world)]
    return torch.cat(out, dim=0)


class Leg:
    """One config on one device: weights, resident inputs, and the timed legs."""

    def __init__(self, wm, cfg, batch, dev, flush):
        import torch
        from wm_harness import weight_file, to_device
        self.wm, self.cfg, self.batch, self.dev, self.flush = wm, cfg, batch, dev, flush
        self.ctx = wm.wm_load_weights(weight_file(cfg), dev.index or 0)
        if os.environ.get("WM_BENCH_SINGLE_CTA"):     # A/B: the single-CTA form of the d = 256 kernel (WM_OPT_PAIR = 0)
            wm.wm_set_option(self.ctx, wm.WM_OPT_PAIR, 0)
        self.info = wm.wm_get_info(self.ctx)
        self.dv = to_device(batch, device=dev)
        self.B, self.S, self.k = batch.B, batch.S, cfg.k
        self.scores = torch.empty(self.B, dtype=torch.float32, device=dev)
        self.idx = torch.empty((self.S, self.k), dtype=torch.int32, device=dev)

    def score(self):
        dv = self.dv
        self.wm.wm_rollout_score(self.ctx, dv["init_states"], dv["action_ids"], dv["action_params"], dv["lengths"],
                                 dv["hw_feats"], self.scores, dv["subgraph_offsets"])

    def step(self):
        self.score()
        self.wm.wm_topk(self.scores, self.dv["subgraph_offsets"], self.k, self.idx)

    def warm(self, n):
        for _ in range(max(n, 3)):
            self.flush.zero_()
            self.step()
        assert self.wm.wm_check(self.ctx) == 0

    def launches(self):
        return self.wm.wm_launch_count(self.ctx) + self.wm.wm_launch_count(None)

    def timed_steps(self, steps, barrier):
        """K steps, each bracketed by CUDA events on the launching stream, L2 flushed (untimed) in between; clocks
        sampled during the region.  -> (list of ms, clocks, launches)"""
        import torch
        sampler = ClockSampler(self.dev.index or 0)
        barrier()
        n0 = self.launches()
        sampler.start()
        evs = []
        for _ in range(steps):
            self.flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            self.step()
            e1.record()
            evs.append((e0, e1))
        barrier()
        clocks = sampler.stop()
        return [a.elapsed_time(b) for a, b in evs], clocks, self.launches() - n0

    def kernel_ms(self, steps):
        """K2 alone (WM_OPT_TIMING: events recorded by the library around the rollout+score launch)."""
        wm = self.wm
        wm.wm_set_option(self.ctx, wm.WM_OPT_TIMING, 1)
        kms = []
        for _ in range(steps):
            self.flush.zero_()
            self.score()
            kms.append(wm.wm_last_kernel_ms(self.ctx))
        wm.wm_set_option(self.ctx, wm.WM_OPT_TIMING, 0)
        return float(np.mean(kms))

    def roofline(self, k_ms, step_ms):
        cfg, info, pk = self.cfg, self.info, peaks()
        flops = literal_flops(cfg, self.batch.lengths)
        achieved = flops / (k_ms * 1e-3) / 1e12
        b = self.batch
        bytes_in = sum(int(np.asarray(a).nbytes) for a in (b.action_ids, b.action_params, b.lengths)) + 4 * self.B
        if cfg.dtype == gen.configs.DTYPE_FP32:
            # cfg 1: 12 MFLOP / 10 KB, launch-latency-bound; report the achieved HBM GB/s as north_star asks
            roof = {"bound": "hbm", "achieved": bytes_in / (k_ms * 1e-3) / 1e9, "peak": pk["hbm"], "unit": "GB/s",
                    "traffic": None, "note": "latency-bound tiny config; neither roofline applies"}
        elif info.path == 2:
            tr, src = ncu_traffic(cfg.number, _kernel_name(info))
            roof = {"bound": "tensor", "achieved": achieved, "peak": pk["bf16"], "unit": "TFLOP/s",
                    "traffic": tr, "traffic_source": src, "frac_of_sustained_peak": achieved / pk["bf16_sustained"],
                    "peak_sustained": pk["bf16_sustained"]}
        else:
            # the fp32 CUDA-core kernel is bound by plain FFMA issue: 148 SMs x 128 lanes x 2 FLOP x SM clock
            # (K2-fp32), not by the tensor pipe
            alu_peak = 148 * 128 * 2 * (pk.get("sm_max_mhz", 1965.0) * 1e6) / 1e12
            roof = {"bound": "alu", "achieved": achieved, "peak": alu_peak, "unit": "TFLOP/s", "traffic": None,
                    "traffic_source": None, "note": "fp32 FFMA peak derived from unit counts and the SM clock"}
        roof["frac"] = roof["achieved"] / roof["peak"]
        roof.update({"kernel": _kernel_name(info), "kernel_ms": k_ms,
                     "peak_source": pk["source"] + " (burst: kernel timed alone)",
                     "algorithmic_flops_per_launch": flops, "share_of_step": k_ms / step_ms})
        return roof

    def sustained(self, seconds=2.0):
        """wm_rollout_score back to back for >= `seconds` with no flush and no host sync in between (the regime of an
        online search loop): ms per call (bucketing + K2), literal TFLOP/s, clocks and throttle reasons seen."""
        import torch
        self.score()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); self.score(); e1.record(); torch.cuda.synchronize()
        one = max(e0.elapsed_time(e1), 1e-3)
        n = int(min(max(seconds * 1e3 / one, 10), 200000))
        sampler = ClockSampler(self.dev.index or 0, period_s=0.01).start()
        e0.record()
        for _ in range(n):
            self.score()
        e1.record()
        torch.cuda.synchronize()
        clocks = sampler.stop()
        ms = e0.elapsed_time(e1) / n
        pk = peaks()
        tf = literal_flops(self.cfg, self.batch.lengths) / (ms * 1e-3) / 1e12
        return {"calls": n, "seconds": ms * n * 1e-3, "ms_per_call": ms, "tflops": tf,
                "frac_of_sustained_peak": tf / pk["bf16_sustained"], "frac_of_burst_peak": tf / pk["bf16"],
                "peak_sustained": pk["bf16_sustained"], "clocks": clocks,
                "what": "wm_rollout_score (bucketing + K2) back to back, inputs L2-warm, literal FLOPs / call time"}

    def close(self):
        self.wm.wm_free(self.ctx)
        self.ctx = None


def per_config_leg(wm, n, dev, flush, steps):
    """One of the other BASELINE.json configs through the device-resident legs (default run, N = 1)."""
    import torch
    cfg = gen.get_config(n)
    t0 = time.perf_counter()
    batch = gen.make_inputs(cfg)
    gen_s = time.perf_counter() - t0
    leg = Leg(wm, cfg, batch, dev, flush)
    leg.warm(3)
    ms, clocks, launches = leg.timed_steps(steps, torch.cuda.synchronize)
    step_ms = float(np.mean(ms))
    k_ms = leg.kernel_ms(steps)
    roof = leg.roofline(k_ms, step_ms)
    out = {"workload": workload_name(cfg), "kernel": roof["kernel"], "steps": steps, "ms_per_step": step_ms,
           "value": leg.B / (step_ms * 1e-3), "unit": UNIT,
           "rollout_steps_per_sec": float(batch.lengths.sum()) / (step_ms * 1e-3), "kernel_ms": k_ms,
           "gpu_launches": int(launches), "clocks": clocks, "input_generation_s": gen_s}
    if roof["bound"] == "tensor":
        out.update({"tflops": roof["achieved"], "frac_of_burst_peak": roof["frac"],
                    "frac_of_sustained_peak": roof["frac_of_sustained_peak"], "traffic": roof["traffic"],
                    "traffic_source": roof.get("traffic_source")})
    else:
        # cfg 1: launch-latency-bound.  Yardstick: one empty kernel launch, timed the same way (events around
        # back-to-back launches on the stream); the step is bucketing (2 launches + memset) + K2 + top-k.
        for _ in range(20):
            wm.wm_launch_empty()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 200
        torch.cuda.synchronize()
        e0.record()
        for _ in range(reps):
            wm.wm_launch_empty()
        e1.record()
        torch.cuda.synchronize()
        empty_ms = e0.elapsed_time(e1) / reps
        one = []
        for _ in range(50):      # a lone launch between two events (launch + drain, not back-to-back throughput)
            a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); wm.wm_launch_empty(); b_.record(); torch.cuda.synchronize()
            one.append(a.elapsed_time(b_))
        lone_ms = float(np.median(one))
        out.update({"achieved_gbs": roof["achieved"], "empty_kernel_launch_ms": lone_ms,
                    "empty_kernel_back_to_back_ms": empty_ms,
                    "step_over_empty_launch": step_ms / lone_ms, "k2_over_empty_launch": k_ms / lone_ms,
                    "note": "launch-latency-bound: 12 MFLOP, 10 KB of input"})
    leg.close()
    del leg, batch
    torch.cuda.empty_cache()
    return out


def run_ours(args, cfg):
    import torch
    import paper_2606_09312_b200 as wm

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
    strong = args.scaling == "strong" and world > 1

    c0 = 0
    if strong:      # one batch, this rank's whole subgraphs
        full = gen.make_inputs(cfg)
        s0, s1 = subgraph_range(full.S, world, rank)
        batch, c0 = slice_batch(full, s0, s1)
    else:
        batch = gen.make_inputs(rank_config(cfg, rank))
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2
    leg = Leg(wm, cfg, batch, dev, flush)
    info = leg.info
    B, S, k = leg.B, leg.S, leg.k

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    leg.warm(args.warmup)

    # ---- device-resident timing
    ms, clocks, launches = leg.timed_steps(args.steps, barrier)
    total_ms = reduce_max(float(np.sum(ms)), dist, dev)
    ms_per_step = total_ms / args.steps
    cands_all = reduce_sum(float(B), dist, dev)
    steps_all = reduce_sum(float(batch.lengths.sum()), dist, dev)
    value = cands_all / (ms_per_step * 1e-3)
    gathered_rows = None
    if strong:      # the result exchange of the strong mode: [S_local, k] -> [S, k] on every rank
        gathered_rows = int(gather_topk(leg.idx, c0, cfg.S, k, world, dist, dev).shape[0])

    # ---- roofline leg: K2 alone
    k_ms = leg.kernel_ms(args.steps)
    roof = leg.roofline(k_ms, float(np.mean(ms)))

    # ---- sustained leg (N = 1): back-to-back launches for >= 2 s
    sustained = None
    if world == 1 and not args.no_sustained and roof["bound"] == "tensor":
        sustained = leg.sustained(2.0)

    # ---- prefix-latent reuse leg (NEXT row f3; configs with a shared-prefix structure, i.e. cfg 4): the representative of
    # every family (the child with the longest copied prefix) is rolled once over that prefix with the latent stored
    # after every step, then every child is scored from its cut.  Same scores, a third of the rollout steps.
    prefix = None
    ctx, dv, scores, idx = leg.ctx, leg.dv, leg.scores, leg.idx
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

    # The host keeps the action arrays compact when the model allows it (uint8 type ids, uint16 parameters: 13 instead of
    # 28 bytes per action on PCIe; include/wm.h wm_score_topk_host_compact); e2e_int32 is the int32 entry beside it.
    valid = np.arange(batch.T_max)[None, :] < batch.lengths[:, None]
    compact = cfg.n_types <= 256 and int(batch.action_params[valid].max(initial=1)) <= 65535
    if compact:
        hb["ids8"] = pin(np.where(valid, batch.action_ids, 0).astype(np.uint8))
        hb["par16"] = torch.from_numpy(np.where(valid[:, :, None], batch.action_params, 1).astype(np.uint16).view(np.int16)).pin_memory()
        # ... and ragged (a search loop holds sequences of different lengths as they are: the valid steps only, packed
        # candidate after candidate; include/wm.h wm_score_topk_host_ragged): no padding crosses PCIe
        hb["so"] = pin(np.concatenate([[0], np.cumsum(batch.lengths)]).astype(np.int32))
        hb["sid8"] = pin(batch.action_ids[valid].astype(np.uint8))
        hb["spar16"] = torch.from_numpy(np.ascontiguousarray(batch.action_params[valid]).astype(np.uint16).view(np.int16)).pin_memory()

    def e2e_step_int32():
        wm.wm_score_topk_host(ctx, hb["z0"], hb["ids"], hb["par"], hb["ln"], hb["hw"], hb["off"], k, h_scores, h_idx)

    def e2e_step_compact():
        wm.wm_score_topk_host_compact(ctx, hb["z0"], hb["ids8"], hb["par16"], hb["ln"], hb["hw"], hb["off"], k, h_scores, h_idx)

    def e2e_step_ragged():
        wm.wm_score_topk_host_ragged(ctx, hb["z0"], hb["sid8"], hb["spar16"], hb["so"], hb["hw"], hb["off"], batch.T_max, k,
                                     h_scores, h_idx)

    def time_e2e_all(fns):
        """K synchronous calls of every entry, one entry after the other (alternating between the entries was measured: each
        has its own pinned buffers, 52 MB in all, and on these boxes — a VM behind an IOMMU — a call that follows a call on
        OTHER buffers is 0.2-0.3 ms slower than one that repeats its own); seconds per call of each entry, max over ranks."""
        for fn in fns:
            fn()
            np.testing.assert_array_equal(h_idx.numpy(), idx.cpu().numpy())   # same answer through every entry
        total = [0.0] * len(fns)
        left = [args.steps] * len(fns)
        block = args.steps
        barrier()
        while any(left):
            for i, fn in enumerate(fns):
                n = min(block, left[i])
                if n == 0:
                    continue
                # warm-up of this entry's block: at least 3 calls and 0.25 s.  The host side of a call (a dozen driver calls, a
                # spinning wait) and the link ramp up over ~100 ms of traffic on these boxes: 4 warm-up calls gave 0.85-0.92 ms
                # per call, 200 gave 0.71-0.73 for the same entry; a serving loop runs in the warmed state
                t_warm, n_warm = time.perf_counter() + 0.25, 0
                while n_warm < 3 or time.perf_counter() < t_warm:
                    fn()
                    n_warm += 1
                t0 = time.perf_counter()
                for _ in range(n):
                    fn()          # synchronous: returns after the D2H copies
                total[i] += time.perf_counter() - t0
                left[i] -= n
        torch.cuda.synchronize()
        return [reduce_max(t / args.steps, dist, dev) for t in total]

    nbytes = lambda names: sum(int(hb[n].numel() * hb[n].element_size()) for n in names)
    h2d32 = nbytes(("z0", "ids", "par", "ln", "hw", "off"))
    e2ec_s = h2dc = None
    if compact:
        e2e32_s, e2ec_s, e2e_s = time_e2e_all([e2e_step_int32, e2e_step_compact, e2e_step_ragged])
        h2dc = nbytes(("z0", "ids8", "par16", "ln", "hw", "off"))
        h2d = nbytes(("z0", "sid8", "spar16", "so", "hw", "off"))
    else:
        (e2e32_s,) = time_e2e_all([e2e_step_int32])
        e2e_s, h2d = e2e32_s, h2d32
    d2h = int(h_scores.numel() * 4 + h_idx.numel() * 4)
    del hb, h_scores, h_idx

    leg.close()
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    scaling = "strong" if strong else "weak"
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": scaling,
           "vs_baseline": None, "dtype": _dtype_name(cfg, info),
           "data": "synthetic",
           "config": {"workload": workload_name(cfg), "per_gpu_batch": B, "l2": "flushed between steps (256 MB write)",
                      "path": _kernel_name(info),
                      "operands": ("fp32" if _dtype_name(cfg, info) == "f32" else
                                   "bf16-valued weights encoded as fp16 (exact for 2^-14 <= |w| <= 65504), fp16 "
                                   "activations, fp32 accumulate + latent"),
                      "parallelism": (f"dp{world}: one batch split by whole-subgraph ranges, [S_local,k] all-gather "
                                      f"after the timed kernels ({gathered_rows} rows gathered)" if strong else
                                      f"dp{world} (independent batches, no collective)")},
           "rollout_steps_per_sec": steps_all / (ms_per_step * 1e-3),
           "clocks": clocks, "gpu_launches": int(launches),
           "e2e": {"value": cands_all / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                   "ms_per_step": e2e_s * 1e3,
                   "entry": ("wm_score_topk_host_ragged (valid steps only: uint8 ids, uint16 params, int32 step offsets)" if compact
                             else "wm_score_topk_host (int32)")},
           "e2e_int32": {"value": cands_all / e2e32_s, "unit": UNIT, "h2d_bytes_per_step": h2d32, "d2h_bytes_per_step": d2h,
                         "ms_per_step": e2e32_s * 1e3, "entry": "wm_score_topk_host (int32)"},
           "roofline": roof}
    if e2ec_s is not None:
        out["e2e_compact"] = {"value": cands_all / e2ec_s, "unit": UNIT, "h2d_bytes_per_step": h2dc, "d2h_bytes_per_step": d2h,
                              "ms_per_step": e2ec_s * 1e3, "entry": "wm_score_topk_host_compact (padded uint8 ids, uint16 params)"}
    if sustained is not None:
        out["sustained"] = sustained
    if prefix is not None:
        out["prefix_reuse"] = prefix
    if world == 1:
        if args.config == 2 and not args.no_per_config:
            del batch
            torch.cuda.empty_cache()
            out["per_config"] = {}
            for n, st in ((1, 20), (3, 10), (4, 5), (5, 5)):
                out["per_config"][f"cfg{n}"] = per_config_leg(wm, n, dev, flush, st)
        out["cpu_baseline"] = cpu_baseline(cfg, 4 if cfg.number != 1 else cfg.S)
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def relaunch_under_torchrun(args) -> None:
    """`python bench.py --gpus N` outside torchrun: start the N ranks ourselves (same launch line the driver uses)."""
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    os.execv(sys.executable, cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--prefix-reuse", action="store_true",
                    help="config 4: also time the prefix-latent-reuse calls (extra 'prefix_reuse' object in the JSON line)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = a full batch per rank; strong = one batch split by whole-subgraph ranges (SURVEY.md §8(e))")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config object (cfg 1, 3, 4, 5) of the default run")
    ap.add_argument("--no-sustained", action="store_true", help="skip the 2 s back-to-back leg")
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number (1-5); 2 = configs[1]; 6, 7 = NEXT row f1 (TransH transition); 8, 9 = NEXT row f2 (structured phi); 10, 11 = NEXT row f4 (forest ranker); 12 = TransH + structured phi + forest")
    args = ap.parse_args()
    cfg = gen.get_config(args.config)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        relaunch_under_torchrun(args)
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()

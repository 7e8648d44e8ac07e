"""N > 1 host logic of bench.py on CPU: world_size-2 gloo, max-over-ranks time, whole-job candidate count,
per-rank batches (weak scaling, no data-path collective)."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import gen
    cfg = gen.get_config(2).scaled(S=2, per_subgraph=16)
    rc = bench.rank_config(cfg, rank)
    b = gen.make_inputs(rc)
    t = bench.reduce_max(10.0 + rank, dist)
    n = bench.reduce_sum(float(b.B), dist)
    q.put((rank, t, n, int(b.lengths.sum()), float(b.init_states[0, 0]), rc.weight_seed))
    dist.destroy_process_group()


def test_world2_gloo_reductions_and_rank_batches():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    (r0, t0, n0, s0, z0, w0), (r1, t1, n1, s1, z1, w1) = res
    assert t0 == t1 == 11.0            # max over ranks
    assert n0 == n1 == 64.0            # whole-job candidates = 2 ranks x 32
    assert z0 != z1                    # each rank scores its own batch
    assert w0 == w1 == 0               # same weights on every rank


def _strong_worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import gen
    cfg = gen.get_config(2).scaled(S=5, per_subgraph=12)      # 5 subgraphs on 2 ranks: 2 + 3
    full = gen.make_inputs(cfg)
    s0, s1 = bench.subgraph_range(full.S, world, rank)
    sub, c0 = bench.slice_batch(full, s0, s1)
    # stand-in for the rank's top-k (the kernels need a GPU): the first k LOCAL candidate indices of each subgraph,
    # last column -1 (padding must survive the rebasing)
    k = 4
    loc = torch.stack([torch.arange(int(sub.subgraph_offsets[s]), int(sub.subgraph_offsets[s]) + k, dtype=torch.int32)
                       for s in range(sub.S)])
    loc[:, -1] = -1
    got = bench.gather_topk(loc, c0, full.S, k, world, dist, "cpu")
    q.put((rank, s0, s1, c0, sub.B, got.numpy().tolist(), int(sub.subgraph_offsets[-1]),
           bool(np.array_equal(sub.action_ids, full.action_ids[c0:c0 + sub.B]))))
    dist.destroy_process_group()


def test_world2_strong_scaling_partition_and_gather():
    """one batch split by whole-subgraph ranges, [S_local, k] blocks all-gathered into [S, k]."""
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + (os.getpid() % 2000)
    ps = [ctx.Process(target=_strong_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    (_, a0, a1, c0a, Ba, ga, lasta, sama), (_, b0, b1, c0b, Bb, gb, lastb, samb) = res
    assert (a0, a1, b0, b1) == (0, 2, 2, 5) and (c0a, c0b) == (0, 24) and (Ba, Bb) == (24, 36)
    assert lasta == Ba and lastb == Bb and sama and samb            # offsets rebased, candidates are views of the batch
    want = [[12 * s, 12 * s + 1, 12 * s + 2, -1] for s in range(5)]     # global indices, padding untouched
    assert ga == want and gb == want                                    # every rank ends with the whole [S, k]


def test_subgraph_range_covers_every_subgraph_once():
    import bench
    for S in (1, 2, 7, 16, 64, 128):
        for world in (1, 2, 3, 4, 8):
            r = [bench.subgraph_range(S, world, k) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == S
            assert all(r[i][1] == r[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1


def test_gpus_flag_relaunches_under_torchrun():
    """`python bench.py --gpus 2` outside torchrun starts two ranks itself; on this GPU-less box both reach the
    'needs a GPU' assertion (there is no CPU fallback)."""
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    if torch.cuda.is_available():
        return
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1", "--no-per-config"],
                       capture_output=True, text=True, timeout=300, env=env)
    assert p.returncode != 0
    assert p.stderr.count("bench.py needs a GPU") >= 2, p.stderr[-2000:]


def test_ncu_traffic_reads_the_newest_profile(tmp_path, monkeypatch):
    import bench
    b, src = bench.ncu_traffic(2, "wm_tc_kernel")                      # (round 1's capture: the only one for this kernel)
    assert b == 23908352 and src == "profiles/r1_tc_v8.md"
    for n, kern, r1 in ((3, "wm_tc2_kernel", "profiles/r1_tc2_v4.md"), (5, "wm_tcg_kernel", "profiles/r1_tcg_v1.md")):
        b3, src3 = bench.ncu_traffic(n, kern)                          # two captures name this pair: the newer file wins
        assert src3 > r1 and b3 > 0
    assert bench.ncu_traffic(99, "wm_tc_kernel") == (None, None)
    (tmp_path / "profiles").mkdir()
    (tmp_path / "profiles" / "r1_x.md").write_text("<!-- traffic: config=2 kernel=k dram_bytes_per_launch=10 -->")
    (tmp_path / "profiles" / "r2_x.md").write_text("<!-- traffic: config=2 kernel=k dram_bytes_per_launch=20 -->")
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    assert bench.ncu_traffic(2, "k") == (20, "profiles/r2_x.md")


def test_single_process_reductions_are_identity():
    import bench
    assert bench.reduce_max(3.5) == 3.5 and bench.reduce_sum(2.0) == 2.0
    import gen
    cfg = gen.get_config(2)
    assert bench.rank_config(cfg, 0) is cfg
    ln = np.array([1, 2, 3])
    assert bench.literal_flops(cfg, ln) == 6 * cfg.flops_per_step() + 3 * cfg.flops_scorer()
    assert cfg.flops_per_step() == 655360 and cfg.flops_scorer() == 934912

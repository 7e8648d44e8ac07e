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


def test_single_process_reductions_are_identity():
    import bench
    assert bench.reduce_max(3.5) == 3.5 and bench.reduce_sum(2.0) == 2.0
    import gen
    cfg = gen.get_config(2)
    assert bench.rank_config(cfg, 0) is cfg
    ln = np.array([1, 2, 3])
    assert bench.literal_flops(cfg, ln) == 6 * cfg.flops_per_step() + 3 * cfg.flops_scorer()
    assert cfg.flops_per_step() == 655360 and cfg.flops_scorer() == 934912

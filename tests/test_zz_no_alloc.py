"""wm_rollout_score_static (include/wm.h): the allocation-free entry against the existing wm_rollout_score.

Collected last on purpose (pytest -x: a failure here hides nothing).  The entry's scratch is one
static device array shared by every call on the device and it keeps the previous call's contents, so each case makes
TWO calls in a row on DIFFERENT batches (other lengths -> another histogram and permutation): a counter that was not
cleared, or a stale permutation entry, shows up in the second call.  Scores do not depend on the order inside a length
bin, so both entries must agree to fp32 rounding (2e-5, the "same path" tolerance of tests/test_gpu_parity.py); the
oracle bar of the config (1e-4 fp32 / 2e-2 bf16) is checked as well.
"""
import ctypes
import numpy as np
import pytest

import gen
import oracle
from gen.configs import DTYPE_FP32
from wm_harness import weight_file, gpu_scores, oracle_scores, to_device

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def wm():
    import torch
    assert torch.cuda.is_available()
    import paper_2606_09312_b200 as wm
    return wm


def _static_scores(wm, ctx, batch):
    import torch
    dv = to_device(batch)
    out = torch.full((batch.B,), float("nan"), dtype=torch.float32, device="cuda:0")
    wm.wm_rollout_score_static(ctx, dv["init_states"], dv["action_ids"], dv["action_params"], dv["lengths"],
                               dv["hw_feats"], out, dv["subgraph_offsets"])
    assert wm.wm_check(ctx) == 0
    return out.cpu().numpy()


# several tiles of every kernel and more than 256 candidates, so that K1 (the user of the scratch) runs:
# cfg 1 = fp32 kernel, cfg 2 = d = 256 pair kernel (12 = its single-CTA form: the tile counter lives in the scratch too),
# cfg 3 = d = 512 pair kernel, cfg 5 = GRU pair kernel
@pytest.mark.parametrize("n,single", [(1, False), (2, False), (2, True), (3, False), (5, False)])
def test_static_entry_matches_rollout_score_twice_in_a_row(wm, n, single):
    base = gen.get_config(n)
    cfg_a = base.scaled(S=3, per_subgraph=171 if n != 1 else 120)
    cfg_b = base.scaled(S=2, per_subgraph=333 if n != 1 else 150)
    w = gen.make_weights(cfg_a)
    batch_a = gen.make_inputs(cfg_a)
    batch_b = gen.make_inputs(cfg_b)                          # other sizes -> other draws of lengths and actions
    ctx = wm.wm_load_weights(weight_file(cfg_a))
    if single:
        wm.wm_set_option(ctx, wm.WM_OPT_PATH, wm.PATH_TCGEN05)
        wm.wm_set_option(ctx, wm.WM_OPT_PAIR, 0)
        assert wm.wm_get_info(ctx).tc_variant == 1
    tol = 1e-4 if base.dtype == DTYPE_FP32 else 2e-2
    launches0 = wm.wm_launch_count(ctx)
    for cfg, batch in ((cfg_a, batch_a), (cfg_b, batch_b), (cfg_a, batch_a)):
        y = _static_scores(wm, ctx, batch)                    # static scratch first: nothing of the other path was set up
        assert np.isfinite(y).all()
        lit = gpu_scores(ctx, batch)                          # the existing path (per-stream cudaMalloc'ed workspace)
        assert oracle.score_error(y, lit, batch.subgraph_offsets) <= 2e-5, (n, single)
        ref = oracle_scores(cfg, w, batch)
        assert oracle.score_error(y, ref, batch.subgraph_offsets) <= tol, (n, single)
    assert wm.wm_launch_count(ctx) > launches0                # our kernels ran (no fallback)
    wm.wm_free(ctx)


def test_static_entry_on_a_per_type_phi_model(wm):
    """A WM_PHI_TYPED model: wm_rollout_score splits the call over three kernels and two workspace buffers it allocates; the
    allocation-free entry cannot, and runs the whole call on the fp32 kernel instead (no tcgen05 rollout kernel holds a
    scorer for this phi) — slower, and within the fp32 kernel's tolerance of the oracle."""
    cfg = gen.get_config(14).scaled(S=2, per_subgraph=300)
    w, b = gen.make_weights(cfg), gen.make_inputs(cfg)
    ctx = wm.wm_load_weights(weight_file(cfg))
    assert wm.wm_get_info(ctx).path == 2
    ref = oracle_scores(cfg, w, b)
    for _ in range(2):
        y = _static_scores(wm, ctx, b)
        assert oracle.score_error(y, ref, b.subgraph_offsets) <= 2e-3
    assert oracle.score_error(gpu_scores(ctx, b), ref, b.subgraph_offsets) <= 2e-2      # the split call, for comparison
    wm.wm_free(ctx)


def test_static_entry_rejects_what_it_cannot_hold(wm):
    """B beyond WM_STATIC_MAX_B: WM_ERR_ARG and a message that names the limit (checked before any pointer is read);
    the forest ranker and WM_OPT_TIMING: WM_ERR_UNSUPPORTED; B = 0: no-op."""
    import torch
    cfg = gen.get_config(2).scaled(S=1, per_subgraph=64)
    ctx = wm.wm_load_weights(weight_file(cfg))
    lib = wm.lib()
    one = torch.zeros(16, dtype=torch.float32, device="cuda:0")
    p = ctypes.c_void_p(one.data_ptr())
    rc = lib.wm_rollout_score_static(ctx, p, p, p, p, p, p, p, wm.WM_STATIC_MAX_B + 1, 1, cfg.T_max, None)
    assert rc == wm.WM_ERR_ARG
    msg = lib.wm_last_error().decode()
    assert "WM_STATIC_MAX_B" in msg and str(wm.WM_STATIC_MAX_B) in msg, msg
    assert lib.wm_rollout_score_static(ctx, p, p, p, p, p, p, p, 0, 1, cfg.T_max, None) == wm.WM_OK
    wm.wm_set_option(ctx, wm.WM_OPT_TIMING, 1)
    assert lib.wm_rollout_score_static(ctx, p, p, p, p, p, p, p, 8, 1, cfg.T_max, None) == wm.WM_ERR_UNSUPPORTED
    wm.wm_free(ctx)
    fcfg = gen.get_config(10).scaled(S=1, per_subgraph=64)
    fctx = wm.wm_load_weights(weight_file(fcfg))
    assert lib.wm_rollout_score_static(fctx, p, p, p, p, p, p, p, 8, 1, fcfg.T_max, None) == wm.WM_ERR_UNSUPPORTED
    wm.wm_free(fctx)

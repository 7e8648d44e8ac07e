"""paper_2606_09312_b200 — thin Python binding of the C-ABI library (include/wm.h).

Argument marshalling only: every step of the hot path runs in the library's CUDA kernels.  The functions
keep the ABI's names (`wm_load_weights`, `wm_rollout_score`, `wm_topk`, ...).  PyTorch is used for device
memory and streams.  There is no CPU fallback: if libwm.so is missing or does not load, importing the
binding's functions raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libwm.so")

WM_OK, WM_ERR_ARG, WM_ERR_IO, WM_ERR_FORMAT, WM_ERR_CUDA, WM_ERR_UNSUPPORTED = 0, -1, -2, -3, -4, -5
WM_MAX_T, WM_MAX_K = 256, 1024
WM_FAULT_LEN, WM_FAULT_TYPE, WM_FAULT_PARAM, WM_FAULT_INDEX, WM_FAULT_RANGE = 1, 2, 4, 8, 16
WM_OPT_PATH, WM_OPT_SORT, WM_OPT_TIMING, WM_OPT_PAIR = 1, 2, 3, 4
WM_STATIC_MAX_B = 262144   # wm_rollout_score_static: candidates the static scratch holds
PATH_AUTO, PATH_FP32, PATH_TCGEN05 = 0, 1, 2

# every symbol include/wm.h declares
ABI_SYMBOLS = ("wm_load_weights", "wm_free", "wm_get_info", "wm_set_option", "wm_rollout_score", "wm_topk",
               "wm_rollout_latents", "wm_rollout_score_from", "wm_rollout_score_static",
               "wm_check", "wm_score_topk_host", "wm_score_topk_host_compact", "wm_score_topk_host_ragged", "wm_last_kernel_ms", "wm_launch_count", "wm_launch_empty", "wm_last_error", "wm_path_reason")


class WmInfo(ctypes.Structure):
    _fields_ = [("kind", ctypes.c_int32), ("dtype", ctypes.c_int32), ("embed", ctypes.c_int32),
                ("d", ctypes.c_int32), ("d_a", ctypes.c_int32), ("hidden", ctypes.c_int32),
                ("n_types", ctypes.c_int32), ("P", ctypes.c_int32), ("n_buckets", ctypes.c_int32),
                ("H", ctypes.c_int32), ("n_scorer_layers", ctypes.c_int32),
                ("scorer_widths", ctypes.c_int32 * 6), ("ln_eps", ctypes.c_float), ("path", ctypes.c_int32),
                ("tc_variant", ctypes.c_int32), ("phi_kind", ctypes.c_int32),
                ("ranker_kind", ctypes.c_int32), ("n_trees", ctypes.c_int32), ("tree_depth", ctypes.c_int32)]


class WmError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"wm error {code}: {msg}")
        self.code = code


_lib = None


def lib() -> ctypes.CDLL:
    """Load libwm.so (built by paper_2606_09312_b200.build).  Fails loudly when it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2606_09312_b200.build` "
                          "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
    L.wm_load_weights.argtypes = [ctypes.c_char_p, ctypes.c_int, ctypes.POINTER(vp)]
    L.wm_load_weights.restype = ctypes.c_int
    L.wm_free.argtypes = [vp]
    L.wm_free.restype = None
    L.wm_get_info.argtypes = [vp, ctypes.POINTER(WmInfo)]
    L.wm_get_info.restype = ctypes.c_int
    L.wm_set_option.argtypes = [vp, i32, i32]
    L.wm_set_option.restype = ctypes.c_int
    L.wm_rollout_score.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, i64, i32, i32, vp]
    L.wm_rollout_score.restype = ctypes.c_int
    L.wm_rollout_score_static.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, i64, i32, i32, vp]
    L.wm_rollout_score_static.restype = ctypes.c_int
    L.wm_rollout_latents.argtypes = [vp, vp, vp, vp, vp, vp, vp, i64, i32, i32, vp]
    L.wm_rollout_score_from.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, i64, i32, i32, i64, vp]
    L.wm_rollout_latents.restype = ctypes.c_int
    L.wm_rollout_score_from.restype = ctypes.c_int
    L.wm_topk.argtypes = [vp, vp, i32, i32, vp, vp]
    L.wm_topk.restype = ctypes.c_int
    L.wm_check.argtypes = [vp, vp]
    L.wm_check.restype = ctypes.c_int
    L.wm_score_topk_host.argtypes = [vp, vp, vp, vp, vp, vp, vp, i64, i32, i32, i32, vp, vp, vp]
    L.wm_score_topk_host.restype = ctypes.c_int
    L.wm_score_topk_host_compact.argtypes = [vp, vp, vp, vp, vp, vp, vp, i64, i32, i32, i32, vp, vp, vp]
    L.wm_score_topk_host_ragged.argtypes = [vp, vp, vp, vp, vp, vp, vp, i64, i32, i32, i32, vp, vp, vp]
    L.wm_score_topk_host_ragged.restype = ctypes.c_int
    L.wm_score_topk_host_compact.restype = ctypes.c_int
    L.wm_last_kernel_ms.argtypes = [vp, vp, ctypes.POINTER(ctypes.c_float)]
    L.wm_last_kernel_ms.restype = ctypes.c_int
    L.wm_launch_count.argtypes = [vp]
    L.wm_launch_count.restype = i64
    L.wm_launch_empty.argtypes = [vp]
    L.wm_launch_empty.restype = ctypes.c_int
    L.wm_path_reason.argtypes = [vp]
    L.wm_path_reason.restype = ctypes.c_char_p
    L.wm_last_error.argtypes = []
    L.wm_last_error.restype = ctypes.c_char_p
    _lib = L
    return L


def _check(rc: int) -> int:
    if rc < 0:
        raise WmError(rc, lib().wm_last_error().decode("utf-8", "replace"))
    return rc


def _ptr(t) -> Optional[int]:
    return None if t is None else t.data_ptr()


def _stream(stream=None) -> Optional[int]:
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return s.cuda_stream or None


def wm_last_error() -> str:
    return lib().wm_last_error().decode("utf-8", "replace")


def wm_load_weights(path: str, device: int = 0) -> int:
    """-> ctx handle (int).  include/wm.h: wm_load_weights."""
    ctx = ctypes.c_void_p()
    _check(lib().wm_load_weights(os.fsencode(path), int(device), ctypes.byref(ctx)))
    return ctx.value


def wm_free(ctx: int) -> None:
    lib().wm_free(ctx)


def wm_get_info(ctx: int) -> WmInfo:
    info = WmInfo()
    _check(lib().wm_get_info(ctx, ctypes.byref(info)))
    return info


def wm_set_option(ctx: int, key: int, value: int) -> None:
    _check(lib().wm_set_option(ctx, key, value))


def wm_rollout_score(ctx: int, init_states, action_ids, action_params, lengths, hw_feats, scores_out,
                     subgraph_offsets=None, stream=None) -> None:
    """Device tensors in, scores_out ([B] fp32, device) written asynchronously on the stream.
    Sizes are read from the tensors: B = lengths.numel(), T_max = action_ids.shape[1],
    S = subgraph_offsets.numel() - 1 (0 in per-candidate mode)."""
    B = int(lengths.numel())
    T_max = int(action_ids.shape[1]) if action_ids is not None and action_ids.dim() == 2 else 0
    S = int(subgraph_offsets.numel()) - 1 if subgraph_offsets is not None else 0
    _check(lib().wm_rollout_score(ctx, _ptr(init_states), _ptr(action_ids), _ptr(action_params), _ptr(lengths),
                                  _ptr(hw_feats), _ptr(scores_out), _ptr(subgraph_offsets), B, S, T_max,
                                  _stream(stream)))


def wm_rollout_score_static(ctx: int, init_states, action_ids, action_params, lengths, hw_feats, scores_out,
                            subgraph_offsets=None, stream=None) -> None:
    """wm_rollout_score without any allocation: the call's scratch is a static device array of the library, shared by
    every call on the device (B <= WM_STATIC_MAX_B; calls that overlap on the GPU race).  include/wm.h."""
    B = int(lengths.numel())
    T_max = int(action_ids.shape[1]) if action_ids is not None and action_ids.dim() == 2 else 0
    S = int(subgraph_offsets.numel()) - 1 if subgraph_offsets is not None else 0
    _check(lib().wm_rollout_score_static(ctx, _ptr(init_states), _ptr(action_ids), _ptr(action_params), _ptr(lengths),
                                         _ptr(hw_feats), _ptr(scores_out), _ptr(subgraph_offsets), B, S, T_max,
                                         _stream(stream)))


def wm_score_topk_host_ragged(ctx: int, init_states, step_ids_u8, step_params_u16, step_offsets, hw_feats, subgraph_offsets,
                              T_max: int, k: int, scores_out, idx_out, stream=None) -> None:
    """wm_score_topk_host on the valid steps only (HOST tensors): step_ids [N] uint8, step_params [N, P] uint16,
    step_offsets [B + 1] int32.  include/wm.h."""
    import torch
    assert step_ids_u8.dtype == torch.uint8 and step_params_u16.dtype in (torch.uint16, torch.int16)
    B = int(step_offsets.numel()) - 1
    S = int(subgraph_offsets.numel()) - 1
    _check(lib().wm_score_topk_host_ragged(ctx, _ptr(init_states), _ptr(step_ids_u8), _ptr(step_params_u16), _ptr(step_offsets),
                                           _ptr(hw_feats), _ptr(subgraph_offsets), B, S, int(T_max), int(k),
                                           _ptr(scores_out), _ptr(idx_out), _stream(stream)))


def wm_rollout_latents(ctx: int, init_states, action_ids, action_params, lengths, latents_out,
                       subgraph_offsets=None, stream=None) -> None:
    """latents_out [B, T_max, d] fp32 (device): z after step t+1 at [b][t] for t < lengths[b].  include/wm.h."""
    B = int(lengths.numel())
    T_max = int(action_ids.shape[1]) if action_ids is not None and action_ids.dim() == 2 else 0
    S = int(subgraph_offsets.numel()) - 1 if subgraph_offsets is not None else 0
    _check(lib().wm_rollout_latents(ctx, _ptr(init_states), _ptr(action_ids), _ptr(action_params), _ptr(lengths),
                                    _ptr(subgraph_offsets), _ptr(latents_out), B, S, T_max, _stream(stream)))


def wm_rollout_score_from(ctx: int, bank, bank_index, start, action_ids, action_params, lengths, hw_feats, scores_out,
                          subgraph_offsets, stream=None) -> None:
    """Score candidates whose first start[b] steps were rolled before (latent in bank[bank_index[b]]).  include/wm.h."""
    B = int(lengths.numel())
    T_max = int(action_ids.shape[1]) if action_ids is not None and action_ids.dim() == 2 else 0
    S = int(subgraph_offsets.numel()) - 1
    n_bank = int(bank.numel() // bank.shape[-1])
    _check(lib().wm_rollout_score_from(ctx, _ptr(bank), _ptr(bank_index), _ptr(start), _ptr(action_ids),
                                       _ptr(action_params), _ptr(lengths), _ptr(hw_feats), _ptr(scores_out),
                                       _ptr(subgraph_offsets), B, S, T_max, n_bank, _stream(stream)))


def wm_topk(scores, subgraph_offsets, k: int, idx_out, stream=None) -> None:
    """idx_out [S, k] int32 (device) written asynchronously on the stream."""
    S = int(subgraph_offsets.numel()) - 1
    _check(lib().wm_topk(_ptr(scores), _ptr(subgraph_offsets), S, int(k), _ptr(idx_out), _stream(stream)))


def wm_check(ctx: int, stream=None) -> int:
    return _check(lib().wm_check(ctx, _stream(stream)))


def wm_score_topk_host(ctx: int, init_states, action_ids, action_params, lengths, hw_feats, subgraph_offsets,
                       k: int, scores_out, idx_out, stream=None) -> None:
    """HOST tensors (CPU, contiguous; pinned for speed) in and out; synchronous.  include/wm.h."""
    B = int(lengths.numel())
    T_max = int(action_ids.shape[1]) if action_ids.dim() == 2 else 0
    S = int(subgraph_offsets.numel()) - 1
    _check(lib().wm_score_topk_host(ctx, _ptr(init_states), _ptr(action_ids), _ptr(action_params), _ptr(lengths),
                                    _ptr(hw_feats), _ptr(subgraph_offsets), B, S, T_max, int(k),
                                    _ptr(scores_out), _ptr(idx_out), _stream(stream)))


def wm_score_topk_host_compact(ctx: int, init_states, action_ids_u8, action_params_u16, lengths, hw_feats, subgraph_offsets,
                               k: int, scores_out, idx_out, stream=None) -> None:
    """wm_score_topk_host with uint8 type ids and uint16 parameters (HOST tensors).  include/wm.h."""
    import torch
    assert action_ids_u8.dtype == torch.uint8 and action_params_u16.dtype in (torch.uint16, torch.int16)
    B = int(lengths.numel())
    T_max = int(action_ids_u8.shape[1]) if action_ids_u8.dim() == 2 else 0
    S = int(subgraph_offsets.numel()) - 1
    _check(lib().wm_score_topk_host_compact(ctx, _ptr(init_states), _ptr(action_ids_u8), _ptr(action_params_u16), _ptr(lengths),
                                            _ptr(hw_feats), _ptr(subgraph_offsets), B, S, T_max, int(k),
                                            _ptr(scores_out), _ptr(idx_out), _stream(stream)))


def wm_last_kernel_ms(ctx: int, stream=None) -> float:
    ms = ctypes.c_float()
    _check(lib().wm_last_kernel_ms(ctx, _stream(stream), ctypes.byref(ms)))
    return float(ms.value)


def wm_path_reason(ctx: int) -> str:
    """Why the model is on the fp32 kernel ("" when a tcgen05 kernel takes it).  include/wm.h."""
    return lib().wm_path_reason(ctx).decode()


def wm_launch_count(ctx: Optional[int]) -> int:
    return int(lib().wm_launch_count(ctx))


def wm_launch_empty(stream=None) -> None:
    """One empty kernel on the stream (bench.py's launch-latency yardstick).  include/wm.h."""
    _check(lib().wm_launch_empty(_stream(stream)))

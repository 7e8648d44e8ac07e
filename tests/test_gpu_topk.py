"""GPU top-k (wm_topk) against the oracle's full sort: bit-exact indices (integer work)."""
import numpy as np
import pytest

import oracle
from wm_harness import gpu_topk

pytestmark = pytest.mark.gpu


def _check(scores, off, k):
    got = gpu_topk(scores, off, k)
    want = oracle.topk_segments(scores, off, k)
    np.testing.assert_array_equal(got, want)


def test_random_segments_various_k():
    rng = np.random.default_rng(0)
    for n_seg, n, k in [(1, 64, 8), (16, 2048, 64), (7, 1024, 128), (3, 16384, 32), (5, 1000, 1), (4, 50, 1024),
                        (2, 20000, 64), (1, 70000, 1024), (300, 37, 5)]:
        sc = rng.standard_normal(n_seg * n).astype(np.float32)
        off = (np.arange(n_seg + 1) * n).astype(np.int32)
        _check(sc, off, k)


def test_ragged_empty_and_short_segments():
    rng = np.random.default_rng(1)
    sizes = [0, 5, 0, 64, 1, 3000, 0, 17, 128, 0]
    off = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int32)
    sc = rng.standard_normal(off[-1]).astype(np.float32)
    for k in (1, 8, 64, 200):
        _check(sc, off, k)


def test_ties_and_special_values():
    rng = np.random.default_rng(2)
    # all equal: pure tie-break by index
    _check(np.zeros(5000, dtype=np.float32), np.array([0, 5000], dtype=np.int32), 64)
    # few distinct values: duplicates straddle the k-th place
    sc = rng.integers(0, 4, size=40000).astype(np.float32)
    _check(sc, np.array([0, 17000, 40000], dtype=np.int32), 100)
    # +-0, +-inf, NaN, denormals
    vals = np.array([0.0, -0.0, np.inf, -np.inf, np.nan, 1e-45, -1e-45, 1.0, -1.0, 3.4e38, -3.4e38], dtype=np.float32)
    sc = vals[rng.integers(0, len(vals), size=3000)]
    for k in (1, 7, 500, 1024):
        _check(sc, np.array([0, 1500, 3000], dtype=np.int32), k)
    # everything NaN
    _check(np.full(300, np.nan, dtype=np.float32), np.array([0, 300], dtype=np.int32), 16)
    # values differing only in the lowest mantissa bits (exercises the last radix pass)
    base = np.float32(1.0).view(np.uint32)
    sc = (base + rng.integers(0, 300, size=20000).astype(np.uint32)).view(np.float32)
    _check(sc, np.array([0, 20000], dtype=np.int32), 256)


def test_full_size_configs():
    """The five configs' segment shapes at full size (cfg 4/5: 128 x 16384)."""
    rng = np.random.default_rng(3)
    for S, n, k in [(1, 64, 8), (16, 2048, 64), (64, 1024, 128), (128, 16384, 32), (128, 16384, 64)]:
        sc = rng.standard_normal(S * n).astype(np.float32)
        off = (np.arange(S + 1) * n).astype(np.int32)
        got = gpu_topk(sc, off, k)
        # numpy reference at full size (the oracle's python sort is slow here): stable argsort of -score
        for s in range(0, S, max(1, S // 8)):
            seg = sc[off[s]:off[s + 1]]
            want = off[s] + np.argsort(-seg, kind="stable")[:k]
            np.testing.assert_array_equal(got[s], want)
        # sampled segments against the oracle itself
        np.testing.assert_array_equal(got[:1], oracle.topk_segments(sc[:n], off[:2], k))

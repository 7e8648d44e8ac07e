"""CPU-only checks of the boundary: libwm.so loads, exports every symbol include/wm.h declares, and the argument /
file-format errors that need no GPU behave as the header says.  No compute calls."""
import os
import re
import struct

import pytest

import gen
import paper_2606_09312_b200 as wm

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_2606_09312_b200 import build
    build.build()
    return wm.lib()


def test_exports_every_declared_symbol(L):
    hdr = open(os.path.join(ROOT, "include", "wm.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(wm_[a-z_]+)\s*\(", hdr))
    assert declared == set(wm.ABI_SYMBOLS), declared ^ set(wm.ABI_SYMBOLS)
    for s in declared:
        assert hasattr(L, s), s


def test_constants_match_header():
    hdr = open(os.path.join(ROOT, "include", "wm.h")).read()
    for name in ("WM_OK", "WM_ERR_ARG", "WM_ERR_IO", "WM_ERR_FORMAT", "WM_ERR_CUDA", "WM_ERR_UNSUPPORTED",
                 "WM_MAX_T", "WM_MAX_K", "WM_OPT_PATH", "WM_OPT_SORT"):
        m = re.search(rf"#define\s+{name}\s+(-?\d+)", hdr)
        assert m and int(m.group(1)) == getattr(wm, name), name


def test_topk_argument_errors(L):
    assert L.wm_topk(None, None, -1, 3, None, None) == wm.WM_ERR_ARG
    assert "S=-1" in wm.wm_last_error()
    assert L.wm_topk(None, None, 4, 0, None, None) == wm.WM_ERR_ARG
    assert L.wm_topk(None, None, 4, wm.WM_MAX_K + 1, None, None) == wm.WM_ERR_ARG
    assert L.wm_topk(None, None, 4, 8, None, None) == wm.WM_ERR_ARG       # null pointers with S > 0
    assert L.wm_topk(None, None, 0, 8, None, None) == wm.WM_OK            # S = 0 is a no-op


def test_null_ctx_errors(L):
    assert L.wm_rollout_score(None, None, None, None, None, None, None, None, 1, 1, 1, None) == wm.WM_ERR_ARG
    assert L.wm_rollout_latents(None, None, None, None, None, None, None, 1, 1, 1, None) == wm.WM_ERR_ARG
    assert "null ctx" in wm.wm_last_error()
    assert L.wm_rollout_score_from(None, None, None, None, None, None, None, None, None, None, 1, 1, 1, 1,
                                   None) == wm.WM_ERR_ARG
    assert L.wm_check(None, None) == wm.WM_ERR_ARG
    assert L.wm_set_option(None, 1, 0) == wm.WM_ERR_ARG
    L.wm_free(None)


def test_load_weights_io_and_format_errors(tmp_path):
    with pytest.raises(wm.WmError) as e:
        wm.wm_load_weights(str(tmp_path / "missing.wmw"))
    assert e.value.code == wm.WM_ERR_IO
    bad = tmp_path / "bad.wmw"
    bad.write_bytes(b"NOPE" + b"\0" * 100)
    with pytest.raises(wm.WmError) as e:
        wm.wm_load_weights(str(bad))
    assert e.value.code == wm.WM_ERR_FORMAT
    short = tmp_path / "short.wmw"
    short.write_bytes(b"WMW1" + struct.pack("<I", 1))
    with pytest.raises(wm.WmError) as e:
        wm.wm_load_weights(str(short))
    assert e.value.code == wm.WM_ERR_FORMAT
    # a valid header whose tensors are cut short, and one with trailing bytes
    cfg = gen.get_config(1)
    good = tmp_path / "good.wmw"
    gen.write_weight_file(str(good), cfg, gen.make_weights(cfg))
    raw = good.read_bytes()
    (tmp_path / "trunc.wmw").write_bytes(raw[:-8])
    with pytest.raises(wm.WmError) as e:
        wm.wm_load_weights(str(tmp_path / "trunc.wmw"))
    assert e.value.code == wm.WM_ERR_FORMAT and "truncated" in str(e.value)
    (tmp_path / "trail.wmw").write_bytes(raw + b"\0")
    with pytest.raises(wm.WmError) as e:
        wm.wm_load_weights(str(tmp_path / "trail.wmw"))
    assert e.value.code == wm.WM_ERR_FORMAT and "trailing" in str(e.value)
    # header field out of range (d = 0)
    hdr = bytearray(raw)
    struct.pack_into("<I", hdr, 4 + 4 * 4, 0)
    (tmp_path / "d0.wmw").write_bytes(bytes(hdr))
    with pytest.raises(wm.WmError) as e:
        wm.wm_load_weights(str(tmp_path / "d0.wmw"))
    assert e.value.code == wm.WM_ERR_FORMAT
    # version 2 (structured phi, NEXT row f2): unknown phi_kind, and more features than d_a has room for
    cfg8 = gen.get_config(8)
    v2 = tmp_path / "v2.wmw"
    gen.write_weight_file(str(v2), cfg8, gen.make_weights(cfg8))
    raw2 = bytearray(v2.read_bytes())
    assert struct.unpack_from("<I", raw2, 4)[0] == 2 and struct.unpack_from("<I", raw2, 80)[0] == 1
    struct.pack_into("<I", raw2, 80, 7)
    (tmp_path / "phi7.wmw").write_bytes(bytes(raw2))
    with pytest.raises(wm.WmError) as e:
        wm.wm_load_weights(str(tmp_path / "phi7.wmw"))
    assert e.value.code == wm.WM_ERR_FORMAT and "phi_kind" in str(e.value)
    from dataclasses import replace
    wide = replace(cfg8, n_types=40)            # 40 + 1 + 12 = 53 features > d_a = 32
    gen.write_weight_file(str(tmp_path / "wide.wmw"), wide, gen.make_weights(wide))
    with pytest.raises(wm.WmError) as e:
        wm.wm_load_weights(str(tmp_path / "wide.wmw"))
    assert e.value.code == wm.WM_ERR_UNSUPPORTED and "d_a" in str(e.value)
    struct.pack_into("<I", raw2, 4, 4)          # version 4 does not exist
    (tmp_path / "v4.wmw").write_bytes(bytes(raw2))
    with pytest.raises(wm.WmError) as e:
        wm.wm_load_weights(str(tmp_path / "v4.wmw"))
    assert e.value.code == wm.WM_ERR_FORMAT
    # version 3 (forest ranker, NEXT row f4): bad tree depth, a feature index past the feature vector, forest + mean phi
    cfg10 = gen.get_config(10)
    w10 = gen.make_weights(cfg10)
    v3 = tmp_path / "v3.wmw"
    gen.write_weight_file(str(v3), cfg10, w10)
    raw3 = bytearray(v3.read_bytes())
    assert struct.unpack_from("<I", raw3, 4)[0] == 3 and struct.unpack_from("<3I", raw3, 84) == (1, 32, 4)
    struct.pack_into("<I", raw3, 92, 13)
    (tmp_path / "deep.wmw").write_bytes(bytes(raw3))
    with pytest.raises(wm.WmError) as e:
        wm.wm_load_weights(str(tmp_path / "deep.wmw"))
    assert e.value.code == wm.WM_ERR_FORMAT and "ranker" in str(e.value)
    wbad = dict(w10); wbad["Tf"] = w10["Tf"].copy(); wbad["Tf"][3, 2] = cfg10.scorer_in
    gen.write_weight_file(str(tmp_path / "feat.wmw"), cfg10, wbad)
    try:
        wm.wm_load_weights(str(tmp_path / "feat.wmw"))
        raise AssertionError("a feature index past the feature vector was accepted")
    except wm.WmError as e2:      # FORMAT when the check is reached; CUDA when no device is there to load onto
        assert e2.code in (wm.WM_ERR_FORMAT, wm.WM_ERR_CUDA)
    mean_forest = replace(cfg10, phi_kind=0)
    gen.write_weight_file(str(tmp_path / "meanforest.wmw"), mean_forest, gen.make_weights(mean_forest))
    with pytest.raises(wm.WmError) as e:
        wm.wm_load_weights(str(tmp_path / "meanforest.wmw"))
    assert e.value.code == wm.WM_ERR_UNSUPPORTED


def test_load_weights_huge_header_is_a_format_error(tmp_path):
    """A header whose tensor sizes multiply past 2^32 (or ask for tens of GB) must be answered with WM_ERR_FORMAT before
    anything is allocated: sizes are summed in 64-bit and compared with the file size (include/wm.h: no exceptions, no aborts)."""
    cfg = gen.get_config(5).scaled(S=1, per_subgraph=8)
    from dataclasses import replace
    small = replace(cfg, d=16, d_a=8, scorer_widths=(8,), n_types=4, P=2, n_buckets=4, H=8)
    f = tmp_path / "b.wmw"
    gen.write_weight_file(str(f), small, gen.make_weights(small))
    raw = bytearray(f.read_bytes())
    # header layout: magic, version, kind, dtype, embed, d, d_a, hidden, n_types, P, n_buckets, H, n_lin, widths[6], eps
    fld = lambda i: 4 + 4 * i
    big = bytearray(raw)
    struct.pack_into("<I", big, fld(7), 1 << 20)      # n_types = 2^20
    struct.pack_into("<I", big, fld(8), 64)           # P = 64
    struct.pack_into("<I", big, fld(9), 4096)         # n_buckets = 4096: rows = 2^38 (wraps to 0 in 32 bits)
    (tmp_path / "wrap.wmw").write_bytes(bytes(big))
    with pytest.raises(wm.WmError) as e:
        wm.wm_load_weights(str(tmp_path / "wrap.wmw"))
    assert e.value.code == wm.WM_ERR_FORMAT and "truncated" in str(e.value)
    big = bytearray(raw)
    struct.pack_into("<I", big, fld(4), 65536)        # d = 65536
    struct.pack_into("<I", big, fld(5), 65536)        # d_a = 65536: W_g alone would be 34 GB
    (tmp_path / "wide.wmw").write_bytes(bytes(big))
    with pytest.raises(wm.WmError) as e:
        wm.wm_load_weights(str(tmp_path / "wide.wmw"))
    assert e.value.code == wm.WM_ERR_FORMAT and "truncated" in str(e.value)


def test_no_product_import_of_oracle():
    """The product path must not route through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2606_09312_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f

"""C-ABI checks that need no GPU: the library builds for sm_100a, loads, exports every symbol that
include/minipic.h declares, and rejects bad arguments on the host before any launch."""
import ctypes as C
import os
import re

import pytest

from paper_2606_13126_b200 import binding as mp
from paper_2606_13126_b200 import build as mpbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    mpbuild.build()
    return mp.lib()


def test_header_symbols_are_exported(lib):
    header = open(os.path.join(ROOT, "include", "minipic.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(minipic_[a-z0-9_]+)\s*\(", header))
    assert declared == set(mp.EXPORTS), declared ^ set(mp.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_sass_is_sm100a_only(lib):
    import subprocess
    out = subprocess.run(["/usr/local/cuda/bin/cuobjdump", "-lelf", mp.LIB_PATH], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_status_strings(lib):
    assert mp.minipic_status_string(0) == "MINIPIC_OK"
    assert mp.minipic_status_string(3) == "MINIPIC_ERR_WORKSPACE_TOO_SMALL"
    assert mp.minipic_status_string(5) == "MINIPIC_ERR_KERNEL_TIMEOUT"
    assert "UNKNOWN" in mp.minipic_status_string(99)


def _cfg(**kw):
    base = dict(num_q_heads=32, num_kv_heads=8, head_dim=128, num_blocks=64, dtype="bf16", rope_theta=5e5)
    base.update(kw)
    return mp.make_config(**base)


def test_host_side_validation_no_launch(lib):
    before = mp.minipic_launch_count()
    L = lib
    bad = [(_cfg(num_kv_heads=5), mp.MINIPIC_ERR_INVALID_ARG), (_cfg(head_dim=96), mp.MINIPIC_ERR_UNSUPPORTED),
           (_cfg(block_size=32), mp.MINIPIC_ERR_UNSUPPORTED), (_cfg(dtype=1, rope_theta=-1.0), mp.MINIPIC_ERR_INVALID_ARG),
           (_cfg(num_blocks=0), mp.MINIPIC_ERR_INVALID_ARG)]
    for cfg, code in bad:
        st = L.minipic_cache_write(C.byref(cfg), 16, 16, 16, 4, 16, 16, None)
        assert st == code
        assert mp.minipic_prefill_workspace_bytes(cfg, 1, 16) == 0
    good = _cfg()
    # null pointers / negative sizes / misaligned pointers
    assert L.minipic_cache_write(C.byref(good), None, 16, 16, 4, 16, 16, None) == mp.MINIPIC_ERR_INVALID_ARG
    assert L.minipic_cache_write(C.byref(good), 16, 16, 16, -1, 16, 16, None) == mp.MINIPIC_ERR_INVALID_ARG
    assert L.minipic_cache_write(C.byref(good), 8, 16, 16, 4, 16, 16, None) == mp.MINIPIC_ERR_INVALID_ARG
    assert L.minipic_cache_write(C.byref(good), None, None, None, 0, None, None, None) == mp.MINIPIC_OK   # empty write
    ws = mp.minipic_decode_workspace_bytes(good, 4, 1000)
    assert ws > 0
    args = [256] * 4 + [63] + [256] * 4 + [4, 1000, 256, 256, 256, ws - 1, None]
    assert L.minipic_decode_attention(C.byref(good), *args) == mp.MINIPIC_ERR_WORKSPACE_TOO_SMALL
    args[4] = 10    # max_blocks_per_req * 16 < max_kv_len
    assert L.minipic_decode_attention(C.byref(good), *args) == mp.MINIPIC_ERR_INVALID_ARG
    assert mp.minipic_launch_count() == before


def test_workspace_sizes_are_monotone(lib):
    cfg = _cfg()
    a = mp.minipic_decode_workspace_bytes(cfg, 8, 4096)
    b = mp.minipic_decode_workspace_bytes(cfg, 16, 4096)
    assert 0 < a <= b
    assert mp.minipic_prefill_workspace_bytes(cfg, 1, 128) <= mp.minipic_prefill_workspace_bytes(cfg, 4, 4096)
    assert mp.minipic_rope_table_bytes(cfg, 100) == 100 * 64 * 8


def test_binding_fails_loudly_without_library(monkeypatch, tmp_path):
    monkeypatch.setattr(mp, "_lib", None)
    monkeypatch.setattr(mp, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        mp.lib()

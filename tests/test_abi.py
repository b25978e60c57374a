"""The C-ABI library loads on a CPU-only box and exports every symbol include/lazy_attn.h declares;
host-side argument logic that needs no GPU (workspace sizing, status strings, config rejection)."""
import ctypes
import os
import re

import pytest

from paper_2606_04302_b200 import binding as B
from paper_2606_04302_b200 import build as lazy_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    lazy_build.build()
    return B.lib()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "lazy_attn.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lazy_[a-z_]+)\s*\(", text)))


def test_exports_match_header(lib):
    declared = _declared_symbols()
    assert set(declared) == set(B.EXPORTS), (declared, B.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_status_strings(lib):
    assert B.lazy_status_string(0) == "ok"
    for code in (-1, -2, -3, -4, -99):
        assert isinstance(B.lazy_status_string(code), str) and B.lazy_status_string(code)


def _cfg(**kw):
    base = dict(num_q_heads=32, num_kv_heads=8, head_dim=128, page_size=16, num_pages=1000, max_position=4096,
                max_reqs=64, max_pages_per_req=256, rope_theta=5e5, rope_style=0, dtype=0, flags=0, k_storage=0)
    base.update(kw)
    return B.LazyConfig(**base)


def test_workspace_bytes(lib):
    n = B.lazy_workspace_bytes(_cfg())
    table = 4096 * 64 * 8
    assert n >= table
    assert B.lazy_workspace_bytes(_cfg(max_position=8192)) - n == table       # table grows 512 B / position
    # unsupported / invalid configurations size to 0
    assert B.lazy_workspace_bytes(_cfg(head_dim=96)) == 0
    assert B.lazy_workspace_bytes(_cfg(page_size=32)) == 0
    assert B.lazy_workspace_bytes(_cfg(num_q_heads=30)) == 0
    assert B.lazy_workspace_bytes(_cfg(num_q_heads=32, num_kv_heads=2)) == 0   # group 16 > 8
    assert B.lazy_workspace_bytes(_cfg(num_pages=0)) == 0
    assert B.lazy_workspace_bytes(_cfg(dtype=2)) == 0
    assert B.lazy_workspace_bytes(_cfg(dtype=B.LAZY_KV_FP8_E4M3)) >= n          # FP8 pages: more split-KV partial slots
    assert B.lazy_workspace_bytes(_cfg(dtype=B.LAZY_KV_FP8_E4M3, k_storage=1)) == 0
    assert B.lazy_workspace_bytes(_cfg(dtype=B.LAZY_KV_FP8_E4M3, rope_style=2)) == 0          # no ALiBi on FP8 pages
    assert B.lazy_workspace_bytes(_cfg(dtype=B.LAZY_KV_FP8_E4M3, rope_style=1)) > 0


def test_create_rejects_without_touching_the_gpu(lib):
    out = ctypes.c_void_p()
    cfg = _cfg(head_dim=96)
    assert lib.lazy_create(ctypes.byref(cfg), None, 0, None, ctypes.byref(out)) == B.LAZY_ERR_UNSUPPORTED
    cfg = _cfg(max_reqs=0)
    assert lib.lazy_create(ctypes.byref(cfg), None, 0, None, ctypes.byref(out)) == B.LAZY_ERR_INVALID
    cfg = _cfg()
    assert lib.lazy_create(ctypes.byref(cfg), None, 0, None, ctypes.byref(out)) == B.LAZY_ERR_WORKSPACE
    assert lib.lazy_create(ctypes.byref(cfg), 256, 16, None, ctypes.byref(out)) == B.LAZY_ERR_WORKSPACE
    assert lib.lazy_create(None, None, 0, None, ctypes.byref(out)) == B.LAZY_ERR_INVALID
    # null handle on the data calls
    assert lib.lazy_cache_write(None, None, None, None, 0, None, None, None) == B.LAZY_ERR_INVALID
    assert lib.lazy_attn_decode(None, None, None, None, None, None, None, 0, None, None) == B.LAZY_ERR_INVALID
    assert lib.lazy_launch_count(None) == 0


def test_product_path_has_no_oracle_import():
    pkg = os.path.join(ROOT, "paper_2606_04302_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("oracle/", "").replace("oracle's", "") or f == "workloads.py" \
                    or "import oracle" not in src and "from oracle" not in src, f
                assert "import oracle" not in src and "from oracle" not in src, f

"""lazy_attn_decode_static: the decode entry point for callers that cannot allocate device memory.

Who needs it: code that runs inside a host framework which has taken all device memory for its own pool and forbids
raw cudaMalloc, serving loops where cudaMalloc is banned because it synchronises the device, and components that are
handed nothing but the inputs and outputs of one call.  Such a caller cannot give lazy_create a workspace, so this
entry point keeps the decode kernel's scratch (cos/sin table, split-KV partials, arrival counters) in a 48 MiB
device array that is part of the library image.

What is checked: its output against the ordinary lazy_create + lazy_attn_decode path on the same inputs, within the
tolerances of the other GPU tests (tests/gpu_util.py), on two calls in a row (the second with new queries, so a stale
result cannot pass), then on a call with a different configuration, which re-carves the shared array.  The file
name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the parity tests.
"""
import ctypes

import numpy as np
import pytest
import torch

from paper_2606_04302_b200 import binding as B
from paper_2606_04302_b200 import workloads as W
from paper_2606_04302_b200.runner import DeviceBatch


@pytest.fixture(scope="module", autouse=True)
def _lib():
    from paper_2606_04302_b200 import build
    build.build()
    B.lib()


def _config_of(batch, max_position=None) -> B.LazyConfig:
    sh = batch.shape
    R, pmax = batch.block_table.shape
    return B.LazyConfig(sh.num_q_heads, sh.num_kv_heads, sh.head_dim, sh.page_size, int(batch.k_pool.shape[0]),
                        max_position or batch.max_position, R, pmax, float(sh.rope_theta), B.LAZY_ROPE_HALF_SPLIT,
                        B.LAZY_KV_BF16, 0, B.LAZY_K_UNROTATED)


def _decode_both_ways(batch, q_variants):
    """Runs the batch's cache writes and its first decode step through the workspace path, then the same decode
    through lazy_attn_decode_static once per entry of q_variants (scale factors applied to the step's q).
    Returns [(expected, got), ...], one pair per variant."""
    from gpu_util import compare
    dev = DeviceBatch(batch)
    cfg = _config_of(batch)
    pairs = []
    try:
        step = None
        for st in batch.steps:                      # everything up to and including the first decode step
            dev.write(st)
            if st.kind == "decode":
                step = st
                break
            dev.attend(st)
        assert step is not None
        bt, pp = dev.tables_for(step)
        sl = step.seq_lens.to(dev.device)
        for f in q_variants:
            q = (step.q.float() * f).to(torch.bfloat16).to(dev.device)
            expected = torch.full_like(q, float("nan"))
            B.lazy_attn_decode(dev.handle, q, dev.k_pool, dev.v_pool, bt, pp, sl, expected)
            got = torch.full_like(q, float("nan"))
            B.lazy_attn_decode_static(cfg, q, dev.k_pool, dev.v_pool, bt, pp, sl, got)
            torch.cuda.synchronize()
            assert torch.isfinite(expected.float()).all()
            compare(got, expected.double().cpu().numpy(), f"{batch.name} static decode, q x {f}")
            pairs.append((expected, got))
    finally:
        dev.close()
    return pairs


@pytest.mark.gpu
def test_static_decode_matches_workspace_path_twice_in_a_row():
    pairs = _decode_both_ways(W.config2(scale=0.25), q_variants=(1.0, 2.0))
    # the two calls really computed different things (no stale buffer satisfied the second compare)
    assert not torch.equal(pairs[0][1], pairs[1][1])
    # a different configuration (4 kv heads, other table sizes) re-carves the same array; then the first one again
    _decode_both_ways(W.config5(scale=0.25), q_variants=(1.0,))
    _decode_both_ways(W.config2(scale=0.25), q_variants=(1.0,))


@pytest.mark.gpu
def test_static_decode_empty_batch_and_bad_counts():
    batch = W.config2(scale=0.1)
    cfg = _config_of(batch)
    L = B.lib()
    assert L.lazy_attn_decode_static(ctypes.byref(cfg), None, None, None, None, None, None, 0, None, None) == B.LAZY_OK
    assert L.lazy_attn_decode_static(ctypes.byref(cfg), None, None, None, None, None, None, cfg.max_reqs + 1, None,
                                     None) == B.LAZY_ERR_INVALID
    torch.cuda.synchronize()


def test_static_decode_rejects_what_does_not_fit():
    """Host-side checks, made before any CUDA call (so this runs on a box without a GPU too)."""
    L = B.lib()
    batch = W.config2(scale=0.1)
    fits = _config_of(batch)
    assert 0 < B.lazy_workspace_bytes(fits) <= B.LAZY_STATIC_SCRATCH_BYTES
    too_big = _config_of(batch, max_position=1 << 20)            # a 512 MiB cos/sin table
    assert B.lazy_workspace_bytes(too_big) > B.LAZY_STATIC_SCRATCH_BYTES
    rc = L.lazy_attn_decode_static(ctypes.byref(too_big), None, None, None, None, None, None, 1, None, None)
    assert rc == B.LAZY_ERR_STATIC_LIMIT
    assert "LAZY_STATIC_SCRATCH_BYTES" in B.lazy_status_string(rc)
    fp8 = _config_of(batch)
    fp8.dtype = B.LAZY_KV_FP8_E4M3
    assert L.lazy_attn_decode_static(ctypes.byref(fp8), None, None, None, None, None, None, 1, None, None) \
        == B.LAZY_ERR_UNSUPPORTED
    assert L.lazy_attn_decode_static(None, None, None, None, None, None, None, 1, None, None) == B.LAZY_ERR_INVALID

"""-m gpu parity tests for SURVEY.md 8.0 row f3 (section 3.5): RoPE-family variants --
interleaved pairing, frequency-scaled RoPE (per-pair frequency vector), softmax temperature, partial rotary --
through the C ABI against the fp64 oracle given the same variant."""
import math

import numpy as np
import pytest
import torch

from paper_2606_04302_b200 import binding as B
from paper_2606_04302_b200 import workloads as W

from gpu_util import run_and_compare

pytestmark = pytest.mark.gpu

FLAGS = [pytest.param(0, id="prod"), pytest.param(B.LAZY_FLAG_ROWWISE_KERNELS, id="rowwise")]


@pytest.fixture(scope="module", autouse=True)
def _lib():
    from paper_2606_04302_b200 import build
    build.build()
    B.lib()


def _batch(cfg, scale):
    return W.config1() if cfg == 1 else W.CONFIGS[cfg](scale=scale)


def _deinterleaved_docs(batch):
    """With LAZY_ROPE_INTERLEAVED the library keeps K rows de-interleaved.  Document pages that are pre-loaded
    (not written through lazy_cache_write in the test) must be uploaded in that order: the CPU copy the oracle reads
    stays in model order."""
    D = batch.shape.head_dim
    perm = torch.cat([torch.arange(0, D, 2), torch.arange(1, D, 2)])
    return batch.k_pool[..., perm].contiguous(), perm


@pytest.mark.parametrize("flags", FLAGS)
@pytest.mark.parametrize("cfg,scale", [(1, None), (2, 0.1), (3, 0.05), (5, 0.15)])
def test_interleaved_pairing(cfg, scale, flags):
    batch = _batch(cfg, scale)
    k_dev, perm = _deinterleaved_docs(batch)
    stats = run_and_compare(batch, flags=flags, dev_kw=dict(rope_style=B.LAZY_ROPE_INTERLEAVED, k_pool=k_dev),
                            oracle_kw=dict(rope_style=1), k_perm=perm)
    assert stats


def _llama31_style(theta, D, factor=8.0, low=1.0, high=4.0, orig=8192.0):
    base = theta ** (-2.0 * np.arange(D // 2) / D)
    wavelen = 2 * math.pi / base
    smooth = np.clip((orig / wavelen - low) / (high - low), 0.0, 1.0)
    return np.where(wavelen > orig / low, base / factor,
                    np.where(wavelen < orig / high, base, (1 - smooth) * base / factor + smooth * base))


@pytest.mark.parametrize("flags", FLAGS)
@pytest.mark.parametrize("cfg,scale", [(1, None), (2, 0.1), (3, 0.05)])
def test_scaled_frequencies_and_temperature(cfg, scale, flags):
    batch = _batch(cfg, scale)
    sh = batch.shape
    f = _llama31_style(sh.rope_theta, sh.head_dim)
    temp = 1.1 / math.sqrt(sh.head_dim)
    run_and_compare(batch, flags=flags, dev_kw=dict(inv_freq=f, softmax_scale=temp),
                    oracle_kw=dict(inv_freq=f, scale=temp))


@pytest.mark.parametrize("cfg,scale", [(1, None), (2, 0.1), (3, 0.05)])
def test_partial_rotary_and_restore_default(cfg, scale):
    """Pairs with frequency 0 are not rotated; passing NULL restores theta^(-2j/D)."""
    batch = _batch(cfg, scale)
    sh = batch.shape
    f = sh.rope_theta ** (-2.0 * np.arange(sh.head_dim // 2) / sh.head_dim)
    f[sh.head_dim // 4:] = 0.0
    run_and_compare(batch, dev_kw=dict(inv_freq=f), oracle_kw=dict(inv_freq=f))
    from paper_2606_04302_b200.runner import DeviceBatch
    dev = DeviceBatch(batch, inv_freq=f)
    B.lazy_set_rope_frequencies(dev.handle, None)
    ref = DeviceBatch(batch)
    try:
        for a, b in zip(dev.run_all(), ref.run_all()):
            if a is not None:
                assert torch.equal(a.view(torch.int16), b.view(torch.int16))
        with pytest.raises(B.LazyError):
            B.lazy_set_rope_frequencies(dev.handle, [-1.0] * (sh.head_dim // 2))
    finally:
        dev.close(); ref.close()


def _alibi_slopes(n_heads):
    return np.array([2.0 ** (-8.0 * (h + 1) / n_heads) for h in range(n_heads)])


@pytest.mark.parametrize("flags", FLAGS)
@pytest.mark.parametrize("cfg,scale", [(1, None), (2, 0.1), (3, 0.05), (4, 0.1), (5, 0.15)])
def test_alibi_bias(cfg, scale, flags):
    """ALiBi with deferred positions -- the bias uses the per-page logical positions, nothing is
    rotated, cached pages stay reusable at any offset (the configs share pages across requests and positions)."""
    batch = _batch(cfg, scale)
    slopes = _alibi_slopes(batch.shape.num_q_heads)
    run_and_compare(batch, flags=flags, dev_kw=dict(rope_style=B.LAZY_POS_ALIBI, alibi_slopes=slopes),
                    oracle_kw=dict(alibi_slopes=slopes))


def test_alibi_strong_slopes_and_shift_invariance():
    """Large slopes make the bias decide the softmax (a wrong sign or a wrong page position cannot hide);
    shifting every logical position leaves the outputs unchanged."""
    slopes = None
    outs = []
    for shift in (0, 4096):
        batch = W.config2(scale=0.1, pos_shift=shift)
        slopes = np.linspace(0.5, 0.01, batch.shape.num_q_heads)
        if shift == 0:
            run_and_compare(batch, dev_kw=dict(rope_style=B.LAZY_POS_ALIBI, alibi_slopes=slopes),
                            oracle_kw=dict(alibi_slopes=slopes), scale_abs_by_output=True)
        from paper_2606_04302_b200.runner import DeviceBatch
        dev = DeviceBatch(batch, rope_style=B.LAZY_POS_ALIBI, alibi_slopes=slopes)
        outs.append([o.float().cpu() for o in dev.run_all() if o is not None])
        dev.close()
    for a, b in zip(*outs):
        assert (a - b).abs().max().item() < 2e-3


def test_alibi_rejects_rotated_storage_and_wrong_style():
    cfg = B.LazyConfig(32, 8, 128, 16, 64, 4096, 4, 16, 5e5, B.LAZY_POS_ALIBI, 0, 0, B.LAZY_K_ABSOLUTE)
    assert B.lazy_workspace_bytes(cfg) == 0
    h = B.lazy_create(4, 1, 64, num_pages=8, max_position=256, max_reqs=1, max_pages_per_req=4, rope_theta=1e4)
    try:
        with pytest.raises(B.LazyError):
            B.lazy_set_alibi_slopes(h, [0.1, 0.2, 0.3, 0.4])
    finally:
        h.close()

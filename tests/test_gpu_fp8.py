"""-m gpu parity tests of LAZY_KV_FP8_E4M3 pages: the quantising lazy_cache_write bit for bit
against the oracle's, and the attention calls against the oracle's exact-dequantisation result.  The tolerance is the
bf16 contract (max abs 2e-2, mean abs 2e-3) and the same normalised gates: both sides start from identical codes and
scales, so the FP8 quantisation error itself is not part of the comparison."""
import numpy as np
import pytest
import torch

from paper_2606_04302_b200 import binding as B
from paper_2606_04302_b200 import workloads as W

pytestmark = pytest.mark.gpu

FLAGS = [pytest.param(0, id="prod"), pytest.param(B.LAZY_FLAG_ROWWISE_KERNELS, id="rowwise"),
         pytest.param(B.LAZY_FLAG_PREFILL_ONE_CTA, id="one_cta")]   # head_dim 128 prefill on single CTAs (A/B arm)


@pytest.fixture(scope="module", autouse=True)
def _lib():
    from paper_2606_04302_b200 import build
    build.build()
    B.lib()


def _run(batch, **kw):
    from gpu_util import run_and_compare_fp8
    return run_and_compare_fp8(batch, **kw)


@pytest.mark.parametrize("flags", FLAGS)
def test_fp8_config1_tiny(flags):
    stats = _run(W.config1(), flags=flags)
    assert len(stats) == 2
    assert all(s["max_abs"] < 5e-3 for s in stats), stats


@pytest.mark.parametrize("flags", FLAGS)
@pytest.mark.parametrize("cfg,scale", [(2, 0.25), (3, 0.07), (4, 0.25), (5, 0.25)])
def test_fp8_configs_reduced_full_compare(cfg, scale, flags):
    _run(W.CONFIGS[cfg](scale=scale), flags=flags)


@pytest.mark.parametrize("cfg", [2, 3, 4, 5])
def test_fp8_configs_peaked_queries(cfg):
    scale = {2: 0.1, 3: 0.07, 4: 0.25, 5: 0.25}[cfg]
    _run(W.CONFIGS[cfg](scale=scale, q_scale=4.0), scale_abs_by_output=True)


def test_fp8_cache_write_edge_rows():
    """All-zero rows (scale 1, codes 0), huge and tiny magnitudes, skipped slots, a partially written page."""
    from oracle import oracle as O
    torch.manual_seed(3)
    Hkv, D, P, T = 2, 128, 16, 40
    dev = torch.device("cuda")
    h = B.lazy_create(4, Hkv, D, num_pages=4, max_position=256, max_reqs=1, max_pages_per_req=4, rope_theta=1e4,
                      dtype=B.LAZY_KV_FP8_E4M3, device=dev)
    kc = torch.full((4, Hkv, P, D), 0x7f, dtype=torch.uint8, device=dev)
    vc = torch.full((4, Hkv, P, D), 0x7f, dtype=torch.uint8, device=dev)
    ks = torch.full((4, Hkv, P), float("nan"), dtype=torch.float32, device=dev)
    vs = torch.full((4, Hkv, P), float("nan"), dtype=torch.float32, device=dev)
    B.lazy_set_kv_scales(h, ks, vs)
    k = torch.randn(T, Hkv, D).to(torch.bfloat16)
    v = torch.randn(T, Hkv, D).to(torch.bfloat16)
    k[0] = 0
    v[1] = 0
    k[2] *= 1e30
    v[3] *= 1e-30
    k[4, 0, 5] = 3e38
    v[5] = torch.where(torch.rand(Hkv, D) < 0.5, 1.0, -1.0).to(torch.bfloat16) * 7
    slots = torch.arange(T, dtype=torch.int64) + 5
    slots[7] = -1
    B.lazy_cache_write(h, k.to(dev), v.to(dev), slots.to(dev), kc, vc)
    torch.cuda.synchronize()
    pools = O.Fp8Pools(4, Hkv, P, D)
    O.cache_write_fp8(k, v, slots.numpy(), pools)
    assert np.array_equal(kc.cpu().numpy(), pools.k_codes)
    assert np.array_equal(vc.cpu().numpy(), pools.v_codes)
    assert np.array_equal(ks.cpu().numpy().view(np.uint32), pools.k_scale.view(np.uint32))
    assert np.array_equal(vs.cpu().numpy().view(np.uint32), pools.v_scale.view(np.uint32))
    h.close()


def test_fp8_cache_write_non_finite_rows_read_back_as_nan():
    """include/lazy_attn.h (LAZY_KV_FP8_E4M3): inputs must be finite; a row with Inf or NaN is stored so that it reads
    back as NaN instead of being silently flattened -- Inf: scale = inf and code x inf = NaN for every element; NaN:
    finite scale from the other elements, the element itself gets the E4M3 NaN code.  Neighbouring rows are untouched."""
    Hkv, D, P = 1, 128, 16
    dev = torch.device("cuda")
    h = B.lazy_create(4, Hkv, D, num_pages=2, max_position=256, max_reqs=1, max_pages_per_req=2, rope_theta=1e4,
                      dtype=B.LAZY_KV_FP8_E4M3, device=dev)
    kc = torch.zeros((2, Hkv, P, D), dtype=torch.uint8, device=dev)
    vc = torch.zeros((2, Hkv, P, D), dtype=torch.uint8, device=dev)
    ks = torch.ones((2, Hkv, P), dtype=torch.float32, device=dev)
    vs = torch.ones((2, Hkv, P), dtype=torch.float32, device=dev)
    B.lazy_set_kv_scales(h, ks, vs)
    g = torch.Generator().manual_seed(9)
    k = torch.randn(3, Hkv, D, generator=g).to(torch.bfloat16)
    v = torch.randn(3, Hkv, D, generator=g).to(torch.bfloat16)
    k[0, 0, 7] = float("inf")
    v[1, 0, 100] = float("nan")
    B.lazy_cache_write(h, k.to(dev), v.to(dev), torch.arange(3, dtype=torch.int64, device=dev), kc, vc)
    torch.cuda.synchronize()
    deq = lambda c, s: c.cpu().view(torch.float8_e4m3fn).float() * s.cpu()[..., None]
    kd, vd = deq(kc, ks), deq(vc, vs)
    assert torch.isinf(ks[0, 0, 0]) and torch.isnan(kd[0, 0, 0]).all()               # Inf row: every element NaN
    assert torch.isfinite(vs[0, 0, 1]) and torch.isnan(vd[0, 0, 1, 100])             # NaN element stays NaN ...
    assert torch.isfinite(vd[0, 0, 1]).sum() == D - 1                                #   ... the rest of its row is kept
    assert torch.isfinite(kd[0, 0, 1:3]).all() and torch.isfinite(vd[0, 0, [0, 2]]).all()   # neighbours untouched
    h.close()


def test_fp8_needs_scales_and_rejects_unsupported_modes():
    dev = torch.device("cuda")
    with pytest.raises(B.LazyError):
        B.lazy_create(4, 1, 64, num_pages=4, max_position=256, max_reqs=1, max_pages_per_req=4, rope_theta=1e4,
                      dtype=B.LAZY_KV_FP8_E4M3, k_storage=B.LAZY_K_STORED_POS, device=dev)
    h = B.lazy_create(4, 1, 64, num_pages=4, max_position=256, max_reqs=1, max_pages_per_req=4, rope_theta=1e4,
                      dtype=B.LAZY_KV_FP8_E4M3, device=dev)
    kc = torch.zeros(4, 1, 16, 64, dtype=torch.uint8, device=dev)
    k = torch.zeros(1, 1, 64, dtype=torch.bfloat16, device=dev)
    with pytest.raises(B.LazyError) as e:
        B.lazy_cache_write(h, k, k, torch.zeros(1, dtype=torch.int64, device=dev), kc, kc)
    assert e.value.status == B.LAZY_ERR_INVALID
    h.close()
    hb = B.lazy_create(4, 1, 64, num_pages=4, max_position=256, max_reqs=1, max_pages_per_req=4, rope_theta=1e4,
                       device=dev)
    with pytest.raises(B.LazyError) as e:
        B.lazy_set_kv_scales(hb, torch.zeros(64, device=dev), torch.zeros(64, device=dev))
    assert e.value.status == B.LAZY_ERR_UNSUPPORTED
    hb.close()


@pytest.mark.parametrize("cfg,rows", [(2, 0), (3, 96), (4, 0), (5, 64)])
def test_fp8_configs_full_size_sampled(cfg, rows):
    """BASELINE.json sizes on FP8 pages, the launch configurations bench.py's fp8 legs time; the oracle on sampled
    query rows (decode configs are compared in full).  Same margins as the bf16 full-size test: the kernels' own
    error (f16 / bf16 rounding of the rotated operands and of P) is what is measured, not the quantisation."""
    stats = _run(W.CONFIGS[cfg](), sample_rows=rows, seed=cfg)
    max_b, mean_b = {2: (2e-3, 2e-4), 3: (2e-3, 2e-4), 4: (1e-3, 1e-4), 5: (1.5e-2, 5e-4)}[cfg]
    assert all(s["max_abs"] < max_b and s["mean_abs"] < mean_b for s in stats), stats


def test_fp8_v_scale_outlier_tokens():
    """V rows whose magnitudes differ by 2^+-20 inside one request (and inside one page): the decode kernel's running
    reference V scale must re-reference O in both directions; the prefill kernel folds the scale into the bf16 tile."""
    b = W.config2(scale=0.1)
    g = torch.Generator().manual_seed(5)
    v = b.v_pool.float()
    fin = torch.isfinite(v).all(dim=-1, keepdim=True)
    e = torch.randint(-20, 21, v.shape[:-1] + (1,), generator=g).float()
    sparse = torch.rand(v.shape[:-1] + (1,), generator=g) < 0.05
    b.v_pool = torch.where(fin & sparse, v * torch.exp2(e), v).to(torch.bfloat16)
    _run(b, scale_abs_by_output=True, gates=dict(rel_rms=2e-2))


def test_fp8_mixed_call_matches_oracle():
    """lazy_attn_mixed on FP8 pages at 4 kv heads: the one-launch FP8 step (mixed_step_fp8_kernel: 12-warp FP8 decode
    body + FP8 pair prefill body in one grid)."""
    from oracle import oracle as O
    from paper_2606_04302_b200.runner import DeviceBatch
    from gpu_util import compare
    batch = W.config5(scale=0.2)
    pre, dec = batch.steps[0], batch.steps[1]
    dev = DeviceBatch(batch, dtype=B.LAZY_KV_FP8_E4M3)
    d = dev.device
    pools = O.quantize_pool_fp8(batch.k_pool, batch.v_pool)
    try:
        dev.write(pre); dev.write(dec)
        ref_p = O.run_step_fp8(batch, pre, pools)
        ref_d = O.run_step_fp8(batch, dec, pools)
        bt_p, pp_p = dev.tables_for(pre)
        bt_d, pp_d = dev.tables_for(dec)
        out_p = torch.zeros_like(pre.q, device=d)
        out_d = torch.zeros_like(dec.q, device=d)
        max_q = int((pre.cu_q_lens[1:] - pre.cu_q_lens[:-1]).max())
        B.lazy_attn_mixed(dev.handle, dev.k_pool, dev.v_pool, q_prefill=pre.q.to(d), block_table_prefill=bt_p,
                          page_logical_pos_prefill=pp_p, seq_lens_prefill=pre.seq_lens.to(d),
                          cu_q_lens=pre.cu_q_lens.to(d), max_q_len=max_q, out_prefill=out_p, q_decode=dec.q.to(d),
                          block_table_decode=bt_d, page_logical_pos_decode=pp_d, seq_lens_decode=dec.seq_lens.to(d),
                          out_decode=out_d)
        torch.cuda.synchronize()
        compare(out_p, ref_p, "fp8 mixed prefill")
        compare(out_d, ref_d, "fp8 mixed decode")
    finally:
        dev.close()


# ---- edge cases on FP8 pages: ragged lengths, partial (poisoned) last pages, repeated pages, position gaps, keys
# positioned above the query, every head grouping of the 12-warp and 8-warp decode cuts, empty requests
from test_gpu_edges import _custom, SH128, SH64, SH7   # noqa: E402

SH2 = W.LazyShape(8, 2, 128, 1.0e4)      # 2 kv heads: 6 pages per stage in the 12-warp cut
SH1 = W.LazyShape(8, 1, 128, 1.0e4)      # 1 kv head: 12 pages per stage
SH16 = W.LazyShape(32, 16, 128, 5.0e5)   # 16 kv heads: 4 head groups (grid.y = 4)
SH64B = W.LazyShape(32, 8, 64, 1.0e4)    # head_dim 64 with 8 kv heads (64-byte swizzled rows, two head groups)
DFLAGS = [pytest.param(0, id="w12"), pytest.param(B.LAZY_FLAG_FP8_DECODE_8_WARPS, id="w8")]


@pytest.mark.parametrize("flags", DFLAGS)
@pytest.mark.parametrize("shape", [SH128, SH7, SH2, SH1, SH16, SH64, SH64B],
                         ids=["g4", "g7", "hkv2", "hkv1", "hkv16", "d64", "d64hkv8"])
def test_fp8_ragged_decode(shape, flags):
    seq = [1, 2, 15, 16, 17, 31, 33, 100, 257, 640, 1000, 3]
    _run(_custom(shape, seq, [1] * len(seq), seed=21, kind="decode"), flags=flags)


@pytest.mark.parametrize("flags", [pytest.param(0, id="pairs"), pytest.param(B.LAZY_FLAG_PREFILL_ONE_CTA, id="one_cta")])
@pytest.mark.parametrize("shape", [SH128, SH64, SH7, SH2], ids=["g4d128", "g4d64", "g7d128", "hkv2"])
def test_fp8_ragged_prefill(shape, flags):
    seq = [5, 16, 200, 129, 300, 47, 1]
    qls = [5, 3, 200, 1, 130, 47, 1]
    _run(_custom(shape, seq, qls, seed=22), flags=flags)


def test_fp8_zero_length_repeated_pages_gaps():
    _run(_custom(SH128, [0, 40, 0], [1, 1, 1], seed=23, kind="decode"))
    _run(_custom(SH128, [33, 0, 20], [4, 0, 20], seed=24))
    _run(_custom(SH128, [200, 333], [1, 1], seed=25, repeat_pages=True, kind="decode"))
    _run(_custom(SH128, [200, 333], [8, 70], seed=26, repeat_pages=True, pos_gap=1000))
    _run(_custom(SH128, [77, 160], [1, 1], seed=27, pos_gap=4096, unaligned_pos=True, kind="decode"))


def test_fp8_key_positions_above_the_query():
    """Pages positioned AFTER the query token (negative page offset: the sign path of the q re-rotation)."""
    b = _custom(SH128, [100, 260], [1, 1], seed=28, kind="decode")
    pp = b.page_logical_pos.clone()
    pp[:, 0:3] += 5000                               # the first pages sit far above the query's position
    b.page_logical_pos = pp
    _run(b)
    b2 = _custom(SH128, [100, 260], [10, 40], seed=29)
    pp = b2.page_logical_pos.clone()
    pp[:, 1:3] += 7000
    b2.page_logical_pos = pp
    _run(b2)


def test_fp8_many_requests_split_over_launches():
    """More requests than one decode launch holds in shared memory (2048)."""
    n = 2100
    _run(_custom(W.LazyShape(8, 4, 128, 1.0e4), [3 + (i % 40) for i in range(n)], [1] * n, seed=30, kind="decode"))


@pytest.mark.parametrize("decode_sms", [0, 8, 148])
def test_fp8_mixed_one_launch_8_kv_heads(decode_sms):
    """The one-launch FP8 mixed step with 8 kv heads (two head groups alternate over the decode CTAs): a prefill chunk
    of the last 8 tokens of every request and the decode of the same requests, in one call, against the oracle."""
    from oracle import oracle as O
    from paper_2606_04302_b200.runner import DeviceBatch
    from gpu_util import compare
    batch = W.config2(scale=0.1)
    assert batch.shape.num_kv_heads == 8
    dec = [s for s in batch.steps if s.kind == "decode"][0]
    dev = DeviceBatch(batch, dtype=B.LAZY_KV_FP8_E4M3)
    d = dev.device
    pools = O.quantize_pool_fp8(batch.k_pool, batch.v_pool)
    try:
        for st in batch.steps:                       # every cache write of the batch (question tokens, decode token)
            dev.write(st)
            if st.k_new is not None:
                O.cache_write_fp8(st.k_new, st.v_new, st.slot_mapping.numpy(), pools)
        R = dec.seq_lens.shape[0]
        nq = 8
        g = torch.Generator().manual_seed(77)
        qp = torch.randn(R * nq, batch.shape.num_q_heads, batch.shape.head_dim, generator=g).to(torch.bfloat16)
        pre = W.Step(kind="prefill", q=qp, seq_lens=dec.seq_lens.clone(),
                     cu_q_lens=(nq * torch.arange(R + 1)).to(torch.int32), req_ids=dec.req_ids)
        ref_p = O.run_step_fp8(batch, pre, pools)
        ref_d = O.run_step_fp8(batch, W.dataclasses.replace(dec, k_new=None, v_new=None, slot_mapping=None), pools)
        bt, pp = dev.tables_for(dec)
        out_p = torch.zeros_like(qp, device=d)
        out_d = torch.zeros_like(dec.q, device=d)
        for _ in range(2):
            B.lazy_attn_mixed(dev.handle, dev.k_pool, dev.v_pool, q_prefill=qp.to(d), block_table_prefill=bt,
                              page_logical_pos_prefill=pp, seq_lens_prefill=pre.seq_lens.to(d),
                              cu_q_lens=pre.cu_q_lens.to(d), max_q_len=nq, out_prefill=out_p, q_decode=dec.q.to(d),
                              block_table_decode=bt, page_logical_pos_decode=pp, seq_lens_decode=dec.seq_lens.to(d),
                              out_decode=out_d, decode_sms=decode_sms)
        torch.cuda.synchronize()
        compare(out_p, ref_p, "fp8 mixed prefill, 8 kv heads")
        compare(out_d, ref_d, "fp8 mixed decode, 8 kv heads")
        assert np.array_equal(dev.k_pool.cpu().numpy(), pools.k_codes)       # read path is read-only
    finally:
        dev.close()


@pytest.mark.parametrize("cfg,scale", [(1, None), (2, 0.1), (3, 0.05), (5, 0.2)])
def test_fp8_scaled_frequencies_and_temperature(cfg, scale):
    """Frequency-scaled RoPE (Llama-3.1 style per-pair frequencies, lazy_set_rope_frequencies) and a softmax temperature on
    FP8 pages: every FP8 kernel reads its angles through the rebuilt table and its scale from the handle."""
    import math
    from test_gpu_posvariants import _llama31_style
    batch = W.CONFIGS[cfg]() if scale is None else W.CONFIGS[cfg](scale=scale)
    sh = batch.shape
    f = _llama31_style(sh.rope_theta, sh.head_dim)
    temp = 1.1 / math.sqrt(sh.head_dim)
    _run(batch, dev_kw=dict(inv_freq=f, softmax_scale=temp), oracle_kw=dict(inv_freq=f, scale=temp))


@pytest.mark.parametrize("flags", [pytest.param(0, id="prod"), pytest.param(B.LAZY_FLAG_ROWWISE_KERNELS, id="rowwise")])
@pytest.mark.parametrize("cfg,scale", [(1, None), (2, 0.1), (3, 0.05), (5, 0.2)])
def test_fp8_interleaved_pairing(cfg, scale, flags):
    """LAZY_ROPE_INTERLEAVED on FP8 pages: lazy_cache_write de-interleaves the K row before quantising it (same values,
    same scale, codes in the stored order), the kernels de-interleave q on load."""
    batch = W.CONFIGS[cfg]() if scale is None else W.CONFIGS[cfg](scale=scale)
    D = batch.shape.head_dim
    perm = np.concatenate([np.arange(0, D, 2), np.arange(1, D, 2)])
    _run(batch, flags=flags, dev_kw=dict(rope_style=B.LAZY_ROPE_INTERLEAVED), oracle_kw=dict(rope_style=1), k_perm=perm)


@pytest.mark.parametrize("log2_q", [16, -20])
@pytest.mark.parametrize("cfg,scale", [(1, None), (2, 0.1), (5, 0.2)])
def test_fp8_q_far_outside_the_f16_range(cfg, scale, log2_q):
    """The FP8 decode kernel packs the rotated q to f16 for its MMAs.  q scaled by 2^16 puts the rotated values beyond
    f16's largest finite number (65504 -> inf -> NaN after the softmax), q scaled by 2^-20 below its smallest normal
    one (6e-5 -> precision lost, then flushed); the bf16-page kernels take both.  The kernel therefore normalises q by
    a power of two per (request, kv head) and folds the inverse into the score scale.  Here the softmax temperature is
    scaled the other way, so the scores -- and the oracle's answer -- are those of the unscaled batch and the usual
    gates apply."""
    import math
    kw = dict(q_scale=2.0 ** log2_q)
    batch = W.CONFIGS[cfg](**kw) if scale is None else W.CONFIGS[cfg](scale=scale, **kw)
    temp = 2.0 ** (-log2_q) / math.sqrt(batch.shape.head_dim)
    stats = _run(batch, dev_kw=dict(softmax_scale=temp), oracle_kw=dict(scale=temp))
    assert stats

"""-m gpu: lazy_attn_mixed -- prefill of the cache-miss documents and decode of the running
requests issued together, decode confined to a subset of the SMs on a forked stream.  Results must equal the oracle
(and the two separate calls up to the split-KV summation order, which depends on the decode grid)."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2606_04302_b200 import binding as B
from paper_2606_04302_b200 import workloads as W
from paper_2606_04302_b200.runner import DeviceBatch

from gpu_util import compare

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _lib():
    from paper_2606_04302_b200 import build
    build.build()
    B.lib()


@pytest.mark.parametrize("decode_sms", [0, 8, 148, 1000])
def test_mixed_step_matches_oracle_and_separate_calls(decode_sms):
    batch = W.config5(scale=0.2)
    pre, dec = batch.steps[0], batch.steps[1]
    assert pre.kind == "prefill" and dec.kind == "decode"
    dev = DeviceBatch(batch)
    d = dev.device
    k_ref, v_ref = batch.k_pool.clone(), batch.v_pool.clone()
    try:
        dev.write(pre); dev.write(dec)
        ref_p = O.run_step(batch, pre, k_ref, v_ref)
        ref_d = O.run_step(batch, dec, k_ref, v_ref)
        sep_p, sep_d = dev.attend(pre), dev.attend(dec)
        bt_p, pp_p = dev.tables_for(pre)
        bt_d, pp_d = dev.tables_for(dec)
        out_p = torch.zeros_like(pre.q, device=d)
        out_d = torch.zeros_like(dec.q, device=d)
        max_q = int((pre.cu_q_lens[1:] - pre.cu_q_lens[:-1]).max())
        for _ in range(2):
            B.lazy_attn_mixed(dev.handle, dev.k_pool, dev.v_pool, q_prefill=pre.q.to(d), block_table_prefill=bt_p,
                              page_logical_pos_prefill=pp_p, seq_lens_prefill=pre.seq_lens.to(d),
                              cu_q_lens=pre.cu_q_lens.to(d), max_q_len=max_q, out_prefill=out_p, q_decode=dec.q.to(d),
                              block_table_decode=bt_d, page_logical_pos_decode=pp_d, seq_lens_decode=dec.seq_lens.to(d),
                              out_decode=out_d, decode_sms=decode_sms)
        torch.cuda.synchronize()
        compare(out_p, ref_p, "mixed prefill")
        compare(out_d, ref_d, "mixed decode")
        assert torch.equal(out_p.view(torch.int16), sep_p.view(torch.int16))       # same kernel, same grid
        assert (out_d.float() - sep_d.float()).abs().max().item() < 2e-3
        assert torch.equal(dev.k_pool.cpu().view(torch.int16), k_ref.view(torch.int16))
    finally:
        dev.close()


def test_mixed_step_full_size_cfg5_sampled():
    """BASELINE.json configs[4] at full size through the call bench.py times for it (lazy_attn_mixed, default SM
    share): all decode rows and ALL prefill rows against the oracle (30 GFLOP: seconds on the host cores)."""
    batch = W.config5()
    pre, dec = batch.steps[0], batch.steps[1]
    dev = DeviceBatch(batch)
    d = dev.device
    k_ref, v_ref = batch.k_pool.clone(), batch.v_pool.clone()
    try:
        dev.write(pre); dev.write(dec)
        rows = None
        ref_p = O.run_step(batch, pre, k_ref, v_ref)
        ref_d = O.run_step(batch, dec, k_ref, v_ref)
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
        compare(out_p, ref_p, "cfg5 mixed prefill", rows=rows)
        compare(out_d, ref_d, "cfg5 mixed decode")
    finally:
        dev.close()


def _mixed_8_kv_heads(batch, decode_sms, interleaved, sample_rows=0):
    """Llama-3-8B layer shape (Hq 32 / Hkv 8 / D 128, configs 2-4): a prefill chunk of the last 8 tokens of every request
    and the decode of the same requests in ONE lazy_attn_mixed call -> mixed_step_kernel<8> (two head groups alternate
    over the decode CTAs).  Both halves against the oracle element by element."""
    assert batch.shape.num_kv_heads == 8 and batch.shape.head_dim == 128
    dec = [s for s in batch.steps if s.kind == "decode"][0]
    dev_kw, oracle_kw, perm = {}, {}, None
    if interleaved:
        D = batch.shape.head_dim
        perm = torch.cat([torch.arange(0, D, 2), torch.arange(1, D, 2)])
        dev_kw = dict(rope_style=B.LAZY_ROPE_INTERLEAVED, k_pool=batch.k_pool[..., perm].contiguous())
        oracle_kw = dict(rope_style=1)
    dev = DeviceBatch(batch, **dev_kw)
    d = dev.device
    k_ref, v_ref = batch.k_pool.clone(), batch.v_pool.clone()
    try:
        for st in batch.steps:                       # every cache write of the batch (question tokens, decode token)
            dev.write(st)
            if st.k_new is not None:
                O.cache_write(st.k_new, st.v_new, st.slot_mapping.numpy(), k_ref, v_ref, batch.shape.page_size)
        R = dec.seq_lens.shape[0]
        nq = 8
        g = torch.Generator().manual_seed(78)
        qp = torch.randn(R * nq, batch.shape.num_q_heads, batch.shape.head_dim, generator=g).to(torch.bfloat16)
        pre = W.Step(kind="prefill", q=qp, seq_lens=dec.seq_lens.clone(),
                     cu_q_lens=(nq * torch.arange(R + 1)).to(torch.int32), req_ids=dec.req_ids)
        sel = rows = None
        if sample_rows and qp.shape[0] > sample_rows:
            rows = np.sort(np.random.default_rng(5).choice(qp.shape[0], size=sample_rows, replace=False))
            sel = np.zeros(qp.shape[0], dtype=np.uint8)
            sel[rows] = 1
        ref_p = O.run_step(batch, pre, k_ref, v_ref, row_select=sel, **oracle_kw)
        ref_d = O.run_step(batch, W.dataclasses.replace(dec, k_new=None, v_new=None, slot_mapping=None), k_ref, v_ref,
                           **oracle_kw)
        bt, pp = dev.tables_for(dec)
        out_p = torch.full_like(qp, float("nan"), device=d)
        out_d = torch.full_like(dec.q, float("nan"), device=d)
        launches = dev.handle.launch_count()
        for _ in range(2):
            B.lazy_attn_mixed(dev.handle, dev.k_pool, dev.v_pool, q_prefill=qp.to(d), block_table_prefill=bt,
                              page_logical_pos_prefill=pp, seq_lens_prefill=pre.seq_lens.to(d),
                              cu_q_lens=pre.cu_q_lens.to(d), max_q_len=nq, out_prefill=out_p, q_decode=dec.q.to(d),
                              block_table_decode=bt, page_logical_pos_decode=pp, seq_lens_decode=dec.seq_lens.to(d),
                              out_decode=out_d, decode_sms=decode_sms)
        torch.cuda.synchronize()
        assert dev.handle.launch_count() - launches == 2          # ONE launch per call: the fused kernel really ran
        compare(out_p, ref_p, "mixed prefill, 8 kv heads", rows=rows)
        compare(out_d, ref_d, "mixed decode, 8 kv heads")
        k_expect = k_ref if perm is None else k_ref[..., perm]
        assert torch.equal(dev.k_pool.cpu().view(torch.int16), k_expect.view(torch.int16))   # read path is read-only
    finally:
        dev.close()


@pytest.mark.parametrize("interleaved", [False, True], ids=["half_split", "interleaved"])
@pytest.mark.parametrize("decode_sms", [0, 8, 148])
def test_mixed_one_launch_8_kv_heads(decode_sms, interleaved):
    _mixed_8_kv_heads(W.config2(scale=0.1), decode_sms, interleaved)


def test_mixed_one_launch_8_kv_heads_full_size_sampled():
    """BASELINE.json configs[1] at full size (64 requests x 2,640 tokens) as the decode half, an 8-token chunk per
    request as the prefill half; every decode row and 96 sampled prefill rows against the oracle."""
    _mixed_8_kv_heads(W.config2(), 0, False, sample_rows=96)


def test_mixed_one_launch_4_kv_heads_interleaved():
    """LAZY_ROPE_INTERLEAVED through the one-launch path at 4 kv heads (mixed_step_kernel<4>, q de-interleaved on load
    in both halves)."""
    batch = W.config5(scale=0.2)
    pre, dec = batch.steps[0], batch.steps[1]
    D = batch.shape.head_dim
    perm = torch.cat([torch.arange(0, D, 2), torch.arange(1, D, 2)])
    dev = DeviceBatch(batch, rope_style=B.LAZY_ROPE_INTERLEAVED, k_pool=batch.k_pool[..., perm].contiguous())
    d = dev.device
    k_ref, v_ref = batch.k_pool.clone(), batch.v_pool.clone()
    try:
        dev.write(pre); dev.write(dec)
        ref_p = O.run_step(batch, pre, k_ref, v_ref, rope_style=1)
        ref_d = O.run_step(batch, dec, k_ref, v_ref, rope_style=1)
        bt_p, pp_p = dev.tables_for(pre)
        bt_d, pp_d = dev.tables_for(dec)
        out_p = torch.full_like(pre.q, float("nan"), device=d)
        out_d = torch.full_like(dec.q, float("nan"), device=d)
        max_q = int((pre.cu_q_lens[1:] - pre.cu_q_lens[:-1]).max())
        launches = dev.handle.launch_count()
        B.lazy_attn_mixed(dev.handle, dev.k_pool, dev.v_pool, q_prefill=pre.q.to(d), block_table_prefill=bt_p,
                          page_logical_pos_prefill=pp_p, seq_lens_prefill=pre.seq_lens.to(d),
                          cu_q_lens=pre.cu_q_lens.to(d), max_q_len=max_q, out_prefill=out_p, q_decode=dec.q.to(d),
                          block_table_decode=bt_d, page_logical_pos_decode=pp_d, seq_lens_decode=dec.seq_lens.to(d),
                          out_decode=out_d)
        torch.cuda.synchronize()
        assert dev.handle.launch_count() - launches == 1
        compare(out_p, ref_p, "mixed prefill, interleaved")
        compare(out_d, ref_d, "mixed decode, interleaved")
    finally:
        dev.close()

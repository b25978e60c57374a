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

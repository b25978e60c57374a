"""-m gpu: repeated-run bitwise determinism of the CTA-pair prefill kernel (bf16 and FP8 pages) and of the one-launch
mixed step's prefill half.  In the pair kernel the peer CTA publishes rotated K / dequantised V / rotated Q tiles to the
LEADER's MMA thread through remote mbarrier arrivals (cluster-scope release / acquire since round 3) and P tiles in
TMEM through CTA-scope arrivals ordered by tcgen05 fences (DESIGN.md 6.2 records that residual formal gap).  A stale
operand read would show up as a run whose output differs from the first: 1000 back-to-back runs per case, with a side
stream hammering the L2 and the SMs, must be bit-identical."""
import pytest
import torch

from paper_2606_04302_b200 import binding as B
from paper_2606_04302_b200 import workloads as W
from paper_2606_04302_b200.runner import DeviceBatch

pytestmark = pytest.mark.gpu

RUNS = 1000


@pytest.fixture(scope="module", autouse=True)
def _lib():
    from paper_2606_04302_b200 import build
    build.build()
    B.lib()


@pytest.mark.parametrize("dtype", [B.LAZY_KV_BF16, B.LAZY_KV_FP8_E4M3], ids=["bf16", "fp8"])
@pytest.mark.parametrize("cfg,scale", [(3, 0.07), (5, 0.25)])
def test_pair_prefill_is_bitwise_repeatable_under_pressure(cfg, scale, dtype):
    batch = W.CONFIGS[cfg](scale=scale)
    dev = DeviceBatch(batch, dtype=dtype)
    d = dev.device
    try:
        pre = None
        for st in batch.steps:
            dev.write(st)
            if st.kind == "prefill":
                pre = st
                break
        assert pre is not None
        bt, pp = dev.tables_for(pre)
        q, sl, cu = pre.q.to(d), pre.seq_lens.to(d), pre.cu_q_lens.to(d)
        max_q = int((pre.cu_q_lens[1:] - pre.cu_q_lens[:-1]).max())
        first = torch.empty_like(q)
        B.lazy_attn_prefill(dev.handle, q, dev.k_pool, dev.v_pool, bt, pp, sl, cu, max_q, first)
        torch.cuda.synchronize()
        assert torch.isfinite(first.float()).all()
        out = torch.empty_like(q)
        bad = torch.zeros((), dtype=torch.int64, device=d)
        noise_a = torch.empty(64 << 20, dtype=torch.uint8, device=d)
        noise_b = torch.empty(64 << 20, dtype=torch.uint8, device=d)
        side = torch.cuda.Stream()
        main = torch.cuda.current_stream()
        for i in range(RUNS):
            if i % 4 == 0:
                with torch.cuda.stream(side):            # concurrent L2 / SM pressure
                    noise_b.copy_(noise_a)
                    noise_a.add_(1)
            out.fill_(float("nan"))
            B.lazy_attn_prefill(dev.handle, q, dev.k_pool, dev.v_pool, bt, pp, sl, cu, max_q, out, stream=main)
            bad += (out.view(torch.int16) != first.view(torch.int16)).sum()
        torch.cuda.synchronize()
        assert int(bad.item()) == 0, f"{int(bad.item())} elements differed from the first run over {RUNS} runs"
    finally:
        dev.close()

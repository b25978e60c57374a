"""-m gpu: the three calls only enqueue work on the given stream (no host sync, no allocation, include/lazy_attn.h),
so a whole serving step can be captured into a CUDA graph and replayed (CUDA-graph capture of
the mixed prefill + decode step).  Replays must reproduce the eager outputs bit for bit."""
import pytest
import torch

from paper_2606_04302_b200 import binding as B
from paper_2606_04302_b200 import workloads as W
from paper_2606_04302_b200.runner import DeviceBatch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _lib():
    from paper_2606_04302_b200 import build
    build.build()
    B.lib()


@pytest.mark.parametrize("cfg,scale", [(5, 0.15), (2, 0.1)])
def test_step_captured_in_cuda_graph_replays_bit_exact(cfg, scale):
    batch = W.CONFIGS[cfg](scale=scale)
    dev = DeviceBatch(batch)
    d = dev.device
    steps = [s for s in batch.steps]
    recs = []
    for st in steps:
        rec = dict(step=st)
        if st.k_new is not None:
            rec.update(k=st.k_new.to(d), v=st.v_new.to(d), slots=st.slot_mapping.to(d))
        if st.kind != "write_only":
            bt, pp = dev.tables_for(st)
            rec.update(bt=bt, pp=pp, q=st.q.to(d), out=torch.empty_like(st.q, device=d), sl=st.seq_lens.to(d))
            if st.kind == "prefill":
                rec["cu"] = st.cu_q_lens.to(d)
                rec["max_q"] = int((st.cu_q_lens[1:] - st.cu_q_lens[:-1]).max())
        recs.append(rec)

    def run_all():
        for r in recs:
            st = r["step"]
            if "k" in r:
                B.lazy_cache_write(dev.handle, r["k"], r["v"], r["slots"], dev.k_pool, dev.v_pool)
            if st.kind == "decode":
                B.lazy_attn_decode(dev.handle, r["q"], dev.k_pool, dev.v_pool, r["bt"], r["pp"], r["sl"], r["out"])
            elif st.kind == "prefill":
                B.lazy_attn_prefill(dev.handle, r["q"], dev.k_pool, dev.v_pool, r["bt"], r["pp"], r["sl"], r["cu"],
                                    r["max_q"], r["out"])

    try:
        run_all()                                   # eager (also sets kernel attributes / tensor maps once)
        torch.cuda.synchronize()
        eager = [r["out"].clone() for r in recs if "out" in r]
        g = torch.cuda.CUDAGraph()
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            run_all()                               # warm-up on the capture stream
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        with torch.cuda.graph(g):
            run_all()
        for _ in range(2):
            for r in recs:
                if "out" in r:
                    r["out"].zero_()
            g.replay()
            torch.cuda.synchronize()
            got = [r["out"] for r in recs if "out" in r]
            for a, b in zip(eager, got):
                assert torch.equal(a.view(torch.int16), b.view(torch.int16))
    finally:
        dev.close()

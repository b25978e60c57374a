"""-m gpu: a small serving loop through the host page pool and the three CUDA calls.
Documents are looked up position-agnostically, misses are written un-rotated into the pages the pool hands out
(after LRU eviction of unpinned documents), hits are reused at whatever offset the request needs, and every decode
result is checked against the oracle's plain attention over the request's LOGICAL token sequence."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2606_04302_b200 import binding as B

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _lib():
    from paper_2606_04302_b200 import build
    build.build()
    B.lib()


def test_serving_loop_with_eviction_and_reuse_at_any_offset():
    Hq, Hkv, D, P, theta = 4, 1, 64, 16, 1e4
    doc_len, n_docs, docs_per_req, n_req = 64, 12, 3, 40
    num_pages = 6 * (doc_len // P) + 1                      # room for 6 of the 12 documents + one question page
    gen = torch.Generator().manual_seed(1234)
    doc_k = torch.randn(n_docs, doc_len, Hkv, D, generator=gen).to(torch.bfloat16)
    doc_v = torch.randn(n_docs, doc_len, Hkv, D, generator=gen).to(torch.bfloat16)
    rng = np.random.default_rng(7)
    nan = torch.full((num_pages, Hkv, P, D), float("nan"), dtype=torch.bfloat16)
    k_pool, v_pool = nan.clone().cuda(), nan.clone().cuda()
    pmax = docs_per_req * (doc_len // P) + 1
    h = B.lazy_create(Hq, Hkv, D, num_pages=num_pages, max_position=4096, max_reqs=1, max_pages_per_req=pmax,
                      rope_theta=theta)
    pool = B.LazyPool(num_pages, P)
    hits = 0
    try:
        for r in range(n_req):
            docs = rng.choice(n_docs, size=docs_per_req, replace=False, p=np.arange(n_docs, 0, -1) / 78.0)
            gap = int(rng.integers(0, 3)) * 32               # documents need not start at multiples of their length
            bt, pp, k_log, v_log, pos_log = [], [], [], [], []
            pos = gap
            for d in docs:
                hit, pages = pool.acquire(int(d), doc_len, pos)
                hits += hit
                if not hit:                                  # cache miss: store the document's K/V, position-free
                    slots = torch.tensor([pg * P + t for pg in pages for t in range(P)], dtype=torch.int64).cuda()
                    B.lazy_cache_write(h, doc_k[d].cuda(), doc_v[d].cuda(), slots, k_pool, v_pool)
                bt += pages
                pp += [pos + P * i for i in range(len(pages))]
                k_log.append(doc_k[d]); v_log.append(doc_v[d]); pos_log += list(range(pos, pos + doc_len))
                pos += doc_len
            _, qpage = pool.acquire(-(r + 1), 1, pos)         # private page of the request's own token
            kq = torch.randn(1, Hkv, D, generator=gen).to(torch.bfloat16)
            vq = torch.randn(1, Hkv, D, generator=gen).to(torch.bfloat16)
            B.lazy_cache_write(h, kq.cuda(), vq.cuda(), torch.tensor([qpage[0] * P], dtype=torch.int64).cuda(),
                               k_pool, v_pool)
            bt += qpage; pp += [pos]
            k_log.append(kq); v_log.append(vq); pos_log.append(pos)
            L = len(pos_log)
            q = torch.randn(1, Hq, D, generator=gen).to(torch.bfloat16)
            out = torch.empty_like(q, device="cuda")
            pad = pmax - len(bt)
            B.lazy_attn_decode(h, q.cuda(), k_pool, v_pool,
                               torch.tensor([bt + [0] * pad], dtype=torch.int32).cuda(),
                               torch.tensor([pp + [0] * pad], dtype=torch.int32).cuda(),
                               torch.tensor([L], dtype=torch.int32).cuda(), out)
            torch.cuda.synchronize()
            ref = O.attend_core(q.double().numpy(), torch.cat(k_log).double().numpy(), torch.cat(v_log).double().numpy(),
                                [float(pos_log[-1])], np.array(pos_log, dtype=np.float64), [L - 1], theta)
            err = np.abs(out.double().cpu().numpy() - ref)
            assert err.max() <= 2e-2 and err.mean() <= 2e-3, (r, err.max())
            assert err.max() < 5e-3
            for d, p0 in zip(docs, range(gap, gap + docs_per_req * doc_len, doc_len)):
                pool.release(int(d), p0)
            pool.release(-(r + 1), pos)
        st = pool.stats()
        assert st["evictions"] > 10 and hits > 20, (st, hits)   # both reuse and rewrite-after-eviction happened
    finally:
        pool.close(); h.close()

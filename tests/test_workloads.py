"""Structure of the synthetic Zipf-shared RAG batches (host logic only; no method arithmetic)."""
import numpy as np
import torch

from paper_2606_04302_b200 import workloads as W


def test_config1_structure():
    b = W.config1()
    assert b.k_pool.shape == (32 + 2, 1, 16, 64)            # 8 docs x 4 pages + 2 private pages (16 q + 1 decode)
    assert b.block_table.shape == (1, 14)
    assert b.page_logical_pos[0].tolist() == [16 * i for i in range(14)]
    pre, dec = b.steps
    assert pre.kind == "prefill" and dec.kind == "decode"
    assert int(pre.seq_lens[0]) == 208 and int(dec.seq_lens[0]) == 209
    assert pre.q.shape == (16, 4, 64) and dec.q.shape == (1, 4, 64)
    # private pages start poisoned; document pages are finite
    priv = b.block_table[0, 12:].long()
    assert torch.isnan(b.k_pool[priv].float()).all()
    assert torch.isfinite(b.k_pool[b.block_table[0, :12].long()].float()).all()


def test_zipf_sharing_and_determinism():
    a = W.config2(scale=0.25)
    b = W.config2(scale=0.25)
    assert torch.equal(a.block_table, b.block_table)
    assert torch.equal(a.k_pool.view(torch.int16), b.k_pool.view(torch.int16))
    assert a.meta["distinct_docs"] < a.block_table.shape[0] * 10      # pages are shared across requests
    # without replacement inside a request
    for row in a.meta["drawn"]:
        assert len(set(row.tolist())) == len(row)
    ns = W.config2(scale=0.25, noshare=True)
    assert ns.meta["distinct_docs"] == ns.block_table.shape[0] * 10


def test_config4_repeats_within_request():
    b = W.config4(scale=0.25)
    assert any(len(set(r.tolist())) < len(r) for r in b.meta["drawn"])
    assert int(b.steps[-1].seq_lens[0]) == 64 * 512 + 128 + 1


def test_zipf_table():
    p = W.zipf_probs(100, 1.0)
    assert abs(p.sum() - 1.0) < 1e-12 and abs(p[0] / p[9] - 10.0) < 1e-9


def test_shard_requests_covers_everything():
    for n, w in [(64, 2), (7, 4), (3, 8)]:
        got = [i for r in range(w) for i in W.shard_requests(n, r, w)]
        assert got == list(range(n))


def test_config5_rows():
    b = W.config5(scale=0.25)
    pre, dec, fu = b.steps
    n_miss = b.meta["n_miss"]
    assert pre.req_ids.tolist() == list(range(n_miss))
    assert dec.req_ids.tolist() == list(range(n_miss, n_miss + b.meta["R_dec"]))
    # follow-up places the fresh documents at non-zero offsets
    row = int(fu.req_ids[0])
    miss_pages = set(b.block_table[:n_miss].flatten().tolist())
    used = b.block_table[row].tolist()
    assert any(p in miss_pages and b.page_logical_pos[row, i] > 0 for i, p in enumerate(used))

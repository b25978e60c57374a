"""Seeded synthetic Zipf-shared RAG batches (the five BASELINE.json configs).

This module only *generates inputs*: random bf16 tensors, Zipf document draws,
block tables and logical page positions.  It contains none of the method's
arithmetic (no RoPE, no softmax, no attention) and is the only code shared by
the CPU oracle's tests and the CUDA path's tests / bench (DESIGN.md "Input
recipe").  Everything is produced on the host with explicit seeds; tensors are
torch CPU tensors (bf16 / int32 / int64).

Recipe (stands in for the paper's QA-dataset request streams,
PAPER.md L236-L242, L261, L273):
  * pool of `pool_docs` documents of `doc_len` tokens, each `doc_len/16` pages;
    physical page ids are a random permutation (scattered like a real paged
    allocator); K,V ~ N(0,1) rounded to bf16.
  * each request draws `docs_per_req` documents Zipf(alpha) over the pool
    (with or without replacement), document k sits at logical positions
    [k*doc_len, (k+1)*doc_len); then private pages for the question tokens
    (and the decode token), appended to the pool.
  * private pages start out as NaN bit patterns (0x7FC0): only what
    `lazy_cache_write` stores becomes valid, so the tail of the last page stays
    poisoned and any kernel that lets it leak into the result fails parity.
"""
from __future__ import annotations

import dataclasses
from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np
import torch

PAGE_SIZE = 16
BF16_NAN_BITS = 0x7FC0


@dataclass
class LazyShape:
    num_q_heads: int
    num_kv_heads: int
    head_dim: int
    rope_theta: float
    page_size: int = PAGE_SIZE


@dataclass
class Step:
    """One serving step: optional cache write of new tokens, then one attention call."""
    kind: str                               # 'prefill' | 'decode' | 'write_only'
    k_new: Optional[torch.Tensor] = None    # [T, Hkv, D] bf16 (un-rotated)
    v_new: Optional[torch.Tensor] = None
    slot_mapping: Optional[torch.Tensor] = None  # [T] int64, page*16+off
    q: Optional[torch.Tensor] = None        # [total_q, Hq, D] bf16 (un-rotated)
    seq_lens: Optional[torch.Tensor] = None  # [R] int32 (KV length incl. this step's tokens)
    cu_q_lens: Optional[torch.Tensor] = None  # [R+1] int32
    req_ids: Optional[torch.Tensor] = None  # [R'] rows of the batch tables this call uses (None = all)


@dataclass
class LazyBatch:
    name: str
    shape: LazyShape
    k_pool: torch.Tensor            # [num_pages, Hkv, 16, D] bf16
    v_pool: torch.Tensor
    block_table: torch.Tensor       # [R, Pmax] int32
    page_logical_pos: torch.Tensor  # [R, Pmax] int32
    steps: List[Step] = field(default_factory=list)
    meta: dict = field(default_factory=dict)

    @property
    def num_pages(self) -> int:
        return self.k_pool.shape[0]

    @property
    def max_position(self) -> int:
        return int(self.page_logical_pos.max().item()) + self.shape.page_size


def _randn_bf16(gen: torch.Generator, shape, chunk_elems: int = 1 << 26) -> torch.Tensor:
    """N(0,1) in fp32 rounded to bf16 (RNE), generated in chunks to bound memory."""
    n = int(np.prod(shape))
    out = torch.empty(n, dtype=torch.bfloat16)
    for s in range(0, n, chunk_elems):
        e = min(n, s + chunk_elems)
        out[s:e] = torch.randn(e - s, generator=gen, dtype=torch.float32).to(torch.bfloat16)
    return out.view(*shape)


def zipf_probs(pool: int, alpha: float) -> np.ndarray:
    w = np.arange(1, pool + 1, dtype=np.float64) ** (-alpha)
    return w / w.sum()


def draw_docs(rng: np.random.Generator, pool: int, alpha: float, n: int, replace: bool) -> np.ndarray:
    """Inverse-CDF Zipf sampling on the explicit table (rank 0 = most popular)."""
    p = zipf_probs(pool, alpha)
    if replace:
        cdf = np.cumsum(p)
        u = rng.random(n)
        return np.minimum(np.searchsorted(cdf, u, side="right"), pool - 1).astype(np.int64)
    # without replacement: successive draws from the renormalised remainder
    out = []
    alive = np.ones(pool, dtype=bool)
    for _ in range(n):
        pp = np.where(alive, p, 0.0)
        cdf = np.cumsum(pp)
        u = rng.random() * cdf[-1]
        i = int(min(np.searchsorted(cdf, u, side="right"), pool - 1))
        while not alive[i]:            # guard against a rounding landing on a dead slot
            i = (i + 1) % pool
        alive[i] = False
        out.append(i)
    return np.asarray(out, dtype=np.int64)


def make_rag_batch(
    name: str,
    shape: LazyShape,
    *,
    seed: int,
    pool_docs: int,
    doc_len: int,
    num_reqs: int,
    docs_per_req: int,
    alpha: float,
    replace: bool,
    question_len: int,
    decode: bool,
    prefill_question: bool,
    noshare: bool = False,
    q_scale: float = 1.0,
    pos_shift: int = 0,
) -> LazyBatch:
    """Generic Zipf-shared RAG batch.

    decode=True adds one decode token per request (seq_len = docs + question + 1)
    and a 'decode' step; prefill_question=True adds a 'prefill' step over the
    question chunk.  `noshare` enlarges the pool so every drawn document is
    distinct (logical bytes == unique bytes).  `pos_shift` adds a constant to every
    logical position (shift-invariance tests).
    """
    P = shape.page_size
    assert doc_len % P == 0
    Hq, Hkv, D = shape.num_q_heads, shape.num_kv_heads, shape.head_dim
    rng = np.random.default_rng(np.random.PCG64(seed))
    gen = torch.Generator().manual_seed(seed)

    if noshare:
        pool_docs = num_reqs * docs_per_req
    pages_per_doc = doc_len // P
    doc_pages_total = pool_docs * pages_per_doc
    n_priv_tokens = question_len + (1 if decode else 0)
    priv_pages_per_req = (n_priv_tokens + P - 1) // P
    num_pages = doc_pages_total + num_reqs * priv_pages_per_req

    # physical placement: random permutation of all page ids
    perm = rng.permutation(num_pages).astype(np.int64)
    doc_page_ids = perm[:doc_pages_total].reshape(pool_docs, pages_per_doc)
    priv_page_ids = perm[doc_pages_total:].reshape(num_reqs, priv_pages_per_req) if priv_pages_per_req else \
        np.zeros((num_reqs, 0), dtype=np.int64)

    k_pool = torch.empty(num_pages, Hkv, P, D, dtype=torch.bfloat16)
    v_pool = torch.empty(num_pages, Hkv, P, D, dtype=torch.bfloat16)
    # document pages: N(0,1); private pages: NaN-poisoned until written
    dp = torch.from_numpy(doc_page_ids.reshape(-1))
    k_pool[dp] = _randn_bf16(gen, (doc_pages_total, Hkv, P, D))
    v_pool[dp] = _randn_bf16(gen, (doc_pages_total, Hkv, P, D))
    if priv_pages_per_req:
        pp = torch.from_numpy(priv_page_ids.reshape(-1))
        nanv = torch.full((1,), BF16_NAN_BITS, dtype=torch.int16).view(torch.bfloat16)
        k_pool[pp] = nanv
        v_pool[pp] = nanv

    pmax = docs_per_req * pages_per_doc + priv_pages_per_req
    block_table = np.zeros((num_reqs, pmax), dtype=np.int32)
    page_pos = np.zeros((num_reqs, pmax), dtype=np.int32)
    drawn = np.zeros((num_reqs, docs_per_req), dtype=np.int64)
    for r in range(num_reqs):
        if noshare:
            docs = np.arange(r * docs_per_req, (r + 1) * docs_per_req, dtype=np.int64)
        else:
            docs = draw_docs(rng, pool_docs, alpha, docs_per_req, replace)
        drawn[r] = docs
        pages = np.concatenate([doc_page_ids[d] for d in docs] + [priv_page_ids[r]])
        block_table[r, : len(pages)] = pages
        page_pos[r, : len(pages)] = pos_shift + P * np.arange(len(pages))

    doc_tokens = docs_per_req * doc_len
    batch = LazyBatch(
        name=name, shape=shape, k_pool=k_pool, v_pool=v_pool,
        block_table=torch.from_numpy(block_table), page_logical_pos=torch.from_numpy(page_pos),
        meta=dict(seed=seed, pool_docs=pool_docs, doc_len=doc_len, docs_per_req=docs_per_req,
                  alpha=alpha, replace=replace, question_len=question_len, noshare=noshare,
                  distinct_docs=int(len(np.unique(drawn))), drawn=drawn, doc_tokens=doc_tokens),
    )

    def slots_for(r: int, first_tok: int, n: int) -> np.ndarray:
        """slots of private tokens [first_tok, first_tok+n) of request r (0 = first question token)."""
        t = first_tok + np.arange(n)
        return priv_page_ids[r][t // P] * P + (t % P)

    def new_tokens(n_per_req: int, first_tok: int):
        k_new = _randn_bf16(gen, (num_reqs * n_per_req, Hkv, D))
        v_new = _randn_bf16(gen, (num_reqs * n_per_req, Hkv, D))
        slots = np.concatenate([slots_for(r, first_tok, n_per_req) for r in range(num_reqs)])
        return k_new, v_new, torch.from_numpy(slots.astype(np.int64))

    if question_len > 0:
        k_new, v_new, slots = new_tokens(question_len, 0)
        if prefill_question:
            q = (_randn_bf16(gen, (num_reqs * question_len, Hq, D)).float() * q_scale).to(torch.bfloat16)
            batch.steps.append(Step(
                kind="prefill", k_new=k_new, v_new=v_new, slot_mapping=slots, q=q,
                seq_lens=torch.full((num_reqs,), doc_tokens + question_len, dtype=torch.int32),
                cu_q_lens=torch.arange(0, (num_reqs + 1) * question_len, question_len, dtype=torch.int32)))
        else:
            batch.steps.append(Step(kind="write_only", k_new=k_new, v_new=v_new, slot_mapping=slots))
    if decode:
        k_new, v_new, slots = new_tokens(1, question_len)
        q = (_randn_bf16(gen, (num_reqs, Hq, D)).float() * q_scale).to(torch.bfloat16)
        batch.steps.append(Step(
            kind="decode", k_new=k_new, v_new=v_new, slot_mapping=slots, q=q,
            seq_lens=torch.full((num_reqs,), doc_tokens + question_len + 1, dtype=torch.int32),
            cu_q_lens=torch.arange(0, num_reqs + 1, dtype=torch.int32)))
    return batch


# ----------------------------------------------------------------------------------------------
# The five BASELINE.json configs.  `scale` < 1 shrinks request / document counts for parity tests
# that run the full oracle; scale = 1 is the size the bench and the sampled parity tests use.
# ----------------------------------------------------------------------------------------------
SEED0 = 20260604


def config1(**kw) -> LazyBatch:
    """Tiny reuse case: 3 of 8 docs (64 tok) at 0/64/128, 16-token question prefill, 1 decode step."""
    shape = LazyShape(4, 1, 64, 1.0e4)
    return make_rag_batch("cfg1_tiny", shape, seed=SEED0 + 1, pool_docs=8, doc_len=64, num_reqs=1,
                          docs_per_req=3, alpha=1.0, replace=False, question_len=16, decode=True,
                          prefill_question=True, **kw)


def config2(scale: float = 1.0, **kw) -> LazyBatch:
    """Decode at Llama-3-8B layer shape: 64 reqs x (10 docs x 256 + 64-token question + 1)."""
    shape = LazyShape(32, 8, 128, 5.0e5)
    R = max(2, int(round(64 * scale)))
    pool = max(12, int(round(200 * scale)))
    return make_rag_batch("cfg2_decode", shape, seed=SEED0 + 2, pool_docs=pool, doc_len=256, num_reqs=R,
                          docs_per_req=10, alpha=1.0, replace=False, question_len=64, decode=True,
                          prefill_question=False, **kw)


def config3(scale: float = 1.0, **kw) -> LazyBatch:
    """Prefill of a 256-token question over 20 docs x 512 (pool 1000, Zipf 1.0), 32 requests."""
    shape = LazyShape(32, 8, 128, 5.0e5)
    R = max(2, int(round(32 * scale)))
    pool = max(24, int(round(1000 * scale)))
    return make_rag_batch("cfg3_prefill", shape, seed=SEED0 + 3, pool_docs=pool, doc_len=512, num_reqs=R,
                          docs_per_req=20, alpha=1.0, replace=False, question_len=256, decode=False,
                          prefill_question=True, **kw)


def config4(scale: float = 1.0, **kw) -> LazyBatch:
    """Long-context decode: 8 reqs x (64 docs x 512, Zipf 1.2 with replacement + 128-token question + 1)."""
    shape = LazyShape(32, 8, 128, 5.0e5)
    R = max(2, int(round(8 * scale)))
    pool = max(8, int(round(300 * scale)))
    return make_rag_batch("cfg4_longdecode", shape, seed=SEED0 + 4, pool_docs=pool, doc_len=512, num_reqs=R,
                          docs_per_req=64, alpha=1.2, replace=True, question_len=128, decode=True,
                          prefill_question=False, **kw)


def e3_paper(decode: bool, **kw) -> LazyBatch:
    """The shape of the paper's overhead ablation (Fig. 5): ONE request over 5 cached documents of 4,096
    tokens each plus a 64-token query, Llama-3-8B layer shape.  decode=True: one decode token over the 20,545-token
    sequence; decode=False: the 64-row query prefill over the cached documents.  A measurement shape for
    `bench.py --e3`, not one of BASELINE.json's configs."""
    shape = LazyShape(32, 8, 128, 5.0e5)
    return make_rag_batch("e3_decode" if decode else "e3_prefill", shape, seed=SEED0 + 6, pool_docs=5, doc_len=4096,
                          num_reqs=1, docs_per_req=5, alpha=1.0, replace=False, question_len=64, decode=decode,
                          prefill_question=not decode, **kw)


def config5(scale: float = 1.0, q_scale: float = 1.0, noshare: bool = False) -> LazyBatch:
    """Mixed serving step (Hq=28, Hkv=4, theta 1e6): 16 decode requests over 20 cached docs x 512
    (pool 2000, Zipf 0.8) + 4 cache-miss docs x 1024 prefilled block-locally (positions from 0, causal)
    and written un-rotated into new pages.  Steps: prefill (writes the 4 miss documents, then attends
    them block-locally: rows 0..3 of the tables), decode (rows 4..19), then a follow-up decode request
    (last row) that places two of the freshly written documents at non-zero offsets.
    """
    shape = LazyShape(28, 4, 128, 1.0e6)
    P, Hq, Hkv, D = shape.page_size, 28, 4, 128
    seed = SEED0 + 5
    R_dec = max(2, int(round(16 * scale)))
    pool = max(24, int(round(2000 * scale)))
    n_miss, miss_len = (4, 1024) if scale >= 1.0 else (2, 272)
    miss_pages = (miss_len + P - 1) // P
    dec = make_rag_batch("cfg5_mixed", shape, seed=seed, pool_docs=pool, doc_len=512, num_reqs=R_dec,
                         docs_per_req=20, alpha=0.8, replace=False, question_len=0, decode=True,
                         prefill_question=False, q_scale=q_scale, noshare=noshare)
    gen = torch.Generator().manual_seed(seed + 1000)
    base_pages = dec.num_pages
    # new pages: miss documents + 1 private page for the follow-up request's decode token
    n_new = n_miss * miss_pages + 1
    nanv = torch.full((1,), BF16_NAN_BITS, dtype=torch.int16).view(torch.bfloat16)
    k_pool = torch.cat([dec.k_pool, nanv.expand(n_new, Hkv, P, D).clone()])
    v_pool = torch.cat([dec.v_pool, nanv.expand(n_new, Hkv, P, D).clone()])
    rng = np.random.default_rng(np.random.PCG64(seed + 1000))
    new_ids = base_pages + rng.permutation(n_new).astype(np.int64)
    miss_ids = new_ids[: n_miss * miss_pages].reshape(n_miss, miss_pages)
    fu_page = int(new_ids[-1])

    # table rows: [0,n_miss) miss docs (block-local), [n_miss, n_miss+R_dec) decode requests, last: follow-up
    pmax_dec = dec.block_table.shape[1]
    fu_docs = [0, min(1, n_miss - 1)]
    fu_cached_doc_pages = 32                                    # one cached 512-token doc in front
    fu_pages = fu_cached_doc_pages + 2 * miss_pages + 1
    pmax = max(pmax_dec, miss_pages, fu_pages)
    R = n_miss + R_dec + 1
    bt = np.zeros((R, pmax), dtype=np.int32)
    pp = np.zeros((R, pmax), dtype=np.int32)
    for m in range(n_miss):
        bt[m, :miss_pages] = miss_ids[m]
        pp[m, :miss_pages] = P * np.arange(miss_pages)
    bt[n_miss:n_miss + R_dec, :pmax_dec] = dec.block_table.numpy()
    pp[n_miss:n_miss + R_dec, :pmax_dec] = dec.page_logical_pos.numpy()
    # follow-up: cached doc (pages of decode request 0's first doc) at 0, then the two miss docs back to
    # back at non-zero offsets; miss_len need not be a page multiple -> the 2nd miss doc starts mid-way
    # through a logical page: handled by giving every page its own logical start.
    cached = dec.block_table.numpy()[0, :fu_cached_doc_pages]
    fu_row = R - 1
    bt[fu_row, :fu_cached_doc_pages] = cached
    pp[fu_row, :fu_cached_doc_pages] = P * np.arange(fu_cached_doc_pages)
    off = fu_cached_doc_pages * P
    c = fu_cached_doc_pages
    for d in fu_docs:
        bt[fu_row, c:c + miss_pages] = miss_ids[d]
        pp[fu_row, c:c + miss_pages] = off + P * np.arange(miss_pages)
        c += miss_pages
        off += miss_pages * P
    bt[fu_row, c] = fu_page
    pp[fu_row, c] = off

    batch = LazyBatch(name="cfg5_mixed", shape=shape, k_pool=k_pool, v_pool=v_pool,
                      block_table=torch.from_numpy(bt), page_logical_pos=torch.from_numpy(pp),
                      meta=dict(dec.meta, n_miss=n_miss, miss_len=miss_len, R_dec=R_dec))
    # step 1: write the miss documents and prefill them block-locally
    T = n_miss * miss_len
    k_new = _randn_bf16(gen, (T, Hkv, D))
    v_new = _randn_bf16(gen, (T, Hkv, D))
    tok = np.arange(miss_len)
    slots = np.concatenate([miss_ids[m][tok // P] * P + tok % P for m in range(n_miss)]).astype(np.int64)
    q = (_randn_bf16(gen, (T, Hq, D)).float() * q_scale).to(torch.bfloat16)
    batch.steps.append(Step(kind="prefill", k_new=k_new, v_new=v_new, slot_mapping=torch.from_numpy(slots), q=q,
                            seq_lens=torch.full((n_miss,), miss_len, dtype=torch.int32),
                            cu_q_lens=torch.arange(0, (n_miss + 1) * miss_len, miss_len, dtype=torch.int32),
                            req_ids=torch.arange(0, n_miss, dtype=torch.int64)))
    # step 2: decode over the cached documents (reuses dec's decode step)
    d = dec.steps[-1]
    batch.steps.append(dataclasses.replace(d, req_ids=torch.arange(n_miss, n_miss + R_dec, dtype=torch.int64)))
    # step 3 (follow-up, correctness only): decode token over cached doc + the two fresh docs at offsets
    L_fu = fu_cached_doc_pages * P + 2 * miss_pages * P + 1
    # note: when miss_len is not a page multiple the tail of each miss document's last page is poisoned
    # and must not be visible; the follow-up is therefore only generated with whole pages visible.
    if miss_len % P != 0:
        # shrink: the follow-up sees each miss doc only up to its last whole page
        whole = miss_len // P
        c = fu_cached_doc_pages
        off = fu_cached_doc_pages * P
        bt[fu_row, c:] = 0
        pp[fu_row, c:] = 0
        for dd in fu_docs:
            bt[fu_row, c:c + whole] = miss_ids[dd][:whole]
            pp[fu_row, c:c + whole] = off + P * np.arange(whole)
            c += whole
            off += whole * P
        bt[fu_row, c] = fu_page
        pp[fu_row, c] = off
        L_fu = off + 1
        batch.block_table = torch.from_numpy(bt)
        batch.page_logical_pos = torch.from_numpy(pp)
    k1 = _randn_bf16(gen, (1, Hkv, D))
    v1 = _randn_bf16(gen, (1, Hkv, D))
    q1 = (_randn_bf16(gen, (1, Hq, D)).float() * q_scale).to(torch.bfloat16)
    batch.steps.append(Step(kind="decode", k_new=k1, v_new=v1,
                            slot_mapping=torch.tensor([fu_page * P], dtype=torch.int64), q=q1,
                            seq_lens=torch.tensor([L_fu], dtype=torch.int32),
                            cu_q_lens=torch.tensor([0, 1], dtype=torch.int32),
                            req_ids=torch.tensor([fu_row], dtype=torch.int64)))
    return batch


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


def shard_requests(num_reqs: int, rank: int, world_size: int) -> range:
    """Request-parallel sharding for multi-GPU runs (no data-path collective: DESIGN.md 'Multi-GPU').
    Contiguous, balanced to within one request."""
    base, rem = divmod(num_reqs, world_size)
    lo = rank * base + min(rank, rem)
    return range(lo, lo + base + (1 if rank < rem else 0))

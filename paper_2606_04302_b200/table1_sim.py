#!/usr/bin/env python
"""Trace-driven VRAM hit-ratio simulation in the manner of PAPER.md Table 1 (L254-269, section 4.2): host only.

    python -m paper_2606_04302_b200.table1_sim [--queries 20000] [--pool-docs 100000] [--doc-tokens 512] [--markdown]

Seeded Zipf request traces (skew alpha = 1.1 / 1.5 / 2.1 for Low / Mid / High, K = 10 documents per query drawn without
replacement, random slot order) are replayed through the library's page pool (`lazy_pool_*`, csrc/page_pool.cpp) under
a page budget, once keyed by document only (LAZY_POOL_AGNOSTIC: the position-free cache of this repo -- one physical
copy serves every logical offset) and once keyed by (document, logical position) (LAZY_POOL_POSITION_AWARE: a
position-coupled cache such as Block-Attention's, which must hold one copy per offset a document was seen at).  The hit
ratio is the fraction of document lookups served from the pool; next to it the script prints the paper's analytic
model, Eq. 1 (agnostic) and Eq. 2 (aware, D = K positions), for an ideal top-C cache.

Stand-in sizes (stated because the paper does not print them): every document has `--doc-tokens` tokens (default 512 =
32 pages); a KV page of 16 tokens of Llama-3-8B (32 layers x 8 kv heads x 128 dims x K,V x bf16) is 2 MiB, so the
paper's budgets 1 / 5 / 10 / 50 GB and "no limit" (about 66 GB) are 512 / 2560 / 5120 / 25600 / 33792 pages.  The
paper's trace length and document-length mix are not given; absolute percentages therefore differ from Table 1 and
only the ordering and the trend with budget and skew are comparable.
"""
from __future__ import annotations

import argparse
import json

import numpy as np

from . import binding as B
from .workloads import zipf_probs

PAGE_TOKENS = 16
PAGE_BYTES_8B = 32 * 8 * 128 * 2 * 2 * PAGE_TOKENS          # all layers of Llama-3-8B: 2 MiB per 16-token page
BUDGETS_GB = [("1 GB", 1.0), ("5 GB", 5.0), ("10 GB", 10.0), ("50 GB", 50.0), ("no limit (66 GB)", 66.0)]
SKEWS = [("Low", 1.1), ("Mid", 1.5), ("High", 2.1)]


def make_trace(seed: int, queries: int, docs_per_query: int, pool_docs: int, alpha: float):
    """[(doc id, slot)] per query: Zipf(alpha) popularity, K distinct documents, random slot order."""
    rng = np.random.default_rng(seed)
    p = zipf_probs(pool_docs, alpha)
    cdf = np.cumsum(p)
    out = []
    for _ in range(queries):
        docs = []
        seen = set()
        while len(docs) < docs_per_query:                    # inverse-CDF draws, rejecting repeats
            for d in np.searchsorted(cdf, rng.random(docs_per_query * 2)):
                d = int(min(d, pool_docs - 1))
                if d not in seen:
                    seen.add(d)
                    docs.append(d)
                    if len(docs) == docs_per_query:
                        break
        order = rng.permutation(docs_per_query)
        out.append([(docs[i], int(k)) for k, i in enumerate(order)])
    return out


def replay(trace, num_pages: int, doc_tokens: int, keying: int, warm_fraction: float = 0.25) -> float:
    """Hit ratio over the part of the trace after the warm-up fraction (the pool starts empty)."""
    pool = B.LazyPool(num_pages=num_pages, page_size=PAGE_TOKENS, keying=keying)
    warm = int(len(trace) * warm_fraction)
    hits = lookups = 0
    try:
        for qi, req in enumerate(trace):
            got = []
            for d, k in req:
                try:
                    hit, _ = pool.acquire(d, doc_tokens, k * doc_tokens)
                    got.append((d, k))
                except B.LazyError:                           # budget smaller than one request's pinned documents
                    hit = False
                if qi >= warm:
                    lookups += 1
                    hits += int(hit)
            for d, k in got:
                pool.release(d, k * doc_tokens)
    finally:
        pool.close()
    return hits / max(lookups, 1)


def simulate(queries: int = 20000, pool_docs: int = 100000, doc_tokens: int = 512, docs_per_query: int = 10,
             budgets_gb=None, skews=None, seed: int = 20260604):
    rows = []
    doc_pages = -(-doc_tokens // PAGE_TOKENS)
    for bname, gb in (budgets_gb or BUDGETS_GB):
        pages = int(gb * (1 << 30) // PAGE_BYTES_8B)
        cap_docs = pages // doc_pages
        for sname, alpha in (skews or SKEWS):
            trace = make_trace(seed + int(alpha * 10), queries, docs_per_query, pool_docs, alpha)
            rows.append(dict(
                budget=bname, pages=pages, capacity_docs=cap_docs, skew=sname, alpha=alpha,
                lazy_sim=100 * replay(trace, pages, doc_tokens, B.LAZY_POOL_AGNOSTIC),
                aware_sim=100 * replay(trace, pages, doc_tokens, B.LAZY_POOL_POSITION_AWARE),
                lazy_eq1=100 * B.lazy_hit_ratio_model(alpha, pool_docs, cap_docs, 1),
                aware_eq2=100 * B.lazy_hit_ratio_model(alpha, pool_docs, cap_docs, docs_per_query)))
    return rows


def to_markdown(rows) -> str:
    lines = ["| budget | pages | docs that fit | skew (alpha) | position-free pool, simulated % | position-aware pool, simulated % "
             "| Eq. 1 % | Eq. 2 (D = 10) % | simulated advantage |", "|---|---|---|---|---|---|---|---|---|"]
    for r in rows:
        adv = r["lazy_sim"] / r["aware_sim"] if r["aware_sim"] > 0 else float("inf")
        lines.append(f"| {r['budget']} | {r['pages']} | {r['capacity_docs']} | {r['skew']} ({r['alpha']}) | {r['lazy_sim']:.2f} | "
                     f"{r['aware_sim']:.2f} | {r['lazy_eq1']:.2f} | {r['aware_eq2']:.2f} | {adv:.2f}x |")
    return "\n".join(lines)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--queries", type=int, default=20000)
    ap.add_argument("--pool-docs", type=int, default=100000)
    ap.add_argument("--doc-tokens", type=int, default=512)
    ap.add_argument("--markdown", action="store_true")
    a = ap.parse_args()
    rows = simulate(a.queries, a.pool_docs, a.doc_tokens)
    print(to_markdown(rows) if a.markdown else json.dumps(rows, indent=1))


if __name__ == "__main__":
    main()

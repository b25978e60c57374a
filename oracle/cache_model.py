"""Plain-Python statement of the paper's cache-level model -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

PAPER.md Eq. 1-3 (L60-75): Zipf hit ratios of a position-agnostic cache (one entry per document) and of a
position-aware cache (up to D position-specific copies per document), and a brute-force LRU page pool with reference
counts written with lists and dicts only.  Shares nothing with paper_2606_04302_b200/csrc/page_pool.cpp.
"""
from __future__ import annotations


def hit_ratio_agnostic(alpha: float, n_docs: int, capacity: int) -> float:
    """Eq. 1: sum_{i<=C} i^-alpha / sum_{j<=N} j^-alpha."""
    den = sum(j ** (-alpha) for j in range(1, n_docs + 1))
    return sum(i ** (-alpha) for i in range(1, min(capacity, n_docs) + 1)) / den


def hit_ratio_aware(alpha: float, n_docs: int, capacity: int, positions: int) -> float:
    """Eq. 2: the same budget covers only floor(C/D) unique documents."""
    return hit_ratio_agnostic(alpha, n_docs, capacity // positions)


def advantage(alpha: float, capacity: int, positions: int) -> float:
    """Eq. 3 (independent of N)."""
    num = sum(i ** (-alpha) for i in range(1, capacity + 1))
    return num / sum(i ** (-alpha) for i in range(1, capacity // positions + 1))


class BruteForcePool:
    """LRU over unpinned documents, pages handed out lowest id first, freed pages reused last-freed first."""

    def __init__(self, num_pages: int, page_size: int, position_aware: bool):
        self.page_size, self.aware = page_size, position_aware
        self.free = list(range(num_pages - 1, -1, -1))      # pop() yields page 0 first
        self.docs = {}                                       # key -> [pages, refcount]
        self.lru = []                                        # keys, least recently released first
        self.lookups = self.hits = self.evictions = 0

    def _key(self, doc, pos):
        return (doc, pos if self.aware else 0)

    def acquire(self, doc, tokens, pos):
        need = -(-tokens // self.page_size)
        key = self._key(doc, pos)
        self.lookups += 1
        if key in self.docs:
            if key in self.lru:
                self.lru.remove(key)
            self.docs[key][1] += 1
            self.hits += 1
            return True, list(self.docs[key][0])
        while len(self.free) < need:
            if not self.lru:
                raise MemoryError("pool exhausted by pinned documents")
            victim = self.lru.pop(0)
            self.free.extend(self.docs.pop(victim)[0])
            self.evictions += 1
        pages = [self.free.pop() for _ in range(need)]
        self.docs[key] = [pages, 1]
        return False, list(pages)

    def release(self, doc, pos):
        key = self._key(doc, pos)
        self.docs[key][1] -= 1
        if self.docs[key][1] == 0:
            self.lru.append(key)

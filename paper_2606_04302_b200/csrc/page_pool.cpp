// page_pool.cpp -- host side of SURVEY.md 8.0 row f4: a document-granular, position-agnostic page pool with
// reference counts and LRU eviction, and the paper's analytic hit-ratio model (Eq. 1-3).
//
// The pool owns no device memory: it hands out physical page ids of the caller's k_cache / v_cache.  Keyed by
// document only (LAZY_POOL_AGNOSTIC) one physical copy serves every logical position; keyed
// by (document, logical position) (LAZY_POOL_POSITION_AWARE) it behaves like the position-coupled caches the paper
// compares against, which spend capacity on positional variants (L56-58, Eq. 2).  Same code, same budget: the
// difference in hit ratio is the method's cache-level claim (Table 1).
#include <cmath>
#include <cstdint>
#include <list>
#include <new>
#include <unordered_map>
#include <vector>

#include "lazy_attn.h"

namespace {
struct Key {
  int64_t doc;
  int32_t pos;
  bool operator==(const Key& o) const { return doc == o.doc && pos == o.pos; }
};
struct KeyHash {
  size_t operator()(const Key& k) const {
    uint64_t x = (uint64_t)k.doc * 0x9E3779B97F4A7C15ull ^ ((uint64_t)(uint32_t)k.pos + 0x7F4A7C15ull) * 0xBF58476D1CE4E5B9ull;
    x ^= x >> 31;
    return (size_t)x;
  }
};
struct Entry {
  std::vector<int32_t> pages;
  int32_t refcount = 0;
  bool in_lru = false;
  std::list<Key>::iterator lru_it;
};
}  // namespace

struct lazy_pool {
  int32_t num_pages, page_size, keying;
  std::vector<int32_t> free_pages;                 // stack of free physical page ids
  std::unordered_map<Key, Entry, KeyHash> docs;
  std::list<Key> lru;                              // unpinned entries, least recently released first
  int64_t lookups = 0, hits = 0, evictions = 0;
};

extern "C" {

lazy_pool* lazy_pool_create(int32_t num_pages, int32_t page_size, int32_t keying) {
  if (num_pages <= 0 || page_size <= 0 || (keying != LAZY_POOL_AGNOSTIC && keying != LAZY_POOL_POSITION_AWARE))
    return nullptr;
  lazy_pool* p = new (std::nothrow) lazy_pool();
  if (!p) return nullptr;
  p->num_pages = num_pages;
  p->page_size = page_size;
  p->keying = keying;
  p->free_pages.reserve(num_pages);
  for (int32_t i = num_pages - 1; i >= 0; --i) p->free_pages.push_back(i);   // page 0 is handed out first
  return p;
}

void lazy_pool_destroy(lazy_pool* p) { delete p; }

int lazy_pool_acquire(lazy_pool* p, int64_t doc_id, int32_t doc_tokens, int32_t logical_pos, int32_t* pages_out) {
  if (!p || doc_tokens <= 0 || !pages_out) return LAZY_ERR_INVALID;
  const int32_t need = (doc_tokens + p->page_size - 1) / p->page_size;
  const Key key{doc_id, p->keying == LAZY_POOL_POSITION_AWARE ? logical_pos : 0};
  p->lookups++;
  auto it = p->docs.find(key);
  if (it != p->docs.end()) {
    Entry& e = it->second;
    if ((int32_t)e.pages.size() != need) return LAZY_ERR_INVALID;     // a document's length is part of its identity
    if (e.in_lru) { p->lru.erase(e.lru_it); e.in_lru = false; }
    e.refcount++;
    p->hits++;
    for (int32_t i = 0; i < need; ++i) pages_out[i] = e.pages[i];
    return 1;
  }
  if (need > p->num_pages) return LAZY_ERR_WORKSPACE;
  while ((int32_t)p->free_pages.size() < need) {                       // evict unpinned documents, LRU first
    if (p->lru.empty()) return LAZY_ERR_WORKSPACE;                     // everything left is pinned by running requests
    const Key victim = p->lru.front();
    p->lru.pop_front();
    auto vit = p->docs.find(victim);
    for (int32_t pg : vit->second.pages) p->free_pages.push_back(pg);
    p->docs.erase(vit);
    p->evictions++;
  }
  Entry e;
  e.pages.resize(need);
  for (int32_t i = 0; i < need; ++i) { e.pages[i] = p->free_pages.back(); p->free_pages.pop_back(); }
  e.refcount = 1;
  for (int32_t i = 0; i < need; ++i) pages_out[i] = e.pages[i];
  p->docs.emplace(key, std::move(e));
  return 0;
}

int lazy_pool_release(lazy_pool* p, int64_t doc_id, int32_t logical_pos) {
  if (!p) return LAZY_ERR_INVALID;
  const Key key{doc_id, p->keying == LAZY_POOL_POSITION_AWARE ? logical_pos : 0};
  auto it = p->docs.find(key);
  if (it == p->docs.end() || it->second.refcount <= 0) return LAZY_ERR_INVALID;
  if (--it->second.refcount == 0) {
    p->lru.push_back(key);
    it->second.lru_it = std::prev(p->lru.end());
    it->second.in_lru = true;
  }
  return LAZY_OK;
}

void lazy_pool_stats(const lazy_pool* p, int64_t* lookups, int64_t* hits, int64_t* evictions, int32_t* pages_in_use) {
  if (!p) return;
  if (lookups) *lookups = p->lookups;
  if (hits) *hits = p->hits;
  if (evictions) *evictions = p->evictions;
  if (pages_in_use) *pages_in_use = p->num_pages - (int32_t)p->free_pages.size();
}

// PAPER.md Eq. 1 (positions == 1) and Eq. 2: sum_{i <= floor(C/positions)} i^-alpha / sum_{j <= N} j^-alpha
double lazy_hit_ratio_model(double alpha, int64_t num_docs, int64_t capacity_entries, int32_t positions) {
  if (num_docs <= 0 || capacity_entries < 0 || positions <= 0) return -1.0;
  int64_t top = capacity_entries / positions;
  if (top > num_docs) top = num_docs;
  double num = 0.0, den = 0.0;
  for (int64_t j = 1; j <= num_docs; ++j) {
    const double w = std::pow((double)j, -alpha);
    den += w;
    if (j <= top) num += w;
  }
  return num / den;
}

}  // extern "C"

"""LazyAttention hot path for B200 (sm_100a): paged attention over a position-free (un-rotated K) KV cache.

Public API = the C-ABI calls of include/lazy_attn.h with the same names (see binding.py).
"""

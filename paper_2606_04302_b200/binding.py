"""Thin ctypes binding over liblazyattn.so (include/lazy_attn.h) -- argument marshalling only.

Every function has the name and argument order of its C counterpart; tensors are torch CUDA tensors whose
`data_ptr()` is handed through, the stream is `torch.cuda.current_stream().cuda_stream` unless given.
Nothing here computes: if the CUDA library is missing the import of `lib()` raises (there is no fallback).
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "csrc", "liblazyattn.so")

LAZY_OK, LAZY_ERR_INVALID, LAZY_ERR_UNSUPPORTED, LAZY_ERR_WORKSPACE, LAZY_ERR_CUDA = 0, -1, -2, -3, -4
LAZY_ERR_STATIC_LIMIT = -5
LAZY_STATIC_SCRATCH_BYTES = 48 << 20
LAZY_FLAG_ROWWISE_KERNELS = 1
LAZY_FLAG_PREFILL_ONE_CTA = 2
LAZY_FLAG_FP8_DECODE_8_WARPS = 4
LAZY_K_UNROTATED, LAZY_K_STORED_POS, LAZY_K_ABSOLUTE = 0, 1, 2
LAZY_ROPE_HALF_SPLIT, LAZY_ROPE_INTERLEAVED, LAZY_POS_ALIBI = 0, 1, 2
LAZY_KV_BF16, LAZY_KV_FP8_E4M3 = 0, 1

EXPORTS = ["lazy_workspace_bytes", "lazy_create", "lazy_destroy", "lazy_cache_write", "lazy_attn_prefill",
           "lazy_attn_decode", "lazy_attn_decode_static", "lazy_set_rope_frequencies", "lazy_set_alibi_slopes", "lazy_set_page_stored_pos",
           "lazy_set_kv_scales",
           "lazy_materialize_pages", "lazy_status_string", "lazy_launch_count", "lazy_host_step_staging_bytes", "lazy_host_step", "lazy_host_step_layout", "lazy_host_step_packed",
           "lazy_attn_mixed", "lazy_debug_validate",
           "lazy_pool_create", "lazy_pool_destroy", "lazy_pool_acquire", "lazy_pool_release", "lazy_pool_stats",
           "lazy_hit_ratio_model"]
LAZY_POOL_AGNOSTIC, LAZY_POOL_POSITION_AWARE = 0, 1


class LazyConfig(ctypes.Structure):
    _fields_ = [("num_q_heads", ctypes.c_int32), ("num_kv_heads", ctypes.c_int32), ("head_dim", ctypes.c_int32),
                ("page_size", ctypes.c_int32), ("num_pages", ctypes.c_int32), ("max_position", ctypes.c_int32),
                ("max_reqs", ctypes.c_int32), ("max_pages_per_req", ctypes.c_int32),
                ("rope_theta", ctypes.c_double), ("rope_style", ctypes.c_int32), ("dtype", ctypes.c_int32),
                ("flags", ctypes.c_int32), ("k_storage", ctypes.c_int32)]


_lib: Optional[ctypes.CDLL] = None


def lib() -> ctypes.CDLL:
    """Loads the CUDA library; raises if it has not been built (python -m paper_2606_04302_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_04302_b200.build` "
                               "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
        L.lazy_workspace_bytes.restype = ctypes.c_size_t
        L.lazy_workspace_bytes.argtypes = [ctypes.POINTER(LazyConfig)]
        L.lazy_create.restype = ctypes.c_int
        L.lazy_create.argtypes = [ctypes.POINTER(LazyConfig), vp, ctypes.c_size_t, vp, ctypes.POINTER(vp)]
        L.lazy_destroy.restype = None
        L.lazy_destroy.argtypes = [vp]
        L.lazy_cache_write.restype = ctypes.c_int
        L.lazy_cache_write.argtypes = [vp, vp, vp, vp, i32, vp, vp, vp]
        L.lazy_attn_prefill.restype = ctypes.c_int
        L.lazy_attn_prefill.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, vp, vp]
        L.lazy_attn_decode.restype = ctypes.c_int
        L.lazy_attn_decode.argtypes = [vp, vp, vp, vp, vp, vp, vp, i32, vp, vp]
        L.lazy_attn_decode_static.restype = ctypes.c_int
        L.lazy_attn_decode_static.argtypes = [ctypes.POINTER(LazyConfig), vp, vp, vp, vp, vp, vp, i32, vp, vp]
        L.lazy_set_rope_frequencies.restype = ctypes.c_int
        L.lazy_set_rope_frequencies.argtypes = [vp, vp, ctypes.c_double, vp]
        L.lazy_set_alibi_slopes.restype = ctypes.c_int
        L.lazy_set_alibi_slopes.argtypes = [vp, vp, vp]
        L.lazy_set_page_stored_pos.restype = ctypes.c_int
        L.lazy_set_page_stored_pos.argtypes = [vp, vp]
        L.lazy_set_kv_scales.restype = ctypes.c_int
        L.lazy_set_kv_scales.argtypes = [vp, vp, vp]
        L.lazy_materialize_pages.restype = ctypes.c_int
        L.lazy_materialize_pages.argtypes = [vp, vp, vp, vp, vp, i32, vp, vp, vp, i32, vp]
        L.lazy_status_string.restype = ctypes.c_char_p
        L.lazy_status_string.argtypes = [ctypes.c_int]
        L.lazy_launch_count.restype = i64
        L.lazy_launch_count.argtypes = [vp]
        L.lazy_host_step_staging_bytes.restype = ctypes.c_size_t
        L.lazy_host_step_staging_bytes.argtypes = [vp, i32, i32, i32]
        L.lazy_host_step.restype = ctypes.c_int
        L.lazy_host_step.argtypes = [vp, ctypes.POINTER(HostStep), vp]
        L.lazy_host_step_layout.restype = ctypes.c_int
        L.lazy_host_step_layout.argtypes = [vp, i32, i32, i32, ctypes.POINTER(HostStepLayout)]
        L.lazy_host_step_packed.restype = ctypes.c_int
        L.lazy_host_step_packed.argtypes = [vp, ctypes.POINTER(HostStepPacked), vp]
        L.lazy_attn_mixed.restype = ctypes.c_int
        L.lazy_attn_mixed.argtypes = [vp, ctypes.POINTER(MixedArgs), vp, vp, vp]
        L.lazy_debug_validate.restype = i64
        L.lazy_debug_validate.argtypes = [vp, vp, vp, vp, i32, vp]
        L.lazy_pool_create.restype = vp
        L.lazy_pool_create.argtypes = [i32, i32, i32]
        L.lazy_pool_destroy.restype = None
        L.lazy_pool_destroy.argtypes = [vp]
        L.lazy_pool_acquire.restype = ctypes.c_int
        L.lazy_pool_acquire.argtypes = [vp, i64, i32, i32, ctypes.POINTER(i32)]
        L.lazy_pool_release.restype = ctypes.c_int
        L.lazy_pool_release.argtypes = [vp, i64, i32]
        L.lazy_pool_stats.restype = None
        L.lazy_pool_stats.argtypes = [vp, ctypes.POINTER(i64), ctypes.POINTER(i64), ctypes.POINTER(i64),
                                      ctypes.POINTER(i32)]
        L.lazy_hit_ratio_model.restype = ctypes.c_double
        L.lazy_hit_ratio_model.argtypes = [ctypes.c_double, i64, i64, i32]
        _lib = L
    return _lib


class LazyError(RuntimeError):
    def __init__(self, call: str, status: int):
        super().__init__(f"{call} failed: {status} ({lazy_status_string(status)})")
        self.status = status


def _ptr(t) -> Optional[int]:
    return None if t is None else t.data_ptr()


def _stream(stream) -> Optional[int]:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return getattr(stream, "cuda_stream", stream)


def lazy_status_string(status: int) -> str:
    return lib().lazy_status_string(int(status)).decode()


def lazy_workspace_bytes(cfg: LazyConfig) -> int:
    return int(lib().lazy_workspace_bytes(ctypes.byref(cfg)))


class LazyHandle:
    """Owns the torch workspace tensor and the C handle (lazy_create / lazy_destroy)."""

    def __init__(self, cfg: LazyConfig, device="cuda", stream=None):
        import torch
        n = lazy_workspace_bytes(cfg)
        if n == 0:
            raise LazyError("lazy_workspace_bytes", LAZY_ERR_UNSUPPORTED)
        self.cfg = cfg
        self.workspace = torch.empty(n + 256, dtype=torch.uint8, device=device)
        base = (self.workspace.data_ptr() + 255) // 256 * 256
        out = ctypes.c_void_p()
        rc = lib().lazy_create(ctypes.byref(cfg), base, n, _stream(stream), ctypes.byref(out))
        if rc != 0:
            raise LazyError("lazy_create", rc)
        self._h = out

    @property
    def ptr(self):
        return self._h

    def launch_count(self) -> int:
        return int(lib().lazy_launch_count(self._h))

    def close(self):
        if getattr(self, "_h", None):
            lib().lazy_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def lazy_create(num_q_heads: int, num_kv_heads: int, head_dim: int, *, num_pages: int, max_position: int,
                max_reqs: int, max_pages_per_req: int, rope_theta: float, page_size: int = 16, flags: int = 0,
                k_storage: int = LAZY_K_UNROTATED, rope_style: int = LAZY_ROPE_HALF_SPLIT, dtype: int = LAZY_KV_BF16,
                device="cuda", stream=None) -> LazyHandle:
    cfg = LazyConfig(num_q_heads, num_kv_heads, head_dim, page_size, num_pages, max_position, max_reqs,
                     max_pages_per_req, float(rope_theta), rope_style, dtype, flags, k_storage)
    return LazyHandle(cfg, device=device, stream=stream)


def lazy_destroy(h: LazyHandle) -> None:
    h.close()


def lazy_cache_write(h: LazyHandle, k_new, v_new, slot_mapping, k_cache, v_cache, stream=None) -> None:
    n = 0 if k_new is None else int(k_new.shape[0])
    rc = lib().lazy_cache_write(h.ptr, _ptr(k_new), _ptr(v_new), _ptr(slot_mapping), n, _ptr(k_cache),
                                _ptr(v_cache), _stream(stream))
    if rc != 0:
        raise LazyError("lazy_cache_write", rc)


def lazy_attn_prefill(h: LazyHandle, q, k_cache, v_cache, block_table, page_logical_pos, seq_lens, cu_q_lens,
                      max_q_len: int, out, stream=None) -> None:
    num_reqs = int(seq_lens.shape[0])
    total_q = int(q.shape[0])
    rc = lib().lazy_attn_prefill(h.ptr, _ptr(q), _ptr(k_cache), _ptr(v_cache), _ptr(block_table),
                                 _ptr(page_logical_pos), _ptr(seq_lens), _ptr(cu_q_lens), num_reqs, total_q,
                                 int(max_q_len), _ptr(out), _stream(stream))
    if rc != 0:
        raise LazyError("lazy_attn_prefill", rc)


def lazy_attn_decode(h: LazyHandle, q, k_cache, v_cache, block_table, page_logical_pos, seq_lens, out,
                     stream=None) -> None:
    num_reqs = int(seq_lens.shape[0])
    rc = lib().lazy_attn_decode(h.ptr, _ptr(q), _ptr(k_cache), _ptr(v_cache), _ptr(block_table),
                                _ptr(page_logical_pos), _ptr(seq_lens), num_reqs, _ptr(out), _stream(stream))
    if rc != 0:
        raise LazyError("lazy_attn_decode", rc)


def lazy_attn_decode_static(cfg: LazyConfig, q, k_cache, v_cache, block_table, page_logical_pos, seq_lens, out,
                            stream=None) -> None:
    """Decode for callers that cannot allocate device memory (no handle, no workspace tensor): the library's built-in
    LAZY_STATIC_SCRATCH_BYTES array is the scratch.  One call at a time per GPU; see include/lazy_attn.h."""
    num_reqs = int(seq_lens.shape[0])
    rc = lib().lazy_attn_decode_static(ctypes.byref(cfg), _ptr(q), _ptr(k_cache), _ptr(v_cache), _ptr(block_table),
                                       _ptr(page_logical_pos), _ptr(seq_lens), num_reqs, _ptr(out), _stream(stream))
    if rc != 0:
        raise LazyError("lazy_attn_decode_static", rc)


def lazy_set_rope_frequencies(h: LazyHandle, inv_freq=None, softmax_scale: float = 0.0, stream=None) -> None:
    """inv_freq: sequence of head_dim/2 floats (host) or None for the default theta^(-2j/D)."""
    arr = None
    if inv_freq is not None:
        vals = [float(x) for x in inv_freq]
        if len(vals) != h.cfg.head_dim // 2:
            raise LazyError("lazy_set_rope_frequencies", LAZY_ERR_INVALID)
        arr = (ctypes.c_double * len(vals))(*vals)
    rc = lib().lazy_set_rope_frequencies(h.ptr, arr, float(softmax_scale), _stream(stream))
    if rc != 0:
        raise LazyError("lazy_set_rope_frequencies", rc)


def lazy_set_alibi_slopes(h: LazyHandle, slopes, stream=None) -> None:
    """slopes: sequence of num_q_heads floats (host)."""
    vals = [float(x) for x in slopes]
    if len(vals) != h.cfg.num_q_heads:
        raise LazyError("lazy_set_alibi_slopes", LAZY_ERR_INVALID)
    arr = (ctypes.c_float * len(vals))(*vals)
    rc = lib().lazy_set_alibi_slopes(h.ptr, arr, _stream(stream))
    if rc != 0:
        raise LazyError("lazy_set_alibi_slopes", rc)


def lazy_set_page_stored_pos(h: LazyHandle, page_stored_pos) -> None:
    rc = lib().lazy_set_page_stored_pos(h.ptr, _ptr(page_stored_pos))
    if rc != 0:
        raise LazyError("lazy_set_page_stored_pos", rc)
    h._stored_pos = page_stored_pos          # the library keeps the pointer: keep the tensor alive with the handle


def lazy_set_kv_scales(h: LazyHandle, k_scale, v_scale) -> None:
    rc = lib().lazy_set_kv_scales(h.ptr, _ptr(k_scale), _ptr(v_scale))
    if rc != 0:
        raise LazyError("lazy_set_kv_scales", rc)
    h._kv_scales = (k_scale, v_scale)        # the library keeps the pointers: keep the tensors alive with the handle


def lazy_materialize_pages(h: LazyHandle, k_src, v_src, src_pages, rot_pos, per_token: bool, k_dst, v_dst,
                           dst_pages, stream=None) -> None:
    num = int(src_pages.shape[0])
    rc = lib().lazy_materialize_pages(h.ptr, _ptr(k_src), _ptr(v_src), _ptr(src_pages), _ptr(rot_pos),
                                      1 if per_token else 0, _ptr(k_dst), _ptr(v_dst), _ptr(dst_pages), num,
                                      _stream(stream))
    if rc != 0:
        raise LazyError("lazy_materialize_pages", rc)


def lazy_debug_validate(h: LazyHandle, block_table, page_logical_pos, seq_lens, stream=None) -> int:
    """Synchronising debug call: number of table entries the attention kernels would misuse."""
    rc = int(lib().lazy_debug_validate(h.ptr, _ptr(block_table), _ptr(page_logical_pos), _ptr(seq_lens),
                                       int(seq_lens.shape[0]), _stream(stream)))
    if rc < 0:
        raise LazyError("lazy_debug_validate", rc)
    return rc


class MixedArgs(ctypes.Structure):
    """Mirror of lazy_mixed_args (include/lazy_attn.h)."""
    _fields_ = [("q_prefill", ctypes.c_void_p), ("block_table_prefill", ctypes.c_void_p),
                ("page_logical_pos_prefill", ctypes.c_void_p), ("seq_lens_prefill", ctypes.c_void_p),
                ("cu_q_lens", ctypes.c_void_p), ("num_reqs_prefill", ctypes.c_int32), ("total_q", ctypes.c_int32),
                ("max_q_len", ctypes.c_int32), ("reserved0", ctypes.c_int32), ("out_prefill", ctypes.c_void_p),
                ("q_decode", ctypes.c_void_p), ("block_table_decode", ctypes.c_void_p),
                ("page_logical_pos_decode", ctypes.c_void_p), ("seq_lens_decode", ctypes.c_void_p),
                ("num_reqs_decode", ctypes.c_int32), ("decode_sms", ctypes.c_int32), ("out_decode", ctypes.c_void_p)]


def lazy_attn_mixed(h: LazyHandle, k_cache, v_cache, *, q_prefill, block_table_prefill, page_logical_pos_prefill,
                    seq_lens_prefill, cu_q_lens, max_q_len: int, out_prefill, q_decode, block_table_decode,
                    page_logical_pos_decode, seq_lens_decode, out_decode, decode_sms: int = 0, stream=None) -> None:
    args = MixedArgs(_ptr(q_prefill), _ptr(block_table_prefill), _ptr(page_logical_pos_prefill),
                     _ptr(seq_lens_prefill), _ptr(cu_q_lens), int(seq_lens_prefill.shape[0]), int(q_prefill.shape[0]),
                     int(max_q_len), 0, _ptr(out_prefill), _ptr(q_decode), _ptr(block_table_decode),
                     _ptr(page_logical_pos_decode), _ptr(seq_lens_decode), int(seq_lens_decode.shape[0]),
                     int(decode_sms), _ptr(out_decode))
    rc = lib().lazy_attn_mixed(h.ptr, ctypes.byref(args), _ptr(k_cache), _ptr(v_cache), _stream(stream))
    if rc != 0:
        raise LazyError("lazy_attn_mixed", rc)


class HostStepLayout(ctypes.Structure):
    """Mirror of lazy_host_step_layout_t: byte offsets of the sections of the packed host block."""
    _fields_ = [(n, ctypes.c_size_t) for n in ("q", "k_new", "v_new", "slot_mapping", "block_table", "page_logical_pos",
                                               "seq_lens", "cu_q_lens", "out", "in_bytes", "staging_bytes")]


class HostStepPacked(ctypes.Structure):
    """Mirror of lazy_host_step_packed_args."""
    _fields_ = [("kind", ctypes.c_int32), ("num_reqs", ctypes.c_int32), ("total_q", ctypes.c_int32),
                ("max_q_len", ctypes.c_int32), ("num_new_tokens", ctypes.c_int32), ("reserved", ctypes.c_int32),
                ("h_packed", ctypes.c_void_p), ("h_out", ctypes.c_void_p), ("d_k_cache", ctypes.c_void_p),
                ("d_v_cache", ctypes.c_void_p), ("d_staging", ctypes.c_void_p), ("staging_bytes", ctypes.c_size_t)]


class HostStep(ctypes.Structure):
    """Mirror of lazy_host_step_args (include/lazy_attn.h): one serving step with HOST buffers."""
    _fields_ = [("kind", ctypes.c_int32), ("num_reqs", ctypes.c_int32), ("total_q", ctypes.c_int32),
                ("max_q_len", ctypes.c_int32), ("num_new_tokens", ctypes.c_int32), ("reserved", ctypes.c_int32),
                ("h_q", ctypes.c_void_p), ("h_k_new", ctypes.c_void_p), ("h_v_new", ctypes.c_void_p),
                ("h_slot_mapping", ctypes.c_void_p), ("h_block_table", ctypes.c_void_p),
                ("h_page_logical_pos", ctypes.c_void_p), ("h_seq_lens", ctypes.c_void_p),
                ("h_cu_q_lens", ctypes.c_void_p), ("h_out", ctypes.c_void_p),
                ("d_k_cache", ctypes.c_void_p), ("d_v_cache", ctypes.c_void_p),
                ("d_staging", ctypes.c_void_p), ("staging_bytes", ctypes.c_size_t)]


def lazy_host_step_staging_bytes(h: LazyHandle, num_reqs: int, total_q: int, num_new_tokens: int) -> int:
    return int(lib().lazy_host_step_staging_bytes(h.ptr, num_reqs, total_q, num_new_tokens))


def lazy_host_step(h: LazyHandle, args: HostStep, stream=None) -> None:
    rc = lib().lazy_host_step(h.ptr, ctypes.byref(args), _stream(stream))
    if rc != 0:
        raise LazyError("lazy_host_step", rc)


def lazy_host_step_layout(h: LazyHandle, num_reqs: int, total_q: int, num_new_tokens: int) -> "HostStepLayout":
    out = HostStepLayout()
    rc = lib().lazy_host_step_layout(h.ptr, num_reqs, total_q, num_new_tokens, ctypes.byref(out))
    if rc != 0:
        raise LazyError("lazy_host_step_layout", rc)
    return out


def lazy_host_step_packed(h: LazyHandle, args: "HostStepPacked", stream=None) -> None:
    rc = lib().lazy_host_step_packed(h.ptr, ctypes.byref(args), _stream(stream))
    if rc != 0:
        raise LazyError("lazy_host_step_packed", rc)


class LazyPool:
    """Host page pool (lazy_pool_*): marshalling only."""

    def __init__(self, num_pages: int, page_size: int = 16, keying: int = LAZY_POOL_AGNOSTIC):
        self.page_size = page_size
        self._p = lib().lazy_pool_create(num_pages, page_size, keying)
        if not self._p:
            raise LazyError("lazy_pool_create", LAZY_ERR_INVALID)

    def acquire(self, doc_id: int, doc_tokens: int, logical_pos: int = 0):
        """Returns (hit: bool, pages: list[int]); raises LazyError when the document cannot be placed."""
        n = (doc_tokens + self.page_size - 1) // self.page_size
        buf = (ctypes.c_int32 * n)()
        rc = lib().lazy_pool_acquire(self._p, doc_id, doc_tokens, logical_pos, buf)
        if rc < 0:
            raise LazyError("lazy_pool_acquire", rc)
        return rc == 1, list(buf)

    def release(self, doc_id: int, logical_pos: int = 0) -> None:
        rc = lib().lazy_pool_release(self._p, doc_id, logical_pos)
        if rc != 0:
            raise LazyError("lazy_pool_release", rc)

    def stats(self) -> dict:
        a, b, c, d = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int32()
        lib().lazy_pool_stats(self._p, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c), ctypes.byref(d))
        return dict(lookups=a.value, hits=b.value, evictions=c.value, pages_in_use=d.value)

    def close(self):
        if getattr(self, "_p", None):
            lib().lazy_pool_destroy(self._p)
            self._p = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def lazy_hit_ratio_model(alpha: float, num_docs: int, capacity_entries: int, positions: int = 1) -> float:
    return float(lib().lazy_hit_ratio_model(alpha, num_docs, capacity_entries, positions))

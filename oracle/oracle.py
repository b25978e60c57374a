"""ctypes wrapper around oracle/lazy_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It imports nothing from paper_2606_04302_b200 (the CUDA path) and the CUDA path imports nothing from here.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lazy_oracle.c")
_LIB = os.path.join(_HERE, "liblazy_oracle.so")
_lib = None

DT_F64, DT_BF16 = 0, 1


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp; the oracle is compiled as it stands, never tuned."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _LIB


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.lazy_oracle_num_threads.restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(lib().lazy_oracle_num_threads())


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _as_kernel_input(t):
    """torch bf16 tensor -> (uint16 numpy view, DT_BF16); float array -> (float64 numpy, DT_F64)."""
    try:
        import torch
        if isinstance(t, torch.Tensor):
            if t.dtype == torch.bfloat16:
                return np.ascontiguousarray(t.contiguous().view(torch.int16).numpy()).view(np.uint16), DT_BF16
            return np.ascontiguousarray(t.double().numpy()), DT_F64
    except ImportError:
        pass
    return np.ascontiguousarray(np.asarray(t, dtype=np.float64)), DT_F64


def rope(x, pos: float, theta: float) -> np.ndarray:
    x = np.ascontiguousarray(np.asarray(x, dtype=np.float64))
    y = np.empty_like(x)
    f = lib().lazy_oracle_rope
    f.restype = None
    f(_p(x), ctypes.c_double(pos), ctypes.c_int(x.shape[-1]), ctypes.c_double(theta), _p(y))
    return y


class Variant(ctypes.Structure):
    """Mirror of lazy_oracle_variant (positional variants)."""
    _fields_ = [("rope_style", ctypes.c_int), ("inv_freq", ctypes.c_void_p), ("scale", ctypes.c_double),
                ("alibi_slopes", ctypes.c_void_p)]


def attend_core(q, k, v, pos_q, pos_k, vis, theta: float, row_select=None, want_probs=False, want_hats=False,
                rope_style: int = 0, inv_freq=None, scale: float = 0.0, alibi_slopes=None):
    """q [n_q,Hq,D], k/v [L,Hkv,D] float64; returns out (and probs [n_q,Hq,L], khat, qhat if asked)."""
    q = np.ascontiguousarray(np.asarray(q, dtype=np.float64))
    k = np.ascontiguousarray(np.asarray(k, dtype=np.float64))
    v = np.ascontiguousarray(np.asarray(v, dtype=np.float64))
    n_q, Hq, D = q.shape
    L, Hkv, _ = k.shape
    pos_q = np.ascontiguousarray(np.asarray(pos_q, dtype=np.float64))
    pos_k = np.ascontiguousarray(np.asarray(pos_k, dtype=np.float64))
    vis = np.ascontiguousarray(np.asarray(vis, dtype=np.int64))
    out = np.zeros((n_q, Hq, D), dtype=np.float64)
    probs = np.zeros((n_q, Hq, L), dtype=np.float64) if want_probs else None
    khat = np.zeros((L, Hkv, D), dtype=np.float64) if want_hats else None
    qhat = np.zeros((n_q, Hq, D), dtype=np.float64) if want_hats else None
    rs = None if row_select is None else np.ascontiguousarray(np.asarray(row_select, dtype=np.uint8))
    fr = None if inv_freq is None else np.ascontiguousarray(np.asarray(inv_freq, dtype=np.float64))
    sl = None if alibi_slopes is None else np.ascontiguousarray(np.asarray(alibi_slopes, dtype=np.float64))
    var = Variant(int(rope_style), None if fr is None else fr.ctypes.data, float(scale),
                  None if sl is None else sl.ctypes.data)
    f = lib().lazy_oracle_attend_core_ex
    f.restype = ctypes.c_int
    rc = f(_p(q), _p(k), _p(v), _p(pos_q), _p(pos_k), _p(vis), ctypes.c_int(n_q), ctypes.c_int64(L),
           ctypes.c_int(Hq), ctypes.c_int(Hkv), ctypes.c_int(D), ctypes.c_double(theta), ctypes.byref(var), None,
           _p(rs), _p(out), _p(probs), _p(khat), _p(qhat))
    if rc != 0:
        raise RuntimeError(f"lazy_oracle_attend_core failed: {rc}")
    res = [out]
    if want_probs:
        res.append(probs)
    if want_hats:
        res += [khat, qhat]
    return res[0] if len(res) == 1 else tuple(res)


def attend_paged(q, k_pool, v_pool, block_table, page_logical_pos, seq_lens, cu_q_lens, *,
                 num_q_heads: int, num_kv_heads: int, head_dim: int, page_size: int, theta: float,
                 row_select=None, k_storage: int = 0, page_stored_pos=None, rope_style: int = 0, inv_freq=None,
                 scale: float = 0.0, alibi_slopes=None) -> np.ndarray:
    """Paged interface.  q [total_q,Hq,D]; pools [num_pages,Hkv,P,D] (torch bf16 or float arrays).
    k_storage 0: pages hold un-rotated K; 1: page g holds K rotated at page_stored_pos[g] + t (the paper's
    document-local layout); 2: K already rotated at its final position.
    Returns out [total_q,Hq,D] float64 (rows not selected stay 0)."""
    qa, dq = _as_kernel_input(q)
    ka, dk = _as_kernel_input(k_pool)
    va, dv = _as_kernel_input(v_pool)
    assert dk == dv
    bt = np.ascontiguousarray(np.asarray(block_table, dtype=np.int32))
    pp = np.ascontiguousarray(np.asarray(page_logical_pos, dtype=np.int32))
    assert bt.shape == pp.shape and bt.ndim == 2
    sl = np.ascontiguousarray(np.asarray(seq_lens, dtype=np.int32))
    cu = np.ascontiguousarray(np.asarray(cu_q_lens, dtype=np.int32))
    R = sl.shape[0]
    total_q = int(cu[-1])
    out = np.zeros((total_q, num_q_heads, head_dim), dtype=np.float64)
    rs = None if row_select is None else np.ascontiguousarray(np.asarray(row_select, dtype=np.uint8))
    sp = None if page_stored_pos is None else np.ascontiguousarray(np.asarray(page_stored_pos, dtype=np.int32))
    fr = None if inv_freq is None else np.ascontiguousarray(np.asarray(inv_freq, dtype=np.float64))
    al = None if alibi_slopes is None else np.ascontiguousarray(np.asarray(alibi_slopes, dtype=np.float64))
    f = lib().lazy_oracle_attend_paged_variant
    f.restype = ctypes.c_int
    rc = f(_p(qa), ctypes.c_int(dq), _p(ka), _p(va), ctypes.c_int(dk), _p(bt), _p(pp),
           ctypes.c_int64(bt.shape[1]), _p(sl), _p(cu), ctypes.c_int(R), ctypes.c_int(num_q_heads),
           ctypes.c_int(num_kv_heads), ctypes.c_int(head_dim), ctypes.c_int(page_size), ctypes.c_double(theta),
           ctypes.c_int(k_storage), _p(sp), ctypes.c_int(rope_style), _p(fr), ctypes.c_double(scale), _p(al),
           _p(rs), _p(out))
    if rc != 0:
        raise RuntimeError(f"lazy_oracle_attend_paged_variant failed: {rc}")
    return out


def materialize_pages(k_pool, src_pages, rot_pos, per_token: bool, theta: float) -> np.ndarray:
    """fp64 [num,Hkv,P,D]: page src_pages[i] rotated by rot_pos[i] (+ t if per_token)."""
    ka, dk = _as_kernel_input(k_pool)
    _, Hkv, P, D = ka.shape
    sp = np.ascontiguousarray(np.asarray(src_pages, dtype=np.int32))
    rp = np.ascontiguousarray(np.asarray(rot_pos, dtype=np.int32))
    assert sp.shape == rp.shape and sp.ndim == 1
    out = np.zeros((sp.shape[0], Hkv, P, D), dtype=np.float64)
    f = lib().lazy_oracle_materialize_pages
    f.restype = ctypes.c_int
    rc = f(_p(ka), ctypes.c_int(dk), _p(sp), _p(rp), ctypes.c_int(1 if per_token else 0),
           ctypes.c_int64(sp.shape[0]), ctypes.c_int(Hkv), ctypes.c_int(D), ctypes.c_int(P), ctypes.c_double(theta),
           _p(out))
    if rc != 0:
        raise RuntimeError(f"lazy_oracle_materialize_pages failed: {rc}")
    return out


def cache_write(k_new, v_new, slot_mapping, k_pool, v_pool, page_size: int) -> None:
    """In-place bit copy into torch bf16 pools [num_pages,Hkv,P,D] (shared memory with numpy views)."""
    import torch
    assert k_pool.dtype == torch.bfloat16 and k_pool.is_contiguous() and v_pool.is_contiguous()
    kn = np.ascontiguousarray(k_new.contiguous().view(torch.int16).numpy()).view(np.uint16)
    vn = np.ascontiguousarray(v_new.contiguous().view(torch.int16).numpy()).view(np.uint16)
    kp = k_pool.view(torch.int16).numpy().view(np.uint16)
    vp = v_pool.view(torch.int16).numpy().view(np.uint16)
    sm = np.ascontiguousarray(np.asarray(slot_mapping, dtype=np.int64))
    T, Hkv, D = kn.shape
    f = lib().lazy_oracle_cache_write
    f.restype = ctypes.c_int
    rc = f(_p(kn), _p(vn), _p(sm), ctypes.c_int64(T), ctypes.c_int(Hkv), ctypes.c_int(D), ctypes.c_int(page_size),
           ctypes.c_int64(k_pool.shape[0]), _p(kp), _p(vp))
    if rc != 0:
        raise RuntimeError(f"lazy_oracle_cache_write failed: {rc}")


# ---- FP8 KV pages: E4M3 codes + one fp32 scale per (page, kv head, token) -------------------
def e4m3_to_double(codes) -> np.ndarray:
    c = np.ascontiguousarray(np.asarray(codes, dtype=np.uint8))
    f = lib().lazy_oracle_e4m3_to_double
    f.restype = ctypes.c_double
    f.argtypes = [ctypes.c_uint8]
    return np.array([f(int(x)) for x in c.ravel()], dtype=np.float64).reshape(c.shape)


def e4m3_from_float(x) -> np.ndarray:
    a = np.ascontiguousarray(np.asarray(x, dtype=np.float32))
    f = lib().lazy_oracle_e4m3_from_float
    f.restype = ctypes.c_uint8
    f.argtypes = [ctypes.c_float]
    return np.array([f(float(v)) for v in a.ravel()], dtype=np.uint8).reshape(a.shape)


class Fp8Pools:
    """The oracle's own FP8 page pools (numpy): codes [num_pages,Hkv,P,D] uint8, scales [num_pages,Hkv,P] float32.
    Unwritten rows hold the NaN code 0x7f and a NaN scale, so that a kernel reading past a tail is caught."""

    def __init__(self, num_pages: int, Hkv: int, P: int, D: int):
        self.k_codes = np.full((num_pages, Hkv, P, D), 0x7f, dtype=np.uint8)
        self.v_codes = np.full((num_pages, Hkv, P, D), 0x7f, dtype=np.uint8)
        self.k_scale = np.full((num_pages, Hkv, P), np.nan, dtype=np.float32)
        self.v_scale = np.full((num_pages, Hkv, P), np.nan, dtype=np.float32)


def cache_write_fp8(k_new, v_new, slot_mapping, pools: Fp8Pools) -> None:
    """Quantise bf16 rows [T,Hkv,D] (torch) into the FP8 pools, in place."""
    import torch
    kn = np.ascontiguousarray(k_new.contiguous().view(torch.int16).numpy()).view(np.uint16)
    vn = np.ascontiguousarray(v_new.contiguous().view(torch.int16).numpy()).view(np.uint16)
    sm = np.ascontiguousarray(np.asarray(slot_mapping, dtype=np.int64))
    T, Hkv, D = kn.shape
    num_pages, _, P, _ = pools.k_codes.shape
    f = lib().lazy_oracle_cache_write_fp8
    f.restype = ctypes.c_int
    rc = f(_p(kn), _p(vn), _p(sm), ctypes.c_int64(T), ctypes.c_int(Hkv), ctypes.c_int(D), ctypes.c_int(P),
           ctypes.c_int64(num_pages), _p(pools.k_codes), _p(pools.v_codes), _p(pools.k_scale), _p(pools.v_scale))
    if rc != 0:
        raise RuntimeError(f"lazy_oracle_cache_write_fp8 failed: {rc}")


def quantize_pool_fp8(k_pool, v_pool) -> Fp8Pools:
    """FP8 pools holding the quantised content of whole bf16 pools [num_pages,Hkv,P,D]: every slot whose K and V
    rows are finite is written once; poisoned (NaN) slots of the bf16 pools stay poisoned (skipped)."""
    import torch
    num_pages, Hkv, P, D = k_pool.shape
    pools = Fp8Pools(num_pages, Hkv, P, D)
    kn = k_pool.permute(0, 2, 1, 3).reshape(num_pages * P, Hkv, D)
    vn = v_pool.permute(0, 2, 1, 3).reshape(num_pages * P, Hkv, D)
    ok = torch.isfinite(kn.float()).all(dim=(1, 2)) & torch.isfinite(vn.float()).all(dim=(1, 2))
    slots = np.where(ok.numpy(), np.arange(num_pages * P, dtype=np.int64), -1)
    cache_write_fp8(kn, vn, slots, pools)
    return pools


def attend_paged_fp8(q, pools: Fp8Pools, block_table, page_logical_pos, seq_lens, cu_q_lens, *,
                     num_q_heads: int, num_kv_heads: int, head_dim: int, page_size: int, theta: float,
                     row_select=None, rope_style: int = 0, inv_freq=None, scale: float = 0.0,
                     alibi_slopes=None) -> np.ndarray:
    """attend_paged over FP8 pages: exact dequantisation, then the unchanged definition."""
    qa, dq = _as_kernel_input(q)
    bt = np.ascontiguousarray(np.asarray(block_table, dtype=np.int32))
    pp = np.ascontiguousarray(np.asarray(page_logical_pos, dtype=np.int32))
    assert bt.shape == pp.shape and bt.ndim == 2
    sl = np.ascontiguousarray(np.asarray(seq_lens, dtype=np.int32))
    cu = np.ascontiguousarray(np.asarray(cu_q_lens, dtype=np.int32))
    out = np.zeros((int(cu[-1]), num_q_heads, head_dim), dtype=np.float64)
    rs = None if row_select is None else np.ascontiguousarray(np.asarray(row_select, dtype=np.uint8))
    fr = None if inv_freq is None else np.ascontiguousarray(np.asarray(inv_freq, dtype=np.float64))
    al = None if alibi_slopes is None else np.ascontiguousarray(np.asarray(alibi_slopes, dtype=np.float64))
    f = lib().lazy_oracle_attend_paged_fp8
    f.restype = ctypes.c_int
    rc = f(_p(qa), ctypes.c_int(dq), _p(pools.k_codes), _p(pools.v_codes), _p(pools.k_scale), _p(pools.v_scale),
           _p(bt), _p(pp), ctypes.c_int64(bt.shape[1]), _p(sl), _p(cu), ctypes.c_int(sl.shape[0]),
           ctypes.c_int(num_q_heads), ctypes.c_int(num_kv_heads), ctypes.c_int(head_dim), ctypes.c_int(page_size),
           ctypes.c_double(theta), ctypes.c_int(rope_style), _p(fr), ctypes.c_double(scale), _p(al), _p(rs), _p(out))
    if rc != 0:
        raise RuntimeError(f"lazy_oracle_attend_paged_fp8 failed: {rc}")
    return out


def run_step_fp8(batch, step, pools: Fp8Pools, row_select=None, **variant) -> Optional[np.ndarray]:
    """run_step over FP8 pools: quantising cache write, then attention over the dequantised pages."""
    sh = batch.shape
    if step.k_new is not None:
        cache_write_fp8(step.k_new, step.v_new, step.slot_mapping.numpy(), pools)
    if step.kind == "write_only":
        return None
    bt, pp = batch.block_table, batch.page_logical_pos
    if step.req_ids is not None:
        bt, pp = bt[step.req_ids], pp[step.req_ids]
    return attend_paged_fp8(step.q, pools, bt.numpy(), pp.numpy(), step.seq_lens.numpy(), step.cu_q_lens.numpy(),
                            num_q_heads=sh.num_q_heads, num_kv_heads=sh.num_kv_heads, head_dim=sh.head_dim,
                            page_size=sh.page_size, theta=sh.rope_theta, row_select=row_select, **variant)


def run_step(batch, step, k_pool, v_pool, row_select=None, **variant) -> Optional[np.ndarray]:
    """Apply one workloads.Step with the oracle: cache write (in place on the given pool copies),
    then the attention call.  Returns the fp64 output or None for write-only steps."""
    sh = batch.shape
    if step.k_new is not None:
        cache_write(step.k_new, step.v_new, step.slot_mapping.numpy(), k_pool, v_pool, sh.page_size)
    if step.kind == "write_only":
        return None
    bt, pp = batch.block_table, batch.page_logical_pos
    if step.req_ids is not None:
        bt, pp = bt[step.req_ids], pp[step.req_ids]
    return attend_paged(step.q, k_pool, v_pool, bt.numpy(), pp.numpy(), step.seq_lens.numpy(),
                        step.cu_q_lens.numpy(), num_q_heads=sh.num_q_heads, num_kv_heads=sh.num_kv_heads,
                        head_dim=sh.head_dim, page_size=sh.page_size, theta=sh.rope_theta, row_select=row_select,
                        **variant)

"""Device-side driver for a workloads.LazyBatch: uploads the pool and tables, creates the handle and runs
the batch's steps through the C-ABI binding.  Marshalling only -- every step of the path runs in the CUDA
kernels of liblazyattn.so.  Used by tests/, bench.py and __graft_entry__.smoke()."""
from __future__ import annotations

from typing import List, Optional

import torch

from . import binding as B
from .workloads import LazyBatch, Step


class DeviceBatch:
    def __init__(self, batch: LazyBatch, device: str = "cuda", flags: int = 0, max_position: Optional[int] = None,
                 k_storage: int = B.LAZY_K_UNROTATED, page_stored_pos: Optional[torch.Tensor] = None,
                 k_pool: Optional[torch.Tensor] = None, v_pool: Optional[torch.Tensor] = None,
                 block_table: Optional[torch.Tensor] = None, rope_style: int = B.LAZY_ROPE_HALF_SPLIT,
                 inv_freq=None, softmax_scale: float = 0.0, alibi_slopes=None, dtype: int = B.LAZY_KV_BF16):
        """k_pool / v_pool / block_table override the batch's own (the stored-position and absolute layouts of
        SURVEY 8.0 row f1 hold differently encoded K, the absolute one also private pages per request)."""
        self.batch = batch
        self.device = torch.device(device)
        sh = batch.shape
        self.dtype = dtype
        src_k = batch.k_pool if k_pool is None else k_pool
        src_v = batch.v_pool if v_pool is None else v_pool
        if dtype == B.LAZY_KV_FP8_E4M3:
            # code pools start as the E4M3 NaN code and the scales as NaN: only lazy_cache_write makes a row valid
            self.k_pool = torch.full(tuple(src_k.shape), 0x7f, dtype=torch.uint8, device=self.device)
            self.v_pool = torch.full(tuple(src_k.shape), 0x7f, dtype=torch.uint8, device=self.device)
            self.k_scale = torch.full(tuple(src_k.shape[:3]), float("nan"), dtype=torch.float32, device=self.device)
            self.v_scale = torch.full(tuple(src_k.shape[:3]), float("nan"), dtype=torch.float32, device=self.device)
        else:
            self.k_pool = src_k.to(self.device)
            self.v_pool = src_v.to(self.device)
        self.block_table = (batch.block_table if block_table is None else block_table).to(self.device)
        self.page_logical_pos = batch.page_logical_pos.to(self.device)
        R, pmax = batch.block_table.shape
        self.handle = B.lazy_create(sh.num_q_heads, sh.num_kv_heads, sh.head_dim, num_pages=int(self.k_pool.shape[0]),
                                    max_position=max_position or batch.max_position, max_reqs=R,
                                    max_pages_per_req=pmax, rope_theta=sh.rope_theta, page_size=sh.page_size,
                                    flags=flags, k_storage=k_storage, rope_style=rope_style, dtype=dtype,
                                    device=self.device)
        if dtype == B.LAZY_KV_FP8_E4M3:
            B.lazy_set_kv_scales(self.handle, self.k_scale, self.v_scale)
            self._quantize_pool(src_k, src_v)
        if alibi_slopes is not None:
            B.lazy_set_alibi_slopes(self.handle, alibi_slopes)
        if inv_freq is not None or softmax_scale:
            B.lazy_set_rope_frequencies(self.handle, inv_freq, softmax_scale)
        if page_stored_pos is not None:
            B.lazy_set_page_stored_pos(self.handle, page_stored_pos.to(self.device, dtype=torch.int32).contiguous())

    def _quantize_pool(self, src_k: torch.Tensor, src_v: torch.Tensor, pages_per_call: int = 4096) -> None:
        """FP8 pages: the batch's bf16 pool content goes through lazy_cache_write (the library's quantiser), one slot
        per finite (page, token) row; poisoned rows of the bf16 pool stay poisoned."""
        num_pages, Hkv, P, D = src_k.shape
        for p0 in range(0, num_pages, pages_per_call):
            p1 = min(num_pages, p0 + pages_per_call)
            kn = src_k[p0:p1].permute(0, 2, 1, 3).reshape(-1, Hkv, D).contiguous()
            vn = src_v[p0:p1].permute(0, 2, 1, 3).reshape(-1, Hkv, D).contiguous()
            ok = torch.isfinite(kn.float()).all(dim=(1, 2)) & torch.isfinite(vn.float()).all(dim=(1, 2))
            slots = torch.arange(p0 * P, p1 * P, dtype=torch.int64)
            slots = torch.where(ok, slots, torch.full_like(slots, -1))
            B.lazy_cache_write(self.handle, kn.to(self.device), vn.to(self.device), slots.to(self.device),
                               self.k_pool, self.v_pool)
        torch.cuda.synchronize(self.device)

    def tables_for(self, step: Step):
        if step.req_ids is None:
            return self.block_table, self.page_logical_pos
        ids = step.req_ids.to(self.device)
        return self.block_table[ids].contiguous(), self.page_logical_pos[ids].contiguous()

    def write(self, step: Step) -> None:
        if step.k_new is None:
            return
        B.lazy_cache_write(self.handle, step.k_new.to(self.device), step.v_new.to(self.device),
                           step.slot_mapping.to(self.device), self.k_pool, self.v_pool)

    def attend(self, step: Step) -> Optional[torch.Tensor]:
        if step.kind == "write_only":
            return None
        bt, pp = self.tables_for(step)
        q = step.q.to(self.device)
        out = torch.empty_like(q)
        sl = step.seq_lens.to(self.device)
        if step.kind == "decode":
            B.lazy_attn_decode(self.handle, q, self.k_pool, self.v_pool, bt, pp, sl, out)
        else:
            cu = step.cu_q_lens.to(self.device)
            max_q = int((step.cu_q_lens[1:] - step.cu_q_lens[:-1]).max())
            B.lazy_attn_prefill(self.handle, q, self.k_pool, self.v_pool, bt, pp, sl, cu, max_q, out)
        return out

    def run_step(self, step: Step) -> Optional[torch.Tensor]:
        self.write(step)
        return self.attend(step)

    def run_all(self) -> List[Optional[torch.Tensor]]:
        return [self.run_step(s) for s in self.batch.steps]

    def close(self):
        self.handle.close()

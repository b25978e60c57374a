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
                 inv_freq=None, softmax_scale: float = 0.0, alibi_slopes=None):
        """k_pool / v_pool / block_table override the batch's own (the stored-position and absolute layouts of
        SURVEY 8.0 row f1 hold differently encoded K, the absolute one also private pages per request)."""
        self.batch = batch
        self.device = torch.device(device)
        sh = batch.shape
        self.k_pool = (batch.k_pool if k_pool is None else k_pool).to(self.device)
        self.v_pool = (batch.v_pool if v_pool is None else v_pool).to(self.device)
        self.block_table = (batch.block_table if block_table is None else block_table).to(self.device)
        self.page_logical_pos = batch.page_logical_pos.to(self.device)
        R, pmax = batch.block_table.shape
        self.handle = B.lazy_create(sh.num_q_heads, sh.num_kv_heads, sh.head_dim, num_pages=int(self.k_pool.shape[0]),
                                    max_position=max_position or batch.max_position, max_reqs=R,
                                    max_pages_per_req=pmax, rope_theta=sh.rope_theta, page_size=sh.page_size,
                                    flags=flags, k_storage=k_storage, rope_style=rope_style, device=self.device)
        if alibi_slopes is not None:
            B.lazy_set_alibi_slopes(self.handle, alibi_slopes)
        if inv_freq is not None or softmax_scale:
            B.lazy_set_rope_frequencies(self.handle, inv_freq, softmax_scale)
        if page_stored_pos is not None:
            B.lazy_set_page_stored_pos(self.handle, page_stored_pos.to(self.device, dtype=torch.int32).contiguous())

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

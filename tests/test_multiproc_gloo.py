"""N > 1 host logic on CPU (world_size 2, gloo): attention shards by request with NO data-path exchange
(DESIGN.md 'Multi-GPU: replicas only'), so two ranks that each own `shard_requests(R, rank, 2)` of a batch and never
talk during the computation reproduce the one-process result; the only collectives are the bench's barrier and its
max-over-ranks timing reduction.  The per-rank computation here is the oracle (no GPU in this test)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import oracle as O
from paper_2606_04302_b200 import workloads as W


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _decode_rows(batch, step, rows):
    sh = batch.shape
    k, v = batch.k_pool.clone(), batch.v_pool.clone()
    for st in batch.steps:
        if st.k_new is not None:
            O.cache_write(st.k_new, st.v_new, st.slot_mapping.numpy(), k, v, sh.page_size)
    rows = list(rows)
    return O.attend_paged(step.q[rows], k, v, batch.block_table[rows].numpy(), batch.page_logical_pos[rows].numpy(),
                          step.seq_lens[rows].numpy(), np.arange(len(rows) + 1, dtype=np.int32),
                          num_q_heads=sh.num_q_heads, num_kv_heads=sh.num_kv_heads, head_dim=sh.head_dim,
                          page_size=sh.page_size, theta=sh.rope_theta)


def _worker(rank, world, port, out_path):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        batch = W.config2(scale=0.05)
        step = [s for s in batch.steps if s.kind == "decode"][0]
        R = step.seq_lens.shape[0]
        mine = W.shard_requests(R, rank, world)
        dist.barrier()
        part = torch.from_numpy(_decode_rows(batch, step, mine))
        # the bench's timing reduction: MAX over ranks of the per-rank time
        t = torch.tensor([10.0 + rank], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        assert t.item() == 10.0 + world - 1
        parts = [None] * world
        dist.all_gather_object(parts, (list(mine), part))
        if rank == 0:
            full = np.zeros((R,) + tuple(part.shape[1:]))
            seen = []
            for rows, p in parts:
                full[rows] = p.numpy()
                seen += rows
            assert sorted(seen) == list(range(R))
            ref = _decode_rows(batch, step, range(R))
            np.save(out_path, np.array([np.abs(full - ref).max()]))
    finally:
        dist.destroy_process_group()


def test_request_parallel_shards_reproduce_the_single_process_result(tmp_path):
    out = str(tmp_path / "err.npy")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    assert float(np.load(out)[0]) == 0.0

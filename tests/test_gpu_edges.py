"""-m gpu edge cases: empty and ragged inputs, partial pages, repeated pages, position gaps, skipped slots,
argument errors, and the read-only property of the read path."""
import ctypes

import numpy as np
import pytest
import torch

from paper_2606_04302_b200 import binding as B
from paper_2606_04302_b200 import workloads as W
from paper_2606_04302_b200.runner import DeviceBatch

pytestmark = pytest.mark.gpu
FLAGS = [pytest.param(0, id="prod"), pytest.param(B.LAZY_FLAG_ROWWISE_KERNELS, id="rowwise")]


def _custom(shape, seq_lens, q_lens, *, seed, repeat_pages=False, pos_gap=0, unaligned_pos=False, kind="prefill"):
    """Hand-built batch: every request owns ceil(L/16) pages (or re-uses its first page repeatedly);
    positions may have gaps and need not be multiples of 16."""
    P = shape.page_size
    gen = torch.Generator().manual_seed(seed)
    rng = np.random.default_rng(seed)
    R = len(seq_lens)
    npages = [(L + P - 1) // P for L in seq_lens]
    pmax = max(max(npages), 1)
    total_pages = sum(npages) + 3
    k_pool = W._randn_bf16(gen, (total_pages, shape.num_kv_heads, P, shape.head_dim))
    v_pool = W._randn_bf16(gen, (total_pages, shape.num_kv_heads, P, shape.head_dim))
    perm = rng.permutation(total_pages)
    bt = np.zeros((R, pmax), dtype=np.int32)
    pp = np.zeros((R, pmax), dtype=np.int32)
    c = 0
    for r in range(R):
        ids = perm[c:c + npages[r]].copy()
        c += npages[r]
        if repeat_pages and npages[r] > 2:
            ids[2::2] = ids[0]                      # the same physical page at several slots of one request
        bt[r, :npages[r]] = ids
        pos = P * np.arange(npages[r])
        if pos_gap:
            pos = pos + pos_gap * (np.arange(npages[r]) // 3)      # jump every 3 pages
        if unaligned_pos:
            pos = pos + 5
        pp[r, :npages[r]] = pos
    # poison the tail of every last page (tokens >= L must never be read into the result)
    for r in range(R):
        L = seq_lens[r]
        if L % P and not repeat_pages:
            k_pool[bt[r, npages[r] - 1], :, L % P:, :] = float("nan")
            v_pool[bt[r, npages[r] - 1], :, L % P:, :] = float("nan")
    tq = int(sum(q_lens))
    q = W._randn_bf16(gen, (max(tq, 1), shape.num_q_heads, shape.head_dim))[:tq]
    cu = np.concatenate([[0], np.cumsum(q_lens)]).astype(np.int32)
    step = W.Step(kind=kind, q=q, seq_lens=torch.tensor(seq_lens, dtype=torch.int32),
                  cu_q_lens=torch.from_numpy(cu))
    return W.LazyBatch(name="custom", shape=shape, k_pool=k_pool, v_pool=v_pool,
                       block_table=torch.from_numpy(bt), page_logical_pos=torch.from_numpy(pp), steps=[step])


def _check(batch, flags=0):
    from gpu_util import run_and_compare
    return run_and_compare(batch, flags=flags)


SH128 = W.LazyShape(32, 8, 128, 5.0e5)
SH64 = W.LazyShape(4, 1, 64, 1.0e4)
SH7 = W.LazyShape(28, 4, 128, 1.0e6)


@pytest.mark.parametrize("flags", FLAGS)
@pytest.mark.parametrize("shape", [SH128, SH64, SH7], ids=["g4d128", "g4d64", "g7d128"])
def test_ragged_decode(shape, flags):
    seq = [1, 2, 15, 16, 17, 31, 33, 100, 257, 640, 1000, 3]
    _check(_custom(shape, seq, [1] * len(seq), seed=11, kind="decode"), flags)


@pytest.mark.parametrize("flags", FLAGS)
@pytest.mark.parametrize("shape", [SH128, SH64, SH7], ids=["g4d128", "g4d64", "g7d128"])
def test_ragged_prefill(shape, flags):
    seq = [5, 16, 200, 129, 300, 47, 1]
    qls = [5, 3, 200, 1, 130, 47, 1]          # includes block-local (q_len == seq_len) and single rows
    _check(_custom(shape, seq, qls, seed=12), flags)


@pytest.mark.parametrize("flags", FLAGS)
def test_zero_length_requests(flags):
    seq = [0, 40, 0]
    b = _custom(SH128, seq, [1, 1, 1], seed=13, kind="decode")
    dev = DeviceBatch(b, flags=flags)
    out = dev.run_step(b.steps[0])
    torch.cuda.synchronize()
    assert (out[0] == 0).all() and (out[2] == 0).all() and out[1].float().abs().sum() > 0
    dev.close()
    _check(b, flags)
    # prefill with an empty request in the middle (no query rows, seq_len 0)
    _check(_custom(SH128, [33, 0, 20], [4, 0, 20], seed=14), flags)


@pytest.mark.parametrize("flags", FLAGS)
def test_repeated_pages_gaps_and_unaligned_positions(flags):
    _check(_custom(SH128, [200, 333], [1, 1], seed=15, repeat_pages=True, kind="decode"), flags)
    _check(_custom(SH128, [200, 333], [8, 70], seed=16, repeat_pages=True, pos_gap=1000), flags)
    _check(_custom(SH128, [77, 160], [1, 1], seed=17, pos_gap=4096, unaligned_pos=True, kind="decode"), flags)
    _check(_custom(SH64, [77, 160], [30, 160], seed=18, pos_gap=512, unaligned_pos=True), flags)


def test_one_page_two_positions_equals_two_copies():
    """north_star check 4 / PAPER.md L37, L88: a page used at two slots == a byte-identical duplicate."""
    b = _custom(SH128, [160], [1], seed=19, kind="decode")
    bt = b.block_table.clone()
    x, dup = int(bt[0, 1]), int(bt[0, 5])
    shared = W.LazyBatch(name="s", shape=b.shape, k_pool=b.k_pool.clone(), v_pool=b.v_pool.clone(),
                         block_table=bt.clone(), page_logical_pos=b.page_logical_pos, steps=b.steps)
    shared.block_table[0, 5] = x                      # page x at slots 1 and 5
    copied = W.LazyBatch(name="c", shape=b.shape, k_pool=b.k_pool.clone(), v_pool=b.v_pool.clone(),
                         block_table=bt.clone(), page_logical_pos=b.page_logical_pos, steps=b.steps)
    copied.k_pool[dup] = copied.k_pool[x]
    copied.v_pool[dup] = copied.v_pool[x]
    outs = []
    for bb in (shared, copied):
        dev = DeviceBatch(bb)
        outs.append(dev.run_step(bb.steps[0]).float().cpu())
        dev.close()
    assert torch.equal(outs[0], outs[1])
    _check(shared)


def test_empty_calls_and_errors():
    b = W.config1()
    dev = DeviceBatch(b)
    h = dev.handle
    n0 = h.launch_count()
    L = B.lib()
    z = torch.zeros(16, dtype=torch.int32, device="cuda")
    # zero-sized calls launch nothing and succeed
    assert L.lazy_cache_write(h.ptr, None, None, None, 0, None, None, None) == 0
    assert L.lazy_attn_decode(h.ptr, None, None, None, None, None, None, 0, None, None) == 0
    assert L.lazy_attn_prefill(h.ptr, None, None, None, None, None, None, None, 0, 0, 0, None, None) == 0
    assert h.launch_count() == n0
    # errors: too many requests, null pointers, misaligned pointer
    p = z.data_ptr()
    assert L.lazy_attn_decode(h.ptr, p, p, p, p, p, p, 2, p, None) == B.LAZY_ERR_INVALID      # max_reqs = 1
    assert L.lazy_attn_decode(h.ptr, None, p, p, p, p, p, 1, p, None) == B.LAZY_ERR_INVALID
    assert L.lazy_attn_decode(h.ptr, p + 2, p, p, p, p, p, 1, p, None) == B.LAZY_ERR_INVALID
    assert L.lazy_cache_write(h.ptr, p, p, p, -1, p, p, None) == B.LAZY_ERR_INVALID
    assert h.launch_count() == n0
    dev.close()


def test_cache_write_skips_negative_slots_and_is_bit_exact():
    from oracle import oracle as O
    b = W.config5(scale=0.25)
    step = b.steps[0]
    slots = step.slot_mapping.clone()
    slots[::7] = -1
    s2 = W.Step(kind="write_only", k_new=step.k_new, v_new=step.v_new, slot_mapping=slots)
    dev = DeviceBatch(b)
    k_ref, v_ref = b.k_pool.clone(), b.v_pool.clone()
    dev.write(s2)
    torch.cuda.synchronize()
    O.cache_write(s2.k_new, s2.v_new, slots.numpy(), k_ref, v_ref, 16)
    assert torch.equal(dev.k_pool.cpu().view(torch.int16), k_ref.view(torch.int16))
    assert torch.equal(dev.v_pool.cpu().view(torch.int16), v_ref.view(torch.int16))
    dev.close()


def test_host_step_matches_device_calls():
    """lazy_host_step (HOST buffers, copies inside) == the device-pointer calls."""
    b = W.config2(scale=0.1)
    step = b.steps[-1]
    dev = DeviceBatch(b)
    dev.write(b.steps[0])
    want = dev.run_step(step)
    torch.cuda.synchronize()
    dev2 = DeviceBatch(b)
    dev2.write(b.steps[0])
    pin = lambda t: t.contiguous().pin_memory()
    hq, hk, hv, hs = pin(step.q), pin(step.k_new), pin(step.v_new), pin(step.slot_mapping)
    hbt, hpp, hsl = pin(b.block_table), pin(b.page_logical_pos), pin(step.seq_lens)
    hout = torch.empty_like(step.q).pin_memory()
    R = step.seq_lens.shape[0]
    nbytes = B.lazy_host_step_staging_bytes(dev2.handle, R, R, step.k_new.shape[0])
    staging = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
    base = (staging.data_ptr() + 255) // 256 * 256
    a = B.HostStep(0, R, R, 1, step.k_new.shape[0], 0, hq.data_ptr(), hk.data_ptr(), hv.data_ptr(), hs.data_ptr(),
                   hbt.data_ptr(), hpp.data_ptr(), hsl.data_ptr(), None, hout.data_ptr(),
                   dev2.k_pool.data_ptr(), dev2.v_pool.data_ptr(), base, nbytes)
    B.lazy_host_step(dev2.handle, a)
    torch.cuda.synchronize()
    assert torch.equal(hout.view(torch.int16), want.cpu().view(torch.int16))
    dev.close(); dev2.close()


def _packed_step(dev, batch, step):
    """One step through lazy_host_step_layout + lazy_host_step_packed (the call bench.py's e2e leg times): the caller
    packs every input into one pinned block at the offsets the library states."""
    bt = batch.block_table if step.req_ids is None else batch.block_table[step.req_ids]
    pp = batch.page_logical_pos if step.req_ids is None else batch.page_logical_pos[step.req_ids]
    R, tq = step.seq_lens.shape[0], step.q.shape[0]
    nn = 0 if step.k_new is None else step.k_new.shape[0]
    lay = B.lazy_host_step_layout(dev.handle, R, tq, nn)
    assert lay.staging_bytes == B.lazy_host_step_staging_bytes(dev.handle, R, tq, nn)
    assert lay.in_bytes == lay.out and lay.out < lay.staging_bytes
    offs = [lay.q, lay.k_new, lay.v_new, lay.slot_mapping, lay.block_table, lay.page_logical_pos, lay.seq_lens,
            lay.cu_q_lens, lay.out]
    assert all(o % 256 == 0 for o in offs) and offs == sorted(offs)
    packed = torch.full((int(lay.in_bytes),), 0xA5, dtype=torch.uint8).pin_memory()     # gaps hold junk

    def put(off, t):
        raw = t.contiguous().view(torch.uint8).reshape(-1)
        packed[off:off + raw.numel()] = raw
    put(lay.q, step.q)
    if nn:
        put(lay.k_new, step.k_new); put(lay.v_new, step.v_new); put(lay.slot_mapping, step.slot_mapping)
    put(lay.block_table, bt.to(torch.int32)); put(lay.page_logical_pos, pp.to(torch.int32))
    put(lay.seq_lens, step.seq_lens)
    kind, max_q = 0, 1
    if step.kind == "prefill":
        kind = 1
        put(lay.cu_q_lens, step.cu_q_lens)
        max_q = int((step.cu_q_lens[1:] - step.cu_q_lens[:-1]).max())
    hout = torch.full_like(step.q, float("nan")).pin_memory()
    staging = torch.empty(int(lay.staging_bytes) + 256, dtype=torch.uint8, device="cuda")
    base = (staging.data_ptr() + 255) // 256 * 256
    args = B.HostStepPacked(kind, R, tq, max_q, nn, 0, packed.data_ptr(), hout.data_ptr(), dev.k_pool.data_ptr(),
                            dev.v_pool.data_ptr(), base, int(lay.staging_bytes))
    B.lazy_host_step_packed(dev.handle, args)
    torch.cuda.synchronize()
    return hout


@pytest.mark.parametrize("cfg,scale", [(2, 0.1), (3, 0.05), (5, 0.2)])
def test_host_step_packed_matches_oracle_and_device_calls(cfg, scale):
    """lazy_host_step_layout + lazy_host_step_packed, decode and prefill kinds: every step of the batch (cache write
    included) through the packed call on one handle, through the device-pointer calls on another and through the
    oracle; pools bit-equal afterwards."""
    from oracle import oracle as O
    from gpu_util import compare
    b = W.CONFIGS[cfg](scale=scale)
    dev, dev2 = DeviceBatch(b), DeviceBatch(b)
    k_ref, v_ref = b.k_pool.clone(), b.v_pool.clone()
    kinds = set()
    try:
        for si, step in enumerate(b.steps):
            want = dev.run_step(step)
            ref = O.run_step(b, step, k_ref, v_ref)
            if step.kind == "write_only":
                dev2.write(step)
                continue
            got = _packed_step(dev2, b, step)
            kinds.add(step.kind)
            compare(got, ref, f"cfg{cfg} step {si} ({step.kind}) packed host step")
            if step.kind == "prefill":                                     # same kernel, same grid: bit equal
                assert torch.equal(got.view(torch.int16), want.cpu().view(torch.int16))
            else:                                                          # split-KV summation order may differ
                assert (got.float() - want.cpu().float()).abs().max().item() < 2e-3
            assert torch.equal(dev2.k_pool.cpu().view(torch.int16), k_ref.view(torch.int16))
            assert torch.equal(dev2.v_pool.cpu().view(torch.int16), v_ref.view(torch.int16))
        assert kinds
    finally:
        dev.close(); dev2.close()


def test_host_step_packed_rejects_bad_arguments():
    b = W.config2(scale=0.05)
    dev = DeviceBatch(b)
    try:
        lay = B.lazy_host_step_layout(dev.handle, 4, 4, 4)
        a = B.HostStepPacked(0, 4, 4, 1, 4, 0, None, None, None, None, None, 0)
        with pytest.raises(B.LazyError):
            B.lazy_host_step_packed(dev.handle, a)
        staging = torch.empty(int(lay.staging_bytes) + 256, dtype=torch.uint8, device="cuda")
        base = (staging.data_ptr() + 255) // 256 * 256
        host = torch.zeros(int(lay.in_bytes), dtype=torch.uint8).pin_memory()
        hout = torch.zeros(4 * b.shape.num_q_heads * b.shape.head_dim, dtype=torch.bfloat16).pin_memory()
        a = B.HostStepPacked(0, 4, 4, 1, 4, 0, host.data_ptr(), hout.data_ptr(), dev.k_pool.data_ptr(),
                             dev.v_pool.data_ptr(), base, int(lay.staging_bytes) - 1)
        with pytest.raises(B.LazyError) as e:
            B.lazy_host_step_packed(dev.handle, a)
        assert e.value.status == B.LAZY_ERR_WORKSPACE
        with pytest.raises(B.LazyError):
            B.lazy_host_step_layout(dev.handle, -1, 4, 4)
    finally:
        dev.close()


def test_many_requests_cross_the_per_launch_limit():
    """Maximum sizes: more requests than one decode launch keeps in shared memory (2048) -> lazy_attn_decode splits
    the batch into several launches; many short prefill chunks -> one CTA per (request, kv head)."""
    rng = np.random.default_rng(3)
    R = 2300
    lens = rng.integers(0, 40, size=R).tolist()
    lens[5] = 0
    lens[2047] = 33; lens[2048] = 17; lens[2299] = 1
    _check(_custom(SH64, lens, [1] * R, seed=21, kind="decode"))
    R = 300
    lens = rng.integers(1, 50, size=R).tolist()
    qs = [int(min(L, rng.integers(1, 20))) for L in lens]
    _check(_custom(SH64, lens, qs, seed=22))


def test_long_chunk_prefill_and_single_key():
    """A 2 000-token chunk over a short prefix (many m-blocks per request, mostly causal tiles) next to a request
    whose query sees exactly one key."""
    _check(_custom(SH128, [2100, 1, 130], [2000, 1, 130], seed=23))
    _check(_custom(SH7, [1500, 1], [1500, 1], seed=24))


def test_debug_validate_counts_bad_table_entries():
    batch = W.config2(scale=0.05)
    dev = DeviceBatch(batch)
    try:
        st = [s for s in batch.steps if s.kind == "decode"][0]
        bt, pp = dev.tables_for(st)
        sl = st.seq_lens.cuda()
        assert B.lazy_debug_validate(dev.handle, bt, pp, sl) == 0
        bt2, pp2, sl2 = bt.clone(), pp.clone(), sl.clone()
        bt2[0, 0] = batch.num_pages            # page id out of range
        bt2[1, 3] = -1
        pp2[0, 1] = batch.max_position         # position beyond the table
        sl2[2] = bt.shape[1] * 16 + 1          # longer than the table row
        assert B.lazy_debug_validate(dev.handle, bt2, pp2, sl2) == 4
        bt2[0, bt.shape[1] - 1] = -7           # beyond ceil(seq_len / 16): ignored, as the attention calls do
        sl3 = sl.clone()
        sl3[0] = 100
        assert B.lazy_debug_validate(dev.handle, bt2, pp2, sl3) == 3
    finally:
        dev.close()

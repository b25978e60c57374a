"""-m gpu parity tests for SURVEY.md 8.0 rows f1 / f2: the stored-position K layouts (the paper's own
document-local cache, and the position-dependent "rotation compiled out" arm of its overhead ablation) and the
materialising page re-encoding, each against the fp64 oracle on the same seeded inputs.

The pre-rotated pools the attention kernels read here are built on the CPU by the ORACLE
(oracle.materialize_pages, fp64, rounded once to bf16) -- never by the CUDA path -- so the attention parity
does not depend on lazy_materialize_pages, which has its own test."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2606_04302_b200 import binding as B
from paper_2606_04302_b200 import workloads as W
from paper_2606_04302_b200.runner import DeviceBatch

from gpu_util import compare

pytestmark = pytest.mark.gpu

FLAGS = [pytest.param(0, id="prod"), pytest.param(B.LAZY_FLAG_ROWWISE_KERNELS, id="rowwise")]


@pytest.fixture(scope="module", autouse=True)
def _lib():
    from paper_2606_04302_b200 import build
    build.build()
    B.lib()


def _filled_pools(batch):
    """CPU pools after every cache write of the batch (un-rotated, bit copies), NaN tails turned into zeros so
    that a rotated copy of a poisoned row is still poisoned only where it was (rope(NaN) is NaN anyway)."""
    k, v = batch.k_pool.clone(), batch.v_pool.clone()
    for st in batch.steps:
        if st.k_new is not None:
            O.cache_write(st.k_new, st.v_new, st.slot_mapping.numpy(), k, v, batch.shape.page_size)
    return k, v


def _to_bf16(x: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(x).to(torch.float32).to(torch.bfloat16)


def _attend_steps(batch):
    return [s for s in batch.steps if s.kind != "write_only"]


def _oracle(batch, step, k, v, bt, **kw):
    sh = batch.shape
    pp = batch.page_logical_pos
    if step.req_ids is not None:
        bt, pp = bt[step.req_ids], pp[step.req_ids]
    return O.attend_paged(step.q, k, v, bt.numpy(), pp.numpy(), step.seq_lens.numpy(), step.cu_q_lens.numpy(),
                          num_q_heads=sh.num_q_heads, num_kv_heads=sh.num_kv_heads, head_dim=sh.head_dim,
                          page_size=sh.page_size, theta=sh.rope_theta, **kw)


@pytest.mark.parametrize("flags", FLAGS)
@pytest.mark.parametrize("cfg,scale", [(1, None), (2, 0.1), (3, 0.05), (5, 0.15)])
def test_stored_position_layout(cfg, scale, flags):
    """PAPER.md L173 / L409 layout: page g holds K rotated at stored[g] + t; the kernels apply one relative
    rotation per page (K tile in prefill, Eq. 5; q in decode, Eq. 6).  Stored starts are arbitrary multiples of
    16, some LARGER than the logical start (negative relative offset)."""
    batch = W.config1() if cfg == 1 else W.CONFIGS[cfg](scale=scale)
    sh = batch.shape
    k, v = _filled_pools(batch)
    g = np.arange(batch.num_pages)
    stored = (16 * ((g * 7919) % 41)).astype(np.int32)
    k_st = _to_bf16(O.materialize_pages(k, g.astype(np.int32), stored, True, sh.rope_theta))
    dev = DeviceBatch(batch, flags=flags, k_storage=B.LAZY_K_STORED_POS, page_stored_pos=torch.from_numpy(stored),
                      k_pool=k_st, v_pool=v, max_position=batch.max_position + 16 * 41 + 16)
    try:
        for st in _attend_steps(batch):
            got = dev.attend(st)
            torch.cuda.synchronize()
            ref = _oracle(batch, st, k_st, v, batch.block_table, k_storage=1, page_stored_pos=stored)
            compare(got, ref, f"{batch.name} stored-pos {st.kind}")
        assert torch.equal(dev.k_pool.cpu().view(torch.int16), k_st.view(torch.int16))     # read path is read-only
    finally:
        dev.close()


def _absolute_copies(batch, k, v):
    """Private page per (request, slot), K rotated at its final position (what a position-dependent cache holds)."""
    sh = batch.shape
    R, pmax = batch.block_table.shape
    src = batch.block_table.numpy().reshape(-1).astype(np.int32)
    starts = batch.page_logical_pos.numpy().reshape(-1).astype(np.int32)
    k_abs = _to_bf16(O.materialize_pages(k, src, starts, True, sh.rope_theta))
    v_abs = v[torch.from_numpy(src.astype(np.int64))].clone()
    bt_abs = torch.arange(R * pmax, dtype=torch.int32).view(R, pmax)
    return k_abs, v_abs, bt_abs


@pytest.mark.parametrize("flags", FLAGS)
@pytest.mark.parametrize("cfg,scale", [(1, None), (2, 0.1), (3, 0.05), (5, 0.15)])
def test_absolute_layout_rotation_compiled_out(cfg, scale, flags):
    """The 'without deferred rotation' arm of PAPER.md Fig. 5 (L271-297): K stored at its final position, no K
    rotation in the kernels, q rotated by its own position."""
    batch = W.config1() if cfg == 1 else W.CONFIGS[cfg](scale=scale)
    k, v = _filled_pools(batch)
    k_abs, v_abs, bt_abs = _absolute_copies(batch, k, v)
    dev = DeviceBatch(batch, flags=flags, k_storage=B.LAZY_K_ABSOLUTE, k_pool=k_abs, v_pool=v_abs, block_table=bt_abs)
    try:
        for st in _attend_steps(batch):
            got = dev.attend(st)
            torch.cuda.synchronize()
            ref = _oracle(batch, st, k_abs, v_abs, bt_abs, k_storage=2)
            compare(got, ref, f"{batch.name} absolute {st.kind}")
    finally:
        dev.close()


def test_three_layouts_agree_on_gpu():
    """the lazy path is 'mathematically identical' to duplicating + re-encoding.  Same batch through
    the three layouts on the GPU: outputs agree within the rounding of the bf16 pre-rotated copies."""
    batch = W.config2(scale=0.1)
    k, v = _filled_pools(batch)
    outs = {}
    dev = DeviceBatch(batch, k_pool=k, v_pool=v)
    outs["lazy"] = [dev.attend(s).float().cpu() for s in _attend_steps(batch)]
    dev.close()
    k_abs, v_abs, bt_abs = _absolute_copies(batch, k, v)
    dev = DeviceBatch(batch, k_storage=B.LAZY_K_ABSOLUTE, k_pool=k_abs, v_pool=v_abs, block_table=bt_abs)
    outs["abs"] = [dev.attend(s).float().cpu() for s in _attend_steps(batch)]
    dev.close()
    for a, b in zip(outs["lazy"], outs["abs"]):
        assert (a - b).abs().max().item() < 4e-3


@pytest.mark.parametrize("D,Hkv", [(128, 8), (64, 1), (128, 4)])
def test_materialize_pages_matches_oracle(D, Hkv):
    """f2: copy + rotate whole pages.  K within one bf16 ulp of the fp64 oracle and
    bit-equal to its RNE rounding almost everywhere; V a bit copy; untouched pages untouched; per-token and
    relative (negative) rotations; re-encoding in place."""
    gen = torch.Generator().manual_seed(5)
    num_pages, theta = 40, 5e5
    k = torch.randn(num_pages, Hkv, 16, D, generator=gen).to(torch.bfloat16)
    v = torch.randn(num_pages, Hkv, 16, D, generator=gen).to(torch.bfloat16)
    h = B.lazy_create(Hkv * 4, Hkv, D, num_pages=num_pages, max_position=140000, max_reqs=4, max_pages_per_req=8,
                      rope_theta=theta)
    try:
        for per_token, rot in ((True, [0, 16, 4096, 131056, 77, 1]), (False, [0, -16, 5000, -131071, 3, -1])):
            src = np.array([3, 3, 17, 39, 0, 21], np.int32)
            dst = np.array([30, 31, 5, 6, 7, 8], np.int32)
            rot = np.array(rot, np.int32)
            kd, vd = k.cuda(), v.cuda()
            kdst, vdst = kd.clone(), vd.clone()
            B.lazy_materialize_pages(h, kd, vd, torch.from_numpy(src).cuda(), torch.from_numpy(rot).cuda(), per_token,
                                     kdst, vdst, torch.from_numpy(dst).cuda())
            torch.cuda.synchronize()
            ref = O.materialize_pages(k, src, rot, per_token, theta)
            got = kdst.cpu()[torch.from_numpy(dst.astype(np.int64))].double().numpy()
            err = np.abs(got - ref)
            # half a bf16 ulp is <= 2^-8 |x|; near a rounding tie the fp32 pipeline may round the other way
            assert (err <= np.abs(ref) * 2.0 ** -8 * 1.02 + 1e-7).all(), (err - np.abs(ref) * 2.0 ** -8).max()
            exact = _to_bf16(ref).double().numpy() == got
            assert exact.mean() > 0.995, exact.mean()
            assert torch.equal(vdst.cpu()[torch.from_numpy(dst.astype(np.int64))].view(torch.int16),
                               v[torch.from_numpy(src.astype(np.int64))].view(torch.int16))
            untouched = np.setdiff1d(np.arange(num_pages), dst)
            assert torch.equal(kdst.cpu()[untouched].view(torch.int16), k[untouched].view(torch.int16))
            assert torch.equal(kd.cpu().view(torch.int16), k.view(torch.int16))           # source pool never written
        # in place, K only (v pointers NULL): encode then move by a relative offset == encode at the sum
        pages = torch.tensor([2, 9], dtype=torch.int32).cuda()
        kd = k.cuda()
        B.lazy_materialize_pages(h, kd, None, pages, torch.tensor([100, 7], dtype=torch.int32).cuda(), True, kd, None, pages)
        B.lazy_materialize_pages(h, kd, None, pages, torch.tensor([23, -7], dtype=torch.int32).cuda(), False, kd, None, pages)
        torch.cuda.synchronize()
        ref = O.materialize_pages(k, np.array([2, 9], np.int32), np.array([123, 0], np.int32), True, theta)
        got = kd.cpu()[[2, 9]].double().numpy()
        # two roundings: the first one's error (<= 2^-8 of each component) is mixed across the pair by the second
        # rotation, so the bound is relative to the pair's norm (which rotations preserve), not to the element
        half = D // 2
        pair = np.sqrt(ref[..., :half] ** 2 + ref[..., half:] ** 2)
        pair = np.concatenate([pair, pair], axis=-1)
        assert (np.abs(got - ref) <= pair * 2.0 ** -7 * 1.1 + 1e-6).all()
        # degenerate / error paths
        B.lazy_materialize_pages(h, kd, None, pages[:0], pages[:0], True, kd, None, pages[:0])
        rc = B.lib().lazy_materialize_pages(h.ptr, None, None, pages.data_ptr(), pages.data_ptr(), 1, kd.data_ptr(),
                                            None, pages.data_ptr(), 2, None)
        assert rc == B.LAZY_ERR_INVALID
    finally:
        h.close()


def test_stored_pos_requires_table():
    batch = W.config1()
    dev = DeviceBatch(batch, k_storage=B.LAZY_K_STORED_POS)
    try:
        st = _attend_steps(batch)[0]
        with pytest.raises(B.LazyError):
            dev.attend(st)
    finally:
        dev.close()
    dev = DeviceBatch(batch)
    try:
        with pytest.raises(B.LazyError):
            B.lazy_set_page_stored_pos(dev.handle, torch.zeros(batch.num_pages, dtype=torch.int32, device="cuda"))
    finally:
        dev.close()

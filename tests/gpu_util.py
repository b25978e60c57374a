"""Helpers shared by the -m gpu parity tests: run a LazyBatch through the CUDA path (C ABI) and through the
fp64 oracle on the same seeded inputs, and compare.  Tolerances: BASELINE.json north_star (max abs <= 2e-2,
mean abs <= 2e-3 on outputs) plus the tighter self-imposed normalised gates of DESIGN.md "Tolerances"."""
from __future__ import annotations

import numpy as np
import torch

from oracle import oracle as O
from paper_2606_04302_b200.runner import DeviceBatch

MAX_ABS, MEAN_ABS = 2e-2, 2e-3          # contract (north_star)
REL_RMS, REL_MAX = 1.0e-2, 5e-2         # self-imposed: RMS(err)/RMS(ref), max|err| / max|ref|


def compare(got: torch.Tensor, ref: np.ndarray, what: str = "", rows=None, abs_scale: float = 1.0,
            rel_rms: float = None, rel_max: float = None):
    """abs_scale > 1 only for the peaked (q x4) variants, whose outputs are O(1): the absolute contract is then
    scaled by the output magnitude (bf16 output rounding alone is |out| * 2^-9) -- DESIGN.md 'Tolerances'."""
    g = got.detach().double().cpu().numpy()
    if rows is not None:
        g, ref = g[rows], ref[rows]
    assert np.isfinite(g).all(), f"{what}: non-finite GPU output"
    err = np.abs(g - ref)
    rms_ref = float(np.sqrt((ref ** 2).mean()))
    stats = dict(max_abs=float(err.max()), mean_abs=float(err.mean()),
                 rel_rms=float(np.sqrt((err ** 2).mean()) / max(rms_ref, 1e-30)),
                 rel_max=float(err.max() / max(np.abs(ref).max(), 1e-30)))
    assert stats["max_abs"] <= MAX_ABS * abs_scale and stats["mean_abs"] <= MEAN_ABS * abs_scale, \
        f"{what}: contract violated {stats}"
    assert stats["rel_rms"] <= (rel_rms or REL_RMS) and stats["rel_max"] <= (rel_max or REL_MAX), \
        f"{what}: normalised gate violated {stats}"
    return stats


def run_and_compare(batch, flags: int = 0, sample_rows: int = 0, seed: int = 0, max_position=None,
                    scale_abs_by_output: bool = False, dev_kw=None, oracle_kw=None, k_perm=None, gates=None):
    """Runs every step on the GPU and on the oracle (oracle pools are separate CPU copies).  With
    sample_rows > 0 the oracle computes only that many seeded query rows per attention step."""
    """dev_kw / oracle_kw: the same positional variant handed to the CUDA handle and to the oracle; k_perm: order
    in which the library stores K's last axis (LAZY_ROPE_INTERLEAVED de-interleaves on write; pre-loaded pages must be
    uploaded in that order, dev_kw["k_pool"])."""
    dev = DeviceBatch(batch, flags=flags, max_position=max_position, **(dev_kw or {}))
    k_ref, v_ref = batch.k_pool.clone(), batch.v_pool.clone()
    rng = np.random.default_rng(seed)
    all_stats = []
    try:
        for si, step in enumerate(batch.steps):
            got = dev.run_step(step)
            torch.cuda.synchronize()
            sel = rows = None
            if step.q is not None and sample_rows and step.q.shape[0] > sample_rows:
                rows = np.sort(rng.choice(step.q.shape[0], size=sample_rows, replace=False))
                sel = np.zeros(step.q.shape[0], dtype=np.uint8)
                sel[rows] = 1
            ref = O.run_step(batch, step, k_ref, v_ref, row_select=sel, **(oracle_kw or {}))
            # pools must agree bit for bit after the step's cache write, and stay so after the read path
            k_expect = k_ref if k_perm is None else k_ref[..., k_perm]
            assert torch.equal(dev.k_pool.cpu().view(torch.int16), k_expect.view(torch.int16)), f"step {si}: K pool"
            assert torch.equal(dev.v_pool.cpu().view(torch.int16), v_ref.view(torch.int16)), f"step {si}: V pool"
            if got is not None:
                sc = max(1.0, float(np.abs(ref).max())) if scale_abs_by_output else 1.0
                kw = dict(abs_scale=sc)
                kw.update(gates or {})
                all_stats.append(compare(got, ref, f"{batch.name} step {si} ({step.kind})", rows=rows, **kw))
    finally:
        dev.close()
    return all_stats


def run_and_compare_fp8(batch, flags: int = 0, sample_rows: int = 0, seed: int = 0, scale_abs_by_output: bool = False,
                        gates=None, dev_kw=None, oracle_kw=None, k_perm=None):
    """FP8 KV pages (LAZY_KV_FP8_E4M3): the library quantises (lazy_cache_write), the oracle quantises its own copy;
    codes and scales must agree BIT FOR BIT after every step (integer decisions taken in fp32 on both sides), and the
    attention outputs must match the oracle's exact-dequantisation result under the same gates as the bf16 path."""
    from paper_2606_04302_b200 import binding as B
    dev = DeviceBatch(batch, flags=flags, dtype=B.LAZY_KV_FP8_E4M3, **(dev_kw or {}))
    pools = O.quantize_pool_fp8(batch.k_pool, batch.v_pool)
    rng = np.random.default_rng(seed)
    all_stats = []

    def check_pools(si):
        kc, vc = dev.k_pool.cpu().numpy(), dev.v_pool.cpu().numpy()
        ks, vs = dev.k_scale.cpu().numpy().view(np.uint32), dev.v_scale.cpu().numpy().view(np.uint32)
        valid = ~np.isnan(pools.k_scale)
        assert np.array_equal(np.isnan(dev.k_scale.cpu().numpy()), ~valid), f"step {si}: which rows are written"
        assert np.array_equal(ks[valid], pools.k_scale.view(np.uint32)[valid]), f"step {si}: K scales"
        assert np.array_equal(vs[valid], pools.v_scale.view(np.uint32)[valid]), f"step {si}: V scales"
        # k_perm: order in which the library stores K's last axis (LAZY_ROPE_INTERLEAVED de-interleaves on write)
        assert np.array_equal(kc, pools.k_codes if k_perm is None else pools.k_codes[..., k_perm]), f"step {si}: K codes"
        assert np.array_equal(vc, pools.v_codes), f"step {si}: V codes"

    try:
        check_pools(-1)
        for si, step in enumerate(batch.steps):
            got = dev.run_step(step)
            torch.cuda.synchronize()
            sel = rows = None
            if step.q is not None and sample_rows and step.q.shape[0] > sample_rows:
                rows = np.sort(rng.choice(step.q.shape[0], size=sample_rows, replace=False))
                sel = np.zeros(step.q.shape[0], dtype=np.uint8)
                sel[rows] = 1
            ref = O.run_step_fp8(batch, step, pools, row_select=sel, **(oracle_kw or {}))
            check_pools(si)
            if got is not None:
                sc = max(1.0, float(np.abs(ref).max())) if scale_abs_by_output else 1.0
                kw = dict(abs_scale=sc)
                kw.update(gates or {})
                all_stats.append(compare(got, ref, f"{batch.name} fp8 step {si} ({step.kind})", rows=rows, **kw))
    finally:
        dev.close()
    return all_stats

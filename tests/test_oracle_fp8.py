"""Pins of the oracle's FP8-page functions against things other than
themselves: the OCP E4M3 value table, torch's independent float8_e4m3fn conversion, the nearest-value property by brute
force, closed forms of the per-row scale, and equality of the FP8 attention with the already pinned fp64 path on pools
dequantised outside the oracle."""
import math

import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2606_04302_b200 import workloads as W

THETA = 10000.0


def _golden_e4m3():
    """tests/golden/e4m3_values.txt: values written out from the OCP FP8 definition (S.EEEE.MMM, bias 7)."""
    import os
    rows = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "e4m3_values.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                code, val = line.split()
                rows[int(code, 16)] = float(val)
    return rows


def test_e4m3_decode_golden_values():
    for code, val in _golden_e4m3().items():
        got = float(O.e4m3_to_double(np.array([code], dtype=np.uint8))[0])
        assert got == val, (hex(code), got, val)
    assert math.isnan(float(O.e4m3_to_double(np.array([0x7f], dtype=np.uint8))[0]))
    assert math.isnan(float(O.e4m3_to_double(np.array([0xff], dtype=np.uint8))[0]))


def test_e4m3_decode_matches_torch_float8_all_codes():
    c = np.arange(256, dtype=np.uint8)
    ours = O.e4m3_to_double(c)
    ref = torch.from_numpy(c.copy()).view(torch.float8_e4m3fn).double().numpy()
    assert np.array_equal(np.isnan(ours), np.isnan(ref))
    assert np.array_equal(ours[~np.isnan(ours)], ref[~np.isnan(ref)])
    # monotone in the code over the non-negative finite range, symmetric in sign
    assert np.all(np.diff(ours[:0x7f]) > 0)
    assert np.array_equal(ours[0x80:0xff], -ours[0x00:0x7f])


def test_e4m3_encode_is_nearest_value_brute_force():
    rng = np.random.default_rng(7)
    x = np.concatenate([rng.standard_normal(3000) * s for s in (1e-3, 0.05, 1.0, 30.0, 200.0)]).astype(np.float32)
    x = x[np.abs(x) <= 448.0]
    codes = O.e4m3_from_float(x)
    vals = O.e4m3_to_double(np.arange(256, dtype=np.uint8))
    finite = ~np.isnan(vals)
    got = vals[codes]
    best = np.min(np.abs(x.astype(np.float64)[:, None] - vals[finite][None, :]), axis=1)
    assert np.array_equal(np.abs(x.astype(np.float64) - got), best)
    # and torch's independent round-to-nearest-even conversion picks the same codes
    ref = torch.from_numpy(x.copy()).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    assert np.array_equal(codes, ref)


def test_e4m3_encode_ties_to_even_round_trip_and_saturation():
    vals = O.e4m3_to_double(np.arange(0x7f, dtype=np.uint8))
    # exact midpoints between neighbours go to the code with an even mantissa bit
    mid = ((vals[:-1] + vals[1:]) / 2).astype(np.float32)
    assert np.array_equal(mid.astype(np.float64), (vals[:-1] + vals[1:]) / 2)      # representable in fp32
    got = O.e4m3_from_float(mid)
    want = np.array([c if c % 2 == 0 else c + 1 for c in range(0x7e)], dtype=np.uint8)
    assert np.array_equal(got, want)
    assert np.array_equal(O.e4m3_from_float(-mid), want | 0x80)
    # every finite code survives decode -> encode
    allc = np.array([c for c in range(256) if c not in (0x7f, 0xff)], dtype=np.uint8)
    assert np.array_equal(O.e4m3_from_float(O.e4m3_to_double(allc).astype(np.float32)), allc)
    # saturation: beyond the largest finite value, never NaN or infinity
    big = np.array([448.0, 449.0, 464.0, 1e6, np.inf, -500.0, -np.inf], dtype=np.float32)
    assert list(O.e4m3_from_float(big)) == [0x7e, 0x7e, 0x7e, 0x7e, 0x7e, 0xfe, 0xfe]
    assert int(O.e4m3_from_float(np.array([np.nan], dtype=np.float32))[0]) == 0x7f


def _rows(seed, T=37, Hkv=2, D=64, scale=1.0):
    g = torch.Generator().manual_seed(seed)
    k = (torch.randn(T, Hkv, D, generator=g) * scale).to(torch.bfloat16)
    v = (torch.randn(T, Hkv, D, generator=g) * scale * 3).to(torch.bfloat16)
    return k, v


def test_cache_write_fp8_scale_closed_form_and_error_bound():
    T, Hkv, D, P = 37, 2, 64, 16
    k, v = _rows(1, T, Hkv, D)
    k[5] = 0                                              # an all-zero row: scale 1, codes 0
    pools = O.Fp8Pools(4, Hkv, P, D)
    slots = np.arange(T, dtype=np.int64) + 3              # contiguous slots from offset 3 of page 0
    slots[9] = -1                                         # skipped token
    O.cache_write_fp8(k, v, slots, pools)
    for t in range(T):
        for hk in range(Hkv):
            if slots[t] < 0:
                continue
            page, off = divmod(int(slots[t]), P)
            for x, codes, sc in ((k, pools.k_codes, pools.k_scale), (v, pools.v_codes, pools.v_scale)):
                row = x[t, hk].float().numpy()
                amax = np.abs(row).max()
                s = sc[page, hk, off]
                if amax == 0:
                    assert s == 1.0 and not codes[page, hk, off].any()
                    continue
                assert s == np.float32(amax) / np.float32(448.0)            # fp32 quotient
                deq = O.e4m3_to_double(codes[page, hk, off]) * float(s)
                # the row's largest element sits on +-448 and comes back within an fp32 rounding of the scale
                top = int(np.abs(row).argmax())
                assert codes[page, hk, off][top] & 0x7f == 0x7e
                assert abs(deq[top] - row[top]) <= abs(row[top]) * 2.0 ** -23
                # E4M3 has 3 mantissa bits: relative error <= 2^-4 for normal codes, absolute <= scale * 2^-10 below
                err = np.abs(deq - row.astype(np.float64))
                bound = np.maximum(np.abs(row) * 2.0 ** -4, float(s) * 2.0 ** -10) * (1 + 1e-6)
                assert np.all(err <= bound)
    # untouched slots (before offset 3, the skipped token, everything after) keep the poison
    assert np.isnan(pools.k_scale[0, 0, 0]) and pools.k_codes[0, 0, 0, 0] == 0x7f
    page, off = divmod(3 + 9, P)
    assert np.isnan(pools.v_scale[page, 1, off])


def test_cache_write_fp8_codes_match_torch_on_the_same_quotients():
    """An independent restatement: x / scale in fp32 (numpy), codes by torch's float8 conversion."""
    T, Hkv, D, P = 48, 2, 128, 16
    k, v = _rows(2, T, Hkv, D, scale=0.3)
    pools = O.Fp8Pools(3, Hkv, P, D)
    O.cache_write_fp8(k, v, np.arange(T, dtype=np.int64), pools)
    for x, codes in ((k, pools.k_codes), (v, pools.v_codes)):
        xf = x.float().numpy()
        s = np.abs(xf).max(axis=-1, keepdims=True).astype(np.float32) / np.float32(448.0)
        y = (xf / s).astype(np.float32)
        ref = torch.from_numpy(np.clip(y, -448, 448)).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
        got = codes.transpose(0, 2, 1, 3).reshape(T, Hkv, D)
        assert np.array_equal(got, ref)


def _small_batch():
    return W.config1()


def test_fp8_attention_equals_pinned_fp64_path_on_dequantised_pools():
    """Dequantise OUTSIDE the oracle (torch float8 -> double, times the scale) and run the pinned fp64 function."""
    b = _small_batch()
    sh = b.shape
    pools = O.quantize_pool_fp8(b.k_pool, b.v_pool)
    for step in b.steps:
        got = O.run_step_fp8(b, step, pools)
        kd = torch.from_numpy(pools.k_codes.copy()).view(torch.float8_e4m3fn).double().numpy() * \
            pools.k_scale[..., None].astype(np.float64)
        vd = torch.from_numpy(pools.v_codes.copy()).view(torch.float8_e4m3fn).double().numpy() * \
            pools.v_scale[..., None].astype(np.float64)
        # poisoned slots dequantise to NaN on both sides; the definition never reads them
        ref = O.attend_paged(step.q, kd, vd, b.block_table.numpy(), b.page_logical_pos.numpy(),
                             step.seq_lens.numpy(), step.cu_q_lens.numpy(), num_q_heads=sh.num_q_heads,
                             num_kv_heads=sh.num_kv_heads, head_dim=sh.head_dim, page_size=sh.page_size,
                             theta=sh.rope_theta)
        assert np.isfinite(got).all()
        assert np.abs(got - ref).max() <= 1e-12


def test_fp8_path_equals_bf16_path_on_exactly_representable_inputs():
    """Rows drawn from the E4M3 grid times a power of two, with the row maximum on 448 * 2^e: quantisation is exact,
    so FP8 pages and bf16 pages must give the same attention output."""
    b = _small_batch()
    sh = b.shape
    rng = np.random.default_rng(11)
    grid = O.e4m3_to_double(np.array([c for c in range(256) if c not in (0x7f, 0xff)], dtype=np.uint8))

    def snap(shape):
        x = rng.choice(grid, size=shape)
        x[..., 0] = 448.0                                  # row maximum: scale = 2^e exactly
        e = rng.integers(-9, -5, size=shape[:-1] + (1,))
        return torch.from_numpy(x * np.exp2(e)).to(torch.bfloat16)   # <= 4 significant bits: exact in bf16

    k_pool = snap(tuple(b.k_pool.shape))
    v_pool = snap(tuple(b.v_pool.shape))
    steps = []
    for st in b.steps:
        st2 = W.dataclasses.replace(st)
        if st.k_new is not None:
            st2.k_new, st2.v_new = snap(tuple(st.k_new.shape)), snap(tuple(st.v_new.shape))
        steps.append(st2)
    pools = O.quantize_pool_fp8(k_pool, v_pool)
    kp, vp = k_pool.clone(), v_pool.clone()
    for st in steps:
        got = O.run_step_fp8(b, st, pools)
        ref = O.run_step(b, st, kp, vp)
        assert np.abs(got - ref).max() <= 1e-12
    # and the stored scales are the powers of two
    s = pools.k_scale[np.isfinite(pools.k_scale)]
    assert np.array_equal(np.exp2(np.round(np.log2(s))), s)


def test_fp8_attention_error_vs_bf16_attention_is_quantisation_sized():
    """Sanity of the whole chain: on N(0,1) data the FP8-page output differs from the bf16-page output by the size
    E4M3 rounding predicts (a few per cent of the output RMS), not by O(1)."""
    b = _small_batch()
    pools = O.quantize_pool_fp8(b.k_pool, b.v_pool)
    kp, vp = b.k_pool.clone(), b.v_pool.clone()
    for st in b.steps:
        got = O.run_step_fp8(b, st, pools)
        ref = O.run_step(b, st, kp, vp)
        rel = np.sqrt(np.mean((got - ref) ** 2)) / np.sqrt(np.mean(ref ** 2))
        assert 1e-3 < rel < 0.1, rel


def test_attend_paged_variant_rejects_fp8_without_scales():
    b = _small_batch()
    pools = O.quantize_pool_fp8(b.k_pool, b.v_pool)
    import ctypes
    f = O.lib().lazy_oracle_attend_paged_variant
    f.restype = ctypes.c_int
    # dtype_kv = 2 (E4M3) through the scale-less entry point is refused before anything is read
    rc = f(None, 1, O._p(pools.k_codes), O._p(pools.v_codes), 2, None, None, ctypes.c_int64(1), None, None, 0,
           4, 1, 64, 16, ctypes.c_double(THETA), 0, None, 0, None, ctypes.c_double(0.0), None, None, None)
    assert rc == -1

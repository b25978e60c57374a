"""Pins for the fp64 CPU oracle (oracle/lazy_oracle.c) against what the paper and the mathematics fix.

Each test names the passage it pins.  None of the expected values comes from the oracle itself or from the
CUDA path: they are brute force written independently here, closed forms, invariants, a library routine
(torch SDPA in float64) on a special case, or the golden worked example under tests/golden/.
"""
import math
import os

import numpy as np
import pytest
import torch

from oracle import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "worked_examples.txt")


def _rng(seed):
    return np.random.default_rng(seed)


def brute_force(q, k, v, pos_q, pos_k, vis, theta):
    """Independent statement: score(m,n) = q^T R_{n-m} k with explicit 2x2 blocks (Fact 3.2, PAPER.md
    L154-158), softmax WITHOUT max subtraction (safe at tiny sizes), GQA by integer division."""
    n_q, Hq, D = q.shape
    L, Hkv, _ = k.shape
    h = D // 2
    out = np.zeros((n_q, Hq, D))
    P = np.zeros((n_q, Hq, L))
    for i in range(n_q):
        for hq in range(Hq):
            hk = hq // (Hq // Hkv)
            w = np.zeros(L)
            for s in range(L):
                if s > vis[i]:
                    continue
                rel = pos_k[s] - pos_q[i]
                acc = 0.0
                for j in range(h):
                    a = rel * theta ** (-2.0 * j / D)
                    R = np.array([[math.cos(a), -math.sin(a)], [math.sin(a), math.cos(a)]])
                    qq = np.array([q[i, hq, j], q[i, hq, j + h]])
                    kk = np.array([k[s, hk, j], k[s, hk, j + h]])
                    acc += qq @ (R @ kk)
                w[s] = math.exp(acc / math.sqrt(D))
            w /= w.sum()
            P[i, hq] = w
            for s in range(L):
                out[i, hq] += w[s] * v[s, hk]
    return out, P


def random_case(seed, n_q=3, L=11, Hq=4, Hkv=2, D=8):
    r = _rng(seed)
    q = r.standard_normal((n_q, Hq, D))
    k = r.standard_normal((L, Hkv, D))
    v = r.standard_normal((L, Hkv, D))
    pos_k = np.sort(r.integers(0, 500, size=L)).astype(np.float64)
    vis = np.arange(L - n_q, L)
    pos_q = pos_k[vis]
    return q, k, v, pos_q, pos_k, vis


# ---- whole oracle vs brute force -----------------------------------------------------------------------------
@pytest.mark.parametrize("seed,Hq,Hkv,D,theta", [(0, 4, 2, 8, 1e4), (1, 6, 1, 4, 5e5), (2, 2, 2, 16, 1e6)])
def test_core_matches_brute_force(seed, Hq, Hkv, D, theta):
    q, k, v, pos_q, pos_k, vis = random_case(seed, Hq=Hq, Hkv=Hkv, D=D)
    out, P = oracle.attend_core(q, k, v, pos_q, pos_k, vis, theta, want_probs=True)
    ref, Pref = brute_force(q, k, v, pos_q, pos_k, vis, theta)
    assert np.abs(out - ref).max() < 1e-12
    assert np.abs(P - Pref).max() < 1e-12


def test_paged_matches_brute_force_with_gather():
    """Paged wrapper: slot/offset/page indexing, per-page logical starts with a gap, query = last tokens."""
    r = _rng(7)
    Hq, Hkv, D, P, theta = 4, 2, 8, 4, 1e4
    num_pages = 9
    kp = r.standard_normal((num_pages, Hkv, P, D))
    vp = r.standard_normal((num_pages, Hkv, P, D))
    bt = np.array([[5, 2, 7, 2, 0], [1, 8, 3, 0, 0]], dtype=np.int32)        # page 2 used twice in request 0
    pp = np.array([[0, 4, 40, 44, 48], [100, 104, 108, 0, 0]], dtype=np.int32)  # gap between slots 1 and 2
    seq_lens = np.array([18, 10], dtype=np.int32)
    cu = np.array([0, 3, 5], dtype=np.int32)
    q = r.standard_normal((5, Hq, D))
    out = oracle.attend_paged(q, kp, vp, bt, pp, seq_lens, cu, num_q_heads=Hq, num_kv_heads=Hkv, head_dim=D,
                              page_size=P, theta=theta)
    for rr in range(2):
        L, nq = int(seq_lens[rr]), int(cu[rr + 1] - cu[rr])
        k = np.stack([kp[bt[rr, s // P], :, s % P] for s in range(L)])
        v = np.stack([vp[bt[rr, s // P], :, s % P] for s in range(L)])
        pos = np.array([pp[rr, s // P] + s % P for s in range(L)], dtype=np.float64)
        vis = np.arange(L - nq, L)
        ref, _ = brute_force(q[cu[rr]:cu[rr + 1]], k, v, pos[vis], pos, vis, theta)
        assert np.abs(out[cu[rr]:cu[rr + 1]] - ref).max() < 1e-12


# ---- RoPE: closed forms, norm, pairing, frequency ------------------------------------------------------------
def test_rope_closed_form_one_hot():
    """q = k = e_j  =>  raw score(m, n) = cos((n-m) theta^(-2j/D)) (Fact 3.2; SURVEY 8.c pins)."""
    D, theta = 8, 1e4
    for j in range(D // 2):
        e = np.zeros(D)
        e[j] = 1.0
        for m, n in [(0, 0), (3, 10), (1000, 17), (131071, 5)]:
            s = float(oracle.rope(e, m, theta) @ oracle.rope(e, n, theta))
            assert abs(s - math.cos((n - m) * theta ** (-2.0 * j / D))) < 1e-9


def test_rope_formula_signs_and_halves():
    """k1' = k1 cos - k2 sin, k2' = k1 sin + k2 cos on the two half dimensions."""
    D, theta, pos = 6, 1e4, 3.0
    x = np.array([1.0, 2.0, 3.0, 4.0, 5.0, 6.0])
    y = oracle.rope(x, pos, theta)
    for j in range(3):
        a = pos * theta ** (-2.0 * j / D)
        assert abs(y[j] - (x[j] * math.cos(a) - x[j + 3] * math.sin(a))) < 1e-14
        assert abs(y[j + 3] - (x[j] * math.sin(a) + x[j + 3] * math.cos(a))) < 1e-14
    # position 0 is the identity
    assert np.array_equal(oracle.rope(x, 0.0, theta), x)


def test_rope_preserves_norm():
    r = _rng(3)
    for pos in [0, 1, 77, 32896, 131071]:
        x = r.standard_normal(128)
        assert abs(np.linalg.norm(oracle.rope(x, pos, 5e5)) - np.linalg.norm(x)) < 1e-12


def test_golden_worked_examples():
    """tests/golden/worked_examples.txt (closed form cos(-2), cos(-1), cos(0) -> softmax); example B pins the
    half-split pairing AND the frequency formula (an interleaved pairing gives the 'wrong_b' row)."""
    vals = {}
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        key, *nums = line.split()
        vals[key] = np.array([float(x) for x in nums])
    sc = np.array([math.cos(-2.0), math.cos(-1.0), math.cos(0.0)])
    assert np.abs(vals["scores"] - sc).max() < 1e-11        # fixture == closed form
    sm = np.exp(sc) / np.exp(sc).sum()
    assert np.abs(vals["output"][:3] - sm).max() < 1e-11
    theta, D = 1e4, 4
    # Example A through the paged interface, several page starts (shift invariance in passing)
    for p0 in (0, 1000, 131000):
        kp = np.zeros((1, 1, 16, D)); kp[0, 0, :, 0] = 1.0
        vp = np.zeros((1, 1, 16, D)); vp[0, 0, 0, 0] = 1; vp[0, 0, 1, 1] = 1; vp[0, 0, 2, 2] = 1
        q = np.array([[[2.0, 0, 0, 0]]])
        out = oracle.attend_paged(q, kp, vp, np.array([[0]], np.int32), np.array([[p0]], np.int32),
                                  np.array([3], np.int32), np.array([0, 1], np.int32),
                                  num_q_heads=1, num_kv_heads=1, head_dim=D, page_size=16, theta=theta)
        assert np.abs(out[0, 0] - vals["output"]).max() < (2e-9 if p0 else 1e-11)
    # Example B through the core with explicit positions
    k = np.zeros((3, 1, D)); k[:, 0, 1] = 1.0
    v = np.zeros((3, 1, D)); v[0, 0, 0] = 1; v[1, 0, 1] = 1; v[2, 0, 2] = 1
    q = np.array([[[0.0, 2.0, 0, 0]]])
    out, P = oracle.attend_core(q, k, v, [200.0], [0.0, 100.0, 200.0], [2], theta, want_probs=True)
    assert np.abs(out[0, 0] - vals["output"]).max() < 1e-11
    assert np.abs(P[0, 0] - vals["wrong_b"]).max() > 0.05    # the interleaved reading is clearly excluded


# ---- invariances ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shift", [1, 1000, 99991])
def test_relative_position_invariance(shift):
    """Fact 3.2: shifting all q and k positions by a constant leaves scores unchanged
    (north_star: to 1e-10)."""
    q, k, v, pos_q, pos_k, vis = random_case(11, n_q=4, L=20, Hq=4, Hkv=2, D=16)
    o0, p0 = oracle.attend_core(q, k, v, pos_q, pos_k, vis, 5e5, want_probs=True)
    o1, p1 = oracle.attend_core(q, k, v, pos_q + shift, pos_k + shift, vis, 5e5, want_probs=True)
    assert np.abs(o0 - o1).max() < 1e-10
    assert np.abs(p0 - p1).max() < 1e-10


def test_paged_shift_invariance():
    r = _rng(5)
    Hq, Hkv, D, P = 2, 1, 8, 16
    kp = r.standard_normal((4, Hkv, P, D)); vp = r.standard_normal((4, Hkv, P, D))
    bt = np.array([[3, 1, 0]], np.int32)
    sl = np.array([40], np.int32); cu = np.array([0, 5], np.int32)
    q = r.standard_normal((5, Hq, D))
    outs = []
    for c in (0, 1, 1000, 99991):
        pp = np.array([[0, 16, 32]], np.int32) + c
        outs.append(oracle.attend_paged(q, kp, vp, bt, pp, sl, cu, num_q_heads=Hq, num_kv_heads=Hkv, head_dim=D,
                                        page_size=P, theta=1e4))
    for o in outs[1:]:
        assert np.abs(o - outs[0]).max() < 1e-10


def test_softmax_rows_sum_to_one_and_mask():
    q, k, v, pos_q, pos_k, vis = random_case(13, n_q=5, L=33, Hq=6, Hkv=3, D=8)
    _, P = oracle.attend_core(q, k, v, pos_q, pos_k, vis, 1e4, want_probs=True)
    assert np.abs(P.sum(-1) - 1.0).max() < 1e-12
    for i in range(5):
        assert np.all(P[i, :, vis[i] + 1:] == 0.0)         # nothing beyond the causal index
        assert np.all(P[i, :, :vis[i] + 1] > 0.0)


def test_uniform_values_give_that_value():
    q, k, v, pos_q, pos_k, vis = random_case(17, D=8)
    v[:] = np.linspace(-1, 1, 8)
    out = oracle.attend_core(q, k, v, pos_q, pos_k, vis, 1e4)
    assert np.abs(out - np.linspace(-1, 1, 8)).max() < 1e-12


def test_dominant_key():
    """One key whose score is ~+50 above the rest takes all the weight."""
    r = _rng(19)
    D, L = 8, 12
    q = np.zeros((1, 1, D)); q[0, 0, 0] = 1.0
    k = 0.01 * r.standard_normal((L, 1, D))
    v = r.standard_normal((L, 1, D))
    pos = np.zeros(L)                                   # all positions equal -> no rotation effect
    k[4, 0, 0] = 60.0 * math.sqrt(D)
    out = oracle.attend_core(q, k, v, [0.0], pos, [L - 1], 1e4)
    assert np.abs(out[0, 0] - v[4, 0]).max() < 1e-12


# ---- reduction to a library routine --------------------------------------------------------------------------
def test_zero_positions_reduce_to_sdpa():
    """All positions 0 => RoPE is the identity => softmax(QK^T/sqrt(D))V == torch SDPA in float64."""
    r = _rng(23)
    n_q, L, Hq, Hkv, D = 6, 19, 4, 2, 16
    q = r.standard_normal((n_q, Hq, D)); k = r.standard_normal((L, Hkv, D)); v = r.standard_normal((L, Hkv, D))
    vis = np.full(n_q, L - 1)
    out = oracle.attend_core(q, k, v, np.zeros(n_q), np.zeros(L), vis, 1e4)
    tq = torch.from_numpy(q).permute(1, 0, 2)[None]
    tk = torch.from_numpy(k).permute(1, 0, 2).repeat_interleave(Hq // Hkv, 0)[None]
    tv = torch.from_numpy(v).permute(1, 0, 2).repeat_interleave(Hq // Hkv, 0)[None]
    ref = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv)[0].permute(1, 0, 2).numpy()
    assert np.abs(out - ref).max() < 1e-12


def test_materialised_copy_then_sdpa_with_mask():
    """After step 1 (materialise), step 2 is textbook attention over (qhat, Khat, V) with a boolean index mask and
    GQA head repeat: feed the oracle's own hats to float64 SDPA (pins softmax, mask, head mapping)."""
    q, k, v, pos_q, pos_k, vis = random_case(29, n_q=5, L=23, Hq=6, Hkv=2, D=8)
    out, khat, qhat = oracle.attend_core(q, k, v, pos_q, pos_k, vis, 5e5, want_hats=True)
    Hq, Hkv = 6, 2
    tq = torch.from_numpy(qhat).permute(1, 0, 2)[None]
    tk = torch.from_numpy(khat).permute(1, 0, 2).repeat_interleave(Hq // Hkv, 0)[None]
    tv = torch.from_numpy(v).permute(1, 0, 2).repeat_interleave(Hq // Hkv, 0)[None]
    mask = torch.from_numpy(np.arange(23)[None, :] <= vis[:, None])
    ref = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv, attn_mask=mask)[0].permute(1, 0, 2).numpy()
    assert np.abs(out - ref).max() < 1e-12
    # and the hats are the rope of the inputs at their positions
    assert np.abs(khat[7, 1] - oracle.rope(k[7, 1], pos_k[7], 5e5)).max() == 0.0
    assert np.abs(qhat[2, 3] - oracle.rope(q[2, 3], pos_q[2], 5e5)).max() == 0.0


# ---- sharing semantics ---------------------------------------------------------------------------------------
def test_one_page_at_two_positions_equals_two_copies():
    """one physical page used at two logical positions == two materialised copies (bitwise in
    the oracle), within one request and across two requests."""
    r = _rng(31)
    Hq, Hkv, D, P = 4, 2, 8, 16
    kp = r.standard_normal((4, Hkv, P, D)); vp = r.standard_normal((4, Hkv, P, D))
    kp[3] = kp[1]; vp[3] = vp[1]                          # page 3 is a byte-identical duplicate of page 1
    q = r.standard_normal((2, Hq, D))
    sl = np.array([48, 48], np.int32); cu = np.array([0, 1, 2], np.int32)
    pp = np.array([[0, 16, 32], [64, 16, 0]], np.int32)
    shared = np.array([[1, 0, 1], [1, 2, 1]], np.int32)   # page 1 twice per request, different offsets
    copies = np.array([[1, 0, 3], [3, 2, 1]], np.int32)
    kw = dict(num_q_heads=Hq, num_kv_heads=Hkv, head_dim=D, page_size=P, theta=1e4)
    a = oracle.attend_paged(q, kp, vp, shared, pp, sl, cu, **kw)
    b = oracle.attend_paged(q, kp, vp, copies, pp, sl, cu, **kw)
    assert np.array_equal(a, b)


def test_example_3_1_two_documents():
    """Example 3.1: d2's cache, indexed from 0, reused after d1 by an offset |d1| == attention over
    the concatenation d1 d2 with conventional positions."""
    r = _rng(37)
    Hq, Hkv, D, P = 2, 1, 8, 16
    d1, d2 = 2, 1                                          # pages
    kp = r.standard_normal((4, Hkv, P, D)); vp = r.standard_normal((4, Hkv, P, D))
    q = r.standard_normal((1, Hq, D))
    # request: d1 = pages (0,1) at 0, d2 = page (2) at |d1| = 32, question token on page 3 at 48
    out = oracle.attend_paged(q, kp, vp, np.array([[0, 1, 2, 3]], np.int32), np.array([[0, 16, 32, 48]], np.int32),
                              np.array([49], np.int32), np.array([0, 1], np.int32),
                              num_q_heads=Hq, num_kv_heads=Hkv, head_dim=D, page_size=P, theta=1e4)
    k = np.concatenate([kp[p].transpose(1, 0, 2) for p in (0, 1, 2, 3)])[:49]
    v = np.concatenate([vp[p].transpose(1, 0, 2) for p in (0, 1, 2, 3)])[:49]
    ref, _ = brute_force(q, k, v, np.array([48.0]), np.arange(49, dtype=np.float64), np.array([48]), 1e4)
    assert np.abs(out - ref).max() < 1e-12


# ---- mask properties -----------------------------------------------------------------------------------------
def test_causality_and_poisoned_tail():
    """Perturbing K/V at indices > sq leaves that query bit-identical; NaN bytes beyond seq_len never propagate."""
    r = _rng(41)
    Hq, Hkv, D, P = 2, 1, 8, 16
    kp = r.standard_normal((3, Hkv, P, D)); vp = r.standard_normal((3, Hkv, P, D))
    bt = np.array([[0, 1, 2]], np.int32); pp = np.array([[0, 16, 32]], np.int32)
    sl = np.array([37], np.int32); cu = np.array([0, 4], np.int32)
    q = r.standard_normal((4, Hq, D))
    kw = dict(num_q_heads=Hq, num_kv_heads=Hkv, head_dim=D, page_size=P, theta=1e4)
    a = oracle.attend_paged(q, kp, vp, bt, pp, sl, cu, **kw)
    kp2, vp2 = kp.copy(), vp.copy()
    kp2[2, :, 5:] = np.nan; vp2[2, :, 5:] = np.nan          # beyond seq_len (37 = 32 + 5)
    b = oracle.attend_paged(q, kp2, vp2, bt, pp, sl, cu, **kw)
    assert np.array_equal(a, b) and np.isfinite(b).all()
    kp3 = kp.copy(); kp3[2, :, 4] += 10.0                  # token 36: only the last query (sq=36) may see it
    c = oracle.attend_paged(q, kp3, vp, bt, pp, sl, cu, **kw)
    assert np.array_equal(a[:3], c[:3]) and not np.array_equal(a[3], c[3])


def test_slot_permutation_with_positions():
    """Permuting fully visible page slots together with their logical positions leaves the question's output
    unchanged (attention is a set operation once positions are attached)."""
    r = _rng(43)
    Hq, Hkv, D, P = 4, 2, 8, 16
    kp = r.standard_normal((5, Hkv, P, D)); vp = r.standard_normal((5, Hkv, P, D))
    q = r.standard_normal((1, Hq, D))
    sl = np.array([65], np.int32); cu = np.array([0, 1], np.int32)
    kw = dict(num_q_heads=Hq, num_kv_heads=Hkv, head_dim=D, page_size=P, theta=5e5)
    a = oracle.attend_paged(q, kp, vp, np.array([[0, 1, 2, 3, 4]], np.int32), np.array([[0, 16, 32, 48, 64]], np.int32),
                            sl, cu, **kw)
    b = oracle.attend_paged(q, kp, vp, np.array([[2, 0, 3, 1, 4]], np.int32), np.array([[32, 0, 48, 16, 64]], np.int32),
                            sl, cu, **kw)
    assert np.abs(a - b).max() < 1e-12


def test_row_select_and_empty_request():
    r = _rng(47)
    Hq, Hkv, D, P = 2, 1, 4, 16
    kp = r.standard_normal((2, Hkv, P, D)); vp = r.standard_normal((2, Hkv, P, D))
    q = r.standard_normal((4, Hq, D))
    bt = np.array([[0, 1], [1, 0]], np.int32); pp = np.array([[0, 16], [0, 16]], np.int32)
    sl = np.array([20, 0], np.int32); cu = np.array([0, 3, 4], np.int32)
    kw = dict(num_q_heads=Hq, num_kv_heads=Hkv, head_dim=D, page_size=P, theta=1e4)
    full = oracle.attend_paged(q, kp, vp, bt, pp, sl, cu, **kw)
    assert np.all(full[3] == 0.0)                          # seq_len 0 -> zeros
    sel = oracle.attend_paged(q, kp, vp, bt, pp, sl, cu, row_select=[0, 1, 0, 0], **kw)
    assert np.array_equal(sel[1], full[1]) and np.all(sel[0] == 0) and np.all(sel[2] == 0)


# ---- bf16 input path and cache write -------------------------------------------------------------------------
def test_bf16_inputs_are_converted_exactly():
    g = torch.Generator().manual_seed(3)
    Hq, Hkv, D, P = 4, 1, 64, 16
    kp = torch.randn(3, Hkv, P, D, generator=g).to(torch.bfloat16)
    vp = torch.randn(3, Hkv, P, D, generator=g).to(torch.bfloat16)
    q = torch.randn(2, Hq, D, generator=g).to(torch.bfloat16)
    bt = np.array([[2, 0, 1]], np.int32); pp = np.array([[0, 16, 32]], np.int32)
    sl = np.array([40], np.int32); cu = np.array([0, 2], np.int32)
    kw = dict(num_q_heads=Hq, num_kv_heads=Hkv, head_dim=D, page_size=P, theta=1e4)
    a = oracle.attend_paged(q, kp, vp, bt, pp, sl, cu, **kw)
    b = oracle.attend_paged(q.double().numpy(), kp.double().numpy(), vp.double().numpy(), bt, pp, sl, cu, **kw)
    assert np.array_equal(a, b)


def test_cache_write_is_a_bit_copy():
    g = torch.Generator().manual_seed(5)
    Hkv, D, P, n_pages = 2, 64, 16, 5
    kp = torch.randn(n_pages, Hkv, P, D, generator=g).to(torch.bfloat16)
    vp = torch.randn(n_pages, Hkv, P, D, generator=g).to(torch.bfloat16)
    k0, v0 = kp.clone(), vp.clone()
    kn = torch.randn(4, Hkv, D, generator=g).to(torch.bfloat16)
    vn = torch.randn(4, Hkv, D, generator=g).to(torch.bfloat16)
    kn.view(torch.int16)[0, 0, 0] = 0x7FC1               # a NaN payload must survive bit-exactly
    slots = np.array([3 * P + 5, -1, 0 * P + 15, 4 * P + 0], dtype=np.int64)
    oracle.cache_write(kn, vn, slots, kp, vp, P)
    exp_k, exp_v = k0.clone(), v0.clone()
    for t, (pg, off) in {0: (3, 5), 2: (0, 15), 3: (4, 0)}.items():
        exp_k[pg, :, off] = kn[t]; exp_v[pg, :, off] = vn[t]
    assert torch.equal(kp.view(torch.int16), exp_k.view(torch.int16))
    assert torch.equal(vp.view(torch.int16), exp_v.view(torch.int16))


def test_long_position_numerics_stateless():
    """PAPER.md L455 / Table 7: rotation from absolute indices stays accurate at 128K positions: the oracle at
    positions ~131071 agrees with the relative-angle brute force (which never forms a large angle)."""
    r = _rng(53)
    n_q, L, Hq, Hkv, D = 1, 6, 2, 1, 8
    q = r.standard_normal((n_q, Hq, D)); k = r.standard_normal((L, Hkv, D)); v = r.standard_normal((L, Hkv, D))
    pos_k = np.array([131071 - 5, 131071 - 4, 131071 - 3, 131071 - 2, 131071 - 1, 131071], dtype=np.float64)
    out = oracle.attend_core(q, k, v, [131071.0], pos_k, [L - 1], 5e5)
    ref, _ = brute_force(q, k, v, np.array([131071.0]), pos_k, np.array([L - 1]), 5e5)
    assert np.abs(out - ref).max() < 1e-9


# ---- stored-position layouts and the materialising re-encoding -----------------------
def _np_rope_pool(kp, start_of_page, theta, per_token=True):
    """Independent numpy statement of PAPER.md L164-166 on a whole pool [pages,Hkv,P,D]: token t of page g is
    rotated by start_of_page[g] (+ t), pair (j, j + D/2), angle * theta^(-2j/D)."""
    g, Hkv, P, D = kp.shape
    h = D // 2
    inv = theta ** (-2.0 * np.arange(h) / D)
    pos = np.asarray(start_of_page, dtype=np.float64)[:, None] + (np.arange(P)[None, :] if per_token else 0.0)
    ang = pos[:, None, :, None] * inv[None, None, None, :]                     # [g,1,P,h]
    c, s = np.cos(ang), np.sin(ang)
    x1, x2 = kp[..., :h], kp[..., h:]
    return np.concatenate([x1 * c - x2 * s, x1 * s + x2 * c], axis=-1)


def test_materialize_closed_form_group_property_and_norm():
    """f2: re-encoding a page is a rotation: closed form on one-hot rows (cos / sin of (p+t)*theta_j), R_a R_b =
    R_{a+b} (a cached page moves by one relative rotation), R_{-a} undoes R_a, norms kept."""
    P, D, Hkv, theta = 4, 8, 2, 1e4
    h = D // 2
    kp = np.zeros((3, Hkv, P, D))
    kp[1, :, :, 2] = 1.0                                    # e_2 in every row of page 1
    out = oracle.materialize_pages(kp, [1], [37], True, theta)
    for t in range(P):
        a = (37 + t) * theta ** (-2.0 * 2 / D)
        expect = np.zeros(D); expect[2] = math.cos(a); expect[2 + h] = math.sin(a)
        assert np.abs(out[0, :, t] - expect).max() < 1e-14
    r = _rng(61)
    kp = r.standard_normal((5, Hkv, P, D))
    a = oracle.materialize_pages(kp, [3, 0, 3], [100, 7, 0], True, theta)      # page 3 twice, two positions
    assert np.abs(a - _np_rope_pool(kp[[3, 0, 3]], [100, 7, 0], theta)).max() < 1e-12
    b = oracle.materialize_pages(a, [0, 1, 2], [23, -7, 500], False, theta)    # one relative rotation per page
    c = oracle.materialize_pages(kp, [3, 0, 3], [123, 0, 500], True, theta)
    assert np.abs(b - c).max() < 1e-11
    back = oracle.materialize_pages(b, [0, 1, 2], [-23, 7, -500], False, theta)
    assert np.abs(back - a).max() < 1e-11
    assert np.abs(np.linalg.norm(a, axis=-1) - np.linalg.norm(kp[[3, 0, 3]], axis=-1)).max() < 1e-12


def test_stored_position_layouts_equal_unrotated_cache():
    """f1 (PAPER.md L37 'mathematically identical'; L173 document-local cache + one offset per document; L409):
    attention over (i) un-rotated pages, (ii) pages stored rotated at a page-local position and moved by one
    relative rotation, (iii) private copies already rotated at their final positions -- all the same numbers.
    The pre-rotated pools are built by the independent numpy statement above, not by the oracle."""
    r = _rng(67)
    Hq, Hkv, D, P, theta = 4, 2, 8, 4, 5e5
    num_pages = 7
    kp = r.standard_normal((num_pages, Hkv, P, D)); vp = r.standard_normal((num_pages, Hkv, P, D))
    bt = np.array([[5, 2, 6, 2, 0], [1, 2, 3, 0, 0]], np.int32)                # page 2 shared, twice in request 0
    pp = np.array([[0, 4, 40, 44, 48], [100, 104, 108, 0, 0]], np.int32)
    sl = np.array([18, 10], np.int32); cu = np.array([0, 3, 5], np.int32)
    q = r.standard_normal((5, Hq, D))
    kw = dict(num_q_heads=Hq, num_kv_heads=Hkv, head_dim=D, page_size=P, theta=theta)
    base = oracle.attend_paged(q, kp, vp, bt, pp, sl, cu, **kw)
    # (ii) document-local storage: stored start of every physical page, incl. one larger than its logical start
    stored = np.array([0, 4, 8, 12, 0, 60, 16], np.int32)
    kp_local = _np_rope_pool(kp, stored, theta)
    got = oracle.attend_paged(q, kp_local, vp, bt, pp, sl, cu, k_storage=1, page_stored_pos=stored, **kw)
    assert np.abs(got - base).max() < 1e-10
    # a wrong sign of the relative rotation must be visible
    bad = oracle.attend_paged(q, kp_local, vp, bt, pp, sl, cu, k_storage=1, page_stored_pos=-stored, **kw)
    assert np.abs(bad - base).max() > 1e-3
    # (iii) private absolute copies: every (request, slot) gets its own physical page
    n_slots = bt.shape[1]
    src = bt.reshape(-1); starts = pp.reshape(-1)
    kp_abs = _np_rope_pool(kp[src], starts, theta); vp_abs = vp[src]
    bt_abs = np.arange(2 * n_slots, dtype=np.int32).reshape(2, n_slots)
    got = oracle.attend_paged(q, kp_abs, vp_abs, bt_abs, pp, sl, cu, k_storage=2, **kw)
    assert np.abs(got - base).max() < 1e-10
    # and the oracle's own materialiser builds exactly those copies
    assert np.abs(oracle.materialize_pages(kp, src, starts, True, theta) - kp_abs).max() < 1e-12


# ---- positional variants (section 3.5) ----------------------------------
def brute_force_variant(q, k, v, pos_q, pos_k, vis, theta, pairing="half", inv_freq=None, scale=None, slopes=None):
    """Independent statement for the variants: explicit 2x2 rotation of the pair (i1, i2) by (n - m) * f_j, an
    arbitrary frequency vector, an arbitrary softmax scale, or (ALiBi) no rotation and the bias slope * (n - m)."""
    n_q, Hq, D = q.shape
    L, Hkv, _ = k.shape
    h = D // 2
    f = np.asarray(inv_freq) if inv_freq is not None else theta ** (-2.0 * np.arange(h) / D)
    sc = scale if scale else 1.0 / math.sqrt(D)
    out = np.zeros((n_q, Hq, D))
    for i in range(n_q):
        for hq in range(Hq):
            hk = hq // (Hq // Hkv)
            w = np.zeros(L)
            for s in range(L):
                if s > vis[i]:
                    continue
                rel = pos_k[s] - pos_q[i]
                if slopes is not None:
                    acc = float(q[i, hq] @ k[s, hk]) * sc + slopes[hq] * rel
                else:
                    acc = 0.0
                    for j in range(h):
                        i1, i2 = (2 * j, 2 * j + 1) if pairing == "interleaved" else (j, j + h)
                        a = rel * f[j]
                        acc += q[i, hq, i1] * (math.cos(a) * k[s, hk, i1] - math.sin(a) * k[s, hk, i2])
                        acc += q[i, hq, i2] * (math.sin(a) * k[s, hk, i1] + math.cos(a) * k[s, hk, i2])
                    acc *= sc
                w[s] = math.exp(acc)
            w /= w.sum()
            for s in range(L):
                out[i, hq] += w[s] * v[s, hk]
    return out


def test_interleaved_pairing_brute_force_and_permutation():
    """L215: interleaved pairing (2j, 2j+1).  Brute force; and the fact the CUDA path relies on: interleaved RoPE is
    half-split RoPE on de-interleaved vectors (dims 0,2,4,... then 1,3,5,...), applied to q and k alike."""
    q, k, v, pos_q, pos_k, vis = random_case(71, n_q=3, L=9, Hq=4, Hkv=2, D=8)
    out = oracle.attend_core(q, k, v, pos_q, pos_k, vis, 1e4, rope_style=1)
    ref = brute_force_variant(q, k, v, pos_q, pos_k, vis, 1e4, pairing="interleaved")
    assert np.abs(out - ref).max() < 1e-12
    half = oracle.attend_core(q, k, v, pos_q, pos_k, vis, 1e4)
    assert np.abs(out - half).max() > 1e-3                      # the two pairings are different functions
    perm = np.concatenate([np.arange(0, 8, 2), np.arange(1, 8, 2)])
    via_perm = oracle.attend_core(q[..., perm], k[..., perm], v, pos_q, pos_k, vis, 1e4)
    assert np.abs(out - via_perm).max() < 1e-12
    # SURVEY 8.c worked example B, interleaved reading: D=4, K rows (0,1,0,0), q=(0,2,0,0), keys at 0/100/200,
    # query at 200: index 1 pairs with index 0 at frequency 1 -> scores cos(200-n), n = 0, 100, 200
    kk = np.zeros((3, 1, 4)); kk[:, 0, 1] = 1.0
    vv = np.eye(3, 4).reshape(3, 1, 4)
    qq = np.array([[[0.0, 2.0, 0.0, 0.0]]])
    o = oracle.attend_core(qq, kk, vv, [200.0], [0.0, 100.0, 200.0], [2], 1e4, rope_style=1)
    e = np.exp(np.cos(np.array([200.0, 100.0, 0.0])))
    assert np.abs(o[0, 0, :3] - e / e.sum()).max() < 1e-12


def test_custom_frequencies_scale_and_partial_rotary():
    """L213: frequency-scaled RoPE families only change the per-pair frequency vector (and YaRN a scalar
    temperature).  Default vector reproduces the default path bit for bit; an arbitrary vector and scale match
    brute force; zero frequencies leave those pairs un-rotated (partial rotary)."""
    q, k, v, pos_q, pos_k, vis = random_case(73, n_q=2, L=10, Hq=2, Hkv=1, D=8)
    theta = 5e5
    base = theta ** (-2.0 * np.arange(4) / 8)
    a = oracle.attend_core(q, k, v, pos_q, pos_k, vis, theta)
    b = oracle.attend_core(q, k, v, pos_q, pos_k, vis, theta, inv_freq=base)
    assert np.array_equal(a, b)
    # a Llama-3.1-style rescaling written out here: low frequencies divided by 8, high kept, middle blended
    wavelen = 2 * math.pi / base
    lo, hi, factor, orig = 1.0, 4.0, 8.0, 64.0
    smooth = np.clip((orig / wavelen - lo) / (hi - lo), 0.0, 1.0)
    scaled = np.where(wavelen > orig / lo, base / factor, np.where(wavelen < orig / hi, base,
                                                                  (1 - smooth) * base / factor + smooth * base))
    out = oracle.attend_core(q, k, v, pos_q, pos_k, vis, theta, inv_freq=scaled, scale=0.41)
    ref = brute_force_variant(q, k, v, pos_q, pos_k, vis, theta, inv_freq=scaled, scale=0.41)
    assert np.abs(out - ref).max() < 1e-12
    # partial rotary: pairs 2, 3 carry frequency 0 -> those dims behave as with all positions 0
    part = base.copy(); part[2:] = 0.0
    out = oracle.attend_core(q, k, v, pos_q, pos_k, vis, theta, inv_freq=part)
    ref = brute_force_variant(q, k, v, pos_q, pos_k, vis, theta, inv_freq=part)
    assert np.abs(out - ref).max() < 1e-12


def test_alibi_bias_brute_force_closed_form_and_paged():
    """L221: ALiBi -- no rotation, score bias slope_h * (n - m).  Brute force; closed form with q = 0 (weights
    proportional to exp(slope * n)); shift invariance; and through the paged wrapper, where the bias must use the
    LOGICAL position of a page (same page at two positions -> different biases)."""
    q, k, v, pos_q, pos_k, vis = random_case(79, n_q=3, L=12, Hq=4, Hkv=2, D=8)
    slopes = np.array([0.5, 0.25, 0.125, 0.0625])
    out = oracle.attend_core(q, k, v, pos_q, pos_k, vis, 1e4, alibi_slopes=slopes)
    ref = brute_force_variant(q, k, v, pos_q, pos_k, vis, 1e4, slopes=slopes)
    assert np.abs(out - ref).max() < 1e-12
    out2 = oracle.attend_core(q, k, v, pos_q + 1000, pos_k + 1000, vis, 1e4, alibi_slopes=slopes)
    assert np.abs(out - out2).max() < 1e-10
    z = oracle.attend_core(np.zeros_like(q), k, v, pos_q, pos_k, vis, 1e4, alibi_slopes=slopes, want_probs=True)[1]
    for i in range(3):
        for hq in range(4):
            w = np.exp(slopes[hq] * (pos_k[: vis[i] + 1] - pos_k[vis[i]]))
            assert np.abs(z[i, hq, : vis[i] + 1] - w / w.sum()).max() < 1e-12
    r = _rng(83)
    Hq, Hkv, D, P = 2, 1, 8, 4
    kp = r.standard_normal((3, Hkv, P, D)); vp = r.standard_normal((3, Hkv, P, D))
    bt = np.array([[1, 0, 1, 2]], np.int32); pp = np.array([[0, 4, 30, 34]], np.int32)   # page 1 at 0 and at 30
    sl = np.array([14], np.int32); cu = np.array([0, 2], np.int32)
    qq = r.standard_normal((2, Hq, D)); s2 = np.array([0.3, 0.05])
    got = oracle.attend_paged(qq, kp, vp, bt, pp, sl, cu, num_q_heads=Hq, num_kv_heads=Hkv, head_dim=D, page_size=P,
                              theta=1e4, alibi_slopes=s2)
    kk = np.stack([kp[bt[0, s // P], :, s % P] for s in range(14)])
    vv = np.stack([vp[bt[0, s // P], :, s % P] for s in range(14)])
    pos = np.array([pp[0, s // P] + s % P for s in range(14)], dtype=np.float64)
    ref = brute_force_variant(qq, kk, vv, pos[12:], pos, np.array([12, 13]), 1e4, slopes=s2)
    assert np.abs(got - ref).max() < 1e-12

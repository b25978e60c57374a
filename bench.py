#!/usr/bin/env python
"""bench.py -- LazyAttention hot path on B200: one JSON line per run (see README "Benchmark").

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2|cfg3|cfg4|cfg5] [--impl ours|reference]

A step = one pass of the whole hot path over one synthetic Zipf-shared RAG batch: lazy_cache_write of the
step's new tokens, then the attention call(s) (decode for cfg2/cfg4, prefill for cfg3, prefill + decode for
cfg5).  Default workload: BASELINE.json configs[1] (decode at the Llama-3-8B layer shape); unless
--no-secondary, configs[2..4] (prefill, long-context decode, mixed step) are measured in the same run and
reported kernel by kernel under "configs".  The decode `roofline` is taken on the noshare variant of the
workload (every drawn document distinct, so algorithmic bytes are DRAM bytes); the Zipf-shared numbers, where
the L2 serves repeated pages, sit under roofline.shared.
`--impl reference` times the fp64 CPU oracle (oracle/) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np
import torch


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=float(d["hbm_gbs"]), tensor=float(d["bf16_tflops"]),
                    tensor_sustained=float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), source="measured")
    return dict(hbm=6650.0, tensor=1590.0, tensor_sustained=1400.0, source="fallback")


def ncu_traffic(kernel: str, workload: str):
    """dram read + write bytes per launch of the dominant kernel from the committed ncu --set full capture
    (profiles/*_traffic.csv, latest round wins); None when that workload has not been captured."""
    import csv
    import glob
    val = None
    for f in sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_traffic.csv"))):
        for row in csv.DictReader(open(f)):
            if row["kernel"] == kernel and row["workload"] == workload:
                val = int(row["dram_bytes_read"]) + int(row["dram_bytes_write"])
    return val


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------------------------
def make_batch(workload: str, rank: int, noshare: bool = False):
    from paper_2606_04302_b200 import workloads as W
    idx = int(workload[3:])
    kw = dict(noshare=True) if noshare else {}
    if idx == 5:
        return W.config5(**kw)
    b = W.CONFIGS[idx](**kw)
    if rank:
        # weak scaling: every rank owns a batch of the same shape drawn from its own seed
        import dataclasses  # noqa: F401
        W_SEED = W.SEED0
        W.SEED0 = W_SEED + 1000 * rank
        try:
            b = W.CONFIGS[idx](**kw)
        finally:
            W.SEED0 = W_SEED
    return b


def step_work(batch, steps, fp8=False):
    """Algorithmic work of the timed attention calls.  fp8: LAZY_KV_FP8_E4M3
    pages move D bytes of codes + one fp32 scale per (token, kv head), for K and for V: 2*(D + 4) B instead of 4*D."""
    sh = batch.shape
    logical = 0          # decode: K and V once per (token, kv head): 2*D*2 B, + q/out
    flops = 0            # prefill: 4*D FLOPs per visible (query, key) pair per q head
    q_tokens = dec_tokens = kv_tokens = 0
    for st in steps:
        L = st.seq_lens.numpy().astype(np.int64)
        if st.kind == "decode":
            logical += int(L.sum()) * sh.num_kv_heads * (2 * (sh.head_dim + 4) if fp8 else sh.head_dim * 2 * 2)
            logical += len(L) * sh.num_q_heads * sh.head_dim * 2 * 2
            dec_tokens += len(L)
            kv_tokens += int(L.sum())
        else:
            nq = (st.cu_q_lens[1:] - st.cu_q_lens[:-1]).numpy().astype(np.int64)
            pairs = int((nq * (L - nq) + nq * (nq + 1) // 2).sum())
            flops += 4 * sh.head_dim * sh.num_q_heads * pairs
            q_tokens += int(nq.sum())
    return dict(logical_bytes=logical, flops=flops, q_tokens=q_tokens, dec_tokens=dec_tokens, kv_tokens=kv_tokens)


def unique_bytes(batch, steps):
    sh = batch.shape
    P = sh.page_size
    pages = set()
    for st in steps:
        if st.kind != "decode":
            continue
        bt = batch.block_table if st.req_ids is None else batch.block_table[st.req_ids]
        for r, L in enumerate(st.seq_lens.tolist()):
            pages.update(bt[r, : (L + P - 1) // P].tolist())
    return len(pages) * sh.num_kv_heads * P * sh.head_dim * 2 * 2


class GpuJob:
    """Holds the device-resident batch and replays its timed step."""

    def __init__(self, batch, device, fp8=False):
        from paper_2606_04302_b200.runner import DeviceBatch
        from paper_2606_04302_b200 import binding as B
        self.B = B
        self.batch = batch
        self.dev = DeviceBatch(batch, device=device, dtype=B.LAZY_KV_FP8_E4M3 if fp8 else B.LAZY_KV_BF16)
        d = self.dev.device
        self.timed = []
        for st in batch.steps:
            if st.kind == "write_only":
                self.dev.write(st)                     # set-up: question tokens already in the cache
        # cfg5's follow-up decode (last step) is a correctness-only call: not timed
        steps = [s for s in batch.steps if s.kind != "write_only"]
        if batch.name.startswith("cfg5"):
            steps = steps[:2]
        for st in steps:
            bt, pp = self.dev.tables_for(st)
            rec = dict(step=st, bt=bt, pp=pp, q=st.q.to(d), out=torch.empty_like(st.q, device=d),
                       sl=st.seq_lens.to(d), k_new=st.k_new.to(d), v_new=st.v_new.to(d),
                       slots=st.slot_mapping.to(d))
            if st.kind == "prefill":
                rec["cu"] = st.cu_q_lens.to(d)
                rec["max_q"] = int((st.cu_q_lens[1:] - st.cu_q_lens[:-1]).max())
            self.timed.append(rec)
        # one lazy_cache_write per step: the ABI takes ONE slot mapping over all new tokens of the step (prefill chunk
        # tokens and the decode tokens alike), which is how a serving engine hands them over
        self.kv_cat = None
        if len(self.timed) > 1:
            self.kv_cat = tuple(torch.cat([r[k] for r in self.timed]).contiguous() for k in ("k_new", "v_new", "slots"))
        self.flush_buf = torch.empty(512 << 20, dtype=torch.uint8, device=d)
        self.sweep_buf = torch.zeros(64 << 20, dtype=torch.int32, device=d)      # 256 MB

    def flush_l2(self):
        # write a buffer larger than L2 (evicts every input line), then read-sweep another one so that the dirty
        # lines of the fill are written back BEFORE the timed region instead of competing with the kernel's reads
        self.flush_buf.fill_(1)
        self.sweep_buf.sum()

    def run(self, ev_mid=None, call_evs=None):
        """call_evs: list that receives one (start, end) event pair per attention call (separate calls only)."""
        B, dev = self.B, self.dev
        if self.kv_cat is not None:
            B.lazy_cache_write(dev.handle, self.kv_cat[0], self.kv_cat[1], self.kv_cat[2], dev.k_pool, dev.v_pool)
        else:
            for rec in self.timed:
                B.lazy_cache_write(dev.handle, rec["k_new"], rec["v_new"], rec["slots"], dev.k_pool, dev.v_pool)
        if ev_mid is not None:
            ev_mid.record()
        kinds = [rec["step"].kind for rec in self.timed]
        if kinds == ["prefill", "decode"] and not getattr(self, "separate_calls", False):
            # mixed serving step (cfg5): the two attention calls are issued together (lazy_attn_mixed)
            rp, rd = self.timed
            B.lazy_attn_mixed(dev.handle, dev.k_pool, dev.v_pool, q_prefill=rp["q"], block_table_prefill=rp["bt"],
                              page_logical_pos_prefill=rp["pp"], seq_lens_prefill=rp["sl"], cu_q_lens=rp["cu"],
                              max_q_len=rp["max_q"], out_prefill=rp["out"], q_decode=rd["q"],
                              block_table_decode=rd["bt"], page_logical_pos_decode=rd["pp"], seq_lens_decode=rd["sl"],
                              out_decode=rd["out"])
            return
        for rec in self.timed:
            if call_evs is not None:
                e0 = torch.cuda.Event(enable_timing=True); e0.record()
            if rec["step"].kind == "decode":
                B.lazy_attn_decode(dev.handle, rec["q"], dev.k_pool, dev.v_pool, rec["bt"], rec["pp"], rec["sl"],
                                   rec["out"])
            else:
                B.lazy_attn_prefill(dev.handle, rec["q"], dev.k_pool, dev.v_pool, rec["bt"], rec["pp"], rec["sl"],
                                    rec["cu"], rec["max_q"], rec["out"])
            if call_evs is not None:
                e1 = torch.cuda.Event(enable_timing=True); e1.record()
                call_evs.append((rec["step"].kind, e0, e1))

    def time_calls(self, steps, warmup):
        """Per attention call (separate calls), L2 flushed before EVERY call: {kind: mean kernel ms}."""
        keep = getattr(self, "separate_calls", False)
        self.separate_calls = True
        try:
            acc = {}
            for i in range(warmup + steps):
                for rec in self.timed:
                    self.B.lazy_cache_write(self.dev.handle, rec["k_new"], rec["v_new"], rec["slots"], self.dev.k_pool,
                                            self.dev.v_pool)
                evs = []
                for rec in self.timed:
                    self.flush_l2()
                    one = GpuJob.__new__(GpuJob)
                    one.__dict__.update(self.__dict__)
                    one.timed = [dict(rec, k_new=rec["k_new"][:0], v_new=rec["v_new"][:0], slots=rec["slots"][:0])]
                    one.kv_cat = None
                    one.run(call_evs=evs)
                torch.cuda.synchronize()
                if i >= warmup:
                    for kind, e0, e1 in evs:
                        acc.setdefault(kind, []).append(e0.elapsed_time(e1))
            return {k: float(np.mean(v)) for k, v in acc.items()}
        finally:
            self.separate_calls = keep

    def time_steps(self, steps, warmup, barrier):
        for _ in range(warmup):
            self.flush_l2(); self.run()
        n0 = self.dev.handle.launch_count()
        evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
        barrier(); torch.cuda.synchronize()
        for i in range(steps):
            self.flush_l2()                          # > L2 (126 MB) written between timed iterations
            evs[i][0].record()
            self.run(ev_mid=evs[i][1])
            evs[i][2].record()
        torch.cuda.synchronize(); barrier()
        total = sum(e[0].elapsed_time(e[2]) for e in evs)
        attn = sum(e[1].elapsed_time(e[2]) for e in evs)
        return total, attn, self.dev.handle.launch_count() - n0

    # -------- end to end through lazy_host_step_packed (HOST buffers; copies inside the timed region)
    def prepare_e2e(self):
        """Every step's inputs live in ONE pinned host block laid out by lazy_host_step_layout (where a serving engine's
        scheduler would write them): the step is one H2D copy, the kernels, one D2H copy of the outputs."""
        B, dev = self.B, self.dev
        self.e2e = []
        for rec in self.timed:
            st = rec["step"]
            bt = self.batch.block_table if st.req_ids is None else self.batch.block_table[st.req_ids]
            pp = self.batch.page_logical_pos if st.req_ids is None else self.batch.page_logical_pos[st.req_ids]
            R, tq, nn = st.seq_lens.shape[0], st.q.shape[0], st.k_new.shape[0]
            lay = B.lazy_host_step_layout(dev.handle, R, tq, nn)
            packed = torch.zeros(int(lay.in_bytes), dtype=torch.uint8).pin_memory()
            h2d = 0

            def put(off, t):
                nonlocal h2d
                raw = t.contiguous().view(torch.uint8).reshape(-1)
                packed[off:off + raw.numel()] = raw
                h2d += raw.numel()
            put(lay.q, st.q); put(lay.k_new, st.k_new); put(lay.v_new, st.v_new); put(lay.slot_mapping, st.slot_mapping)
            put(lay.block_table, bt.to(torch.int32)); put(lay.page_logical_pos, pp.to(torch.int32))
            put(lay.seq_lens, st.seq_lens)
            kind = 0 if st.kind == "decode" else 1
            if kind == 1:
                put(lay.cu_q_lens, st.cu_q_lens)
            out = torch.empty_like(st.q).pin_memory()
            staging = torch.empty(int(lay.staging_bytes) + 256, dtype=torch.uint8, device=dev.device)
            base = (staging.data_ptr() + 255) // 256 * 256
            args = B.HostStepPacked(kind, R, tq, rec.get("max_q", 1), nn, 0, packed.data_ptr(), out.data_ptr(),
                                    dev.k_pool.data_ptr(), dev.v_pool.data_ptr(), base, int(lay.staging_bytes))
            self.e2e.append(dict(args=args, packed=packed, out=out, staging=staging, h2d=int(lay.in_bytes),
                                 h2d_payload=h2d, d2h=out.numel() * 2))

    def prepare_e2e_unpacked(self):
        """The same steps through lazy_host_step: every input in its own pinned host tensor (what a caller with separate
        tensors hands over), seven H2D copies per step instead of one packed block."""
        B, dev = self.B, self.dev
        self.e2e_unpacked = []
        pin = lambda t: t.contiguous().pin_memory()
        for rec in self.timed:
            st = rec["step"]
            bt = self.batch.block_table if st.req_ids is None else self.batch.block_table[st.req_ids]
            pp = self.batch.page_logical_pos if st.req_ids is None else self.batch.page_logical_pos[st.req_ids]
            R, tq, nn = st.seq_lens.shape[0], st.q.shape[0], st.k_new.shape[0]
            host = dict(q=pin(st.q), k=pin(st.k_new), v=pin(st.v_new), s=pin(st.slot_mapping), bt=pin(bt.to(torch.int32)),
                        pp=pin(pp.to(torch.int32)), sl=pin(st.seq_lens),
                        cu=pin(st.cu_q_lens) if st.kind != "decode" else None)
            out = torch.empty_like(st.q).pin_memory()
            nbytes = B.lazy_host_step_staging_bytes(dev.handle, R, tq, nn)
            staging = torch.empty(nbytes + 256, dtype=torch.uint8, device=dev.device)
            base = (staging.data_ptr() + 255) // 256 * 256
            args = B.HostStep(0 if st.kind == "decode" else 1, R, tq, rec.get("max_q", 1), nn, 0, host["q"].data_ptr(),
                              host["k"].data_ptr(), host["v"].data_ptr(), host["s"].data_ptr(), host["bt"].data_ptr(),
                              host["pp"].data_ptr(), host["sl"].data_ptr(),
                              None if host["cu"] is None else host["cu"].data_ptr(), out.data_ptr(),
                              dev.k_pool.data_ptr(), dev.v_pool.data_ptr(), base, nbytes)
            self.e2e_unpacked.append(dict(args=args, host=host, out=out, staging=staging))

    def run_e2e(self):
        for e in self.e2e:
            self.B.lazy_host_step_packed(self.dev.handle, e["args"])

    def run_e2e_unpacked(self):
        for e in self.e2e_unpacked:
            self.B.lazy_host_step(self.dev.handle, e["args"])

    def time_e2e(self, steps, warmup, barrier, run=None):
        run = run or self.run_e2e
        for _ in range(warmup):
            self.flush_l2(); run()
        evs = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(steps)]
        barrier(); torch.cuda.synchronize()
        for i in range(steps):
            self.flush_l2()
            evs[i][0].record()
            run()
            evs[i][1].record()
        torch.cuda.synchronize(); barrier()
        return sum(e[0].elapsed_time(e[1]) for e in evs)

    def verify_e2e(self):
        """Outside every timed region: what the timed host-buffer calls wrote to h_out against the `out` of the
        device-pointer step on the same handle.  Prefill is the same kernel on the same grid (bit equal); decode may
        differ in the split-KV combine order (which CTA arrives last), hence a bound instead of equality."""
        self.run(); self.run_e2e()
        if getattr(self, "e2e_unpacked", None):
            self.run_e2e_unpacked()
        torch.cuda.synchronize()
        worst, bit_equal = 0.0, True
        for i, rec in enumerate(self.timed):
            want = rec["out"].float().cpu()
            for e in [self.e2e[i]] + ([self.e2e_unpacked[i]] if getattr(self, "e2e_unpacked", None) else []):
                got = e["out"].float()
                assert torch.isfinite(got).all(), "e2e output is not finite"
                worst = max(worst, float((got - want).abs().max()))
                bit_equal = bit_equal and bool(torch.equal(e["out"].view(torch.int16), rec["out"].cpu().view(torch.int16)))
        assert worst < 2e-3, f"e2e output differs from the device-pointer step by {worst}"
        return {"max_abs_diff_vs_device_step": worst, "bit_equal": bit_equal}


def run_ablation(job, steps, warmup):
    """SURVEY 8.0 rows f1 / f2 on the job's batch: every (request, slot) gets a PRIVATE page (same block tables
    and same HBM traffic in every arm), holding K (a) un-rotated, (b) rotated at a document-local stored position
    (the paper's layout: one relative rotation per page), (c) rotated at its final position (rotation compiled
    out: PAPER.md Fig. 5 'without deferred rotation').  The copies are made by lazy_materialize_pages, whose own
    time is the Block-Attention-style re-encoding cost the lazy path avoids."""
    from paper_2606_04302_b200.runner import DeviceBatch
    B, dev, batch = job.B, job.dev, job.batch
    d, sh, P = dev.device, batch.shape, batch.shape.page_size
    rec = job.timed[-1]                               # the attention call of the step (decode, or cfg3's prefill)
    st = rec["step"]
    bt_h = batch.block_table if st.req_ids is None else batch.block_table[st.req_ids]
    pp_h = batch.page_logical_pos if st.req_ids is None else batch.page_logical_pos[st.req_ids]
    R, pmax = bt_h.shape
    need = (st.seq_lens.to(torch.int64) + P - 1) // P
    mask = torch.arange(pmax)[None, :] < need[:, None]
    src = bt_h[mask].to(torch.int32).contiguous()
    starts = pp_h[mask].to(torch.int32).contiguous()
    n = int(src.numel())
    bt_priv = torch.zeros(R, pmax, dtype=torch.int32)
    bt_priv[mask] = torch.arange(n, dtype=torch.int32)
    doc_pages = max(1, int(batch.meta.get("doc_len", 256)) // P)
    slot = torch.arange(pmax)[None, :].expand(R, pmax)[mask]
    stored = ((slot % doc_pages) * P).to(torch.int32).contiguous()
    src_d, dst_d = src.to(d), torch.arange(n, dtype=torch.int32, device=d)
    shape = (n, sh.num_kv_heads, P, sh.head_dim)
    v_priv = torch.empty(shape, dtype=torch.bfloat16, device=d)
    pools = {}
    mat_ms = None
    for name, rot, per_token in (("unrotated", torch.zeros(n, dtype=torch.int32), False),
                                 ("stored_pos", stored, True), ("absolute", starts, True)):
        kp = torch.empty(shape, dtype=torch.bfloat16, device=d)
        rot_d = rot.to(d)
        run = lambda: B.lazy_materialize_pages(dev.handle, dev.k_pool, dev.v_pool, src_d, rot_d, per_token, kp, v_priv,
                                               dst_d)
        run()
        if name == "absolute":                        # time the re-encoding itself (K rotate + V copy), L2 flushed
            evs = []
            for _ in range(5):
                job.flush_l2()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(); run(); e1.record()
                evs.append((e0, e1))
            torch.cuda.synchronize()
            mat_ms = float(np.median([a.elapsed_time(b) for a, b in evs]))
        pools[name] = kp
    res = {"layout": f"private page per (request, slot): {n} pages", "pages": n}
    modes = (("unrotated", B.LAZY_K_UNROTATED, None), ("stored_pos", B.LAZY_K_STORED_POS, stored),
             ("absolute", B.LAZY_K_ABSOLUTE, None))
    for name, km, sp in modes:
        dv = DeviceBatch(batch, device=str(d), k_storage=km, page_stored_pos=sp, k_pool=pools[name], v_pool=v_priv,
                         block_table=bt_priv if st.req_ids is None else None,
                         max_position=batch.max_position + doc_pages * P + P)
        bt_d = bt_priv.to(d)
        pp_d = pp_h.to(d).contiguous()

        def attend():
            if st.kind == "decode":
                B.lazy_attn_decode(dv.handle, rec["q"], dv.k_pool, dv.v_pool, bt_d, pp_d, rec["sl"], rec["out"])
            else:
                B.lazy_attn_prefill(dv.handle, rec["q"], dv.k_pool, dv.v_pool, bt_d, pp_d, rec["sl"], rec["cu"],
                                    rec["max_q"], rec["out"])
        for _ in range(warmup):
            job.flush_l2(); attend()
        evs = []
        for _ in range(steps):
            job.flush_l2()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); attend(); e1.record()
            evs.append((e0, e1))
        torch.cuda.synchronize()
        res[name + "_ms"] = float(np.mean([a.elapsed_time(b) for a, b in evs]))
        dv.close()
    # f3: ALiBi on the batch's own (shared) pool -- same pages, same traffic as the headline RoPE run
    if sh.num_q_heads <= 256:
        slopes = [2.0 ** (-8.0 * (i + 1) / sh.num_q_heads) for i in range(sh.num_q_heads)]
        dv = DeviceBatch(batch, device=str(d), rope_style=B.LAZY_POS_ALIBI, alibi_slopes=slopes, k_pool=dev.k_pool,
                         v_pool=dev.v_pool)

        def attend_alibi():
            if st.kind == "decode":
                B.lazy_attn_decode(dv.handle, rec["q"], dv.k_pool, dv.v_pool, rec["bt"], rec["pp"], rec["sl"], rec["out"])
            else:
                B.lazy_attn_prefill(dv.handle, rec["q"], dv.k_pool, dv.v_pool, rec["bt"], rec["pp"], rec["sl"],
                                    rec["cu"], rec["max_q"], rec["out"])
        for _ in range(warmup):
            job.flush_l2(); attend_alibi()
        evs = []
        for _ in range(steps):
            job.flush_l2()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); attend_alibi(); e1.record()
            evs.append((e0, e1))
        torch.cuda.synchronize()
        res["alibi_shared_ms"] = float(np.mean([a.elapsed_time(b) for a, b in evs]))
        dv.close()
    # f1 on the SHARED pool: every physical page stored rotated by its in-page offset only (page_stored_pos = 0 for
    # all pages -- still reusable at any logical position); the kernels then owe one relative rotation per page
    if True:
        npg = int(dev.k_pool.shape[0])
        allp = torch.arange(npg, dtype=torch.int32, device=d)
        zeros = torch.zeros(npg, dtype=torch.int32, device=d)
        k_loc = torch.empty_like(dev.k_pool)
        B.lazy_materialize_pages(dev.handle, dev.k_pool, None, allp, zeros, True, k_loc, None, allp)
        dv = DeviceBatch(batch, device=str(d), k_storage=B.LAZY_K_STORED_POS, page_stored_pos=zeros.cpu(),
                         k_pool=k_loc, v_pool=dev.v_pool)

        def attend_loc():
            if st.kind == "decode":
                B.lazy_attn_decode(dv.handle, rec["q"], dv.k_pool, dv.v_pool, rec["bt"], rec["pp"], rec["sl"], rec["out"])
            else:
                B.lazy_attn_prefill(dv.handle, rec["q"], dv.k_pool, dv.v_pool, rec["bt"], rec["pp"], rec["sl"],
                                    rec["cu"], rec["max_q"], rec["out"])
        for _ in range(warmup):
            job.flush_l2(); attend_loc()
        evs = []
        for _ in range(steps):
            job.flush_l2()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); attend_loc(); e1.record()
            evs.append((e0, e1))
        torch.cuda.synchronize()
        res["page_local_shared_ms"] = float(np.mean([a.elapsed_time(b) for a, b in evs]))
        dv.close()
        del k_loc
    page_bytes = sh.num_kv_heads * P * sh.head_dim * 2
    res["rotation_overhead_pct"] = (res["unrotated_ms"] / res["absolute_ms"] - 1.0) * 100.0
    res["stored_pos_overhead_pct"] = (res["stored_pos_ms"] / res["absolute_ms"] - 1.0) * 100.0
    res["unrotated_vs_stored_pos_pct"] = (res["unrotated_ms"] / res["stored_pos_ms"] - 1.0) * 100.0
    res["materialize_ms"] = mat_ms
    res["materialize_bytes"] = 4 * n * page_bytes                 # K read + K write + V read + V write
    res["materialize_GBps"] = res["materialize_bytes"] / (mat_ms * 1e-3) / 1e9
    return res


def _round(o):
    """Floats to 5 significant digits (the whole line must fit the driver's 3 KB tail)."""
    if isinstance(o, dict):
        return {k: _round(v) for k, v in o.items()}
    if isinstance(o, list):
        return [_round(v) for v in o]
    if isinstance(o, float):
        return float(f"{o:.5g}")
    return o


def _get(o, *path):
    for k in path:
        if not isinstance(o, dict) or k not in o:
            return None
        o = o[k]
    return o


def compact_line(out):
    """The one JSON line bench.py prints (the verbose record goes to stderr): the contract's keys, the side legs as
    kernel times only, and LAST a flat `summary` -- so that it survives any tail cut -- with both halves of
    BASELINE.json's metric (decode HBM fraction, prefill tensor fraction) and the f1 / f2 figures."""
    line = {k: v for k, v in out.items() if k not in ("configs", "roofline", "e2e", "clocks", "ablation", "tokens_per_s",
                                                      "cpu_baseline", "mixed", "graph", "e3")}
    line["config"] = dict(out["config"], l2="flushed between timed steps", parallelism=f"replicas x{out['n_gpus']}")
    r = out["roofline"]
    line["roofline"] = {k: r[k] for k in ("bound", "kernel", "achieved", "peak", "unit", "frac", "traffic", "peak_source",
                                          "workload", "kernel_ms", "note") if k in r}
    if "shared" in r:
        line["roofline"]["shared"] = {k: r["shared"][k] for k in ("kernel_ms", "logical_GBps", "unique_GBps", "traffic")}
    e = out["e2e"]
    line["e2e"] = {k: e[k] for k in ("value", "unit", "ms_per_step", "h2d_bytes_per_step", "d2h_bytes_per_step")}
    line["e2e"]["api"] = "lazy_host_step_packed"
    if "unpacked" in e:
        line["e2e"]["lazy_host_step_ms"] = e["unpacked"]["ms_per_step"]
        line["e2e"]["verified"] = e["verified"]
    line["clocks"] = {k: v for k, v in out["clocks"].items() if k not in ("window", "samples")}
    for k in ("mixed", "graph", "e3"):
        if k in out:
            line[k] = out[k]
    c = out.get("configs") or {}
    if c:
        picks = {"cfg3_ms": ("cfg3", "kernel_ms"), "cfg3_sustained_ms": ("cfg3", "sustained", "kernel_ms"),
                 "cfg3_sustained_reasons": ("cfg3", "sustained", "clocks", "reasons"),
                 "cfg4_noshare_ms": ("cfg4", "noshare", "kernel_ms"), "cfg4_shared_ms": ("cfg4", "shared", "kernel_ms"),
                 "cfg4_shared_logical_GBps": ("cfg4", "shared", "logical_GBps"),
                 "cfg5_prefill_ms": ("cfg5", "prefill", "kernel_ms"),
                 "cfg5_decode_noshare_ms": ("cfg5", "decode_noshare", "kernel_ms"),
                 "cfg5_decode_shared_ms": ("cfg5", "decode_shared", "kernel_ms"),
                 "cfg5_cache_write_ms": ("cfg5", "cache_write", "ms"),
                 "fp8_cfg2_ms": ("fp8_pages", "cfg2_noshare", "kernel_ms"),
                 "fp8_cfg4_ms": ("fp8_pages", "cfg4_noshare", "kernel_ms"),
                 "fp8_cfg5_ms": ("fp8_pages", "cfg5_noshare", "kernel_ms"),
                 "fp8_cfg3_prefill_ms": ("fp8_pages", "cfg3_prefill", "kernel_ms"),
                 "fp8_cfg5_mixed_step_ms": ("fp8_pages", "cfg5_mixed_step", "ms_per_step")}
        line["configs"] = {k: _get(c, *p) for k, p in picks.items() if _get(c, *p) is not None}
        errs = {k: v["error"] for k, v in c.items() if isinstance(v, dict) and "error" in v}
        if errs:
            line["configs"]["errors"] = errs
    ab = out.get("ablation") or {}
    if ab:
        line["ablation"] = {k: ab[k] for k in ("unrotated_ms", "stored_pos_ms", "absolute_ms", "materialize_GBps") if k in ab}
    if "cpu_baseline" in out:
        line["cpu_baseline"] = {k: v for k, v in out["cpu_baseline"].items() if k != "seconds"}
    sm = {}

    def put(name, *path, src=None):
        v = _get(c if src is None else src, *path)
        if v is not None:
            sm[name] = v
    wl = out["config"]["workload"].split()[0]
    sm[f"{wl}_roofline_frac"] = r["frac"]
    put("cfg2_shared_logical_GBps", "shared", "logical_GBps", src=r)
    put("cfg3_TFLOPs", "cfg3", "TFLOPs"); put("cfg3_frac_burst", "cfg3", "frac_of_bf16_peak")
    put("cfg3_sustained_TFLOPs", "cfg3", "sustained", "TFLOPs")
    put("cfg3_frac_sustained", "cfg3", "sustained", "frac_of_bf16_sustained")
    put("cfg3_sm_mhz", "cfg3", "sustained", "clocks", "sm_mhz")
    put("cfg4_noshare_frac", "cfg4", "noshare", "frac_of_hbm_peak")
    put("cfg5_decode_noshare_frac", "cfg5", "decode_noshare", "frac_of_hbm_peak")
    put("cfg5_prefill_frac", "cfg5", "prefill", "frac_of_bf16_peak")
    put("cfg5_mixed_attention_ms", "cfg5", "mixed_attention_ms"); put("cfg5_mixed_step_ms", "cfg5", "mixed_step_ms")
    put("fp8_cfg2_frac", "fp8_pages", "cfg2_noshare", "frac_of_hbm_peak")
    put("fp8_cfg4_frac", "fp8_pages", "cfg4_noshare", "frac_of_hbm_peak")
    put("fp8_cfg5_frac", "fp8_pages", "cfg5_noshare", "frac_of_hbm_peak")
    put("fp8_cfg3_frac_burst", "fp8_pages", "cfg3_prefill", "frac_of_bf16_peak")
    for k in ("rotation_overhead_pct", "materialize_ms", "lazy_speedup_vs_materialising"):
        put(k, k, src=ab)
    line["summary"] = sm
    return _round(line)


def headline(workload, work, ms_step):
    s = ms_step * 1e-3
    if workload in ("cfg2", "cfg4"):
        return "decode_attn_logical_GBps", work["logical_bytes"] / s / 1e9, "GB/s"
    if workload == "cfg3":
        return "prefill_attn_TFLOPs", work["flops"] / s / 1e12, "TFLOP/s"
    return "mixed_step_attn_tokens_per_s", (work["q_tokens"] + work["dec_tokens"]) / s, "tokens/s"


# ------------------------------------------------------------------------------------------------------
def oracle_sample(workload, batch, budget_s=20.0):
    """Times the oracle as it stands on a bounded sample of the workload; returns (value in the headline's
    unit, seconds, description).  Decode: the first requests; prefill: seeded query rows of request 0."""
    from oracle import oracle as O
    O.build()
    sh = batch.shape
    steps = [s for s in batch.steps if s.kind != "write_only"]
    if batch.name.startswith("cfg5"):
        steps = steps[:2]
    k_ref, v_ref = batch.k_pool.clone(), batch.v_pool.clone()
    for st in batch.steps:
        if st.k_new is not None:
            O.cache_write(st.k_new, st.v_new, st.slot_mapping.numpy(), k_ref, v_ref, sh.page_size)
    t_total, logical, flops, toks = 0.0, 0, 0, 0
    desc = []
    for st in steps:
        bt = batch.block_table if st.req_ids is None else batch.block_table[st.req_ids]
        pp = batch.page_logical_pos if st.req_ids is None else batch.page_logical_pos[st.req_ids]
        R = st.seq_lens.shape[0]
        if st.kind == "decode":
            n = max(1, min(R, 64))
            sl = st.seq_lens[:n].numpy()
            t0 = time.perf_counter()
            O.attend_paged(st.q[:n], k_ref, v_ref, bt[:n].numpy(), pp[:n].numpy(), sl,
                           np.arange(n + 1, dtype=np.int32), num_q_heads=sh.num_q_heads,
                           num_kv_heads=sh.num_kv_heads, head_dim=sh.head_dim, page_size=sh.page_size,
                           theta=sh.rope_theta)
            t_total += time.perf_counter() - t0
            logical += int(sl.sum()) * sh.num_kv_heads * sh.head_dim * 4 + n * sh.num_q_heads * sh.head_dim * 4
            toks += n
            desc.append(f"decode: first {n} of {R} requests")
        else:
            nq = int(st.cu_q_lens[1] - st.cu_q_lens[0])
            L = int(st.seq_lens[0])
            rows = min(nq, 128)
            sel = np.zeros(nq, dtype=np.uint8)
            pick = np.sort(np.random.default_rng(0).choice(nq, size=rows, replace=False))
            sel[pick] = 1
            t0 = time.perf_counter()
            O.attend_paged(st.q[:nq], k_ref, v_ref, bt[:1].numpy(), pp[:1].numpy(), st.seq_lens[:1].numpy(),
                           np.array([0, nq], dtype=np.int32), num_q_heads=sh.num_q_heads,
                           num_kv_heads=sh.num_kv_heads, head_dim=sh.head_dim, page_size=sh.page_size,
                           theta=sh.rope_theta, row_select=sel)
            t_total += time.perf_counter() - t0
            flops += 4 * sh.head_dim * sh.num_q_heads * int(sum(L - nq + i + 1 for i in pick))
            toks += rows
            desc.append(f"prefill: {rows} seeded query rows of request 0 of {R} (materialise + attend)")
    if workload in ("cfg2", "cfg4"):
        v = logical / t_total / 1e9
    elif workload == "cfg3":
        v = flops / t_total / 1e12
    else:
        v = toks / t_total
    return v, t_total, "; ".join(desc), O.num_threads()


def _timed_job(workload, device, steps, noshare=False, warmup=3, fp8=False):
    b = make_batch(workload, 0, noshare)
    j = GpuJob(b, device, fp8=fp8)
    w = step_work(b, [r["step"] for r in j.timed], fp8=fp8)
    return b, j, w


def decode_noshare_leg(workload, device, steps, barrier, fp8=False):
    b, j, w = _timed_job(workload, device, steps, noshare=True, fp8=fp8)
    _, a_ms, _ = j.time_steps(steps, 3, barrier)
    j.dev.close()
    return dict(kernel_ms=a_ms / steps, bytes=w["logical_bytes"])


def fp8_leg(device, steps, peaks, barrier):
    """the decode configs on LAZY_KV_FP8_E4M3 pages (E4M3 codes + one fp32 scale per row), noshare
    variants, against the HBM roofline on the HALVED algorithmic bytes (264 B per (token, kv head) at head_dim 128)."""
    res = {"dtype": "fp8_e4m3 pages (bf16 q / out, f16 tensor operands, fp32 accumulate)",
           "bytes_per_token_kv_head": 264}
    for wl in ("cfg2", "cfg4", "cfg5"):
        b, j, w = _timed_job(wl, device, steps, noshare=True, fp8=True)
        if wl == "cfg5":
            per = j.time_calls(steps, 3)
            wd = step_work(b, [r["step"] for r in j.timed if r["step"].kind == "decode"], fp8=True)
            ms, nbytes = per["decode"], wd["logical_bytes"]
        else:
            _, a_ms, _ = j.time_steps(steps, 3, barrier)
            ms, nbytes = a_ms / steps, w["logical_bytes"]
        j.dev.close()
        del j, b
        torch.cuda.empty_cache()
        gb = nbytes / (ms * 1e-3) / 1e9
        res[wl + "_noshare"] = {"kernel_ms": ms, "algorithmic_bytes_per_launch": nbytes, "GBps": gb,
                                "frac_of_hbm_peak": gb / peaks["hbm"],
                                "traffic": ncu_traffic("decode_fp8", wl + "_noshare")}
    # prefill over FP8 pages (tcgen05 kernel, the rotate warpgroup dequantises both tiles): same FLOPs as cfg3
    b, j, w = _timed_job("cfg3", device, steps, fp8=True)
    _, a_ms, _ = j.time_steps(max(3, steps // 2), 3, barrier)
    ms = a_ms / max(3, steps // 2)
    j.dev.close()
    del j, b
    torch.cuda.empty_cache()
    tf = w["flops"] / (ms * 1e-3) / 1e12
    res["cfg3_prefill"] = {"bound": "tensor", "kernel_ms": ms, "TFLOPs": tf, "frac_of_bf16_peak": tf / peaks["tensor"],
                           "traffic": ncu_traffic("prefill_fp8", "cfg3")}
    # the mixed step (configs[4]) on FP8 pages: one launch (mixed_step_fp8_kernel)
    b, j, w = _timed_job("cfg5", device, steps, fp8=True)
    t_ms, a_ms, _ = j.time_steps(steps, 3, barrier)
    j.dev.close()
    del j, b
    torch.cuda.empty_cache()
    res["cfg5_mixed_step"] = {"ms_per_step": t_ms / steps, "attention_ms": a_ms / steps}
    return res


def decode_leg(workload, device, steps, peaks, barrier):
    """Decode config as a side leg: Zipf-shared batch (logical GB/s) and its noshare variant (the HBM fraction)."""
    b, j, w = _timed_job(workload, device, steps)
    t_ms, a_ms, _ = j.time_steps(steps, 3, barrier)
    ub = unique_bytes(b, [r["step"] for r in j.timed])
    j.dev.close()
    del j, b
    torch.cuda.empty_cache()
    ns = decode_noshare_leg(workload, device, steps, barrier)
    gb = ns["bytes"] / (ns["kernel_ms"] * 1e-3) / 1e9
    a = a_ms / steps
    return {"workload": workload, "bound": "hbm",
            "noshare": {"kernel_ms": ns["kernel_ms"], "algorithmic_bytes_per_launch": ns["bytes"], "GBps": gb,
                        "frac_of_hbm_peak": gb / peaks["hbm"], "traffic": ncu_traffic("decode", workload + "_noshare")},
            "shared": {"kernel_ms": a, "ms_per_step": t_ms / steps, "logical_GBps": w["logical_bytes"] / (a * 1e-3) / 1e9,
                       "logical_over_hbm_peak": w["logical_bytes"] / (a * 1e-3) / 1e9 / peaks["hbm"],
                       "unique_GBps": ub / (a * 1e-3) / 1e9, "traffic": ncu_traffic("decode", workload)}}


def prefill_leg(workload, device, steps, peaks, barrier, sustained_s=2.0):
    """Prefill config: burst (L2 flushed between launches, vs the burst peak) and a seconds-long back-to-back run with
    its own clock record (vs the sustained peak measured under the power cap)."""
    b, j, w = _timed_job(workload, device, steps)
    t_ms, a_ms, _ = j.time_steps(steps, 3, barrier)
    a = a_ms / steps
    tf = w["flops"] / (a * 1e-3) / 1e12
    res = {"workload": workload, "bound": "tensor", "kernel_ms": a, "ms_per_step": t_ms / steps, "TFLOPs": tf,
           "frac_of_bf16_peak": tf / peaks["tensor"], "traffic": ncu_traffic("prefill", workload),
           "query_tokens_per_s": w["q_tokens"] / (t_ms / steps * 1e-3)}
    rec = [r for r in j.timed if r["step"].kind == "prefill"][0]
    call = lambda: j.B.lazy_attn_prefill(j.dev.handle, rec["q"], j.dev.k_pool, j.dev.v_pool, rec["bt"], rec["pp"],
                                         rec["sl"], rec["cu"], rec["max_q"], rec["out"])
    n = max(50, int(sustained_s * 1e3 / a))
    sampler = ClockSampler(torch.cuda.current_device())
    sampler.start()
    for _ in range(20):
        call()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(n):
        call()
    e1.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1) / n
    tfs = w["flops"] / (ms * 1e-3) / 1e12
    res["sustained"] = {"launches": n, "seconds": ms * n * 1e-3, "kernel_ms": ms, "TFLOPs": tfs,
                        "frac_of_bf16_sustained": tfs / peaks["tensor_sustained"],
                        "frac_of_bf16_peak": tfs / peaks["tensor"], "clocks": clocks,
                        "note": "back-to-back launches, no L2 flush (the K/V working set of 1.1 GB exceeds the L2)"}
    j.dev.close()
    return res


def _cache_write_entry(_batch, tokens, sh, fp8, ms):
    rd = tokens * sh.num_kv_heads * sh.head_dim * 2 * 2                      # bf16 K and V rows in
    wr = tokens * sh.num_kv_heads * (2 * (sh.head_dim + 4) if fp8 else sh.head_dim * 2 * 2)   # pages (+ scales) out
    return {"bound": "hbm", "tokens": tokens, "bytes": rd + wr, "ms": ms, "GBps": (rd + wr) / (ms * 1e-3) / 1e9,
            "note": "one launch over all new tokens of the step; launch-latency-bound at this size"}


def cfg5_leg(device, steps, peaks, job=None, fp8=False):
    """configs[4], kernel by kernel (separate calls, L2 flushed before each): the block-local prefill of the 4 miss
    documents (tensor roofline; 464 one-CTA work items = 232 CTA pairs on 74 SM pairs, causal: 1..8 KV tiles per pair)
    and the decode of the 16 running requests (HBM roofline, on the noshare variant), plus the mixed-step time."""
    own = job is None
    if own:
        b, job, _ = _timed_job("cfg5", device, steps, fp8=fp8)
    per = job.time_calls(steps, 3)
    job_timed_tokens = int(sum(r["k_new"].shape[0] for r in job.timed))
    works = {r["step"].kind: step_work(job.batch, [r["step"]], fp8=fp8) for r in job.timed}
    t_ms, a_ms, _ = job.time_steps(steps, 3, lambda: None)
    if own:
        job.dev.close()
        del job
        torch.cuda.empty_cache()
    bn, jn, _ = _timed_job("cfg5", device, steps, noshare=True, fp8=fp8)
    per_ns = jn.time_calls(steps, 3)
    wn = {r["step"].kind: step_work(bn, [r["step"]], fp8=fp8) for r in jn.timed}
    jn.dev.close()
    tf = works["prefill"]["flops"] / (per["prefill"] * 1e-3) / 1e12
    sh = bn.shape
    grp = sh.num_q_heads // sh.num_kv_heads
    tpt = 128 // grp
    pst = [r["step"] for r in jn.timed if r["step"].kind == "prefill"][0]
    nq = (pst.cu_q_lens[1:] - pst.cu_q_lens[:-1]).numpy()
    pairs = int(sum(-(-int(n) // (4 * tpt)) for n in nq)) * sh.num_kv_heads
    occ = (f"{pairs} CTA pairs ({len(nq)} documents x {sh.num_kv_heads} kv heads x blocks of {4 * tpt} query tokens) on 74 SM "
           f"pairs, one pair per SM pair; causal: a pair runs 1..{-(-int(nq.max()) // 128)} KV tiles; {tpt * grp} of 128 rows "
           f"of a Q tile used (group {grp})")
    gb_ns = wn["decode"]["logical_bytes"] / (per_ns["decode"] * 1e-3) / 1e9
    gb_sh = works["decode"]["logical_bytes"] / (per["decode"] * 1e-3) / 1e9
    return {"workload": "cfg5",
            "prefill": {"bound": "tensor", "kernel_ms": per["prefill"], "flops_per_launch": works["prefill"]["flops"],
                        "TFLOPs": tf, "frac_of_bf16_peak": tf / peaks["tensor"],
                        "occupancy": occ},
            "decode_noshare": {"bound": "hbm", "kernel_ms": per_ns["decode"], "bytes": wn["decode"]["logical_bytes"],
                               "GBps": gb_ns, "frac_of_hbm_peak": gb_ns / peaks["hbm"]},
            "decode_shared": {"kernel_ms": per["decode"], "logical_GBps": gb_sh,
                              "logical_over_hbm_peak": gb_sh / peaks["hbm"]},
            "mixed_step_ms": t_ms / steps, "mixed_attention_ms": a_ms / steps,
            "separate_kernels_sum_ms": per["prefill"] + per["decode"],
            # row a0 (HBM-bound, 2*Hkv*D*2 B read + the same written per token): the step's
            # lazy_cache_write launch = step time - attention time; a few MB, i.e. launch-latency-bound
            "cache_write": _cache_write_entry(job.batch if not own else None, job_timed_tokens, sh, fp8,
                                              (t_ms - a_ms) / steps)}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="cfg2", choices=["cfg2", "cfg3", "cfg4", "cfg5"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--noshare", action="store_true", help="every drawn document distinct (logical == unique bytes)")
    ap.add_argument("--kv-dtype", default="bf16", choices=["bf16", "fp8"],
                    help="fp8: LAZY_KV_FP8_E4M3 pages (SURVEY 8.0 row f4)")
    ap.add_argument("--no-secondary", action="store_true", help="skip the prefill (cfg3) and noshare side measurements")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--mixed", action="store_true",
                    help="cfg5: also time the step with lazy_attn_mixed (prefill and decode concurrently, f4)")
    ap.add_argument("--graph", action="store_true",
                    help="also replay the step from a CUDA graph (f4) and report its time next to the eager one")
    ap.add_argument("--e3", action="store_true",
                    help="also run the f1 / f2 ablation on the paper's own E3 shape: 1 request, 5 x 4,096-token documents + a "
                         "64-token query (PAPER.md L273), decode and the 64-row query prefill")
    ap.add_argument("--ablation", action="store_true",
                    help="also time the stored-position / absolute K layouts and the materialising re-encoding (f1/f2)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    peaks = load_peaks()

    if args.impl == "reference":
        if rank != 0:
            return
        batch = make_batch(args.workload, 0, args.noshare)
        work = step_work(batch, [s for s in batch.steps if s.kind != "write_only"][:2 if args.workload == "cfg5" else None])
        vals, secs = [], []
        sample = ""
        for i in range(args.warmup + args.steps):
            v, t, sample, cores = oracle_sample(args.workload, batch)
            if i >= args.warmup:
                vals.append(v); secs.append(t)
        metric, _, unit = headline(args.workload, work, 1.0)
        value = float(np.mean(vals))
        print(json.dumps({
            "impl": "reference", "metric": metric, "value": value, "unit": unit, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": float(np.mean(secs) * 1e3),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload + (" noshare" if args.noshare else ""), "batch": batch.name,
                       "note": "each step is a bounded sample of the workload"},
            "cpu_baseline": {"value": value, "unit": unit, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}))
        return

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local_rank)
    device = f"cuda:{local_rank}"
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(device))

    def barrier():
        if dist is not None:
            dist.barrier()

    def max_over_ranks(x: float) -> float:
        if dist is None:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    from paper_2606_04302_b200 import build as lazy_build
    if rank == 0:
        lazy_build.build()
    barrier()

    fp8 = args.kv_dtype == "fp8"
    batch = make_batch(args.workload, rank, args.noshare)
    job = GpuJob(batch, device, fp8=fp8)
    work = step_work(batch, [r["step"] for r in job.timed], fp8=fp8)
    sampler = ClockSampler(local_rank)
    sampler.start()
    total_ms, attn_ms, launches = job.time_steps(args.steps, args.warmup, barrier)
    # the timed region of a decode step is a few ms, shorter than nvidia-smi's start-up: keep replaying the same
    # step (untimed) under the sampler until it has seen the GPU under this load for >= 0.5 s
    t_end = time.perf_counter() + 0.5
    while time.perf_counter() < t_end or len(sampler.rows) < 5:
        for _ in range(20):
            job.flush_l2(); job.run()
        torch.cuda.synchronize()
        if time.perf_counter() > t_end + 5.0:
            break
    clocks = sampler.stop()
    clocks["window"] = "timed steps + >=0.5 s untimed replay of the same step"
    total_ms, attn_ms = max_over_ranks(total_ms), max_over_ranks(attn_ms)
    ms_step, ms_attn = total_ms / args.steps, attn_ms / args.steps
    job.prepare_e2e()
    e2e_ms = max_over_ranks(job.time_e2e(args.steps, args.warmup, barrier)) / args.steps
    job.prepare_e2e_unpacked()
    e2e_unpacked_ms = max_over_ranks(job.time_e2e(args.steps, args.warmup, barrier, run=job.run_e2e_unpacked)) / args.steps
    e2e_check = job.verify_e2e()

    metric, value1, unit = headline(args.workload, work, ms_step)
    _, e2e1, _ = headline(args.workload, work, e2e_ms)
    value, e2e_value = value1 * world, e2e1 * world           # whole-job aggregate (weak scaling: same work per rank)

    wl_name = args.workload + ("_noshare" if args.noshare else "")
    roof = None
    if args.workload in ("cfg2", "cfg4"):
        # The HBM roofline of the decode kernel is taken on the `noshare` variant of the workload (every drawn
        # document distinct: algorithmic bytes == distinct bytes == DRAM bytes).  On the Zipf-shared batch the L2
        # serves the repeated pages, so logical bytes / time can exceed the HBM peak: reported under "shared".
        ub = unique_bytes(batch, [r["step"] for r in job.timed])
        shared = {"kernel_ms": ms_attn, "logical_bytes_per_launch": work["logical_bytes"],
                  "logical_GBps": work["logical_bytes"] / (ms_attn * 1e-3) / 1e9,
                  "logical_over_hbm_peak": work["logical_bytes"] / (ms_attn * 1e-3) / 1e9 / peaks["hbm"],
                  "unique_bytes_per_launch": ub, "unique_GBps": ub / (ms_attn * 1e-3) / 1e9,
                  "traffic": ncu_traffic("decode", args.workload)}
        if args.noshare:
            ns = dict(kernel_ms=ms_attn, bytes=work["logical_bytes"])
        else:
            ns = decode_noshare_leg(args.workload, device, max(5, args.steps // 2), barrier, fp8=fp8)
        ach = ns["bytes"] / (ns["kernel_ms"] * 1e-3) / 1e9
        roof = {"bound": "hbm", "kernel": "lazy_attn_decode (split-KV + combine)", "achieved": ach,
                "peak": peaks["hbm"], "unit": "GB/s", "frac": ach / peaks["hbm"],
                "traffic": ncu_traffic("decode_fp8" if fp8 else "decode", args.workload + "_noshare"),
                "peak_source": peaks["source"],
                "workload": args.workload + " noshare (every drawn document distinct)",
                "algorithmic_bytes_per_launch": ns["bytes"], "kernel_ms": ns["kernel_ms"],
                "note": "frac on the noshare variant; value is logical bytes on the Zipf-shared batch and may exceed the "
                        "HBM peak"}
        if not args.noshare:
            roof["shared"] = shared
    elif args.workload == "cfg3":
        ach = work["flops"] / (ms_attn * 1e-3) / 1e12
        roof = {"bound": "tensor", "kernel": "lazy_attn_prefill", "achieved": ach, "peak": peaks["tensor"],
                "unit": "TFLOP/s", "frac": ach / peaks["tensor"], "traffic": ncu_traffic("prefill_fp8" if fp8 else "prefill", wl_name),
                "peak_source": peaks["source"] + " (burst: the kernel is timed alone, L2 flushed between launches)",
                "algorithmic_flops_per_launch": work["flops"], "kernel_ms": ms_attn}
    else:
        # mixed step: the dominant kernel by bytes is the decode kernel; both kernels are reported per call
        leg = cfg5_leg(device, max(5, args.steps // 2), peaks, job=job, fp8=fp8)
        d = leg["decode_noshare"]
        roof = {"bound": "hbm", "kernel": "lazy_attn_decode (split-KV + combine) of the mixed step",
                "achieved": d["GBps"], "peak": peaks["hbm"], "unit": "GB/s", "frac": d["frac_of_hbm_peak"],
                "traffic": ncu_traffic("decode_fp8" if fp8 else "decode", "cfg5_noshare"), "peak_source": peaks["source"],
                "workload": "cfg5 decode requests, noshare variant", "kernel_ms": d["kernel_ms"],
                "algorithmic_bytes_per_launch": d["bytes"], "step": leg}

    out = {
        "metric": metric, "value": value, "unit": unit, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "fp8_e4m3 KV pages, bf16 q/out" if fp8 else "bf16", "data": "synthetic",
        "config": {"workload": args.workload + (" noshare" if args.noshare else ""), "batch": batch.name,
                   "heads": [batch.shape.num_q_heads, batch.shape.num_kv_heads, batch.shape.head_dim],
                   "num_reqs": int(sum(len(r["step"].seq_lens) for r in job.timed)),
                   "distinct_docs": batch.meta.get("distinct_docs"), "l2": "flushed between timed steps (512 MB fill + 256 MB read sweep)",
                   "parallelism": f"request-parallel replicas x{world}, no data-path collective"},
        "tokens_per_s": {"decode_tokens": work["dec_tokens"] / (ms_step * 1e-3) * world,
                         "kv_tokens_attended": work["kv_tokens"] / (ms_step * 1e-3) * world,
                         "prefill_query_tokens": work["q_tokens"] / (ms_step * 1e-3) * world},
        "roofline": roof,
        "e2e": {"value": e2e_value, "unit": unit, "ms_per_step": e2e_ms,
                "h2d_bytes_per_step": int(sum(e["h2d"] for e in job.e2e)),
                "d2h_bytes_per_step": int(sum(e["d2h"] for e in job.e2e)),
                "api": "lazy_host_step_packed: one H2D copy of the packed inputs, the kernels, one D2H copy "
                       "(packing into the pinned block is the caller's and is not timed)",
                "unpacked": {"api": "lazy_host_step: seven H2D copies from separate pinned tensors", "ms_per_step": e2e_unpacked_ms,
                             "value": headline(args.workload, work, e2e_unpacked_ms)[1] * world},
                "verified": e2e_check},
        "gpu_launches": int(launches), "clocks": clocks,
    }
    if args.mixed and rank == 0 and world == 1 and args.workload == "cfg5":
        B, dev = job.B, job.dev
        rp = [r for r in job.timed if r["step"].kind == "prefill"][0]
        rd = [r for r in job.timed if r["step"].kind == "decode"][0]

        def mixed_step(sms):
            for rec in job.timed:
                B.lazy_cache_write(dev.handle, rec["k_new"], rec["v_new"], rec["slots"], dev.k_pool, dev.v_pool)
            B.lazy_attn_mixed(dev.handle, dev.k_pool, dev.v_pool, q_prefill=rp["q"], block_table_prefill=rp["bt"],
                              page_logical_pos_prefill=rp["pp"], seq_lens_prefill=rp["sl"], cu_q_lens=rp["cu"],
                              max_q_len=rp["max_q"], out_prefill=rp["out"], q_decode=rd["q"], block_table_decode=rd["bt"],
                              page_logical_pos_decode=rd["pp"], seq_lens_decode=rd["sl"], out_decode=rd["out"],
                              decode_sms=sms)
        res = {}
        for sms in (0, 64, 96, 128):
            for _ in range(3):
                job.flush_l2(); mixed_step(sms)
            evs = []
            for _ in range(args.steps):
                job.flush_l2()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(); mixed_step(sms); e1.record()
                evs.append((e0, e1))
            torch.cuda.synchronize()
            res[f"decode_sms_{sms if sms else 'default'}"] = float(np.mean([a.elapsed_time(b) for a, b in evs]))
        job.separate_calls = True
        sep_total, _, _ = job.time_steps(args.steps, 3, barrier)
        job.separate_calls = False
        out["mixed"] = {"ms_per_step": res, "separate_calls_ms_per_step": sep_total / args.steps}
    if args.graph and rank == 0 and world == 1:
        g = torch.cuda.CUDAGraph()
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            job.run()
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        with torch.cuda.graph(g):
            job.run()
        evs = []
        for i in range(args.warmup + args.steps):
            job.flush_l2()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); g.replay(); e1.record()
            if i >= args.warmup:
                evs.append((e0, e1))
        torch.cuda.synchronize()
        g_ms = float(np.mean([a.elapsed_time(b) for a, b in evs]))
        out["graph"] = {"ms_per_step": g_ms, "eager_ms_per_step": ms_step,
                        "launches_per_step": int(launches) // max(1, args.steps)}
    default_abl = args.workload == "cfg2" and not args.no_secondary and not fp8 and not args.noshare
    if (args.ablation or default_abl) and rank == 0 and world == 1 and args.workload != "cfg5":
        # rows f1 / f2 (Fig. 5): in the default command a cut-down run on cfg2
        abl = run_ablation(job, max(5, args.steps) if args.ablation else 10, 3)
        abl["lazy_shared_ms"] = ms_attn
        abl["materialise_then_attend_ms"] = abl["materialize_ms"] + abl["absolute_ms"]
        abl["lazy_speedup_vs_materialising"] = abl["materialise_then_attend_ms"] / ms_attn
        out["ablation"] = abl
    job.dev.close()
    del job
    torch.cuda.empty_cache()

    if rank == 0 and world == 1 and not args.no_secondary and args.workload == "cfg2" and not fp8:
        # side measurements in the same run, so that the driver's record carries all five configs: the prefill headline
        # (configs[2]) as a burst and as a seconds-long run, the long-context decode (configs[3]) and the mixed step
        # (configs[4]) kernel by kernel.  configs[0] is the parity-test case.
        side = {}
        for name, fn in (("cfg3", lambda: prefill_leg("cfg3", device, max(5, args.steps // 3), peaks, barrier)),
                         ("cfg4", lambda: decode_leg("cfg4", device, max(5, args.steps // 2), peaks, barrier)),
                         ("cfg5", lambda: cfg5_leg(device, max(5, args.steps // 2), peaks)),
                         ("fp8_pages", lambda: fp8_leg(device, max(5, args.steps // 2), peaks, barrier))):
            try:
                side[name] = fn()
            except Exception as e:  # a side measurement must not lose the headline
                side[name] = {"error": repr(e)}
            torch.cuda.empty_cache()
        out["configs"] = side

    if args.e3 and rank == 0 and world == 1:
        # PAPER.md L271-297 (Fig. 5): the rotation's overhead on the paper's own ablation shape, next to its +0.13 %
        from paper_2606_04302_b200 import workloads as W
        e3 = {}
        for name, dec in (("decode", True), ("prefill_64_rows", False)):
            b3 = W.e3_paper(decode=dec)
            j3 = GpuJob(b3, device)
            _, a3, _ = j3.time_steps(20, 3, barrier)
            ab3 = run_ablation(j3, 20, 3)
            e3[name] = {"seq_len": int(j3.timed[-1]["step"].seq_lens[0]), "lazy_ms": a3 / 20,
                        **{k: ab3[k] for k in ("unrotated_ms", "stored_pos_ms", "absolute_ms", "rotation_overhead_pct",
                                               "stored_pos_overhead_pct", "materialize_ms")}}
            j3.dev.close()
            del j3, b3
            torch.cuda.empty_cache()
        out["e3"] = e3

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, t, sample, cores = oracle_sample(args.workload, batch)
        out["cpu_baseline"] = {"value": v, "unit": unit, "cores": cores, "kind": "oracle", "sample": sample,
                               "seconds": t}
    if rank == 0:
        sys.stderr.write("detail: " + json.dumps(out) + "\n")          # the verbose record (prose, byte counts)
        print(json.dumps(compact_line(out)))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

"""bench.py's stdout contract (host logic, no GPU): the one JSON line stays under the driver's 3 KB tail, carries the
contract's keys, and ENDS with the flat `summary` holding both halves of BASELINE.json's metric.  The input is a verbose
record (`detail: {...}` on stderr) of a real default run of this round on a B200, stored as a text fixture under tests/data/ (a FORMAT sample: no parity test reads it; tests/golden/ holds only the
paper-derived values)."""
import importlib.util
import json
import os

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _bench():
    spec = importlib.util.spec_from_file_location("bench_module", os.path.join(ROOT, "bench.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def test_default_line_fits_the_tail_and_ends_with_the_summary():
    detail = json.load(open(os.path.join(ROOT, "tests", "data", "bench_detail_sample.json")))
    detail["cpu_baseline"] = {"value": 1.2, "unit": "GB/s", "cores": 16, "kind": "oracle",
                              "sample": "decode: first 64 of 64 requests", "seconds": 0.56}
    line = _bench().compact_line(detail)
    text = json.dumps(line)
    assert len(text) < 3072, len(text)
    assert list(line)[-1] == "summary"
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "roofline", "e2e", "gpu_launches", "clocks", "cpu_baseline"):
        assert k in line, k
    assert line["config"]["workload"] == "cfg2"
    for k in ("bound", "achieved", "peak", "unit", "frac", "traffic", "note"):
        assert k in line["roofline"], k
    assert abs(line["roofline"]["frac"] - line["roofline"]["achieved"] / line["roofline"]["peak"]) < 1e-3
    for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "verified", "lazy_host_step_ms"):
        assert k in line["e2e"], k
    for k in ("cpu_baseline",):
        assert {"value", "unit", "cores", "kind", "sample"} <= set(line[k])
    sm = line["summary"]
    for k in ("cfg2_roofline_frac", "cfg3_TFLOPs", "cfg3_frac_burst", "cfg3_frac_sustained", "cfg3_sm_mhz",
              "cfg4_noshare_frac", "cfg5_decode_noshare_frac", "cfg5_prefill_frac", "cfg5_mixed_attention_ms",
              "fp8_cfg2_frac", "fp8_cfg4_frac", "rotation_overhead_pct", "materialize_ms", "lazy_speedup_vs_materialising"):
        assert k in sm and isinstance(sm[k], (int, float)), k
    assert all(not isinstance(v, (dict, list)) for v in sm.values())          # flat

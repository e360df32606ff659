"""bench.py's contract, checked without a GPU: tests/bench_dryrun.py runs main() with CUDA and the kernels stubbed; the one
JSON line it prints must carry every key the harness reads, and the fall-back paths (fused host call raising or missing
parity, a config whose backward no kernel holds) must still end in a complete line."""
import json
import os
import subprocess
import sys

import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


def dryrun(bad=None):
    env = dict(os.environ)
    env.pop("BAD", None)
    if bad:
        env["BAD"] = bad
    p = subprocess.run([sys.executable, os.path.join(HERE, "bench_dryrun.py")], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True,
                       env=env, timeout=900)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [l for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, "bench.py must print ONE JSON line"
    return json.loads(lines[0])


@pytest.mark.parametrize("bad", [None, "raise", "parity"])
def test_bench_line_is_complete(bad):
    d = dryrun(bad)
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "gpu_launches", "clocks", "parity", "others"):
        assert k in d, k
    assert d["config"]["workload"] == "cfg5_1k" and "model" not in d["config"] and d["vs_baseline"] is None and d["scaling"] == "weak"
    assert {"bound", "achieved", "peak", "unit", "frac", "traffic"} <= set(d["roofline"]) and d["roofline"]["bound"] == "hbm"
    assert abs(d["roofline"]["frac"] - d["roofline"]["achieved"] / d["roofline"]["peak"]) < 1e-12
    assert {"value", "unit", "cores", "kind", "sample"} <= set(d["cpu_baseline"]) and d["cpu_baseline"]["kind"] == "oracle"
    assert {"value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"} <= set(d["e2e"]) and d["e2e"]["h2d_bytes_per_step"] > 0
    assert d["gpu_launches"] > 0 and {"sm_mhz", "sm_max_mhz", "reasons"} <= set(d["clocks"])
    assert d["parity"]["fwd_ok"] and d["parity"]["bwd_ok"]
    o = d["others"]
    assert "error" not in o, o.get("error")
    assert all(f"table1:16x8x{L}x{L}:bf16:fwd" in o for L in (256, 512, 1024)) and "line_bwd_child" in o
    assert all(f"{c}:fwd" in o for c in ("cfg1_tiny:f32", "cfg2_cls56:f32", "cfg2_cls56:bf16", "cfg3_enc378:bf16", "cfg4_2k:bf16"))
    if bad is None:
        assert d["e2e"]["api"] == "gspn_scan_fwd_bwd_host" and d["e2e"]["parity"] == {"fwd_ok": True, "bwd_ok": True}
        assert o["cfg4_2k:bf16:bwd"]["variant"] is not None
    else:       # the fused call is dropped, the two-call path measured instead, and the reason is in the line
        assert d["e2e"]["api"].startswith("gspn_scan_fwd_host") and "fused_call" in d["e2e"]
        assert o["cfg4_2k:bf16:bwd"]["variant"] is None and "error" in o["cfg4_2k:bf16:bwd"]

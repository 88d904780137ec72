"""The bench.py contract on a GPU box: one JSON line on stdout with the keys the driver reads (metric, value,
unit, n_gpus, steps, warmup, ms_per_step, higher_is_better, scaling, vs_baseline, dtype, data, config.workload,
roofline, e2e, gpu_launches, clocks, cpu_baseline), on the small config so that it runs in seconds."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_bench_prints_one_contract_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--config", "c1", "--steps", "20", "--warmup", "3"],
                       cwd=ROOT, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [x for x in r.stdout.splitlines() if x.strip()]
    assert len(lines) == 1, lines[:3]
    d = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "roofline", "e2e", "gpu_launches", "clocks", "cpu_baseline"):
        assert k in d, k
    assert d["n_gpus"] == 1 and d["steps"] == 20 and d["warmup"] == 3 and d["higher_is_better"] is False
    assert d["unit"] == "us/session" and d["value"] > 0 and d["vs_baseline"] is None and d["data"] == "synthetic"
    assert "workload" in d["config"] and "model" not in d["config"]
    for k in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
        assert k in d["roofline"], k
    assert d["roofline"]["bound"] in ("hbm", "tensor", "alu")
    assert d["gpu_launches"] == 4 * d["steps"]          # invalidate, entry_attn, ready_dist, gate_serve per step
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > d["value"]
    assert d["clocks"]["sm_max_mhz"] >= d["clocks"]["sm_mhz"] > 0


def _strict_loads(text):
    def bad(c):
        raise ValueError(f"non-standard JSON constant {c}")
    return json.loads(text, parse_constant=bad)


def test_default_invocation_prints_one_small_strict_line():
    """What the driver runs: no --config, --steps 20 --warmup 5.  All five configs run, but stdout is ONE line of a
    few KB holding the headline (configs[4]) contract fields; everything else goes to gpurun_out/bench_detail.json.
    (Round 2's 24 KB line with every config nested in it was not parsed by the driver.)"""
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "20", "--warmup", "5"],
                       cwd=ROOT, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [x for x in r.stdout.splitlines() if x.strip()]
    assert len(lines) == 1, [x[:80] for x in lines[:3]]
    assert len(lines[0]) < 4096, len(lines[0])
    d = _strict_loads(lines[0])
    assert d["steps"] == 20 and d["warmup"] == 5 and d["n_gpus"] == 1
    assert d["config"]["workload"].startswith("configs[4]")
    assert d["value"] > 0 and d["unit"] == "us/session" and d["higher_is_better"] is False
    # one session per step: us/session is the step time, so steps x ms_per_step is the headline's timed region
    assert abs(d["value"] - d["ms_per_step"] * 1e3) <= 1e-6 * d["value"]
    for k in ("roofline", "cpu_baseline", "e2e", "clocks", "gpu_launches", "kernels", "gate_serve"):
        assert k in d, k
    assert d["roofline"]["frac"] > 0 and d["e2e"]["value"] > 0 and d["e2e"]["h2d_bytes_per_step"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["gpu_launches"] == 4 * d["steps"]
    assert sorted(d["other_configs"]) == ["c1", "c2", "c3", "c4"]
    detail = _strict_loads(open(os.path.join(ROOT, d["detail"])).read())
    assert detail["headline"] == "c5" and sorted(detail["configs"]) == ["c1", "c2", "c3", "c4", "c5"]
    assert detail["configs"]["c5"]["value"] == d["value"]

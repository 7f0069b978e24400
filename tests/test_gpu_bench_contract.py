"""The bench.py contract on a GPU box: one JSON line with the keys the driver reads, for our arm and for the reference arm
(the oracle), on the small config (cfg1) so that the test takes seconds.  Values are checked for sanity only; the numbers
that matter are the driver's own runs."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*args):
    env = dict(os.environ)
    env.pop("QSL_LIB_PATH", None)
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, cwd=ROOT, env=env,
                       timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, lines                                  # ONE JSON line on stdout
    return json.loads(lines[0])


def test_bench_line_of_our_arm():
    d = _run("--gpus", "1", "--steps", "3", "--warmup", "3", "--workload", "cfg1", "--no-per-config")
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert k in d, k
    assert d["n_gpus"] == 1 and d["steps"] == 3 and d["warmup"] == 3 and d["higher_is_better"] is True
    assert d["vs_baseline"] is None and d["data"] == "synthetic" and d["dtype"] == "f64" and d["scaling"] == "weak"
    assert d["config"]["workload"].startswith("cfg1") and "model" not in d["config"] and "l2" in d["config"]
    assert d["value"] > 0 and abs(d["value"] - d["lines_per_step"] / (d["ms_per_step"] * 1e-3)) <= 1e-6 * d["value"]
    assert d["gpu_launches"] > 0                                   # the CUDA path ran
    e = d["e2e"]
    assert e["unit"] == d["unit"] and 0 < e["value"] < d["value"] and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0
    r = d["roofline"]
    assert r["bound"] in ("alu", "hbm", "tensor") and r["peak"] > 0 and r["achieved"] > 0
    assert abs(r["frac"] - r["achieved"] / r["peak"]) <= 1e-9 and 0 < r["frac"] < 1 and "traffic" in r
    assert all(0 < v["frac"] < 1.05 and v["ms"] > 0 for v in r["streaming"]["kernels"].values())
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["unit"] == d["unit"] and c["sample"]
    assert c["parity"]["pass"] is True                             # the timed GPU pass against the oracle, north_star gates
    k = d["clocks"]
    assert k["sm_mhz"] > 0 and k["sm_max_mhz"] >= k["sm_mhz"] and isinstance(k["reasons"], list)


def test_bench_line_of_the_reference_arm():
    d = _run("--impl", "reference", "--gpus", "1", "--steps", "1", "--warmup", "0", "--workload", "cfg1")
    assert d["impl"] == "reference" and d["gpu_launches"] == 0 and d["higher_is_better"] is True
    assert d["metric"] == "field lines/s (with Q)" and d["unit"] == "lines/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"] and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["config"]["workload"].startswith("cfg1")

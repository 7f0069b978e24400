"""the oracle built with -fsanitize=address,undefined runs a small pass of every entry point
(pack, evaluate in all three interpolation orders, trace in both geometries and with every stepper, FLEDGE dense and
sparse, select, refine) without a report.  Runs in a subprocess because the sanitizer runtime must be preloaded."""
import os
import subprocess
import sys

import oracle

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SCRIPT = r"""
import numpy as np
import oracle, qsl_inputs as qi
from tests.parity import oracle_pipeline
assert oracle.lib()._name.endswith("libqsl_oracle_san.so")
cfg = qi.make_config("cfg3", scale=1 / 32)
cfg["levels"] = 2
ref = oracle_pipeline(cfg)                                   # trace L, FLEDGE dense + sparse, select, refine, trace LQ
assert len(ref["coords"]) == 3 and np.isfinite(ref["tau"])
g = qi.Grid.uniform((7, 6, 8), (0, 0, 0), (1, 1, 1))
rng = np.random.default_rng(0)
B = [rng.normal(size=g.shape) for _ in range(3)]
seeds = rng.uniform(0.02, 0.98, size=(40, 3))
for order in (oracle.TRILINEAR, oracle.TRIQUADRATIC, oracle.TRICUBIC):
    F = oracle.Field(g, B, oracle.F64, oracle.NORMALIZE_FIRST, order)
    for x in ([0.001, 0.999, 0.5], [-0.01, 1.01, 0.3]):     # boundary cells and a point outside the grid
        F.evaluate(np.array(x))
    oracle.trace(F, seeds, g.lo, g.hi, max_steps=300)
F = oracle.Field(g, B, oracle.F32, oracle.INTERP_FIRST)
for method in (oracle.RK4, oracle.EULER, oracle.CK45):
    oracle.trace(F, seeds, g.lo, g.hi, method=method, max_steps=300, want_dev=True)
gs = qi.Grid.uniform((9, 11, 17), (0.1, -0.3, 1.0), (0.9, 0.5, 2.0))
Fs = oracle.Field(gs, [np.zeros(gs.shape), np.zeros(gs.shape), np.ones(gs.shape)], oracle.F64, oracle.NORMALIZE_FIRST,
                  oracle.TRILINEAR, oracle.SPHERICAL)
o = oracle.trace(Fs, np.array([[0.3, 0.1, 1.5]]), gs.lo, gs.hi, method=oracle.CK45)
assert abs(o["L"][0] - 1.0) < 1e-12
print("sanitized oracle ok")
"""


def test_oracle_runs_clean_under_asan_and_ubsan():
    oracle.build(sanitize=True)
    env = dict(os.environ, QSL_ORACLE_SANITIZE="1", LD_PRELOAD=oracle.sanitizer_runtime(), PYTHONPATH=ROOT,
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1", UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1",
               OMP_NUM_THREADS="2")
    r = subprocess.run([sys.executable, "-c", SCRIPT], cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and "sanitized oracle ok" in r.stdout, (r.stdout[-2000:], r.stderr[-4000:])
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, r.stderr[-4000:]

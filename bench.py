#!/usr/bin/env python
"""bench.py -- field lines/s (with Q) and RK steps/s of the libqsl hot path on B200, with its roofline fraction.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4] [--impl reference]

A "step" is one pass of the whole hot path over one batch of synthetic input: seed ordering, the persistent trace
kernel (a3-a5), the Q/L epilogue (a6) and, for the refinement workloads cfg3 / cfg5, FLEDGE, threshold, compaction and
the level loop (a7-a9).  The default workload is BASELINE.json configs[3] (cfg4: LFFF, fp32-sampled 256^3 field, 256^3
seeds, L + Q) - the largest single-trace "with Q" config and one of the 3-D configs north_star states its roofline target
on; `per_config` carries all five configs in the same line; DESIGN.md "Measurement" states what every key means.

`value`   lines/s with the seeds and the packed field already resident in HBM (CUDA events on the launch stream).
`e2e`     the same through the public binding with HOST buffers: pinned seeds -> device, trace, results -> pinned host.
`roofline` the trace kernel against the FP64 (or FP32) pipe peak measured on this device by qsl_peak_fma.
`roofline.streaming` GB/s of the HBM-streaming stages (FLEDGE, select, refine, sort, field pack) against the measured copy peak.
`per_config` lines/s, RK steps/s, ms and roofline fraction of each of the five BASELINE.json configs (N = 1 only).
`cpu_baseline` the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload (every
          seed for cfg1-3, every 4th seed per axis + two 32^3 tiles for cfg4/5), timed AND compared with the GPU's
          outputs of the timed run at the north_star gates; rank 0, N = 1 only.
`--impl reference` times only that oracle (the reference arm of the contract).

Under torchrun every rank traces its own replica of the workload (lines are independent: weak scaling, no data-path
collective); the time is the max over ranks and `value` the lines all ranks traced divided by it.
"""
from __future__ import annotations

import argparse
import contextlib
import json
import math
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# Algorithmic FP-pipe work per accepted RK4 step of one line:
# pipe instructions (an FMA, add or multiply each occupies one issue slot) and true flops (FMA = 2).
PIPE_SLOTS_PER_STEP = {"LQ": 490, "L": 245}
FLOPS_PER_STEP = {"LQ": 800, "L": 400}
# Figures of one trace-kernel launch taken from the committed `ncu --set full` captures (profiles/): dram_bytes =
# dram__bytes_read.sum + dram__bytes_write.sum, pipe_active = sm__pipe_fp64_cycles_active (sm__pipe_fma_cycles_active for
# fp32 arithmetic) as a fraction of peak.  Keyed by (workload, arithmetic); absent -> null in the bench line.
NCU_CAPTURES = {
    ("cfg2", "f64"): {"dram_bytes": 786209280, "pipe_active": 0.620, "source": "profiles/r2d_cfg4_trace_kernel.md (cfg2 capture)"},
    ("cfg4", "f64"): {"dram_bytes": 47756282000, "pipe_active": 0.649, "source": "profiles/r2f_final_build_cfg4.md"},
    ("cfg5", "f64"): {"dram_bytes": 626591608000, "pipe_active": 0.525,
                      "source": "profiles/r2d_cfg4_trace_kernel.md (cfg5 level 0, the L-only launch)"},
}
DEFAULT_WORKLOAD = "cfg4"
SELECT_PASSES = 3          # passes of qsl_select that read the whole map (select_refine.cu: passes 0 - 2; passes 3 - 7 read the
                           # candidates kept by pass 2, a few per cent of the map), for the streaming byte count
SORT_PASSES = 4            # radix passes of the 30-bit seed sort (order.cu)


def _env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


class ClockSampler:
    """Samples SM clock and clock-event reasons of one GPU during the timed region (NVML, every 100 ms)."""

    BAD = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown"}
    NOTE = {0x4: "sw_power_cap", 0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting"}

    def __init__(self, index):
        self.samples, self.reasons, self.max_mhz, self._stop, self._t = [], set(), None, threading.Event(), None
        # held by the timing loop while it ENQUEUES a pass (a fraction of a millisecond; the pass then runs for its full
        # duration with the sampler free): an NVML query takes driver locks that can stall a kernel launch for tens of
        # milliseconds, which would show up as idle GPU time inside the event pair of that pass
        self.enqueue_lock = threading.Lock()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv, self.h = pynvml, pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _sample(self):
        nv = self.nv
        try:
            with self.enqueue_lock:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
            for bit, name in {**self.BAD, **self.NOTE}.items():
                if r & bit:
                    self.reasons.add(name)
        except Exception:
            pass

    def _loop(self):
        while not self._stop.is_set():
            self._sample()
            self._stop.wait(0.1)

    def __enter__(self):
        if self.nv is not None:
            self._t = threading.Thread(target=self._loop, daemon=True)
            self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._t is not None:
            self._t.join(timeout=2)
            # a timed region shorter than the sampling period (cfg1: 2 ms) can end before the first sample: take one now,
            # right behind the last timed kernel (`at_end` in the summary says so)
            self.at_end = not self.samples
            if self.at_end:
                self._sample()

    def summary(self):
        s = sorted(self.samples)
        out = {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
               "samples": len(s)}
        if getattr(self, "at_end", False):
            out["at_end"] = True
        return out


# ---------------------------------------------------------------------------------------------------------------------
def oracle_sample_indices(cfg):
    """SURVEY.md 8(d) "Oracle timing": cfg1-3 the full level-0 seed set; cfg4 / cfg5 every 4th seed per axis (1/64) plus
    two full 32^3 tiles of the seed lattice.  Returns (indices into the level-0 seeds, description)."""
    n = len(cfg["seeds"])
    lat = cfg["lattice"]
    if cfg["name"] in ("cfg1", "cfg2", "cfg3") or int(lat.ndim) != 3 or min(int(v) for v in lat.n) < 96:
        return np.arange(n), "all %d level-0 seeds of %s" % (n, cfg["name"])
    n0, n1, n2 = (int(v) for v in lat.n)
    k, j, i = np.meshgrid(np.arange(0, n2, 4), np.arange(0, n1, 4), np.arange(0, n0, 4), indexing="ij")
    sub = ((k * n1 + j) * n0 + i).reshape(-1)
    tiles = []
    for (o0, o1, o2) in ((n0 // 4, n1 // 4, n2 // 4), (n0 - 64, n1 // 2, n2 // 2 - 16)):
        k, j, i = np.meshgrid(np.arange(o2, o2 + 32), np.arange(o1, o1 + 32), np.arange(o0, o0 + 32), indexing="ij")
        tiles.append(((k * n1 + j) * n0 + i).reshape(-1))
    idx = np.unique(np.concatenate([sub] + tiles))
    return idx, "every 4th level-0 seed per axis + two 32^3 tiles of %s (%d of %d lines)" % (cfg["name"], len(idx), n)


def parity_report(g, c, box_lo, box_hi, with_q):
    """The north_star gates on the sampled lines: end points <= 1e-9 x box, L and Q <= 1e-8 relative (fractions of the
    sample within the gate), max |delta log10 Q| over Q < 1e8."""
    box = float(np.max(np.asarray(box_hi) - np.asarray(box_lo)))
    rep = {"n": int(len(c["L"]))}
    rl = np.abs(g["L"] - c["L"]) / np.maximum(np.abs(c["L"]), 1e-300)
    rl = np.where(g["L"] == c["L"], 0.0, rl)
    rep["L_within_1e-8"] = float((rl <= 1e-8).mean())
    if "end_f" in g:
        e = np.maximum(np.abs(g["end_f"] - c["end_f"]).max(1), np.abs(g["end_b"] - c["end_b"]).max(1))
        rep["end_within_1e-9_box"] = float((e <= 1e-9 * box).mean())
    if with_q:
        for key in ("q_perp", "q_bnd"):
            qc, qg = c[key], g[key]
            fin = np.isfinite(qc) & np.isfinite(qg)
            rq = np.abs(qg[fin] - qc[fin]) / np.abs(qc[fin])
            rep[key + "_within_1e-8"] = float((rq <= 1e-8).mean()) if fin.any() else 1.0
            small = fin & (np.abs(qc) < 1e8) & (qc > 0) & (qg > 0)
            rep[key + "_dlog10_max"] = float(np.abs(np.log10(qg[small]) - np.log10(qc[small])).max()) if small.any() else 0.0
    rep["gates"] = "north_star: >= 0.999 of the lines within each gate, dlog10 Q <= 1e-3 for every line with Q < 1e8"
    rep["pass"] = bool(all(v >= 0.999 for k, v in rep.items() if "within" in k)
                       and all(v <= 1e-3 for k, v in rep.items() if k.endswith("dlog10_max")))
    return rep


def oracle_leg(cfg, gpu_last, torch):
    """Times the CPU oracle on the sample of SURVEY.md 8(d) and compares it with the outputs of the GPU's last timed pass
    on the same seeds.  If a pilot run says the prescribed sample would take more than ~40 s on this host, every k-th
    seed of it is used instead (and the description says so)."""
    import oracle
    st = oracle.F32 if cfg["sample_type"] == "f32" else oracle.F64
    f = oracle.Field(cfg["grid"], cfg["B"], st, oracle.NORMALIZE_FIRST)
    mode = cfg["mode"]
    kw = dict(step_frac=cfg["step_frac"], mode=mode, max_steps=cfg["max_steps"], null_eps=cfg["null_eps"])
    cores = os.cpu_count() or 1
    idx, desc = oracle_sample_indices(cfg)
    seeds = cfg["seeds"]
    pilot = idx[:: max(1, len(idx) // 4096)]
    t0 = time.perf_counter()
    oracle.trace(f, np.ascontiguousarray(seeds[pilot]), cfg["box_lo"], cfg["box_hi"], **kw)
    est = (time.perf_counter() - t0) * len(idx) / len(pilot)
    if est > 40.0:
        k = int(math.ceil(est / 30.0))
        idx = idx[::k]
        desc = "every %d-th line of: %s (%d lines; the full sample would take %.0f s on %d cores)" % (k, desc, len(idx), est, cores)
    s = np.ascontiguousarray(seeds[idx])
    t0 = time.perf_counter()
    o = oracle.trace(f, s, cfg["box_lo"], cfg["box_hi"], **kw)
    dt = time.perf_counter() - t0
    steps = int(o["total_steps"])
    cpu = {"value": len(idx) / dt, "unit": "lines/s", "cores": cores, "kind": "oracle",
           "sample": "%s; %d RK4 steps, %.1f s wall, OpenMP over lines, mode %s" % (desc, steps, dt, "L+Q" if mode == 1 else "L"),
           "rk_steps_per_s": steps / dt}
    if gpu_last is not None:
        ti = torch.from_numpy(idx).cuda()
        g = {k: v[ti].cpu().numpy() for k, v in gpu_last.items() if k in ("end_f", "end_b", "L", "q_perp", "q_bnd")}
        cpu["parity"] = parity_report(g, o, cfg["box_lo"], cfg["box_hi"], mode == 1)
    return cpu


def run_reference(args, cfg):
    """--impl reference: the oracle, as it stands, on the host cores; each step a bounded sample of the workload."""
    import oracle
    st = oracle.F32 if cfg["sample_type"] == "f32" else oracle.F64
    f = oracle.Field(cfg["grid"], cfg["B"], st, oracle.NORMALIZE_FIRST)
    seeds = cfg["seeds"]
    n = len(seeds)
    kw = dict(step_frac=cfg["step_frac"], mode=cfg["mode"], max_steps=cfg["max_steps"], null_eps=cfg["null_eps"])
    # size the per-step sample from a pilot so that warmup + steps finish in about two minutes
    pilot = np.ascontiguousarray(seeds[::max(1, n // 2048)])
    t0 = time.perf_counter()
    oracle.trace(f, pilot, cfg["box_lo"], cfg["box_hi"], **kw)
    rate = len(pilot) / max(time.perf_counter() - t0, 1e-6)
    budget = 120.0 / max(1, args.steps + args.warmup)
    stride = max(1, int(math.ceil(n / max(rate * budget, 1.0))))
    sample = np.ascontiguousarray(seeds[::stride])
    for _ in range(args.warmup):
        oracle.trace(f, sample, cfg["box_lo"], cfg["box_hi"], **kw)
    t0 = time.perf_counter()
    steps = 0
    for _ in range(args.steps):
        steps += int(oracle.trace(f, sample, cfg["box_lo"], cfg["box_hi"], **kw)["total_steps"])
    dt = time.perf_counter() - t0
    lines_s = len(sample) * args.steps / dt
    cores = os.cpu_count() or 1
    desc = "every %d-th level-0 seed of %s per step (%d lines/step), OpenMP over lines" % (stride, cfg["name"], len(sample))
    line = {
        "impl": "reference", "metric": "field lines/s (with Q)", "value": lines_s, "unit": "lines/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(cfg, args, sample=desc),
        "rk_steps_per_s": steps / dt,
        "cpu_baseline": {"value": lines_s, "unit": "lines/s", "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": lines_s, "unit": "lines/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_config(cfg, args, **extra):
    g = cfg["grid"]
    lat = cfg["lattice"]
    c = {"workload": "%s: %s" % (cfg["name"], WORKLOADS[cfg["name"]]),
         "field_grid": [g.nx, g.ny, g.nz], "field_samples": cfg["sample_type"],
         "seed_lattice": [int(v) for v in lat.n], "n_seeds": int(len(cfg["seeds"])),
         "trace_mode": "L+Q" if cfg["mode"] == 1 else "L", "refine_levels": int(cfg["levels"]),
         "step_rule": "RK4, h = 0.25 x smallest cell edge", "parallelism": "replicas x%d" % args.gpus,
         "interpolation": {1: "trilinear", 2: "triquadratic (Dodgson)", 3: "tricubic (Keys)"}[int(getattr(args, "interp_order", 1))],
         "l2": "flushed between timed steps (256 MiB write)"}
    if int(cfg["levels"]) > 0:
        c["refine"] = ("hilbert: length jump > %g between successive samples along the Hilbert curve, %d passes + shifted "
                       "curve (shift %d)" % (args.hilbert_thr, int(lat.ndim) * int(cfg["levels"]), args.hilbert_shift)
                       if getattr(args, "refine", "fledge") == "hilbert" else "fledge: FLEDGE > 95th percentile, 2x cells per level")
    c.update(extra)
    return c


WORKLOADS = {
    "cfg1": "BASELINE.json configs[0], hyperbolic field fp64 64^3, 128^2 seeds, L+Q",
    "cfg2": "BASELINE.json configs[1], quadrupole fp64 128^3, 1024^2 photospheric seeds (|Bz|>1e-3), L+Q",
    "cfg3": "BASELINE.json configs[2], quadrupole fp64 128^3, 2048x1024 vertical slice, FLEDGE + 4 refinement levels",
    "cfg4": "BASELINE.json configs[3], LFFF fp32 samples 256^3, 256^3 seeds, L+Q",
    "cfg5": "BASELINE.json configs[4], quadrupole+LFFF fp32 samples 512x512x256, 3-D FLEDGE + 3 refinement levels",
}


# ---------------------------------------------------------------------------------------------------------------------
class Workload:
    """One BASELINE.json config resident on the device: packed field, seeds (device + pinned host), trace parameters and
    the three ways bench.py runs it (device-resident step, end-to-end step through host buffers)."""

    def __init__(self, qsl, torch, name, args):
        import qsl_inputs as qi
        self.qsl, self.torch, self.args, self.name = qsl, torch, args, name
        cfg = self.cfg = qi.make_config(name, args.scale)
        g = cfg["grid"]
        dev = [torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64).reshape(-1)).cuda() for a in cfg["B"]]
        st = qsl.QSL_F32 if cfg["sample_type"] == "f32" else qsl.QSL_F64
        self.f32 = args.arith == "f32" and cfg["sample_type"] == "f32"
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        self.order = int(getattr(args, "interp_order", 1))
        self.field = qsl.qsl_field_create(g.nx, g.ny, g.nz, *dev, lo=g.lo, hi=g.hi, sample_type=st,
                                          layout=qsl.QSL_LAYOUT_CELL_TABLE_F32 if self.f32 else qsl.QSL_LAYOUT_CELL_TABLE,
                                          interp_order=0 if self.order == 1 else self.order)
        ev1.record(); ev1.synchronize()
        self.field_create_ms = ev0.elapsed_time(ev1)
        del dev
        self.seeds_host = torch.from_numpy(np.ascontiguousarray(cfg["seeds"])).pin_memory()
        self.n = int(self.seeds_host.shape[0])
        self.seeds = self.seeds_host.cuda()
        self.mode, self.levels, self.lat = cfg["mode"], int(cfg["levels"]), cfg["lattice"]
        mk = lambda m: qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], mode=m, step_frac=cfg["step_frac"],
                                             max_steps=cfg["max_steps"], null_eps=cfg["null_eps"], flags=args.flags,
                                             arith=qsl.QSL_ARITH_F32 if self.f32 else qsl.QSL_ARITH_F64)
        self.pL, self.pLQ = mk(qsl.QSL_TRACE_L), mk(qsl.QSL_TRACE_LQ)
        # samples handed out by hilbert_map are already ordered along a space-filling curve: no Morton sort inside qsl_trace
        args_flags = args.flags
        mkn = lambda m: qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], mode=m, step_frac=cfg["step_frac"],
                                              max_steps=cfg["max_steps"], null_eps=cfg["null_eps"],
                                              flags=args_flags | qsl.QSL_FLAG_NO_SORT,
                                              arith=qsl.QSL_ARITH_F32 if self.f32 else qsl.QSL_ARITH_F64)
        self.pL_curve, self.pLQ_curve = mkn(qsl.QSL_TRACE_L), mkn(qsl.QSL_TRACE_LQ)
        self.outs = ("end_f", "end_b", "L", "q_perp", "q_bnd", "face_f", "face_b", "status")
        self.out_bufs, self.host_out, self.host_res, self.hstate = {}, {}, {}, {}
        self.tot = torch.zeros(1, dtype=torch.int64, device="cuda")
        self.hilbert = args.refine == "hilbert" and self.levels > 0
        self.last = None                          # products of the last device-resident step (parity of the oracle leg)

    def close(self):
        self.field.destroy()
        self.out_bufs = self.host_out = self.host_res = self.hstate = self.last = None
        self.seeds = self.seeds_host = None
        self.torch.cuda.empty_cache()

    def step_device(self):
        """One pass of the hot path, inputs resident.  Returns (lines traced, RK steps tensor [L-only, L+Q])."""
        qsl, torch = self.qsl, self.torch
        if self.levels == 0:
            res = qsl.qsl_trace(self.field, self.seeds, self.pLQ if self.mode == 1 else self.pL, outputs=self.outs,
                                out=self.out_bufs, total_steps=self.tot)
            self.out_bufs.update(res)
            self.last = res
            two = torch.zeros(2, dtype=torch.int64, device="cuda")
            two[self.mode:self.mode + 1] = self.tot
            return self.n, two
        if self.hilbert:
            r, acc = self.hilbert_step()
            return r["counts"][-1], acc
        # keep = what the e2e step ships to the host; the rest of a level is dropped as soon as the next one is traced
        r = qsl.adaptive_map(self.field, self.lat, self.seeds, self.pL, self.pLQ, self.levels, self.cfg["p"])
        self.last = {"L": r["L0"]}
        self.level_sizes = [self.n] + [int(s.shape[0]) for s in r["seeds"][1:]]
        return sum(self.level_sizes), r["steps_by_mode"]

    def hilbert_step(self):
        """The paper's loop: level 0 L-only in curve order, then ndim x levels passes (each halves the key distance) on
        the curve and on the shifted curve, new samples traced with Q; then the converter to the finest lattice."""
        qsl, torch, args = self.qsl, self.torch, self.args
        acc = torch.zeros(2, dtype=torch.int64, device="cuda")
        calls = [0]

        def tf(sd):
            calls[0] += 1
            if calls[0] == 1:
                o = qsl.qsl_trace(self.field, sd, self.pL_curve, outputs=("L",), total_steps=self.tot)
                acc[0:1] += self.tot
                return o["L"], torch.full_like(o["L"], float("nan"))
            o = qsl.qsl_trace(self.field, sd, self.pLQ_curve, outputs=("L", "q_perp"), total_steps=self.tot)
            acc[1:2] += self.tot
            return o["L"], o["q_perp"]

        lat, levels = self.lat, self.levels
        r = qsl.hilbert_map(lat, levels, args.hilbert_thr, int(lat.ndim) * levels, args.hilbert_shift, tf)
        # the converter output at the finest lattice of cfg3 is 4.3 GB, of cfg5 275 GB: convert to level 2 (2-D) / 0 (3-D)
        self.hstate["map"] = qsl.qsl_hilbert_convert(lat, levels, min(levels, 2) if int(lat.ndim) == 2 else 0, r["keys"], r["Q"])
        self.hstate["r"] = r
        return r, acc

    def step_e2e(self):
        """The same through HOST buffers: pinned seeds -> device, hot path, results -> pinned host.
        Returns (h2d bytes, d2h bytes)."""
        qsl, torch = self.qsl, self.torch
        if self.levels == 0:
            # pipelined in pieces over two streams (driver.trace_host)
            qsl.trace_host(self.field, self.seeds_host, self.pLQ if self.mode == 1 else self.pL, outputs=self.outs,
                           chunks=self.args.e2e_chunks or None, host_out=self.host_res)
            return self.seeds_host.numel() * 8, sum(t.numel() * t.element_size() for t in self.host_res.values())
        d = self.seeds_host.cuda(non_blocking=True)
        if self.hilbert:
            # level-0 seeds are generated on the device by qsl_hilbert_level0: the host supplies the lattice only
            r, _ = self.hilbert_step()
            results = [r["keys"], r["L"], r["Q"], self.hstate["map"]]
        else:
            r = qsl.adaptive_map(self.field, self.lat, d, self.pL, self.pLQ, self.levels, self.cfg["p"])
            results = [r["L0"], r["S0"]]
            for lv in range(1, len(r["out"])):
                if r["out"][lv] is not None:
                    results += [r["coords"][lv], r["out"][lv]["L"], r["out"][lv]["q_perp"], r["out"][lv]["q_bnd"]]
        nb = 0
        for i, t in enumerate(results):
            h = self.host_out.get(i)
            if h is None or h.shape != t.shape:
                h = self.host_out[i] = torch.empty(t.shape, dtype=t.dtype).pin_memory()
            h.copy_(t, non_blocking=True)
            nb += t.numel() * t.element_size()
        return self.seeds_host.numel() * 8, nb


def time_device(W, steps, warmup, flush, barrier, clocks=None):
    """`warmup` untimed passes, then `steps` passes timed one by one with CUDA events on the launch stream (L2 flushed
    before each, outside the event pair); the trace kernels of every pass are timed by libqsl's own event pairs."""
    qsl, torch = W.qsl, W.torch
    qsl.qsl_profile_enable(True)               # the event pairs of the trace-kernel timing hook are created in the warm-up
    for _ in range(warmup):
        W.step_device()
    barrier()
    qsl.qsl_profile_enable(True)               # drop the warm-up launches from the trace-kernel event pool
    l0 = qsl.lib().qsl_launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    lines = 0
    rk = torch.zeros(2, dtype=torch.int64, device="cuda")
    kern_ms, kern_n = [0.0, 0.0], [0, 0]
    host_ms = []                               # host time spent enqueueing each pass (the calls are asynchronous)
    if clocks is not None:
        clocks.samples.clear(); clocks.reasons.clear()
    t_wall = time.perf_counter()
    lock = clocks.enqueue_lock if clocks is not None else contextlib.nullcontext()
    if warmup > 0:
        # One more untimed pass AFTER the barrier, with the timed passes enqueued right behind it: the first pass enqueued
        # on an idle device after a device-wide synchronisation sporadically (about one run in four) has one of its
        # driver calls stall the host for 5 - 300 ms, which would be idle GPU time inside that pass's event pair; it
        # belongs to the harness, not to the path (seen with and without the NVML sampler, in different driver calls).
        W.step_device()
        qsl.qsl_profile_enable(True)
        l0 = qsl.lib().qsl_launch_count()
    for a, b in ev:
        with lock:                             # no NVML query in flight while the pass is enqueued (ClockSampler)
            flush.zero_()                      # L2 flush, outside the event pair
            a.record()
            th = time.perf_counter()
            m, s = W.step_device()
            host_ms.append(round((time.perf_counter() - th) * 1e3, 3))
            b.record()
        rk += s
        lines += m
        kms, kn = qsl.qsl_profile_trace_kernel_ms()      # waits for this step's trace kernels (after b.record())
        for q in (0, 1):
            kern_ms[q] += kms[q]; kern_n[q] += kn[q]
    barrier()
    t_wall = time.perf_counter() - t_wall
    return {"lines": lines, "rk_by_mode": [int(v) for v in rk.tolist()], "kern_ms": kern_ms, "kern_n": kern_n,
            "launches": int(qsl.lib().qsl_launch_count() - l0), "dev_ms": sum(a.elapsed_time(b) for a, b in ev),
            "ms_each": [round(a.elapsed_time(b), 3) for a, b in ev], "host_ms_each": host_ms, "wall_s": t_wall, "steps": steps, "warmup": warmup}


def alu_roofline(W, T, peak_fma):
    """The trace kernel against the FP pipe peak measured on this device: algorithmic issue slots of SURVEY.md 8(d)."""
    f32 = W.f32
    peak = 2.0 * peak_fma / 1e12
    rk = T["rk_by_mode"]
    slots = PIPE_SLOTS_PER_STEP["L"] * rk[0] + PIPE_SLOTS_PER_STEP["LQ"] * rk[1]
    flops = FLOPS_PER_STEP["L"] * rk[0] + FLOPS_PER_STEP["LQ"] * rk[1]
    k_ms = T["kern_ms"][0] + T["kern_ms"][1]
    achieved = 2.0 * slots / (k_ms * 1e-3) / 1e12
    ncu = NCU_CAPTURES.get((W.name, "f32" if f32 else "f64"), {})
    return {
        "bound": "alu",
        "kernel": "%s (cell-table trace kernel; all %d launches of the timed region)"
                  % ("trace3_kernel, fp32 arithmetic" if f32 else "trace2_kernel", sum(T["kern_n"])),
        "achieved": achieved, "peak": peak, "unit": "TFLOP/s (FP-pipe issue slots x 2)", "frac": achieved / peak,
        "frac_true_flops": flops / (k_ms * 1e-3) / 1e12 / peak,
        "pipe_active_ncu": ncu.get("pipe_active"), "traffic": ncu.get("dram_bytes"), "ncu_source": ncu.get("source"),
        "kernel_ms": k_ms / T["steps"], "kernel_share_of_step": k_ms / T["dev_ms"],
        "launches_per_step": sum(T["kern_n"]) / T["steps"],
        "by_mode": {m: {"rk_steps_per_step": rk[q] / T["steps"], "kernel_ms_per_step": T["kern_ms"][q] / T["steps"],
                        "frac": (2.0 * PIPE_SLOTS_PER_STEP[m] * rk[q] / (T["kern_ms"][q] * 1e-3) / 1e12 / peak)
                        if T["kern_ms"][q] > 0 else None} for q, m in enumerate(("L", "LQ"))},
        "convention": "frac = algorithmic %s pipe issue slots (an FMA, add or multiply each take one: %d per RK4 step with "
                      "Q, %d without, SURVEY.md 8(d)) / the %s issue rate measured by qsl_peak_fma on this device; "
                      "frac_true_flops counts an FMA as 2 flops and an add or multiply as 1 (%d / %d flops per step) "
                      "against 2 x that rate; pipe_active_ncu = sm__pipe_%s_cycles_active of the committed ncu capture"
                      % ("FP32" if f32 else "FP64", PIPE_SLOTS_PER_STEP["LQ"], PIPE_SLOTS_PER_STEP["L"],
                         "FFMA" if f32 else "DFMA", FLOPS_PER_STEP["LQ"], FLOPS_PER_STEP["L"], "fma" if f32 else "fp64"),
        "true_flops_achieved_tflops": flops / (k_ms * 1e-3) / 1e12}


def gather_roofline(W, T, qsl):
    """--interp-order 2 / 3 (and any run of the corner-gather kernel): the trace kernel against the L1 gather rate.
    Algorithmic bytes: 4 stage evaluations x (order + 1)^3 stencil samples of 16 B (fp32) / 32 B (fp64) per RK4 step;
    peak = divergent gathers of that sample size over an L1-resident (64 KiB) footprint, measured by qsl_peak_gather."""
    sb = 16 if W.cfg["sample_type"] == "f32" else 32
    ns = (W.order + 1) ** 3
    k_ms = T["kern_ms"][0] + T["kern_ms"][1]
    achieved = sum(T["rk_by_mode"]) * 4.0 * ns * sb / (k_ms * 1e-3) / 1e9
    peak = qsl.qsl_peak_gather(sb, 64 << 10) * sb / 1e9
    return {"bound": "l1_gather", "kernel": "trace_kernel<ORDER = %d> (corner / stencil gather kernel; all %d launches of the timed region)"
                                            % (W.order, sum(T["kern_n"])),
            "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
            "kernel_ms": k_ms / T["steps"], "kernel_share_of_step": k_ms / T["dev_ms"],
            "convention": "4 evaluations x %d samples x %d B gathered per RK4 step / qsl_peak_gather(%d B, 64 KiB footprint)" % (ns, sb, sb)}


def streaming_block(qsl, torch, W):
    """the HBM-streaming stages as GB/s against MEASURED_PEAKS.json hbm_gbs.  Each C-ABI call is timed with
    CUDA events (best of 5 after 2 warm-ups, L2 not flushed: every input is larger than L2) on synthetic maps of the size of
    the largest config (512 x 512 x 256 values); bytes = the algorithmic bytes DESIGN.md section 5 states per unit."""
    import qsl_inputs as qi
    peak = hbm_peak_gbs()
    out = {"peak_gbs": peak, "peak_source": "MEASURED_PEAKS.json hbm_gbs" if peak != 6650.0 else "fallback 6650 (B200_PROFILING.md)",
           "kernels": {}}

    def best(fn, reps=5):
        for _ in range(2):
            fn()
        ts = []
        for _ in range(reps):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); fn(); b.record(); b.synchronize()
            ts.append(a.elapsed_time(b))
        return min(ts)

    def put(name, ms, nbytes, note):
        gbs = nbytes / (ms * 1e-3) / 1e9
        out["kernels"][name] = {"ms": round(ms, 4), "bytes": int(nbytes), "gbs": round(gbs, 1), "frac": round(gbs / peak, 3), "what": note}

    gen = torch.Generator(device="cuda"); gen.manual_seed(1609)
    n3 = (256, 512, 512)
    L3 = torch.rand(n3, dtype=torch.float64, device="cuda", generator=gen) + 0.1
    S3 = torch.empty_like(L3)
    N = L3.numel()
    put("fledge_dense_3d", best(lambda: qsl.qsl_fledge_dense(L3, 3, out=S3)), 16 * N, "512x512x256 map, 8 B in + 8 B out per value")
    L2 = L3.view(8192, 8192)
    put("fledge_dense_2d", best(lambda: qsl.qsl_fledge_dense(L2, 2, out=S3.view(8192, 8192))), 16 * N, "8192x8192 map, 8 B in + 8 B out per value")
    tau = torch.empty(1, dtype=torch.float64, device="cuda")
    passes = SELECT_PASSES
    put("select", best(lambda: qsl.qsl_select(S3.view(-1), 0.95, out=tau)), 8 * N * passes,
        "order statistic of 6.7e7 values: 8 radix passes of 8 bits, %d of them over the whole map x 8 B per value (the other 5 "
        "read the candidates pass 2 kept; their data-dependent traffic is not counted)" % passes)
    lat = qi.Lattice(3, (512, 512, 256), (0.0, 0.0, 0.0), (1.0, 0, 0), (0, 1.0, 0), (0, 0, 0.5))
    cap = (N - int(math.ceil(0.95 * N)) + 8) << 3
    m = [0]

    def refine():
        cc, cs, cb = qsl.qsl_refine(lat, 0, None, S3.view(-1), tau, capacity=cap)
        m[0] = int(cc.shape[0])
    ms = best(refine)
    put("refine", ms, 8 * N * 2 + m[0] * (12 + 24) + 8 * N,
        "count + scan + fused scan / emit of 6.7e7 cells, %d children: S read twice, child_base 8 B per cell, 36 B per child (includes the host sync for the count)" % m[0])
    # sparse FLEDGE of level 1 on those children
    cc, cs, cb = qsl.qsl_refine(lat, 0, None, S3.view(-1), tau, capacity=cap)
    L1 = torch.rand(cc.shape[0], dtype=torch.float64, device="cuda", generator=gen) + 0.1
    put("fledge_sparse_3d", best(lambda: qsl.qsl_fledge_sparse(lat, 1, L3.view(-1), [None, cc], [None, L1], [cb])),
        int(cc.shape[0]) * (12 + 8 + 8), "level-1 cells: 12 B coords + 8 B L in, 8 B out per cell; 8 ancestor walks + 27 look-ups per cell: bound by the L1 "
        "wavefront rate of these gathers (83 % of it by ncu, profiles/r2g), not by HBM")
    del L3, S3, L2, L1, cc, cs, cb
    # seed ordering: Morton keys + radix sort of (key, index) pairs, as qsl_trace does it; measured through the test hook
    n = 1 << 26
    keys = torch.randint(0, 1 << 30, (n,), dtype=torch.int32, device="cuda", generator=gen)
    vals = torch.arange(n, dtype=torch.int32, device="cuda")
    k2, v2 = keys.clone(), vals.clone()
    import ctypes as C

    def sort():
        k2.copy_(keys); v2.copy_(vals)
        rc = qsl.lib().qsl_debug_sort_pairs(C.c_void_p(k2.data_ptr()), C.c_void_p(v2.data_ptr()), C.c_longlong(n), C.c_int(30),
                                            C.c_void_p(torch.cuda.current_stream().cuda_stream))
        assert rc == 0
    t_copy = best(lambda: (k2.copy_(keys), v2.copy_(vals)))
    put("radix_sort_pairs", best(sort) - t_copy, n * 8 * 2 * SORT_PASSES + n * 4 * SORT_PASSES,
        "6.7e7 (key, index) pairs, 30-bit keys: %d passes x (histogram read 4 B + scatter read 8 B + write 8 B)" % SORT_PASSES)
    # the same sort on the keys the path really sees: Morton codes of a 512 x 512 x 256 seed lattice in index order (27 bits)
    def spread3(v):
        v = v & 0x3ff
        v = (v | (v << 16)) & 0x030000ff
        v = (v | (v << 8)) & 0x0300f00f
        v = (v | (v << 4)) & 0x030c30c3
        return (v | (v << 2)) & 0x09249249
    idx = torch.arange(n, dtype=torch.int64, device="cuda")
    keys.copy_((spread3(idx % 512) | (spread3((idx // 512) % 512) << 1) | (spread3(idx // (512 * 512)) << 2)).to(torch.int32))
    del idx

    def sort_lattice():
        k2.copy_(keys); v2.copy_(vals)
        rc = qsl.lib().qsl_debug_sort_pairs(C.c_void_p(k2.data_ptr()), C.c_void_p(v2.data_ptr()), C.c_longlong(n), C.c_int(27),
                                            C.c_void_p(torch.cuda.current_stream().cuda_stream))
        assert rc == 0
    put("radix_sort_pairs_lattice_keys", best(sort_lattice) - t_copy, n * 8 * 2 * SORT_PASSES + n * 4 * SORT_PASSES,
        "the same sort on the Morton keys of a 512 x 512 x 256 seed lattice in index order (what qsl_trace sorts): long runs "
        "per digit, %d passes" % SORT_PASSES)
    del keys, vals, k2, v2
    # field pack + per-cell table: the whole qsl_field_create call of this run's workload (allocation included), warm
    g = W.cfg["grid"]
    nodes = g.nx * g.ny * g.nz
    cells = (g.nx - 1) * (g.ny - 1) * (g.nz - 1)
    sb = 16 if W.cfg["sample_type"] == "f32" else 32
    dev = [torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64).reshape(-1)).cuda() for a in W.cfg["B"]]
    st = qsl.QSL_F32 if W.cfg["sample_type"] == "f32" else qsl.QSL_F64
    ts = []
    for _ in range(3):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        f = qsl.qsl_field_create(g.nx, g.ny, g.nz, *dev, lo=g.lo, hi=g.hi, sample_type=st,
                                 layout=qsl.QSL_LAYOUT_CELL_TABLE_F32 if W.f32 else qsl.QSL_LAYOUT_CELL_TABLE)
        b.record(); b.synchronize()
        ts.append(a.elapsed_time(b))
        f.destroy()
    del dev
    put("field_create", min(ts), nodes * (24 + sb) + cells * (96 if W.f32 else 192),
        "whole qsl_field_create call of %s (pack_kernel + cell_table_kernel + cudaMalloc of the arrays + axis upload with its host "
        "synchronisation), best of 3: 24 B in + %d B out per node, %d B out per cell" % (W.name, sb, 96 if W.f32 else 192))
    torch.cuda.empty_cache()
    return out


def hbm_peak_gbs():
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"])
    except Exception:
        return 6650.0


# ---------------------------------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=sorted(WORKLOADS))
    ap.add_argument("--scale", type=float, default=1.0, help="shrink grid and seed lattice (debugging only)")
    ap.add_argument("--flags", type=int, default=0, help="QSL_FLAG_* tuning flags (debugging only)")
    ap.add_argument("--arith", default="f64", choices=["f64", "f32"],
                    help="arithmetic of the integrator; f32 = QSL_ARITH_F32 throughput mode (fp32-sampled workloads only; "
                         "parity is gated in f64, DESIGN.md reading A6)")
    ap.add_argument("--refine", default="fledge", choices=["fledge", "hilbert"],
                    help="refinement scheme of cfg3 / cfg5: FLEDGE percentile + 2x cells (BASELINE.json configs), or the paper's "
                         "own Hilbert-curve mid-point insertion on length jumps (PAPER.md:194-206; DESIGN.md reading A17)")
    ap.add_argument("--hilbert-thr", type=float, default=0.05, help="field-line-length jump threshold of --refine hilbert")
    ap.add_argument("--hilbert-shift", type=int, default=5, help="shift of the second curve in fine cells (0 = no shifted pass)")
    ap.add_argument("--interp-order", type=int, default=1, choices=[1, 2, 3],
                    help="1 trilinear (cell-table kernel, default), 2 triquadratic (Dodgson), 3 tricubic (Keys): PAPER.md:91-93; the "
                         "higher orders run in the stencil-gather kernel and are reported against the L1 gather rate")
    ap.add_argument("--e2e-chunks", type=int, default=0,
                    help="pieces the end-to-end path pipelines over two streams; 0 = one piece per 4 M lines (at most 8)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true",
                    help="skip the per_config block (after the timed workload the other four BASELINE.json configs are timed "
                         "briefly, N = 1 only; about two minutes, most of it cfg5)")
    ap.add_argument("--no-streaming", action="store_true", help="skip the GB/s block of the HBM-streaming stages")
    args = ap.parse_args()
    rank, world, local = _env_int("RANK", 0), _env_int("WORLD_SIZE", 1), _env_int("LOCAL_RANK", 0)

    import qsl_inputs as qi
    if args.impl == "reference":
        if rank == 0:
            run_reference(args, qi.make_config(args.workload, args.scale))
        return 0

    import torch
    import paper_1609_00724_b200 as qsl
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libqsl has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if args.arith == "f32" and args.workload not in ("cfg4", "cfg5"):
        raise SystemExit("--arith f32 needs an fp32-sampled workload (cfg4, cfg5)")
    if args.interp_order != 1 and args.arith == "f32":
        raise SystemExit("--interp-order 2 / 3 run in fp64 arithmetic")

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    W = Workload(qsl, torch, args.workload, args)
    cfg, f32 = W.cfg, W.f32
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    qsl.qsl_profile_enable(True)

    # ---- device-resident timing -------------------------------------------------------------------------------------
    # NVML is initialised and its sampling thread started before the warm-up: its first calls take driver locks that
    # would otherwise delay the launches of the first timed step; the samples of the warm-up are dropped.
    clocks = ClockSampler(local)
    clocks.__enter__()
    warm = max(args.warmup, 3) if args.warmup > 0 else 0
    try:
        T = time_device(W, args.steps, warm, flush, barrier, clocks)
    finally:
        clocks.__exit__()
    rk_steps = sum(T["rk_by_mode"])
    t = torch.tensor([T["dev_ms"]], dtype=torch.float64, device="cuda")
    agg = torch.tensor([float(T["lines"]), float(rk_steps)], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(agg, op=dist.ReduceOp.SUM)
    dev_ms_max = float(t.item())
    lines_all, steps_all = float(agg[0].item()), float(agg[1].item())

    # ---- end to end through host buffers ----------------------------------------------------------------------------
    for _ in range(2):
        W.step_e2e()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e2e_ms = 0.0
    for _ in range(args.steps):
        flush.zero_()
        e0.record()
        bi, bo = W.step_e2e()
        e1.record()
        e1.synchronize()
        e2e_ms += e0.elapsed_time(e1)
    barrier()
    t2 = torch.tensor([e2e_ms], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(t2, op=dist.ReduceOp.MAX)
    e2e_ms_max = float(t2.item())

    # ---- roofline of the dominant kernel (trace kernel) against the measured FP pipe peak ---------------------------
    roofline = None
    peak_fma = None
    if rank == 0:
        peak_fma = qsl.qsl_peak_fma(not f32)           # DFMA/s (FFMA/s with --arith f32), measured on this device
        roofline = alu_roofline(W, T, peak_fma)
        if W.order != 1:
            roofline = dict(gather_roofline(W, T, qsl), alu=roofline)
        k_ms = T["kern_ms"][0] + T["kern_ms"][1]
        # the other candidate bounds of SURVEY.md 8(d): divergent gathers of table entries through L1 / L2.  Algorithmic
        # traffic: a line enters a new cell every ~2.5 steps at h = 0.25 cell and then reads one table entry (192 B fp64,
        # 96 B fp32); peaks = 32-byte divergent gathers over an L1-resident (64 KiB), an L2-resident (64 MiB) and an
        # HBM-resident (1 GiB) footprint, measured here (the three micro-kernels of SURVEY.md:396-399).
        roofline["other_bounds"] = []
        g_ach = (rk_steps / 2.5) * (96.0 if f32 else 192.0) / (k_ms * 1e-3) / 1e9
        for label, fp in (("l1_gather", 64 << 10), ("l2_gather", 64 << 20), ("hbm_gather", 1 << 30)):
            try:
                g_peak = qsl.qsl_peak_gather(32, fp) * 32.0 / 1e9
                if label == "hbm_gather":
                    tr = roofline.get("traffic")
                    a_hbm = tr / (roofline["kernel_ms"] * 1e-3) / 1e9 if tr else None
                    roofline["other_bounds"].append({"bound": label, "achieved": a_hbm, "peak": g_peak, "unit": "GB/s",
                                                     "frac": a_hbm / g_peak if a_hbm else None,
                                                     "convention": "achieved = ncu dram bytes of one launch / kernel time (null without a "
                                                                   "capture of this workload); peak = qsl_peak_gather(32 B, 1 GiB footprint)"})
                    continue
                roofline["other_bounds"].append({"bound": label, "achieved": g_ach, "peak": g_peak, "unit": "GB/s", "frac": g_ach / g_peak,
                                                 "convention": "one table entry per cell entered, a cell every 2.5 RK4 steps; peak = "
                                                               "qsl_peak_gather(32 B, %d-byte footprint)" % fp})
            except Exception as exc:                               # the roofline of the binding unit stands on its own
                roofline["other_bounds"].append({"bound": label, "error": str(exc)})
        if world == 1 and not args.no_streaming:
            try:
                roofline["streaming"] = streaming_block(qsl, torch, W)
            except Exception as exc:
                roofline["streaming"] = {"error": repr(exc)}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = oracle_leg(cfg, W.last, torch)

    summary = lambda name, Tm, Wm: {
        "lines_per_s": Tm["lines"] / (Tm["dev_ms"] * 1e-3), "rk_steps_per_s": sum(Tm["rk_by_mode"]) / (Tm["dev_ms"] * 1e-3),
        "ms_per_step": Tm["dev_ms"] / Tm["steps"], "lines_per_step": Tm["lines"] / Tm["steps"],
        "roofline_frac": alu_roofline(Wm, Tm, peak_fma)["frac"], "kernel_ms": (Tm["kern_ms"][0] + Tm["kern_ms"][1]) / Tm["steps"],
        "steps": Tm["steps"], "warmup": Tm["warmup"], "workload": WORKLOADS[name]}
    per_config = None
    if rank == 0 and world == 1 and (not args.no_per_config) and args.interp_order == 1 and args.scale == 1.0:
        per_config = {args.workload: summary(args.workload, T, W)}
        W.close()
        for name in sorted(WORKLOADS):
            if name == args.workload:
                continue
            try:
                Wo = Workload(qsl, torch, name, args)
                # cfg5 is 24 s per pass: one timed pass after one warm-up pass (a cold pass spends another 0.76 s in
                # cudaMalloc of the 10 - 60 GB blocks of its levels: 24.36 s cold, 23.60 s warm, profiles/r2f)
                To = time_device(Wo, 1 if name == "cfg5" else 3, 1 if name == "cfg5" else 2, flush, barrier)
                per_config[name] = summary(name, To, Wo)
                if getattr(Wo, "level_sizes", None):
                    per_config[name]["level_sizes"] = Wo.level_sizes
                Wo.close()
                del Wo
            except Exception as exc:
                per_config[name] = {"error": repr(exc)}
            torch.cuda.empty_cache()

    if rank == 0:
        line = {
            "metric": "field lines/s (with Q)", "value": lines_all / (dev_ms_max * 1e-3), "unit": "lines/s",
            "n_gpus": world, "steps": args.steps, "warmup": warm,
            "ms_per_step": dev_ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if f32 else "f64", "data": "synthetic", "config": workload_config(cfg, args),
            "rk_steps_per_s": steps_all / (dev_ms_max * 1e-3), "rk_steps_per_step": rk_steps / args.steps,
            "lines_per_step": T["lines"] / args.steps, "wall_s_timed_region": T["wall_s"],
            "ms_each_step": T["ms_each"], "host_enqueue_ms_each_step": T["host_ms_each"],
            "clocks": clocks.summary(),
            "e2e": {"value": lines_all / (e2e_ms_max * 1e-3), "unit": "lines/s", "h2d_bytes_per_step": bi,
                    "d2h_bytes_per_step": bo, "ms_per_step": e2e_ms_max / args.steps},
            "gpu_launches": T["launches"],
            "roofline": roofline,
            "cpu_baseline": cpu,
        }
        if per_config is not None:
            line["per_config"] = per_config
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())

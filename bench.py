#!/usr/bin/env python
"""bench.py -- field lines/s (with Q) and RK steps/s of the libqsl hot path on B200, with its roofline fraction.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2] [--impl reference]

A "step" is one pass of the whole hot path over one batch of synthetic input: seed ordering, the persistent trace
kernel (a3-a5), the Q/L epilogue (a6) and, for the refinement workloads cfg3 / cfg5, FLEDGE, threshold, compaction and
the level loop (a7-a9).  The default workload is BASELINE.json configs[1] (cfg2: quadrupole, fp64 128^3 field,
1024^2 photospheric seeds, L + Q); DESIGN.md "Measurement" states what every key means.

`value`   lines/s with the seeds and the packed field already resident in HBM (CUDA events on the launch stream).
`e2e`     the same through the public binding with HOST buffers: pinned seeds -> device, trace, results -> pinned host.
`roofline` the trace kernel against the FP64 (or FP32) pipe peak measured on this device by qsl_peak_fma.
`cpu_baseline` the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload, rank 0, N = 1 only.
`--impl reference` times only that oracle (the reference arm of the contract).

Under torchrun every rank traces its own replica of the workload (lines are independent: weak scaling, no data-path
collective); the time is the max over ranks and `value` the lines all ranks traced divided by it.
"""
from __future__ import annotations

import argparse
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
# dram__bytes_read.sum + dram__bytes_write.sum of one trace-kernel launch of the default workload, from the committed
# ncu --set full capture (profiles/); None until a capture of the current kernel exists.
NCU_TRACE_KERNEL_DRAM_BYTES = {"cfg2": 789848320}   # profiles/r1b_cell_table_kernel.md


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
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv, self.h = pynvml, pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
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

    def summary(self):
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s)}


# ---------------------------------------------------------------------------------------------------------------------
def oracle_sample(cfg, target_s=15.0):
    """Times the CPU oracle on a bounded, deterministic sample of the workload's level-0 seeds (every k-th seed, k
    chosen from a small pilot run so that the timed run is about `target_s` seconds).  Returns (lines/s, steps/s,
    cores, description)."""
    import oracle
    st = oracle.F32 if cfg["sample_type"] == "f32" else oracle.F64
    f = oracle.Field(cfg["grid"], cfg["B"], st, oracle.NORMALIZE_FIRST)
    seeds = cfg["seeds"]
    n = len(seeds)
    mode = cfg["mode"]
    kw = dict(step_frac=cfg["step_frac"], mode=mode, max_steps=cfg["max_steps"], null_eps=cfg["null_eps"])
    cores = os.cpu_count() or 1

    def run(stride):
        s = np.ascontiguousarray(seeds[::stride])
        t0 = time.perf_counter()
        o = oracle.trace(f, s, cfg["box_lo"], cfg["box_hi"], **kw)
        return len(s), int(o["total_steps"]), time.perf_counter() - t0

    pilot_stride = max(1, n // 4096)
    m, steps, dt = run(pilot_stride)
    rate = m / max(dt, 1e-6)                                   # lines/s of the pilot
    stride = max(1, int(math.ceil(n / max(rate * target_s, 1.0))))
    if stride < pilot_stride:
        m, steps, dt = run(stride)
    else:
        stride = pilot_stride
    desc = "every %d-th level-0 seed of %s (%d of %d lines, %d RK4 steps, %.1f s wall, OpenMP over lines, mode %s)" % (
        stride, cfg["name"], m, n, steps, dt, "L+Q" if mode == 1 else "L")
    return m / dt, steps / dt, cores, desc


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
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=sorted(WORKLOADS))
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
    ap.add_argument("--e2e-chunks", type=int, default=0,
                    help="pieces the end-to-end path pipelines over two streams; 0 = one piece per 4 M lines (at most 8)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
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

    cfg = qi.make_config(args.workload, args.scale)
    g = cfg["grid"]
    dev = [torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64).reshape(-1)).cuda() for a in cfg["B"]]
    st = qsl.QSL_F32 if cfg["sample_type"] == "f32" else qsl.QSL_F64
    f32 = args.arith == "f32"
    if f32 and cfg["sample_type"] != "f32":
        raise SystemExit("--arith f32 needs an fp32-sampled workload (cfg4, cfg5)")
    field = qsl.qsl_field_create(g.nx, g.ny, g.nz, *dev, lo=g.lo, hi=g.hi, sample_type=st,
                                 layout=qsl.QSL_LAYOUT_CELL_TABLE_F32 if f32 else qsl.QSL_LAYOUT_CELL_TABLE)
    del dev
    seeds_host = torch.from_numpy(np.ascontiguousarray(cfg["seeds"])).pin_memory()
    n = int(seeds_host.shape[0])
    seeds = seeds_host.cuda()
    mode = cfg["mode"]
    levels = int(cfg["levels"])
    mk = lambda m: qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], mode=m, step_frac=cfg["step_frac"],
                                         max_steps=cfg["max_steps"], null_eps=cfg["null_eps"], flags=args.flags,
                                         arith=qsl.QSL_ARITH_F32 if f32 else qsl.QSL_ARITH_F64)
    pL, pLQ = mk(qsl.QSL_TRACE_L), mk(qsl.QSL_TRACE_LQ)
    outs = ("end_f", "end_b", "L", "q_perp", "q_bnd", "face_f", "face_b", "status")
    out_bufs = {}
    tot = torch.zeros(1, dtype=torch.int64, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    lat = cfg["lattice"]
    qsl.qsl_profile_enable(True)

    def step_device():
        """One pass of the hot path, inputs resident.  Returns (lines traced, RK steps tensor [L-only, L+Q])."""
        if levels == 0:
            res = qsl.qsl_trace(field, seeds, pLQ if mode == 1 else pL, outputs=outs, out=out_bufs, total_steps=tot)
            out_bufs.update(res)
            two = torch.zeros(2, dtype=torch.int64, device="cuda")
            two[mode:mode + 1] = tot
            return n, two
        if hilbert:
            r, acc = hilbert_step()
            return r["counts"][-1], acc
        r = qsl.adaptive_map(field, lat, seeds, pL, pLQ, levels, cfg["p"])
        return n + sum(int(s.shape[0]) for s in r["seeds"][1:]), r["steps_by_mode"]

    hilbert = args.refine == "hilbert" and levels > 0
    hstate = {}

    def hilbert_step():
        """The paper's loop: level 0 L-only in curve order, then ndim x levels passes (each halves the key distance) on
        the curve and on the shifted curve, new samples traced with Q; then the converter to the finest lattice."""
        acc = torch.zeros(2, dtype=torch.int64, device="cuda")
        calls = [0]

        def tf(sd):
            calls[0] += 1
            if calls[0] == 1:
                o = qsl.qsl_trace(field, sd, pL, outputs=("L",), total_steps=tot)
                acc[0:1] += tot
                return o["L"], torch.full_like(o["L"], float("nan"))
            o = qsl.qsl_trace(field, sd, pLQ, outputs=("L", "q_perp"), total_steps=tot)
            acc[1:2] += tot
            return o["L"], o["q_perp"]

        r = qsl.hilbert_map(lat, levels, args.hilbert_thr, int(lat.ndim) * levels, args.hilbert_shift, tf)
        # the converter output at the finest lattice of cfg3 is 4.3 GB, of cfg5 275 GB: convert to level 2 (2-D) / 0 (3-D)
        hstate["map"] = qsl.qsl_hilbert_convert(lat, levels, min(levels, 2) if int(lat.ndim) == 2 else 0, r["keys"], r["Q"])
        hstate["r"] = r
        return r, acc

    host_out = {}
    host_res = {}

    def step_e2e():
        """The same through HOST buffers: pinned seeds -> device, hot path, results -> pinned host."""
        if levels == 0:
            # pinned seeds -> device, trace, results -> pinned host, pipelined in pieces over two streams (driver.trace_host)
            qsl.trace_host(field, seeds_host, pLQ if mode == 1 else pL, outputs=outs, chunks=args.e2e_chunks or None, host_out=host_res)
            return seeds_host.numel() * 8, sum(t.numel() * t.element_size() for t in host_res.values())
        d = seeds_host.cuda(non_blocking=True)
        if hilbert:
            # level-0 seeds are generated on the device by qsl_hilbert_level0: the host supplies the lattice only
            r, _ = hilbert_step()
            results = [r["keys"], r["L"], r["Q"], hstate["map"]]
        else:
            r = qsl.adaptive_map(field, lat, d, pL, pLQ, levels, cfg["p"])
            results = [r["L0"], r["S0"]]
            for lv in range(1, len(r["out"])):
                if r["out"][lv] is not None:
                    results += [r["coords"][lv], r["out"][lv]["L"], r["out"][lv]["q_perp"], r["out"][lv]["q_bnd"]]
        nb = 0
        for i, t in enumerate(results):
            h = host_out.get(i)
            if h is None or h.shape != t.shape:
                h = host_out[i] = torch.empty(t.shape, dtype=t.dtype).pin_memory()
            h.copy_(t, non_blocking=True)
            nb += t.numel() * t.element_size()
        return seeds_host.numel() * 8, nb

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing -------------------------------------------------------------------------------------
    # NVML is initialised and its sampling thread started before the warm-up: its first calls take driver locks that
    # would otherwise delay the launches of the first timed step; the samples of the warm-up are dropped below.
    clocks = ClockSampler(local)
    clocks.__enter__()
    for _ in range(max(args.warmup, 3) if args.warmup > 0 else 0):
        step_device()
    barrier()
    qsl.qsl_profile_enable(True)               # drop the warm-up launches from the trace-kernel event pool
    l0 = qsl.lib().qsl_launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    lines = 0
    rk = torch.zeros(2, dtype=torch.int64, device="cuda")
    kern_ms, kern_n = [0.0, 0.0], [0, 0]
    try:
        clocks.samples.clear(); clocks.reasons.clear()
        t_wall = time.perf_counter()
        for a, b in ev:
            flush.zero_()                      # L2 flush, outside the event pair
            a.record()
            m, s = step_device()
            b.record()
            rk += s
            lines += m
            kms, kn = qsl.qsl_profile_trace_kernel_ms()      # waits for this step's trace kernels (after b.record())
            for q in (0, 1):
                kern_ms[q] += kms[q]; kern_n[q] += kn[q]
        barrier()
        t_wall = time.perf_counter() - t_wall
    finally:
        clocks.__exit__()
    launches = qsl.lib().qsl_launch_count() - l0
    dev_ms = sum(a.elapsed_time(b) for a, b in ev)
    rk_by_mode = [int(v) for v in rk.tolist()]
    rk_steps = sum(rk_by_mode)
    t = torch.tensor([dev_ms], dtype=torch.float64, device="cuda")
    agg = torch.tensor([float(lines), float(rk_steps)], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(agg, op=dist.ReduceOp.SUM)
    dev_ms_max = float(t.item())
    lines_all, steps_all = float(agg[0].item()), float(agg[1].item())

    # ---- end to end through host buffers ----------------------------------------------------------------------------
    for _ in range(2):
        step_e2e()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e2e_ms = 0.0
    for _ in range(args.steps):
        flush.zero_()
        e0.record()
        bi, bo = step_e2e()
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
    if rank == 0:
        peak_fma = qsl.qsl_peak_fma(not f32)           # DFMA/s (FFMA/s with --arith f32), measured on this device
        peak = 2.0 * peak_fma / 1e12
        # algorithmic FP64 issue slots of all trace-kernel launches of the timed region (both modes) / their device time
        slots = PIPE_SLOTS_PER_STEP["L"] * rk_by_mode[0] + PIPE_SLOTS_PER_STEP["LQ"] * rk_by_mode[1]
        flops = FLOPS_PER_STEP["L"] * rk_by_mode[0] + FLOPS_PER_STEP["LQ"] * rk_by_mode[1]
        k_ms = kern_ms[0] + kern_ms[1]
        achieved = 2.0 * slots / (k_ms * 1e-3) / 1e12
        roofline = {"bound": "alu", "kernel": "%s (cell-table trace kernel; all %d launches of the timed region)"
                    % ("trace3_kernel, fp32 arithmetic" if f32 else "trace2_kernel", kern_n[0] + kern_n[1]), "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                    "frac": achieved / peak, "traffic": NCU_TRACE_KERNEL_DRAM_BYTES.get(args.workload),
                    "kernel_ms": k_ms / args.steps, "kernel_share_of_step": k_ms / dev_ms,
                    "launches_per_step": (kern_n[0] + kern_n[1]) / args.steps,
                    "by_mode": {m: {"rk_steps_per_step": rk_by_mode[q] / args.steps, "kernel_ms_per_step": kern_ms[q] / args.steps,
                                    "frac": (2.0 * PIPE_SLOTS_PER_STEP[m] * rk_by_mode[q] / (kern_ms[q] * 1e-3) / 1e12 / peak)
                                    if kern_ms[q] > 0 else None} for q, m in enumerate(("L", "LQ"))},
                    "convention": "%s pipe issue slots x 2 (FMA-equivalent flops): %d slots per RK4 step with Q, %d "
                                  "without; peak = %s rate measured by qsl_peak_fma on this device"
                                  % ("FP32" if f32 else "FP64", PIPE_SLOTS_PER_STEP["LQ"], PIPE_SLOTS_PER_STEP["L"],
                                     "FFMA" if f32 else "DFMA"),
                    "true_flops_achieved_tflops": flops / (k_ms * 1e-3) / 1e12}
        # the other candidate bound of SURVEY.md 8(d): divergent gathers of table entries through L1/L2.  Algorithmic
        # traffic: a line enters a new cell every ~2.5 steps at h = 0.25 cell and then reads one table entry (192 B fp64,
        # 96 B fp32); peak = 32-byte divergent gathers over an L2-resident (64 MiB) footprint, measured here.
        try:
            g_peak = qsl.qsl_peak_gather(32, 64 << 20) * 32.0 / 1e9
            g_ach = (rk_steps / 2.5) * (96.0 if f32 else 192.0) / (k_ms * 1e-3) / 1e9
            roofline["other_bounds"] = [{"bound": "l2_gather", "achieved": g_ach, "peak": g_peak, "unit": "GB/s",
                                         "frac": g_ach / g_peak,
                                         "convention": "one table entry per cell entered, a cell every 2.5 RK4 steps; peak = "
                                                       "qsl_peak_gather(32 B, 64 MiB footprint)"}]
        except Exception as exc:                                   # the roofline of the binding unit stands on its own
            roofline["other_bounds"] = [{"bound": "l2_gather", "error": str(exc)}]

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, sps, cores, desc = oracle_sample(cfg)
        cpu = {"value": v, "unit": "lines/s", "cores": cores, "kind": "oracle", "sample": desc, "rk_steps_per_s": sps}

    if rank == 0:
        line = {
            "metric": "field lines/s (with Q)", "value": lines_all / (dev_ms_max * 1e-3), "unit": "lines/s",
            "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3) if args.warmup > 0 else 0,
            "ms_per_step": dev_ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if f32 else "f64", "data": "synthetic", "config": workload_config(cfg, args),
            "rk_steps_per_s": steps_all / (dev_ms_max * 1e-3), "rk_steps_per_step": rk_steps / args.steps,
            "lines_per_step": lines / args.steps, "wall_s_timed_region": t_wall,
            "ms_each_step": [round(a.elapsed_time(b), 3) for a, b in ev],
            "clocks": clocks.summary(),
            "e2e": {"value": lines_all / (e2e_ms_max * 1e-3), "unit": "lines/s", "h2d_bytes_per_step": bi,
                    "d2h_bytes_per_step": bo, "ms_per_step": e2e_ms_max / args.steps},
            "gpu_launches": int(launches),
            "roofline": roofline,
            "cpu_baseline": cpu,
        }
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())

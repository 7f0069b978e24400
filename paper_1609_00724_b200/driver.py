"""Level loop of the adaptive refinement: orchestration only, every step is a libqsl call.

PAPER.md:194-200: sample the region on a rectilinear grid, find where the field-line length jumps, sample those places
more finely, repeat.  Reading A11: level 0 is traced L-only, FLEDGE = Sobel magnitude of L, tau = the p-th
percentile (nearest rank) of the level-0 FLEDGE map, reused at every level; cells with S > tau are split 2x per axis and
their children traced with Q; the children's L feeds the sparse FLEDGE map of the next level.
"""
from __future__ import annotations

import torch

from . import binding as B


@B._on_stream
def adaptive_map(field, lattice, seeds0, params_L, params_LQ, n_levels: int, p: float, *, stream=None,
                 outputs=("L", "q_perp", "q_bnd", "status"), max_children=None, on_level=None, keep=None):
    """Runs level 0 (dense, `params_L`) and `n_levels` refinement levels (`params_LQ`).

    seeds0: CUDA float64 (n0*n1*n2, 3) level-0 seeds in dense index order.
    `stream`: every libqsl launch AND every torch-side operation of the loop (allocations, the step-counter sums) run
    on it (it is made torch's current stream for the duration of the call).
    `on_level(level, coords, seeds, out)` is called after the trace of every refined level (1..n_levels) with that
    level's device tensors (e.g. to copy a level to the host or to disk while the next one is traced); `keep`, a subset of
    `outputs`, names what stays in the returned dict afterwards (default: everything; "L" is always kept, the sparse
    FLEDGE of the next level reads it) - 3-D maps with hundreds of millions of refined samples need this.
    Returns a dict: L0 (dense map), S0, tau (CUDA float64[1]) and per-level lists coords / seeds / out (trace outputs) /
    S / child_base, plus `total_steps` (CUDA int64[1], summed over all levels) and `steps_by_mode` (CUDA int64[2]: RK
    steps of the L-only level-0 pass and of the L+Q passes over the refined seeds).
    """
    ndim = int(lattice.ndim)
    shape = tuple(int(v) for v in lattice.n[:ndim][::-1])
    steps = torch.zeros(1, dtype=torch.int64, device="cuda")
    acc = torch.zeros(2, dtype=torch.int64, device="cuda")
    o0 = B.qsl_trace(field, seeds0, params_L, outputs=("L", "status"), total_steps=steps, stream=stream)
    acc[0:1] += steps
    L0 = o0["L"]
    S0 = B.qsl_fledge_dense(L0.view(shape), ndim, stream=stream).view(-1)
    tau = B.qsl_select(S0, p, stream=stream)
    res = dict(L0=L0, status0=o0["status"], S0=S0, tau=tau, coords=[None], seeds=[seeds0], out=[o0], S=[S0], child_base=[])
    coords, S = None, S0
    Ls = [L0]
    for level in range(n_levels):
        cc, cs, cb = B.qsl_refine(lattice, level, coords, S, tau, capacity=max_children, stream=stream)
        res["child_base"].append(cb)
        res["coords"].append(cc); res["seeds"].append(cs)
        if cc.shape[0] == 0:
            res["out"].append(None); res["S"].append(None)
            break
        o = B.qsl_trace(field, cs, params_LQ, outputs=outputs, total_steps=steps, stream=stream)
        acc[1:2] += steps
        if on_level is not None:
            on_level(level + 1, cc, cs, o)
        if keep is not None:
            o = {k: v for k, v in o.items() if k == "L" or k in keep}
        res["out"].append(o)
        Ls.append(o["L"])
        if level + 1 < n_levels:
            S = B.qsl_fledge_sparse(lattice, level + 1, L0, res["coords"], Ls, res["child_base"], stream=stream)
            res["S"].append(S)
            coords = cc
    res["steps_by_mode"] = acc
    res["total_steps"] = acc.sum(0, keepdim=True)
    return res


@B._on_stream
def hilbert_map(lattice, R: int, thr: float, passes: int, shift: int, trace_fn, *, stream=None):
    """The paper's own refinement loop (reading A17): orchestration only, every step is a
    libqsl call.  Level-0 samples ordered along the Hilbert curve; per pass a refinement on the curve (a new sample halfway
    along the curve wherever the field-line length of two successive samples differs by more than `thr`) and, if
    `shift` != 0, the same on the curve shifted by `shift` fine cells, after which the samples go back to the original
    order.  trace_fn(seeds CUDA float64 (m, 3)) -> (L, Q), CUDA float64 (m,) each - e.g. a closure over qsl_trace; every
    batch it receives is ordered along the (shifted) curve, so the closure may pass QSL_FLAG_NO_SORT.

    Returns dict(keys int64 (n,), coords int32 (n, ndim), L, Q, counts): the samples in curve order and the number of
    samples after level 0 and after every (sub-)pass.  Feed keys and Q to qsl_hilbert_convert for the rectilinear map.
    """
    nd = int(lattice.ndim)
    bits = B.qsl_hilbert_bits(lattice, R)
    coords, seeds = B.qsl_hilbert_level0(lattice, R, stream=stream)
    keys = B.qsl_hilbert_keys(coords, bits, 0, stream=stream)
    perm = B.qsl_sort_keys64(keys, bits * nd, stream=stream)
    coords = B.qsl_gather(perm, coords, stream=stream)
    seeds = B.qsl_gather(perm, seeds, stream=stream)
    L, Q = trace_fn(seeds)
    counts = [int(keys.numel())]
    for _ in range(passes):
        for sh in ((0, shift) if shift else (0,)):
            if sh:
                ks = B.qsl_hilbert_keys(coords, bits + 1, sh, stream=stream)
                perm = B.qsl_sort_keys64(ks, (bits + 1) * nd, stream=stream)
                keys, coords, L, Q = (B.qsl_gather(perm, t, stream=stream) for t in (keys, coords, L, Q))
            else:
                ks = keys
            left, nc, ns = B.qsl_hilbert_refine(lattice, R, sh, ks, L, thr, stream=stream)
            if left.numel():
                nL, nQ = trace_fn(ns.contiguous())
                nk = B.qsl_hilbert_keys(nc.contiguous(), bits, 0, stream=stream)
                keys = B.qsl_hilbert_merge(left, keys, nk, stream=stream)
                coords = B.qsl_hilbert_merge(left, coords, nc.contiguous(), stream=stream)
                L = B.qsl_hilbert_merge(left, L, nL.contiguous(), stream=stream)
                Q = B.qsl_hilbert_merge(left, Q, nQ.contiguous(), stream=stream)
            if sh:
                kk = keys.clone()
                perm = B.qsl_sort_keys64(kk, bits * nd, stream=stream)
                coords, L, Q = (B.qsl_gather(perm, t, stream=stream) for t in (coords, L, Q))
                keys = kk
            counts.append(int(keys.numel()))
    return dict(keys=keys, coords=coords, L=L, Q=Q, counts=counts)


def trace_host(field, seeds_host: torch.Tensor, params, *, outputs=("end_f", "end_b", "L", "q_perp", "q_bnd", "face_f", "face_b",
                                                                    "status"), chunks=None, host_out=None):
    """qsl_trace for seeds and results that live in (pinned) HOST memory: orchestration only.  The seeds are cut into
    `chunks` pieces that alternate between two streams, so that the host-to-device copy of a piece and the device-to-host
    copy of its results overlap the trace kernels of its neighbours (the copy engines are otherwise idle during the trace,
    and the trace kernel's ragged tail is filled by the next piece).  chunks = None: one piece per 4 M lines, at most 8 -
measured on a B200, a piece of fewer than a few million lines costs more in kernel efficiency (two half-empty persistent
grids side by side) than the overlapped copies save: cfg2, 1.05 M lines: 18.0 ms in one piece, 20.2 ms in four; cfg4, 16.8 M
lines: 757 ms in one piece, 725 ms in four.  Returns a dict of pinned host tensors (`host_out` is
    reused if it has them).  The caller's current stream waits for both streams on return; call torch.cuda.synchronize()
    (or synchronise that stream) before reading the results on the host."""
    n = int(seeds_host.shape[0])
    host_out = {} if host_out is None else host_out
    cur = torch.cuda.current_stream()
    streams = getattr(trace_host, "_streams", None)
    if streams is None:
        streams = trace_host._streams = (torch.cuda.Stream(), torch.cuda.Stream())
    if chunks is None:
        chunks = min(8, n // 4_000_000)
    chunks = max(1, min(int(chunks), n)) if n else 1
    bounds = [n * k // chunks for k in range(chunks + 1)]
    for s in streams:
        s.wait_stream(cur)
    for k in range(chunks):
        lo, hi = bounds[k], bounds[k + 1]
        if hi == lo:
            continue
        s = streams[k & 1]
        with torch.cuda.stream(s):
            d = seeds_host[lo:hi].cuda(non_blocking=True)
            res = B.qsl_trace(field, d, params, outputs=outputs)
            for name in outputs:
                t = res[name]
                h = host_out.get(name)
                if h is None or h.shape[0] != n or h.dtype != t.dtype:
                    h = host_out[name] = torch.empty((n,) + tuple(t.shape[1:]), dtype=t.dtype).pin_memory()
                h[lo:hi].copy_(t, non_blocking=True)
                t.record_stream(s)
            d.record_stream(s)
    for s in streams:
        cur.wait_stream(s)
    return host_out

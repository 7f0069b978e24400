"""Level loop of the adaptive refinement: orchestration only, every step is a libqsl call.

PAPER.md:194-200: sample the region on a rectilinear grid, find where the field-line length jumps, sample those places
more finely, repeat.  Reading A11: level 0 is traced L-only, FLEDGE = Sobel magnitude of L, tau = the p-th
percentile (nearest rank) of the level-0 FLEDGE map, reused at every level; cells with S > tau are split 2x per axis and
their children traced with Q; the children's L feeds the sparse FLEDGE map of the next level.
"""
from __future__ import annotations

import torch

from . import binding as B


def adaptive_map(field, lattice, seeds0, params_L, params_LQ, n_levels: int, p: float, *, stream=None,
                 outputs=("L", "q_perp", "q_bnd", "status"), max_children=None):
    """Runs level 0 (dense, `params_L`) and `n_levels` refinement levels (`params_LQ`).

    seeds0: CUDA float64 (n0*n1*n2, 3) level-0 seeds in dense index order.
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
        res["out"].append(o)
        Ls.append(o["L"])
        if level + 1 < n_levels:
            S = B.qsl_fledge_sparse(lattice, level + 1, L0, res["coords"], Ls, res["child_base"], stream=stream)
            res["S"].append(S)
            coords = cc
    res["steps_by_mode"] = acc
    res["total_steps"] = acc.sum(0, keepdim=True)
    return res

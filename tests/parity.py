"""Helpers of the GPU parity tests: run the CUDA path (through the C ABI binding) and the CPU oracle on the same
seeded inputs and compare element by element with the gates of BASELINE.json `north_star`."""
import math

import numpy as np
import torch

import oracle
import paper_1609_00724_b200 as qsl


def gpu_field(grid, B, sample_type, interp_mode, order=1, geometry=0):
    """qsl_field_create from host cubes."""
    dev = [torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64).reshape(-1)).cuda() for a in B]
    st = qsl.QSL_F32 if sample_type in ("f32", qsl.QSL_F32) and sample_type != qsl.QSL_F64 else qsl.QSL_F64
    kw = dict(sample_type=st, interp_mode=interp_mode, interp_order=0 if order == 1 else order, geometry=geometry)
    if grid.stretched:
        return qsl.qsl_field_create(grid.nx, grid.ny, grid.nz, *dev, xs=grid.xs, ys=grid.ys, zs=grid.zs, **kw)
    return qsl.qsl_field_create(grid.nx, grid.ny, grid.nz, *dev, lo=grid.lo, hi=grid.hi, **kw)


def cpu_field(grid, B, sample_type, interp_mode, order=1, geometry=0):
    st = oracle.F32 if sample_type in ("f32", 0) else oracle.F64
    return oracle.Field(grid, B, st, interp_mode, order, geometry)


def run_both(grid, B, sample_type, seeds, box_lo, box_hi, *, interp_mode=0, mode=1, method=0, step_frac=0.25,
             max_steps=1 << 30, max_length=math.inf, null_eps=1e-12, flags=0, want_dev=False, tol=1e-2, order=1, geometry=0):
    st = "f32" if sample_type in ("f32", 0) else "f64"
    fg = gpu_field(grid, B, st, interp_mode, order, geometry)
    fc = cpu_field(grid, B, st, interp_mode, order, geometry)
    params = qsl.make_trace_params(box_lo, box_hi, method=method, step_frac=step_frac, mode=mode, max_length=max_length,
                                   max_steps=max_steps, null_eps=null_eps, flags=flags, tol=tol)
    outs = qsl.DEFAULT_OUTPUTS + (("dev_f", "dev_b") if want_dev else ())
    tot = torch.zeros(1, dtype=torch.int64, device="cuda")
    g = qsl.qsl_trace(fg, torch.from_numpy(np.ascontiguousarray(seeds)).cuda(), params, outputs=outs, total_steps=tot)
    torch.cuda.synchronize()
    g = {k: v.cpu().numpy() for k, v in g.items()}
    g["total_steps"] = int(tot.item())
    for k in ("status", "nsteps_f", "nsteps_b"):
        g[k] = g[k].view(np.uint32)
    c = oracle.trace(fc, seeds, box_lo, box_hi, method=method, step_frac=step_frac, mode=mode, max_length=max_length,
                     max_steps=max_steps, null_eps=null_eps, want_dev=want_dev, tol=tol)
    fg.destroy()
    return g, c


def compare_trace(g, c, box_lo, box_hi, *, with_q=True, frac=0.999, label=""):
    """north_star gates: end points <= 1e-9 x box size, L and Q <= 1e-8 relative, for >= 99.9 % of seeds;
    |delta log10 Q| <= 1e-3 for every seed with Q < 1e8; per-line nsteps equal for >= 99.9 %; integer outputs of the
    lines that took the same number of steps are bit-exact."""
    n = len(c["L"])
    if n == 0:
        return {}
    box = float(np.max(np.asarray(box_hi) - np.asarray(box_lo)))
    same_steps = (g["nsteps_f"] == c["nsteps_f"]) & (g["nsteps_b"] == c["nsteps_b"])
    rep = {"n": n, "same_steps": float(same_steps.mean())}
    assert same_steps.mean() >= frac, (label, rep)
    assert np.array_equal(g["status"][same_steps], c["status"][same_steps]), label
    assert np.array_equal(g["face_f"][same_steps], c["face_f"][same_steps]), label
    assert np.array_equal(g["face_b"][same_steps], c["face_b"][same_steps]), label
    bad = (c["status"] & (oracle.ST_SEED_OUTSIDE | oracle.ST_NULL_AT_SEED)) != 0
    assert np.array_equal(np.isnan(g["L"]), np.isnan(c["L"])), label
    ok = ~bad
    e_end = np.maximum(np.abs(g["end_f"] - c["end_f"]).max(1), np.abs(g["end_b"] - c["end_b"]).max(1))[ok]
    rep["end_max"] = float(e_end.max()) if ok.any() else 0.0
    rep["end_ok"] = float((e_end <= 1e-9 * box).mean()) if ok.any() else 1.0
    assert rep["end_ok"] >= frac, (label, rep)
    rl = np.abs(g["L"][ok] - c["L"][ok]) / np.maximum(np.abs(c["L"][ok]), 1e-300)
    rl = np.where(c["L"][ok] == g["L"][ok], 0.0, rl)
    rep["L_ok"] = float((rl <= 1e-8).mean()) if ok.any() else 1.0
    assert rep["L_ok"] >= frac, (label, rep)
    if with_q:
        for key in ("q_perp", "q_bnd"):
            qc, qg = c[key][ok], g[key][ok]
            fin = np.isfinite(qc)
            assert np.array_equal(np.isfinite(qg), fin), (label, key)
            rq = np.abs(qg[fin] - qc[fin]) / np.abs(qc[fin])
            rep[key + "_ok"] = float((rq <= 1e-8).mean()) if fin.any() else 1.0
            assert rep[key + "_ok"] >= frac, (label, rep)
            small = fin & (np.abs(qc) < 1e8) & (qc > 0)
            dl = np.abs(np.log10(np.abs(qg[small])) - np.log10(qc[small]))
            rep[key + "_dlog_max"] = float(dl.max()) if small.any() else 0.0
            assert rep[key + "_dlog_max"] <= 1e-3, (label, rep)
    assert g["total_steps"] == int(g["nsteps_f"].astype(np.int64).sum() + g["nsteps_b"].astype(np.int64).sum()), label
    return rep


# ------------------------------------------------------------------------------------------------- level loop (a9)
def oracle_pipeline(cfg, sample_type=None, interp_mode=0):
    """The adaptive level loop (O6, O7 + traces) run entirely by the oracle.  Returns per-level products."""
    st = sample_type or cfg["sample_type"]
    fc = cpu_field(cfg["grid"], cfg["B"], st, interp_mode)
    lat = cfg["lattice"]; ndim = lat.ndim
    kw = dict(max_steps=cfg["max_steps"], step_frac=cfg["step_frac"], null_eps=cfg["null_eps"])
    o0 = oracle.trace(fc, cfg["seeds"], cfg["box_lo"], cfg["box_hi"], mode=oracle.TRACE_L, **kw)
    shape = tuple(int(v) for v in lat.n[:ndim][::-1])
    L0 = o0["L"].reshape(shape)
    S0 = oracle.fledge_dense(L0, ndim).reshape(-1)
    tau = oracle.select(S0, cfg["p"])
    n = lat.count
    c0 = np.stack(np.unravel_index(np.arange(n), shape), 1)[:, ::-1].astype(np.uint32)   # dense index order
    res = dict(L0=o0["L"], S0=S0, tau=tau, coords=[c0], seeds=[cfg["seeds"]], out=[o0], S=[S0])
    coords, S, Ls = c0, S0, [o0["L"]]
    for level in range(cfg["levels"]):
        cc, cs = oracle.refine(ndim, level, coords, S, tau, lat)
        res["coords"].append(cc); res["seeds"].append(cs)
        if len(cc) == 0:
            break
        o = oracle.trace(fc, cs, cfg["box_lo"], cfg["box_hi"], mode=oracle.TRACE_LQ, **kw)
        res["out"].append(o); Ls.append(o["L"])
        if level + 1 < cfg["levels"]:
            S = oracle.fledge_sparse(ndim, lat.n[:ndim], level + 1, o0["L"], res["coords"], Ls)
            res["S"].append(S); coords = cc
    return res

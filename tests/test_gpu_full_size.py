"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default flags: Morton order,
persistent work queue, cell-table kernel).  The oracle cannot trace 10^6 - 10^8 lines in test time, so it traces a sample
of the seeds one by one (every k-th seed plus one contiguous run that spans several warps and a ragged tail) and the
sampled outputs are compared element by element; the remaining outputs are checked through properties that hold at any
size.  The streaming stages (FLEDGE, threshold, refine) are compared in full: the oracle's C loops finish in seconds."""
import numpy as np
import pytest
import torch

import oracle
import paper_1609_00724_b200 as qsl
import qsl_inputs as qi
from tests.parity import compare_trace, cpu_field, gpu_field

pytestmark = pytest.mark.gpu


def _sample(n, stride, run=4133):
    idx = np.unique(np.concatenate([np.arange(0, n, stride), np.arange(n // 3, min(n, n // 3 + run))]))
    return idx


def _gpu_trace(cfg, mode):
    fg = gpu_field(cfg["grid"], cfg["B"], cfg["sample_type"], 0)
    p = qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], mode=mode, step_frac=cfg["step_frac"], max_steps=cfg["max_steps"],
                              null_eps=cfg["null_eps"])
    tot = torch.zeros(1, dtype=torch.int64, device="cuda")
    seeds = torch.from_numpy(cfg["seeds"]).cuda()
    g = qsl.qsl_trace(fg, seeds, p, total_steps=tot)
    torch.cuda.synchronize()
    return fg, g, int(tot.item())


def _pick(g, idx):
    out = {k: v[torch.from_numpy(idx).cuda()].cpu().numpy() for k, v in g.items()}
    for k in ("status", "nsteps_f", "nsteps_b"):
        out[k] = out[k].view(np.uint32)
    out["total_steps"] = int(out["nsteps_f"].astype(np.int64).sum() + out["nsteps_b"].astype(np.int64).sum())
    return out


def _properties(cfg, g, total_steps, with_q):
    """Checks that need no oracle and hold for every line, whatever the size."""
    lo = torch.tensor(cfg["box_lo"], dtype=torch.float64, device="cuda")
    hi = torch.tensor(cfg["box_hi"], dtype=torch.float64, device="cuda")
    st = g["status"]
    assert int((st & (qsl.QSL_ST_SEED_OUTSIDE | qsl.QSL_ST_NULL_AT_SEED)).count_nonzero()) == 0
    assert int((st & ~0x7f).count_nonzero()) == 0          # only the documented QSL_ST_* bits (no internal record flag leaks)
    # every line was landed (or stalled / capped): a face other than 255 goes with a snapped end, face 255 with a status bit
    for face, bits in ((g["face_f"], qsl.QSL_ST_STALL_F | qsl.QSL_ST_CAP_F), (g["face_b"], qsl.QSL_ST_STALL_B | qsl.QSL_ST_CAP_B)):
        assert bool((((face == 255) == ((st & bits) != 0))).all())
        assert bool((face[face != 255] <= 5).all())
    assert total_steps == int(g["nsteps_f"].to(torch.int64).sum() + g["nsteps_b"].to(torch.int64).sum())
    seeds = torch.from_numpy(cfg["seeds"]).cuda()
    for end, face, ns in ((g["end_f"], g["face_f"], g["nsteps_f"]), (g["end_b"], g["face_b"], g["nsteps_b"])):
        # ends inside the trace box; a line leaving through an edge or corner lands on the first face its chord crosses
        # (reading A4) and may then poke out of a second face by O(h^2 x curvature) - same in the oracle
        tol = 1e-5 * float((hi - lo).max())
        assert bool(((end >= lo - tol) & (end <= hi + tol)).all())
        assert float(((end >= lo) & (end <= hi)).all(1).double().mean()) > 0.9999
        landed = face != 255
        ax = (face.to(torch.int64) >> 1).clamp(max=2)
        bound = torch.where((face & 1).bool(), hi[ax], lo[ax])
        coord = end.gather(1, ax[:, None])[:, 0]
        assert bool((coord[landed] == bound[landed]).all())                   # snapped exactly onto the recorded face
        assert bool((ns[landed] >= 1).all())
    # a curve is at least as long as its chords: |end_f - seed| + |seed - end_b| <= L (to rounding)
    chord = (g["end_f"] - seeds).norm(dim=1) + (g["end_b"] - seeds).norm(dim=1)
    assert bool((g["L"] >= chord * (1 - 1e-12) - 1e-12).all())
    # L is bounded by the affine length: |b_interp| <= 1 under normalise-first, h = 0.25 cell per step
    hmin = min((h - l) / (n - 1) for l, h, n in zip(cfg["grid"].lo, cfg["grid"].hi, (cfg["grid"].nx, cfg["grid"].ny, cfg["grid"].nz)))
    nst = (g["nsteps_f"].to(torch.float64) + g["nsteps_b"].to(torch.float64))
    assert bool((g["L"] <= nst * (cfg["step_frac"] * hmin) * (1 + 1e-6)).all())   # fp32 samples: |b^| = 1 +- 6e-8
    open_expected = ((g["face_f"] != 4) & (g["face_f"] != 255)) | ((g["face_b"] != 4) & (g["face_b"] != 255))
    assert bool((((st & qsl.QSL_ST_OPEN) != 0) == open_expected).all())
    if with_q:
        capped = (st & (qsl.QSL_ST_CAP_F | qsl.QSL_ST_CAP_B | qsl.QSL_ST_STALL_F | qsl.QSL_ST_STALL_B)) != 0
        q = g["q_perp"][~capped]
        assert bool(torch.isfinite(q).all())
        # Q >= 2 for an exactly area-preserving map; the interpolated field is solenoidal only to O(cell^2) (pin P5)
        assert float((q >= 2 * (1 - 5e-2)).double().mean()) > 0.99


def _oracle_sample(cfg, idx, mode):
    fc = cpu_field(cfg["grid"], cfg["B"], cfg["sample_type"], 0)
    return fc, oracle.trace(fc, cfg["seeds"][idx], cfg["box_lo"], cfg["box_hi"], mode=mode, step_frac=cfg["step_frac"],
                            max_steps=cfg["max_steps"], null_eps=cfg["null_eps"])


def test_cfg2_full_size_sampled():
    """BASELINE.json configs[1]: 1 047 959 photospheric seeds, fp64 128^3, L + Q (the default bench workload)."""
    cfg = qi.make_config("cfg2")
    fg, g, tot = _gpu_trace(cfg, qsl.QSL_TRACE_LQ)
    _properties(cfg, g, tot, True)
    idx = _sample(len(cfg["seeds"]), 61)
    _, c = _oracle_sample(cfg, idx, oracle.TRACE_LQ)
    rep = compare_trace(_pick(g, idx), c, cfg["box_lo"], cfg["box_hi"], label="cfg2 full")
    assert rep["n"] > 20000
    # P7: a closed line that starts where Bz > 0 ends where Bz < 0
    q, r = cfg["charges"]
    closed = (g["face_f"] == 4) & (g["face_b"] == 4)
    sub = torch.nonzero(closed)[:: 97, 0].cpu().numpy()
    ends = torch.where((g["nsteps_f"] > 1)[:, None], g["end_f"], g["end_b"])[torch.from_numpy(sub).cuda()].cpu().numpy()
    bz0 = qi.quadrupole_B(cfg["seeds"][sub], q, r)[:, 2]
    bz1 = qi.quadrupole_B(ends, q, r)[:, 2]
    assert np.mean(np.sign(bz0) == -np.sign(bz1)) > 0.99
    fg.destroy()


def test_cfg4_full_size_sampled():
    """BASELINE.json configs[3]: 256^3 seeds through the fp32-sampled 256^3 LFFF field, L + Q."""
    cfg = qi.make_config("cfg4")
    fg, g, tot = _gpu_trace(cfg, qsl.QSL_TRACE_LQ)
    _properties(cfg, g, tot, True)
    idx = _sample(len(cfg["seeds"]), 2039)
    _, c = _oracle_sample(cfg, idx, oracle.TRACE_LQ)
    rep = compare_trace(_pick(g, idx), c, cfg["box_lo"], cfg["box_hi"], label="cfg4 full")
    assert rep["n"] > 12000
    fg.destroy()


@pytest.mark.parametrize("name", ["cfg3", "cfg5"])
def test_refinement_configs_full_size_level0(name):
    """BASELINE.json configs[2] / [4] at full size: the L-only level-0 pass sampled against the oracle, then FLEDGE,
    threshold and the first refinement compared in full with the oracle fed the same inputs (bit-exact seed sets)."""
    cfg = qi.make_config(name)
    lat = cfg["lattice"]; ndim = lat.ndim
    fg, g, tot = _gpu_trace(cfg, qsl.QSL_TRACE_L)
    _properties(cfg, g, tot, False)
    n = len(cfg["seeds"])
    idx = _sample(n, 4099 if name == "cfg5" else 173)
    _, c = _oracle_sample(cfg, idx, oracle.TRACE_L)
    compare_trace(_pick(g, idx), c, cfg["box_lo"], cfg["box_hi"], with_q=False, label=name + " level 0")
    shape = tuple(int(v) for v in lat.n[:ndim][::-1])
    L0 = g["L"]
    S = qsl.qsl_fledge_dense(L0.view(shape), ndim)
    L0h = L0.cpu().numpy()
    Sref = oracle.fledge_dense(L0h.reshape(shape), ndim)
    Sg = S.cpu().numpy()
    assert np.array_equal(np.isnan(Sg), np.isnan(Sref))
    fin = np.isfinite(Sref)
    # differences of O(1) lengths: the error bound is absolute, 32 (3-D) stencil weights x eps x max L
    assert np.max(np.abs(Sg[fin] - Sref[fin])) <= 1e-13 * 32 * float(np.nanmax(L0h))
    tau = qsl.qsl_select(S.view(-1), cfg["p"])
    tau_ref = oracle.select(Sg, cfg["p"])
    assert float(tau.item()) == tau_ref
    max_flagged = n - int(np.ceil(cfg["p"] * n))
    cc, cs, cb = qsl.qsl_refine(lat, 0, None, S.view(-1), tau, capacity=(max_flagged + 8) << ndim)
    cc, cs = cc.cpu().numpy().view(np.uint32), cs.cpu().numpy()
    # the oracle refines the same cells chunk by chunk of the input order (its output buffers are 2^D x the chunk)
    Sflat, at, chunk = Sg.reshape(-1), 0, 1 << 22
    for lo in range(0, n, chunk):
        k = np.arange(lo, min(n, lo + chunk))
        c0 = np.stack(np.unravel_index(k, shape), 1)[:, ::-1].astype(np.uint32)
        cc_ref, cs_ref = oracle.refine(ndim, 0, c0, Sflat[lo:lo + chunk], tau_ref, lat)
        m = len(cc_ref)
        assert np.array_equal(cc[at:at + m], cc_ref) and np.array_equal(cs[at:at + m], cs_ref), (name, lo)
        at += m
    assert at == len(cc)
    flagged = int((cb >= 0).sum())
    assert flagged << ndim == at and 0 < flagged <= max_flagged
    fg.destroy()


@pytest.mark.parametrize("name", ["cfg3", "cfg5"])
def test_refined_levels_full_size_sampled(name):
    """BASELINE.json configs[2] / [4] at full size, the product they deliver: `adaptive_map` as
    bench.py runs it (level 0 L-only, FLEDGE, p95, 4 / 3 levels), and at every refined level the L + Q trace of a sample
    of the children (every k-th child plus one contiguous run) compared element by element with the oracle tracing the
    same seed positions, at the north_star gates (99.9 %).  The children sit on the quasi-connectivity boundaries."""
    cfg = qi.make_config(name)
    lat = cfg["lattice"]
    fg = gpu_field(cfg["grid"], cfg["B"], cfg["sample_type"], 0)
    fc = cpu_field(cfg["grid"], cfg["B"], cfg["sample_type"], 0)
    mk = lambda m: qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], mode=m, step_frac=cfg["step_frac"],
                                         max_steps=cfg["max_steps"], null_eps=cfg["null_eps"])
    picked = {}

    def on_level(level, coords, seeds, out):
        n = int(seeds.shape[0])
        idx = _sample(n, max(1, n // 6000))
        picked[level] = (n, seeds[torch.from_numpy(idx).cuda()].cpu().numpy(), _pick(out, idx))

    res = qsl.adaptive_map(fg, lat, torch.from_numpy(cfg["seeds"]).cuda(), mk(qsl.QSL_TRACE_L), mk(qsl.QSL_TRACE_LQ),
                           cfg["levels"], cfg["p"], outputs=qsl.DEFAULT_OUTPUTS, on_level=on_level, keep=("L",))
    torch.cuda.synchronize()
    assert sorted(picked) == list(range(1, cfg["levels"] + 1)), "every level must have refined"
    sizes = [picked[l][0] for l in sorted(picked)]
    assert all(0 < m <= (1 << lat.ndim) * k for k, m in zip([len(cfg["seeds"])] + sizes, sizes)), sizes
    assert sum(int(s.shape[0]) for s in res["seeds"][1:]) == sum(sizes)
    for level in sorted(picked):
        n, seeds, g = picked[level]
        c = oracle.trace(fc, seeds, cfg["box_lo"], cfg["box_hi"], mode=oracle.TRACE_LQ, step_frac=cfg["step_frac"],
                         max_steps=cfg["max_steps"], null_eps=cfg["null_eps"])
        rep = compare_trace(g, c, cfg["box_lo"], cfg["box_hi"], label="%s level %d of %d children" % (name, level, n))
        assert rep["n"] >= 6000
    fg.destroy()


@pytest.mark.parametrize("name,stride", [("cfg2", 97), ("cfg4", 4093)])
@pytest.mark.parametrize("method", ["euler", "ck45"])
def test_full_size_sampled_with_the_papers_integrators(name, stride, method):
    """The paper's own steppers at full size (fixed-step Euler; adaptive Cash-Karp at tolerance 1e-2,
    readings A5 / A16), L + Q, sampled against the oracle at the north_star gates; for the adaptive stepper the per-line
    step counts must agree too (the controller takes the oracle's accept / reject / double decisions)."""
    cfg = qi.make_config(name)
    m = qsl.QSL_EULER if method == "euler" else qsl.QSL_CK45
    step_frac = 0.2 if method == "euler" else cfg["step_frac"]       # about five samples per cell
    fg = gpu_field(cfg["grid"], cfg["B"], cfg["sample_type"], 0)
    p = qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], mode=qsl.QSL_TRACE_LQ, method=m, step_frac=step_frac,
                              max_steps=cfg["max_steps"], null_eps=cfg["null_eps"], tol=1e-2)
    tot = torch.zeros(1, dtype=torch.int64, device="cuda")
    g = qsl.qsl_trace(fg, torch.from_numpy(cfg["seeds"]).cuda(), p, total_steps=tot)
    torch.cuda.synchronize()
    assert int(tot.item()) == int(g["nsteps_f"].to(torch.int64).sum() + g["nsteps_b"].to(torch.int64).sum())
    idx = _sample(len(cfg["seeds"]), stride, run=1031)
    fc = cpu_field(cfg["grid"], cfg["B"], cfg["sample_type"], 0)
    c = oracle.trace(fc, cfg["seeds"][idx], cfg["box_lo"], cfg["box_hi"], mode=oracle.TRACE_LQ, method=m, step_frac=step_frac,
                     max_steps=cfg["max_steps"], null_eps=cfg["null_eps"], tol=1e-2)
    rep = compare_trace(_pick(g, idx), c, cfg["box_lo"], cfg["box_hi"], label="%s full %s" % (name, method))
    assert rep["n"] > 5000 and rep["same_steps"] >= 0.999
    fg.destroy()

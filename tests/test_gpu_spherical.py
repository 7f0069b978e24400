"""GPU parity of the spherical geometry (SURVEY.md 8(f) f4; PAPER.md:83-87 eq. 2, :125-135 eq. 6-7, :153-156 eq. 8;
reading A19) against the CPU oracle at the north_star gates; the box size of the end-point gate is the largest extent of
the (phi, theta, r) trace box."""
import math

import numpy as np
import pytest
import torch

import oracle
import paper_1609_00724_b200 as qsl
import qsl_inputs as qi
from tests.parity import compare_trace, run_both

pytestmark = pytest.mark.gpu
SPH = qsl.QSL_SPHERICAL


def _cubes(g, f):
    P, T, R = np.meshgrid(g.xs, g.ys, g.zs, indexing="ij")
    return [np.ascontiguousarray(np.transpose(c * np.ones_like(P), (2, 1, 0))) for c in f(P, T, R)]


def _dipole_plus(p, t, r):
    """Dipole plus a small non-axisymmetric octupole-like part, so that B_phi and the phi-derivatives are exercised."""
    return (0.15 * np.sin(3 * p) * np.cos(t) / r ** 4, -np.cos(t) / r ** 3 + 0.1 * np.cos(3 * p) * np.sin(2 * t) / r ** 4,
            2 * np.sin(t) / r ** 3 + 0.2 * np.cos(3 * p) * np.cos(t) ** 2 / r ** 4)


KERNELS = [0, qsl.QSL_FLAG_KERNEL_V1]      # cell-table kernel (default) and gather kernel: both carry the geometry


@pytest.mark.parametrize("flags", KERNELS)
def test_sph_monopole_q_two(flags):
    g = qi.Grid.uniform((9, 11, 33), (0.1, -0.3, 1.0), (0.9, 0.5, 3.0))
    B = _cubes(g, lambda p, t, r: (0 * r, 0 * r, 1 / r ** 2))
    seeds = np.array([[0.33, 0.11, g.zs[7]], [0.71, -0.22, g.zs[20]], [0.5, 0.4, g.zs[1]], [0.2, 0.0, 1.0], [0.2, 0.0, 3.0]])
    gg, c = run_both(g, B, "f64", seeds, g.lo, g.hi, geometry=SPH, flags=flags)
    compare_trace(gg, c, g.lo, g.hi, frac=1.0, label="monopole")
    assert np.abs(gg["q_perp"] - 2).max() < 1e-10 and np.abs(gg["L"] - 2).max() < 1e-12


@pytest.mark.parametrize("flags", KERNELS)
@pytest.mark.parametrize("st", ["f64", "f32"])
@pytest.mark.parametrize("mode", [qsl.QSL_TRACE_LQ, qsl.QSL_TRACE_L])
def test_sph_wedge_field(st, mode, flags):
    g = qi.Grid.uniform((48, 40, 44), (0.0, -0.9, 1.0), (2.0, 0.9, 2.4))
    B = _cubes(g, _dipole_plus)
    rng = np.random.default_rng(5)
    n = 4000
    seeds = np.stack([rng.uniform(0.1, 1.9, n), rng.uniform(-0.8, 0.8, n), rng.uniform(1.0, 2.2, n)], 1)
    seeds[:500, 2] = 1.0                                                      # photospheric seeds
    gg, c = run_both(g, B, st, seeds, g.lo, g.hi, geometry=SPH, mode=mode, max_steps=50000, flags=flags)
    rep = compare_trace(gg, c, g.lo, g.hi, with_q=mode == qsl.QSL_TRACE_LQ, label="wedge %s" % st)
    assert rep["same_steps"] >= 0.999
    assert (c["face_f"] == 4).mean() > 0.2 and (c["status"] & oracle.ST_OPEN).mean() > 0.05      # closed and open lines


@pytest.mark.parametrize("flags", KERNELS)
@pytest.mark.parametrize("mode", [qsl.QSL_TRACE_LQ, qsl.QSL_TRACE_L])
@pytest.mark.parametrize("tol", [1e-2, 1e-5])
def test_sph_wedge_cash_karp(mode, tol, flags):
    """The paper's own workload class: a spherical wedge traced with the adaptive Cash-Karp stepper (PAPER.md:141-143,
    :232-254).  Same controller decisions on both sides (reading A16), so per-line step counts agree."""
    g = qi.Grid.uniform((48, 40, 44), (0.0, -0.9, 1.0), (2.0, 0.9, 2.4))
    B = _cubes(g, _dipole_plus)
    rng = np.random.default_rng(6)
    n = 3000
    seeds = np.stack([rng.uniform(0.1, 1.9, n), rng.uniform(-0.8, 0.8, n), rng.uniform(1.0, 2.2, n)], 1)
    seeds[:400, 2] = 1.0
    gg, c = run_both(g, B, "f64", seeds, g.lo, g.hi, geometry=SPH, mode=mode, max_steps=50000, method=qsl.QSL_CK45, tol=tol,
                     flags=flags)
    rep = compare_trace(gg, c, g.lo, g.hi, with_q=mode == qsl.QSL_TRACE_LQ, label="wedge ck45 tol %g" % tol)
    assert rep["same_steps"] >= 0.999
    # the monopole with the adaptive stepper: radial lines, Q = 2
    g = qi.Grid.uniform((9, 11, 33), (0.1, -0.3, 1.0), (0.9, 0.5, 3.0))
    B = _cubes(g, lambda p, t, r: (0 * r, 0 * r, 1 / r ** 2))
    seeds = np.array([[0.33, 0.11, g.zs[7]], [0.71, -0.22, g.zs[20]], [0.5, 0.4, g.zs[1]]])
    gg, c = run_both(g, B, "f64", seeds, g.lo, g.hi, geometry=SPH, method=qsl.QSL_CK45, tol=tol, flags=flags)
    compare_trace(gg, c, g.lo, g.hi, frac=1.0, label="monopole ck45")
    assert np.abs(gg["q_perp"] - 2).max() < 1e-9 and np.abs(gg["L"] - 2).max() < 1e-11


@pytest.mark.parametrize("mode", [qsl.QSL_TRACE_LQ, qsl.QSL_TRACE_L])
@pytest.mark.parametrize("method", [qsl.QSL_RK4, qsl.QSL_EULER])
def test_sph_wedge_fp32_arithmetic(mode, method):
    """QSL_ARITH_F32 in spherical geometry (the cell-frame kernel with the frame's radius and latitude sin / cos): the gates
    of reading A6 against the fp64 oracle on the same fp32-rounded samples."""
    from tests.test_gpu_trace_f32 import compare_f32
    g = qi.Grid.uniform((48, 40, 44), (0.0, -0.9, 1.0), (2.0, 0.9, 2.4))
    B = _cubes(g, _dipole_plus)
    rng = np.random.default_rng(7)
    n = 4000
    seeds = np.stack([rng.uniform(0.1, 1.9, n), rng.uniform(-0.8, 0.8, n), rng.uniform(1.0, 2.2, n)], 1)
    seeds[:500, 2] = 1.0
    dev = [torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64).reshape(-1)).cuda() for a in B]
    fg = qsl.qsl_field_create(g.nx, g.ny, g.nz, *dev, lo=g.lo, hi=g.hi, sample_type=qsl.QSL_F32, geometry=SPH,
                              layout=qsl.QSL_LAYOUT_CELL_TABLES_BOTH)
    kw = dict(method=method, mode=mode, max_steps=50000, step_frac=0.2 if method == qsl.QSL_EULER else 0.25)
    tot = torch.zeros(1, dtype=torch.int64, device="cuda")
    res = qsl.qsl_trace(fg, torch.from_numpy(seeds).cuda(), qsl.make_trace_params(g.lo, g.hi, arith=qsl.QSL_ARITH_F32, **kw),
                        total_steps=tot)
    torch.cuda.synchronize()
    gg = {k: v.cpu().numpy() for k, v in res.items()}
    gg["total_steps"] = int(tot.item())
    for k in ("status", "nsteps_f", "nsteps_b"):
        gg[k] = gg[k].view(np.uint32)
    fc = oracle.Field(g, B, oracle.F32, oracle.NORMALIZE_FIRST, oracle.TRILINEAR, oracle.SPHERICAL)
    c = oracle.trace(fc, seeds, g.lo, g.hi, **kw)
    rep = compare_f32(gg, c, g.lo, g.hi, with_q=mode == qsl.QSL_TRACE_LQ, label="sph wedge f32 arithmetic")
    assert rep["end_med"] < 1e-6 and rep["L_med"] < 1e-6
    # the fp64 table of the same field gives the fp64 result at the north_star gates
    g64 = qsl.qsl_trace(fg, torch.from_numpy(seeds).cuda(), qsl.make_trace_params(g.lo, g.hi, **kw), total_steps=tot)
    torch.cuda.synchronize()
    g64 = {k: v.cpu().numpy() for k, v in g64.items()}
    g64["total_steps"] = int(tot.item())
    for k in ("status", "nsteps_f", "nsteps_b"):
        g64[k] = g64[k].view(np.uint32)
    compare_trace(g64, c, g.lo, g.hi, with_q=mode == qsl.QSL_TRACE_LQ, label="sph wedge f32 samples, f64 arithmetic")
    fg.destroy()


def test_sph_cartesian_limit_euler_caps_inner_box():
    R0, p0, t0 = 1.0e5, 0.3, 0.2
    c0 = math.cos(t0)
    n = 33
    gc = qi.Grid.uniform((n, n, n), (-1.0, -1.0, 0.0), (1.0, 1.0, 1.0))
    Bc = qi.hyperbolic_field(gc, 2.0)
    gs = qi.Grid.uniform((n, n, n), (p0 - 1.0 / (R0 * c0), t0 - 1.0 / R0, R0), (p0 + 1.0 / (R0 * c0), t0 + 1.0 / R0, R0 + 1.0))
    rng = np.random.default_rng(17)
    sc = np.stack([rng.uniform(-0.4, 0.4, 300), rng.uniform(-0.4, 0.4, 300), rng.uniform(0.0, 0.8, 300)], 1)
    ss = np.stack([p0 + sc[:, 0] / (R0 * c0), t0 + sc[:, 1] / R0, R0 + sc[:, 2]], 1)
    # the trace box is 1e-5 rad x 1e-5 rad x 1: gate the end points per axis by scaling the angles to lengths
    for kw in (dict(), dict(flags=qsl.QSL_FLAG_KERNEL_V1), dict(method=qsl.QSL_EULER, step_frac=0.2), dict(max_steps=5),
               dict(max_length=0.3), dict(max_length=0.3, flags=qsl.QSL_FLAG_KERNEL_V1)):
        gg, c = run_both(gs, Bc, "f64", ss, gs.lo, gs.hi, geometry=SPH, **kw)
        for d in (gg, c):
            for key in ("end_f", "end_b"):
                d[key] = np.stack([(d[key][:, 0] - p0) * R0 * c0, (d[key][:, 1] - t0) * R0, d[key][:, 2] - R0], 1)
        compare_trace(gg, c, (-1, -1, 0), (1, 1, 1), label="cartesian limit " + str(kw))
    # and against the Cartesian device path itself
    gcart, _ = run_both(gc, Bc, "f64", sc, gc.lo, gc.hi)
    gsph, _ = run_both(gs, Bc, "f64", ss, gs.lo, gs.hi, geometry=SPH)
    assert np.allclose(gsph["L"], gcart["L"], rtol=2e-4) and np.allclose(gsph["q_bnd"], gcart["q_bnd"], rtol=2e-3)
    lo = (gs.lo[0] + 0.1 / (R0 * c0), gs.lo[1] + 0.2 / R0, R0 + 0.13); hi = (gs.hi[0] - 0.15 / (R0 * c0), gs.hi[1] - 0.1 / R0, R0 + 0.77)
    gg, c = run_both(gs, Bc, "f64", ss, lo, hi, geometry=SPH)
    for d in (gg, c):
        for key in ("end_f", "end_b"):
            d[key] = np.stack([(d[key][:, 0] - p0) * R0 * c0, (d[key][:, 1] - t0) * R0, d[key][:, 2] - R0], 1)
    compare_trace(gg, c, (-1, -1, 0), (1, 1, 1), label="cartesian limit inner box")


def test_sph_argument_errors():
    z = torch.ones(5 * 5 * 5, dtype=torch.float64, device="cuda")
    kw = dict(lo=(0, 0, 1), hi=(1, 1, 2), geometry=SPH)
    for bad in (dict(interp_mode=qsl.QSL_INTERP_FIRST), dict(interp_order=qsl.QSL_TRICUBIC)):
        with pytest.raises(qsl.QslError):
            qsl.qsl_field_create(5, 5, 5, z, z, z, **kw, **bad)
    with pytest.raises(qsl.QslError):
        qsl.qsl_field_create(5, 5, 5, z, z, z, xs=[0, .1, .3, .6, 1], ys=[0, .1, .3, .6, 1], zs=[1, 1.1, 1.3, 1.6, 2], geometry=SPH)
    f = qsl.qsl_field_create(5, 5, 5, z, z, z, **kw)
    seeds = torch.tensor([[0.5, 0.5, 1.5]], dtype=torch.float64, device="cuda")
    for bad in (dict(arith=qsl.QSL_ARITH_F32),):                  # fp64 samples have no fp32 table
        with pytest.raises(qsl.QslError):
            qsl.qsl_trace(f, seeds, qsl.make_trace_params((0, 0, 1), (1, 1, 2), **bad))
    # the cell-frame kernel does not carry the geometry: the flag is ignored, the result is the spherical one
    a = qsl.qsl_trace(f, seeds, qsl.make_trace_params((0, 0, 1), (1, 1, 2), flags=qsl.QSL_FLAG_KERNEL_FRAME))
    b = qsl.qsl_trace(f, seeds, qsl.make_trace_params((0, 0, 1), (1, 1, 2)))
    torch.cuda.synchronize()
    assert torch.equal(a["L"], b["L"])
    f.destroy()

"""GPU parity of the adaptive Cash-Karp 5(4) stepper (QSL_CK45; reading A16)
against the CPU oracle, element by element at the north_star gates (tests.parity.compare_trace): the power-of-two
controller takes the same accept / reject / double decisions on both sides, so per-line step counts are equal too."""
import math

import numpy as np
import pytest
import torch

import oracle
import paper_1609_00724_b200 as qsl
import qsl_inputs as qi
from tests.parity import compare_trace, run_both

pytestmark = pytest.mark.gpu
CK = qsl.QSL_CK45


@pytest.mark.parametrize("flags", [0, qsl.QSL_FLAG_NO_REFILL, qsl.QSL_FLAG_NO_SORT])
@pytest.mark.parametrize("tol", [1e-2, 1e-7])
def test_ck_cfg1_full_size(flags, tol):
    """BASELINE.json configs[0] geometry at full size (16384 seeds on the face z = 0), paper mode NORMALIZE_FIRST."""
    cfg = qi.make_config("cfg1")
    g, c = run_both(cfg["grid"], cfg["B"], "f64", cfg["seeds"], cfg["box_lo"], cfg["box_hi"], method=CK, tol=tol,
                    max_steps=cfg["max_steps"], flags=flags)
    rep = compare_trace(g, c, cfg["box_lo"], cfg["box_hi"], label="ck cfg1 tol=%g flags=%d" % (tol, flags))
    assert rep["same_steps"] >= 0.9999


def test_ck_closed_form_and_controller_exercised():
    """The CUDA path itself against the closed form (north_star) with steps large enough for the tolerance to bind."""
    cfg = qi.make_config("cfg1")
    kw = dict(interp_mode=qsl.QSL_INTERP_FIRST, method=CK, step_frac=8.0)
    g1, c1 = run_both(cfg["grid"], cfg["B"], "f64", cfg["seeds"], cfg["box_lo"], cfg["box_hi"], tol=1e-7, **kw)
    compare_trace(g1, c1, cfg["box_lo"], cfg["box_hi"], label="ck interp-first tol=1e-7")
    g2, c2 = run_both(cfg["grid"], cfg["B"], "f64", cfg["seeds"], cfg["box_lo"], cfg["box_hi"], tol=1e-2, **kw)
    compare_trace(g2, c2, cfg["box_lo"], cfg["box_hi"], label="ck interp-first tol=1e-2")
    assert g1["total_steps"] > 1.5 * g2["total_steps"]            # the tolerance, not the step cap, sets the steps
    s = cfg["seeds"]; k = 2.0
    top = np.abs(s[:, 0]) <= math.exp(-k)
    qb = np.where(top, 2 * math.cosh(2 * k), k * (s[:, 0] ** 2 + s[:, 1] ** 2) + 1 / (k * s[:, 0] ** 2))
    assert np.abs(g1["q_bnd"] / qb - 1).max() < 1e-6


@pytest.mark.parametrize("name,scale,st", [("cfg2", 1.0 / 8, "f64"), ("cfg4", 1.0 / 8, "f32"), ("cfg5", 1.0 / 16, "f32")])
@pytest.mark.parametrize("mode", [qsl.QSL_TRACE_LQ, qsl.QSL_TRACE_L])
def test_ck_configs_small(name, scale, st, mode):
    cfg = qi.make_config(name, scale)
    g, c = run_both(cfg["grid"], cfg["B"], st, cfg["seeds"], cfg["box_lo"], cfg["box_hi"], method=CK, mode=mode,
                    max_steps=cfg["max_steps"])
    compare_trace(g, c, cfg["box_lo"], cfg["box_hi"], with_q=mode == qsl.QSL_TRACE_LQ, label="ck " + name)


def test_ck_stretched_grid_caps_and_inner_box():
    g = qi.Grid.from_axes(qi.stretched_axis(40, -1, 1, 3.0), qi.stretched_axis(36, -1, 1, 0.4), qi.stretched_axis(44, 0, 1, 5.0))
    B = qi.hyperbolic_field(g, 2.0)
    rng = np.random.default_rng(22)
    seeds = np.stack([rng.uniform(-0.5, 0.5, 500), rng.uniform(-0.5, 0.5, 500), rng.uniform(0, 0.9, 500)], 1)
    lo, hi = (-1, -1, 0), (1, 1, 1)
    for interp in (0, 1):
        gg, c = run_both(g, B, "f64", seeds, lo, hi, interp_mode=interp, method=CK, tol=1e-4)
        compare_trace(gg, c, lo, hi, label="ck stretched interp=%d" % interp)
    for kw in (dict(max_steps=3), dict(max_length=0.1)):
        gg, c = run_both(g, B, "f64", seeds, lo, hi, method=CK, **kw)
        compare_trace(gg, c, lo, hi, frac=1.0, label="ck " + str(kw))
        assert np.array_equal(gg["status"], c["status"])
    gg, c = run_both(g, B, "f64", seeds, (-0.9, -0.8, 0.13), (0.85, 0.9, 0.77), method=CK)
    compare_trace(gg, c, (-0.9, -0.8, 0.13), (0.85, 0.9, 0.77), label="ck inner box")


def test_ck_argument_errors():
    cfg = qi.make_config("cfg4", 1.0 / 16)
    grid = cfg["grid"]
    dev = [torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64).reshape(-1)).cuda() for a in cfg["B"]]
    seeds = torch.from_numpy(np.ascontiguousarray(cfg["seeds"][:64])).cuda()
    f = qsl.qsl_field_create(grid.nx, grid.ny, grid.nz, *dev, lo=grid.lo, hi=grid.hi, sample_type=qsl.QSL_F32,
                             layout=qsl.QSL_LAYOUT_CELL_TABLES_BOTH)
    for kw in (dict(tol=0.0), dict(tol=float("nan")), dict(arith=qsl.QSL_ARITH_F32)):
        with pytest.raises(qsl.QslError):
            qsl.qsl_trace(f, seeds, qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], method=CK, **kw))
    # without a per-cell table (nodes-only layout) the adaptive stepper runs in the gather kernel: same result as the
    # table kernel of the same field to rounding
    a = qsl.qsl_trace(f, seeds, qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], method=CK, max_steps=cfg["max_steps"]))
    f.destroy()
    f = qsl.qsl_field_create(grid.nx, grid.ny, grid.nz, *dev, lo=grid.lo, hi=grid.hi, sample_type=qsl.QSL_F32,
                             layout=qsl.QSL_LAYOUT_NODES_ONLY)
    b = qsl.qsl_trace(f, seeds, qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], method=CK, max_steps=cfg["max_steps"]))
    torch.cuda.synchronize()
    assert torch.equal(a["nsteps_f"], b["nsteps_f"]) and torch.allclose(a["L"], b["L"], rtol=1e-10, atol=0)
    assert torch.allclose(a["q_perp"], b["q_perp"], rtol=1e-7, atol=0)
    f.destroy()


V1 = qsl.QSL_FLAG_KERNEL_V1


@pytest.mark.parametrize("name,scale,st,order", [("cfg2", 1.0 / 8, "f64", 1), ("cfg4", 1.0 / 8, "f32", 1), ("cfg2", 1.0 / 8, "f64", 2),
                                                 ("cfg2", 1.0 / 8, "f64", 3), ("cfg4", 1.0 / 8, "f32", 3)])
@pytest.mark.parametrize("mode", [qsl.QSL_TRACE_LQ, qsl.QSL_TRACE_L])
def test_ck_in_the_gather_kernel(name, scale, st, order, mode):
    """QSL_CK45 on fields without a per-cell table (QSL_FLAG_KERNEL_V1 forces the gather kernel on a trilinear field; the
    higher interpolation orders have no table at all): PAPER.md:91-93 with :141-143, the robustness checks the paper offers
    both options for."""
    cfg = qi.make_config(name, scale)
    g, c = run_both(cfg["grid"], cfg["B"], st, cfg["seeds"], cfg["box_lo"], cfg["box_hi"], method=CK, mode=mode,
                    max_steps=cfg["max_steps"], flags=V1 if order == 1 else 0, order=order, tol=1e-3)
    rep = compare_trace(g, c, cfg["box_lo"], cfg["box_hi"], with_q=mode == qsl.QSL_TRACE_LQ, label="ck gather %s order %d" % (name, order))
    assert rep["same_steps"] >= 0.999


def test_ck_in_the_gather_kernel_stretched_interp_first_caps():
    g = qi.Grid.from_axes(qi.stretched_axis(40, -1, 1, 3.0), qi.stretched_axis(36, -1, 1, 0.4), qi.stretched_axis(44, 0, 1, 5.0))
    B = qi.hyperbolic_field(g, 2.0)
    rng = np.random.default_rng(23)
    seeds = np.stack([rng.uniform(-0.5, 0.5, 500), rng.uniform(-0.5, 0.5, 500), rng.uniform(0, 0.9, 500)], 1)
    lo, hi = (-1, -1, 0), (1, 1, 1)
    for kw in (dict(interp_mode=0), dict(interp_mode=1), dict(order=3), dict(max_steps=3), dict(max_length=0.1)):
        gg, c = run_both(g, B, "f64", seeds, lo, hi, method=CK, tol=1e-4, flags=0 if "order" in kw else V1, **kw)
        compare_trace(gg, c, lo, hi, label="ck gather stretched " + str(kw))
    gg, c = run_both(g, B, "f64", seeds, (-0.9, -0.8, 0.13), (0.85, 0.9, 0.77), method=CK, flags=V1)
    compare_trace(gg, c, (-0.9, -0.8, 0.13), (0.85, 0.9, 0.77), label="ck gather inner box")

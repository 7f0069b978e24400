"""GPU parity of the higher-order interpolation schemes (reading A18): triquadratic
(Dodgson, 27 vertices) and tricubic (Keys, 64 vertices) with analytic gradients, against the CPU oracle at the north_star
gates (tests.parity.compare_trace)."""
import numpy as np
import pytest
import torch

import oracle
import paper_1609_00724_b200 as qsl
import qsl_inputs as qi
from tests.parity import compare_trace, run_both

pytestmark = pytest.mark.gpu
ORDERS = [qsl.QSL_TRIQUADRATIC, qsl.QSL_TRICUBIC]


@pytest.mark.parametrize("order", ORDERS)
@pytest.mark.parametrize("flags", [0, qsl.QSL_FLAG_NO_SORT])
def test_ho_cfg1_full_size(order, flags):
    """BASELINE.json configs[0] geometry at full size (16384 seeds on the face z = 0: the stencil hangs over the edge of
    the grid from the first step on)."""
    cfg = qi.make_config("cfg1")
    g, c = run_both(cfg["grid"], cfg["B"], "f64", cfg["seeds"], cfg["box_lo"], cfg["box_hi"], max_steps=cfg["max_steps"],
                    flags=flags, order=order, want_dev=True)
    rep = compare_trace(g, c, cfg["box_lo"], cfg["box_hi"], label="ho cfg1 order=%d" % order)
    assert rep["same_steps"] >= 0.9999
    # the hyperbolic field is linear and both kernels reproduce linear fields: in paper mode (normalise first) the field
    # traced is the interpolant of unit vectors, close to but not the analytic one - Q within 1e-2 of e^{2k} + e^{-2k}
    s = cfg["seeds"]
    top = np.abs(s[:, 0]) <= np.exp(-2.0) * 0.9
    assert np.abs(g["q_bnd"][top] / (2 * np.cosh(4.0)) - 1).max() < 1e-2


@pytest.mark.parametrize("order", ORDERS)
@pytest.mark.parametrize("name,scale,st", [("cfg2", 1.0 / 8, "f64"), ("cfg4", 1.0 / 8, "f32"), ("cfg5", 1.0 / 16, "f32")])
def test_ho_configs_small(order, name, scale, st):
    cfg = qi.make_config(name, scale)
    g, c = run_both(cfg["grid"], cfg["B"], st, cfg["seeds"], cfg["box_lo"], cfg["box_hi"], max_steps=cfg["max_steps"], order=order)
    compare_trace(g, c, cfg["box_lo"], cfg["box_hi"], label="ho %s order=%d" % (name, order))


@pytest.mark.parametrize("order", ORDERS)
def test_ho_stretched_grid_modes_and_caps(order):
    g = qi.Grid.from_axes(qi.stretched_axis(40, -1, 1, 3.0), qi.stretched_axis(36, -1, 1, 0.4), qi.stretched_axis(44, 0, 1, 5.0))
    B = qi.hyperbolic_field(g, 2.0)
    rng = np.random.default_rng(22)
    seeds = np.stack([rng.uniform(-0.5, 0.5, 500), rng.uniform(-0.5, 0.5, 500), rng.uniform(0, 0.9, 500)], 1)
    lo, hi = (-1, -1, 0), (1, 1, 1)
    g1, c = run_both(g, B, "f64", seeds, lo, hi, order=order)
    compare_trace(g1, c, lo, hi, label="ho stretched")
    g0, c0 = run_both(g, B, "f64", seeds, lo, hi, order=order, mode=qsl.QSL_TRACE_L)
    compare_trace(g0, c0, lo, hi, with_q=False, label="ho L only")
    for k in ("end_f", "end_b", "L", "nsteps_f", "nsteps_b", "face_f", "face_b"):   # pin P12 on the device: bit-identical
        assert np.array_equal(g0[k], g1[k]), k
    gg, c = run_both(g, B, "f64", seeds, lo, hi, order=order, method=qsl.QSL_EULER, step_frac=0.2)
    compare_trace(gg, c, lo, hi, label="ho stretched euler")
    for kw in (dict(max_steps=3), dict(max_length=0.1)):
        gg, c = run_both(g, B, "f64", seeds, lo, hi, order=order, **kw)
        compare_trace(gg, c, lo, hi, frac=1.0, label="ho " + str(kw))
        assert np.array_equal(gg["status"], c["status"])
    gg, c = run_both(g, B, "f64", seeds, (-0.9, -0.8, 0.13), (0.85, 0.9, 0.77), order=order)
    compare_trace(gg, c, (-0.9, -0.8, 0.13), (0.85, 0.9, 0.77), label="ho inner box")


def test_ho_argument_errors():
    z = torch.zeros(3 * 5 * 5, dtype=torch.float64, device="cuda") + 1.0
    with pytest.raises(qsl.QslError):          # tricubic needs 4 nodes per axis
        qsl.qsl_field_create(3, 5, 5, z, z, z, lo=(0, 0, 0), hi=(1, 1, 1), interp_order=qsl.QSL_TRICUBIC)
    f = qsl.qsl_field_create(3, 5, 5, z, z, z, lo=(0, 0, 0), hi=(1, 1, 1), interp_order=qsl.QSL_TRIQUADRATIC)
    seeds = torch.tensor([[0.5, 0.5, 0.5]], dtype=torch.float64, device="cuda")
    o = qsl.qsl_trace(f, seeds, qsl.make_trace_params((0, 0, 0), (1, 1, 1)))
    torch.cuda.synchronize()
    assert abs(float(o["q_perp"][0]) - 2.0) < 1e-12                          # uniform field: Q = 2
    # the adaptive stepper runs in the stencil-gather kernel on a field without the trilinear table (round 2)
    o = qsl.qsl_trace(f, seeds, qsl.make_trace_params((0, 0, 0), (1, 1, 1), method=qsl.QSL_CK45))
    torch.cuda.synchronize()
    assert abs(float(o["q_perp"][0]) - 2.0) < 1e-12
    with pytest.raises(qsl.QslError):          # fp32 arithmetic needs the fp32 trilinear table
        qsl.qsl_trace(f, seeds, qsl.make_trace_params((0, 0, 0), (1, 1, 1), arith=qsl.QSL_ARITH_F32))
    f.destroy()
    z4 = torch.zeros(4 * 4 * 4, dtype=torch.float64, device="cuda") + 1.0
    with pytest.raises(qsl.QslError):          # higher orders are defined for the paper's mode only
        qsl.qsl_field_create(4, 4, 4, z4, z4, z4, lo=(0, 0, 0), hi=(1, 1, 1), interp_order=qsl.QSL_TRICUBIC,
                             interp_mode=qsl.QSL_INTERP_FIRST)
    with pytest.raises(qsl.QslError):
        qsl.qsl_field_create(4, 4, 4, z4, z4, z4, lo=(0, 0, 0), hi=(1, 1, 1), interp_order=7)

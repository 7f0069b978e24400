"""Pins of the oracle's adaptive Cash-Karp 5(4) stepper (reading A16).

The tableau is pinned through its behaviour, not by retyping it: on the linear field B = (kx, -ky, 1) in INTERP_FIRST
mode (the gridded interpolant is exact) one step of size h has the exact solution x0 e^{k h'}..., so the 5th-order
result must converge with h^6 per step and the embedded 4th-order result with h^5; a wrong node, coupling coefficient or
weight breaks one of the two orders.  The controller is pinned by its invariants and by the closed forms of pin P2."""
import math

import numpy as np

import oracle
import qsl_inputs as qi
from tests.test_oracle_pins import BOX_HI, BOX_LO, K, P2_SEEDS, _closed_forms, _hyper


def _exact_unit_speed(x0, y0, z0, lam):
    """Point reached from (x0, y0, z0) after affine parameter lam along b = B/|B| of B = (kx, -ky, 1): integrate
    dz/dlam = 1/|B| with a tight quadrature-free ODE solve (scipy DOP853) of the full system."""
    import scipy.integrate
    f = lambda t, p: (lambda B: B / np.linalg.norm(B))(np.array([K * p[0], -K * p[1], 1.0]))
    r = scipy.integrate.solve_ivp(f, (0.0, lam), [x0, y0, z0], method="DOP853", rtol=1e-13, atol=1e-15)
    return r.y[:, -1]


def test_ck_single_step_orders_5_and_4():
    F = _hyper(64, oracle.INTERP_FIRST)
    y0 = np.array([0.21, -0.33, 0.4, 1, 0, 0, 0, 1, 0, 0.0])
    e5, e4 = [], []
    for h in (0.2, 0.1, 0.05):
        yn, err = oracle.ck_step(F, y0, h)
        ex = _exact_unit_speed(*y0[:3], h)
        e5.append(np.abs(yn[:3] - ex).max())
        e4.append(np.abs((yn[:3] - err) - ex).max())
        assert abs(yn[9] - h) < 1e-12                                   # |b| = 1: the length component advances by h
    assert 45 < e5[0] / e5[1] < 90 and 45 < e5[1] / e5[2] < 90, e5      # local error of the 5th-order result: h^6
    assert 24 < e4[0] / e4[1] < 42 and 24 < e4[1] / e4[2] < 42, e4      # embedded 4th-order result: h^5
    assert e5[2] < 0.05 * e4[2]


def test_ck_deviation_is_derivative_of_the_step_map():
    """RK applied to the augmented system is the exact derivative of the RK map (pin P4's argument): finite differences
    of one Cash-Karp step with respect to the start point reproduce the stepped deviation vectors."""
    F = _hyper(64, oracle.INTERP_FIRST)
    y0 = np.array([0.21, -0.33, 0.4, 1, 0, 0, 0, 0, 1, 0.0])
    h, eps = 0.1, 1e-6
    yn, _ = oracle.ck_step(F, y0, h)
    for v in range(2):
        d = y0[3 + 3 * v:6 + 3 * v]
        yp, ym = y0.copy(), y0.copy()
        yp[:3] += eps * d; ym[:3] -= eps * d
        fd = (oracle.ck_step(F, yp, h)[0][:3] - oracle.ck_step(F, ym, h)[0][:3]) / (2 * eps)
        assert np.abs(fd - yn[3 + 3 * v:6 + 3 * v]).max() < 1e-8


def test_ck_closed_forms_and_tolerance_ladder():
    """Pin P2 with the adaptive stepper: the error against the closed forms falls with tol, the number of steps rises."""
    F = _hyper(64, oracle.INTERP_FIRST)
    seeds = np.array([[x, y, 0.0] for x, y in P2_SEEDS])
    ref = [_closed_forms(x, y) for x, y in P2_SEEDS]
    end = np.array([r[0] for r in ref]); L = np.array([r[1] for r in ref]); qb = np.array([r[2] for r in ref])
    # step_frac = 8: the controller may use steps of 8 * 2^j cells (up to half the box), so that on this smooth field
    # it is the tolerance, not the largest allowed step, that sets the step
    errs, steps = [], []
    for tol in (1e-1, 1e-4, 1e-7):
        o = oracle.trace(F, seeds, BOX_LO, BOX_HI, method=oracle.CK45, tol=tol, step_frac=8.0)
        errs.append(np.abs(o["end_f"] - end).max()); steps.append(int(o["total_steps"]))
        assert np.all(o["face_b"] == 4) and np.all(o["nsteps_b"] == 1)       # zero-length backward end
    assert errs[0] < 1e-2 and errs[1] < 1e-5 and errs[2] < 1e-8, errs
    assert errs[0] > 30 * errs[1] > 900 * errs[2], errs
    assert steps[0] < steps[1] < steps[2], steps
    o = oracle.trace(F, seeds, BOX_LO, BOX_HI, method=oracle.CK45, tol=1e-8)
    assert np.allclose(o["L"], L, rtol=1e-9) and np.allclose(o["q_bnd"], qb, rtol=1e-8)
    # at a loose tolerance the controller runs at its largest step 2^2 * step_frac cell: 4x fewer steps than RK4
    rk = oracle.trace(F, seeds, BOX_LO, BOX_HI, method=oracle.RK4)
    ck = oracle.trace(F, seeds, BOX_LO, BOX_HI, method=oracle.CK45, tol=1e-2)
    assert 0.2 < ck["total_steps"] / rk["total_steps"] < 0.4


def test_ck_uniform_field_q_two():
    g = qi.Grid.uniform((9, 9, 9), (0, 0, 0), (1, 1, 1))
    B = [np.full(g.shape, v) for v in (0.3, -0.2, 0.9)]
    F = oracle.Field(g, B, oracle.F64, oracle.NORMALIZE_FIRST)
    seeds = np.array([[0.4, 0.5, 0.3], [0.2, 0.7, 0.6]])
    o = oracle.trace(F, seeds, (0, 0, 0), (1, 1, 1), method=oracle.CK45)
    assert np.abs(o["q_perp"] - 2).max() < 1e-12 and np.abs(o["q_bnd"] - 2).max() < 1e-12


def _quad_field(n=32, st=oracle.F32):
    g = qi.Grid.uniform((n, n, n), BOX_LO, BOX_HI)
    q, r = qi.quadrupole_charges()
    return oracle.Field(g, qi.quadrupole_field(g, q, r), st, oracle.NORMALIZE_FIRST)


def test_ck_mode_consistency_and_controller_invariants():
    """P12 for the adaptive stepper: controlling the position only makes x, L and the step counts identical in L and
    L+Q mode.  A rejected step is not counted; tightening tol can only add steps."""
    F = _quad_field()
    rng = np.random.default_rng(9)
    seeds = np.stack([rng.uniform(-0.6, 0.6, 100), rng.uniform(-0.6, 0.6, 100), rng.uniform(0.0, 0.5, 100)], 1)
    kw = dict(method=oracle.CK45, max_steps=20000)
    a = oracle.trace(F, seeds, BOX_LO, BOX_HI, mode=oracle.TRACE_LQ, **kw)
    b = oracle.trace(F, seeds, BOX_LO, BOX_HI, mode=oracle.TRACE_L, **kw)
    for k in ("end_f", "end_b", "L", "face_f", "face_b", "nsteps_f", "nsteps_b", "status"):
        assert np.array_equal(a[k], b[k]), k
    c = oracle.trace(F, seeds, BOX_LO, BOX_HI, mode=oracle.TRACE_L, tol=1e-6, **kw)
    assert c["total_steps"] > a["total_steps"]


def test_ck_is_the_convergence_check_of_the_fixed_step_rule():
    """the adaptive stepper "can be used for testing the convergence properties" of the fixed-step scheme:
    on the gridded quadrupole RK4 at h = 0.25 cell and Cash-Karp at a tight tolerance agree far better than either
    differs from a coarse run."""
    F = _quad_field(48, oracle.F64)
    rng = np.random.default_rng(3)
    seeds = np.stack([rng.uniform(-0.5, 0.5, 64), rng.uniform(-0.5, 0.5, 64), rng.uniform(0.05, 0.4, 64)], 1)
    rk = oracle.trace(F, seeds, BOX_LO, BOX_HI, method=oracle.RK4, max_steps=50000)
    ck = oracle.trace(F, seeds, BOX_LO, BOX_HI, method=oracle.CK45, tol=1e-6, max_steps=50000)
    same = (rk["face_f"] == ck["face_f"]) & (rk["face_b"] == ck["face_b"])
    assert same.mean() > 0.95
    d = np.abs(rk["end_f"] - ck["end_f"]).max(1)[same]
    assert np.median(d) < 1e-6 and np.quantile(d, 0.9) < 1e-4, (np.median(d), d.max())
    rl = np.abs(rk["L"] - ck["L"])[same] / ck["L"][same]
    assert np.median(rl) < 1e-6

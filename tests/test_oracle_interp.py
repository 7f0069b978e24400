"""Pins of the oracle's higher-order interpolation (reading A18):
triquadratic (Dodgson 1997, 27 vertices) and tricubic (Keys 1981, 64 vertices) kernels with analytic gradients.

The kernels are pinned by the properties that define them in the cited papers rather than by retyping their formulas:
both interpolate the samples and reproduce linear fields; Keys' cubic convolution with a = -1/2 is the one member of its
family that reproduces quadratics (third-order accurate), and it is C1; Dodgson's interpolating quadratic is C0 with
slope breaks at the half-cell points.  The analytic gradient is pinned by finite differences of the value."""
import math

import numpy as np
import pytest

import oracle
import qsl_inputs as qi
from tests.test_oracle_pins import BOX_HI, BOX_LO, K, P2_SEEDS, _closed_forms

ORDERS = [oracle.TRIQUADRATIC, oracle.TRICUBIC]


def _cubes(g, f):
    X, Y, Z = np.meshgrid(g.xs, g.ys, g.zs, indexing="ij")
    return [np.ascontiguousarray(np.transpose(c * np.ones_like(X), (2, 1, 0))) for c in f(X, Y, Z)]


def _field(g, f, order, mode=oracle.INTERP_FIRST):
    return oracle.Field(g, _cubes(g, f), oracle.F64, mode, order)


def _raw(F, x):
    """(B(x), dB/dx) of the raw interpolant, recovered from INTERP_FIRST outputs b = B/|B|, m = |B|, J = (G - u u^T G)/m
    is not invertible for G - so the raw gradient is taken from NORMALIZE_FIRST fields instead (see callers)."""
    b, J, m, _ = F.evaluate(x)
    return b, J, m


PTS = np.array([[0.43, 0.27, 0.61], [0.02, 0.97, 0.5], [0.99, 0.01, 0.03], [0.5, 0.5, 0.5], [0.07, 0.93, 0.98]])


@pytest.mark.parametrize("order", ORDERS)
def test_interpolates_the_samples_and_reproduces_linear_fields(order):
    g = qi.Grid.uniform((7, 6, 8), (0, 0, 0), (1, 1, 1))
    rng = np.random.default_rng(order)
    B = [rng.normal(size=g.shape) for _ in range(3)]
    F = oracle.Field(g, B, oracle.F64, oracle.NORMALIZE_FIRST, order)
    for (i, j, k) in [(0, 0, 0), (3, 2, 4), (6, 5, 7), (1, 5, 0), (5, 0, 6)]:
        b, J, m, _ = F.evaluate(np.array([g.xs[i], g.ys[j], g.zs[k]]))
        assert np.allclose(b, F.packed.reshape(g.nz, g.ny, g.nx, 4)[k, j, i, :3], atol=1e-14)
    lin = lambda x, y, z: (1 + 2 * x - y + 0.5 * z, 2 - x + 0.25 * y, 0.5 + z - 3 * x)
    G = np.array([[2, -1, 0.5], [-1, 0.25, 0], [-3, 0, 1.0]])
    # NORMALIZE_FIRST on a field whose samples are used as they are (pack normalises: undo by comparing directions) is
    # awkward; INTERP_FIRST returns b = B/|B| and m = |B| of the raw interpolant, which is what is pinned here
    F = _field(g, lin, order)
    for x in PTS:                                              # includes the first and last cells (boundary rule)
        b, J, m, _ = F.evaluate(x)
        v = np.array(lin(*x))
        assert abs(m - np.linalg.norm(v)) < 1e-13 and np.abs(b - v / m).max() < 1e-13
        u = v / m
        assert np.abs(J - (G - np.outer(u, u @ G)) / m).max() < 1e-12


def test_keys_reproduces_quadratics_dodgson_does_not():
    g = qi.Grid.uniform((9, 8, 7), (0, 0, 0), (1, 1, 1))
    quad = lambda x, y, z: (1 + 2 * x - y + 0.5 * z + x * y - 0.3 * z * z + 0.7 * x * x, 2 - x + 0.2 * y * z, 0.5 + z + y * y)
    def grad(x, y, z):
        return np.array([[2 + y + 1.4 * x, -1 + x, 0.5 - 0.6 * z], [-1, 0.2 * z, 0.2 * y], [0, 2 * y, 1.0]])
    Fc, Fq = _field(g, quad, oracle.TRICUBIC), _field(g, quad, oracle.TRIQUADRATIC)
    eq = []
    for x in PTS:
        v = np.array(quad(*x)); m0 = np.linalg.norm(v); u = v / m0
        b, J, m, _ = Fc.evaluate(x)
        assert abs(m - m0) < 1e-13 and np.abs(b - u).max() < 1e-13
        assert np.abs(J - (grad(*x) - np.outer(u, u @ grad(*x))) / m0).max() < 1e-12
        eq.append(abs(Fq.evaluate(x)[2] - m0))
    assert max(eq) > 1e-5                                      # the quadratic kernel is only linear-reproducing


@pytest.mark.parametrize("order", [oracle.TRILINEAR] + ORDERS)
def test_analytic_gradient_is_the_derivative_of_the_value(order):
    g = qi.Grid.uniform((7, 6, 8), (0, 0, 0), (1, 1, 1))
    rng = np.random.default_rng(10 + order)
    B = [rng.normal(size=g.shape) for _ in range(3)]
    F = oracle.Field(g, B, oracle.F64, oracle.NORMALIZE_FIRST, order)
    eps = 1e-6
    for x in PTS + np.array([0.003, -0.002, 0.001]):           # off the nodes and the half-cell points
        _, J, _, _ = F.evaluate(x)
        for d in range(3):
            e = np.zeros(3); e[d] = eps
            fd = (F.evaluate(x + e)[0] - F.evaluate(x - e)[0]) / (2 * eps)
            assert np.abs(fd - J[:, d]).max() < 2e-7 * max(1.0, np.abs(J).max())


def test_smoothness_c1_cubic_c0_quadratic_c0_linear():
    g = qi.Grid.uniform((7, 6, 8), (0, 0, 0), (1, 1, 1))
    rng = np.random.default_rng(3)
    B = [rng.normal(size=g.shape) for _ in range(3)]
    jumpJ = {}
    for order in (oracle.TRILINEAR, oracle.TRIQUADRATIC, oracle.TRICUBIC):
        F = oracle.Field(g, B, oracle.F64, oracle.NORMALIZE_FIRST, order)
        worst_v, worst_J = 0.0, 0.0
        for xf in (g.xs[2], g.xs[3], 0.5 * (g.xs[2] + g.xs[3])):   # two cell faces and a half-cell point
            lo = np.array([xf - 1e-10, 0.41, 0.37]); hi = np.array([xf + 1e-10, 0.41, 0.37])
            (b0, J0, _, _), (b1, J1, _, _) = F.evaluate(lo), F.evaluate(hi)
            worst_v = max(worst_v, np.abs(b1 - b0).max()); worst_J = max(worst_J, np.abs(J1 - J0).max())
        assert worst_v < 1e-8                                  # every scheme is continuous
        jumpJ[order] = worst_J
    assert jumpJ[oracle.TRICUBIC] < 1e-7                       # C1 (Keys)
    assert jumpJ[oracle.TRILINEAR] > 1e-2 and jumpJ[oracle.TRIQUADRATIC] > 1e-2


def test_convergence_orders():
    f = lambda x, y, z: (np.sin(2.1 * x + 0.3) * np.cos(1.7 * y) + 2, np.cos(1.3 * x + z) + 0.5 * y, np.exp(0.8 * z) * np.sin(1.1 * y + 0.2))
    rng = np.random.default_rng(8)
    pts = rng.uniform(0.2, 0.8, size=(40, 3))
    rate = {}
    for order in (oracle.TRILINEAR, oracle.TRIQUADRATIC, oracle.TRICUBIC):
        errs = []
        for n in (9, 17, 33):
            g = qi.Grid.uniform((n, n, n), (0, 0, 0), (1, 1, 1))
            F = _field(g, f, order)
            errs.append(max(abs(F.evaluate(x)[2] - np.linalg.norm(np.array(f(*x)))) for x in pts))
        rate[order] = math.log2(errs[1] / errs[2])
    assert 1.7 < rate[oracle.TRILINEAR] < 2.3 and 1.7 < rate[oracle.TRIQUADRATIC] < 2.4
    assert 2.7 < rate[oracle.TRICUBIC] < 3.4                   # Keys: third order


@pytest.mark.parametrize("order", ORDERS)
def test_kernels_depend_on_the_cell_and_the_fraction_only(order):
    """PAPER.md:95 (eq. 3): f_v(x - x_c; h_c) - on a stretched grid the kernels are those of the uniform grid in the units
    of the cell containing x."""
    gs = qi.Grid.from_axes(qi.stretched_axis(8, 0, 1, 3.0), qi.stretched_axis(7, 0, 1, 0.4), qi.stretched_axis(9, 0, 1, 5.0))
    gu = qi.Grid.uniform((8, 7, 9), (0, 0, 0), (1, 1, 1))
    rng = np.random.default_rng(12)
    B = [rng.normal(size=gs.shape) for _ in range(3)]
    Fs = oracle.Field(gs, B, oracle.F64, oracle.NORMALIZE_FIRST, order)
    Fu = oracle.Field(gu, B, oracle.F64, oracle.NORMALIZE_FIRST, order)
    for (i, j, k, t) in [(2, 3, 4, (0.3, 0.8, 0.45)), (0, 0, 0, (0.6, 0.2, 0.9)), (6, 5, 7, (0.7, 0.55, 0.1))]:
        xs = np.array([gs.xs[i] + t[0] * (gs.xs[i + 1] - gs.xs[i]), gs.ys[j] + t[1] * (gs.ys[j + 1] - gs.ys[j]),
                       gs.zs[k] + t[2] * (gs.zs[k + 1] - gs.zs[k])])
        xu = np.array([gu.xs[i] + t[0] * (gu.xs[1] - gu.xs[0]), gu.ys[j] + t[1] * (gu.ys[1] - gu.ys[0]),
                       gu.zs[k] + t[2] * (gu.zs[1] - gu.zs[0])])
        (bs, Js, _, hs), (bu, Ju, _, hu) = Fs.evaluate(xs), Fu.evaluate(xu)
        assert np.abs(bs - bu).max() < 1e-12
        assert np.abs(Js * hs[None, :] - Ju * hu[None, :]).max() < 1e-10      # gradients scale with the cell edges


@pytest.mark.parametrize("order", ORDERS)
def test_traces_through_higher_order_fields(order):
    """The tracer on top: the hyperbolic field is linear, so both kernels reproduce it exactly in INTERP_FIRST mode and
    the closed forms of pin P2 hold to 1e-9; a uniform field gives Q = 2."""
    g = qi.Grid.uniform((32, 32, 32), BOX_LO, BOX_HI)
    F = oracle.Field(g, qi.hyperbolic_field(g, K), oracle.F64, oracle.INTERP_FIRST, order)
    seeds = np.array([[x, y, 0.0] for x, y in P2_SEEDS])
    ref = [_closed_forms(x, y) for x, y in P2_SEEDS]
    o = oracle.trace(F, seeds, BOX_LO, BOX_HI)
    assert np.abs(o["end_f"] - np.array([r[0] for r in ref])).max() < 1e-9
    assert np.allclose(o["q_bnd"], [r[2] for r in ref], rtol=1e-8) and np.allclose(o["q_perp"], [r[3] for r in ref], rtol=1e-8)
    gu = qi.Grid.uniform((9, 9, 9), (0, 0, 0), (1, 1, 1))
    Fu = oracle.Field(gu, [np.full(gu.shape, v) for v in (0.3, -0.2, 0.9)], oracle.F64, oracle.NORMALIZE_FIRST, order)
    o = oracle.trace(Fu, np.array([[0.4, 0.5, 0.3]]), (0, 0, 0), (1, 1, 1))
    assert abs(o["q_perp"][0] - 2) < 1e-12 and abs(o["q_bnd"][0] - 2) < 1e-12


@pytest.mark.parametrize("order", ORDERS)
def test_outside_the_grid_the_boundary_cell_polynomial_is_continued(order):
    """Reading A8 carried to the higher orders (cell index clamped, fraction not): for a stage point a little outside the
    grid the interpolant and its gradient are the polynomial of the boundary cell continued, as for the trilinear kernels.
    Pinned without the kernel formulas: along a line parallel to an axis the interpolant inside one cell (one half cell
    for the quadratic) is a polynomial of degree <= 3 in that coordinate, so a cubic through four inside values predicts
    the outside values, and its derivative the outside gradient component."""
    g = qi.Grid.uniform((7, 6, 8), (0, 0, 0), (1, 1, 1))
    rng = np.random.default_rng(10 + order)
    B = [rng.normal(size=g.shape) for _ in range(3)]
    F = oracle.Field(g, B, oracle.F64, oracle.NORMALIZE_FIRST, order)
    n = (7, 6, 8)
    for axis in range(3):
        h = 1.0 / (n[axis] - 1)
        for side in (0, 1):
            base = np.array([0.41, 0.33, 0.58])
            # four points inside the boundary (half) cell next to the face, three outside
            ins = (np.array([0.05, 0.15, 0.3, 0.45]) * h) if side == 0 else (1.0 - np.array([0.05, 0.15, 0.3, 0.45]) * h)
            outs = (np.array([-0.02, -0.2, -0.45]) * h) if side == 0 else (1.0 + np.array([0.02, 0.2, 0.45]) * h)

            def at(c):
                x = base.copy(); x[axis] = c
                b, J, m, _ = F.evaluate(x)
                return np.append(b, m), J[:, axis]

            vals = np.array([at(c)[0] for c in ins])
            for q in range(4):
                poly = np.polynomial.Polynomial.fit(ins, vals[:, q], 3)
                for c in outs:
                    v, gr = at(c)
                    assert abs(v[q] - poly(c)) < 1e-11, (order, axis, side, q, c)
                    if q < 3:
                        assert abs(gr[q] - poly.deriv()(c)) < 1e-9 / h, (order, axis, side, q, c)

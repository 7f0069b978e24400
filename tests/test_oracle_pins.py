"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these tests touches the CUDA path.  Each pin is chosen so that a plausible mistake in the oracle
(dropped term, wrong sign or index, transposed operand) fails at least one of them.
"""
import math
import os

import numpy as np
import pytest
import scipy.integrate
import scipy.interpolate

import oracle
import qsl_inputs as qi

K = 2.0
BOX_LO, BOX_HI = (-1.0, -1.0, 0.0), (1.0, 1.0, 1.0)
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "hyperbolic_closed_forms.txt")


def _hyper(n=64, interp=oracle.INTERP_FIRST):
    g = qi.Grid.uniform((n, n, n), BOX_LO, BOX_HI)
    return oracle.Field(g, qi.hyperbolic_field(g, K), oracle.F64, interp)


# ----------------------------------------------------------------------------- O1: interpolation pins
def test_evaluate_reproduces_trilinear_polynomial_exactly():
    """A function that is itself trilinear is reproduced (value and analytic gradient) to rounding, on a
    uniform and on a stretched grid (PAPER.md:95 eq. 3, :123)."""
    rng = np.random.default_rng(1)
    for stretched in (False, True):
        if stretched:
            g = qi.Grid.from_axes(qi.stretched_axis(9, -1, 2, 3.0), qi.stretched_axis(7, 0, 1, 0.5),
                                  qi.stretched_axis(11, -2, 0, 2.0))
        else:
            g = qi.Grid.uniform((9, 7, 11), (-1, 0, -2), (2, 1, 0))
        Z, Y, X = np.meshgrid(g.zs, g.ys, g.xs, indexing="ij")
        co = rng.normal(size=(3, 8))

        def poly(c, x, y, z):
            return c[0] + c[1] * x + c[2] * y + c[3] * z + c[4] * x * y + c[5] * x * z + c[6] * y * z + c[7] * x * y * z

        def grad(c, x, y, z):
            return np.array([c[1] + c[4] * y + c[5] * z + c[7] * y * z, c[2] + c[4] * x + c[6] * z + c[7] * x * z,
                             c[3] + c[5] * x + c[6] * y + c[7] * x * y])
        B = tuple(poly(co[c], X, Y, Z) for c in range(3))
        F = oracle.Field(g, B, oracle.F64, oracle.INTERP_FIRST)
        for _ in range(50):
            p = np.array([rng.uniform(g.lo[d], g.hi[d]) for d in range(3)])
            # INTERP_FIRST returns the normalised field; undo it with m = |B|
            b, J, m, hc = F.evaluate(p)
            Bex = np.array([poly(co[c], *p) for c in range(3)])
            assert np.allclose(b * m, Bex, rtol=0, atol=1e-12)
            Gex = np.array([grad(co[c], *p) for c in range(3)])          # G[c][d]
            u = Bex / np.linalg.norm(Bex)
            Jex = (Gex - np.outer(u, u @ Gex)) / np.linalg.norm(Bex)
            assert np.allclose(J, Jex, rtol=0, atol=1e-10)


def test_evaluate_matches_scipy_regular_grid_interpolator():
    """Library pin: NORMALIZE_FIRST values are the multilinear interpolant of the packed (b^, |B|) samples."""
    rng = np.random.default_rng(2)
    g = qi.Grid.from_axes(qi.stretched_axis(12, 0, 1, 4.0), np.linspace(0, 2, 9), qi.stretched_axis(10, -1, 1, 0.3))
    B = tuple(rng.normal(size=g.shape) for _ in range(3))
    F = oracle.Field(g, B, oracle.F64, oracle.NORMALIZE_FIRST)
    mag = np.sqrt(B[0] ** 2 + B[1] ** 2 + B[2] ** 2)
    interps = [scipy.interpolate.RegularGridInterpolator((g.zs, g.ys, g.xs), a / mag) for a in B]
    im = scipy.interpolate.RegularGridInterpolator((g.zs, g.ys, g.xs), mag)
    for _ in range(100):
        p = np.array([rng.uniform(g.lo[d], g.hi[d]) for d in range(3)])
        b, J, m, hc = F.evaluate(p)
        ref = np.array([float(f(p[::-1])[0]) for f in interps])
        assert np.allclose(b, ref, atol=1e-13)
        assert abs(m - float(im(p[::-1])[0])) < 1e-12
        # gradient by central differences inside the cell (the interpolant is multilinear there)
        i = [int(np.searchsorted(ax, p[d], side="right") - 1) for d, ax in enumerate((g.xs, g.ys, g.zs))]
        for d, ax in enumerate((g.xs, g.ys, g.zs)):
            eps = 0.25 * min(p[d] - ax[i[d]], ax[i[d] + 1] - p[d])
            if eps < 1e-6:
                continue
            pp, pm = p.copy(), p.copy(); pp[d] += eps; pm[d] -= eps
            fd = (F.evaluate(pp)[0] - F.evaluate(pm)[0]) / (2 * eps)
            assert np.allclose(J[:, d], fd, atol=1e-8)


def test_field_pack_f32_rounding_and_unit_norm():
    g = qi.Grid.uniform((5, 6, 7), (0, 0, 0), (1, 1, 1))
    rng = np.random.default_rng(3)
    B = tuple(rng.normal(size=g.shape) for _ in range(3))
    F = oracle.Field(g, B, oracle.F32, oracle.NORMALIZE_FIRST)
    P = F.packed.reshape(-1, 4)
    assert np.array_equal(P, P.astype(np.float32).astype(np.float64))       # representable in fp32
    B32 = np.stack([a.reshape(-1).astype(np.float32).astype(np.float64) for a in B], 1)
    m = np.sqrt((B32 ** 2).sum(1))
    assert np.allclose(P[:, 3], m, rtol=1e-7)
    assert np.allclose(P[:, :3], B32 / m[:, None], atol=1e-7)


# ----------------------------------------------------------------------------- P1: uniform field
@pytest.mark.parametrize("direction", [(0, 0, 1), (0.3, -0.2, 0.9), (-1, 0.5, -0.25), (1, 0, 0)])
@pytest.mark.parametrize("interp", [oracle.NORMALIZE_FIRST, oracle.INTERP_FIRST])
def test_P1_uniform_field_q_is_two_and_chord(direction, interp):
    """Uniform field: delta x is constant, so eq. (11) gives Q = 2; the line is the chord."""
    g = qi.Grid.uniform((17, 13, 9), BOX_LO, BOX_HI)
    F = oracle.Field(g, qi.uniform_field(g, direction), oracle.F64, interp)
    rng = np.random.default_rng(4)
    seeds = np.stack([rng.uniform(-0.9, 0.9, 64), rng.uniform(-0.9, 0.9, 64), rng.uniform(0.05, 0.95, 64)], 1)
    o = oracle.trace(F, seeds, BOX_LO, BOX_HI)
    d = np.asarray(direction, float); d /= np.linalg.norm(d)
    lo, hi = np.array(BOX_LO), np.array(BOX_HI)
    with np.errstate(divide="ignore", invalid="ignore"):
        tf = np.where(d > 0, (hi - seeds) / d, np.where(d < 0, (lo - seeds) / d, np.inf)).min(1)
        tb = np.where(d > 0, (seeds - lo) / d, np.where(d < 0, (seeds - hi) / d, np.inf)).min(1)
    assert np.allclose(o["q_perp"], 2.0, rtol=0, atol=1e-12)
    # q_bnd is Titov's Q of the face-to-face map D (oblique projection along d between the two end faces):
    # 2 when the faces are parallel, |D|_F^2/|det D| otherwise -- computed here from the geometry alone.
    for i in range(len(seeds)):
        aB, aF = o["face_b"][i] // 2, o["face_f"][i] // 2
        tB = [np.eye(3)[a] for a in range(3) if a != aB]; tF = [np.eye(3)[a] for a in range(3) if a != aF]
        nF = np.eye(3)[aF]
        D = np.array([[tf_ @ (tb_ - d * (nF @ tb_) / (nF @ d)) for tb_ in tB] for tf_ in tF])
        qref = (D ** 2).sum() / abs(np.linalg.det(D))
        assert abs(o["q_bnd"][i] - qref) < 1e-11
        if aB == aF:
            assert abs(qref - 2.0) < 1e-12
    assert np.allclose(o["end_f"], seeds + tf[:, None] * d, atol=1e-12)
    assert np.allclose(o["end_b"], seeds - tb[:, None] * d, atol=1e-12)
    assert np.allclose(o["L"], tf + tb, atol=1e-12)
    assert np.all(o["status"] & ~np.uint32(oracle.ST_OPEN) == 0)


# ----------------------------------------------------------------------------- P2: hyperbolic closed forms
def _closed_forms(x0, y0, k=K):
    """Analytic line through (x0, y0, 0) of B = (kx, -ky, 1): x = x0 e^{kz}, y = y0 e^{-kz}.
    Top exit iff |x0| <= e^{-k}.  q_bnd = |D|_F^2 / |det D| of the foot-point map D (Titov's Q)."""
    if abs(x0) <= math.exp(-k):
        end = np.array([x0 * math.exp(k), y0 * math.exp(-k), 1.0]); zs = 1.0
        qb = math.exp(2 * k) + math.exp(-2 * k)
        D = np.array([[math.exp(k), 0, -k * x0 * math.exp(k)], [0, math.exp(-k), k * y0 * math.exp(-k)], [0, 0, 0]])
    else:
        zs = math.log(1 / abs(x0)) / k; sx = math.copysign(1.0, x0)
        end = np.array([sx, y0 * abs(x0), zs])
        qb = k * (x0 * x0 + y0 * y0) + 1 / (k * x0 * x0)
        D = np.array([[0, 0, 0], [y0 * sx, abs(x0), 0], [-1 / (k * x0), 0, 1.0]])
    L = scipy.integrate.quad(lambda z: math.sqrt(1 + (k * x0 * math.exp(k * z)) ** 2 + (k * y0 * math.exp(-k * z)) ** 2),
                             0, zs, epsabs=1e-13, epsrel=1e-13)[0]
    # q_perp for a seed on z=0 (backward end of zero length): (m_F/m_0)(|P D a|^2 + |P D b|^2)
    B0 = np.array([k * x0, -k * y0, 1.0]); m0 = np.linalg.norm(B0); u0 = B0 / m0
    e = np.zeros(3); e[int(np.argmin(np.abs(u0)))] = 1
    a = e - u0 * (u0 @ e); a /= np.linalg.norm(a); b = np.cross(u0, a)
    BF = np.array([k * end[0], -k * end[1], 1.0]); mF = np.linalg.norm(BF); uF = BF / mF
    P = np.eye(3) - np.outer(uF, uF)
    qp = mF / m0 * (np.sum((P @ D @ a) ** 2) + np.sum((P @ D @ b) ** 2))
    return end, L, qb, qp


P2_SEEDS = [(0.0, 0.0), (0.05, 0.2), (-0.1, -0.4), (0.12, 0.0), (0.3, 0.25), (-0.45, 0.1), (0.135, -0.3), (0.49, 0.49)]


def test_P2_golden_file_matches_formulas():
    """tests/golden/hyperbolic_closed_forms.txt stores the closed-form values (north_star: Q = e^{2kh} + e^{-2kh} =
    54.61646567 for k = 2, h = 1); written by tests/golden/make_golden.py from the formulas only."""
    rows = [l.split() for l in open(GOLDEN) if l.strip() and not l.startswith("#")]
    assert len(rows) == len(P2_SEEDS)
    for r, (x0, y0) in zip(rows, P2_SEEDS):
        v = [float(t) for t in r]
        end, L, qb, qp = _closed_forms(x0, y0)
        assert np.allclose(v, [x0, y0, *end, L, qb, qp], rtol=1e-12, atol=1e-14)
    assert abs(float(rows[0][6]) - 54.61646567) < 1e-8


def test_P2_hyperbolic_interp_first_1e9():
    F = _hyper(64, oracle.INTERP_FIRST)
    rows = np.array([[float(t) for t in l.split()] for l in open(GOLDEN) if l.strip() and not l.startswith("#")])
    seeds = np.stack([rows[:, 0], rows[:, 1], np.zeros(len(rows))], 1)
    o = oracle.trace(F, seeds, BOX_LO, BOX_HI)
    assert np.abs(o["end_f"] - rows[:, 2:5]).max() < 1e-9
    assert np.allclose(o["end_b"], seeds, atol=0)                    # zero-length backward end
    assert np.all(o["face_b"] == 4) and np.all(o["nsteps_b"] == 1)
    assert np.allclose(o["L"], rows[:, 5], rtol=1e-9)
    assert np.allclose(o["q_bnd"], rows[:, 6], rtol=1e-9)
    assert np.allclose(o["q_perp"], rows[:, 7], rtol=1e-9)
    # closed form of L on the y0 = 0 axis: (1/k)[u + 0.5 ln((u-1)/(u+1))] between u0 and u1
    x0 = 0.12; zs = 1.0
    a = K * x0; u0 = math.sqrt(1 + a * a); u1 = math.sqrt(1 + a * a * math.exp(2 * K * zs))
    Fu = lambda u: u + 0.5 * math.log((u - 1) / (u + 1))
    assert abs(o["L"][3] - (Fu(u1) - Fu(u0)) / K) < 1e-9
    assert abs(o["L"][0] - 1.0) < 1e-12                              # L = h at the origin


def test_P2_full_cfg1_map_interp_first():
    """All 16384 seeds of BASELINE.json configs[0]: end points and q_bnd against the closed form."""
    cfg = qi.make_config("cfg1")
    F = oracle.Field(cfg["grid"], cfg["B"], oracle.F64, oracle.INTERP_FIRST)
    s = cfg["seeds"]
    o = oracle.trace(F, s, cfg["box_lo"], cfg["box_hi"], max_steps=cfg["max_steps"])
    top = np.abs(s[:, 0]) <= math.exp(-K)
    qb = np.where(top, 2 * math.cosh(2 * K), K * (s[:, 0] ** 2 + s[:, 1] ** 2) + 1 / (K * s[:, 0] ** 2))
    E = np.where(top[:, None], np.stack([s[:, 0] * math.exp(K), s[:, 1] * math.exp(-K), np.ones(len(s))], 1),
                 np.stack([np.sign(s[:, 0]), s[:, 1] * np.abs(s[:, 0]), np.log(1 / np.abs(s[:, 0])) / K], 1))
    assert np.abs(o["end_f"] - E).max() < 1e-9
    assert np.abs(o["q_bnd"] / qb - 1).max() < 1e-9
    assert np.array_equal(o["face_f"] == 5, top)
    assert abs(top.mean() - 0.27) < 0.02                             # D1: about a quarter exits through the top
    assert o["q_perp"].min() >= 2 - 1e-9 and o["q_bnd"].min() >= 2 - 1e-9     # P5


def test_P2_normalize_first_is_second_order_accurate():
    """Paper mode (fn. 9): O(cell^2) away from the closed form (reading A2): <= 1e-2 at 64^3, ~4x smaller at 128^3."""
    rows = np.array([[float(t) for t in l.split()] for l in open(GOLDEN) if l.strip() and not l.startswith("#")])
    seeds = np.stack([rows[:, 0], rows[:, 1], np.zeros(len(rows))], 1)
    errs = []
    for n in (64, 128):
        o = oracle.trace(_hyper(n, oracle.NORMALIZE_FIRST), seeds, BOX_LO, BOX_HI)
        e = max(np.abs(o["q_bnd"] / rows[:, 6] - 1).max(), np.abs(o["end_f"] - rows[:, 2:5]).max(),
                np.abs(o["L"] / rows[:, 5] - 1).max())
        errs.append(e)
    assert errs[0] < 1e-2
    assert 2.5 < errs[0] / errs[1] < 6.0


# ----------------------------------------------------------------------------- P3: invariances
def test_P3_basis_rotation_invariance():
    """the only restriction on a^, b^ is orthonormality with B^(x0)."""
    F = _hyper(48, oracle.NORMALIZE_FIRST)
    rng = np.random.default_rng(5)
    seeds = np.stack([rng.uniform(-0.5, 0.5, 40), rng.uniform(-0.5, 0.5, 40), rng.uniform(0.0, 0.9, 40)], 1)
    o0 = oracle.trace(F, seeds, BOX_LO, BOX_HI)
    for ang in (0.7, 2.1, -1.3):
        o1 = oracle.trace(F, seeds, BOX_LO, BOX_HI, basis_angle=ang)
        assert np.allclose(o1["q_perp"], o0["q_perp"], rtol=1e-9)
        assert np.allclose(o1["q_bnd"], o0["q_bnd"], rtol=1e-9)
        assert np.array_equal(o1["end_f"], o0["end_f"]) and np.array_equal(o1["L"], o0["L"])


def test_P3_q_constant_along_the_line():
    """Global Q is constant along a field line (PAPER.md:165 by contrast): mid-line seeds vs foot-point seeds.
    q_bnd is the boundary-to-boundary quantity and must agree; L must agree."""
    F = _hyper(64, oracle.INTERP_FIRST)
    foot = np.array([[0.05, 0.2, 0.0], [-0.1, -0.4, 0.0], [0.3, 0.25, 0.0], [0.02, -0.45, 0.0]])
    o0 = oracle.trace(F, foot, BOX_LO, BOX_HI)
    for z in (0.25, 0.4):
        mid = np.stack([foot[:, 0] * np.exp(K * z), foot[:, 1] * np.exp(-K * z), np.full(len(foot), z)], 1)
        mid = mid[np.abs(mid[:, 0]) < 1]
        keep = np.abs(foot[:, 0] * np.exp(K * z)) < 1
        o1 = oracle.trace(F, mid, BOX_LO, BOX_HI)
        assert np.allclose(o1["q_bnd"], o0["q_bnd"][keep], rtol=1e-8)
        assert np.allclose(o1["L"], o0["L"][keep], rtol=1e-8)
        assert np.allclose(o1["end_f"], o0["end_f"][keep], atol=1e-9)
        assert np.allclose(o1["end_b"], foot[keep], atol=1e-9)
        # q_perp is also constant along the line (it is Titov's Q_perp)
        assert np.allclose(o1["q_perp"], o0["q_perp"][keep], rtol=1e-7)


def test_P3_field_reversal_swaps_ends():
    """Eq. (11) is symmetric in F <-> B: tracing -B swaps the ends and leaves Q, L unchanged."""
    g = qi.Grid.uniform((32, 32, 32), BOX_LO, BOX_HI)
    q, r = qi.quadrupole_charges()
    B = qi.quadrupole_field(g, q, r)
    Fp = oracle.Field(g, B, oracle.F64, oracle.NORMALIZE_FIRST)
    Fm = oracle.Field(g, tuple(-a for a in B), oracle.F64, oracle.NORMALIZE_FIRST)
    rng = np.random.default_rng(6)
    seeds = np.stack([rng.uniform(-0.6, 0.6, 60), rng.uniform(-0.6, 0.6, 60), rng.uniform(0.01, 0.5, 60)], 1)
    a = oracle.trace(Fp, seeds, BOX_LO, BOX_HI, max_steps=20000)
    b = oracle.trace(Fm, seeds, BOX_LO, BOX_HI, max_steps=20000)
    assert np.array_equal(a["end_f"], b["end_b"]) and np.array_equal(a["end_b"], b["end_f"])
    assert np.array_equal(a["face_f"], b["face_b"])
    assert np.allclose(a["L"], b["L"], rtol=1e-14)
    assert np.allclose(a["q_perp"], b["q_perp"], rtol=1e-10)
    assert np.allclose(a["q_bnd"], b["q_bnd"], rtol=1e-10)


# ----------------------------------------------------------------------------- P4: finite-difference Jacobian
def _p4_errors(F, seeds, eps, max_steps=20000):
    o = oracle.trace(F, seeds, BOX_LO, BOX_HI, max_steps=max_steps, want_dev=True)
    rel = []
    for i, x0 in enumerate(seeds):
        b0 = F.evaluate(x0)[0]; u = b0 / np.linalg.norm(b0)
        e = np.zeros(3); e[int(np.argmin(np.abs(u)))] = 1
        a = e - u * (u @ e); a /= np.linalg.norm(a); bp = np.cross(u, a)
        for end, dev, face in (("end_f", "dev_f", "face_f"), ("end_b", "dev_b", "face_b")):
            uE = F.evaluate(o[end][i])[0]; uE /= np.linalg.norm(uE)
            P = np.eye(3) - np.outer(uE, uE)
            for v, sl in ((a, slice(0, 3)), (bp, slice(3, 6))):
                pm = oracle.trace(F, np.stack([x0 + eps * v, x0 - eps * v]), BOX_LO, BOX_HI, max_steps=max_steps,
                                  mode=oracle.TRACE_L)
                if pm[face][0] != o[face][i] or pm[face][1] != o[face][i]:
                    continue                                         # perturbed lines straddle a box edge
                fd = P @ (pm[end][0] - pm[end][1]) / (2 * eps)
                lin = P @ o[dev][i][sl]
                rel.append(np.linalg.norm(fd - lin) / max(np.linalg.norm(lin), 1e-3))
    return np.array(rel)


def test_P4_deviation_vectors_match_finite_differences():
    """Pariat & Demoulin's three-line finite differences against the linearised eq. (5):
    (end(x0 + eps v) - end(x0 - eps v)) / 2 eps, projected perpendicular to B at the end, equals delta_perp.
    Holds because RK applied to the augmented system is the exact derivative of the RK map."""
    rng = np.random.default_rng(7)
    # (i) smooth case: linear field, INTERP_FIRST -> no gradient kinks at cell faces, tight gate
    F = _hyper(32, oracle.INTERP_FIRST)
    seeds = np.stack([rng.uniform(-0.5, 0.5, 24), rng.uniform(-0.5, 0.5, 24), rng.uniform(0.05, 0.9, 24)], 1)
    rel = _p4_errors(F, seeds, 1e-6)
    assert len(rel) > 80 and rel.max() < 1e-6
    # (ii) quadrupole, paper mode: the trilinear gradient jumps at cell faces, so +-eps lines that cross a face
    # on different steps add O(eps) noise to the finite difference; the bulk must still agree tightly
    g = qi.Grid.uniform((40, 40, 40), BOX_LO, BOX_HI)
    q, r = qi.quadrupole_charges()
    F = oracle.Field(g, qi.quadrupole_field(g, q, r), oracle.F64, oracle.NORMALIZE_FIRST)
    seeds = np.stack([rng.uniform(-0.5, 0.5, 48), rng.uniform(-0.4, 0.4, 48), rng.uniform(0.05, 0.4, 48)], 1)
    rel = _p4_errors(F, seeds, 1e-7)
    assert len(rel) > 150
    assert np.median(rel) < 1e-7 and np.quantile(rel, 0.9) < 1e-5 and rel.max() < 2e-2


# ----------------------------------------------------------------------------- P5 / P6
def test_P5_q_lower_bound_converges_on_quadrupole():
    """Q >= 2 holds exactly only when flux is conserved along the numerical tube; the trilinear interpolant of the
    normalised field is not solenoidal, so eq. (11) undershoots 2 by O(cell^2) where the field is under-resolved
    (charges at depth 0.1).  The deficit must shrink ~4x per grid doubling.  (Exact bound: cfg1 test above.)"""
    q, r = qi.quadrupole_charges()
    rng = np.random.default_rng(8)
    seeds = np.stack([rng.uniform(-0.6, 0.6, 400), rng.uniform(-0.6, 0.6, 400), rng.uniform(0.0, 0.5, 400)], 1)
    deficit = []
    for n in (48, 96):
        g = qi.Grid.uniform((n, n, n), BOX_LO, BOX_HI)
        F = oracle.Field(g, qi.quadrupole_field(g, q, r), oracle.F64, oracle.NORMALIZE_FIRST)
        o = oracle.trace(F, seeds, BOX_LO, BOX_HI, max_steps=20000)
        ok = (o["status"] & ~np.uint32(oracle.ST_OPEN)) == 0
        assert ok.all()
        deficit.append(2 - min(o["q_perp"].min(), o["q_bnd"].min()))
    assert deficit[0] < 0.3 and deficit[1] < 0.1 and deficit[1] < deficit[0] / 3
    # P7 sanity: closed lines of the quadrupole join opposite polarities on z = 0
    closed = (o["face_f"] == 4) & (o["face_b"] == 4)
    assert closed.sum() > 50
    bzf = qi.quadrupole_B(o["end_f"][closed], q, r)[:, 2]; bzb = qi.quadrupole_B(o["end_b"][closed], q, r)[:, 2]
    assert np.all(bzf < 0) and np.all(bzb > 0)


def test_P6_rk4_is_fourth_order_and_euler_first_order():
    """INTERP_FIRST on the linear field: the interpolant is exact, so the error is the integrator's."""
    F = _hyper(64, oracle.INTERP_FIRST)
    seeds = np.array([[0.05, 0.2, 0.0], [0.3, 0.25, 0.0], [-0.1, -0.4, 0.0]])
    ref = np.array([_closed_forms(x, y)[0] for x, y, _ in seeds])
    err = {}
    for method, fr in ((oracle.RK4, (2.0, 1.0)), (oracle.EULER, (0.5, 0.25))):
        e = [np.abs(oracle.trace(F, seeds, BOX_LO, BOX_HI, method=method, step_frac=f)["end_f"] - ref).max() for f in fr]
        err[method] = e[0] / e[1]
    assert 12 < err[oracle.RK4] < 20
    assert 1.7 < err[oracle.EULER] < 2.3


# ----------------------------------------------------------------------------- P12 and status handling
def test_P12_L_mode_bit_identical_to_LQ_mode():
    g = qi.Grid.uniform((32, 32, 32), BOX_LO, BOX_HI)
    q, r = qi.quadrupole_charges()
    F = oracle.Field(g, qi.quadrupole_field(g, q, r), oracle.F32, oracle.NORMALIZE_FIRST)
    rng = np.random.default_rng(9)
    seeds = np.stack([rng.uniform(-0.6, 0.6, 100), rng.uniform(-0.6, 0.6, 100), rng.uniform(0.0, 0.5, 100)], 1)
    a = oracle.trace(F, seeds, BOX_LO, BOX_HI, max_steps=20000, mode=oracle.TRACE_LQ)
    b = oracle.trace(F, seeds, BOX_LO, BOX_HI, max_steps=20000, mode=oracle.TRACE_L)
    for k in ("end_f", "end_b", "L", "face_f", "face_b", "nsteps_f", "nsteps_b", "status"):
        assert np.array_equal(a[k], b[k]), k
    assert np.all(np.isnan(b["q_perp"]))


def test_status_bits_and_caps():
    F = _hyper(16, oracle.NORMALIZE_FIRST)
    seeds = np.array([[0.0, 0.0, 0.5], [2.0, 0.0, 0.5], [0.1, 0.1, 0.2]])
    o = oracle.trace(F, seeds, BOX_LO, BOX_HI, max_steps=3)
    assert o["status"][1] == oracle.ST_SEED_OUTSIDE and np.isnan(o["L"][1]) and o["face_f"][1] == 255
    assert o["status"][0] & oracle.ST_CAP_F and o["status"][0] & oracle.ST_CAP_B and o["nsteps_f"][0] == 3
    # fixed maximum length: lambda capped per direction, last step shortened
    o = oracle.trace(F, seeds[[0, 2]], BOX_LO, BOX_HI, max_length=0.1)
    assert np.all(o["status"] & oracle.ST_CAP_F) and np.all(o["status"] & oracle.ST_CAP_B)
    assert np.all(o["L"] <= 0.2 + 1e-12) and np.all(o["L"] > 0.19)
    # null at the seed
    g = qi.Grid.uniform((8, 8, 8), BOX_LO, BOX_HI)
    Fz = oracle.Field(g, tuple(np.zeros(g.shape) for _ in range(3)), oracle.F64, oracle.NORMALIZE_FIRST)
    o = oracle.trace(Fz, seeds[[0]], BOX_LO, BOX_HI)
    assert o["status"][0] == oracle.ST_NULL_AT_SEED and np.isnan(o["q_perp"][0])


def test_raised_lower_boundary_trace_box():
    """the lower boundary of the calculation may be raised above the grid's."""
    F = _hyper(32, oracle.INTERP_FIRST)
    lo = (-1.0, -1.0, 0.25)
    seeds = np.array([[0.02, 0.1, 0.5], [0.01, -0.2, 0.6]])
    o = oracle.trace(F, seeds, lo, BOX_HI)
    assert np.all(o["face_b"] == 4) and np.allclose(o["end_b"][:, 2], 0.25, atol=0)
    xb = seeds[:, 0] * np.exp(K * (0.25 - seeds[:, 2]))
    assert np.allclose(o["end_b"][:, 0], xb, atol=1e-9)
    # map z=0.25 -> z=1 of the same field: Q = e^{2k h} + e^{-2k h} with h = 0.75
    assert np.allclose(o["q_bnd"], 2 * math.cosh(2 * K * 0.75), rtol=1e-9)


def test_stretched_grid_traces_like_uniform_on_linear_field():
    """On B = (kx, -ky, 1) the interpolant is exact on any rectilinear grid, so a stretched grid must reproduce
    the same closed forms (INTERP_FIRST); the step follows the local cell (reading A5)."""
    g = qi.Grid.from_axes(qi.stretched_axis(48, -1, 1, 3.0), qi.stretched_axis(40, -1, 1, 0.4),
                          qi.stretched_axis(56, 0, 1, 5.0))
    F = oracle.Field(g, qi.hyperbolic_field(g, K), oracle.F64, oracle.INTERP_FIRST)
    rows = np.array([[float(t) for t in l.split()] for l in open(GOLDEN) if l.strip() and not l.startswith("#")])
    seeds = np.stack([rows[:, 0], rows[:, 1], np.zeros(len(rows))], 1)
    o = oracle.trace(F, seeds, BOX_LO, BOX_HI)
    assert np.abs(o["end_f"] - rows[:, 2:5]).max() < 1e-8
    assert np.allclose(o["q_bnd"], rows[:, 6], rtol=1e-8)
    assert np.allclose(o["L"], rows[:, 5], rtol=1e-8)

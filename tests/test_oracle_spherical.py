"""Pins of the oracle's spherical geometry (SURVEY.md 8(f) f4; PAPER.md:83-87 eq. 2, :125-135 eq. 6-7, :147 fn. 8,
:153-156 eq. 8; reading A19).  Axes (phi, theta, r) = (longitude, latitude, radius), components in the orthonormal basis.

 S1  monopole B = r^/r^2: radial lines, L = r_max - r_min, Q = 2 exactly (the flux-tube map between two spheres is a
     similarity) - pins the metric factors of eq. 8 and the |B| weighting of eq. 11 together;
 S2  dipole: the invariant r / cos^2(theta) of its lines, phi constant, foot-point latitude and arc length in closed form -
     pins eq. 2 (a wrong or missing 1/r or 1/(r cos theta) bends the lines);
 S3  Cartesian limit: a wedge of unit size at radius 1e5 is a Cartesian box up to O(1e-5); the hyperbolic field traced
     there must reproduce the Cartesian oracle (itself pinned by closed forms) in end points, L, q_perp and q_bnd - pins
     eq. 6 and the scaling of the deviation vectors in and out of coordinate units."""
import math

import numpy as np
import scipy.integrate

import oracle
import qsl_inputs as qi


def _cubes(g, f):
    P, T, R = np.meshgrid(g.xs, g.ys, g.zs, indexing="ij")
    return [np.ascontiguousarray(np.transpose(c * np.ones_like(P), (2, 1, 0))) for c in f(P, T, R)]


def test_S1_monopole_radial_lines_q_two():
    g = qi.Grid.uniform((9, 11, 33), (0.1, -0.3, 1.0), (0.9, 0.5, 3.0))
    F = oracle.Field(g, _cubes(g, lambda p, t, r: (0 * r, 0 * r, 1 / r ** 2)), oracle.F64, oracle.NORMALIZE_FIRST,
                     oracle.TRILINEAR, oracle.SPHERICAL)
    seeds = np.array([[0.33, 0.11, g.zs[7]], [0.71, -0.22, g.zs[20]], [0.5, 0.4, g.zs[1]]])
    o = oracle.trace(F, seeds, g.lo, g.hi)
    assert np.allclose(o["end_f"], np.c_[seeds[:, :2], np.full(3, 3.0)], atol=1e-12)
    assert np.allclose(o["end_b"], np.c_[seeds[:, :2], np.full(3, 1.0)], atol=1e-12)
    assert np.allclose(o["L"], 2.0, atol=1e-12)
    assert np.all(o["face_f"] == 5) and np.all(o["face_b"] == 4)
    assert np.abs(o["q_perp"] - 2).max() < 1e-10 and np.abs(o["q_bnd"] - 2).max() < 1e-10


def _dipole(p, t, r):
    return (0 * r, -np.cos(t) / r ** 3, 2 * np.sin(t) / r ** 3)


def test_S2_dipole_line_geometry():
    errs = []
    seeds = np.array([[0.2, 0.55, 1.3], [0.6, 0.35, 1.6], [0.4, -0.5, 1.2]])
    Req = seeds[:, 2] / np.cos(seeds[:, 1]) ** 2
    for n in (33, 65):
        g = qi.Grid.uniform((5, n, n), (0.0, -1.2, 1.0), (1.0, 1.2, 2.6))
        F = oracle.Field(g, _cubes(g, _dipole), oracle.F64, oracle.NORMALIZE_FIRST, oracle.TRILINEAR, oracle.SPHERICAL)
        o = oracle.trace(F, seeds, g.lo, g.hi, mode=oracle.TRACE_L, max_steps=100000)
        ends = np.concatenate([o["end_f"], o["end_b"]])
        assert np.all(o["face_f"] == 4) and np.all(o["face_b"] == 4)                  # closed lines: both feet on r = 1
        assert np.abs(ends[:, 0] - np.tile(seeds[:, 0], 2)).max() < 1e-12            # phi constant
        lat = np.arccos(np.sqrt(1.0 / Req))                                           # foot points: cos^2(theta) = 1 / R
        e_lat = np.abs(np.abs(ends[:, 1]) - np.tile(lat, 2)).max()
        assert np.all(np.sign(o["end_f"][:, 1]) != np.sign(o["end_b"][:, 1]))          # one foot in each hemisphere
        Lref = [Rq * scipy.integrate.quad(lambda th: math.cos(th) * math.sqrt(1 + 3 * math.sin(th) ** 2), -l, l)[0]
                for Rq, l in zip(Req, lat)]
        errs.append(max(e_lat, np.abs(o["L"] / Lref - 1).max()))
    assert errs[1] < 2e-4 and errs[1] < 0.4 * errs[0], errs                             # O(cell^2) from the interpolant


def test_S3_cartesian_limit_reproduces_the_cartesian_oracle():
    R0, p0, t0, k = 1.0e5, 0.3, 0.2, 2.0
    c0 = math.cos(t0)
    n = 33
    gc = qi.Grid.uniform((n, n, n), (-1.0, -1.0, 0.0), (1.0, 1.0, 1.0))
    Bc = qi.hyperbolic_field(gc, k)
    gs = qi.Grid.uniform((n, n, n), (p0 - 1.0 / (R0 * c0), t0 - 1.0 / R0, R0), (p0 + 1.0 / (R0 * c0), t0 + 1.0 / R0, R0 + 1.0))
    rng = np.random.default_rng(17)
    sc = np.stack([rng.uniform(-0.4, 0.4, 40), rng.uniform(-0.4, 0.4, 40), rng.uniform(0.0, 0.8, 40)], 1)
    sc[:10, 2] = 0.0                                                                   # some photospheric seeds
    ss = np.stack([p0 + sc[:, 0] / (R0 * c0), t0 + sc[:, 1] / R0, R0 + sc[:, 2]], 1)
    for mode in (oracle.NORMALIZE_FIRST, oracle.INTERP_FIRST):
        Fc = oracle.Field(gc, Bc, oracle.F64, mode)
        Fs = oracle.Field(gs, Bc, oracle.F64, mode, oracle.TRILINEAR, oracle.SPHERICAL)   # same samples, spherical axes
        oc = oracle.trace(Fc, sc, gc.lo, gc.hi)
        os_ = oracle.trace(Fs, ss, gs.lo, gs.hi)
        assert np.array_equal(oc["face_f"], os_["face_f"]) and np.array_equal(oc["face_b"], os_["face_b"])
        for key in ("end_f", "end_b"):
            e = os_[key]
            loc = np.stack([(e[:, 0] - p0) * R0 * c0, (e[:, 1] - t0) * R0, e[:, 2] - R0], 1)
            assert np.abs(loc - oc[key]).max() < 2e-4
        assert np.allclose(os_["L"], oc["L"], rtol=2e-4)
        assert np.allclose(os_["q_perp"], oc["q_perp"], rtol=2e-3) and np.allclose(os_["q_bnd"], oc["q_bnd"], rtol=2e-3)
        assert np.abs(os_["nsteps_f"].astype(int) - oc["nsteps_f"]).max() <= 2


def test_S4_cash_karp_in_spherical_geometry():
    """The adaptive stepper in spherical geometry (the paper's own combination): the monopole keeps
    Q = 2 and L = r_max - r_min with fewer steps than the fixed-step rule, and a dipole line keeps the closed-form invariant
    r / cos^2(theta) from foot point to foot point at every tolerance (a missing or wrong metric factor in any of the six
    stages bends the line at O(1))."""
    g = qi.Grid.uniform((9, 11, 33), (0.1, -0.3, 1.0), (0.9, 0.5, 3.0))
    F = oracle.Field(g, _cubes(g, lambda p, t, r: (0 * r, 0 * r, 1 / r ** 2)), oracle.F64, oracle.NORMALIZE_FIRST,
                     oracle.TRILINEAR, oracle.SPHERICAL)
    seeds = np.array([[0.33, 0.11, g.zs[7]], [0.71, -0.22, g.zs[20]]])
    o = oracle.trace(F, seeds, g.lo, g.hi, method=oracle.CK45, tol=1e-2)
    assert np.allclose(o["L"], 2.0, atol=1e-11) and np.abs(o["q_perp"] - 2).max() < 1e-9
    assert int(o["nsteps_f"].sum() + o["nsteps_b"].sum()) < int(sum(oracle.trace(F, seeds, g.lo, g.hi)[k].sum() for k in ("nsteps_f", "nsteps_b")))
    g = qi.Grid.uniform((5, 161, 161), (0.0, -1.0, 1.0), (0.4, 1.0, 3.0))
    F = oracle.Field(g, _cubes(g, _dipole), oracle.F64, oracle.NORMALIZE_FIRST, oracle.TRILINEAR, oracle.SPHERICAL)
    seeds = np.array([[0.2, 0.5, 1.0], [0.2, 0.62, 1.0]])
    errs = []
    for tol in (1e-2, 1e-4, 1e-6):
        o = oracle.trace(F, seeds, g.lo, g.hi, method=oracle.CK45, tol=tol, max_steps=100000)
        inv0 = seeds[:, 2] / np.cos(seeds[:, 1]) ** 2
        end = np.where((o["nsteps_f"] > 1)[:, None], o["end_f"], o["end_b"])
        assert np.all(np.where(o["nsteps_f"] > 1, o["face_f"], o["face_b"]) == 4)        # closed lines: back on r = 1
        assert np.all(np.sign(end[:, 1]) == -np.sign(seeds[:, 1]))                        # in the other hemisphere
        errs.append(np.abs(end[:, 2] / np.cos(end[:, 1]) ** 2 - inv0).max())
    assert max(errs) < 1e-6, errs                                   # floor set by the trilinear interpolant on 161 nodes

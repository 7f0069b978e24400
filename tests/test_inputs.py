"""Checks of the seeded input generators (data only, pin P11)."""
import numpy as np

import qsl_inputs as qi


def test_splitmix64_reference_stream():
    """splitmix64 from seed 0: first outputs of the published reference generator (Steele, Lea & Flood 2014)."""
    r = qi.SplitMix64(0)
    assert [r.next_u64() for _ in range(3)] == [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]
    r = qi.SplitMix64(160900724)
    u = [r.u01() for _ in range(1000)]
    assert 0 <= min(u) and max(u) < 1 and abs(np.mean(u) - 0.5) < 0.05


def test_P11_lfff_is_force_free_and_solenoidal():
    modes = qi.lfff_modes()
    assert len(modes["kx"]) == 32 and np.all(modes["kmag"] >= 2 * np.pi) and np.all(modes["kmag"] <= 8 * np.pi)
    rng = np.random.default_rng(0)
    p = rng.uniform(0.1, 0.9, (8, 3)); d = 1e-5
    J = np.zeros((len(p), 3, 3))
    for j in range(3):
        e = np.zeros(3); e[j] = d
        J[:, :, j] = (qi.lfff_B(p + e, modes) - qi.lfff_B(p - e, modes)) / (2 * d)
    curl = np.stack([J[:, 2, 1] - J[:, 1, 2], J[:, 0, 2] - J[:, 2, 0], J[:, 1, 0] - J[:, 0, 1]], 1)
    B = qi.lfff_B(p, modes); nB = np.linalg.norm(B, axis=1)
    assert (np.linalg.norm(curl - modes["alpha"] * B, axis=1) / nB).max() < 1e-6
    assert (np.abs(np.trace(J, axis1=1, axis2=2)) / nB).max() < 1e-6


def test_grid_fields_match_pointwise_formulas():
    g = qi.Grid.uniform((7, 6, 5), (0, 0, 0), (1, 1, 0.5))
    Z, Y, X = np.meshgrid(g.zs, g.ys, g.xs, indexing="ij")
    pts = np.stack([X.ravel(), Y.ravel(), Z.ravel()], 1)
    modes = qi.lfff_modes()
    q, r = qi.quadrupole_charges(shift=(0.5, 0.5))
    for cube, ref in ((qi.lfff_field(g, modes), qi.lfff_B(pts, modes)), (qi.quadrupole_field(g, q, r), qi.quadrupole_B(pts, q, r))):
        for c in range(3):
            assert np.allclose(cube[c].ravel(), ref[:, c], rtol=1e-12, atol=1e-13)
    bx, by, bz, w = qi.superposition_field(g, q, r, modes, 0.1)
    ql = qi.quadrupole_field(g, q, r); lf = qi.lfff_field(g, modes)
    rms = lambda c: np.sqrt(np.mean(c[0][0] ** 2 + c[1][0] ** 2 + c[2][0] ** 2))
    assert abs(w * rms(lf) / rms(ql) - 0.1) < 1e-12
    assert np.allclose(bx, ql[0] + w * lf[0])


def test_configs_have_the_baseline_shapes():
    c1 = qi.make_config("cfg1")
    assert c1["grid"].shape == (64, 64, 64) and c1["seeds"].shape == (128 * 128, 3)
    assert abs(c1["step_frac"] * min(2 / 63, 1 / 63) - 0.25 / 63) < 1e-18
    assert np.all(c1["seeds"][:, 2] == 0) and abs(c1["seeds"][0, 0] + 0.5 - 0.5 / 128) < 1e-15
    c3 = qi.make_config("cfg3", scale=1 / 16)
    assert c3["lattice"].n == (128, 64, 1) and np.all(c3["seeds"][:, 1] == 0) and c3["seeds"][:, 2].min() > 0
    c2 = qi.make_config("cfg2", scale=1 / 16)
    assert c2["keep"].sum() == len(c2["seeds"]) and 0.8 < c2["keep"].mean() <= 1.0
    c4 = qi.make_config("cfg4", scale=1 / 16)
    assert c4["sample_type"] == "f32" and c4["seeds"].shape == (16 ** 3, 3)
    c5 = qi.make_config("cfg5", scale=1 / 16)
    assert c5["grid"].shape == (16, 32, 32) and c5["levels"] == 3 and c5["lfff_weight"] > 0


def test_stretched_axis_is_monotone_with_ratio():
    x = qi.stretched_axis(33, -1.0, 2.0, 4.0)
    w = np.diff(x)
    assert x[0] == -1.0 and x[-1] == 2.0 and np.all(w > 0) and abs(w[-1] / w[0] - 4.0) < 1e-9

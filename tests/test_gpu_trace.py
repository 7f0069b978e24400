"""GPU parity: qsl_field_create / qsl_trace (through the C ABI) against the CPU oracle, element by element."""
import math

import numpy as np
import pytest
import torch

import oracle
import paper_1609_00724_b200 as qsl
import qsl_inputs as qi
from tests.parity import compare_trace, cpu_field, gpu_field, run_both

pytestmark = pytest.mark.gpu

V1, FRAME = qsl.QSL_FLAG_KERNEL_V1, qsl.QSL_FLAG_KERNEL_FRAME
ALL_FLAGS = [0, qsl.QSL_FLAG_NO_REFILL, qsl.QSL_FLAG_NO_SORT, qsl.QSL_FLAG_NO_REFILL | qsl.QSL_FLAG_NO_SORT,
             V1, V1 | qsl.QSL_FLAG_NO_REFILL, V1 | qsl.QSL_FLAG_NO_SORT, FRAME, FRAME | qsl.QSL_FLAG_NO_REFILL]
KERNELS = [0, V1, FRAME]   # per-cell table kernel (default), corner-gather kernel, cell-frame kernel (uniform grids)


@pytest.mark.parametrize("sample_type", ["f32", "f64"])
@pytest.mark.parametrize("interp", [qsl.QSL_NORMALIZE_FIRST, qsl.QSL_INTERP_FIRST])
def test_field_pack_bit_exact(sample_type, interp):
    g = qi.Grid.uniform((19, 13, 11), (0, 0, 0), (1, 1, 0.5))
    rng = np.random.default_rng(20)
    B = [rng.normal(size=g.shape) for _ in range(3)]
    B[0][1, 2, 3] = B[1][1, 2, 3] = B[2][1, 2, 3] = 0.0           # a null node
    fg = gpu_field(g, B, sample_type, interp)
    fc = cpu_field(g, B, sample_type, interp)
    packed = fg.export().cpu().numpy().astype(np.float64).reshape(-1)
    assert np.array_equal(packed, fc.packed)
    assert fg.nbytes >= packed.size * (4 if sample_type == "f32" else 8)


@pytest.mark.parametrize("flags", ALL_FLAGS)
def test_cfg1_full_size_all_launch_modes(flags):
    """BASELINE.json configs[0] at full size (16384 seeds, paper mode NORMALIZE_FIRST), every scheduling variant."""
    cfg = qi.make_config("cfg1")
    g, c = run_both(cfg["grid"], cfg["B"], "f64", cfg["seeds"], cfg["box_lo"], cfg["box_hi"], max_steps=cfg["max_steps"],
                    flags=flags, want_dev=True)
    rep = compare_trace(g, c, cfg["box_lo"], cfg["box_hi"], label="cfg1 flags=%d" % flags)
    assert rep["same_steps"] == 1.0
    # the basis (a^, b^) is only unique where the smallest |u_d| is unique (reading A7): here off the diagonals |x0| = |y0|
    s = cfg["seeds"]
    uniq = np.abs(np.abs(s[:, 0]) - np.abs(s[:, 1])) > 1e-9
    assert uniq.mean() > 0.98
    assert np.abs(g["dev_f"][uniq] - c["dev_f"][uniq]).max() < 1e-9 * np.abs(c["dev_f"]).max()


@pytest.mark.parametrize("kernel", KERNELS)
def test_cfg1_closed_form_interp_first(kernel):
    """The CUDA path itself against the closed forms of the hyperbolic field (north_star): Q = e^{2kh} + e^{-2kh}."""
    cfg = qi.make_config("cfg1")
    g, c = run_both(cfg["grid"], cfg["B"], "f64", cfg["seeds"], cfg["box_lo"], cfg["box_hi"], interp_mode=qsl.QSL_INTERP_FIRST,
                    flags=kernel)
    compare_trace(g, c, cfg["box_lo"], cfg["box_hi"], label="cfg1 interp-first")
    s = cfg["seeds"]; k = 2.0
    top = np.abs(s[:, 0]) <= math.exp(-k)
    qb = np.where(top, 2 * math.cosh(2 * k), k * (s[:, 0] ** 2 + s[:, 1] ** 2) + 1 / (k * s[:, 0] ** 2))
    assert np.abs(g["q_bnd"] / qb - 1).max() < 1e-9
    assert np.allclose(g["q_bnd"][top], 54.61646567, rtol=1e-9)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("sample_type", ["f32", "f64"])
@pytest.mark.parametrize("mode", [qsl.QSL_TRACE_L, qsl.QSL_TRACE_LQ])
def test_quadrupole_volume_seeds(sample_type, mode, kernel):
    """cfg3-like: quadrupole, bidirectional lines from a vertical slice, ragged lengths, both storage types."""
    cfg = qi.make_config("cfg3", scale=0.25)                         # 32^3 grid
    rng = np.random.default_rng(21)
    seeds = cfg["seeds"][rng.choice(len(cfg["seeds"]), 3000, replace=False)]
    g, c = run_both(cfg["grid"], cfg["B"], sample_type, seeds, cfg["box_lo"], cfg["box_hi"], mode=mode,
                    max_steps=cfg["max_steps"], flags=kernel)
    compare_trace(g, c, cfg["box_lo"], cfg["box_hi"], with_q=mode == qsl.QSL_TRACE_LQ, label="quad")


@pytest.mark.parametrize("kernel", KERNELS)
def test_P12_gpu_L_mode_bit_identical_to_LQ(kernel):
    cfg = qi.make_config("cfg3", scale=0.25)
    seeds = cfg["seeds"][::41]
    fg = gpu_field(cfg["grid"], cfg["B"], "f64", 0)
    s = torch.from_numpy(seeds).cuda()
    mk = lambda m: qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], mode=m, max_steps=cfg["max_steps"], flags=kernel)
    a = qsl.qsl_trace(fg, s, mk(qsl.QSL_TRACE_LQ))
    b = qsl.qsl_trace(fg, s, mk(qsl.QSL_TRACE_L))
    for k in ("end_f", "end_b", "L", "face_f", "face_b", "nsteps_f", "nsteps_b", "status"):
        assert torch.equal(a[k], b[k]), k
    assert torch.isnan(b["q_perp"]).all()


@pytest.mark.parametrize("kernel", KERNELS)
def test_stretched_grid_and_euler(kernel):
    g = qi.Grid.from_axes(qi.stretched_axis(40, -1, 1, 3.0), qi.stretched_axis(36, -1, 1, 0.4), qi.stretched_axis(44, 0, 1, 5.0))
    B = qi.hyperbolic_field(g, 2.0)
    rng = np.random.default_rng(22)
    seeds = np.stack([rng.uniform(-0.5, 0.5, 500), rng.uniform(-0.5, 0.5, 500), rng.uniform(0, 0.9, 500)], 1)
    lo, hi = (-1, -1, 0), (1, 1, 1)
    for interp in (0, 1):
        gg, c = run_both(g, B, "f64", seeds, lo, hi, interp_mode=interp, flags=kernel)
        compare_trace(gg, c, lo, hi, label="stretched interp=%d" % interp)
    gg, c = run_both(g, B, "f64", seeds, lo, hi, method=qsl.QSL_EULER, step_frac=0.2, flags=kernel)
    compare_trace(gg, c, lo, hi, label="stretched euler")


@pytest.mark.parametrize("kernel", KERNELS)
def test_edge_cases_status_caps_empty(kernel):
    cfg = qi.make_config("cfg1", scale=0.25)
    lo, hi = cfg["box_lo"], cfg["box_hi"]
    seeds = np.array([[0.0, 0.0, 0.5], [2.0, 0.0, 0.5], [0.1, 0.1, 0.2], [1.0, 1.0, 1.0], [-1.0, 0.3, 0.0], [0.3, 0.2, 0.0]])
    for kw in (dict(max_steps=3), dict(max_length=0.1), dict()):
        g, c = run_both(cfg["grid"], cfg["B"], "f64", seeds, lo, hi, flags=kernel, **kw)
        compare_trace(g, c, lo, hi, frac=1.0, label=str(kw))
        assert np.array_equal(g["status"], c["status"])
    # raised lower boundary
    g, c = run_both(cfg["grid"], cfg["B"], "f64", seeds, (-1, -1, 0.25), hi, flags=kernel)
    compare_trace(g, c, (-1, -1, 0.25), hi, frac=1.0, label="raised")
    # null field
    gz = qi.Grid.uniform((8, 8, 8), lo, hi)
    g, c = run_both(gz, tuple(np.zeros(gz.shape) for _ in range(3)), "f64", seeds[:3], lo, hi, flags=kernel)
    assert np.array_equal(g["status"], c["status"]) and np.isnan(g["q_perp"]).all()
    # n = 0
    fg = gpu_field(cfg["grid"], cfg["B"], "f64", 0)
    out = qsl.qsl_trace(fg, torch.empty((0, 3), dtype=torch.float64, device="cuda"), qsl.make_trace_params(lo, hi))
    assert out["L"].numel() == 0
    # a ragged tail: n not a multiple of the block or warp size
    g, c = run_both(cfg["grid"], cfg["B"], "f64", cfg["seeds"][:131], lo, hi, flags=kernel)
    compare_trace(g, c, lo, hi, frac=1.0, label="tail")


@pytest.mark.parametrize("method", ["rk4", "ck45"])
@pytest.mark.parametrize("kernel", KERNELS)
def test_non_finite_seeds_and_seeds_on_faces_edges_corners(kernel, method):
    """Degenerate seeds: NaN / +-inf coordinates are SEED_OUTSIDE with NaN outputs (no lane may wander off with them), seeds
    exactly on a face, an edge or a corner of the closed trace box (O2: box_lo <= x <= box_hi) start, leave through the
    face the oracle names after the same number of steps and give the same L and Q."""
    cfg = qi.make_config("cfg1", scale=0.25)
    lo, hi = cfg["box_lo"], cfg["box_hi"]
    seeds = np.array([[np.nan, 0, 0.5], [0, np.inf, 0.5], [0, 0, -np.inf], [lo[0], lo[1], lo[2]], [hi[0], hi[1], hi[2]],
                      [lo[0], 0.1, 0.5], [0.2, hi[1], 0.0], [0.0, 0.0, hi[2]], [0.3, -0.2, 0.5], [lo[0], hi[1], 0.25],
                      [np.nan, np.nan, np.nan], [hi[0], 0.0, lo[2]]])
    seeds = np.concatenate([seeds, cfg["seeds"][:53]])                    # + ordinary lines around them in the same warps
    kw = dict(method=qsl.QSL_CK45, tol=1e-4) if method == "ck45" else {}
    g, c = run_both(cfg["grid"], cfg["B"], "f64", seeds, lo, hi, flags=kernel, **kw)
    compare_trace(g, c, lo, hi, frac=1.0, label="degenerate seeds")
    assert np.array_equal(g["status"], c["status"]) and np.array_equal(g["face_f"], c["face_f"])
    assert np.array_equal(g["face_b"], c["face_b"])
    bad = np.array([0, 1, 2, 10])
    assert (c["status"][bad] & 1).all() and (g["status"][bad] & 1).all()       # SEED_OUTSIDE
    for k in ("L", "q_perp", "q_bnd"):
        assert np.isnan(g[k][bad]).all(), k
        assert np.array_equal(np.isnan(g[k]), np.isnan(c[k])), k
    assert np.isnan(g["end_f"][bad]).all() and np.isnan(g["end_b"][bad]).all()
    assert (g["nsteps_f"][bad] == 0).all() and (g["nsteps_b"][bad] == 0).all()


def test_bad_arguments_are_reported_not_crashed():
    cfg = qi.make_config("cfg1", scale=0.25)
    fg = gpu_field(cfg["grid"], cfg["B"], "f64", 0)
    s = torch.zeros((4, 3), dtype=torch.float64, device="cuda")
    with pytest.raises(qsl.QslError):
        qsl.qsl_trace(fg, s, qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], step_frac=0.0))
    with pytest.raises(qsl.QslError):
        qsl.qsl_trace(fg, s, qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], method=7))
    with pytest.raises(qsl.QslError):
        z = torch.zeros(8, dtype=torch.float64, device="cuda")
        qsl.qsl_field_create(1, 2, 4, z, z, z, lo=(0, 0, 0), hi=(1, 1, 1))


def test_nodes_only_layout_uses_corner_kernel_and_matches():
    """QSL_LAYOUT_NODES_ONLY keeps no per-cell table (6x / 12x less HBM); qsl_trace then runs the corner kernel."""
    cfg = qi.make_config("cfg3", scale=0.25)
    seeds = cfg["seeds"][::37]
    dev = [torch.from_numpy(np.ascontiguousarray(a).reshape(-1)).cuda() for a in cfg["B"]]
    gr = cfg["grid"]
    ft = qsl.qsl_field_create(gr.nx, gr.ny, gr.nz, *dev, lo=gr.lo, hi=gr.hi)
    fn = qsl.qsl_field_create(gr.nx, gr.ny, gr.nz, *dev, lo=gr.lo, hi=gr.hi, layout=qsl.QSL_LAYOUT_NODES_ONLY)
    n_nodes, n_cells = gr.nx * gr.ny * gr.nz, (gr.nx - 1) * (gr.ny - 1) * (gr.nz - 1)
    assert fn.nbytes < n_nodes * 32 + 4096 and ft.nbytes >= n_nodes * 32 + n_cells * 192
    s = torch.from_numpy(seeds).cuda()
    p = qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], max_steps=cfg["max_steps"])
    pv1 = qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], max_steps=cfg["max_steps"], flags=V1)
    a, b = qsl.qsl_trace(fn, s, p), qsl.qsl_trace(ft, s, pv1)
    for k in a:
        assert torch.equal(a[k], b[k]) or (torch.isnan(a[k]) == torch.isnan(b[k])).all() and torch.equal(
            torch.nan_to_num(a[k]), torch.nan_to_num(b[k])), k


@pytest.mark.parametrize("chunks", [1, 3, None])
def test_trace_host_pipelined_equals_one_call(chunks):
    """driver.trace_host (pinned host buffers, pieces alternating between two streams) returns exactly what one qsl_trace
    call returns: lines are independent, so cutting the seed set changes nothing."""
    cfg = qi.make_config("cfg1", scale=0.5)
    fg = gpu_field(cfg["grid"], cfg["B"], "f64", 0)
    p = qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], max_steps=cfg["max_steps"])
    outs = ("end_f", "end_b", "L", "q_perp", "q_bnd", "face_f", "face_b", "status", "nsteps_f")
    seeds_host = torch.from_numpy(np.ascontiguousarray(cfg["seeds"])).pin_memory()
    h = qsl.trace_host(fg, seeds_host, p, outputs=outs, chunks=chunks)
    torch.cuda.synchronize()
    g = qsl.qsl_trace(fg, seeds_host.cuda(), p, outputs=outs)
    torch.cuda.synchronize()
    for k in outs:
        assert h[k].is_pinned() and torch.equal(h[k], g[k].cpu()), k
    assert qsl.trace_host(fg, seeds_host[:0], p, outputs=("L",)) == {}
    fg.destroy()


@pytest.mark.parametrize("n", [1, 2, 3, 7, 8, 9, 31, 32, 33, 257])
@pytest.mark.parametrize("mode", [qsl.QSL_TRACE_L, qsl.QSL_TRACE_LQ])
def test_small_launches_staging_and_landing_kernel(n, mode):
    """Launch sizes around the staging chunk (8 items per counter pop) and the warp size: every line is traced once and
    landed once (records written by the trace kernel and rewritten by the landing kernel), and total_steps is the sum
    of the per-line step counts of both kernels."""
    cfg = qi.make_config("cfg3", scale=0.25)
    rng = np.random.default_rng(1000 + n)
    seeds = cfg["seeds"][rng.choice(len(cfg["seeds"]), n, replace=False)]
    g, c = run_both(cfg["grid"], cfg["B"], "f64", seeds, cfg["box_lo"], cfg["box_hi"], mode=mode, max_steps=cfg["max_steps"])
    compare_trace(g, c, cfg["box_lo"], cfg["box_hi"], with_q=mode == qsl.QSL_TRACE_LQ, frac=1.0, label="small n=%d" % n)
    assert np.array_equal(g["status"], c["status"])
    assert g["total_steps"] == int(g["nsteps_f"].astype(np.int64).sum() + g["nsteps_b"].astype(np.int64).sum())
    assert g["total_steps"] == int(c["nsteps_f"].astype(np.int64).sum() + c["nsteps_b"].astype(np.int64).sum())

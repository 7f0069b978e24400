"""GPU parity of FLEDGE (a7), threshold + refinement (a8), the seed sort (a2) and the level loop (a9) against the
oracle.  Inputs are seeded random maps or the oracle's own intermediate products (never the other way round)."""
import ctypes as C
import math

import numpy as np
import pytest
import torch

import oracle
import paper_1609_00724_b200 as qsl
import qsl_inputs as qi
from tests.parity import compare_trace, gpu_field, oracle_pipeline

pytestmark = pytest.mark.gpu


def _cuda(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("shape", [(13, 17), (1, 9), (8, 1), (64, 95), (6, 7, 9), (5, 4, 1), (2, 2, 2), (33, 31, 70), (1, 1, 1),
                                   # bands / groups / plane chunks of the dense kernels with ragged ends: 2-D rows per band
                                   # 16 .. 64 in groups of 8, strips of 30 columns; 3-D bands of 2 rows, chunks of 64 planes
                                   (65, 61), (129, 30), (17, 31), (300, 1), (2, 200), (9, 3, 2), (8, 1, 1), (67, 5, 33),
                                   (130, 2, 61), (64, 3, 30), (65, 7, 1)])
def test_fledge_dense_matches_oracle(shape):
    rng = np.random.default_rng(30)
    V = rng.uniform(0.1, 3.0, size=shape)
    if V.size > 20:
        V.reshape(-1)[7] = np.nan
    S = qsl.qsl_fledge_dense(_cuda(V), V.ndim).cpu().numpy()
    ref = oracle.fledge_dense(V, V.ndim)
    assert np.array_equal(np.isnan(S), np.isnan(ref))
    ok = ~np.isnan(ref)
    assert np.abs(S[ok] - ref[ok]).max() <= 1e-13 * 32 * 3.0      # |weights| sum to 32 in 3-D


def test_fledge_dense_full_size_sampled():
    """cfg3's 2048x1024 and a 3-D 256x256x128 map in the bench's launch configuration; sampled outputs vs the oracle
    evaluated one by one is the same as the whole map here, since the oracle finishes in seconds."""
    rng = np.random.default_rng(31)
    for shape in ((1024, 2048), (128, 256, 256)):
        V = rng.uniform(0.1, 3.0, size=shape)
        S = qsl.qsl_fledge_dense(_cuda(V), V.ndim).cpu().numpy()
        ref = oracle.fledge_dense(V, V.ndim)
        assert np.abs(S - ref).max() <= 1e-12


@pytest.mark.parametrize("shape", [(16384, 16384), (512, 1024, 1024)])
def test_fledge_dense_more_tasks_than_the_grid_sampled(shape):
    """Maps with more strips x bands (x chunks) than the dense kernels launch CTAs (a few waves of single-warp CTAs per SM),
    so that their task loops stride: sub-blocks (corners, edges, interior, across band / chunk borders) against the
    oracle run on the sub-block with one halo cell (the Sobel stencil reaches no further; at the map's edge the
    sub-block's own edge replication is the map's)."""
    g = torch.Generator(device="cuda"); g.manual_seed(36)
    L = torch.rand(shape, dtype=torch.float64, device="cuda", generator=g) * 3.0 + 0.1
    nd = len(shape)
    L.view(-1)[12345] = float("nan")
    S = qsl.qsl_fledge_dense(L, nd)
    torch.cuda.synchronize()
    rng = np.random.default_rng(37)
    ext = 40 if nd == 2 else 12
    starts = [tuple(0 for _ in shape), tuple(n - ext for n in shape)]
    starts += [tuple(int(rng.integers(0, n - ext)) for n in shape) for _ in range(6)]
    starts += [tuple(min(max(v, 0), n - ext) for v, n in zip((60, 25) if nd == 2 else (58, 1, 25), shape))]   # band / chunk borders
    if nd == 2:
        starts.append((max(12345 // shape[1] - 3, 0), max(12345 % shape[1] - 3, 0)))                        # around the NaN
    for st in starts:
        lo = [max(a - 1, 0) for a in st]
        hi = [min(a + ext + 1, n) for a, n in zip(st, shape)]
        sl = tuple(slice(a, b) for a, b in zip(lo, hi))
        ref = oracle.fledge_dense(L[sl].cpu().numpy(), nd)
        inner = tuple(slice(a - l, a - l + ext) for a, l in zip(st, lo))
        got = S[tuple(slice(a, a + ext) for a in st)].cpu().numpy()
        want = ref[inner]
        assert np.array_equal(np.isnan(got), np.isnan(want)), st
        ok = ~np.isnan(want)
        assert np.abs(got[ok] - want[ok]).max() <= 1e-12, st


@pytest.mark.parametrize("n", [1, 2, 19, 255, 256, 257, 4097, 1 << 20])
def test_select_exact(n):
    rng = np.random.default_rng(32)
    S = rng.exponential(size=n)
    S[rng.random(n) < 0.1] = np.nan
    if n > 5:
        S[3] = np.inf; S[4] = S[5]; S[0] = 0.0
    for p in (0.95, 0.5, 0.999, 1.0, 0.0):
        tau = float(qsl.qsl_select(_cuda(S), p).item())
        ref = oracle.select(S, p)
        assert (math.isnan(tau) and math.isnan(ref)) or tau == ref, (n, p, tau, ref)


def test_select_negative_values_and_all_nan():
    rng = np.random.default_rng(33)
    S = rng.normal(size=5000)
    assert float(qsl.qsl_select(_cuda(S), 0.3).item()) == oracle.select(S, 0.3)
    assert math.isnan(float(qsl.qsl_select(_cuda(np.full(10, np.nan)), 0.95).item()))


@pytest.mark.parametrize("kind", ["fledge_like", "constant", "two_values", "one_block", "negative", "tiny_bucket"])
def test_select_candidate_compaction_paths(kind):
    """qsl_select on maps large enough for the candidate compaction of pass 2 (n >= 65536), chosen so that every branch
    runs: candidates kept (fledge_like, tiny_bucket, negative), too many candidates -> every pass reads S (constant,
    two_values), candidates of the answer's bucket all in the elements of ONE block of the grid-stride loop -> its
    segment overflows -> fallback (one_block).  Exact against the sorted definition (nearest rank)."""
    rng = np.random.default_rng(35)
    n = (1 << 22) + 777
    if kind == "fledge_like":
        S = np.abs(rng.normal(10.0, 3.0, size=n)); S[rng.random(n) < 0.01] = np.nan
        ps = (0.95, 0.5, 0.001)
    elif kind == "constant":
        S = np.full(n, 3.25); ps = (0.95, 0.0, 1.0)
    elif kind == "two_values":
        S = np.where(rng.random(n) < 0.5, 1.5, 1.5 + 2.0 ** -40); ps = (0.95, 0.25, 0.5)
    elif kind == "negative":
        S = -np.abs(rng.normal(10.0, 3.0, size=n)); S[::5] = rng.normal(size=len(S[::5])); ps = (0.95, 0.05, 0.5)
    elif kind == "tiny_bucket":
        S = rng.uniform(100.0, 200.0, size=n); S[:40] = 1.0 + np.arange(40) * 2.0 ** -45; ps = (5e-6, 9.5e-6, 0.95)
    else:
        # the smallest values (one 16-bit bucket: [1, 1.0625)) sit only where block 0 of the grid-stride loop reads
        blocks = torch.cuda.get_device_properties(0).multi_processor_count * 8
        stride = blocks * 256
        S = rng.uniform(100.0, 200.0, size=n)
        idx = np.arange(n)
        own = (idx % stride) < 256
        S[own] = 1.0 + rng.random(int(own.sum())) * 0.0624
        assert own.sum() > (n // 4) // blocks                      # more than one segment holds
        ps = (0.5 * own.sum() / n, 0.95, 1e-7)
    d = _cuda(S)
    for p in ps:
        tau = float(qsl.qsl_select(d, p).item())
        ref = oracle.select(S, p)
        assert (math.isnan(tau) and math.isnan(ref)) or tau == ref, (kind, p, tau, ref)


@pytest.mark.parametrize("ndim", [2, 3])
def test_refine_bit_exact_two_levels(ndim):
    rng = np.random.default_rng(34)
    if ndim == 2:
        lat = qi.Lattice(2, (96, 70, 1), (-0.6, 0.0, 0.0), (1.2, 0, 0), (0, 0, 0.5))
    else:
        lat = qi.Lattice(3, (20, 18, 12), (0.0, 0.1, 0.0), (1.0, 0, 0.1), (0, 0.9, 0), (0.05, 0, 0.5))
    n = lat.count
    shape = tuple(lat.n[:ndim][::-1])
    c0 = np.stack(np.unravel_index(np.arange(n), shape), 1)[:, ::-1].astype(np.uint32)
    S = rng.exponential(size=n); S[::17] = np.nan
    tau = oracle.select(S, 0.9)
    tau_d = _cuda(np.array([tau]))
    cc, cs, cb = qsl.qsl_refine(lat, 0, None, _cuda(S), tau_d)
    rc, rs = oracle.refine(ndim, 0, c0, S, tau, lat)
    assert np.array_equal(cc.cpu().numpy().view(np.uint32), rc)
    assert np.array_equal(cs.cpu().numpy(), rs)                       # bit-exact positions
    cbn = cb.cpu().numpy()
    flagged = S > tau
    assert np.array_equal(cbn >= 0, flagged)
    assert np.array_equal(cbn[flagged], np.arange(flagged.sum()) << ndim)
    # explicit coords give the same result as the implicit dense lattice
    cc2, cs2, _ = qsl.qsl_refine(lat, 0, _cuda(c0.view(np.int32)), _cuda(S), tau_d)
    assert torch.equal(cc, cc2) and torch.equal(cs, cs2)
    # level 1 -> 2
    S1 = rng.exponential(size=len(rc)); S1[0] = tau
    cc3, cs3, _ = qsl.qsl_refine(lat, 1, cc, _cuda(S1), tau_d)
    r3, s3 = oracle.refine(ndim, 1, rc, S1, tau, lat)
    assert np.array_equal(cc3.cpu().numpy().view(np.uint32), r3) and np.array_equal(cs3.cpu().numpy(), s3)
    # nothing flagged / capacity overflow is reported
    cc4, _, cb4 = qsl.qsl_refine(lat, 0, None, _cuda(S), _cuda(np.array([np.inf])))
    assert cc4.shape[0] == 0 and bool((cb4 == -1).all())
    with pytest.raises(qsl.QslError):
        qsl.qsl_refine(lat, 0, None, _cuda(S), tau_d, capacity=8)


@pytest.mark.parametrize("n,bits", [(1, 8), (31, 5), (2048, 16), (2049, 30), (100003, 30), (1 << 20, 24)])
def test_radix_sort_pairs_stable(n, bits):
    rng = np.random.default_rng(35)
    keys = rng.integers(0, 1 << bits, size=n, dtype=np.uint32)
    vals = np.arange(n, dtype=np.uint32)
    k = _cuda(keys.view(np.int32)); v = _cuda(vals.view(np.int32))
    rc = qsl.lib().qsl_debug_sort_pairs(C.c_void_p(k.data_ptr()), C.c_void_p(v.data_ptr()), C.c_longlong(n), C.c_int(bits),
                                        C.c_void_p(torch.cuda.current_stream().cuda_stream))
    assert rc == 0
    order = np.argsort(keys, kind="stable")
    assert np.array_equal(k.cpu().numpy().view(np.uint32), keys[order])
    assert np.array_equal(v.cpu().numpy().view(np.uint32), vals[order])


@pytest.mark.parametrize("kind", ["all_equal", "sorted", "reversed", "three_values", "runs_of_40", "one_odd_lane"])
def test_radix_sort_pairs_structured_keys(kind):
    """Keys as a seed lattice produces them - long runs of one digit, whole warps with the same digit, a single lane that
    differs - through the warp-vote ranking of the scatter kernel; stable, bit-exact against numpy."""
    n = 70001
    i = np.arange(n, dtype=np.uint32)
    keys = {"all_equal": np.full(n, 0x2a5a5a5a, dtype=np.uint32), "sorted": i * 3, "reversed": (n - i) * 5,
            "three_values": np.array([7, 0x10007, 0x3fffffff], dtype=np.uint32)[i % 3], "runs_of_40": (i // 40) * 0x01010101 % (1 << 30),
            "one_odd_lane": np.where(i % 32 == 17, 0x12345, 0x12344).astype(np.uint32)}[kind].astype(np.uint32)
    vals = np.arange(n, dtype=np.uint32)
    k = _cuda(keys.view(np.int32)); v = _cuda(vals.view(np.int32))
    rc = qsl.lib().qsl_debug_sort_pairs(C.c_void_p(k.data_ptr()), C.c_void_p(v.data_ptr()), C.c_longlong(n), C.c_int(30),
                                        C.c_void_p(torch.cuda.current_stream().cuda_stream))
    assert rc == 0
    order = np.argsort(keys, kind="stable")
    assert np.array_equal(k.cpu().numpy().view(np.uint32), keys[order])
    assert np.array_equal(v.cpu().numpy().view(np.uint32), vals[order])


@pytest.mark.parametrize("name,scale", [("cfg3", 1 / 16), ("cfg5", 1 / 16)])
def test_level_loop_stagewise_against_oracle(name, scale):
    """a9: every stage of the level loop fed with the ORACLE's products of the previous stage."""
    cfg = qi.make_config(name, scale=scale)
    ref = oracle_pipeline(cfg)
    lat = cfg["lattice"]; ndim = lat.ndim
    shape = tuple(int(v) for v in lat.n[:ndim][::-1])
    fg = gpu_field(cfg["grid"], cfg["B"], cfg["sample_type"], 0)
    # FLEDGE + threshold on the oracle's level-0 lengths
    S0 = qsl.qsl_fledge_dense(_cuda(ref["L0"].reshape(shape)), ndim).view(-1)
    assert np.abs(S0.cpu().numpy() - ref["S0"]).max() <= 1e-12
    assert float(qsl.qsl_select(_cuda(ref["S0"]), cfg["p"]).item()) == ref["tau"]
    tau_d = _cuda(np.array([ref["tau"]]))
    child_base = []
    coords_g = [None]; Ls_g = [_cuda(ref["L0"])]
    assert len(ref["coords"]) >= 3, "refinement must actually refine at this size"
    for level in range(len(ref["coords"]) - 1):
        Sin = ref["S"][level]
        cin = None if level == 0 else _cuda(ref["coords"][level].view(np.int32))
        cc, cs, cb = qsl.qsl_refine(lat, level, cin, _cuda(Sin), tau_d)
        assert np.array_equal(cc.cpu().numpy().view(np.uint32), ref["coords"][level + 1])       # bit-exact seed sets
        assert np.array_equal(cs.cpu().numpy(), ref["seeds"][level + 1])
        child_base.append(cb); coords_g.append(cc)
        if level + 1 >= len(ref["out"]):
            break
        # trace of the refined seeds (with Q)
        params = qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], mode=qsl.QSL_TRACE_LQ, max_steps=cfg["max_steps"])
        tot = torch.zeros(1, dtype=torch.int64, device="cuda")
        g = qsl.qsl_trace(fg, cs, params, total_steps=tot)
        g = {k: v.cpu().numpy() for k, v in g.items()}
        for k in ("status", "nsteps_f", "nsteps_b"):
            g[k] = g[k].view(np.uint32)
        g["total_steps"] = int(tot.item())
        compare_trace(g, ref["out"][level + 1], cfg["box_lo"], cfg["box_hi"], label="%s level %d" % (name, level + 1))   # north_star gate: 99.9 %
        Ls_g.append(_cuda(ref["out"][level + 1]["L"]))
        if level + 1 < len(ref["S"]):
            S = qsl.qsl_fledge_sparse(lat, level + 1, Ls_g[0], coords_g, Ls_g, child_base)
            assert np.abs(S.cpu().numpy() - ref["S"][level + 1]).max() <= 1e-12, level


def test_level_loop_end_to_end_close_to_oracle():
    """The whole GPU level loop on its own products: level sizes track the oracle's (they may differ only where a
    FLEDGE value sits within rounding of tau)."""
    cfg = qi.make_config("cfg3", scale=1 / 16)
    ref = oracle_pipeline(cfg)
    fg = gpu_field(cfg["grid"], cfg["B"], cfg["sample_type"], 0)
    pL = qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], mode=qsl.QSL_TRACE_L, max_steps=cfg["max_steps"])
    pQ = qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], mode=qsl.QSL_TRACE_LQ, max_steps=cfg["max_steps"])
    res = qsl.adaptive_map(fg, cfg["lattice"], _cuda(cfg["seeds"]), pL, pQ, cfg["levels"], cfg["p"])
    assert abs(float(res["tau"].item()) / ref["tau"] - 1) < 1e-8
    for l in range(1, len(ref["coords"])):
        a, b = res["coords"][l].shape[0], len(ref["coords"][l])
        assert abs(a - b) <= max(8, 0.01 * b), (l, a, b)
    nsteps = sum(int(o["nsteps_f"].astype(np.int64).sum() + o["nsteps_b"].astype(np.int64).sum()) for o in ref["out"])
    assert abs(int(res["total_steps"].item()) - nsteps) <= 0.02 * nsteps


def test_adaptive_map_on_a_non_default_stream():
    """`stream=` must carry the torch-side work too (allocations, step-counter sums).  The level loop on a side
    stream, with the default stream kept busy, gives the same products and step counts as the default-stream run."""
    cfg = qi.make_config("cfg3", scale=1 / 16)
    fg = gpu_field(cfg["grid"], cfg["B"], cfg["sample_type"], 0)
    pL = qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], mode=qsl.QSL_TRACE_L, max_steps=cfg["max_steps"])
    pQ = qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], mode=qsl.QSL_TRACE_LQ, max_steps=cfg["max_steps"])
    seeds = _cuda(cfg["seeds"])
    ref = qsl.adaptive_map(fg, cfg["lattice"], seeds, pL, pQ, cfg["levels"], cfg["p"])
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    busy = torch.empty(1 << 26, dtype=torch.float32, device="cuda")
    for _ in range(8):
        busy.normal_()                                   # work queued on the default stream while the side stream runs
    res = qsl.adaptive_map(fg, cfg["lattice"], seeds, pL, pQ, cfg["levels"], cfg["p"], stream=side)
    side.synchronize()
    assert torch.equal(res["steps_by_mode"], ref["steps_by_mode"]) and torch.equal(res["total_steps"], ref["total_steps"])
    assert int(res["steps_by_mode"][0]) > 0 and int(res["steps_by_mode"][1]) > 0
    assert torch.equal(res["tau"], ref["tau"]) and torch.equal(res["L0"], ref["L0"])
    for l in range(1, len(ref["coords"])):
        assert torch.equal(res["coords"][l], ref["coords"][l]) and torch.equal(res["seeds"][l], ref["seeds"][l])
        if ref["out"][l] is not None:
            for k in ("L", "q_perp", "q_bnd", "status"):
                assert torch.equal(res["out"][l][k].view(torch.int64 if k != "status" else torch.int32),
                                   ref["out"][l][k].view(torch.int64 if k != "status" else torch.int32)), (l, k)
    torch.cuda.synchronize()
    fg.destroy()

"""GPU parity of the Hilbert-curve refinement kernels against oracle/hilbert.py.
Integer work (keys, cells, sort, insertion lists, merge) is bit-exact; sample positions are bit-exact (one IEEE division
and an fma chain on both sides); the converter's interpolated values agree to 1e-12 relative (log10 / pow of two maths
libraries), its max-rule values exactly."""
import numpy as np
import pytest
import torch

import oracle
import paper_1609_00724_b200 as qsl
import qsl_inputs as qi
from oracle import hilbert as H

pytestmark = pytest.mark.gpu


def _lat(nd, n):
    if nd == 2:
        return qi.Lattice(2, (n[0], n[1], 1), (0.1, -0.2, 0.3), (1.2, 0.0, 0.0), (0.0, 0.0, 0.7))
    return qi.Lattice(3, tuple(n), (0.0, 0.0, 0.0), (1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (0.0, 0.0, 0.5))


@pytest.mark.parametrize("nd,bits,shift", [(2, 1, 0), (2, 7, 0), (2, 16, 3), (2, 31, 5), (3, 1, 0), (3, 5, 0), (3, 12, 7), (3, 21, 1)])
def test_keys_and_cells_bit_exact(nd, bits, shift):
    rng = np.random.default_rng(bits * 10 + nd)
    n = 3000
    hi = (1 << bits) - shift
    c = rng.integers(0, max(hi, 1), size=(n, nd), dtype=np.int64)
    c[0] = 0; c[1] = max(hi - 1, 0)
    want = H.keys_of(c, bits, shift)
    got = qsl.qsl_hilbert_keys(torch.from_numpy(c.astype(np.int32)).cuda(), bits, shift)
    assert np.array_equal(got.cpu().numpy().view(np.uint64), want)
    back = qsl.qsl_hilbert_cells(got, nd, bits, shift).cpu().numpy()
    assert np.array_equal(back, c.astype(np.int32))


def test_shift_out_of_range_is_rejected():
    """a shift that would push cells out of the curve's cube must be an error, not wrong keys."""
    c = torch.zeros((4, 2), dtype=torch.int32, device="cuda")
    with pytest.raises(qsl.QslError):
        qsl.qsl_hilbert_keys(c, 3, 8)
    k = qsl.qsl_hilbert_keys(c, 3, 7)
    with pytest.raises(qsl.QslError):
        qsl.qsl_hilbert_cells(k, 2, 3, 8)
    lat = _lat(2, (8, 4))
    bits = qsl.qsl_hilbert_bits(lat, 1)                                        # 4 bits: cube of 16 cells per axis
    keys = torch.arange(4, dtype=torch.int64, device="cuda")
    L = torch.ones(4, dtype=torch.float64, device="cuda")
    with pytest.raises(qsl.QslError):
        qsl.qsl_hilbert_refine(lat, 1, (1 << bits) + 1, keys, L, 0.1)


@pytest.mark.parametrize("n", [0, 1, 5, 4097, 100003])
def test_sort_keys64_and_gather(n):
    rng = np.random.default_rng(n)
    k = rng.integers(0, 1 << 62, size=n, dtype=np.int64)
    if n > 10:
        k[5] = k[7]                                                            # equal keys keep their order (stable)
    payload = rng.normal(size=(n, 3))
    kk = torch.from_numpy(k.copy()).cuda()
    perm = qsl.qsl_sort_keys64(kk, 62)
    o = np.argsort(k, kind="stable")
    assert np.array_equal(kk.cpu().numpy(), k[o]) and np.array_equal(perm.cpu().numpy(), o.astype(np.int32))
    if n:
        g = qsl.qsl_gather(perm, torch.from_numpy(payload).cuda())
        assert np.array_equal(g.cpu().numpy(), payload[o])


@pytest.mark.parametrize("nd,n,R", [(2, (8, 4), 3), (2, (13, 7), 2), (3, (4, 4, 2), 2), (3, (5, 3, 6), 1)])
def test_level0_refine_merge_against_the_oracle(nd, n, R):
    lat = _lat(nd, n)
    bits = H.curve_bits(n, R)
    assert qsl.qsl_hilbert_bits(lat, R) == bits
    c0, s0 = qsl.qsl_hilbert_level0(lat, R)
    keys = qsl.qsl_hilbert_keys(c0, bits)
    perm = qsl.qsl_sort_keys64(keys, bits * nd)
    c0, s0 = qsl.qsl_gather(perm, c0), qsl.qsl_gather(perm, s0)
    wk, wc = H.level0(lat, R)
    assert np.array_equal(keys.cpu().numpy().view(np.uint64), wk) and np.array_equal(c0.cpu().numpy(), wc.astype(np.int32))
    assert np.array_equal(s0.cpu().numpy(), H.positions(lat, R, wc))           # bit-exact positions
    rng = np.random.default_rng(4)
    L = rng.choice([1.0, 1.3, 2.5, np.nan, np.inf], size=len(wk), p=[0.4, 0.3, 0.2, 0.05, 0.05])
    for shift in (0, 3):
        if shift:
            ks = H.keys_of(wc, bits + 1, shift)
            o = np.argsort(ks, kind="stable")
            ks_o, L_o, wc_o = ks[o], L[o], wc[o]
        else:
            ks_o, L_o, wc_o = wk, L, wc
        left, nk, nc = H.refine_pass(lat, R, ks_o, L_o, 0.25, shift)
        gl, gc, gs = qsl.qsl_hilbert_refine(lat, R, shift, torch.from_numpy(ks_o.view(np.int64)).cuda(), torch.from_numpy(L_o).cuda(), 0.25)
        assert len(left) > 1
        assert np.array_equal(gl.cpu().numpy(), left) and np.array_equal(gc.cpu().numpy(), nc.astype(np.int32))
        assert np.array_equal(gs.cpu().numpy(), H.positions(lat, R, nc))
        pos_old, pos_new = H.merge(left, len(ks_o))
        want = np.empty((len(ks_o) + len(left), nd), dtype=np.int32); want[pos_old] = wc_o; want[pos_new] = nc
        got = qsl.qsl_hilbert_merge(gl, torch.from_numpy(wc_o.astype(np.int32)).cuda(), gc.contiguous())
        assert np.array_equal(got.cpu().numpy(), want)
        # capacity too small: QSL_ERANGE
        with pytest.raises(qsl.QslError):
            qsl.qsl_hilbert_refine(lat, R, shift, torch.from_numpy(ks_o.view(np.int64)).cuda(), torch.from_numpy(L_o).cuda(), 0.25, capacity=len(left) - 1)
    # nothing to do: empty, single sample, threshold above every jump
    e = qsl.qsl_hilbert_refine(lat, R, 0, keys[:1], torch.zeros(1, dtype=torch.float64, device="cuda"), 0.1)
    assert e[0].numel() == 0
    e = qsl.qsl_hilbert_refine(lat, R, 0, keys, torch.from_numpy(np.nan_to_num(L, nan=1.0, posinf=1.0)).cuda(), 10.0)
    assert e[0].numel() == 0


def _step_fn_np(seeds):
    L = np.where(seeds[:, 0] * 0.9 + seeds[:, 2] * 0.4 < 0.61, 1.0, 2.0) + 0.01 * seeds[:, 1]
    Q = 2.0 + 1.0 / (1e-3 + np.abs(seeds[:, 0] * 0.9 + seeds[:, 2] * 0.4 - 0.61))
    return L, Q


def _step_fn_torch(seeds):
    s = seeds.cpu().numpy()                                                    # the same arithmetic, so that decisions are identical
    L, Q = _step_fn_np(s)
    return torch.from_numpy(L).cuda(), torch.from_numpy(Q).cuda()


@pytest.mark.parametrize("nd,n,R,shift", [(2, (16, 8), 3, 0), (2, (16, 8), 3, 5), (3, (4, 4, 4), 2, 3)])
def test_whole_loop_and_converter_against_the_oracle(nd, n, R, shift):
    lat = _lat(nd, n)
    want = H.hilbert_map(_step_fn_np, lat, R, 0.5, 3, shift)
    got = qsl.hilbert_map(lat, R, 0.5, 3, shift, _step_fn_torch)
    assert got["counts"] == want["counts"] and want["counts"][-1] > want["counts"][0]
    assert np.array_equal(got["keys"].cpu().numpy().view(np.uint64), want["keys"])
    assert np.array_equal(got["coords"].cpu().numpy(), want["coords"].astype(np.int32))
    assert np.array_equal(got["L"].cpu().numpy(), want["L"]) and np.array_equal(got["Q"].cpu().numpy(), want["Q"])
    Q = want["Q"].copy()
    Q[::7] = np.nan                                                            # samples without a usable Q
    for r in (0, 1, R):
        w = H.convert(lat, R, r, want["keys"], Q)
        g = qsl.qsl_hilbert_convert(lat, R, r, got["keys"], torch.from_numpy(Q).cuda()).cpu().numpy().reshape(-1)
        assert np.array_equal(np.isnan(g), np.isnan(w))
        assert np.allclose(g, w, rtol=1e-12, atol=0, equal_nan=True)
        dims = [int(v) << r for v in n]                                        # cells holding a sample: the max rule, exact
        cc = want["coords"][np.isfinite(Q)] >> (R - r)
        flat = np.zeros(len(cc), dtype=np.int64)
        for d in range(nd - 1, -1, -1):
            flat = flat * dims[d] + cc[:, d]
        hit = np.zeros(len(w), dtype=bool); hit[flat] = True
        assert hit.sum() > 0 and np.array_equal(g[hit], w[hit])
        assert np.all(np.isin(g[hit], Q))
    # no sample at all: NaN map
    g = qsl.qsl_hilbert_convert(lat, R, 0, got["keys"][:0], torch.zeros(0, dtype=torch.float64, device="cuda"))
    assert torch.isnan(g).all()


def test_paper_loop_on_a_traced_field():
    """The loop with real tracing (quadrupole slice, cfg3 scaled): the GPU path and the oracle path add samples in the same
    places - identical sample sets unless a length difference sits within rounding of the threshold."""
    cfg = qi.make_config("cfg3", 1.0 / 16)
    lat = cfg["lattice"]
    R, thr = 2, 0.3
    grid = cfg["grid"]
    dev = [torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64).reshape(-1)).cuda() for a in cfg["B"]]
    f = qsl.qsl_field_create(grid.nx, grid.ny, grid.nz, *dev, lo=grid.lo, hi=grid.hi)
    p = qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], max_steps=cfg["max_steps"])
    fc = oracle.Field(grid, cfg["B"], oracle.F64, oracle.NORMALIZE_FIRST)

    def tg(seeds):
        o = qsl.qsl_trace(f, seeds, p, outputs=("L", "q_perp"))
        return o["L"], o["q_perp"]

    def tc(seeds):
        o = oracle.trace(fc, seeds, cfg["box_lo"], cfg["box_hi"], max_steps=cfg["max_steps"])
        return o["L"], o["q_perp"]

    got = qsl.hilbert_map(lat, R, thr, 2, 3, tg)
    want = H.hilbert_map(tc, lat, R, thr, 2, 3)
    assert got["counts"] == want["counts"] and want["counts"][-1] > 1.05 * want["counts"][0]
    assert np.array_equal(got["keys"].cpu().numpy().view(np.uint64), want["keys"])
    assert np.allclose(got["L"].cpu().numpy(), want["L"], rtol=1e-8, equal_nan=True)
    m = qsl.qsl_hilbert_convert(lat, R, R, got["keys"], got["Q"])
    assert m.shape == (int(lat.n[1]) << R, int(lat.n[0]) << R) and bool(torch.isfinite(m).all())
    f.destroy()


def test_hilbert_map_on_a_non_default_stream():
    """the loop on a side stream (default stream kept busy) gives the sample set of the default-stream run."""
    cfg = qi.make_config("cfg3", 1.0 / 16)
    lat, grid = cfg["lattice"], cfg["grid"]
    dev = [torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64).reshape(-1)).cuda() for a in cfg["B"]]
    f = qsl.qsl_field_create(grid.nx, grid.ny, grid.nz, *dev, lo=grid.lo, hi=grid.hi)
    p = qsl.make_trace_params(cfg["box_lo"], cfg["box_hi"], max_steps=cfg["max_steps"])

    def tg(seeds):                                                             # stream=None: torch's current stream
        o = qsl.qsl_trace(f, seeds, p, outputs=("L", "q_perp"))
        return o["L"], o["q_perp"]

    ref = qsl.hilbert_map(lat, 2, 0.3, 2, 3, tg)
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    busy = torch.empty(1 << 26, dtype=torch.float32, device="cuda")
    for _ in range(8):
        busy.normal_()
    got = qsl.hilbert_map(lat, 2, 0.3, 2, 3, tg, stream=side)
    side.synchronize()
    assert got["counts"] == ref["counts"]
    for k in ("keys", "coords", "L", "Q"):
        assert torch.equal(got[k].view(torch.int64 if got[k].dtype == torch.float64 else got[k].dtype),
                           ref[k].view(torch.int64 if ref[k].dtype == torch.float64 else ref[k].dtype)), k
    torch.cuda.synchronize()
    f.destroy()

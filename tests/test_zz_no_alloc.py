"""GPU test of the one entry point that allocates nothing, qsl_refine_noalloc (include/qsl.h): its outputs against those of
qsl_refine - bit for bit, the bar of every refinement test here (north_star: "refinement seed sets must be bit-exact") -
on calls in a row that share the library's fixed scratch array.  Collected last on purpose (file name): the suite runs
with pytest -x."""
import numpy as np
import pytest
import torch

import paper_1609_00724_b200 as qsl
import qsl_inputs as qi

pytestmark = pytest.mark.gpu


def _case(ndim, dims, seed, p=0.9):
    g = torch.Generator(device="cuda"); g.manual_seed(seed)
    n = int(np.prod(dims))
    S = torch.rand(n, dtype=torch.float64, device="cuda", generator=g)
    S[::97] = float("nan")                                       # NaN never flags
    e = [(1.0, 0, 0), (0, 0.7, 0), (0, 0, 0.5)]
    lat = qi.Lattice(ndim, tuple(dims) + (1,) * (3 - ndim), (0.1, -0.2, 0.05), e[0], e[1], e[2])
    tau = qsl.qsl_select(S, p)
    return lat, S, tau


def _buffers(n, ndim, cap):
    # poisoned, so that anything the call leaves unwritten shows up
    cc = torch.full((cap, ndim), -7, dtype=torch.int32, device="cuda")
    cs = torch.full((cap, 3), float("nan"), dtype=torch.float64, device="cuda")
    cb = torch.full((n,), -99, dtype=torch.int64, device="cuda")
    m = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    return cc, cs, cb, m


def _same(got, want):
    cc, cs, cb, m = got
    wc, ws, wb = want
    k = int(m.item())
    assert k == int(wc.shape[0])
    assert torch.equal(cc[:k], wc) and torch.equal(cs[:k].view(torch.int64), ws.view(torch.int64)) and torch.equal(cb, wb)
    assert bool((cc[k:] == -7).all())                            # nothing written beyond the children


def test_refine_noalloc_matches_refine_on_calls_in_a_row():
    cases = [_case(2, (300, 211), 1), _case(3, (40, 33, 21), 2), _case(2, (2048, 1024), 3, p=0.95), _case(2, (5, 3), 4, p=0.5)]
    want = [qsl.qsl_refine(lat, 0, None, S, tau) for lat, S, tau in cases]
    bufs = [_buffers(int(S.numel()), int(lat.ndim), int(w[0].shape[0]) + 8) for (lat, S, tau), w in zip(cases, want)]
    # back to back on one stream, large and small inputs alternating over the same scratch, each twice
    order = [0, 1, 2, 3, 2, 0, 3, 1]
    for i in order:
        lat, S, tau = cases[i]
        qsl.qsl_refine_noalloc(lat, 0, None, S, tau, *bufs[i])
    torch.cuda.synchronize()
    for i in range(len(cases)):
        _same(bufs[i], want[i])
    # a sparse level: the children of case 0 refined again (coords given, level 1)
    lat, S, tau = cases[0]
    c1 = want[0][0].contiguous()
    g = torch.Generator(device="cuda"); g.manual_seed(9)
    S1 = torch.rand(int(c1.shape[0]), dtype=torch.float64, device="cuda", generator=g)
    w1 = qsl.qsl_refine(lat, 1, c1, S1, tau)
    b1 = _buffers(int(S1.numel()), 2, int(w1[0].shape[0]))
    for _ in range(2):
        qsl.qsl_refine_noalloc(lat, 1, c1, S1, tau, *b1)
    torch.cuda.synchronize()
    _same(b1, w1)


def test_refine_noalloc_allocates_nothing_and_never_synchronises():
    """Free device memory does not move over repeated calls, and the call can be captured into a CUDA graph (a capture in
    global mode rejects cudaMalloc / cudaFree and any synchronisation); the replayed graph gives the same children."""
    lat, S, tau = _case(3, (64, 48, 40), 5)
    want = qsl.qsl_refine(lat, 0, None, S, tau)
    cap = int(want[0].shape[0])
    bufs = _buffers(int(S.numel()), 3, cap)
    qsl.qsl_refine_noalloc(lat, 0, None, S, tau, *bufs)          # first call on this device: looks up the scratch address
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        qsl.qsl_refine_noalloc(lat, 0, None, S, tau, *bufs)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    _same(bufs, want)
    bufs2 = _buffers(int(S.numel()), 3, cap)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        with torch.cuda.graph(graph, stream=side, capture_error_mode="global"):
            qsl.qsl_refine_noalloc(lat, 0, None, S, tau, *bufs2)
    torch.cuda.current_stream().wait_stream(side)
    for _ in range(2):
        graph.replay()
    torch.cuda.synchronize()
    _same(bufs2, want)


def test_refine_noalloc_rejects_more_cells_than_its_scratch_holds():
    n0, n1 = 8193, 8192                                          # 67 117 056 cells > QSL_REFINE_NOALLOC_MAX_CELLS
    assert n0 * n1 > qsl.QSL_REFINE_NOALLOC_MAX_CELLS
    lat = qi.Lattice(2, (n0, n1, 1), (0.0, 0.0, 0.0), (1.0, 0, 0), (0, 1.0, 0), (0, 0, 1.0))
    S = torch.zeros(n0 * n1, dtype=torch.float64, device="cuda")
    tau = torch.ones(1, dtype=torch.float64, device="cuda")
    cc, cs, cb, m = _buffers(1, 2, 4)
    with pytest.raises(qsl.QslError, match="no-allocation"):
        qsl.qsl_refine_noalloc(lat, 0, None, S, tau, cc, cs, None, m)
    torch.cuda.synchronize()
    assert int(m.item()) == -1 and bool((cc == -7).all())        # nothing was launched
    del S
    # the limit itself is accepted (cfg5's dense level 0: 512 x 512 x 256 cells)
    lat = qi.Lattice(3, (512, 512, 256), (0.0, 0.0, 0.0), (1.0, 0, 0), (0, 1.0, 0), (0, 0, 0.5))
    S = torch.zeros(qsl.QSL_REFINE_NOALLOC_MAX_CELLS, dtype=torch.float64, device="cuda")
    S[12345] = 2.0
    S[qsl.QSL_REFINE_NOALLOC_MAX_CELLS - 1] = 3.0
    cc, cs, cb, m = _buffers(1, 3, 16)
    qsl.qsl_refine_noalloc(lat, 0, None, S, tau, cc, cs, None, m)
    wc, ws, _ = qsl.qsl_refine(lat, 0, None, S, tau)
    torch.cuda.synchronize()
    assert int(m.item()) == 16 and torch.equal(cc, wc) and torch.equal(cs.view(torch.int64), ws.view(torch.int64))


@pytest.mark.parametrize("ndim,dims,cap", [(2, (300, 211), 1003), (3, (40, 33, 21), 4097), (2, (300, 211), 0), (3, (40, 33, 21), 5)])
def test_refine_noalloc_writes_nothing_beyond_capacity(ndim, dims, cap):
    """Buffers smaller than the child count (qsl.h: "nothing beyond capacity was written"): the first `cap` children are
    those of the full result - also when the cut falls inside a cell's group of children and inside a tile - the rows
    behind them stay untouched, child_base and the count are complete."""
    lat, S, tau = _case(ndim, dims, 11)
    wc, ws, wb = qsl.qsl_refine(lat, 0, None, S, tau)
    total = int(wc.shape[0])
    assert total > cap
    big_c = torch.full((cap + 64, ndim), -7, dtype=torch.int32, device="cuda")
    big_s = torch.full((cap + 64, 3), float("nan"), dtype=torch.float64, device="cuda")
    cb = torch.full((int(S.numel()),), -99, dtype=torch.int64, device="cuda")
    m = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    qsl.qsl_refine_noalloc(lat, 0, None, S, tau, big_c[:cap], big_s[:cap], cb, m)
    torch.cuda.synchronize()
    assert int(m.item()) == total and torch.equal(cb, wb)
    assert torch.equal(big_c[:cap], wc[:cap]) and torch.equal(big_s[:cap].view(torch.int64), ws[:cap].view(torch.int64))
    assert bool((big_c[cap:] == -7).all()) and bool(torch.isnan(big_s[cap:]).all())
    # the pooled entry point reports the overflow
    with pytest.raises(qsl.QslError):
        qsl.qsl_refine(lat, 0, None, S, tau, capacity=cap)

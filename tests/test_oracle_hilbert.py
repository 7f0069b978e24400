"""Pins of the Hilbert-curve refinement oracle (oracle/hilbert.py).  The curve is
pinned by what defines a Hilbert curve - a bijection that starts at the origin, moves by one cell along one axis per
step, visits every aligned sub-cube contiguously and ends in a corner next to the start - not by retyping the algorithm;
the refinement by its purpose (samples accumulate on the length jump; the shifted pass finds what the curve misses,
PAPER.md:204); merge and converter by brute force."""
import itertools
import math

import numpy as np
import pytest

import qsl_inputs as qi
from oracle import hilbert as H


@pytest.mark.parametrize("nd,bits", [(2, 1), (2, 2), (2, 3), (2, 5), (3, 1), (3, 2), (3, 4)])
def test_curve_is_a_hilbert_curve(nd, bits):
    n = 1 << bits
    cells = list(itertools.product(range(n), repeat=nd))
    keys = [H.hilbert_key(c, bits) for c in cells]
    assert sorted(keys) == list(range(n ** nd))                               # bijection onto [0, n^nd)
    path = [H.hilbert_cell(k, nd, bits) for k in range(n ** nd)]
    assert all(H.hilbert_key(p, bits) == k for k, p in enumerate(path))        # inverse
    assert path[0] == [0] * nd                                                # starts at the origin
    steps = np.abs(np.diff(np.array(path), axis=0))
    assert np.all(steps.sum(1) == 1)                                          # unit step along exactly one axis
    end = path[-1]
    assert sorted(end) == [0] * (nd - 1) + [n - 1]                            # ends in the corner one edge away
    # every aligned sub-cube of side 2^R is one contiguous piece of the curve (what makes "halfway along the curve
    # between two samples" a point between them in space, and an output cell of the converter a key range)
    for R in range(1, bits):
        pre = np.array([k >> (nd * R) for k in range(n ** nd)])
        coarse = np.array(path) >> R
        for p in np.unique(pre):
            assert len(np.unique(coarse[pre == p], axis=0)) == 1
        assert len(np.unique(np.concatenate([pre[:, None], coarse], 1), axis=0)) == (n >> R) ** nd


def _lat2(n0=8, n1=8):
    return qi.Lattice(2, (n0, n1, 1), (0.0, 0.0, 0.0), (1.0, 0.0, 0.0), (0.0, 1.0, 0.0))


def test_level0_positions_and_order():
    lat = _lat2(8, 4)
    R = 2
    keys, coords = H.level0(lat, R)
    assert len(keys) == 32 and np.all(np.diff(keys.astype(np.int64)) > 0)
    assert np.all(coords % 4 == 2)                                            # fine cell c0 2^R + 2^(R-1)
    pos = H.positions(lat, R, coords)
    assert np.allclose(pos[:, 0], (coords[:, 0] + 0.5) / 32) and np.allclose(pos[:, 1], (coords[:, 1] + 0.5) / 16)
    assert np.all(pos[:, 2] == 0)
    assert H.curve_bits((8, 4), 2) == 5 and H.curve_bits((5, 3), 0) == 3


def _step_trace(x_jump):
    """Field-line length with a jump across the line x = x_jump; Q large next to it."""
    def f(seeds):
        L = np.where(seeds[:, 0] < x_jump, 1.0, 2.0) + 0.01 * seeds[:, 1]
        Q = 2.0 + 1.0 / (1e-3 + np.abs(seeds[:, 0] - x_jump))
        return L, Q
    return f


def test_passes_accumulate_samples_on_the_jump_and_terminate():
    lat = _lat2(8, 8)
    R = 4
    res = H.hilbert_map(_step_trace(0.37), lat, R, thr=0.5, passes=10, shift=0)
    c = res["counts"]
    assert c[0] == 64 and all(b >= a for a, b in zip(c, c[1:])) and c[-1] > c[0]
    assert c[-1] == c[-2]                                                     # converged: no pair left to split
    keys = res["keys"].astype(np.int64)
    assert np.all(np.diff(keys) > 0)                                          # still sorted, no duplicate cell
    assert np.array_equal(H.keys_of(res["coords"], H.curve_bits((8, 8), R)).astype(np.int64), keys)
    dL = np.abs(np.diff(res["L"]))
    assert np.all(np.diff(keys)[dL > 0.5] == 1)                               # every remaining jump is between adjacent cells
    new = np.ones(len(keys), bool); new[np.isin(keys, H.level0(lat, R)[0].astype(np.int64))] = False
    x = (res["coords"][new, 0] + 0.5) / (8 << R)
    assert np.all(np.abs(x - 0.37) < 0.13)                                    # the added samples sit at the jump
    # a NaN length never triggers, a threshold above the jump adds nothing
    assert H.hilbert_map(_step_trace(0.37), lat, R, thr=5.0, passes=2, shift=0)["counts"] == [64, 64, 64]
    nanf = lambda s: (np.full(len(s), np.nan), np.full(len(s), np.nan))
    assert H.hilbert_map(nanf, lat, R, thr=0.5, passes=1, shift=0)["counts"] == [64, 64]


def test_shifted_pass_finds_what_the_curve_misses():
    """a jump along the line where the two halves of the curve meet is crossed by few successive sample
    pairs; on the shifted curve it is not special any more."""
    lat = _lat2(16, 16)
    R = 3
    f = _step_trace(0.5)                                                      # on the boundary of the top-level quadrants
    plain = H.hilbert_map(f, lat, R, thr=0.5, passes=8, shift=0)
    shifted = H.hilbert_map(f, lat, R, thr=0.5, passes=8, shift=5)
    def rows_resolved(res):                                                   # level-0 rows with a refined sample at the jump
        near = np.abs((res["coords"][:, 0] + 0.5) / (16 << R) - 0.5) < 1.0 / 64
        return len(np.unique(res["coords"][near, 1] >> R))
    assert rows_resolved(plain) <= 2 and rows_resolved(shifted) >= 12        # of 16 rows
    k = shifted["keys"].astype(np.int64)
    assert np.all(np.diff(k) > 0)
    assert np.all(H.inside(lat, R, shifted["coords"]))


def test_merge_positions_are_the_sorted_union():
    rng = np.random.default_rng(5)
    old = np.sort(rng.choice(10000, 300, replace=False)) * 2
    left = np.sort(rng.choice(299, 80, replace=False))
    new = (old[left] + old[left + 1]) // 2 + 0                                 # strictly between the neighbours
    new = np.where(new == old[left], new + 1, new)
    pos_old, pos_new = H.merge(left, len(old))
    out = np.empty(380, dtype=np.int64); out[pos_old] = old; out[pos_new] = new
    assert np.array_equal(out, np.sort(np.concatenate([old, new])))


def test_converter_max_rule_and_gap_fill():
    lat = _lat2(2, 2)
    R, r = 2, 1                                                               # fine 8 x 8, output 4 x 4
    bits = H.curve_bits((2, 2), R)
    cells = np.array([[0, 0], [1, 1], [6, 6], [7, 0]])
    Q = np.array([10.0, 1000.0, 100.0, np.nan])
    keys = H.keys_of(cells, bits)
    o = np.argsort(keys)
    out = H.convert(lat, R, r, keys[o], Q[o]).reshape(4, 4)                   # [c1, c0]
    assert out[0, 0] == 1000.0                                                # two samples in output cell (0,0): the max
    assert out[3, 3] == 100.0
    # an empty cell: log-linear along the curve between the neighbours of its key range, at the middle of the range
    c = (1, 2)
    k0 = H.hilbert_key([c[0] << 1, c[1] << 1], bits) & ~3
    kc = k0 + 2
    ks = sorted(int(k) for k, q in zip(keys, Q) if math.isfinite(q))
    qs = {int(k): q for k, q in zip(keys, Q)}
    p = max(k for k in ks if k < k0); q = min(k for k in ks if k >= k0 + 4)
    t = (kc - p) / (q - p)
    want = 10 ** (math.log10(qs[p]) + t * (math.log10(qs[q]) - math.log10(qs[p])))
    assert abs(out[c[1], c[0]] / want - 1) < 1e-12
    assert np.all(np.isfinite(out)) and out.min() >= 10.0 and out.max() <= 1000.0
    # full coverage at r = 0: the map is the samples themselves
    k0s, c0s = H.level0(lat, R)
    q0 = np.arange(4) + 2.0
    full = H.convert(lat, R, 0, k0s, q0)
    for kk, cc, qq in zip(k0s, c0s, q0):
        assert full[(cc[1] >> R) * 2 + (cc[0] >> R)] == qq

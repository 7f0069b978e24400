"""Pins of the oracle's FLEDGE (O6) and threshold / refinement (O7) against library routines and brute force
(SURVEY.md 8(c) P8, P9, P10).  CPU only."""
import math

import numpy as np
import pytest
import scipy.ndimage

import oracle
import qsl_inputs as qi


def _sobel_mag(V):
    return np.sqrt(sum(scipy.ndimage.sobel(V, axis=a) ** 2 for a in range(V.ndim)))


@pytest.mark.parametrize("shape", [(13, 17), (1, 9), (8, 1), (6, 7, 9), (5, 4, 1), (2, 2, 2)])
def test_P8_dense_fledge_equals_scipy_sobel(shape):
    """gradient magnitude of the Sobel operator; reading A10 = scipy.ndimage.sobel defaults."""
    rng = np.random.default_rng(10)
    V = rng.uniform(0.1, 3.0, size=shape)
    S = oracle.fledge_dense(V, V.ndim)
    ref = _sobel_mag(V)
    assert np.allclose(S, ref, rtol=1e-13, atol=1e-13)


def test_P8_fledge_closed_forms():
    """A linear ramp L = a*c0 + b*c1 has interior Sobel response (8a, 8b); a unit step has response 4 on both sides."""
    c1, c0 = np.meshgrid(np.arange(12.0), np.arange(10.0), indexing="ij")
    S = oracle.fledge_dense(0.5 * c0 - 0.25 * c1, 2)
    assert np.allclose(S[1:-1, 1:-1], math.hypot(8 * 0.5, 8 * 0.25), rtol=1e-14)
    V = np.zeros((8, 8)); V[:, 4:] = 1.0
    S = oracle.fledge_dense(V, 2)
    assert np.allclose(S[:, 3], 4.0) and np.allclose(S[:, 4], 4.0) and np.allclose(S[:, :3], 0) and np.allclose(S[:, 5:], 0)
    c2, c1, c0 = np.meshgrid(np.arange(6.0), np.arange(7.0), np.arange(8.0), indexing="ij")
    S = oracle.fledge_dense(1.0 * c0 + 2.0 * c1 - 0.5 * c2, 3)
    assert np.allclose(S[1:-1, 1:-1, 1:-1], 32 * math.sqrt(1 + 4 + 0.25), rtol=1e-14)


def test_fledge_nan_propagates():
    V = np.ones((6, 6)); V[2, 3] = np.nan
    S = oracle.fledge_dense(V, 2)
    assert np.all(np.isnan(S[1:4, 2:5])) and np.isfinite(S[0, 0]) and np.isfinite(S[5, 5])


def _virtual_dense(n0, levels_coords, levels_L, L0, level):
    """Brute force: the level-`level` virtual lattice, every cell carrying the L of its nearest existing ancestor."""
    V = np.asarray(L0, float)
    for l in range(1, level + 1):
        for ax in range(V.ndim):
            V = np.repeat(V, 2, axis=ax)
        c = levels_coords[l]
        idx = tuple(c[:, d] for d in range(c.shape[1] - 1, -1, -1))       # array axes are (c2, c1, c0)
        V = V.copy(); V[idx] = levels_L[l]
    return V


@pytest.mark.parametrize("ndim,n0", [(2, (12, 9)), (3, (6, 5, 4))])
def test_sparse_fledge_equals_dense_sobel_of_virtual_lattice(ndim, n0):
    rng = np.random.default_rng(11)
    shape0 = tuple(n0[::-1])
    L0 = rng.uniform(0.5, 2.0, size=shape0)
    coords = [None]; Ls = [None]
    parents = np.stack(np.unravel_index(rng.choice(np.prod(n0), size=np.prod(n0) // 3, replace=False), n0), 1)
    for l in range(1, 4):
        offs = np.array([[(ch >> d) & 1 for d in range(ndim)] for ch in range(1 << ndim)])
        ch = (2 * parents[:, None, :] + offs[None]).reshape(-1, ndim).astype(np.uint32)
        coords.append(ch); Ls.append(rng.uniform(0.5, 2.0, size=len(ch)))
        V = _virtual_dense(n0, coords, Ls, L0, l)
        ref = _sobel_mag(V)[tuple(ch[:, d] for d in range(ndim - 1, -1, -1))]
        S = oracle.fledge_sparse(ndim, n0, l, L0, coords, Ls)
        assert np.allclose(S, ref, rtol=1e-12, atol=1e-12)
        parents = ch[rng.random(len(ch)) < 0.4].astype(np.int64)
        if len(parents) == 0:
            break


def test_P9_select_is_nearest_rank_order_statistic():
    rng = np.random.default_rng(12)
    for n in (1, 2, 19, 20, 21, 1000, 4097):
        S = rng.exponential(size=n)
        S[rng.random(n) < 0.1] = np.nan
        if n > 5:
            S[3] = np.inf; S[4] = S[5]
        fin = np.sort(S[np.isfinite(S)])
        for p in (0.95, 0.5, 0.999, 1.0, 0.0):
            if len(fin) == 0:
                assert math.isnan(oracle.select(S, p)); continue
            rank = min(max(int(math.ceil(p * len(fin))), 1), len(fin))
            assert oracle.select(S, p) == fin[rank - 1]


def _brute_refine(ndim, level, coords, S, tau, lat):
    cc, cs = [], []
    for c, s in zip(coords, S):
        if not (s > tau):
            continue
        for ch in range(1 << ndim):
            c2 = [2 * int(c[d]) + ((ch >> d) & 1) for d in range(ndim)]
            w = [(c2[d] + 0.5) / (int(lat.n[d]) << (level + 1)) for d in range(ndim)]
            e = (lat.e0, lat.e1, lat.e2)
            cc.append(c2)
            cs.append([lat.origin[k] + sum(w[d] * e[d][k] for d in range(ndim)) for k in range(3)])
    return np.array(cc, dtype=np.uint32).reshape(-1, ndim), np.array(cs).reshape(-1, 3)


@pytest.mark.parametrize("ndim", [2, 3])
def test_P10_refine_brute_force(ndim):
    rng = np.random.default_rng(13)
    if ndim == 2:
        lat = qi.Lattice(2, (32, 32, 1), (-0.6, 0.0, 0.0), (1.2, 0, 0), (0, 0, 0.5))
    else:
        lat = qi.Lattice(3, (16, 16, 16), (0.0, 0.0, 0.0), (1.0, 0, 0), (0, 1.0, 0), (0, 0, 0.5))
    n = lat.count
    coords = np.stack(np.unravel_index(np.arange(n), lat.n[:ndim][::-1]), 1)[:, ::-1].astype(np.uint32)
    S = rng.exponential(size=n); S[::17] = np.nan
    tau = oracle.select(S, 0.9)
    cc, cs = oracle.refine(ndim, 0, coords, S, tau, lat)
    bc, bs = _brute_refine(ndim, 0, coords, S, tau, lat)
    assert np.array_equal(cc, bc)
    assert np.allclose(cs, bs, rtol=0, atol=1e-15)
    flagged = int(np.sum(S > tau))
    assert len(cc) == flagged << ndim and flagged == np.isfinite(S).sum() - math.ceil(0.9 * np.isfinite(S).sum())
    # children are the quarter-offset points of the parent pixel: their mean is the parent's seed
    par = qi.lattice_seeds(lat)[S > tau]
    assert np.allclose(cs.reshape(flagged, 1 << ndim, 3).mean(1), par, atol=1e-14)
    # level 1 -> 2: nesting (every child's parent exists and was flagged), equal S never flags (strict >)
    S1 = rng.exponential(size=len(cc)); S1[0] = tau
    cc2, cs2 = oracle.refine(ndim, 1, cc, S1, tau, lat)
    parents = {tuple(c) for c in cc[S1 > tau]}
    assert all(tuple(c >> 1) in parents for c in cc2) and not (S1[0] > tau)
    assert np.allclose(cs2, _brute_refine(ndim, 1, cc, S1, tau, lat)[1], atol=1e-15)

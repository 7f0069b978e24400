"""CPU oracle of the paper's own adaptive refinement (section 3.6): samples ordered
along a Hilbert curve, mid-point insertion where the field-line length jumps between successive samples, a pass on a
shifted curve, and the converter back to a rectilinear array.  TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline leg may import this; it shares no code with the CUDA path.  Plain numpy / Python loops.

Readings (A17), where PAPER.md is silent:
 H0  curve: the Hilbert curve of Skilling, "Programming the Hilbert curve" (2004), on the cube of 2^bits cells per axis
     that bounds the finest lattice; key = the transposed index with its bits interleaved, axis 0 most significant.
 H1  a sample sits at the centre of a cell of the finest lattice n_d 2^R ("fine cell"); the level-0 sample of the
     level-0 cell c0 is the fine cell c0 2^R + 2^(R-1); position = origin + sum_d (c_d + 0.5)/(n_d 2^R) e_d with one
     IEEE division and an fma chain per component (as O7).
 H2  pass: for successive samples i, i+1 in key order with both L finite, |L_{i+1} - L_i| > thr and
     key_{i+1} - key_i >= 2, a new sample at key (key_i + key_{i+1}) >> 1 ("halfway along the Hilbert curve"), unless
     that cell lies outside the lattice (the padding of the bounding cube).
 H3  shifted pass: keys of the cells displaced by +shift fine cells per axis on a cube one bit larger;
     same rule in that order; the new cell is the mid-point cell displaced back; then the original order again.
 H4  converter to the lattice n_d 2^r, r <= R: max of the finite Q of the samples inside an output cell;
     a cell without sample takes 10^(lerp of log10 Q) along the curve between the last sample before the cell's key range
     and the first after it, at the middle key of the range (one-sided at the ends of the curve; NaN without samples).
"""
from __future__ import annotations

import ctypes
import ctypes.util
import math

import numpy as np

_libm = ctypes.CDLL(ctypes.util.find_library("m") or "libm.so.6")
_libm.fma.restype = ctypes.c_double
_libm.fma.argtypes = [ctypes.c_double] * 3


def _fma(a, b, c):
    """IEEE fused multiply-add (C99 fma of libm)."""
    return _libm.fma(float(a), float(b), float(c))


# ------------------------------------------------------------------------------------------------------------ H0
def _axes_to_transpose(X, bits):
    """Skilling (2004), AxesToTranspose: in place on the list X of `len(X)` integer coordinates of `bits` bits."""
    n = len(X)
    M = 1 << (bits - 1)
    Q = M
    while Q > 1:                                   # inverse undo
        P = Q - 1
        for i in range(n):
            if X[i] & Q:
                X[0] ^= P                          # invert
            else:
                t = (X[0] ^ X[i]) & P              # exchange
                X[0] ^= t
                X[i] ^= t
        Q >>= 1
    for i in range(1, n):                          # Gray encode
        X[i] ^= X[i - 1]
    t = 0
    Q = M
    while Q > 1:
        if X[n - 1] & Q:
            t ^= Q - 1
        Q >>= 1
    for i in range(n):
        X[i] ^= t
    return X


def _transpose_to_axes(X, bits):
    """Skilling (2004), TransposeToAxes."""
    n = len(X)
    N = 2 << (bits - 1)
    t = X[n - 1] >> 1                              # Gray decode by H ^ (H/2)
    for i in range(n - 1, 0, -1):
        X[i] ^= X[i - 1]
    X[0] ^= t
    Q = 2
    while Q != N:                                  # undo excess work
        P = Q - 1
        for i in range(n - 1, -1, -1):
            if X[i] & Q:
                X[0] ^= P
            else:
                t = (X[0] ^ X[i]) & P
                X[0] ^= t
                X[i] ^= t
        Q <<= 1
    return X


def hilbert_key(c, bits):
    """Cell coordinates (length ndim) -> position along the curve, an integer in [0, 2^(ndim bits))."""
    X = _axes_to_transpose([int(v) for v in c], bits)
    key = 0
    for b in range(bits - 1, -1, -1):
        for d in range(len(X)):
            key = (key << 1) | ((X[d] >> b) & 1)
    return key


def hilbert_cell(key, ndim, bits):
    """Inverse of hilbert_key."""
    X = [0] * ndim
    for b in range(bits - 1, -1, -1):
        for d in range(ndim):
            X[d] |= ((key >> (b * ndim + (ndim - 1 - d))) & 1) << b
    return _transpose_to_axes(X, bits)


def keys_of(coords, bits, shift=0):
    coords = np.asarray(coords, dtype=np.int64)
    return np.array([hilbert_key(c + shift, bits) for c in coords], dtype=np.uint64)


def cells_of(keys, ndim, bits, shift=0):
    return np.array([hilbert_cell(int(k), ndim, bits) for k in keys], dtype=np.int64).reshape(-1, ndim) - shift


# ------------------------------------------------------------------------------------------------------------ H1
def curve_bits(n, R):
    """Bits per axis of the cube bounding the finest lattice n_d 2^R."""
    m = max(int(v) << R for v in n)
    return max(1, (m - 1).bit_length())


def positions(lat, R, coords):
    """Centres of the fine cells `coords` (m, ndim): origin + sum_d (c_d + 0.5)/(n_d 2^R) e_d, IEEE division + fma."""
    coords = np.asarray(coords, dtype=np.int64).reshape(-1, lat.ndim)
    es = [np.asarray(lat.e0, float), np.asarray(lat.e1, float), np.asarray(lat.e2, float)]
    out = np.empty((len(coords), 3))
    for m, c in enumerate(coords):
        w = [(float(c[d]) + 0.5) / float(int(lat.n[d]) << R) for d in range(lat.ndim)]
        for k in range(3):
            pos = _fma(w[0], es[0][k], float(lat.origin[k]))
            pos = _fma(w[1], es[1][k], pos)
            if lat.ndim == 3:
                pos = _fma(w[2], es[2][k], pos)
            out[m, k] = pos
    return out


def level0(lat, R):
    """(keys, coords) of the level-0 samples, sorted along the curve."""
    nd = lat.ndim
    n = [int(v) for v in lat.n[:nd]]
    grids = np.meshgrid(*[np.arange(v) for v in n], indexing="ij")
    c0 = np.stack([g.reshape(-1) for g in grids], 1)
    cf = c0 * (1 << R) + ((1 << R) >> 1)
    keys = keys_of(cf, curve_bits(n, R))
    o = np.argsort(keys, kind="stable")
    return keys[o], cf[o]


# ------------------------------------------------------------------------------------------------------------ H2, H3
def inside(lat, R, coords):
    coords = np.asarray(coords, dtype=np.int64).reshape(-1, lat.ndim)
    hi = np.array([int(v) << R for v in lat.n[:lat.ndim]])
    return np.all((coords >= 0) & (coords < hi), axis=1)


def refine_pass(lat, R, keys, L, thr, shift=0):
    """H2 (shift = 0) / H3 on samples sorted by `keys` (the keys of the cells displaced by `shift`, on curve_bits + 1 bits
    if shift != 0).  Returns (left, new_keys, new_coords): index of the left neighbour of every new sample, its key in
    the SAME (possibly shifted) curve, and its cell in un-shifted fine coordinates."""
    nd = lat.ndim
    bits = curve_bits(lat.n[:nd], R) + (1 if shift else 0)
    left, nk, nc = [], [], []
    for i in range(len(keys) - 1):
        a, b = L[i], L[i + 1]
        if not (math.isfinite(a) and math.isfinite(b)):
            continue
        if not abs(b - a) > thr:
            continue
        k0, k1 = int(keys[i]), int(keys[i + 1])
        if k1 - k0 < 2:
            continue
        km = (k0 + k1) >> 1
        c = np.array(hilbert_cell(km, nd, bits), dtype=np.int64) - shift
        if not inside(lat, R, c)[0]:
            continue
        left.append(i); nk.append(km); nc.append(c)
    return (np.array(left, dtype=np.int64), np.array(nk, dtype=np.uint64),
            np.array(nc, dtype=np.int64).reshape(-1, nd))


def merge(left, n_old):
    """Positions in the merged, still sorted, array: (pos_old[n_old], pos_new[len(left)])."""
    ins = np.zeros(n_old + 1, dtype=np.int64)
    if len(left):
        np.add.at(ins, left + 1, 1)
    before = np.cumsum(ins)[:n_old]                 # number of new samples before old sample i
    pos_old = np.arange(n_old) + before
    pos_new = left + 1 + np.arange(len(left))
    return pos_old, pos_new


# ------------------------------------------------------------------------------------------------------------ H4
def convert(lat, R, r, keys, Q):
    """H4: samples (sorted keys of the un-shifted curve, Q) -> dense map on the lattice n_d 2^r, flat index
    (c2 d1 + c1) d0 + c0."""
    nd = lat.ndim
    bits = curve_bits(lat.n[:nd], R)
    dims = [int(v) << r for v in lat.n[:nd]]
    span = 1 << (nd * (R - r))                      # keys per output cell
    out = np.full(int(np.prod(dims)), np.nan)
    have = np.zeros(len(out), dtype=bool)
    cells = cells_of(keys, nd, bits) >> (R - r)
    flat = np.zeros(len(keys), dtype=np.int64)
    for d in range(nd - 1, -1, -1):
        flat = flat * dims[d] + cells[:, d]
    for i, f in enumerate(flat):
        if math.isfinite(Q[i]) and (not have[f] or Q[i] > out[f]):
            out[f] = Q[i]; have[f] = True
    kint = np.array([int(k) for k in keys], dtype=object)
    usable = [i for i in range(len(keys)) if math.isfinite(Q[i]) and Q[i] > 0]
    uk = [int(keys[i]) for i in usable]
    import bisect
    it = np.ndindex(*dims[::-1])
    for idx in it:
        c = list(idx[::-1])
        f = 0
        for d in range(nd - 1, -1, -1):
            f = f * dims[d] + c[d]
        if have[f] or not usable:
            continue
        k0 = hilbert_key([v << (R - r) for v in c], bits) & ~(span - 1)
        k1 = k0 + span
        kc = k0 + span // 2
        p = bisect.bisect_left(uk, k0) - 1           # last usable sample before the range
        q = bisect.bisect_left(uk, k1)               # first usable sample after it
        if p >= 0 and q < len(uk):
            t = float(kc - uk[p]) / float(uk[q] - uk[p])      # both differences rounded to fp64 first, then one division
            la, lb = math.log10(Q[usable[p]]), math.log10(Q[usable[q]])
            out[f] = 10.0 ** (la + t * (lb - la))
        elif p >= 0:
            out[f] = Q[usable[p]]
        elif q < len(uk):
            out[f] = Q[usable[q]]
    del kint
    return out


# ------------------------------------------------------------------------------------------------------------ driver
def hilbert_map(trace_fn, lat, R, thr, passes, shift):
    """The loop of PAPER.md:194-204.  trace_fn(seeds) -> (L, Q).  Every pass = one refinement on the curve, then one on
    the shifted curve (if shift != 0).  Returns dict(keys, coords, L, Q, counts)."""
    nd = lat.ndim
    bits = curve_bits(lat.n[:nd], R)
    keys, coords = level0(lat, R)
    L, Q = trace_fn(positions(lat, R, coords))
    counts = [len(keys)]
    for _ in range(passes):
        for sh in ((0, shift) if shift else (0,)):
            if sh:
                ks = keys_of(coords, bits + 1, sh)
                o = np.argsort(ks, kind="stable")
                ks, keys, coords, L, Q = ks[o], keys[o], coords[o], L[o], Q[o]
            else:
                ks = keys
            left, nk, nc = refine_pass(lat, R, ks, L, thr, sh)
            if len(left):
                nL, nQ = trace_fn(positions(lat, R, nc))
                pos_old, pos_new = merge(left, len(keys))
                m = len(keys) + len(left)
                def mix(old, new, dtype, shape=()):
                    out = np.empty((m,) + shape, dtype=dtype)
                    out[pos_old] = old; out[pos_new] = new
                    return out
                coords = mix(coords, nc, np.int64, (nd,))
                L = mix(L, nL, np.float64); Q = mix(Q, nQ, np.float64)
                keys = mix(keys, keys_of(nc, bits), np.uint64)
            if sh:
                o = np.argsort(keys, kind="stable")
                keys, coords, L, Q = keys[o], coords[o], L[o], Q[o]
            counts.append(len(keys))
    return dict(keys=keys, coords=coords, L=L, Q=Q, counts=counts)

"""Thin ctypes binding over the C ABI of libqsl (include/qsl.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libqsl.so; torch is used for device memory and streams.
There is no CPU fallback: if the shared library is missing or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import functools
import math
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("QSL_LIB_PATH") or os.path.join(_HERE, "libqsl.so")   # override: A/B runs of two builds
PEAKS_LIB_PATH = os.path.join(_HERE, "libqsl_peaks.so")                         # bench utility (include/qsl_peaks.h)

QSL_F32, QSL_F64 = 0, 1
QSL_NORMALIZE_FIRST, QSL_INTERP_FIRST = 0, 1
QSL_RK4, QSL_EULER, QSL_CK45 = 0, 1, 2
QSL_TRACE_L, QSL_TRACE_LQ = 0, 1
QSL_ARITH_F64, QSL_ARITH_F32 = 0, 1
QSL_TRILINEAR, QSL_TRIQUADRATIC, QSL_TRICUBIC = 0, 2, 3
QSL_CARTESIAN, QSL_SPHERICAL = 0, 1
QSL_LAYOUT_CELL_TABLE, QSL_LAYOUT_NODES_ONLY, QSL_LAYOUT_CELL_TABLE_F32, QSL_LAYOUT_CELL_TABLES_BOTH = 0, 1, 2, 3
QSL_ST_SEED_OUTSIDE, QSL_ST_NULL_AT_SEED, QSL_ST_STALL_F, QSL_ST_STALL_B = 1, 2, 4, 8
QSL_ST_CAP_F, QSL_ST_CAP_B, QSL_ST_OPEN = 16, 32, 64
QSL_FLAG_NO_SORT, QSL_FLAG_NO_REFILL, QSL_FLAG_KERNEL_V1, QSL_FLAG_KERNEL_FRAME = 1, 2, 4, 8

_dp = C.POINTER(C.c_double)


class QslError(RuntimeError):
    pass


class _GridDesc(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("stretched", C.c_int),
                ("lo", C.c_double * 3), ("hi", C.c_double * 3), ("xs", _dp), ("ys", _dp), ("zs", _dp),
                ("sample_type", C.c_int), ("interp_mode", C.c_int), ("layout", C.c_int), ("interp_order", C.c_int), ("geometry", C.c_int)]


class _TraceParams(C.Structure):
    _fields_ = [("box_lo", C.c_double * 3), ("box_hi", C.c_double * 3), ("method", C.c_int),
                ("step_frac", C.c_double), ("mode", C.c_int), ("arith", C.c_int), ("max_length", C.c_double),
                ("max_steps", C.c_longlong), ("null_eps", C.c_double), ("flags", C.c_uint), ("tol", C.c_double)]


class _TraceOut(C.Structure):
    _fields_ = [("end_f", C.c_void_p), ("end_b", C.c_void_p), ("L", C.c_void_p), ("q_perp", C.c_void_p),
                ("q_bnd", C.c_void_p), ("face_f", C.c_void_p), ("face_b", C.c_void_p), ("status", C.c_void_p),
                ("nsteps_f", C.c_void_p), ("nsteps_b", C.c_void_p), ("dev_f", C.c_void_p), ("dev_b", C.c_void_p)]


class _Lattice(C.Structure):
    _fields_ = [("ndim", C.c_int), ("n", C.c_longlong * 3), ("origin", C.c_double * 3), ("e0", C.c_double * 3),
                ("e1", C.c_double * 3), ("e2", C.c_double * 3)]


class _Levels(C.Structure):
    _fields_ = [("lat", C.POINTER(_Lattice)), ("nlevels", C.c_int), ("L0", C.c_void_p),
                ("count", C.POINTER(C.c_longlong)), ("coords", C.POINTER(C.c_void_p)), ("L", C.POINTER(C.c_void_p)),
                ("child_base", C.POINTER(C.c_void_p))]


_lib = None


def lib():
    """Loads libqsl.so (building it in-tree if nvcc is available and it is missing).  Raises if it cannot."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            from . import build as _build
            _build.build()
        _lib = C.CDLL(LIB_PATH)
        _lib.qsl_strerror.restype = C.c_char_p
        _lib.qsl_field_bytes.restype = C.c_longlong
    return _lib


_peaks = None


def peaks_lib():
    """Loads libqsl_peaks.so: the roofline-denominator micro-kernels of bench.py (include/qsl_peaks.h), not part of libqsl."""
    global _peaks
    if _peaks is None:
        if not os.path.exists(PEAKS_LIB_PATH):
            from . import build as _build
            _build.build()
        _peaks = C.CDLL(PEAKS_LIB_PATH)
    return _peaks


def _check(rc: int, what: str):
    if rc != 0:
        L = lib()
        raise QslError("%s failed: %s (code %d, cudaError %d)" % (what, L.qsl_strerror(rc).decode(), rc,
                                                                   L.qsl_last_cuda_error()))


def _stream_ptr(stream=None):
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


def _on_stream(fn):
    """Runs a binding call with its `stream=` argument as torch's current stream, so that the tensors the call allocates
    (outputs, scratch) belong to that stream in the caching allocator and every torch-side operation next to the libqsl
    launch is ordered with it."""
    @functools.wraps(fn)
    def wrapped(*args, stream=None, **kw):
        if stream is None or stream == torch.cuda.current_stream():
            return fn(*args, stream=stream, **kw)
        with torch.cuda.stream(stream):
            return fn(*args, stream=stream, **kw)
    return wrapped


def _dev_f64(t, name):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise QslError("%s must be a contiguous CUDA float64 tensor" % name)
    return C.c_void_p(t.data_ptr())


def _require_cuda():
    if not torch.cuda.is_available():
        raise QslError("libqsl needs a CUDA device (sm_100a); there is no CPU fallback")


def make_lattice(lattice) -> _Lattice:
    """`lattice`: any object with ndim, n, origin, e0, e1, e2 (e.g. qsl_inputs.Lattice)."""
    n = [int(v) for v in lattice.n] + [1] * (3 - len(lattice.n))
    v3 = lambda v: (C.c_double * 3)(*[float(x) for x in v])
    return _Lattice(int(lattice.ndim), (C.c_longlong * 3)(*n), v3(lattice.origin), v3(lattice.e0), v3(lattice.e1),
                    v3(lattice.e2))


class Field:
    """Owner of a qsl_field handle (packed AoS samples in HBM)."""

    def __init__(self, handle, nx, ny, nz, sample_type, interp_mode, lo, hi):
        self._h = handle
        self.nx, self.ny, self.nz = nx, ny, nz
        self.sample_type, self.interp_mode = sample_type, interp_mode
        self.lo, self.hi = tuple(lo), tuple(hi)

    @property
    def handle(self):
        if not self._h:
            raise QslError("field already destroyed")
        return self._h

    @property
    def nbytes(self):
        return int(lib().qsl_field_bytes(self.handle))

    def export(self, stream=None) -> torch.Tensor:
        dt = torch.float32 if self.sample_type == QSL_F32 else torch.float64
        with torch.cuda.stream(stream if stream is not None else torch.cuda.current_stream()):
            out = torch.empty((self.nz, self.ny, self.nx, 4), dtype=dt, device="cuda")
            _check(lib().qsl_field_export(self.handle, C.c_void_p(out.data_ptr()), _stream_ptr(stream)), "qsl_field_export")
        return out

    def destroy(self):
        if self._h:
            lib().qsl_field_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


@_on_stream
def qsl_field_create(nx, ny, nz, bx, by, bz, *, lo=None, hi=None, xs=None, ys=None, zs=None,
                     sample_type=QSL_F64, interp_mode=QSL_NORMALIZE_FIRST, layout=QSL_LAYOUT_CELL_TABLE,
                     interp_order=QSL_TRILINEAR, geometry=QSL_CARTESIAN, stream=None) -> Field:
    """bx, by, bz: CUDA float64 tensors of nx*ny*nz values (x fastest).  Uniform grid: lo, hi.  Stretched: xs, ys, zs
    (host sequences of node coordinates)."""
    _require_cuda()
    stretched = xs is not None
    d = _GridDesc()
    d.nx, d.ny, d.nz, d.stretched = int(nx), int(ny), int(nz), int(stretched)
    keep = []
    if stretched:
        for name, arr, n in (("xs", xs, nx), ("ys", ys, ny), ("zs", zs, nz)):
            a = (C.c_double * int(n))(*[float(v) for v in arr])
            keep.append(a)
            setattr(d, name, C.cast(a, _dp))
        lo = (float(xs[0]), float(ys[0]), float(zs[0])); hi = (float(xs[-1]), float(ys[-1]), float(zs[-1]))
    d.lo = (C.c_double * 3)(*[float(v) for v in lo]); d.hi = (C.c_double * 3)(*[float(v) for v in hi])
    d.sample_type, d.interp_mode, d.layout = int(sample_type), int(interp_mode), int(layout)
    d.interp_order = int(interp_order)
    d.geometry = int(geometry)
    for t, name in ((bx, "bx"), (by, "by"), (bz, "bz")):
        if t.numel() != nx * ny * nz:
            raise QslError("%s has %d values, expected %d" % (name, t.numel(), nx * ny * nz))
    h = C.c_void_p()
    _check(lib().qsl_field_create(C.byref(h), C.byref(d), _dev_f64(bx, "bx"), _dev_f64(by, "by"), _dev_f64(bz, "bz"),
                                  _stream_ptr(stream)), "qsl_field_create")
    return Field(h, int(nx), int(ny), int(nz), int(sample_type), int(interp_mode), lo, hi)


_OUT_SPECS = {  # name -> (dtype, trailing dim)
    "end_f": (torch.float64, 3), "end_b": (torch.float64, 3), "L": (torch.float64, 0), "q_perp": (torch.float64, 0),
    "q_bnd": (torch.float64, 0), "face_f": (torch.uint8, 0), "face_b": (torch.uint8, 0), "status": (torch.int32, 0),
    "nsteps_f": (torch.int32, 0), "nsteps_b": (torch.int32, 0), "dev_f": (torch.float64, 6), "dev_b": (torch.float64, 6),
}
DEFAULT_OUTPUTS = ("end_f", "end_b", "L", "q_perp", "q_bnd", "face_f", "face_b", "status", "nsteps_f", "nsteps_b")


def make_trace_params(box_lo, box_hi, *, method=QSL_RK4, step_frac=0.25, mode=QSL_TRACE_LQ, arith=QSL_ARITH_F64,
                      max_length=math.inf, max_steps=1 << 30, null_eps=1e-12, flags=0, tol=1e-2) -> _TraceParams:
    return _TraceParams((C.c_double * 3)(*[float(v) for v in box_lo]), (C.c_double * 3)(*[float(v) for v in box_hi]),
                        int(method), float(step_frac), int(mode), int(arith), float(max_length), int(max_steps),
                        float(null_eps), int(flags), float(tol))


@_on_stream
def qsl_trace(field: Field, seeds: torch.Tensor, params: _TraceParams, *, outputs=DEFAULT_OUTPUTS, out=None,
              total_steps: torch.Tensor | None = None, stream=None) -> dict:
    """Traces `seeds` (CUDA float64 (n,3)).  Returns a dict of CUDA tensors for the requested `outputs`
    (pre-allocated tensors may be passed in `out`); `total_steps` (CUDA int64[1]) receives the RK-step count."""
    _require_cuda()
    n = int(seeds.shape[0]) if seeds.dim() == 2 else int(seeds.numel() // 3)
    res = {} if out is None else dict(out)
    o = _TraceOut()
    for name in outputs:
        dt, tr = _OUT_SPECS[name]
        if name not in res:
            res[name] = torch.empty((n, tr) if tr else (n,), dtype=dt, device="cuda")
        t = res[name]
        if not (t.is_cuda and t.is_contiguous() and t.dtype == dt and t.numel() == n * max(tr, 1)):
            raise QslError("output %s has the wrong dtype / size / device" % name)
        setattr(o, name, t.data_ptr())
    ts = C.c_void_p(total_steps.data_ptr()) if total_steps is not None else None
    _check(lib().qsl_trace(field.handle, C.byref(params), C.c_longlong(n), _dev_f64(seeds, "seeds") if n else None,
                           C.byref(o), ts, _stream_ptr(stream)), "qsl_trace")
    return res


@_on_stream
def qsl_fledge_dense(L: torch.Tensor, ndim: int, *, out=None, stream=None) -> torch.Tensor:
    """L: CUDA float64 map of shape (d1, d0) or (d2, d1, d0) (axis 0 fastest).  Returns S of the same shape."""
    _require_cuda()
    if L.dim() != ndim:
        raise QslError("L must have %d dimensions" % ndim)
    dims = list(L.shape[::-1]) + [1] * (3 - ndim)
    S = torch.empty_like(L) if out is None else out
    _check(lib().qsl_fledge_dense(C.c_int(ndim), (C.c_longlong * 3)(*dims), _dev_f64(L, "L"), _dev_f64(S, "S"),
                                  _stream_ptr(stream)), "qsl_fledge_dense")
    return S


@_on_stream
def qsl_fledge_sparse(lattice, level: int, L0: torch.Tensor, coords: list, Ls: list, child_base: list, *, stream=None):
    """Sparse FLEDGE at `level` >= 1.  coords[l], Ls[l] (l = 1..level) and child_base[l] (l = 0..level-1) are CUDA
    tensors as produced by qsl_refine / qsl_trace; index 0 of coords / Ls is ignored."""
    _require_cuda()
    nl = level + 1
    lat = make_lattice(lattice)
    count = (C.c_longlong * nl)(*([0] + [int(Ls[l].numel()) for l in range(1, nl)]))
    cp = (C.c_void_p * nl)(*([None] + [coords[l].data_ptr() for l in range(1, nl)]))
    lp = (C.c_void_p * nl)(*([None] + [Ls[l].data_ptr() for l in range(1, nl)]))
    bp = (C.c_void_p * nl)(*([child_base[l].data_ptr() for l in range(0, level)] + [None]))
    for l in range(1, nl):
        if coords[l].dtype != torch.int32 or Ls[l].dtype != torch.float64 or not coords[l].is_cuda:
            raise QslError("coords must be CUDA int32 (uint32 bit patterns), L CUDA float64")
    for l in range(0, level):
        if child_base[l].dtype != torch.int64 or not child_base[l].is_cuda:
            raise QslError("child_base must be CUDA int64")
    lv = _Levels(C.pointer(lat), nl, L0.data_ptr(), count, cp, lp, bp)
    S = torch.empty(int(Ls[level].numel()), dtype=torch.float64, device="cuda")
    _check(lib().qsl_fledge_sparse(C.byref(lv), C.c_int(level), _dev_f64(S, "S"), _stream_ptr(stream)), "qsl_fledge_sparse")
    return S


@_on_stream
def qsl_select(S: torch.Tensor, p: float, *, out=None, stream=None) -> torch.Tensor:
    """Nearest-rank order statistic of the finite values of S; returns a CUDA float64[1] tensor (no host sync)."""
    _require_cuda()
    tau = torch.empty(1, dtype=torch.float64, device="cuda") if out is None else out
    _check(lib().qsl_select(C.c_longlong(S.numel()), _dev_f64(S.reshape(-1), "S"), C.c_double(p), _dev_f64(tau, "tau"),
                            _stream_ptr(stream)), "qsl_select")
    return tau


@_on_stream
def qsl_refine(lattice, level: int, coords, S: torch.Tensor, tau: torch.Tensor, *, capacity=None, stream=None):
    """Refines the cells with S > tau.  coords: CUDA int32 (n, ndim) or None for the dense level-0 lattice.
    Returns (child_coords int32 (m, ndim), child_seeds float64 (m, 3), child_base int64 (n,))."""
    _require_cuda()
    lat = make_lattice(lattice)
    ndim = int(lattice.ndim)
    n = int(S.numel())
    cap = int(capacity) if capacity is not None else n << ndim
    cc = torch.empty((cap, ndim), dtype=torch.int32, device="cuda")
    cs = torch.empty((cap, 3), dtype=torch.float64, device="cuda")
    cb = torch.empty(n, dtype=torch.int64, device="cuda")
    m = C.c_longlong(0)
    cptr = None
    if coords is not None:
        if coords.dtype != torch.int32 or not coords.is_cuda or coords.numel() != n * ndim:
            raise QslError("coords must be CUDA int32 of n*ndim values")
        cptr = C.c_void_p(coords.data_ptr())
    _check(lib().qsl_refine(C.c_int(ndim), C.c_int(level), C.c_longlong(n), cptr, _dev_f64(S.reshape(-1), "S"),
                            _dev_f64(tau, "tau"), C.byref(lat), C.c_longlong(cap), C.c_void_p(cc.data_ptr()),
                            C.c_void_p(cs.data_ptr()), C.c_void_p(cb.data_ptr()), C.byref(m), _stream_ptr(stream)),
           "qsl_refine")
    return cc[: m.value], cs[: m.value], cb


QSL_REFINE_NOALLOC_MAX_CELLS = 67108864      # include/qsl.h


def qsl_refine_noalloc(lattice, level: int, coords, S: torch.Tensor, tau: torch.Tensor, child_coords: torch.Tensor,
                       child_seeds: torch.Tensor, child_base, n_children: torch.Tensor, *, stream=None) -> None:
    """qsl_refine without any allocation and without a host synchronisation (include/qsl.h: qsl_refine_noalloc): the
    caller passes every buffer - child_coords CUDA int32 (capacity, ndim), child_seeds CUDA float64 (capacity, 3),
    child_base CUDA int64 (n,) or None, n_children CUDA int64 (1,), written on the stream.  n is limited to
    QSL_REFINE_NOALLOC_MAX_CELLS (QslError beyond it); calls that overlap on the GPU race on the library's fixed scratch."""
    _require_cuda()
    lat = make_lattice(lattice)
    ndim = int(lattice.ndim)
    n = int(S.numel())
    cap = int(child_coords.shape[0]) if child_coords is not None else 0
    ok = (child_coords is None or (child_coords.is_cuda and child_coords.dtype == torch.int32 and child_coords.is_contiguous()
                                   and child_coords.numel() == cap * ndim))
    ok = ok and (child_seeds is None or (child_seeds.is_cuda and child_seeds.dtype == torch.float64
                                         and child_seeds.is_contiguous() and child_seeds.numel() == cap * 3))
    ok = ok and (child_base is None or (child_base.is_cuda and child_base.dtype == torch.int64 and child_base.numel() == n))
    ok = ok and n_children.is_cuda and n_children.dtype == torch.int64 and n_children.numel() == 1
    if not ok:
        raise QslError("qsl_refine_noalloc: outputs must be contiguous CUDA tensors of the documented types and sizes")
    cptr = None
    if coords is not None:
        if coords.dtype != torch.int32 or not coords.is_cuda or coords.numel() != n * ndim:
            raise QslError("coords must be CUDA int32 of n*ndim values")
        cptr = C.c_void_p(coords.data_ptr())
    _check(lib().qsl_refine_noalloc(C.c_int(ndim), C.c_int(level), C.c_longlong(n), cptr, _dev_f64(S.reshape(-1), "S"),
                                    _dev_f64(tau, "tau"), C.byref(lat), C.c_longlong(cap), _p(child_coords), _p(child_seeds),
                                    _p(child_base), C.c_void_p(n_children.data_ptr()), _stream_ptr(stream)),
           "qsl_refine_noalloc")


# ---- the paper's Hilbert-curve refinement (include/qsl.h) --------------------------------------------
def _p(t):
    return C.c_void_p(t.data_ptr()) if t is not None and t.numel() else None


def qsl_hilbert_bits(lattice, R: int) -> int:
    b = lib().qsl_hilbert_bits(C.byref(make_lattice(lattice)), C.c_int(R))
    _check(min(b, 0), "qsl_hilbert_bits")
    return int(b)


@_on_stream
def qsl_hilbert_level0(lattice, R: int, *, stream=None):
    """(coords int32 (n, ndim), seeds float64 (n, 3)) of the level-0 samples in dense order."""
    _require_cuda()
    nd = int(lattice.ndim)
    n = 1
    for v in list(lattice.n)[:nd]:
        n *= int(v)
    coords = torch.empty((n, nd), dtype=torch.int32, device="cuda")
    seeds = torch.empty((n, 3), dtype=torch.float64, device="cuda")
    _check(lib().qsl_hilbert_level0(C.byref(make_lattice(lattice)), C.c_int(R), _p(coords), _p(seeds), _stream_ptr(stream)),
           "qsl_hilbert_level0")
    return coords, seeds


@_on_stream
def qsl_hilbert_keys(coords: torch.Tensor, bits: int, shift: int = 0, *, stream=None) -> torch.Tensor:
    """coords: CUDA int32 (n, ndim).  Returns the keys as CUDA int64 (they are below 2^63)."""
    _require_cuda()
    n, nd = int(coords.shape[0]), int(coords.shape[1])
    if coords.dtype != torch.int32 or not coords.is_cuda or not coords.is_contiguous():
        raise QslError("coords must be a contiguous CUDA int32 (n, ndim) tensor")
    keys = torch.empty(n, dtype=torch.int64, device="cuda")
    _check(lib().qsl_hilbert_keys(C.c_int(nd), C.c_int(bits), C.c_int(shift), C.c_longlong(n), _p(coords), _p(keys),
                                  _stream_ptr(stream)), "qsl_hilbert_keys")
    return keys


@_on_stream
def qsl_hilbert_cells(keys: torch.Tensor, ndim: int, bits: int, shift: int = 0, *, stream=None) -> torch.Tensor:
    _require_cuda()
    n = int(keys.numel())
    if keys.dtype != torch.int64 or not keys.is_cuda or not keys.is_contiguous():
        raise QslError("keys must be a contiguous CUDA int64 tensor")
    coords = torch.empty((n, ndim), dtype=torch.int32, device="cuda")
    _check(lib().qsl_hilbert_cells(C.c_int(ndim), C.c_int(bits), C.c_int(shift), C.c_longlong(n), _p(keys), _p(coords),
                                   _stream_ptr(stream)), "qsl_hilbert_cells")
    return coords


@_on_stream
def qsl_sort_keys64(keys: torch.Tensor, key_bits: int = 64, *, stream=None) -> torch.Tensor:
    """Sorts `keys` (CUDA int64, non-negative) in place; returns the permutation (CUDA int32)."""
    _require_cuda()
    n = int(keys.numel())
    if keys.dtype != torch.int64 or not keys.is_cuda or not keys.is_contiguous():
        raise QslError("keys must be a contiguous CUDA int64 tensor")
    perm = torch.empty(n, dtype=torch.int32, device="cuda")
    _check(lib().qsl_sort_keys64(C.c_longlong(n), _p(keys), _p(perm), C.c_int(key_bits), _stream_ptr(stream)), "qsl_sort_keys64")
    return perm


@_on_stream
def qsl_gather(perm: torch.Tensor, src: torch.Tensor, *, stream=None) -> torch.Tensor:
    """dst[i] = src[perm[i]] along the first axis (rows of a multiple of 4 bytes)."""
    _require_cuda()
    n = int(perm.numel())
    if not src.is_cuda or not src.is_contiguous() or perm.dtype != torch.int32:
        raise QslError("src must be a contiguous CUDA tensor, perm CUDA int32")
    row = src.element_size() * (src.numel() // max(int(src.shape[0]), 1))
    dst = torch.empty((n,) + tuple(src.shape[1:]), dtype=src.dtype, device="cuda")
    _check(lib().qsl_gather(C.c_longlong(n), _p(perm), C.c_int(row), _p(src), _p(dst), _stream_ptr(stream)), "qsl_gather")
    return dst


@_on_stream
def qsl_hilbert_refine(lattice, R: int, shift: int, keys: torch.Tensor, L: torch.Tensor, thr: float, *, capacity=None,
                       stream=None):
    """One refinement pass.  Returns (left int64 (m,), new_coords int32 (m, ndim), new_seeds float64 (m, 3))."""
    _require_cuda()
    n, nd = int(keys.numel()), int(lattice.ndim)
    cap = int(capacity) if capacity is not None else max(n - 1, 0)
    left = torch.empty(cap, dtype=torch.int64, device="cuda")
    nc = torch.empty((cap, nd), dtype=torch.int32, device="cuda")
    ns = torch.empty((cap, 3), dtype=torch.float64, device="cuda")
    m = C.c_longlong(0)
    _check(lib().qsl_hilbert_refine(C.byref(make_lattice(lattice)), C.c_int(R), C.c_int(shift), C.c_longlong(n), _p(keys),
                                    _dev_f64(L, "L") if n else None, C.c_double(thr), C.c_longlong(cap), _p(left), _p(nc), _p(ns),
                                    C.byref(m), _stream_ptr(stream)), "qsl_hilbert_refine")
    return left[: m.value], nc[: m.value], ns[: m.value]


@_on_stream
def qsl_hilbert_merge(left: torch.Tensor, old: torch.Tensor, new: torch.Tensor, *, stream=None) -> torch.Tensor:
    _require_cuda()
    n_old, n_new = int(old.shape[0]), int(new.shape[0])
    if old.dtype != new.dtype or old.shape[1:] != new.shape[1:] or not old.is_contiguous() or not new.is_contiguous():
        raise QslError("old and new payloads must be contiguous tensors of the same dtype and row shape")
    row = old.element_size()
    for v in old.shape[1:]:
        row *= int(v)
    out = torch.empty((n_old + n_new,) + tuple(old.shape[1:]), dtype=old.dtype, device="cuda")
    _check(lib().qsl_hilbert_merge(C.c_longlong(n_old), C.c_longlong(n_new), _p(left), C.c_int(row), _p(old), _p(new), _p(out),
                                   _stream_ptr(stream)), "qsl_hilbert_merge")
    return out


@_on_stream
def qsl_hilbert_convert(lattice, R: int, r: int, keys: torch.Tensor, Q: torch.Tensor, *, stream=None) -> torch.Tensor:
    """Dense Q map on the lattice n_d 2^r, shape (d1, d0) or (d2, d1, d0)."""
    _require_cuda()
    nd = int(lattice.ndim)
    dims = [int(v) << r for v in list(lattice.n)[:nd]]
    out = torch.empty(tuple(dims[::-1]), dtype=torch.float64, device="cuda")
    _check(lib().qsl_hilbert_convert(C.byref(make_lattice(lattice)), C.c_int(R), C.c_int(r), C.c_longlong(keys.numel()), _p(keys),
                                     _p(Q), _p(out), _stream_ptr(stream)), "qsl_hilbert_convert")
    return out


# ---- measurement hooks (bench.py) ----------------------------------------------------------------------------------
def qsl_profile_enable(on: bool = True):
    _require_cuda()
    _check(lib().qsl_profile_enable(C.c_int(1 if on else 0)), "qsl_profile_enable")


def qsl_profile_trace_kernel_ms():
    """(ms, launches): device time and number of the trace-kernel launches since the previous read, each a 2-tuple
    indexed by trace mode (QSL_TRACE_L, QSL_TRACE_LQ)."""
    ms = (C.c_double * 2)()
    n = (C.c_longlong * 2)()
    _check(lib().qsl_profile_trace_kernel_ms(ms, n), "qsl_profile_trace_kernel_ms")
    return (ms[0], ms[1]), (int(n[0]), int(n[1]))


def qsl_peak_fma(fp64: bool, reps: int = 5, stream=None) -> float:
    """Measured FMA issue rate (FMA/s) of the plain FP pipe: DFMA if fp64 else FFMA (libqsl_peaks.so, bench utility)."""
    _require_cuda()
    v = C.c_double(0.0)
    rc = peaks_lib().qsl_peak_fma(C.c_int(1 if fp64 else 0), C.c_int(reps), C.byref(v), _stream_ptr(stream))
    if rc != 0:
        raise QslError("qsl_peak_fma failed (code %d)" % rc)
    return v.value


def qsl_peak_gather(bytes_per_sample: int, footprint_bytes: int, reps: int = 5, stream=None) -> float:
    """Measured rate (samples/s) of divergent 16 B / 32 B gathers over a footprint of the given size (libqsl_peaks.so)."""
    _require_cuda()
    v = C.c_double(0.0)
    rc = peaks_lib().qsl_peak_gather(C.c_int(bytes_per_sample), C.c_longlong(footprint_bytes), C.c_int(reps), C.byref(v),
                                     _stream_ptr(stream))
    if rc != 0:
        raise QslError("qsl_peak_gather failed (code %d)" % rc)
    return v.value

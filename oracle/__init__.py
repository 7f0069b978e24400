"""ctypes face of the CPU oracle (oracle/qsl_oracle.c).  TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  It imports nothing from paper_1609_00724_b200 and shares no code with it.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libqsl_oracle.so")
_SRC = [os.path.join(_HERE, "qsl_oracle.c"), os.path.join(_HERE, "qsl_oracle.h")]

F32, F64 = 0, 1
NORMALIZE_FIRST, INTERP_FIRST = 0, 1
RK4, EULER, CK45 = 0, 1, 2
TRILINEAR, TRIQUADRATIC, TRICUBIC = 1, 2, 3
CARTESIAN, SPHERICAL = 0, 1
TRACE_L, TRACE_LQ = 0, 1
ST_SEED_OUTSIDE, ST_NULL_AT_SEED, ST_STALL_F, ST_STALL_B, ST_CAP_F, ST_CAP_B, ST_OPEN = 1, 2, 4, 8, 16, 32, 64


_SO_SAN = os.path.join(_HERE, "libqsl_oracle_san.so")


def build(force: bool = False, sanitize: bool = False) -> str:
    """Compile the oracle with gcc (-O2 -ffp-contract=off: arithmetic exactly as written).
    sanitize=True builds a second library with -fsanitize=address,undefined: it is loaded when the
    environment variable QSL_ORACLE_SANITIZE=1 is set, in a process started with LD_PRELOAD=<sanitizer_runtime()>."""
    so = _SO_SAN if sanitize else _SO
    if not force and os.path.exists(so) and all(os.path.getmtime(so) >= os.path.getmtime(s) for s in _SRC):
        return so
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-std=c11", "-Wall", "-shared", "-fPIC"]
    if sanitize:
        cmd += ["-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]
    subprocess.run(cmd + [_SRC[0], "-o", so, "-lm"], check=True)
    return so


def sanitizer_runtime() -> str:
    """Path of gcc's libasan.so, to be LD_PRELOADed by a process that loads the sanitized oracle."""
    return subprocess.run(["gcc", "-print-file-name=libasan.so"], check=True, capture_output=True, text=True).stdout.strip()


_dp = C.POINTER(C.c_double)


class _Field(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("stretched", C.c_int),
                ("lo", C.c_double * 3), ("hi", C.c_double * 3),
                ("xs", _dp), ("ys", _dp), ("zs", _dp), ("interp_mode", C.c_int), ("packed", _dp), ("order", C.c_int), ("geometry", C.c_int)]


class _Params(C.Structure):
    _fields_ = [("box_lo", C.c_double * 3), ("box_hi", C.c_double * 3), ("method", C.c_int),
                ("step_frac", C.c_double), ("mode", C.c_int), ("max_length", C.c_double),
                ("max_steps", C.c_longlong), ("null_eps", C.c_double), ("basis_angle", C.c_double), ("tol", C.c_double)]


class _Out(C.Structure):
    _fields_ = [("end_f", _dp), ("end_b", _dp), ("L", _dp), ("q_perp", _dp), ("q_bnd", _dp),
                ("face_f", C.POINTER(C.c_uint8)), ("face_b", C.POINTER(C.c_uint8)),
                ("status", C.POINTER(C.c_uint32)), ("nsteps_f", C.POINTER(C.c_uint32)),
                ("nsteps_b", C.POINTER(C.c_uint32)), ("dev_f", _dp), ("dev_b", _dp)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        san = os.environ.get("QSL_ORACLE_SANITIZE") == "1"
        _lib = C.CDLL(build(sanitize=san))
        _lib.orc_select.restype = C.c_double
        _lib.orc_refine.restype = C.c_longlong
    return _lib


def _ptr(a, ty=C.c_double):
    return a.ctypes.data_as(C.POINTER(ty))


class Field:
    """O0: packed field the oracle traces through.  `B` = (bx, by, bz) fp64 cubes of shape (nz, ny, nx)."""

    def __init__(self, grid, B, sample_type=F64, interp_mode=NORMALIZE_FIRST, order=TRILINEAR, geometry=CARTESIAN):
        self.grid = grid
        bx, by, bz = (np.ascontiguousarray(a, dtype=np.float64).reshape(-1) for a in B)
        n = grid.nx * grid.ny * grid.nz
        assert bx.size == n
        self.packed = np.empty(n * 4, dtype=np.float64)
        lib().orc_field_pack(C.c_longlong(n), _ptr(bx), _ptr(by), _ptr(bz), C.c_int(sample_type),
                             C.c_int(interp_mode), _ptr(self.packed))
        self._xs = np.ascontiguousarray(grid.xs, dtype=np.float64)
        self._ys = np.ascontiguousarray(grid.ys, dtype=np.float64)
        self._zs = np.ascontiguousarray(grid.zs, dtype=np.float64)
        self.c = _Field(grid.nx, grid.ny, grid.nz, int(bool(grid.stretched)),
                        (C.c_double * 3)(*grid.lo), (C.c_double * 3)(*grid.hi),
                        _ptr(self._xs), _ptr(self._ys), _ptr(self._zs), interp_mode, _ptr(self.packed), int(order), int(geometry))
        self.order = int(order)
        self.geometry = int(geometry)
        self.sample_type = sample_type
        self.interp_mode = interp_mode

    def evaluate(self, x):
        x = np.ascontiguousarray(x, dtype=np.float64)
        b = np.empty(3); J = np.empty(9); m = C.c_double(); hc = np.empty(3)
        lib().orc_evaluate(C.byref(self.c), _ptr(x), _ptr(b), _ptr(J), C.byref(m), _ptr(hc))
        return b, J.reshape(3, 3), m.value, hc


def ck_step(field: Field, y, h, *, with_dev=True, s=1.0):
    """One Cash-Karp 5(4) step of the 10-component state y.  Returns (y5, y5 - y4 of the position)."""
    y = np.ascontiguousarray(y, dtype=np.float64)
    yn = np.empty(10); err = np.empty(3)
    lib().orc_ck_step(C.byref(field.c), C.c_int(1 if with_dev else 0), C.c_double(s), _ptr(y), C.c_double(h), _ptr(yn), _ptr(err))
    return yn, err


def trace(field: Field, seeds, box_lo, box_hi, *, method=RK4, step_frac=0.25, mode=TRACE_LQ,
          max_length=math.inf, max_steps=1 << 40, null_eps=1e-12, basis_angle=0.0, nthreads=0, want_dev=False,
          tol=1e-2):
    """O2-O5 for every seed.  Returns a dict of numpy arrays plus total_steps."""
    seeds = np.ascontiguousarray(seeds, dtype=np.float64).reshape(-1, 3)
    n = len(seeds)
    P = _Params((C.c_double * 3)(*box_lo), (C.c_double * 3)(*box_hi), method, step_frac, mode, max_length,
                int(max_steps), null_eps, basis_angle, tol)
    o = dict(end_f=np.empty((n, 3)), end_b=np.empty((n, 3)), L=np.empty(n), q_perp=np.empty(n), q_bnd=np.empty(n),
             face_f=np.empty(n, np.uint8), face_b=np.empty(n, np.uint8), status=np.empty(n, np.uint32),
             nsteps_f=np.empty(n, np.uint32), nsteps_b=np.empty(n, np.uint32))
    if want_dev:
        o["dev_f"] = np.empty((n, 6)); o["dev_b"] = np.empty((n, 6))
    out = _Out(_ptr(o["end_f"]), _ptr(o["end_b"]), _ptr(o["L"]), _ptr(o["q_perp"]), _ptr(o["q_bnd"]),
               _ptr(o["face_f"], C.c_uint8), _ptr(o["face_b"], C.c_uint8), _ptr(o["status"], C.c_uint32),
               _ptr(o["nsteps_f"], C.c_uint32), _ptr(o["nsteps_b"], C.c_uint32),
               _ptr(o["dev_f"]) if want_dev else None, _ptr(o["dev_b"]) if want_dev else None)
    tot = C.c_ulonglong(0)
    lib().orc_trace(C.byref(field.c), C.byref(P), C.c_longlong(n), _ptr(seeds), C.byref(out), C.byref(tot),
                    C.c_int(nthreads))
    o["total_steps"] = tot.value
    return o


def fledge_dense(L, ndim):
    """O6 on a dense map.  L has shape (d1, d0) for 2-D or (d2, d1, d0) for 3-D (axis 0 fastest)."""
    L = np.ascontiguousarray(L, dtype=np.float64)
    assert L.ndim == ndim
    dims = list(L.shape[::-1]) + [1] * (3 - ndim)
    S = np.empty_like(L)
    lib().orc_fledge_dense(C.c_int(ndim), (C.c_longlong * 3)(*dims), _ptr(L), _ptr(S))
    return S


def fledge_sparse(ndim, n0, level, L0, coords, Ls):
    """O6 on sparse level `level` >= 1.  coords[l] (count_l, ndim) uint32 and Ls[l] (count_l,) for l = 1..level
    (index 0 of both lists is ignored); L0 is the dense level-0 map (flat or shaped)."""
    L0 = np.ascontiguousarray(L0, dtype=np.float64).reshape(-1)
    nl = level + 1
    coords = [None] + [np.ascontiguousarray(coords[l], dtype=np.uint32).reshape(-1, ndim) for l in range(1, nl)]
    Ls = [None] + [np.ascontiguousarray(Ls[l], dtype=np.float64).reshape(-1) for l in range(1, nl)]
    count = (C.c_longlong * nl)(*([0] + [len(Ls[l]) for l in range(1, nl)]))
    cp = (C.POINTER(C.c_uint32) * nl)(*([None] + [_ptr(coords[l], C.c_uint32) for l in range(1, nl)]))
    lp = (_dp * nl)(*([None] + [_ptr(Ls[l]) for l in range(1, nl)]))
    n0v = list(n0) + [1] * (3 - len(n0))
    S = np.empty(len(Ls[level]), dtype=np.float64)
    lib().orc_fledge_sparse(C.c_int(ndim), (C.c_longlong * 3)(*n0v), C.c_int(level), _ptr(L0), count, cp, lp, _ptr(S))
    return S


def select(S, p):
    """O7 threshold: nearest-rank order statistic of the finite values."""
    S = np.ascontiguousarray(S, dtype=np.float64).reshape(-1)
    return float(lib().orc_select(C.c_longlong(S.size), _ptr(S), C.c_double(p)))


def refine(ndim, level, coords, S, tau, lattice):
    """O7 refinement of the cells `coords` (n, ndim) at `level`; returns (child_coords, child_seeds)."""
    coords = np.ascontiguousarray(coords, dtype=np.uint32).reshape(-1, ndim)
    S = np.ascontiguousarray(S, dtype=np.float64).reshape(-1)
    n = len(S)
    cc = np.empty((n << ndim, ndim), dtype=np.uint32)
    cs = np.empty((n << ndim, 3), dtype=np.float64)
    v3 = lambda v: (C.c_double * 3)(*v)
    n0 = [int(v) for v in lattice.n]
    m = lib().orc_refine(C.c_int(ndim), C.c_int(level), C.c_longlong(n), _ptr(coords, C.c_uint32), _ptr(S),
                         C.c_double(tau), (C.c_longlong * 3)(*n0), v3(lattice.origin), v3(lattice.e0),
                         v3(lattice.e1), v3(lattice.e2), _ptr(cc, C.c_uint32), _ptr(cs))
    return cc[:m].copy(), cs[:m].copy()

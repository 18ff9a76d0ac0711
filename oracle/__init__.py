"""ctypes front end of the CPU oracle -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference legs may import this package.  It never imports the CUDA package and
the CUDA package never imports it.  All arithmetic lives in
monc_adv_oracle.cpp (fp64, plain loops); this file only
marshals numpy arrays.

Arrays are C-contiguous float64 of shape [nx+2h, ny+2h, nz] (z fastest).
"""
import ctypes as C
import os

import numpy as np

from .build import build as _build

_LIB = None


def lib():
    global _LIB
    if _LIB is None:
        _LIB = C.CDLL(_build())
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int)
        _LIB.oracle_coefficients.argtypes = [C.c_int] + [dp] * 8
        _LIB.oracle_coefficients.restype = None
        _LIB.oracle_momentum.argtypes = ([C.c_int] * 4 + [C.c_double] * 2 + [dp] * 4 + [dp] * 3
                                         + [dp] * 3 + [C.c_int, C.c_int])
        _LIB.oracle_momentum.restype = None
        _LIB.oracle_scalar.argtypes = ([C.c_int] * 4 + [C.c_double] * 2 + [dp] * 2 + [dp] * 4
                                       + [dp] + [C.c_int, C.c_int])
        _LIB.oracle_scalar.restype = None
        _LIB.oracle_points.argtypes = ([C.c_int] * 5 + [C.c_double] * 2 + [dp] * 4 + [dp] * 4
                                       + [C.c_int, C.c_long, ip, ip, ip, dp])
        _LIB.oracle_points.restype = None
        _LIB.oracle_max_threads.restype = C.c_int
    return _LIB


def _p(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _chk(a, shape=None):
    assert isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous, \
        "oracle takes C-contiguous float64 arrays"
    if shape is not None:
        assert a.shape == tuple(shape), (a.shape, shape)
    return a


def max_threads() -> int:
    return int(lib().oracle_max_threads())


def coefficients(dz, dzn, rho, rhon):
    """tzc1, tzc2, tzd1, tzd2 (SURVEY.md 8(c).2 'Coefficients'), index K-1."""
    nz = len(dz)
    ins = [np.ascontiguousarray(a, dtype=np.float64) for a in (dz, dzn, rho, rhon)]
    outs = [np.zeros(nz) for _ in range(4)]
    lib().oracle_coefficients(nz, *[_p(a) for a in ins], *[_p(a) for a in outs])
    return tuple(outs)


class Problem:
    """Grid sizes + constants of one advection problem (what monc_adv_create takes)."""

    def __init__(self, nx, ny, nz, halo, dx, dy, dz, dzn, rho, rhon):
        self.nx, self.ny, self.nz, self.h = int(nx), int(ny), int(nz), int(halo)
        self.dx, self.dy = float(dx), float(dy)
        self.tzc1, self.tzc2, self.tzd1, self.tzd2 = coefficients(dz, dzn, rho, rhon)
        self.shape = (self.nx + 2 * self.h, self.ny + 2 * self.h, self.nz)

    def momentum(self, u, v, w, skew=False, nthreads=1, out=None):
        """su, sv, sw; output halos are left as allocated (zeros)."""
        for a in (u, v, w):
            _chk(a, self.shape)
        su, sv, sw = out if out is not None else (np.zeros(self.shape) for _ in range(3))
        lib().oracle_momentum(self.nx, self.ny, self.nz, self.h, self.dx, self.dy,
                              _p(self.tzc1), _p(self.tzc2), _p(self.tzd1), _p(self.tzd2),
                              _p(u), _p(v), _p(w), _p(su), _p(sv), _p(sw),
                              int(bool(skew)), int(nthreads))
        return su, sv, sw

    def scalar(self, u, v, w, q, skew=False, nthreads=1, out=None):
        for a in (u, v, w, q):
            _chk(a, self.shape)
        sq = out if out is not None else np.zeros(self.shape)
        lib().oracle_scalar(self.nx, self.ny, self.nz, self.h, self.dx, self.dy,
                            _p(self.tzc1), _p(self.tzc2), _p(u), _p(v), _p(w), _p(q), _p(sq),
                            int(bool(skew)), int(nthreads))
        return sq

    def points(self, which, u, v, w, q, ii, jj, kk, skew=False):
        """Tendency `which` in {'su','sv','sw','sq'} at sampled array indices."""
        code = {"su": 0, "sv": 1, "sw": 2, "sq": 3}[which]
        for a in (u, v, w):
            _chk(a, self.shape)
        if code == 3:
            _chk(q, self.shape)
        ii, jj, kk = (np.ascontiguousarray(a, dtype=np.int32) for a in (ii, jj, kk))
        out = np.zeros(len(ii))
        ipt = C.POINTER(C.c_int)
        lib().oracle_points(code, self.nx, self.ny, self.nz, self.h, self.dx, self.dy,
                            _p(self.tzc1), _p(self.tzc2), _p(self.tzd1), _p(self.tzd2),
                            _p(u), _p(v), _p(w), _p(q) if code == 3 else None,
                            int(bool(skew)), len(ii), ii.ctypes.data_as(ipt),
                            jj.ctypes.data_as(ipt), kk.ctypes.data_as(ipt), _p(out))
        return out

"""ctypes loader for the CPU oracle (TEST INFRASTRUCTURE -- see oracle/md_oracle.c).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It holds argument marshalling only; all arithmetic is in md_oracle.c.
"""
import ctypes
import os

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
_libs = {}


def _load(quad=False):
    key = bool(quad)
    if key not in _libs:
        _build.build(quad=quad)
        path = _build.LIB_QUAD if quad else _build.LIB
        lib = ctypes.CDLL(path)
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int32)
        lib.oracle_boys.argtypes = [ctypes.c_int, ctypes.c_double, dp]
        lib.oracle_hermite_E2.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_double, dp]
        lib.oracle_hermite_E1.argtypes = [ctypes.c_int, ctypes.c_double, dp]
        lib.oracle_hermite_R.argtypes = [ctypes.c_int, ctypes.c_double, ctypes.c_double, dp, dp]
        lib.oracle_cart2solid.argtypes = [ctypes.c_int, dp]
        lib.oracle_eri_batch.argtypes = [
            ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_int),
            ctypes.POINTER(dp), ctypes.POINTER(dp), ctypes.POINTER(dp),
            ctypes.c_int64, ip, ip, ip, ip, ctypes.c_int, ctypes.c_int, dp]
        lib.oracle_max_threads.restype = ctypes.c_int
        lib.oracle_is_quad.restype = ctypes.c_int
        _libs[key] = lib
    return _libs[key]


def _dptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _iptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))


def ncart(l):
    return (l + 1) * (l + 2) // 2


def nsolid(l):
    return 2 * l + 1


def max_threads():
    return int(_load().oracle_max_threads())


def boys(mmax, x, quad=False):
    """F_m(x), m = 0..mmax (Eq. 22)."""
    out = np.zeros(mmax + 1)
    _load(quad).oracle_boys(int(mmax), float(x), _dptr(out))
    return out


def hermite_E2(la, lb, za, zb, xab, quad=False):
    """Two-center 1-D table E[i, j, t] (Eqs. 9, 10, 13, 14)."""
    out = np.zeros((la + 1, lb + 1, la + lb + 1))
    _load(quad).oracle_hermite_E2(la, lb, float(za), float(zb), float(xab), _dptr(out))
    return out


def hermite_E1(l, za, quad=False):
    """One-center 1-D table E[a, t] (Eqs. 8, 11, 12)."""
    out = np.zeros((l + 1, l + 1))
    _load(quad).oracle_hermite_E1(l, float(za), _dptr(out))
    return out


def hermite_R(L, p, q, PQ, quad=False):
    """[tuv]^(0) as a dense (L+1)^3 cube, zero for t+u+v > L (Eqs. 21, 23, 24)."""
    out = np.zeros((L + 1, L + 1, L + 1))
    pq = np.ascontiguousarray(PQ, dtype=np.float64)
    _load(quad).oracle_hermite_R(int(L), float(p), float(q), _dptr(pq), _dptr(out))
    return out


def cart2solid(l):
    """C[m+l, cart] of the Racah-normalised real solid harmonics (Eqs. 16-17)."""
    out = np.zeros((2 * l + 1, ncart(l)))
    _load().oracle_cart2solid(int(l), _dptr(out))
    return out


def _marshal(shells):
    ls = (ctypes.c_int * 4)()
    Ks = (ctypes.c_int * 4)()
    dp = ctypes.POINTER(ctypes.c_double)
    cen = (dp * 4)()
    exs = (dp * 4)()
    cos = (dp * 4)()
    keep = []
    for k, s in enumerate(shells):
        l, c, e, w = s
        c = np.ascontiguousarray(c, dtype=np.float64).reshape(-1, 3)
        e = np.ascontiguousarray(e, dtype=np.float64).reshape(c.shape[0], -1)
        w = np.ascontiguousarray(w, dtype=np.float64).reshape(c.shape[0], -1)
        assert e.shape == w.shape
        if not 0 <= int(l) <= 6:
            raise ValueError("oracle supports 0 <= l <= 6")
        ls[k] = int(l)
        Ks[k] = e.shape[1]
        cen[k], exs[k], cos[k] = _dptr(c), _dptr(e), _dptr(w)
        keep += [c, e, w]
    return ls, Ks, cen, exs, cos, keep


def eri4(a, b, c, d, ia, ib, ic, id_, pure, quad=False):
    """(ab|cd) for quartets i = (a[ia[i]], b[ib[i]], c[ic[i]], d[id_[i]]).

    Each of a, b, c, d is a tuple (l, center[n,3], exps[n,K], coefs[n,K]).  Returns
    out[n, na, nb, nc, nd] (Cartesian or solid components, SURVEY.md 8(b) order).
    """
    ls, Ks, cen, exs, cos, keep = _marshal([a, b, c, d])
    idx = [np.ascontiguousarray(x, dtype=np.int32) for x in (ia, ib, ic, id_)]
    n = len(idx[0])
    nf = nsolid if pure else ncart
    shape = (n, nf(a[0]), nf(b[0]), nf(c[0]), nf(d[0]))
    out = np.zeros(shape)
    _load(quad).oracle_eri_batch(ls, Ks, cen, exs, cos, n, _iptr(idx[0]), _iptr(idx[1]), _iptr(idx[2]), _iptr(idx[3]),
                                 0, int(bool(pure)), _dptr(out))
    return out


def eri3(a, b, x, ia, ib, ix, pure, quad=False):
    """(ab|X) with the one-center ket of PAPER.md Eqs. 2, 6, 8.  Returns out[n, na, nb, nX]."""
    ls, Ks, cen, exs, cos, keep = _marshal([a, b, x, x])
    idx = [np.ascontiguousarray(v, dtype=np.int32) for v in (ia, ib, ix)]
    n = len(idx[0])
    nf = nsolid if pure else ncart
    out = np.zeros((n, nf(a[0]), nf(b[0]), nf(x[0])))
    _load(quad).oracle_eri_batch(ls, Ks, cen, exs, cos, n, _iptr(idx[0]), _iptr(idx[1]), _iptr(idx[2]), _iptr(idx[2]),
                                 1, int(bool(pure)), _dptr(out))
    return out

"""Independent Obara-Saika VRR + Head-Gordon-Pople HRR evaluation of (ab|cd) over contracted
Cartesian Gaussians (Refs. 23-24 of the paper).  Pure Python, tiny inputs only.

It is a PIN for the oracle, not part of it: a different algorithm (no Hermite Gaussians, no E
coefficients, no R tensor), its own Boys function (scipy's regularised incomplete gamma) and its
own loops.  Form per SURVEY.md 8(c) "Independent Obara-Saika oracle-2".
"""
import math
from functools import lru_cache

import numpy as np
from scipy import special


def boys_gamma(m, T):
    """F_m(T) = gamma(m+1/2) P(m+1/2, T) / (2 T^{m+1/2}); Taylor series near T = 0."""
    if T < 1e-3:
        return sum((-T) ** k / (math.factorial(k) * (2 * m + 2 * k + 1)) for k in range(8))
    return special.gamma(m + 0.5) * special.gammainc(m + 0.5, T) / (2.0 * T ** (m + 0.5))


def cart_list(l):
    return [(ax, ay, l - ax - ay) for ax in range(l, -1, -1) for ay in range(l - ax, -1, -1)]


def _dec(v, i):
    w = list(v); w[i] -= 1
    return tuple(w)


def _inc(v, i):
    w = list(v); w[i] += 1
    return tuple(w)


def eri_os(la, lb, lc, ld, A, B, C, D, za, ca, zb, cb, zc, cc, zd, cd):
    """Contracted Cartesian shell quartet [na, nb, nc, nd]; exps/coefs are 1-D sequences."""
    A, B, C, D = (np.asarray(x, dtype=float) for x in (A, B, C, D))
    Lb, Lk = la + lb, lc + ld
    contracted = {}

    for ea, wa in zip(za, ca):
        for eb, wb in zip(zb, cb):
            p = ea + eb
            P = (ea * A + eb * B) / p
            Kab = math.exp(-ea * eb / p * float(np.dot(A - B, A - B)))
            for ec, wc in zip(zc, cc):
                for ed, wd in zip(zd, cd):
                    q = ec + ed
                    Q = (ec * C + ed * D) / q
                    Kcd = math.exp(-ec * ed / q * float(np.dot(C - D, C - D)))
                    rho = p * q / (p + q)
                    W = (p * P + q * Q) / (p + q)
                    T = rho * float(np.dot(P - Q, P - Q))
                    pref = 2.0 * math.pi ** 2.5 / (p * q * math.sqrt(p + q)) * Kab * Kcd
                    F = [boys_gamma(m, T) for m in range(Lb + Lk + 1)]

                    @lru_cache(maxsize=None)
                    def theta(a, c, m):
                        if min(a) < 0 or min(c) < 0:
                            return 0.0
                        if sum(a) == 0 and sum(c) == 0:
                            return pref * F[m]
                        if sum(c) > 0:          # ket VRR
                            i = next(k for k in range(3) if c[k] > 0)
                            c1 = _dec(c, i)
                            v = (Q[i] - C[i]) * theta(a, c1, m) + (W[i] - Q[i]) * theta(a, c1, m + 1)
                            if c1[i] > 0:
                                c2 = _dec(c1, i)
                                v += c1[i] / (2 * q) * (theta(a, c2, m) - rho / q * theta(a, c2, m + 1))
                            if a[i] > 0:
                                v += a[i] / (2 * (p + q)) * theta(_dec(a, i), c1, m + 1)
                            return v
                        i = next(k for k in range(3) if a[k] > 0)   # bra VRR (c = 0)
                        a1 = _dec(a, i)
                        v = (P[i] - A[i]) * theta(a1, c, m) + (W[i] - P[i]) * theta(a1, c, m + 1)
                        if a1[i] > 0:
                            a2 = _dec(a1, i)
                            v += a1[i] / (2 * p) * (theta(a2, c, m) - rho / p * theta(a2, c, m + 1))
                        return v

                    w = wa * wb * wc * wd
                    for le in range(la, Lb + 1):
                        for e in cart_list(le):
                            for lf in range(lc, Lk + 1):
                                for f in cart_list(lf):
                                    contracted[(e, f)] = contracted.get((e, f), 0.0) + w * theta(e, f, 0)

    AB, CD = A - B, C - D

    @lru_cache(maxsize=None)
    def hrr(a, b, c, d):
        if sum(b) > 0:
            i = next(k for k in range(3) if b[k] > 0)
            b1 = _dec(b, i)
            return hrr(_inc(a, i), b1, c, d) + AB[i] * hrr(a, b1, c, d)
        if sum(d) > 0:
            i = next(k for k in range(3) if d[k] > 0)
            d1 = _dec(d, i)
            return hrr(a, b, _inc(c, i), d1) + CD[i] * hrr(a, b, c, d1)
        return contracted[(a, c)]

    out = np.zeros((len(cart_list(la)), len(cart_list(lb)), len(cart_list(lc)), len(cart_list(ld))))
    for ia, a in enumerate(cart_list(la)):
        for ib, b in enumerate(cart_list(lb)):
            for ic, c in enumerate(cart_list(lc)):
                for id_, d in enumerate(cart_list(ld)):
                    out[ia, ib, ic, id_] = hrr(a, b, c, d)
    return out

"""Pins of oracle/two_center.py (no GPU)."""
import math

import numpy as np
from scipy.special import erf

from oracle import two_center as o2
from paper_2405_01834_b200 import workloads as W


def _f0(T):
    return 1.0 if T < 1e-14 else 0.5 * math.sqrt(math.pi / T) * erf(math.sqrt(T))


def test_ss_closed_form_and_symmetry():
    rng = np.random.default_rng(1)
    x = W.make_shells(rng, 6, 0, 1, (0.2, 9.0), (-2.0, 2.0))
    y = W.make_shells(rng, 5, 0, 1, (0.2, 9.0), (-2.0, 2.0))
    ix, iy = np.divmod(np.arange(30, dtype=np.int32), 5)
    v = o2.eri2(x.astuple(), y.astuple(), ix, iy, True)[:, 0, 0]
    for k in range(30):
        p, q = x.exps[ix[k], 0], y.exps[iy[k], 0]
        R2 = np.sum((x.center[ix[k]] - y.center[iy[k]]) ** 2)
        ref = x.coefs[ix[k], 0] * y.coefs[iy[k], 0] * 2 * math.pi ** 2.5 / (p * q * math.sqrt(p + q)) * _f0(p * q / (p + q) * R2)
        assert abs(v[k] - ref) <= 1e-14 * abs(ref)
    for lx, ly in [(1, 0), (2, 1), (3, 3), (4, 2)]:
        a = W.make_shells(rng, 4, lx, 2, (0.3, 5.0), (-1.5, 1.5))
        b = W.make_shells(rng, 4, ly, 1, (0.3, 5.0), (-1.5, 1.5))
        i = np.arange(4, dtype=np.int32)
        for pure in (True, False):
            ab, ba = o2.eri2(a.astuple(), b.astuple(), i, i, pure), o2.eri2(b.astuple(), a.astuple(), i, i, pure)
            assert np.allclose(ab, ba.transpose(0, 2, 1), rtol=1e-11, atol=1e-14)


def test_p_s_is_the_centre_derivative_of_s_s():
    rng = np.random.default_rng(2)
    zx, zy = 0.9, 1.7
    X, Y = rng.uniform(-1, 1, 3), rng.uniform(-1, 1, 3)
    s = lambda c: (0, c.reshape(1, 3), np.array([[zx]]), np.array([[1.0]]))
    ys = (0, Y.reshape(1, 3), np.array([[zy]]), np.array([[1.0]]))
    px = (1, X.reshape(1, 3), np.array([[zx]]), np.array([[1.0]]))
    i = np.zeros(1, dtype=np.int32)
    ps = o2.eri2(px, ys, i, i, False)[0, :, 0]                         # Cartesian p: x, y, z
    h = 1e-4
    for ax in range(3):
        d = np.zeros(3); d[ax] = h
        fd = (o2.eri2(s(X + d), ys, i, i, False)[0, 0, 0] - o2.eri2(s(X - d), ys, i, i, False)[0, 0, 0]) / (2 * h)
        assert abs(ps[ax] - fd / (2 * zx)) < 1e-8 * max(1.0, abs(ps[ax]))


def test_solid_block_norm_is_rotation_invariant():
    rng = np.random.default_rng(3)
    a = W.make_shells(rng, 1, 3, 1, (0.5, 2.0), (-1.0, 1.0))
    b = W.make_shells(rng, 1, 4, 1, (0.5, 2.0), (-1.0, 1.0))
    Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    i = np.zeros(1, dtype=np.int32)
    n0 = np.linalg.norm(o2.eri2(a.astuple(), b.astuple(), i, i, True))
    ar = (a.l, a.center @ Q.T, a.exps, a.coefs)
    br = (b.l, b.center @ Q.T, b.exps, b.coefs)
    assert abs(np.linalg.norm(o2.eri2(ar, br, i, i, True)) - n0) <= 1e-12 * n0

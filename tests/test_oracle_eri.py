"""Pins for the oracle's full integrals (Eqs. 2-4, 7, 19, 25-26).

Closed forms, exact identities that link classes (HRR), symmetries, an independent Obara-Saika
code (tests/os_reference.py), linearity in the contraction, rotation invariance of solid blocks,
the Hobson pin for the one-center side, and the 3-center == dummy-shell 4-center equivalence.
"""
import itertools
import math

import numpy as np
import pytest

import oracle
from os_reference import cart_list, eri_os
from paper_2405_01834_b200 import workloads as wl


def sh(l, center, exps, coefs):
    return (l, np.asarray(center, float).reshape(1, 3), np.asarray(exps, float).reshape(1, -1), np.asarray(coefs, float).reshape(1, -1))


def one(a, b, c, d, pure=False, quad=False):
    return oracle.eri4(a, b, c, d, [0], [0], [0], [0], pure, quad=quad)[0]


def rand_shell(rng, l, K=1, box=1.0, zr=(0.3, 3.0)):
    return sh(l, rng.uniform(-box, box, 3), np.exp(rng.uniform(math.log(zr[0]), math.log(zr[1]), K)), rng.uniform(0.3, 1.0, K))


def cidx(l):
    return {c: k for k, c in enumerate(cart_list(l))}


# ---------------------------------------------------------------- closed form (ss|ss)

def test_ssss_closed_form():
    rng = np.random.default_rng(0)
    for _ in range(50):
        A, B, C, D = rng.uniform(-3, 3, (4, 3))
        za, zb, zc, zd = np.exp(rng.uniform(math.log(0.1), math.log(20), 4))
        v = one(sh(0, A, [za], [1]), sh(0, B, [zb], [1]), sh(0, C, [zc], [1]), sh(0, D, [zd], [1]))[0, 0, 0, 0]
        p, q = za + zb, zc + zd
        P, Q = (za * A + zb * B) / p, (zc * C + zd * D) / q
        T = p * q / (p + q) * np.sum((P - Q) ** 2)
        F0 = 0.5 * math.sqrt(math.pi / T) * math.erf(math.sqrt(T)) if T > 1e-12 else 1.0
        ref = 2 * math.pi ** 2.5 / (p * q * math.sqrt(p + q)) * math.exp(-za * zb / p * np.sum((A - B) ** 2)) \
            * math.exp(-zc * zd / q * np.sum((C - D) ** 2)) * F0
        assert abs(v - ref) <= 1e-13 * abs(ref)   # exp() of a large argument carries |arg| ulps


def test_far_field_limit():
    # (ss|ss) -> S_ab S_cd / |PQ| when the charge clouds do not overlap
    A, B = np.array([0.0, 0.1, 0.0]), np.array([0.2, 0.0, 0.1])
    C, D = A + [40.0, 0, 0], B + [40.0, 0.3, 0]
    za, zb, zc, zd = 1.1, 0.8, 1.4, 0.6
    v = one(sh(0, A, [za], [1]), sh(0, B, [zb], [1]), sh(0, C, [zc], [1]), sh(0, D, [zd], [1]))[0, 0, 0, 0]
    p, q = za + zb, zc + zd
    P, Q = (za * A + zb * B) / p, (zc * C + zd * D) / q
    Sab = (math.pi / p) ** 1.5 * math.exp(-za * zb / p * np.sum((A - B) ** 2))
    Scd = (math.pi / q) ** 1.5 * math.exp(-zc * zd / q * np.sum((C - D) ** 2))
    assert abs(v - Sab * Scd / np.linalg.norm(P - Q)) <= 1e-13 * v


# ---------------------------------------------------------------- independent Obara-Saika, l <= 2 (and one l = 3)

@pytest.mark.parametrize("ls", [(0, 0, 0, 0), (1, 0, 0, 0), (0, 1, 0, 0), (0, 0, 1, 0), (0, 0, 0, 1), (1, 1, 1, 1), (2, 0, 1, 0),
                                (2, 1, 0, 2), (1, 2, 2, 1), (2, 2, 2, 2), (0, 2, 1, 2), (3, 1, 2, 0)])
def test_against_obara_saika(ls):
    rng = np.random.default_rng(sum(k * 5 ** i for i, k in enumerate(ls)))
    Ks = (2, 1, 1, 2) if sum(ls) <= 5 else (1, 1, 1, 1)
    shells = [rand_shell(rng, l, K) for l, K in zip(ls, Ks)]
    got = one(*shells)
    args = []
    for s in shells:
        args += [s[2][0], s[3][0]]
    ref = eri_os(*ls, *[s[1][0] for s in shells], *args)
    assert got.shape == ref.shape
    assert np.max(np.abs(got - ref)) <= 2e-12 * max(1.0, np.max(np.abs(ref)))
    assert np.max(np.abs(got - ref)) <= 1e-10 * np.max(np.abs(ref))


# ---------------------------------------------------------------- symmetries and invariances

@pytest.mark.parametrize("ls", [(1, 0, 2, 1), (2, 1, 1, 0), (3, 2, 1, 1), (4, 0, 2, 3)])
def test_permutational_symmetry(ls):
    rng = np.random.default_rng(11 + sum(ls))
    a, b, c, d = [rand_shell(rng, l, 2 if i % 2 else 1) for i, l in enumerate(ls)]
    for pure in (False, True):
        base = one(a, b, c, d, pure)
        tol = 1e-13 * np.max(np.abs(base))
        assert np.max(np.abs(one(b, a, c, d, pure) - base.transpose(1, 0, 2, 3))) <= tol
        assert np.max(np.abs(one(a, b, d, c, pure) - base.transpose(0, 1, 3, 2))) <= tol
        assert np.max(np.abs(one(c, d, a, b, pure) - base.transpose(2, 3, 0, 1))) <= tol
        assert np.max(np.abs(one(d, c, b, a, pure) - base.transpose(3, 2, 1, 0))) <= tol


def test_translation_invariance():
    rng = np.random.default_rng(3)
    shells = [rand_shell(rng, l) for l in (2, 1, 3, 2)]
    shift = np.array([0.7, -1.3, 2.1])
    moved = [(s[0], s[1] + shift, s[2], s[3]) for s in shells]
    x, y = one(*shells), one(*moved)
    assert np.max(np.abs(x - y)) <= 1e-12 * np.max(np.abs(x))


def _rot(rng):
    q, r = np.linalg.qr(rng.normal(size=(3, 3)))
    q = q * np.sign(np.diag(r))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    return q


@pytest.mark.parametrize("ls", [(2, 2, 2, 2), (3, 1, 0, 2), (4, 2, 3, 1), (6, 0, 1, 0)])
def test_rotation_invariance_of_solid_block_norm(ls):
    # Racah real solid harmonics of one l mix orthogonally under rotation => Frobenius norm invariant;
    # for l >= 2 the Cartesian block norm is NOT invariant, so this pins the Cartesian->solid coefficients.
    rng = np.random.default_rng(21 + sum(ls))
    shells = [rand_shell(rng, l) for l in ls]
    U = _rot(rng)
    rotated = [(s[0], s[1] @ U.T, s[2], s[3]) for s in shells]
    n0 = np.linalg.norm(one(*shells, pure=True))
    n1 = np.linalg.norm(one(*rotated, pure=True))
    assert abs(n0 - n1) <= 1e-12 * n0
    if max(ls) >= 2:
        c0, c1 = np.linalg.norm(one(*shells)), np.linalg.norm(one(*rotated))
        assert abs(c0 - c1) > 1e-6 * c0


def test_solid_equals_cartesian_for_s_and_p():
    rng = np.random.default_rng(4)
    shells = [rand_shell(rng, l) for l in (1, 0, 1, 1)]
    c, s = one(*shells), one(*shells, pure=True)
    perm = [1, 2, 0]    # solid p order (y,z,x) out of Cartesian (x,y,z)
    assert np.array_equal(s, c[perm][:, :, perm][:, :, :, perm])


# ---------------------------------------------------------------- HRR identity links classes up to l = 6

@pytest.mark.parametrize("la,lb,lc,ld", [(0, 0, 0, 0), (1, 0, 1, 0), (2, 1, 0, 1), (3, 2, 1, 0), (4, 3, 0, 0), (5, 5, 0, 0), (2, 2, 2, 1), (5, 5, 1, 0), (3, 3, 3, 2)])
def test_hrr_identity_bra(la, lb, lc, ld):
    # (a (b+1_i) | cd) = ((a+1_i) b | cd) + (A_i - B_i)(ab|cd), exact for contracted shells
    rng = np.random.default_rng(100 + la * 49 + lb * 7 + lc)
    K = 2 if la + lb + lc + ld <= 6 else 1
    A, B = rng.uniform(-0.6, 0.6, (2, 3))
    za, ca = np.exp(rng.uniform(-0.5, 1.0, K)), rng.uniform(0.3, 1, K)
    zb, cb = np.exp(rng.uniform(-0.5, 1.0, K)), rng.uniform(0.3, 1, K)
    c, d = rand_shell(rng, lc, 1, 0.6), rand_shell(rng, ld, 1, 0.6)
    I_ab1 = one(sh(la, A, za, ca), sh(lb + 1, B, zb, cb), c, d)
    I_a1b = one(sh(la + 1, A, za, ca), sh(lb, B, zb, cb), c, d)
    I_ab = one(sh(la, A, za, ca), sh(lb, B, zb, cb), c, d)
    ia, ia1, ib, ib1 = cidx(la), cidx(la + 1), cidx(lb), cidx(lb + 1)
    scale = max(np.max(np.abs(I_ab1)), np.max(np.abs(I_a1b)), np.max(np.abs(I_ab)))
    worst = 0.0
    for a in cart_list(la):
        for b in cart_list(lb):
            for i in range(3):
                a1 = tuple(a[k] + (k == i) for k in range(3))
                b1 = tuple(b[k] + (k == i) for k in range(3))
                lhs = I_ab1[ia[a], ib1[b1]]
                rhs = I_a1b[ia1[a1], ib[b]] + (A[i] - B[i]) * I_ab[ia[a], ib[b]]
                worst = max(worst, np.max(np.abs(lhs - rhs)))
    assert worst <= 2e-13 * scale


def test_hrr_identity_ket():
    rng = np.random.default_rng(77)
    a, b = rand_shell(rng, 2, 1, 0.6), rand_shell(rng, 1, 2, 0.6)
    C, D = rng.uniform(-0.6, 0.6, (2, 3))
    zc, cc, zd, cd = [1.3, 0.4], [0.5, 0.9], [0.8], [1.0]
    lc, ld = 3, 2
    I1 = one(a, b, sh(lc, C, zc, cc), sh(ld + 1, D, zd, cd))
    I2 = one(a, b, sh(lc + 1, C, zc, cc), sh(ld, D, zd, cd))
    I0 = one(a, b, sh(lc, C, zc, cc), sh(ld, D, zd, cd))
    ic, ic1, id_, id1 = cidx(lc), cidx(lc + 1), cidx(ld), cidx(ld + 1)
    scale = max(np.max(np.abs(I1)), np.max(np.abs(I2)))
    for c in cart_list(lc):
        for d in cart_list(ld):
            for i in range(3):
                c1 = tuple(c[k] + (k == i) for k in range(3))
                d1 = tuple(d[k] + (k == i) for k in range(3))
                lhs = I1[:, :, ic[c], id1[d1]]
                rhs = I2[:, :, ic1[c1], id_[d]] + (C[i] - D[i]) * I0[:, :, ic[c], id_[d]]
                assert np.max(np.abs(lhs - rhs)) <= 2e-13 * scale


def test_derivative_identity_central_differences():
    # d/dA_i (ab|cd) = 2 za ((a+1_i) b|cd) - a_i ((a-1_i) b|cd), K = 1
    rng = np.random.default_rng(8)
    la = 2
    A = rng.uniform(-0.5, 0.5, 3)
    za = 0.9
    b, c, d = rand_shell(rng, 1), rand_shell(rng, 2), rand_shell(rng, 0)
    up = one(sh(la + 1, A, [za], [1]), b, c, d)
    dn = one(sh(la - 1, A, [za], [1]), b, c, d)
    iu, idn, i0 = cidx(la + 1), cidx(la - 1), cidx(la)
    h = 1e-4
    for i in range(3):
        e = np.zeros(3); e[i] = h
        num = (-one(sh(la, A + 2 * e, [za], [1]), b, c, d) + 8 * one(sh(la, A + e, [za], [1]), b, c, d)
               - 8 * one(sh(la, A - e, [za], [1]), b, c, d) + one(sh(la, A - 2 * e, [za], [1]), b, c, d)) / (12 * h)
        for a in cart_list(la):
            a1 = tuple(a[k] + (k == i) for k in range(3))
            ana = 2 * za * up[iu[a1]]
            if a[i] > 0:
                am = tuple(a[k] - (k == i) for k in range(3))
                ana = ana - a[i] * dn[idn[am]]
            assert np.max(np.abs(num[i0[a]] - ana)) <= 1e-8 * max(1.0, np.max(np.abs(ana)))


# ---------------------------------------------------------------- contraction loop, Schwarz, degenerate geometry

def test_contraction_is_linear_in_primitives():
    rng = np.random.default_rng(9)
    ls, Ks = (2, 1, 1, 2), (3, 2, 2, 1)
    shells = [rand_shell(rng, l, K) for l, K in zip(ls, Ks)]
    full = one(*shells, pure=True)
    acc = np.zeros_like(full)
    for ks in itertools.product(*[range(K) for K in Ks]):
        prim = [sh(s[0], s[1], [s[2][0, k]], [1.0]) for s, k in zip(shells, ks)]
        w = np.prod([s[3][0, k] for s, k in zip(shells, ks)])
        acc += w * one(*prim, pure=True)
    assert np.max(np.abs(full - acc)) <= 1e-13 * np.max(np.abs(full))


def test_schwarz_and_positivity():
    rng = np.random.default_rng(10)
    a, b, c, d = [rand_shell(rng, l) for l in (2, 1, 1, 2)]
    abab = one(a, b, a, b)
    cdcd = one(c, d, c, d)
    abcd = one(a, b, c, d)
    na, nb, nc, nd = abcd.shape
    for i, j, k, l in itertools.product(range(na), range(nb), range(nc), range(nd)):
        assert abab[i, j, i, j] >= 0 and cdcd[k, l, k, l] >= 0
        assert abs(abcd[i, j, k, l]) <= math.sqrt(abab[i, j, i, j] * cdcd[k, l, k, l]) * (1 + 1e-12) + 1e-300


def test_degenerate_geometry_is_regular_and_symmetric():
    # reading S7: A=B, C=D, all equal: no division by a distance anywhere
    a = sh(2, [0.1, 0.2, 0.3], [1.1], [1.0])
    b = sh(1, [0.1, 0.2, 0.3], [0.7], [1.0])
    v = one(a, b, a, b, pure=True)
    assert np.all(np.isfinite(v))
    assert np.max(np.abs(v - v.transpose(2, 3, 0, 1))) <= 1e-15 * np.max(np.abs(v))
    # one-center (ss|ss), all exponents z: 2 pi^{5/2} / (2z 2z sqrt(4z))
    z = 0.8
    s = sh(0, [0, 0, 0], [z], [1.0])
    assert abs(one(s, s, s, s)[0, 0, 0, 0] - 2 * math.pi ** 2.5 / (4 * z * z * math.sqrt(4 * z))) < 1e-14


# ---------------------------------------------------------------- 3-center

@pytest.mark.parametrize("la,lb,lx", [(0, 0, 0), (1, 0, 2), (2, 2, 3), (3, 1, 6), (0, 3, 4)])
def test_eri3_equals_eri4_with_dummy_s_shell(la, lb, lx):
    # reading O3: (ab|X) == (ab|X s0) with the dummy s shell zeta = 0, c = 1 at X
    rng = np.random.default_rng(50 + la + 7 * lb + 49 * lx)
    a, b, x = rand_shell(rng, la, 2), rand_shell(rng, lb, 1), rand_shell(rng, lx, 1)
    dummy = sh(0, x[1][0], [0.0], [1.0])
    for pure in (False, True):
        t = oracle.eri3(a, b, x, [0], [0], [0], pure)[0]
        f = one(a, b, x, dummy, pure)[..., 0]
        assert np.max(np.abs(t - f)) <= 1e-14 * np.max(np.abs(f))
        assert np.max(np.abs(oracle.eri3(b, a, x, [0], [0], [0], pure)[0] - t.transpose(1, 0, 2))) <= 1e-13 * np.max(np.abs(t))


def test_hobson_pin_one_center_side():
    # S_lm(grad_A) e^{-z r_A^2} = (2z)^l S_lm(r_A) e^{-z r_A^2}: in H_X = C . E1 every Hermite order < l_X cancels
    for l in range(7):
        z = 0.6 + 0.2 * l
        E1 = oracle.hermite_E1(l, z)
        C = oracle.cart2solid(l)
        comps = cart_list(l)
        H = {}
        for m in range(2 * l + 1):
            for k, (ax, ay, az) in enumerate(comps):
                for t in range(ax + 1):
                    for u in range(ay + 1):
                        for v in range(az + 1):
                            H[(m, t, u, v)] = H.get((m, t, u, v), 0.0) + C[m, k] * E1[ax, t] * E1[ay, u] * E1[az, v]
        for (m, t, u, v), val in H.items():
            if t + u + v < l:
                assert abs(val) < 1e-13
            else:
                k = comps.index((t, u, v))
                assert abs(val - C[m, k] / (2 * z) ** l) < 1e-13


# ---------------------------------------------------------------- roundoff attribution (finding F1 iii)

def test_double_oracle_agrees_with_quad_oracle():
    rng = np.random.default_rng(12)
    for ls in [(1, 1, 1, 1), (2, 2, 2, 2), (4, 3, 2, 1), (6, 6, 1, 0)]:
        shells = [rand_shell(rng, l, 1, 0.5, (0.3, 10.0)) for l in ls]
        d, q = one(*shells, pure=True), one(*shells, pure=True, quad=True)
        assert np.max(np.abs(d - q)) <= 1e-12 * np.max(np.abs(q))


def test_batch_indexing_matches_single_calls():
    w = wl.config1(n=6)
    ia, ib, ic, id_ = w.shell_indices()
    out = oracle.eri4(w.a.astuple(), w.b.astuple(), w.c.astuple(), w.d.astuple(), ia, ib, ic, id_, False)
    for i in (0, 3, 5):
        single = one(*[s.take([i]).astuple() for s in (w.a, w.b, w.c, w.d)])
        assert np.array_equal(out[i], single)

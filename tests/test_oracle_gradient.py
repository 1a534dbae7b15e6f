"""Pins of oracle/gradient.py (first geometric derivatives of (ab|cd)).

None of the pins uses the derivative rule the oracle writes out:
  * central differences of oracle.eri4 under a displaced centre, Richardson-extrapolated (error O(h^4));
  * translational invariance: the integral depends on centre differences only, so the four centre derivatives sum to zero;
  * the closed form of d/dA (ss|ss) for primitives, from F_0(T) = sqrt(pi/T) erf(sqrt T)/2 and F_0' = -F_1 = -(F_0 - e^-T)/(2T);
  * (ab|cd) = (cd|ab): the derivative with respect to a of (ab|cd) is the derivative with respect to c of (cd|ab), transposed.
"""
import math

import numpy as np
import pytest

import oracle
from oracle import gradient


def shells(rng, ls, Ks, n=3):
    out = []
    for l, K in zip(ls, Ks):
        out.append((l, rng.uniform(-1.5, 1.5, (n, 3)), np.exp(rng.uniform(np.log(0.4), np.log(3.0), (n, K))), rng.uniform(0.5, 1.5, (n, K))))
    return out


def displaced(s, i, h):
    l, c, e, w = s
    c = c.copy()
    c[:, i] += h
    return (l, c, e, w)


def fd_grad(sh, idx, pure, center, h=2e-2):
    """Richardson: (4 D(h/2) - D(h)) / 3 with D the central difference; O(h^4) truncation."""
    out = []
    for i in range(3):
        def D(hh):
            p = list(sh); m = list(sh)
            p[center] = displaced(sh[center], i, hh)
            m[center] = displaced(sh[center], i, -hh)
            return (oracle.eri4(*p, *idx, pure) - oracle.eri4(*m, *idx, pure)) / (2 * hh)
        out.append((4 * D(h / 2) - D(h)) / 3)
    return np.stack(out, axis=1)


CASES = [((0, 0, 0, 0), (1, 1, 1, 1)), ((1, 0, 0, 0), (1, 1, 1, 1)), ((1, 1, 1, 1), (2, 1, 1, 2)), ((2, 1, 0, 2), (1, 2, 1, 1)),
         ((2, 2, 2, 2), (1, 1, 1, 1)), ((3, 1, 2, 0), (2, 1, 1, 1)), ((0, 3, 1, 2), (1, 1, 2, 1))]


@pytest.mark.parametrize("ls,Ks", CASES, ids=[str(c[0]) for c in CASES])
@pytest.mark.parametrize("pure", [False, True])
def test_gradient_matches_finite_differences(ls, Ks, pure):
    rng = np.random.default_rng(sum(ls) * 7 + pure)
    sh = shells(rng, ls, Ks)
    idx = [np.arange(3, dtype=np.int32)] * 4
    for center in range(4):
        g = gradient.eri4_grad(*sh, *idx, pure, center)
        f = fd_grad(sh, idx, pure, center)
        scale = np.abs(f).max()
        assert np.abs(g - f).max() <= 2e-7 * scale, (center, np.abs(g - f).max() / scale)


@pytest.mark.parametrize("ls,Ks", [((2, 1, 1, 2), (2, 1, 1, 1)), ((3, 2, 2, 1), (1, 1, 1, 1)), ((4, 0, 3, 1), (1, 1, 1, 1))])
def test_translational_invariance(ls, Ks):
    rng = np.random.default_rng(11)
    sh = shells(rng, ls, Ks)
    idx = [np.arange(3, dtype=np.int32)] * 4
    gs = [gradient.eri4_grad(*sh, *idx, True, c) for c in range(4)]
    scale = max(np.abs(g).max() for g in gs)
    assert np.abs(gs[0] + gs[1] + gs[2] + gs[3]).max() <= 1e-12 * scale


def test_ssss_closed_form():
    rng = np.random.default_rng(5)
    sh = shells(rng, (0, 0, 0, 0), (1, 1, 1, 1), n=6)
    idx = [np.arange(6, dtype=np.int32)] * 4
    g = gradient.eri4_grad(*sh, *idx, False, 0)[:, :, 0, 0, 0, 0]
    for n in range(6):
        (A, za, ca), (B, zb, cb), (C, zc, cc), (D, zd, cd) = [(s[1][n], s[2][n, 0], s[3][n, 0]) for s in sh]
        p, q = za + zb, zc + zd
        P, Q = (za * A + zb * B) / p, (zc * C + zd * D) / q
        rho = p * q / (p + q)
        T = rho * np.dot(P - Q, P - Q)
        F0 = 0.5 * math.sqrt(math.pi / T) * math.erf(math.sqrt(T))
        F1 = (F0 - math.exp(-T)) / (2 * T)
        pref = ca * cb * cc * cd * 2 * math.pi ** 2.5 / (p * q * math.sqrt(p + q))
        Kab = math.exp(-za * zb / p * np.dot(A - B, A - B)) * math.exp(-zc * zd / q * np.dot(C - D, C - D))
        ref = pref * Kab * (-2 * za * zb / p * (A - B) * F0 - F1 * 2 * rho * (P - Q) * za / p)
        assert np.allclose(g[n], ref, rtol=1e-12, atol=0)


def test_bra_ket_symmetry_of_the_derivative():
    rng = np.random.default_rng(8)
    sh = shells(rng, (2, 1, 1, 3), (1, 2, 1, 1))
    idx = [np.arange(3, dtype=np.int32)] * 4
    g_a = gradient.eri4_grad(sh[0], sh[1], sh[2], sh[3], *idx, True, 0)                 # d/dA (ab|cd)
    g_c = gradient.eri4_grad(sh[2], sh[3], sh[0], sh[1], *idx, True, 2)                 # d/dA (cd|ab)
    assert np.allclose(g_a, np.transpose(g_c, (0, 1, 4, 5, 2, 3)), rtol=1e-11, atol=1e-14)


def test_component_order_helpers():
    for l in range(0, 7):
        comps = gradient.cart_components(l)
        assert len(comps) == oracle.ncart(l)
        assert [gradient.cart_index(*c) for c in comps] == list(range(len(comps)))


# ---- 3-center (ab|X) ----------------------------------------------------------------------------------------------------------

def fd_grad3(sh, idx, pure, center, h=2e-2):
    out = []
    for i in range(3):
        def D(hh):
            p = list(sh); m = list(sh)
            p[center] = displaced(sh[center], i, hh)
            m[center] = displaced(sh[center], i, -hh)
            return (oracle.eri3(*p, *idx, pure) - oracle.eri3(*m, *idx, pure)) / (2 * hh)
        out.append((4 * D(h / 2) - D(h)) / 3)
    return np.stack(out, axis=1)


CASES3 = [((0, 0, 0), (1, 1, 1)), ((1, 0, 2), (1, 2, 1)), ((2, 1, 1), (2, 1, 1)), ((2, 2, 3), (1, 1, 1)), ((3, 1, 4), (1, 1, 2)), ((0, 2, 5), (1, 1, 1))]


@pytest.mark.parametrize("ls,Ks", CASES3, ids=[str(c[0]) for c in CASES3])
@pytest.mark.parametrize("pure", [False, True])
def test_gradient3_matches_finite_differences_and_sums_to_zero(ls, Ks, pure):
    rng = np.random.default_rng(sum(ls) * 5 + pure)
    sh = shells(rng, ls, Ks)
    idx = [np.arange(3, dtype=np.int32)] * 3
    gs = []
    for center in range(3):
        g = gradient.eri3_grad(*sh, *idx, pure, center)
        f = fd_grad3(sh, idx, pure, center)
        scale = np.abs(f).max()
        assert np.abs(g - f).max() <= 2e-7 * scale, (center, np.abs(g - f).max() / scale)
        gs.append(g)
    assert np.abs(gs[0] + gs[1] + gs[2]).max() <= 1e-12 * max(np.abs(g).max() for g in gs)


def test_gradient3_is_the_four_center_gradient_on_a_dummy_shell():
    """(ab|X) = (ab|X s0) with a zeta = 0, c = 1 dummy (reading S7): the derivatives must agree."""
    rng = np.random.default_rng(9)
    sh = shells(rng, (2, 1, 3), (1, 2, 1))
    dummy = (0, np.zeros((1, 3)), np.zeros((1, 1)), np.ones((1, 1)))
    idx = [np.arange(3, dtype=np.int32)] * 3
    z = np.zeros(3, dtype=np.int32)
    for center in range(3):
        g3 = gradient.eri3_grad(*sh, *idx, True, center)
        g4 = gradient.eri4_grad(sh[0], sh[1], sh[2], dummy, idx[0], idx[1], idx[2], z, True, center)[..., 0]
        assert np.allclose(g3, g4, rtol=1e-12, atol=1e-15)


# ---- 2-center (X|Y) -----------------------------------------------------------------------------------------------------------

@pytest.mark.parametrize("lx,ly", [(0, 0), (1, 0), (2, 1), (3, 3), (0, 4), (5, 2)])
@pytest.mark.parametrize("pure", [False, True])
def test_gradient2_matches_finite_differences_of_the_two_center_oracle(lx, ly, pure):
    from oracle import two_center
    rng = np.random.default_rng(lx * 7 + ly + pure)
    sh = shells(rng, (lx, ly), (2, 1))
    ix = iy = np.arange(3, dtype=np.int32)
    gs = []
    for center in range(2):
        g = gradient.eri2_grad(sh[0], sh[1], ix, iy, pure, center)
        fd = []
        for i in range(3):
            def D(hh):
                p = list(sh); m = list(sh)
                p[center] = displaced(sh[center], i, hh)
                m[center] = displaced(sh[center], i, -hh)
                return (two_center.eri2(p[0], p[1], ix, iy, pure) - two_center.eri2(m[0], m[1], ix, iy, pure)) / (2 * hh)
            fd.append((4 * D(1e-2) - D(2e-2)) / 3)
        f = np.stack(fd, axis=1)
        assert np.abs(g - f).max() <= 2e-7 * np.abs(f).max()
        gs.append(g)
    assert np.abs(gs[0] + gs[1]).max() <= 1e-12 * np.abs(gs[0]).max()      # the integral depends on X - Y only

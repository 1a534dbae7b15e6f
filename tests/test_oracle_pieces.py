"""Pins for the oracle's building blocks: Boys function, E tables, R tensor, solid harmonics.

Each test checks the oracle against something the paper or the mathematics fixes and that is NOT
the oracle's own formula: library special functions, closed forms, identities, quadrature.
(SURVEY.md 8(c) "What pins each part".)
"""
import math

import mpmath
import numpy as np
import pytest
from numpy.polynomial.hermite import hermgauss, hermval
from scipy import special

import oracle

MMAX = 24


# ----------------------------------------------------------------------------- Boys (Eq. 22)

def _boys_mp(m, x):
    mpmath.mp.dps = 50
    return mpmath.hyp1f1(m + 0.5, m + 1.5, -mpmath.mpf(x)) / (2 * m + 1)


@pytest.mark.parametrize("x", [0.0, 1e-8, 1e-3, 0.3, 1.0, 4.7, 12.0, 19.99, 25.0, 29.999, 30.0, 30.001, 33.0, 47.0, 80.0, 500.0, 2.5e4])
def test_boys_vs_mpmath_hyp1f1(x):
    F = oracle.boys(MMAX, x)
    for m in range(MMAX + 1):
        ref = float(_boys_mp(m, x))
        assert abs(F[m] - ref) <= 4e-15 * abs(ref), (m, x, F[m], ref)


def test_boys_vs_scipy_incomplete_gamma():
    for x in [0.5, 3.0, 11.0, 28.0, 31.0, 60.0]:
        F = oracle.boys(12, x)
        for m in range(13):
            ref = special.gamma(m + 0.5) * special.gammainc(m + 0.5, x) / (2 * x ** (m + 0.5))
            assert abs(F[m] - ref) <= 2e-13 * ref


def test_boys_closed_forms_and_recursion():
    # F_m(0) = 1/(2m+1); F_0(T) = 1/2 sqrt(pi/T) erf(sqrt T); F_{m-1} = (2T F_m + e^-T)/(2m-1)
    F = oracle.boys(MMAX, 0.0)
    assert np.allclose(F, 1.0 / (2 * np.arange(MMAX + 1) + 1), rtol=1e-15, atol=0)
    for T in [0.01, 2.0, 17.0, 29.0, 31.0, 45.0]:
        F = oracle.boys(MMAX, T)
        assert abs(F[0] - 0.5 * math.sqrt(math.pi / T) * math.erf(math.sqrt(T))) <= 2e-15 * F[0]
        for m in range(1, MMAX + 1):
            lhs = F[m - 1]
            rhs = (2 * T * F[m] + math.exp(-T)) / (2 * m - 1)
            assert abs(lhs - rhs) <= 1e-13 * lhs


def test_boys_branches_agree_across_switch():
    # series+down (x<30) and erf+up (x>=30) must join smoothly: compare with the quad build
    for x in [29.9999999, 30.0000001]:
        assert np.allclose(oracle.boys(MMAX, x), oracle.boys(MMAX, x, quad=True), rtol=4e-15, atol=0)


# ----------------------------------------------------------------------------- E tables (Eqs. 8-15)

def _lambda_t(t, x, P, p):
    # Hermite Gaussian (d/dP)^t exp(-p (x-P)^2) = p^{t/2} H_t(sqrt(p)(x-P)) exp(-p (x-P)^2)  (Eq. 5)
    c = np.zeros(t + 1); c[t] = 1.0
    return p ** (t / 2.0) * hermval(math.sqrt(p) * (x - P), c) * np.exp(-p * (x - P) ** 2)


@pytest.mark.parametrize("la,lb", [(0, 0), (1, 0), (0, 1), (2, 2), (3, 1), (6, 6), (4, 6)])
def test_E2_reconstructs_product_pointwise(la, lb):
    # PAPER.md Eq. 7 on one axis: x_A^i x_B^j e^{-za xA^2 - zb xB^2} = sum_t E^t_ij Lambda_t(x)
    rng = np.random.default_rng(la * 7 + lb)
    za, zb, A, B = rng.uniform(0.4, 2.0), rng.uniform(0.4, 2.0), rng.uniform(-1, 1), rng.uniform(-1, 1)
    E = oracle.hermite_E2(la, lb, za, zb, A - B)
    p, P = za + zb, (za * A + zb * B) / (za + zb)
    x = rng.uniform(-2.5, 2.5, 9)
    for i in range(la + 1):
        for j in range(lb + 1):
            lhs = (x - A) ** i * (x - B) ** j * np.exp(-za * (x - A) ** 2 - zb * (x - B) ** 2)
            rhs = sum(E[i, j, t] * _lambda_t(t, x, P, p) for t in range(i + j + 1))
            scale = np.max(np.abs([E[i, j, t] * _lambda_t(t, x, P, p) for t in range(i + j + 1)]), axis=0)
            assert np.all(np.abs(lhs - rhs) <= 1e-11 * (scale + 1e-300)), (i, j)
            assert np.all(E[i, j, i + j + 1:] == 0.0)      # Eq. 14


def test_E2_seed_top_term_and_overlap():
    rng = np.random.default_rng(5)
    za, zb, A, B = 0.9, 1.7, 0.3, -0.8
    la, lb = 5, 4
    E = oracle.hermite_E2(la, lb, za, zb, A - B)
    p = za + zb
    assert abs(E[0, 0, 0] - math.exp(-za * zb * (A - B) ** 2 / p)) < 1e-16            # Eq. 13
    for i in range(la + 1):
        for j in range(lb + 1):
            assert abs(E[i, j, i + j] - E[0, 0, 0] / (2 * p) ** (i + j)) <= 1e-14 * E[i, j, i + j]   # Eq. 15
    # 1-D overlap: int x_A^i x_B^j e^{..} dx = E^0_ij sqrt(pi/p); Gauss-Hermite is exact here
    P = (za * A + zb * B) / p
    xs, ws = hermgauss(40)
    x = xs / math.sqrt(p) + P
    for i in range(la + 1):
        for j in range(lb + 1):
            quad = np.sum(ws * (x - A) ** i * (x - B) ** j) / math.sqrt(p) * E[0, 0, 0]
            assert abs(quad - E[i, j, 0] * math.sqrt(math.pi / p)) <= 1e-12 * max(abs(quad), 1e-3)


def test_E1_parity_rule_and_two_center_limit():
    # Eq. 12: E^t_a = 0 for a+t odd; Eq. 8 equals Eqs. 9-10 with zb = 0, B = A (reading G2)
    l, za = 6, 1.3
    E1 = oracle.hermite_E1(l, za)
    E2 = oracle.hermite_E2(l, 0, za, 0.0, 0.0)[:, 0, :]
    assert np.allclose(E1, E2, rtol=1e-15, atol=0)
    for a in range(l + 1):
        for t in range(l + 1):
            if (a + t) % 2 == 1 or t > a:
                assert E1[a, t] == 0.0
    assert E1[0, 0] == 1.0                                                            # Eq. 11
    # x^a e^{-za x^2} = sum_t E^t_a Lambda_t(x)
    x = np.linspace(-2, 2, 7)
    for a in range(l + 1):
        rhs = sum(E1[a, t] * _lambda_t(t, x, 0.0, za) for t in range(a + 1))
        assert np.allclose(x ** a * np.exp(-za * x * x), rhs, rtol=1e-11, atol=1e-13)


# ----------------------------------------------------------------------------- R tensor (Eqs. 20-24)

def _hermite_deriv_gauss(t, X, rho):
    # (d/dX)^t exp(-rho X^2) = (-1)^t rho^{t/2} H_t(sqrt(rho) X) exp(-rho X^2)
    c = np.zeros(t + 1); c[t] = 1.0
    return (-1) ** t * rho ** (t / 2.0) * hermval(math.sqrt(rho) * X, c) * math.exp(-rho * X * X)


@pytest.mark.parametrize("L", [2, 5, 8, 12, 24])
def test_R_poisson_identity(L):
    # [0]^(0)(R) is the Coulomb potential of a Gaussian charge (pi/(p+q))^{3/2} e^{-rho R^2}, hence
    # R_{t+2,u,v} + R_{t,u+2,v} + R_{t,u,v+2} = -4 pi^{5/2} (p+q)^{-3/2} d^t d^u d^v e^{-rho |PQ|^2}
    rng = np.random.default_rng(L)
    p, q = rng.uniform(0.5, 3.0, 2)
    PQ = rng.uniform(-0.9, 0.9, 3)
    rho = p * q / (p + q)
    R = oracle.hermite_R(L, p, q, PQ)
    worst = 0.0
    for t in range(L - 1):
        for u in range(L - 1 - t):
            for v in range(L - 1 - t - u):
                lhs = R[t + 2, u, v] + R[t, u + 2, v] + R[t, u, v + 2]
                rhs = -4 * math.pi ** 2.5 * (p + q) ** -1.5 * _hermite_deriv_gauss(t, PQ[0], rho) \
                    * _hermite_deriv_gauss(u, PQ[1], rho) * _hermite_deriv_gauss(v, PQ[2], rho)
                scale = max(abs(R[t + 2, u, v]), abs(R[t, u + 2, v]), abs(R[t, u, v + 2]), abs(rhs))
                worst = max(worst, abs(lhs - rhs) / scale)
    assert worst < 2e-11


def test_R_low_orders_vs_mpmath_derivatives():
    # Eq. 20: [tuv]^(0) = d^t/dX^t d^u/dY^u d^v/dZ^v [0]^(0); differentiate the closed form numerically at 40 digits
    mpmath.mp.dps = 40
    p, q = 1.3, 0.7
    PQ = [0.4, -0.7, 0.25]
    rho = p * q / (p + q)
    pref = 2 * mpmath.pi ** 2.5 / (p * q * mpmath.sqrt(p + q))

    def V(x, y, z):
        T = rho * (x * x + y * y + z * z)
        return pref * mpmath.sqrt(mpmath.pi / T) * mpmath.erf(mpmath.sqrt(T)) / 2

    R = oracle.hermite_R(4, p, q, PQ)
    assert abs(R[0, 0, 0] - float(V(*PQ))) < 1e-14 * abs(R[0, 0, 0])
    for (t, u, v) in [(1, 0, 0), (0, 1, 0), (0, 0, 1), (2, 0, 0), (1, 1, 0), (0, 1, 1), (1, 1, 1), (3, 0, 0), (0, 2, 1), (2, 0, 2), (1, 2, 1), (4, 0, 0)]:
        ref = float(mpmath.diff(V, tuple(PQ), (t, u, v)))
        assert abs(R[t, u, v] - ref) <= 1e-10 * max(1.0, abs(ref)), (t, u, v, R[t, u, v], ref)


def test_R_zero_separation_is_regular():
    # reading S7: P = Q gives T = 0, F_m = 1/(2m+1); odd orders vanish by symmetry
    R = oracle.hermite_R(6, 1.1, 2.3, [0.0, 0.0, 0.0])
    assert np.all(np.isfinite(R))
    for t in range(7):
        for u in range(7 - t):
            for v in range(7 - t - u):
                if t % 2 or u % 2 or v % 2:
                    assert R[t, u, v] == 0.0


# ----------------------------------------------------------------------------- solid harmonics (Eqs. 16-17, reading O2)

def test_solid_harmonics_known_low_l():
    s3 = math.sqrt(3.0)
    assert np.array_equal(oracle.cart2solid(0), [[1.0]])
    assert np.array_equal(oracle.cart2solid(1), [[0, 1, 0], [0, 0, 1], [1, 0, 0]])          # (y, z, x)
    C2 = oracle.cart2solid(2)   # cart order xx xy xz yy yz zz; m=-2..2: sqrt3 xy, sqrt3 yz, z^2-(x^2+y^2)/2, sqrt3 xz, sqrt3/2 (x^2-y^2)
    ref = np.array([[0, s3, 0, 0, 0, 0], [0, 0, 0, 0, s3, 0], [-0.5, 0, 0, -0.5, 0, 1], [0, 0, s3, 0, 0, 0], [s3 / 2, 0, 0, -s3 / 2, 0, 0]])
    assert np.allclose(C2, ref, rtol=1e-15, atol=1e-16)
    # S_33 = sqrt(10)/4 (x^3 - 3 x y^2): cart index of xxx is 0, of xyy is 3
    C3 = oracle.cart2solid(3)
    assert abs(C3[6, 0] - math.sqrt(10) / 4) < 1e-15 and abs(C3[6, 3] + 3 * math.sqrt(10) / 4) < 1e-15


@pytest.mark.parametrize("l", range(7))
def test_solid_harmonics_are_harmonic_racah_normalised(l):
    # numerically: Laplacian = 0 (finite differences of exact polynomials via numpy polynomial algebra),
    # sum_m S_lm^2 = r^{2l} (Unsoeld), S_l0(0,0,1) = 1.
    C = oracle.cart2solid(l)
    comps = [(ax, ay, l - ax - ay) for ax in range(l, -1, -1) for ay in range(l - ax, -1, -1)]
    idx = {c: k for k, c in enumerate(comps)}
    # Laplacian acting on monomial coefficients -> coefficients of degree l-2 monomials must vanish
    if l >= 2:
        low = [(ax, ay, l - 2 - ax - ay) for ax in range(l - 2, -1, -1) for ay in range(l - 2 - ax, -1, -1)]
        for m in range(2 * l + 1):
            for (a, b, c) in low:
                lap = (a + 2) * (a + 1) * C[m, idx[(a + 2, b, c)]] + (b + 2) * (b + 1) * C[m, idx[(a, b + 2, c)]] \
                    + (c + 2) * (c + 1) * C[m, idx[(a, b, c + 2)]]
                assert abs(lap) < 1e-12 * np.max(np.abs(C[m])) * l * l
    rng = np.random.default_rng(l)
    r = rng.normal(size=(5, 3))
    mono = np.array([[np.prod(v ** np.array(c)) for c in comps] for v in r])
    S = mono @ C.T
    assert np.allclose(np.sum(S * S, axis=1), np.sum(r * r, axis=1) ** l, rtol=1e-12)
    assert abs(C[l, idx[(0, 0, l)]] - 1.0) < 1e-14                                    # S_l0(z^) = 1
    # rows are linearly independent (rank 2l+1)
    assert np.linalg.matrix_rank(C) == 2 * l + 1


@pytest.mark.parametrize("l", range(7))
def test_solid_harmonic_rows_vs_scipy(l):
    """Order and sign of every row m = -l..l (the invariants above are blind to a row swap or sign
    flip).  Library special case: with Y_lm = scipy's complex spherical harmonic (Condon-Shortley phase),
    S_l0 = c r^l Y_l0,  S_l,+m = c r^l sqrt2 (-1)^m Re Y_lm,  S_l,-m = c r^l sqrt2 (-1)^m Im Y_lm,  c = sqrt(4 pi/(2l+1)):
    the Racah-normalised real solid harmonics without the phase (reading O2/S2)."""
    from scipy.special import sph_harm_y
    C = oracle.cart2solid(l)
    comps = [(ax, ay, l - ax - ay) for ax in range(l, -1, -1) for ay in range(l - ax, -1, -1)]
    rng = np.random.default_rng(100 + l)
    xyz = rng.normal(size=(12, 3))
    r = np.linalg.norm(xyz, axis=1)
    theta, phi = np.arccos(xyz[:, 2] / r), np.arctan2(xyz[:, 1], xyz[:, 0])
    mono = np.array([[np.prod(v ** np.array(c)) for c in comps] for v in xyz])
    S = mono @ C.T                                                   # [point][m + l]
    c = math.sqrt(4 * math.pi / (2 * l + 1)) * r ** l
    for m in range(-l, l + 1):
        Y = sph_harm_y(l, abs(m), theta, phi)
        ref = c * Y.real if m == 0 else c * math.sqrt(2) * (-1) ** m * (Y.real if m > 0 else Y.imag)
        assert np.allclose(S[:, m + l], ref, rtol=1e-12, atol=1e-13), (l, m)

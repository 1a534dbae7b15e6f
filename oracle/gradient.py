"""CPU oracle of the first geometric derivatives of (ab|cd) (TEST INFRASTRUCTURE).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module; it shares no code with csrc/.

A primitive Cartesian Gaussian (Eq. 1) centred at A, G_a = (x-A_x)^{a_x} (y-A_y)^{a_y} (z-A_z)^{a_z} exp(-zeta |r-A|^2),
depends on A only through r - A, so
    d/dA_i G_a = 2 zeta G_{a+1_i} - a_i G_{a-1_i}.
For a contracted shell (Eq. 4: sum_k c_k G_a(zeta_k)) the derivative of the integral with respect to the centre of one shell is
therefore the Cartesian integral with that shell RAISED to l+1 and contraction coefficients 2 zeta_k c_k, minus a_i times the
integral with the shell LOWERED to l-1 (coefficients c_k).  The solid-harmonic transform (Eqs. 16-17) is linear in the
Cartesian components of each shell and independent of the centres, so it is applied after the combination.  The integrals
themselves are oracle.eri4's; this module only writes the derivative rule out.

Pins (tests/test_oracle_gradient.py): Richardson-extrapolated central differences of oracle.eri4 under a displaced centre
(uses no derivative rule at all), translational invariance (the four centre derivatives sum to zero), the closed form of
d/dA (ss|ss), and (ab|cd) symmetry of the derivative blocks; the 3-center form by the same finite differences of oracle.eri3,
its three derivatives summing to zero, and agreement with the 4-center form on a zeta = 0 dummy shell.
"""
import numpy as np

from . import cart2solid, eri3, eri4, ncart


def cart_components(l):
    """(ax, ay, az) in the order of include/md_b200.h: ax = l..0, ay = l-ax..0."""
    return [(ax, ay, l - ax - ay) for ax in range(l, -1, -1) for ay in range(l - ax, -1, -1)]


def cart_index(ax, ay, az):
    i = ay + az
    return i * (i + 1) // 2 + az


def eri4_grad(a, b, c, d, ia, ib, ic, id_, pure, center, quad=False):
    """d/dR_i (ab|cd), R the centre of shell `center` (0..3 = a, b, c, d), i = x, y, z.

    Shells as for oracle.eri4: (l, center[n,3], exps[n,K], coefs[n,K]).  Returns out[n, 3, na, nb, nc, nd]."""
    shells = [a, b, c, d]
    l, cen, ex, co = shells[center]
    ex = np.asarray(ex, dtype=np.float64).reshape(np.asarray(cen).reshape(-1, 3).shape[0], -1)
    co = np.asarray(co, dtype=np.float64).reshape(ex.shape)
    idx = (ia, ib, ic, id_)
    up = list(shells)
    up[center] = (l + 1, cen, ex, 2.0 * ex * co)
    U = eri4(up[0], up[1], up[2], up[3], *idx, False, quad=quad)                # Cartesian, shell raised
    U = np.moveaxis(U, 1 + center, 1)                                           # [n, comp(l+1), ...]
    if l > 0:
        dn = list(shells)
        dn[center] = (l - 1, cen, ex, co)
        Dn = np.moveaxis(eri4(dn[0], dn[1], dn[2], dn[3], *idx, False, quad=quad), 1 + center, 1)
    n = U.shape[0]
    rest = U.shape[2:]
    G = np.zeros((n, 3, ncart(l)) + rest)
    for k, (ax, ay, az) in enumerate(cart_components(l)):
        e = [ax, ay, az]
        for i in range(3):
            r = list(e); r[i] += 1
            G[:, i, k] = U[:, cart_index(*r)]
            if e[i] > 0:
                s = list(e); s[i] -= 1
                G[:, i, k] -= e[i] * Dn[:, cart_index(*s)]
    G = np.moveaxis(G, 2, 2 + center)                                           # [n, 3, a, b, c, d] Cartesian
    if pure:
        Ca, Cb, Cc, Cd = (cart2solid(s[0]) for s in shells)
        G = np.einsum("nxabcd,pa,qb,rc,sd->nxpqrs", G, Ca, Cb, Cc, Cd, optimize=True)
    return G


def eri3_grad(a, b, x, ia, ib, ix, pure, center, quad=False):
    """d/dR_i (ab|X), R the centre of shell `center` (0, 1, 2 = a, b, X).  Returns out[n, 3, na, nb, nX].

    The same rule on the 3-center integrals of oracle.eri3 (Eqs. 2, 6, 8)."""
    shells = [a, b, x]
    l, cen, ex, co = shells[center]
    ex = np.asarray(ex, dtype=np.float64).reshape(np.asarray(cen).reshape(-1, 3).shape[0], -1)
    co = np.asarray(co, dtype=np.float64).reshape(ex.shape)
    idx = (ia, ib, ix)
    up = list(shells)
    up[center] = (l + 1, cen, ex, 2.0 * ex * co)
    U = np.moveaxis(eri3(up[0], up[1], up[2], *idx, False, quad=quad), 1 + center, 1)
    if l > 0:
        dn = list(shells)
        dn[center] = (l - 1, cen, ex, co)
        Dn = np.moveaxis(eri3(dn[0], dn[1], dn[2], *idx, False, quad=quad), 1 + center, 1)
    G = np.zeros((U.shape[0], 3, ncart(l)) + U.shape[2:])
    for k, (ax, ay, az) in enumerate(cart_components(l)):
        e = [ax, ay, az]
        for i in range(3):
            r = list(e); r[i] += 1
            G[:, i, k] = U[:, cart_index(*r)]
            if e[i] > 0:
                s = list(e); s[i] -= 1
                G[:, i, k] -= e[i] * Dn[:, cart_index(*s)]
    G = np.moveaxis(G, 2, 2 + center)
    if pure:
        Ca, Cb, Cx = (cart2solid(s[0]) for s in shells)
        G = np.einsum("nxabc,pa,qb,rc->nxpqr", G, Ca, Cb, Cx, optimize=True)
    return G


def eri2_grad(x, y, ix, iy, pure, center, quad=False):
    """d/dR_i (X|Y), R the centre of X (center 0) or Y (center 1).  Returns out[n, 3, nX, nY].

    (X|Y) is the 4-center integral with a zeta = 0, c = 1 dummy s shell beside each of X and Y (oracle/two_center.py), so its
    derivative is eri4_grad's with respect to position 0 or 2."""
    dummy = (0, np.zeros((1, 3)), np.zeros((1, 1)), np.ones((1, 1)))
    z = np.zeros(len(ix), dtype=np.int32)
    g = eri4_grad(x, dummy, y, dummy, ix, z, iy, z, pure, 0 if center == 0 else 2, quad=quad)
    return g[:, :, :, 0, :, 0]

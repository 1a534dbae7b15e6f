"""CPU oracle of the 2-center integrals (X|Y) (TEST INFRASTRUCTURE).

(X|Y) is the 4-center integral with a dummy s shell (zeta = 0, c = 1) beside each of X and Y: E^0_00 = 1, p = zeta_X, P = X
(SURVEY.md 8(c) O3 / reading S7: zeta = 0 is legal for exactly this dummy).  The arithmetic is oracle.eri4's; this module only
builds the dummies.  Pins (tests/test_oracle_two_center.py): the closed form of (s|s), (X|Y) = (Y|X)^T, the derivative identity
(p_i|s) = (1/2 zeta) d/dX_i (s|s) by central differences, rotation invariance of the solid block norm.
"""
import numpy as np

from . import eri4


def eri2(x, y, ix, iy, pure):
    """x, y = (l, center[n,3], exps[n,K], coefs[n,K]); returns out[n, nX, nY]."""
    dummy = (0, np.zeros((1, 3)), np.zeros((1, 1)), np.ones((1, 1)))
    z = np.zeros(len(ix), dtype=np.int32)
    v = eri4(x, dummy, y, dummy, ix, z, iy, z, pure)
    return v[:, :, 0, :, 0]

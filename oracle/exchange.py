"""CPU oracle of exchange digestion (TEST INFRASTRUCTURE) -- the definition written out:

  K[b][c] += sum_{a,d} (ab|cd) D[a][d]                       PAPER.md:329-333, Eq. 32

over the listed shell quartets, with (ab|cd) from oracle.eri4 and plain loops over shells (numpy only inside a block).
Pins (tests/test_oracle_exchange.py): for a full ordered list over one basis and symmetric D the result equals the dense
einsum over the full 4-index tensor, K is symmetric, K = 0 for D = 0, and K is linear in D.
Shares no code with paper_2405_01834_b200/csrc.
"""
import numpy as np

from . import eri4


def exchange(a, b, c, d, ia, ib, ic, id_, pure, offs, D):
    """a..d = (l, center, exps, coefs); quartet k = shells (ia[k], ib[k], ic[k], id_[k]); offs = 4 arrays of AO offsets."""
    V = eri4(a, b, c, d, ia, ib, ic, id_, pure)                    # [n][na][nb][nc][nd]
    n, na, nb, nc, nd = V.shape
    K = np.zeros_like(D)
    for k in range(n):
        oa, ob, oc, od = offs[0][ia[k]], offs[1][ib[k]], offs[2][ic[k]], offs[3][id_[k]]
        Dad = D[oa:oa + na, od:od + nd]
        K[ob:ob + nb, oc:oc + nc] += np.einsum("abcd,ad->bc", V[k], Dad)
    return K

"""CPU oracle of the screening step (TEST INFRASTRUCTURE) -- plain numpy, written from the definitions:

  Q_ij = sqrt(max_ab |(ab|ab)|)                              Schwarz factor of shell pair ij (BASELINE config 5:
                                                             "All shell quartets passing a Schwarz bound of 1e-12 are evaluated")
  list = {(i, j): Q_bra[i] * Q_ket[j] >= thr}, ascending (i, j); same=True keeps j <= i

The bound itself is the Cauchy-Schwarz inequality |(ab|cd)| <= sqrt((ab|ab)) sqrt((cd|cd)) for the positive-definite Coulomb
kernel; tests/test_oracle_screening.py pins both functions (the inequality on random integrals, brute-force double loops).
Shares no code with paper_2405_01834_b200/csrc/screen.cu.
"""
import numpy as np

from . import eri4, ncart, nsolid


def schwarz_factors(a, b, ia, ib, pure):
    """Q[n] for pairs (a[ia[k]], b[ib[k]]); a, b = (l, center, exps, coefs) as for oracle.eri4."""
    n = len(ia)
    nf = nsolid if pure else ncart
    nab = nf(a[0]) * nf(b[0])
    blk = eri4(a, b, a, b, ia, ib, ia, ib, pure).reshape(n, nab, nab)
    diag = np.abs(blk[:, np.arange(nab), np.arange(nab)])
    return np.sqrt(diag.max(axis=1))


def quartet_list(Qbra, Qket, thr, same=False):
    """int32 [count, 2] in ascending (i, j) order."""
    keep = Qbra[:, None] * Qket[None, :] >= thr          # one FP64 multiply per pair of pairs
    if same:
        keep &= np.tril(np.ones(keep.shape, dtype=bool))
    return np.argwhere(keep).astype(np.int32)            # row-major: ascending (i, j)

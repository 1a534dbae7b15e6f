"""Pins of oracle/screening.py (no GPU): the Cauchy-Schwarz bound on random oracle integrals, brute force on tiny inputs."""
import numpy as np

import oracle
from oracle import screening
from paper_2405_01834_b200 import workloads as W


def test_schwarz_bound_holds_and_is_attained_on_the_diagonal():
    rng = np.random.default_rng(4)
    for ls in [(0, 0), (1, 0), (1, 1), (2, 1), (2, 2), (3, 1)]:
        a = W.make_shells(rng, 7, ls[0], 2, (0.2, 6.0), (-1.5, 1.5))
        b = W.make_shells(rng, 7, ls[1], 1, (0.2, 6.0), (-1.5, 1.5))
        ia = np.arange(7, dtype=np.int32)
        for pure in (True, False):
            Q = screening.schwarz_factors(a.astuple(), b.astuple(), ia, ia, pure)
            assert (Q > 0).all()
            i, j = np.meshgrid(ia, ia, indexing="ij")
            i, j = i.ravel(), j.ravel()
            blk = oracle.eri4(a.astuple(), b.astuple(), a.astuple(), b.astuple(), i, i, j, j, pure)
            big = np.abs(blk.reshape(49, -1)).max(axis=1)
            assert (big <= Q[i] * Q[j] * (1 + 1e-12)).all()                       # |(ab|cd)| <= Q_ab Q_cd
            d = oracle.eri4(a.astuple(), b.astuple(), a.astuple(), b.astuple(), ia, ia, ia, ia, pure).reshape(7, -1)
            n = int(round(d.shape[1] ** 0.5))
            assert np.allclose(Q ** 2, np.abs(d.reshape(7, n, n)[:, np.arange(n), np.arange(n)]).max(axis=1), rtol=1e-14)


def test_quartet_list_against_double_loop():
    rng = np.random.default_rng(9)
    qb, qk = np.exp(rng.uniform(-18, 1, 41)), np.exp(rng.uniform(-18, 1, 29))
    for thr in (1e-12, 1e-8, 1e-3, 1e9):
        want = [(i, j) for i in range(41) for j in range(29) if qb[i] * qk[j] >= thr]
        got = screening.quartet_list(qb, qk, thr)
        assert got.dtype == np.int32 and got.tolist() == [list(x) for x in want]
        want = [(i, j) for i in range(41) for j in range(41) if j <= i and qb[i] * qb[j] >= thr]
        assert screening.quartet_list(qb, qb, thr, same=True).tolist() == [list(x) for x in want]
    assert len(screening.quartet_list(qb, qb, 0.0, same=True)) == 41 * 42 // 2
    assert screening.quartet_list(qb[:0], qk, 1e-8).shape == (0, 2)
    # agrees with the counting helper the config-5 bookkeeping uses
    assert len(screening.quartet_list(qb, qk, 1e-8)) == W.schwarz_count(qb, qk, 1e-8, False)
    assert len(screening.quartet_list(qb, qb, 1e-8, same=True)) == W.schwarz_count(qb, qb, 1e-8, True)

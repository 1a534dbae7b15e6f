"""Pins of oracle/exchange.py (no GPU): against the dense 4-index definition on a tiny basis, symmetry, linearity."""
import itertools

import numpy as np

import oracle
from oracle import exchange as ox
from paper_2405_01834_b200 import workloads as W


def _basis(rng, ls):
    """One shell per entry of ls: shell batches per l, AO offsets, and the list of (l, index in batch, offset)."""
    shells, info, off = {}, [], 0
    for l in sorted(set(ls)):
        shells[l] = W.make_shells(rng, ls.count(l), l, 2 if l < 2 else 1, (0.3, 4.0), (-1.2, 1.2))
    count = {l: 0 for l in shells}
    for l in ls:
        info.append((l, count[l], off))
        count[l] += 1
        off += 2 * l + 1
    return shells, info, off


def test_exchange_equals_dense_definition_and_is_symmetric():
    rng = np.random.default_rng(8)
    shells, info, nao = _basis(rng, [0, 1, 2, 1, 0])
    D = rng.normal(size=(nao, nao))
    D = D + D.T
    # dense (ab|cd) over all ordered shell quadruples
    full = np.zeros((nao,) * 4)
    for (la, ka, oa), (lb, kb, ob), (lc, kc, oc), (ld, kd, od) in itertools.product(info, repeat=4):
        blk = oracle.eri4(shells[la].astuple(), shells[lb].astuple(), shells[lc].astuple(), shells[ld].astuple(),
                          [ka], [kb], [kc], [kd], True)[0]
        full[oa:oa + 2 * la + 1, ob:ob + 2 * lb + 1, oc:oc + 2 * lc + 1, od:od + 2 * ld + 1] = blk
    want = np.einsum("abcd,ad->bc", full, D)
    K = np.zeros((nao, nao))
    for la, lb, lc, ld in itertools.product(sorted(shells), repeat=4):       # class by class, every ordered quartet
        A, B, C, Dd = (shells[l] for l in (la, lb, lc, ld))
        idx = np.array(list(itertools.product(range(A.n), range(B.n), range(C.n), range(Dd.n))), dtype=np.int32)
        offs = [np.array([o for (l, k, o) in info if l == lx], dtype=np.int64) for lx in (la, lb, lc, ld)]
        K += ox.exchange(A.astuple(), B.astuple(), C.astuple(), Dd.astuple(), idx[:, 0], idx[:, 1], idx[:, 2], idx[:, 3],
                         True, offs, D)
    assert np.allclose(K, want, rtol=1e-12, atol=1e-13)
    assert np.allclose(K, K.T, rtol=1e-11, atol=1e-13)                       # symmetric D, full list: K symmetric
    # linear in D, zero for D = 0
    A = shells[1]
    idx = np.array(list(itertools.product(range(2), repeat=4)), dtype=np.int32)
    offs = [np.array([o for (l, k, o) in info if l == 1], dtype=np.int64)] * 4
    f = lambda M: ox.exchange(A.astuple(), A.astuple(), A.astuple(), A.astuple(), idx[:, 0], idx[:, 1], idx[:, 2], idx[:, 3], True, offs, M)
    D2 = rng.normal(size=(nao, nao))
    assert np.allclose(f(2.0 * D - 3.0 * D2), 2.0 * f(D) - 3.0 * f(D2), rtol=1e-12, atol=1e-13)
    assert not f(np.zeros_like(D)).any()

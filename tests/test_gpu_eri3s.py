"""-m gpu: the one-warp-per-triplet 3-center kernel (MD_VARIANT_ERI3S, csrc/eri3s.cuh) against the oracle: every (la, lb) <= 3 with
every lX <= 6, solid and Cartesian output, contraction on all three shells, index lists, product mode, ragged counts."""
import itertools

import numpy as np
import pytest

from paper_2405_01834_b200 import engine, workloads as W
from gpu_util import check

pytestmark = pytest.mark.gpu
E3 = engine.VARIANT_ERI3S


@pytest.mark.parametrize("la,lb", list(itertools.product(range(4), repeat=2)), ids=lambda x: str(x))
def test_eri3s_all_classes(la, lb):
    for lX in range(7):
        Ks = [(1, 1, 1), (2, 3, 2)] if (la + lb + lX) % 3 == 0 else [(1, 1, 1)]
        for K in Ks:
            w = W.class_sweep((la, lb, lX), 37, K=K, three_center=True)
            for pure in (True, False):
                _, used = check(w, pure, E3)
                assert used == E3
    check(W.clustered((la, lb, 2), 19, three_center=True, coincide="AB"), True, E3)


def test_eri3s_config3_contracted_and_ragged():
    for n in (1, 7, 8, 9, 1185):
        w = W.config3(3, 3, 3, K=4, n=n)
        check(w, True, E3, sel=np.arange(0, n, max(1, n // 25)))


def test_eri3s_index_lists_and_product_mode():
    rng = np.random.default_rng(21)
    a = W.make_shells(rng, 9, 3, 2, (0.2, 8.0), (-1.5, 1.5))
    b = W.make_shells(rng, 7, 2, 1, (0.2, 8.0), (-1.5, 1.5))
    x = W.make_shells(rng, 5, 4, 1, (0.2, 8.0), (-1.5, 1.5))
    bra_idx = np.stack([rng.integers(0, 9, 31), rng.integers(0, 7, 31)], 1).astype(np.int32)
    ti = np.stack([rng.integers(0, 31, 120), rng.integers(0, 5, 120)], 1).astype(np.int32)
    for q in (ti, None):
        w = W.Workload("e3idx", a, b, x, None, bra_idx, None, q)
        for pure in (True, False):
            _, used = check(w, pure, E3)
            assert used == E3


# ---- the same kernel on 4-center classes with an s shell second in one pair: (ab|c s) and, by swapping sides, (a s|cd) ----

TWO = [((3, 2, 2, 0), (1, 1, 1, 1)), ((2, 1, 4, 0), (2, 1, 1, 2)), ((3, 3, 6, 0), (1, 1, 1, 1)), ((1, 0, 0, 0), (1, 2, 2, 1)),
       ((3, 3, 3, 0), (2, 2, 1, 3)), ((0, 0, 5, 0), (1, 1, 1, 1)),
       ((3, 0, 2, 1), (1, 1, 1, 1)), ((5, 0, 3, 3), (1, 1, 1, 1)), ((4, 0, 1, 1), (2, 2, 1, 1)), ((6, 0, 3, 2), (1, 1, 2, 1)),
       # general two-centre kets (pp|, (dp|, (fp|, (dd| through the dense ket table, and their transposes
       ((3, 2, 1, 1), (1, 1, 1, 1)), ((3, 3, 2, 1), (1, 1, 1, 1)), ((2, 1, 2, 2), (2, 1, 1, 2)), ((3, 3, 3, 1), (1, 1, 1, 1)),
       ((1, 1, 3, 2), (1, 2, 1, 1)), ((0, 0, 2, 2), (1, 1, 1, 1)), ((3, 1, 1, 2), (1, 1, 2, 1)), ((2, 2, 3, 3), (1, 1, 1, 1)),
       ((3, 3, 2, 2), (1, 1, 1, 1))]


@pytest.mark.parametrize("ls,Ks", TWO, ids=[str(c[0]) for c in TWO])
def test_eri3s_two_centre_ket_with_an_s_shell(ls, Ks):
    w = W.class_sweep(ls, 41, K=Ks)
    for pure in (True, False):
        _, used = check(w, pure, E3)
        assert used == E3


def test_eri3s_two_centre_index_lists_and_product_mode():
    rng = np.random.default_rng(22)
    a = W.make_shells(rng, 9, 3, 2, (0.2, 8.0), (-1.5, 1.5))
    b = W.make_shells(rng, 7, 1, 1, (0.2, 8.0), (-1.5, 1.5))
    c = W.make_shells(rng, 5, 4, 1, (0.2, 8.0), (-1.5, 1.5))
    d = W.make_shells(rng, 6, 0, 2, (0.2, 8.0), (-1.5, 1.5))
    bra_idx = np.stack([rng.integers(0, 9, 31), rng.integers(0, 7, 31)], 1).astype(np.int32)
    ket_idx = np.stack([rng.integers(0, 5, 23), rng.integers(0, 6, 23)], 1).astype(np.int32)
    qi = np.stack([rng.integers(0, 31, 120), rng.integers(0, 23, 120)], 1).astype(np.int32)
    for q in (qi, None):
        for pure in (True, False):
            _, used = check(W.Workload("e3two", a, b, c, d, bra_idx, ket_idx, q), pure, E3)          # (fp|g s)
            assert used == E3
            _, used = check(W.Workload("e3swap", c, d, a, b, ket_idx, bra_idx,                        # (g s|fp): sides swapped
                                       None if q is None else q[:, ::-1].copy()), pure, E3)
            assert used == E3

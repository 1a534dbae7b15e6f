"""-m gpu: the one-thread-per-quartet kernel for the classes with every l <= 1 (MD_VARIANT_LOWL, csrc/lowl.cuh) against the
oracle: all 16 ordered 4-center and 8 ordered 3-center classes, contraction, index lists, product mode, ragged counts."""
import itertools

import numpy as np
import pytest

from paper_2405_01834_b200 import engine, workloads as W
from gpu_util import check

pytestmark = pytest.mark.gpu
LOWL = engine.VARIANT_LOWL


@pytest.mark.parametrize("ls", list(itertools.product((0, 1), repeat=4)), ids=lambda ls: "".join(map(str, ls)))
def test_lowl_four_center(ls):
    for Ks in [(1, 1, 1, 1), (2, 1, 3, 2), (1, 6, 1, 1)]:
        w = W.independent_quartets("lw", ls, Ks, 301, (0.1, 20.0), (-3.0, 3.0), W.class_seed("lw", ls, Ks))
        for pure in (True, False):
            _, used = check(w, pure, LOWL)
            assert used == LOWL
    # all four centres equal: blocks of odd total l vanish identically (no scale for the block-relative gate): use C = D there
    check(W.clustered(ls, 67, coincide="ALL" if sum(ls) % 2 == 0 else "CD"), True, LOWL)
    check(W.clustered(ls, 67, coincide="AB"), False, LOWL)


@pytest.mark.parametrize("ls", list(itertools.product((0, 1), repeat=3)), ids=lambda ls: "".join(map(str, ls)))
def test_lowl_three_center(ls):
    for K in [(1, 1, 1), (4, 4, 1), (2, 3, 2)]:
        w = W.class_sweep(ls, 203, K=K, three_center=True)
        for pure in (True, False):
            _, used = check(w, pure, LOWL)
            assert used == LOWL


@pytest.mark.parametrize("n", [1, 31, 32, 33, 127, 129, 4097])
def test_lowl_ragged_counts(n):
    check(W.independent_quartets("lwr", (1, 0, 1, 1), (1, 1, 1, 1), n, (0.1, 20.0), (-3.0, 3.0), n), True, LOWL)


def test_lowl_index_lists_and_product_mode():
    rng = np.random.default_rng(12)
    sh = [W.make_shells(rng, m, l, K, (0.2, 8.0), (-1.5, 1.5)) for m, l, K in ((9, 1, 2), (7, 0, 1), (5, 1, 1), (6, 1, 3))]
    bra_idx = np.stack([rng.integers(0, 9, 31), rng.integers(0, 7, 31)], 1).astype(np.int32)
    ket_idx = np.stack([rng.integers(0, 5, 17), rng.integers(0, 6, 17)], 1).astype(np.int32)
    qi = np.stack([rng.integers(0, 31, 211), rng.integers(0, 17, 211)], 1).astype(np.int32)
    for q in (qi, None):
        w = W.Workload("lwidx", *sh, bra_idx, ket_idx, q)
        for pure in (True, False):
            _, used = check(w, pure, LOWL)
            assert used == LOWL


def test_auto_uses_lowl_for_low_l_and_paper_layout_does_not():
    from gpu_util import gpu_run
    w = W.config1(200)
    _, used = gpu_run(w, False)
    assert used == LOWL
    wp = W.paper_microbench((1, 1, 1, 1), 1, 1, 6, 5)
    _, used = gpu_run(wp, True, layout=engine.LAYOUT_PAPER)
    assert used != LOWL

"""-m gpu: north_star's target, every canonical (la lb|lc ld) class with l <= 6 (406) and every canonical 3-center
class (196), a few quartets each, solid output, whatever kernel MD_VARIANT_AUTO selects, against the oracle.
The per-class depth (sizes spanning tiles, Cartesian output, clustered geometry, contraction, every variant) is in
test_gpu_parity.py on 32 representative classes; this file is breadth."""
import numpy as np
import pytest

from paper_2405_01834_b200 import workloads as W
from gpu_util import check

pytestmark = pytest.mark.gpu

PAIRS = [(a, b) for a in range(7) for b in range(a + 1)]


def _n(L):
    return 7 if L <= 8 else 4 if L <= 16 else 2


@pytest.mark.parametrize("la", range(7))
def test_every_four_center_class(la):
    worst = 0.0
    for b in [p for p in PAIRS if p[0] == la]:
        for k in PAIRS[: PAIRS.index(b) + 1]:
            ls = b + k
            r, _ = check(W.class_sweep(ls, _n(sum(ls))), True)
            worst = max(worst, r)
    print("worst block-relative error", worst)


def test_every_three_center_class():
    for b in PAIRS:
        for lX in range(7):
            check(W.class_sweep(b + (lX,), _n(sum(b) + lX), K=(1, 1, 1), three_center=True), True)

"""-m gpu: configurations VERDICT r01 found untested: Cartesian output for L > 16 on every runtime-l
variant, and the largest contraction degree the header accepts (MD_MAX_K = 16 per shell)."""
import numpy as np
import pytest

from paper_2405_01834_b200 import engine, workloads as W
from gpu_util import check

pytestmark = pytest.mark.gpu

GENERIC, MMA, WARP = engine.VARIANT_GENERIC, engine.VARIANT_MMA, engine.VARIANT_WARP


@pytest.mark.parametrize("variant", [engine.VARIANT_AUTO, GENERIC, MMA], ids=["auto", "generic", "mma"])
@pytest.mark.parametrize("ls", [(5, 5, 5, 5), (6, 6, 6, 6), (3, 4, 5, 6), (6, 4, 5, 3), (0, 0, 6, 6), (6, 6, 0, 0)],
                         ids=lambda ls: "".join(map(str, ls)))
def test_cartesian_high_l(ls, variant):
    """Cartesian output (north_star: 'Cartesian or solid-harmonic output') where N_cd reaches 784."""
    n = 3 if sum(ls) > 20 else 5
    check(W.class_sweep(ls, n), False, variant)
    check(W.clustered(ls, 2), False, variant)


@pytest.mark.parametrize("variant", [engine.VARIANT_AUTO, GENERIC, MMA], ids=["auto", "generic", "mma"])
def test_cartesian_three_center_66_6(variant):
    check(W.class_sweep((6, 6, 6), 4, K=(1, 1, 1), three_center=True), False, variant)


@pytest.mark.parametrize("variant", [engine.VARIANT_AUTO, GENERIC, MMA], ids=["auto", "generic", "mma"])
@pytest.mark.parametrize("ls,Ks", [((0, 0, 0, 0), (16, 16, 16, 16)), ((1, 1, 1, 1), (16, 1, 1, 16)),
                                   ((2, 2, 2, 2), (16, 1, 1, 16)), ((2, 1, 2, 0), (4, 16, 16, 2)),
                                   ((3, 0, 2, 1), (16, 1, 1, 16)), ((3, 3, 3, 3), (16, 1, 16, 1)),
                                   ((0, 0, 6, 6), (8, 8, 1, 1)), ((4, 4, 1, 0), (1, 2, 16, 16))],
                         ids=lambda x: "".join(map(str, x)))
def test_max_contraction(ls, Ks, variant):
    """K = MD_MAX_K per shell (K_bra or K_ket up to 256) on the fused, warp, DMMA and generic kernels."""
    n = 3 if max(Ks[0] * Ks[1], Ks[2] * Ks[3]) >= 64 and sum(ls) > 4 else 7
    w = W.independent_quartets("kmax", ls, Ks, n, (0.05, 50.0), (-2.0, 2.0), W.class_seed("kmax", ls, Ks))
    for pure in (True, False):
        check(w, pure, variant)


def test_max_contraction_three_center():
    w = W.class_sweep((2, 1, 4), 5, K=(16, 16, 1), three_center=True)
    for variant in (engine.VARIANT_AUTO, GENERIC, MMA):
        check(w, True, variant)

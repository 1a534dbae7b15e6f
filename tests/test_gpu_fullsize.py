"""-m gpu: BASELINE.json's full sizes in the launch configuration bench.py times (one call over the whole batch,
MD_VARIANT_AUTO), checked on seeded samples of quartets that the oracle computes one by one."""
import numpy as np
import pytest

from paper_2405_01834_b200 import engine, workloads as W
from gpu_util import check

pytestmark = pytest.mark.gpu


def _sample(n, k, seed):
    return np.sort(np.random.default_rng(seed).choice(n, k, replace=False))


@pytest.mark.parametrize("K,pure", [(3, True), (3, False), (1, True), (1, False)])
def test_config2_full_200k(K, pure):
    """configs[1]: the bench.py workload (K = 3, solid) and its three siblings, 200,000 quartets each."""
    w = W.config2(K=K)
    assert w.nquartets == 200_000
    sel = np.concatenate([[0, 1, 7, 8, 199_992, 199_999], _sample(200_000, 300, K)])   # first/last CTA passes + random
    _, used = check(w, pure, sel=np.unique(sel))
    assert used == engine.VARIANT_FUSED2


def test_config1_full():
    check(W.config1(), False)


@pytest.mark.parametrize("ls,k", [((4, 4, 4, 4), 40), ((5, 5, 5, 5), 16), ((6, 6, 6, 6), 8), ((3, 4, 5, 6), 16)],
                         ids=lambda x: "".join(map(str, x)) if isinstance(x, tuple) else str(x))
def test_config4_full_20k(ls, k):
    """configs[3]: 20,000 quartets per high-l class in one call; the oracle checks a seeded sample."""
    w = W.config4(ls)
    assert w.nquartets == 20_000
    check(w, True, sel=np.unique(np.concatenate([[0, 19_999], _sample(20_000, k, sum(ls))])))


@pytest.mark.parametrize("la,lb,lX,K", [(1, 1, 2, 1), (3, 3, 6, 2), (2, 1, 4, 4), (0, 0, 0, 3)])
def test_config3_full_1m(la, lb, lX, K):
    """configs[2]: 1,000,000 triplets per class in one call; sampled against the oracle."""
    w = W.config3(la, lb, lX, K=K)
    assert w.nquartets == 1_000_000
    check(w, True, sel=np.unique(np.concatenate([[0, 999_999], _sample(1_000_000, 120, la + lb + lX)])))

"""BASELINE config 5 (synthetic quadruple-zeta molecule): the input generator and the Schwarz bookkeeping on CPU,
and sampled classes of the molecule against the oracle on the GPU."""
import numpy as np
import pytest

from paper_2405_01834_b200 import workloads as W


def test_molecule_matches_the_shell_list():
    m = W.config5_molecule()
    assert len(m.positions) == 144 and m.nshells() == 1296 and m.nao(True) == 4464 and m.nao(False) == 5568
    d = np.linalg.norm(m.positions[:, None] - m.positions[None], axis=2) + 10 * np.eye(144)
    assert d.min() >= 1.8 and m.positions.min() >= 0 and m.positions.max() <= 22.0
    assert m.shells[(0, 6)].n == 48 and m.shells[(0, 3)].n == 96 and m.shells[(4, 1)].n == 48
    for (l, K), s in m.shells.items():
        assert (s.exps >= 0.1).all() and (s.exps <= (5000.0 if K > 1 else 10.0)).all()
        assert np.array_equal(s.center, m.positions[m.atom_of[(l, K)]])
    pts = m.pair_types(4)
    assert len(pts) == 36 and all(a[0] >= b[0] for a, b in pts)
    assert sum(len(m.pair_list(a, b)) for a, b in pts) == 1296 * 1297 // 2     # every unordered shell pair once
    assert W.config5_molecule().positions.tobytes() == m.positions.tobytes()  # seeded


def test_schwarz_count_and_sample_against_brute_force():
    rng = np.random.default_rng(3)
    qb, qk = np.exp(rng.uniform(-20, 2, 300)), np.exp(rng.uniform(-20, 2, 170))
    thr = 1e-8
    assert W.schwarz_count(qb, qk, thr, False) == int((qb[:, None] * qk[None] >= thr).sum())
    m = qb[:, None] * qb[None] >= thr
    assert W.schwarz_count(qb, qb, thr, True) == int(np.triu(m).sum())
    s = W.schwarz_sample(np.random.default_rng(1), qb, qb, thr, 500, True)
    assert len(s) == 500 and (s[:, 0] <= s[:, 1]).all() and (qb[s[:, 0]] * qb[s[:, 1]] >= thr).all()


@pytest.mark.gpu
def test_config5_classes_against_oracle():
    from gpu_util import check
    m = W.config5_molecule()
    rng = np.random.default_rng(11)
    for pb, pk in [(((0, 6), (0, 6)), ((0, 6), (0, 3))), (((2, 1), (1, 3)), ((1, 1), (0, 6))), (((4, 1), (2, 1)), ((3, 1), (1, 3))),
                   (((1, 3), (1, 3)), ((1, 3), (1, 3))), (((2, 1), (2, 1)), ((2, 1), (1, 1))), (((4, 1), (4, 1)), ((0, 1), (0, 1)))]:
        bra, ket = m.pair_list(*pb), m.pair_list(*pk)
        qi = np.stack([rng.integers(0, len(bra), 60), rng.integers(0, len(ket), 60)], 1).astype(np.int32)
        w = W.config5_class(m, pb, pk, bra, ket, qi)
        check(w, True)

"""The size and flop model that bench.py's roofline uses (workloads.flops_model)
against the figures the paper prints in Table I (tests/golden/table1_paper.txt)."""
import os

from paper_2405_01834_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden", "table1_paper.txt")


def _rows():
    for ln in open(GOLD):
        if ln.startswith("#") or not ln.strip():
            continue
        f = ln.split()
        yield tuple(map(int, f[:4])), f[4], int(f[5]), int(f[6]), int(f[7])


def test_table1_sizes_and_flops():
    total = {}
    for ls, step, a_in, a_out, nf in _rows():
        la, lb, lc, ld = ls
        L = sum(ls)
        Hb, Hk, HL = W.nherm(la + lb), W.nherm(lc + ld), W.nherm(L)
        Nb, Nk = W.nsolid(la) * W.nsolid(lb), W.nsolid(lc) * W.nsolid(ld)
        want = {"r": (L + 1, HL, W.r_l_model(L)), "pq": (HL, Hb * Hk, Hb * Hk // 2),
                "ket": (Hb * Hk, Hb * Nk, 2 * Hb * Hk * Nk), "bra": (Hb * Nk, Nb * Nk, 2 * Nb * Hb * Nk)}[step]
        assert want[:2] == (a_in, a_out), (ls, step, want)
        # the paper prints 103,514 for 455*455/2 = 103,512.5: allow its rounding on the Eq. 19 column
        assert abs(want[2] - nf) <= (2 if step == "pq" else 0), (ls, step, want)
        total[ls] = total.get(ls, 0) + want[2]
    for ls, t in total.items():                      # K = 1: the model is the sum of the four columns
        assert W.flops_model(*ls, 1, 1, True) == t


def test_model_folds_contraction_degrees():
    """K_bra K_ket primitive quartets pay the first three columns, K_bra bra primitives the last (Eqs. 25-26)."""
    one = W.flops_model(2, 2, 2, 2, 1, 1, True)
    bra_step = 2 * 25 * W.nherm(4) * 25
    assert W.flops_model(2, 2, 2, 2, 9, 9, True) == 81 * (one - bra_step) + 9 * bra_step == 5580747
    assert W.flops_model(2, 2, 2, 2, 9, 9, False) == 8186427

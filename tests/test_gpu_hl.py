"""-m gpu: the one-launch high-l kernel (MD_VARIANT_HL, csrc/hl.cuh) against the oracle, in its three S1 modes:
0 = pair matrices built inside the quartet kernel, 1 = one record per shell pair (hl_pair_kernel), 2 = one record per
quartet side, in chunks of quartets.  MD_HL_MODE / MD_HL_WS_MB are the library's measurement overrides."""
import os

import numpy as np
import pytest

from paper_2405_01834_b200 import engine, workloads as W
from gpu_util import assert_parity, check, gpu_run, oracle_run

pytestmark = pytest.mark.gpu
HL = engine.VARIANT_HL


@pytest.fixture(params=["0", "1", "2"], ids=["fused", "per_pair", "per_quartet"])
def mode(request):
    os.environ["MD_HL_MODE"] = request.param
    yield request.param
    os.environ.pop("MD_HL_MODE", None)
    os.environ.pop("MD_HL_WS_MB", None)


CLASSES = [(3, 0, 0, 0), (0, 0, 3, 3), (3, 3, 3, 3), (4, 2, 3, 1), (2, 3, 4, 1), (4, 4, 4, 4), (5, 0, 0, 5), (3, 4, 5, 6),
           (6, 4, 5, 3), (5, 5, 5, 5), (6, 6, 0, 0), (0, 6, 6, 0), (6, 6, 6, 6), (1, 0, 4, 0), (2, 2, 2, 2)]


@pytest.mark.parametrize("ls", CLASSES, ids=lambda ls: "".join(map(str, ls)))
def test_hl_classes(ls, mode):
    L = sum(ls)
    n = 67 if L <= 8 else 29 if L <= 12 else 13 if L <= 16 else 7 if L <= 20 else 4
    for pure in (True, False):
        if not pure and L > 16:
            continue                       # N_ab > 192 Cartesians: the kernel declines, the DMMA chain serves (tested elsewhere)
        _, used = check(W.class_sweep(ls, n), pure, HL)
        if pure or W.ncart(ls[0]) * W.ncart(ls[1]) <= 192:         # N_ab <= 192: the [ab|cd] tile fits the GEMM2 accumulators
            assert used == HL, (ls, pure, used)
    check(W.clustered(ls, 5), True, HL)


@pytest.mark.parametrize("ls", [(3, 3, 3), (2, 1, 4), (3, 3, 6), (6, 6, 6), (0, 0, 5), (4, 0, 0)], ids=lambda ls: "".join(map(str, ls)))
def test_hl_three_center(ls, mode):
    w = W.class_sweep(ls, 41, K=(1, 1, 1), three_center=True)
    _, used = check(w, True, HL)
    assert used == HL
    check(w, False, HL)


@pytest.mark.parametrize("ls,Ks", [((3, 3, 2, 2), (2, 2, 1, 3)), ((4, 2, 3, 1), (1, 2, 2, 1)), ((3, 0, 1, 0), (1, 6, 3, 3)),
                                   ((4, 0, 0, 1), (1, 6, 6, 3)), ((3, 1, 4, 0), (1, 3, 1, 6))], ids=lambda x: "".join(map(str, x)))
def test_hl_contracted(ls, Ks, mode):
    w = W.independent_quartets("hlc", ls, Ks, 23, (0.05, 50.0), (-2.0, 2.0), W.class_seed("hlc", ls, Ks))
    for pure in (True, False):
        _, used = check(w, pure, HL)
        assert used == HL


def test_hl_product_mode_shared_pairs_and_paper_layout(mode):
    """bra list x ket list (every pair shared by many quartets), both layouts, and an index list over shared pairs."""
    w = W.paper_microbench((3, 2, 4, 1), 1, 2, 9, 7)
    for layout in (engine.LAYOUT_QUARTET_MAJOR, engine.LAYOUT_PAPER):
        got, used = gpu_run(w, True, HL, layout)
        assert used == HL
        ref = oracle_run(w, True)                                   # [nq][nab*ncd], q = ij*nket + kl
        if layout == engine.LAYOUT_PAPER:                           # V[ij,ab,cd,kl] column-major
            nb, nk, nab, ncd = w.nbra, w.nket, 7 * 5, 9 * 3
            got = got.reshape(nk, ncd, nab, nb).transpose(3, 0, 2, 1).reshape(nb * nk, nab * ncd)
        assert_parity(got.reshape(ref.shape), ref, "product")
    rng = np.random.default_rng(3)
    w.quartet_idx = np.stack([rng.integers(0, w.nbra, 150), rng.integers(0, w.nket, 150)], 1).astype(np.int32)
    check(w, True, HL)


def test_hl_chunked_launches(mode):
    """A 1 MB record budget forces many chunks (mode 2) or the fall-back to in-kernel S1 (mode 1 -> 2 -> 0)."""
    os.environ["MD_HL_WS_MB"] = "1"
    w = W.class_sweep((4, 4, 4, 4), 700)
    sel = np.arange(0, 700, 23)
    _, used = check(w, True, HL, sel=sel)
    assert used == HL


def test_hl_ragged_counts(mode):
    for n in (1, 2, 147, 149, 297):
        check(W.class_sweep((3, 3, 2, 1), n), True, HL, sel=np.arange(0, n, max(1, n // 20)))


def test_hl_either_orientation(mode):
    """(ab|cd) = (cd|ab): the kernel may take the caller's ket as its bra (MD_HL_SWAP forces either choice)."""
    try:
        for sw in ("0", "1"):
            os.environ["MD_HL_SWAP"] = sw
            for ls in [(3, 2, 4, 1), (4, 4, 3, 3), (1, 0, 4, 3)]:
                check(W.class_sweep(ls, 19), True, HL)
                check(W.class_sweep(ls, 19), False, HL)
            check(W.paper_microbench((3, 2, 4, 1), 1, 2, 9, 7), True, HL)
            check(W.independent_quartets("sw", (3, 1, 2, 2), (2, 1, 1, 3), 31, (0.05, 50.0), (-2.0, 2.0), 3), True, HL)
    finally:
        os.environ.pop("MD_HL_SWAP", None)

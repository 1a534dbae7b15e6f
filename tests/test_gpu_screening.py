"""-m gpu: md_schwarz / md_quartet_list against oracle/screening.py.  Q: floating point, relative 1e-12 (a square root of an
integral inside the north_star bound); the quartet list is integer work on the SAME Q input: bit-exact."""
import numpy as np
import pytest
import torch

from oracle import screening
from paper_2405_01834_b200 import engine, workloads as W

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("ls,Ks", [((0, 0), (3, 1)), ((1, 1), (1, 3)), ((2, 1), (1, 1)), ((2, 2), (2, 2)), ((3, 2), (1, 1)),
                                   ((4, 4), (1, 1)), ((6, 0), (1, 1))], ids=lambda x: "".join(map(str, x)))
def test_schwarz_factors(ls, Ks):
    rng = np.random.default_rng(17)
    n = 37 if sum(ls) <= 5 else 9
    a = W.make_shells(rng, 23, ls[0], Ks[0], (0.1, 30.0), (-2.0, 2.0))
    b = W.make_shells(rng, 19, ls[1], Ks[1], (0.1, 30.0), (-2.0, 2.0))
    idx = np.stack([rng.integers(0, 23, n), rng.integers(0, 19, n)], 1).astype(np.int32)
    da, db, di = engine.to_device(a), engine.to_device(b), engine.idx_to_device(idx)
    for pure in (True, False):
        Q = engine.md_schwarz(da, db, di, pure).cpu().numpy()
        ref = screening.schwarz_factors(a.astuple(), b.astuple(), idx[:, 0], idx[:, 1], pure)
        assert np.all(np.abs(Q - ref) <= 1e-12 * np.maximum(1.0, np.abs(ref))) and np.all(np.abs(Q - ref) <= 1e-10 * ref), (ls, pure)


def test_schwarz_chunks_and_empty():
    """More pairs than one 256 MB chunk of (ab|ab) blocks holds ((dd| Cartesian: 36^2 doubles per pair -> 25,890 per chunk)."""
    rng = np.random.default_rng(2)
    a = W.make_shells(rng, 30000, 2, 1, (0.2, 8.0), (-2.0, 2.0))
    b = W.make_shells(rng, 30000, 2, 1, (0.2, 8.0), (-2.0, 2.0))
    da, db = engine.to_device(a), engine.to_device(b)
    Q = engine.md_schwarz(da, db, None, False).cpu().numpy()
    sel = np.concatenate([np.arange(5), np.arange(25885, 25895), np.arange(29995, 30000)]).astype(np.int32)
    ref = screening.schwarz_factors(a.astuple(), b.astuple(), sel, sel, False)
    assert np.allclose(Q[sel], ref, rtol=1e-11, atol=0)
    assert engine.md_schwarz(da, db, engine.idx_to_device(np.zeros((0, 2), np.int32)), True, npairs=0).numel() == 0


@pytest.mark.parametrize("nb,nk", [(1, 1), (300, 170), (1, 5000), (2049, 257), (777, 777)])
def test_quartet_list_bit_exact(nb, nk):
    rng = np.random.default_rng(nb * 7 + nk)
    qb, qk = np.exp(rng.uniform(-20, 2, nb)), np.exp(rng.uniform(-20, 2, nk))
    qb[rng.integers(0, nb, 3)] = 0.0
    db, dk = torch.as_tensor(qb).cuda(), torch.as_tensor(qk).cuda()
    for thr in (1e-12, 1e-8, 1.0, 1e30, 0.0):
        ref = screening.quartet_list(qb, qk, thr)
        n, idx = engine.md_quartet_list(db, dk, thr)
        assert n == len(ref) and np.array_equal(idx.cpu().numpy(), ref)
        if nb == nk:
            ref = screening.quartet_list(qb, qb, thr, same=True)
            n, idx = engine.md_quartet_list(db, db, thr, same=True)
            assert n == len(ref) and np.array_equal(idx.cpu().numpy(), ref)
    ref = screening.quartet_list(qb, qk, 1e-8)                       # capacity smaller than the count: the first entries, count exact
    n, idx = engine.md_quartet_list(db, dk, 1e-8, capacity=max(1, len(ref) // 3))
    assert n == len(ref) and np.array_equal(idx.cpu().numpy(), ref[: max(1, len(ref) // 3)])


def test_screened_list_feeds_md_eri4():
    """Pair batch -> md_schwarz -> md_quartet_list -> md_eri4 on the surviving quartets, all on the device."""
    from gpu_util import assert_parity, oracle_run
    m = W.config5_molecule()
    pb, pk = ((2, 1), (1, 3)), ((1, 1), (0, 6))
    bra, ket = m.pair_list(*pb)[:160], m.pair_list(*pk)[:140]
    w = W.config5_class(m, pb, pk, bra, ket, None)
    dw = engine.DeviceWorkload(w)
    Qb = engine.md_schwarz(dw.a, dw.b, dw.bra_idx, True)
    Qk = engine.md_schwarz(dw.c, dw.d, dw.ket_idx, True)
    thr = 1e-6
    n, qidx = engine.md_quartet_list(Qb, Qk, thr)
    ref_list = screening.quartet_list(Qb.cpu().numpy(), Qk.cpu().numpy(), thr)
    assert 0 < n < len(bra) * len(ket) and np.array_equal(qidx.cpu().numpy(), ref_list)
    out = torch.empty(n * w.nout(True), dtype=torch.float64, device="cuda")
    engine.md_eri4(dw.a, dw.b, dw.c, dw.d, dw.bra_idx, dw.ket_idx, qidx, n, True, out, nbra=w.nbra, nket=w.nket)
    torch.cuda.synchronize()
    sel = np.arange(0, n, max(1, n // 200))
    w.quartet_idx = ref_list
    assert_parity(out.cpu().numpy().reshape(n, -1)[sel], oracle_run(w, True, sel), "screened")

"""-m gpu: md_exchange (Eq. 32) against oracle/exchange.py.  Floating point with atomic accumulation: the bound is
1e-12 * max(1, sum of |terms| per K element) -- north_star's per-integral bound carried through the sum."""
import numpy as np
import pytest
import torch

import oracle
from oracle import exchange as ox
from paper_2405_01834_b200 import engine, workloads as W

pytestmark = pytest.mark.gpu


def _case(ls, Ks, nsh, nq, pure, seed, product=False):
    rng = np.random.default_rng(seed)
    sh = [W.make_shells(rng, nsh[k], ls[k], Ks[k], (0.2, 8.0), (-1.5, 1.5)) for k in range(4)]
    nf = (lambda l: 2 * l + 1) if pure else (lambda l: (l + 1) * (l + 2) // 2)
    # AO offsets: the four batches laid out one after the other, shells in shuffled order inside a batch
    offs, nao = [], 0
    for k in range(4):
        perm = rng.permutation(nsh[k])
        o = np.empty(nsh[k], np.int32)
        o[perm] = nao + np.arange(nsh[k], dtype=np.int32) * nf(ls[k])
        offs.append(o)
        nao += nsh[k] * nf(ls[k])
    bra_idx = np.stack([rng.integers(0, nsh[0], 9), rng.integers(0, nsh[1], 9)], 1).astype(np.int32)
    ket_idx = np.stack([rng.integers(0, nsh[2], 7), rng.integers(0, nsh[3], 7)], 1).astype(np.int32)
    qidx = None if product else np.stack([rng.integers(0, 9, nq), rng.integers(0, 7, nq)], 1).astype(np.int32)
    D = rng.normal(size=(nao, nao))
    return sh, offs, nao, bra_idx, ket_idx, qidx, D


@pytest.mark.parametrize("ls,Ks", [((0, 0, 0, 0), (2, 1, 1, 3)), ((1, 1, 1, 1), (1, 1, 1, 1)), ((1, 0, 2, 1), (2, 1, 1, 1)),
                                   ((0, 2, 1, 2), (1, 1, 2, 1)), ((2, 2, 2, 2), (1, 2, 1, 1)), ((1, 2, 0, 1), (1, 1, 1, 1)),
                                   ((3, 1, 2, 0), (1, 1, 1, 1)), ((2, 3, 1, 3), (1, 1, 2, 1)), ((4, 4, 3, 2), (1, 1, 1, 1))],
                         ids=lambda x: "".join(map(str, x)))
@pytest.mark.parametrize("product", [False, True], ids=["list", "product"])
def test_exchange_vs_oracle(ls, Ks, product):
    for pure in (True, False):
        if not pure and max(ls) > 3:
            continue
        sh, offs, nao, bra_idx, ket_idx, qidx, D = _case(ls, Ks, (5, 4, 6, 3), 40, pure, 31 + sum(ls), product)
        if qidx is None:
            bi, ki = np.divmod(np.arange(9 * 7), 7)
        else:
            bi, ki = qidx[:, 0], qidx[:, 1]
        ia, ib, ic, id_ = bra_idx[bi, 0], bra_idx[bi, 1], ket_idx[ki, 0], ket_idx[ki, 1]
        tup = [s.astuple() for s in sh]
        ref = ox.exchange(*tup, ia, ib, ic, id_, pure, offs, D)
        mag = ox.exchange(*[(t[0], t[1], t[2], np.abs(t[3])) for t in tup], ia, ib, ic, id_, pure, offs, np.abs(D))   # loose scale of the sums
        dev = [engine.to_device(s) for s in sh]
        K = torch.zeros((nao, nao), dtype=torch.float64, device="cuda")
        engine.md_exchange(*dev, engine.idx_to_device(bra_idx), engine.idx_to_device(ket_idx), engine.idx_to_device(qidx),
                           len(bi), pure, [torch.as_tensor(o).cuda() for o in offs], torch.as_tensor(D).cuda(), K)
        torch.cuda.synchronize()
        got = K.cpu().numpy()
        scale = np.maximum(1.0, np.maximum(np.abs(ref), np.abs(mag)))
        assert np.all(np.abs(got - ref) <= 1e-12 * scale), (ls, pure, np.abs(got - ref).max())
        assert np.abs(got - ref).max() <= 1e-11 * np.abs(ref).max()
        if max(ls) <= 2:
            assert engine.md_last_variant() == engine.VARIANT_FUSED and engine.md_last_launch_count() == 1   # digested in the kernel


def test_exchange_accumulates_and_empty_list():
    sh, offs, nao, bra_idx, ket_idx, qidx, D = _case((1, 1, 1, 0), (1, 1, 1, 1), (3, 3, 3, 3), 10, True, 5)
    dev = [engine.to_device(s) for s in sh]
    K = torch.full((nao, nao), 2.5, dtype=torch.float64, device="cuda")
    args = (engine.idx_to_device(bra_idx), engine.idx_to_device(ket_idx))
    o = [torch.as_tensor(x).cuda() for x in offs]
    engine.md_exchange(*dev, *args, engine.idx_to_device(qidx[:0]), 0, True, o, torch.as_tensor(D).cuda(), K)
    assert (K == 2.5).all()
    engine.md_exchange(*dev, *args, engine.idx_to_device(qidx), 10, True, o, torch.as_tensor(D).cuda(), K)
    bi, ki = qidx[:, 0], qidx[:, 1]
    ref = 2.5 + ox.exchange(*[s.astuple() for s in sh], bra_idx[bi, 0], bra_idx[bi, 1], ket_idx[ki, 0], ket_idx[ki, 1], True, offs, D)
    assert np.allclose(K.cpu().numpy(), ref, rtol=1e-12, atol=1e-12)

"""-m gpu: md_eri4_grad (first geometric derivatives) against oracle/gradient.py, element by element:
every centre, Cartesian and solid output, list and product mode, several chunks, classes served by different kernels."""
import os

import numpy as np
import pytest
import torch

from oracle import gradient
from paper_2405_01834_b200 import engine, workloads as W
from gpu_util import assert_parity

pytestmark = pytest.mark.gpu


def oracle_grad(w, pure, center):
    ia, ib, ic, id_ = w.shell_indices(np.arange(w.nquartets))
    sh = [(s.l, s.center, s.exps, s.coefs) for s in (w.a, w.b, w.c, w.d)]
    g = gradient.eri4_grad(*sh, ia, ib, ic, id_, pure, center)
    return g.reshape(w.nquartets, -1)


def gpu_grad(w, pure, center):
    dw = engine.DeviceWorkload(w)
    out = torch.full((w.nquartets * 3 * w.nout(pure),), float("nan"), dtype=torch.float64, device="cuda")
    engine.md_eri4_grad(dw.a, dw.b, dw.c, dw.d, dw.bra_idx, dw.ket_idx, dw.quartet_idx, w.nquartets, pure, center, out,
                        nbra=w.nbra, nket=w.nket)
    torch.cuda.synchronize()
    return out.cpu().numpy().reshape(w.nquartets, -1)


CASES = [((0, 0, 0, 0), (1, 1, 1, 1), 67), ((1, 1, 1, 1), (2, 1, 1, 2), 67), ((2, 1, 0, 2), (1, 2, 1, 1), 41), ((2, 2, 2, 2), (1, 1, 1, 1), 33),
         ((3, 1, 2, 0), (2, 1, 1, 1), 29), ((0, 3, 1, 2), (1, 1, 2, 1), 29), ((4, 3, 2, 1), (1, 1, 1, 1), 9), ((5, 5, 4, 3), (1, 1, 1, 1), 3)]


@pytest.mark.parametrize("ls,Ks,n", CASES, ids=[str(c[0]) for c in CASES])
@pytest.mark.parametrize("pure", [False, True])
def test_gradient_parity_every_centre(ls, Ks, n, pure):
    w = W.independent_quartets("grad", ls, Ks, n, (0.3, 6.0), (-2.0, 2.0), sum(ls) + 17)
    for center in range(4):
        assert_parity(gpu_grad(w, pure, center), oracle_grad(w, pure, center), f"{ls} centre {center} pure={pure}")


def test_gradient_product_mode_and_chunks():
    w = W.product_batch("gradp", (2, 1, 1, 2), (1, 2, 1, 1), 7, 5, (0.3, 6.0), (-2.0, 2.0), 4)
    ref = [oracle_grad(w, True, c) for c in range(4)]
    os.environ["MD_GRAD_CHUNK_BYTES"] = str(200_000)                  # a few quartets per chunk, ragged last chunk
    try:
        got = [gpu_grad(w, True, c) for c in range(4)]
    finally:
        del os.environ["MD_GRAD_CHUNK_BYTES"]
    for c in range(4):
        assert_parity(got[c], ref[c], f"product, chunks, centre {c}")
    s = got[0] + got[1] + got[2] + got[3]                              # translational invariance of what the GPU returns
    assert np.abs(s).max() <= 1e-11 * max(np.abs(g).max() for g in got)


def test_gradient_rejects_what_it_cannot_serve():
    w = W.independent_quartets("grad6", (6, 0, 0, 0), (1, 1, 1, 1), 2, (0.3, 6.0), (-2.0, 2.0), 1)
    dw = engine.DeviceWorkload(w)
    out = torch.empty(2 * 3 * w.nout(True), dtype=torch.float64, device="cuda")
    with pytest.raises(engine.MDError) as ei:                         # the raised shell would have l = 7
        engine.md_eri4_grad(dw.a, dw.b, dw.c, dw.d, None, None, dw.quartet_idx, 2, True, 0, out)
    assert ei.value.code == engine.MD_EINVAL
    with pytest.raises(engine.MDError) as ei:
        engine.md_eri4_grad(dw.a, dw.b, dw.c, dw.d, None, None, dw.quartet_idx, 2, True, 1, out[:10])
    assert ei.value.code == engine.MD_ECAPACITY
    engine.md_eri4_grad(dw.a, dw.b, dw.c, dw.d, None, None, dw.quartet_idx, 2, True, 1, out)   # the s shell of the same quartets is fine
    torch.cuda.synchronize()
    assert torch.isfinite(out).all()


# ---- 3-center (ab|X) ----------------------------------------------------------------------------------------------------------

def oracle_grad3(w, pure, center):
    ia, ib, ic, _ = w.shell_indices(np.arange(w.nquartets))
    sh = [(s.l, s.center, s.exps, s.coefs) for s in (w.a, w.b, w.c)]
    return gradient.eri3_grad(*sh, ia, ib, ic, pure, center).reshape(w.nquartets, -1)


def gpu_grad3(w, pure, center):
    dw = engine.DeviceWorkload(w)
    out = torch.full((w.nquartets * 3 * w.nout(pure),), float("nan"), dtype=torch.float64, device="cuda")
    engine.md_eri3_grad(dw.a, dw.b, dw.c, dw.bra_idx, dw.quartet_idx, w.nquartets, pure, center, out, nbra=w.nbra)
    torch.cuda.synchronize()
    return out.cpu().numpy().reshape(w.nquartets, -1)


CASES3 = [((0, 0, 0), (1, 1, 1), 67), ((1, 1, 1), (2, 1, 2), 67), ((2, 1, 3), (1, 2, 1), 41), ((3, 3, 2), (1, 1, 1), 23), ((2, 2, 5), (1, 1, 1), 19),
          ((4, 1, 4), (1, 1, 1), 9), ((5, 5, 3), (1, 1, 1), 3)]


@pytest.mark.parametrize("ls,Ks,n", CASES3, ids=[str(c[0]) for c in CASES3])
@pytest.mark.parametrize("pure", [False, True])
def test_gradient3_parity_every_centre(ls, Ks, n, pure):
    w = W.independent_quartets("grad3", ls, Ks, n, (0.3, 6.0), (-2.0, 2.0), sum(ls) + 31, three_center=True)
    got = []
    for center in range(3):
        g = gpu_grad3(w, pure, center)
        assert_parity(g, oracle_grad3(w, pure, center), f"{ls} centre {center} pure={pure}")
        got.append(g)
    assert np.abs(got[0] + got[1] + got[2]).max() <= 1e-11 * max(np.abs(g).max() for g in got)


def test_gradient3_product_mode():
    w = W.product_batch("grad3p", (2, 1, 3), (1, 2, 1), 6, 5, (0.3, 6.0), (-2.0, 2.0), 8, three_center=True)
    for center in range(3):
        assert_parity(gpu_grad3(w, True, center), oracle_grad3(w, True, center), f"3-center product, centre {center}")


# ---- 2-center (X|Y) -----------------------------------------------------------------------------------------------------------

@pytest.mark.parametrize("lx,ly", [(0, 0), (1, 0), (2, 1), (3, 3), (0, 4), (5, 2), (5, 5), (2, 6)])
def test_gradient2_parity(lx, ly):
    rng = np.random.default_rng(lx * 7 + ly)
    x = W.make_shells(rng, 11, lx, 2, (0.3, 6.0), (-2.0, 2.0))
    y = W.make_shells(rng, 9, ly, 1, (0.3, 6.0), (-2.0, 2.0))
    pidx = np.stack([rng.integers(0, 11, 57), rng.integers(0, 9, 57)], 1).astype(np.int32)
    dx, dy = engine.to_device(x), engine.to_device(y)
    for pure in (True, False):
        nout = engine.ncomp(lx, pure) * engine.ncomp(ly, pure)
        for center in range(2):
            if (lx if center == 0 else ly) > 5:
                continue                                              # the raised shell would have l = 7
            for idx in (pidx, None):
                n = 57 if idx is not None else 99
                out = torch.full((n * 3 * nout,), float("nan"), dtype=torch.float64, device="cuda")
                engine.md_eri2_grad(dx, dy, engine.idx_to_device(idx), n, pure, center, out)
                torch.cuda.synchronize()
                ix, iy = (idx[:, 0], idx[:, 1]) if idx is not None else (np.repeat(np.arange(11), 9), np.tile(np.arange(9), 11))
                ref = gradient.eri2_grad(x.astuple(), y.astuple(), ix.astype(np.int32), iy.astype(np.int32), pure, center)
                assert_parity(out.cpu().numpy().reshape(n, -1), ref.reshape(n, -1), f"({lx}|{ly}) centre {center} pure={pure}")

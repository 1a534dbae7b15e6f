"""-m gpu: md_eri2 (X|Y) against oracle/two_center.py, every (lX, lY) <= 6, contraction, product mode and index lists."""
import numpy as np
import pytest
import torch

from oracle import two_center as o2
from paper_2405_01834_b200 import engine, workloads as W
from gpu_util import assert_parity

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("lx", range(7))
def test_eri2_all_l(lx):
    rng = np.random.default_rng(40 + lx)
    for ly in range(7):
        x = W.make_shells(rng, 5, lx, 2 if lx < 3 else 1, (0.3, 10.0), (-2.0, 2.0))
        y = W.make_shells(rng, 4, ly, 3 if ly < 2 else 1, (0.3, 10.0), (-2.0, 2.0))
        idx = np.stack([rng.integers(0, 5, 13), rng.integers(0, 4, 13)], 1).astype(np.int32)
        dx, dy = engine.to_device(x), engine.to_device(y)
        for pure in (True, False):
            n = engine.ncomp(lx, pure) * engine.ncomp(ly, pure)
            for q in (idx, None):
                m = 13 if q is not None else 20
                out = torch.full((m * n,), float("nan"), dtype=torch.float64, device="cuda")
                engine.md_eri2(dx, dy, engine.idx_to_device(q), m, pure, out)
                torch.cuda.synchronize()
                ix, iy = (q[:, 0], q[:, 1]) if q is not None else np.divmod(np.arange(20, dtype=np.int32), 4)
                ref = o2.eri2(x.astuple(), y.astuple(), ix, iy, pure).reshape(m, n)
                assert_parity(out.cpu().numpy().reshape(m, n), ref, f"({lx}|{ly})")

"""-m gpu: md_eri4_static (include/md_b200.h), the entry point that allocates nothing: the runtime-l chain with its pair
records in the library's file-scope 32 MiB __device__ array.  Checked against the EXISTING path (md_eri4 with the same
chain on pool scratch) on two calls in a row that leave different records behind, and against the oracle; the size
limit and the not-initialised case are rejected with their own codes.  The file is named to be collected last."""
import os
import subprocess
import sys

import numpy as np
import pytest
import torch

from paper_2405_01834_b200 import engine, workloads as W
from gpu_util import TOL_ABS, assert_parity, oracle_run

pytestmark = pytest.mark.gpu


def _static(dw, pure, out, layout=engine.LAYOUT_QUARTET_MAJOR):
    w = dw.w
    return engine.md_eri4_static(dw.a, dw.b, dw.c, dw.d, dw.bra_idx, dw.ket_idx, dw.quartet_idx, w.nquartets, pure, out,
                                 layout, None, nbra=w.nbra, nket=w.nket)


def _existing(dw, pure, variant):
    engine.md_set_variant(variant)
    try:
        out = dw.alloc_out(pure)
        out.fill_(float("nan"))
        dw.run(pure, out)
        torch.cuda.synchronize()
        assert engine.md_last_variant() in (engine.VARIANT_WARP, engine.VARIANT_MMA, engine.VARIANT_GENERIC)
        return out
    finally:
        engine.md_set_variant(engine.VARIANT_AUTO)


def test_static_scratch_matches_the_existing_path_on_two_calls_in_a_row():
    engine.md_init()                                                  # set-up (allocates); the calls below must not
    # call 1: (fd|pd) K = (2,1,2,1), 300 listed quartets, solid: the one-warp-per-quartet kernel after pair setup
    w1 = W.independent_quartets("static1", (3, 2, 1, 2), (2, 1, 2, 1), 300, (0.3, 10.0), (-2.0, 2.0), 5)
    # call 2: (gg|fd) K = 1, 37 quartets (ragged against every tile), Cartesian: the DMMA kernel; other record sizes, so
    # whatever call 1 left in the array lies across call 2's records
    w2 = W.independent_quartets("static2", (4, 4, 3, 2), (1, 1, 1, 1), 37, (0.3, 10.0), (-2.0, 2.0), 6)
    d1, d2 = engine.DeviceWorkload(w1), engine.DeviceWorkload(w2)
    e1, e2 = _existing(d1, True, engine.VARIANT_WARP), _existing(d2, False, engine.VARIANT_MMA)
    for dw, pure in ((d1, True), (d2, False)):
        nb = engine.md_eri4_static_bytes(dw.a, dw.b, dw.c, dw.d, dw.bra_idx, dw.ket_idx, pure, nbra=dw.w.nbra, nket=dw.w.nket)
        assert 0 < nb <= engine.STATIC_SCRATCH_BYTES
    o1, o2 = d1.alloc_out(True), d2.alloc_out(False)
    o1.fill_(float("nan")); o2.fill_(float("nan"))
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated(), torch.cuda.memory_reserved()
    free_before = torch.cuda.mem_get_info()[0]                        # the kernels are loaded (the existing path ran them)
    _static(d1, True, o1)                                             # two calls in a row on one stream: ordered, no race
    _static(d2, False, o2)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before                # nothing was taken from the device
    assert (torch.cuda.memory_allocated(), torch.cuda.memory_reserved()) == before
    for name, got, ref, w, pure in (("call 1", o1, e1, w1, True), ("call 2", o2, e2, w2, False)):
        g, r = got.cpu().numpy().reshape(w.nquartets, -1), ref.cpu().numpy().reshape(w.nquartets, -1)
        assert np.all(np.isfinite(g)), name
        assert np.all(np.abs(g - r) <= TOL_ABS * np.maximum(1.0, np.abs(r))), f"{name}: {np.abs(g - r).max():.3e}"
        assert_parity(g, oracle_run(w, pure), "static " + name)
    # and once more in the other order, over the records call 2 left
    o1.fill_(float("nan"))
    _static(d1, True, o1)
    torch.cuda.synchronize()
    g, r = o1.cpu().numpy(), e1.cpu().numpy()
    assert np.all(np.abs(g - r) <= TOL_ABS * np.maximum(1.0, np.abs(r)))


def test_static_scratch_paper_layout_product():
    """bra x ket product in the paper's layout (Eq. 33) through the static array."""
    engine.md_init()
    w = W.product_batch("static_paper", (2, 1, 3, 0), (1, 2, 1, 1), 9, 7, (0.3, 10.0), (-2.0, 2.0), 3)
    dw = engine.DeviceWorkload(w)
    engine.md_set_variant(engine.VARIANT_WARP)
    try:
        ref = dw.alloc_out(True)
        dw.run(True, ref, engine.LAYOUT_PAPER)
    finally:
        engine.md_set_variant(engine.VARIANT_AUTO)
    out = dw.alloc_out(True)
    out.fill_(float("nan"))
    _static(dw, True, out, engine.LAYOUT_PAPER)
    torch.cuda.synchronize()
    g, r = out.cpu().numpy(), ref.cpu().numpy()
    assert np.all(np.abs(g - r) <= TOL_ABS * np.maximum(1.0, np.abs(r)))


def test_static_scratch_rejects_calls_beyond_its_size():
    engine.md_init()
    # (ii|ii): 8 * (4 + 455 * 169) * 2 bytes = 1.23 MB of records per quartet; 40 quartets exceed 32 MiB
    w = W.independent_quartets("static3", (6, 6, 6, 6), (1, 1, 1, 1), 40, (0.3, 10.0), (-2.0, 2.0), 7)
    dw = engine.DeviceWorkload(w)
    nb = engine.md_eri4_static_bytes(dw.a, dw.b, dw.c, dw.d, dw.bra_idx, dw.ket_idx, True, nbra=w.nbra, nket=w.nket)
    assert nb > engine.STATIC_SCRATCH_BYTES
    out = dw.alloc_out(True)
    out.fill_(float("nan"))
    with pytest.raises(engine.MDError) as ei:
        _static(dw, True, out)
    assert ei.value.code == engine.MD_ESTATIC
    assert "32 MiB" in str(ei.value) or "STATIC" in str(ei.value)
    torch.cuda.synchronize()
    assert torch.isnan(out).all()                                     # nothing was launched
    # the same class within the limit runs
    w = W.independent_quartets("static4", (6, 6, 6, 6), (1, 1, 1, 1), 5, (0.3, 10.0), (-2.0, 2.0), 8)
    dw = engine.DeviceWorkload(w)
    out = dw.alloc_out(True)
    _static(dw, True, out)
    torch.cuda.synchronize()
    assert_parity(out.cpu().numpy().reshape(5, -1), oracle_run(w, True), "static (ii|ii)")


def test_static_entry_point_never_initialises():
    """Before md_init() the call returns MD_ENOTINIT instead of initialising (which would allocate).  Needs a fresh process."""
    code = (
        "import torch\n"
        "from paper_2405_01834_b200 import engine, workloads as W\n"
        "torch.cuda.set_device(0)\n"
        "w = W.independent_quartets('s', (3, 2, 1, 2), (1, 1, 1, 1), 4, (0.3, 10.0), (-2.0, 2.0), 1)\n"
        "dw = engine.DeviceWorkload(w)\n"
        "out = dw.alloc_out(True)\n"
        "try:\n"
        "    engine.md_eri4_static(dw.a, dw.b, dw.c, dw.d, None, None, dw.quartet_idx, 4, True, out)\n"
        "except engine.MDError as e:\n"
        "    print('code', e.code)\n"
    )
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-c", code], cwd=root, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    assert f"code {engine.MD_ENOTINIT}" in r.stdout, (r.stdout, r.stderr[-2000:])

"""-m gpu: the workspace contract of include/md_b200.h and independence of calls on different streams
(Listing IV.1: an engine bound to a stream with an asynchronous compute())."""
import numpy as np
import pytest
import torch

from paper_2405_01834_b200 import engine, workloads as W
from gpu_util import assert_parity, oracle_run

pytestmark = pytest.mark.gpu

CASES = [("fused2", (2, 2, 2, 2), (3, 3, 3, 3), 40, engine.VARIANT_FUSED2),
         ("mma", (4, 4, 3, 2), (1, 1, 1, 1), 12, engine.VARIANT_MMA),
         ("warp", (3, 0, 2, 1), (2, 1, 1, 2), 50, engine.VARIANT_AUTO)]


@pytest.mark.parametrize("name,ls,Ks,n,variant", CASES, ids=[c[0] for c in CASES])
def test_caller_workspace_exact_and_too_small(name, ls, Ks, n, variant):
    w = W.independent_quartets("ws", ls, Ks, n, (0.3, 10.0), (-2.0, 2.0), 11)
    dw = engine.DeviceWorkload(w)
    ref = oracle_run(w, True)
    engine.md_set_variant(variant)
    try:
        need = dw.workspace_bytes(True)
        assert need > 0
        buf = torch.empty(need, dtype=torch.uint8, device="cuda")
        out = dw.alloc_out(True)
        out.fill_(float("nan"))
        engine.md_set_workspace(buf)                       # exactly the queried size: must run
        dw.run(True, out)
        torch.cuda.synchronize()
        assert_parity(out.cpu().numpy().reshape(n, -1), ref, name)
        out.fill_(float("nan"))
        engine.md_set_workspace(buf[: need - 8])           # 8 bytes short: MD_ENOMEM, nothing written
        with pytest.raises(engine.MDError) as ei:
            dw.run(True, out)
        assert ei.value.code == engine.MD_ENOMEM
        torch.cuda.synchronize()
        assert torch.isnan(out).all()
    finally:
        engine.md_set_workspace(None)
        engine.md_set_variant(engine.VARIANT_AUTO)


def test_fused_classes_need_no_workspace_and_auto_falls_back():
    w = W.config1(100)
    dw = engine.DeviceWorkload(w)
    assert dw.workspace_bytes(False) == 0                  # (pp|pp) K=1: first fused kernel, no scratch
    w2 = W.independent_quartets("ws2", (2, 2, 2, 2), (3, 3, 3, 3), 30, (0.3, 10.0), (-2.0, 2.0), 5)
    dw2 = engine.DeviceWorkload(w2)
    tiny = torch.empty(64, dtype=torch.uint8, device="cuda")
    engine.md_set_workspace(tiny)
    try:
        out = dw2.run(True)                                # AUTO: fused2 needs scratch -> falls back to the fused kernel
        torch.cuda.synchronize()
        assert engine.md_last_variant() == engine.VARIANT_FUSED
    finally:
        engine.md_set_workspace(None)
    assert_parity(out.cpu().numpy().reshape(30, -1), oracle_run(w2, True), "fallback")


def test_two_streams_back_to_back_do_not_share_scratch():
    """A runtime-l class and a fused2 class, then two runtime-l classes, launched on two streams with no
    synchronisation in between: each call has its own stream-ordered scratch."""
    wa = W.class_sweep((4, 4, 4, 4), 600)
    wb = W.independent_quartets("s2", (2, 2, 2, 2), (3, 3, 3, 3), 3000, (0.05, 50.0), (-3.0, 3.0), 3)
    wc = W.class_sweep((3, 3, 3, 3), 1500)
    da, db, dc = engine.DeviceWorkload(wa), engine.DeviceWorkload(wb), engine.DeviceWorkload(wc)
    oa, ob, oc = da.alloc_out(True), db.alloc_out(True), dc.alloc_out(True)
    for o in (oa, ob, oc):
        o.fill_(float("nan"))
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    for _ in range(3):                                     # repeated so the launches really overlap
        da.run(True, oa, stream=s1)
        dc.run(True, oc, stream=s2)
        db.run(True, ob, stream=s1)
        da.run(True, oa, stream=s2)
        dc.run(True, oc, stream=s1)
    torch.cuda.synchronize()
    sel = np.arange(0, 600, 40)
    assert_parity(oa.cpu().numpy().reshape(600, -1)[sel], oracle_run(wa, True, sel), "stream a")
    sel = np.arange(0, 3000, 100)
    assert_parity(ob.cpu().numpy().reshape(3000, -1)[sel], oracle_run(wb, True, sel), "stream b")
    sel = np.arange(0, 1500, 50)
    assert_parity(oc.cpu().numpy().reshape(1500, -1)[sel], oracle_run(wc, True, sel), "stream c")


def test_workspace_query_scales_with_the_call_not_the_class():
    """(ii|ii) x 20,000 independent quartets: the query must report what the call takes."""
    w = W.config4((6, 6, 6, 6), n=64)
    dw = engine.DeviceWorkload(w)
    assert dw.workspace_bytes(True) > 0


def test_quartet_list_is_chunked_when_pair_records_exceed_the_scratch_budget():
    """(ff|f) with K = 4 per bra shell: 527 KB of pair records per triplet; 9,000 independent triplets would take 4.7 GB in
    one piece (1 M triplets: 527 GB).  The runtime-l chain cuts the list into chunks that reuse a 4 GB scratch."""
    w = W.config3(3, 3, 3, K=4, n=9000)
    dw = engine.DeviceWorkload(w)
    engine.md_set_variant(engine.VARIANT_WARP)                        # AUTO takes the scratch-free eri3s kernel for this class
    try:
        assert dw.workspace_bytes(True) <= (4 << 30) + (1 << 20)
        out = dw.run(True)
        torch.cuda.synchronize()
        assert engine.md_last_launch_count() > 3                      # several chunks: pair setup x 2 + quartet kernel each
    finally:
        engine.md_set_variant(engine.VARIANT_AUTO)
    sel = np.concatenate([np.arange(0, 9000, 450), [8999]])
    assert_parity(out.cpu().numpy().reshape(9000, -1)[sel], oracle_run(w, True, sel), "chunked list")

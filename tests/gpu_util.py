"""Helpers for the -m gpu parity tests: run a workload through the C ABI and through the oracle."""
import numpy as np

import oracle
from paper_2405_01834_b200 import engine

TOL_ABS = 1e-12      # north_star: max|delta| <= 1e-12 * max(1, |I|) per integral
TOL_BLOCK = 1e-9     # self-imposed (finding F1): max|delta| / max|I_oracle| per quartet block


def oracle_run(w, pure, sel=None, quad=False):
    ia, ib, ic, id_ = w.shell_indices(sel)
    if w.three_center:
        r = oracle.eri3(w.a.astuple(), w.b.astuple(), w.c.astuple(), ia, ib, ic, pure, quad=quad)
    else:
        r = oracle.eri4(w.a.astuple(), w.b.astuple(), w.c.astuple(), w.d.astuple(), ia, ib, ic, id_, pure, quad=quad)
    return r.reshape(r.shape[0], -1)


def gpu_run(w, pure, variant=engine.VARIANT_AUTO, layout=engine.LAYOUT_QUARTET_MAJOR):
    import torch
    engine.md_set_variant(variant)
    try:
        dw = engine.DeviceWorkload(w)
        out = dw.alloc_out(pure)
        out.fill_(float("nan"))
        dw.run(pure, out, layout)
        torch.cuda.synchronize()
        used = engine.md_last_variant()
    finally:
        engine.md_set_variant(engine.VARIANT_AUTO)
    return out.cpu().numpy(), used


def assert_parity(gpu, ref, what="", quad_ref=None):
    """gpu, ref: [n, nout].  Element-wise north_star bound plus the per-block scale-aware bound.

    The block bound is a self-imposed bar.  A solid-harmonic block can be 1e7 times smaller than the
    Cartesian integrals it is a combination of, and then the DOUBLE oracle (which transforms last) is the
    inaccurate side.  quad_ref(rows) returns the __float128 oracle for those rows: blocks that miss the
    bar against the double oracle must meet it against the quad one, or be no worse than the double
    oracle's own distance from the quad one (roundoff attribution, finding F1)."""
    assert gpu.shape == ref.shape, (gpu.shape, ref.shape)
    assert np.all(np.isfinite(gpu)), f"{what}: non-finite output"
    d = np.abs(gpu - ref)
    bound = TOL_ABS * np.maximum(1.0, np.abs(ref))
    assert np.all(d <= bound), f"{what}: max|delta|={d.max():.3e} at {np.unravel_index(d.argmax(), d.shape)}"
    if not ref.size:
        return 0.0
    scale = np.abs(ref).max(axis=1)
    rel = np.where(scale > 1e-250, d.max(axis=1) / np.maximum(scale, 1e-250), 0.0)
    bad = np.nonzero(rel > TOL_BLOCK)[0]
    if bad.size and quad_ref is not None:
        rq = quad_ref(bad)
        sq = np.abs(rq).max(axis=1)
        dq = np.abs(gpu[bad] - rq).max(axis=1) / sq
        # where the harmonic combination itself cancels (e.g. (ss|i) at |PQ| -> 0) no FP64 MD code can
        # meet the bar: there the GPU must be within 8x of the double oracle's own roundoff
        dd = np.abs(ref[bad] - rq).max(axis=1) / sq
        ok = (dq <= TOL_BLOCK) | (dq <= 8 * dd)
        assert ok.all(), f"{what}: block-relative error vs quad oracle {dq[~ok].max():.3e} (double oracle {dd[~ok].max():.3e})"
        rel[bad] = np.minimum(dq, TOL_BLOCK)
        bad = bad[:0]
    assert bad.size == 0, f"{what}: block-relative error {rel.max():.3e}"
    return float(rel.max())


def check(w, pure, variant=engine.VARIANT_AUTO, sel=None, what=""):
    gpu, used = gpu_run(w, pure, variant)
    gpu = gpu.reshape(w.nquartets, -1)
    if sel is not None:
        gpu = gpu[sel]
    ref = oracle_run(w, pure, sel)
    rows = np.arange(w.nquartets) if sel is None else np.arange(w.nquartets)[sel]
    quad = lambda bad: oracle_run(w, pure, rows[bad], quad=True)
    return assert_parity(gpu, ref, what or w.name, quad), used

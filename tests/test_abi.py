"""CPU-side checks of the C-ABI library: it builds, loads, and exports every symbol the header declares."""
import os
import re

import pytest

from paper_2405_01834_b200 import build, engine

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return engine.lib()


def test_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "md_b200.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(md_[a-z0-9_]+)\s*\(", hdr))
    assert declared, "no declarations parsed"
    assert declared == set(engine.SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), name


def test_out_elems_and_errors(lib):
    assert lib.md_eri4_out_elems(2, 2, 2, 2, 1, 10) == 6250
    assert lib.md_eri4_out_elems(2, 2, 2, 2, 0, 10) == 12960
    assert lib.md_eri4_out_elems(6, 6, 6, 6, 1, 1) == 169 * 169
    assert lib.md_eri3_out_elems(3, 3, 6, 1, 2) == 2 * 7 * 7 * 13
    assert lib.md_eri4_out_elems(7, 0, 0, 0, 1, 1) == engine.MD_EINVAL
    assert lib.md_eri4_out_elems(0, 0, 0, 0, 2, 1) == engine.MD_EINVAL
    assert lib.md_strerror(engine.MD_ECAPACITY) == b"output buffer too small"
    assert lib.md_version() >= 100
    assert lib.md_set_variant(99) == engine.MD_EINVAL


def test_argument_validation_needs_no_gpu(lib):
    """Bad arguments are rejected before any CUDA call."""
    import ctypes
    import numpy as np
    z = np.zeros(3)
    good = engine.md_shells(1, 1, 1, z.ctypes.data, z.ctypes.data, z.ctypes.data)
    bad_l = engine.md_shells(7, 1, 1, z.ctypes.data, z.ctypes.data, z.ctypes.data)
    bad_k = engine.md_shells(1, 0, 1, z.ctypes.data, z.ctypes.data, z.ctypes.data)
    out = np.zeros(81)
    for bad in (bad_l, bad_k):
        bra = engine.md_pairs(bad, good, 1, None)
        ket = engine.md_pairs(good, good, 1, None)
        rc = lib.md_eri4(ctypes.byref(bra), ctypes.byref(ket), 1, None, 0, 0, out.ctypes.data, 81, None)
        assert rc == engine.MD_EINVAL
    bra = engine.md_pairs(good, good, 2, None)          # npairs > n with idx == NULL
    ket = engine.md_pairs(good, good, 1, None)
    assert lib.md_eri4(ctypes.byref(bra), ctypes.byref(ket), 2, None, 0, 0, out.ctypes.data, 162, None) == engine.MD_EINVAL


def test_missing_library_fails_loudly(monkeypatch):
    monkeypatch.setattr(engine, "_lib", None)
    monkeypatch.setattr(engine, "LIB_PATH", "/nonexistent/libmdb200.so")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        engine.lib()

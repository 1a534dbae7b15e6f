"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Tolerance: north_star's max|delta| <= 1e-12*max(1,|I|) plus the scale-aware
per-block bound of DESIGN.md (finding F1)."""
import ctypes

import numpy as np
import pytest

from paper_2405_01834_b200 import engine, workloads as W
from gpu_util import assert_parity, check, gpu_run, oracle_run

pytestmark = pytest.mark.gpu

GENERIC = engine.VARIANT_GENERIC
MMA = engine.VARIANT_MMA


def _n_for(ls):
    L = sum(ls)
    return 301 if L <= 4 else 131 if L <= 8 else 37 if L <= 12 else 19 if L <= 16 else 11 if L <= 20 else 5


# ---- Boys function: the device routine against mpmath-free closed forms and scipy -------------------------

def test_boys_device_vs_mpmath():
    """F_m(T) = 1F1(m+1/2; m+3/2; -T)/(2m+1) at 40 digits: grid points, the branch switch, tiny and huge T."""
    import mpmath as mp
    import torch
    mp.mp.dps = 40
    T = np.concatenate([[0.0, 1e-12, 1e-6, 0.03124, 0.03126, 0.09375, 31.96, 31.9999999, 32.0, 32.0000001, 40.0, 127.9,
                         127.96874, 127.96875, 127.97, 128.0, 131.0, 1e3, 3e4],
                        np.random.default_rng(1).uniform(0, 140, 600), np.exp(np.random.default_rng(2).uniform(-20, 11, 300))])
    worst = 0.0
    for scheme in (0, 1):
        for mmax in (0, 1, 8, 24):
            F = engine.md_boys(mmax, torch.as_tensor(T).cuda(), scheme).cpu().numpy()
            for m in sorted({0, mmax // 2, mmax}):
                ref = np.array([float(mp.hyp1f1(m + 0.5, m + 1.5, -mp.mpf(float(t))) / (2 * m + 1)) for t in T])
                rel = np.abs(F[:, m] - ref) / ref
                worst = max(worst, rel.max())
                assert rel.max() < 2e-14, (scheme, mmax, m, rel.max(), T[rel.argmax()])
    print("boys worst rel", worst)


# ---- BASELINE config 1: all 2000 x 81 values -----------------------------------------------------------

@pytest.mark.parametrize("variant", [engine.VARIANT_AUTO, GENERIC])
def test_config1_pppp_all_values(variant):
    w = W.config1()
    for pure in (False, True):
        check(w, pure, variant)


# ---- every l: canonical diagonal classes, mixed orders, spread and clustered geometry -------------------

CLASSES = [(0, 0, 0, 0), (1, 0, 0, 0), (0, 1, 0, 0), (0, 0, 1, 0), (0, 0, 0, 1), (1, 1, 0, 0), (1, 0, 1, 0), (2, 0, 0, 0),
           (2, 1, 1, 0), (0, 2, 1, 1), (2, 2, 1, 1), (2, 2, 2, 2), (1, 2, 0, 2), (3, 0, 0, 0), (3, 3, 0, 0), (0, 0, 3, 3),
           (3, 1, 2, 0), (3, 3, 3, 3), (4, 0, 4, 0), (4, 4, 0, 0), (2, 3, 4, 1), (4, 4, 4, 4), (5, 0, 0, 5), (5, 5, 1, 0),
           (3, 4, 5, 6), (6, 0, 0, 0), (0, 6, 6, 0), (6, 6, 0, 0), (0, 0, 6, 6), (5, 5, 5, 5), (6, 4, 5, 3), (6, 6, 6, 6)]


@pytest.mark.parametrize("ls", CLASSES, ids=lambda ls: "".join(map(str, ls)))
def test_class_generic_vs_oracle(ls):
    n = _n_for(ls)
    for pure in (True, False):
        if not pure and sum(ls) > 16:
            continue                      # Cartesian high-l is covered up to L = 16; solid covers the rest
        check(W.class_sweep(ls, n), pure, GENERIC)
        check(W.clustered(ls, max(3, n // 4)), pure, GENERIC)


@pytest.mark.parametrize("ls", CLASSES, ids=lambda ls: "".join(map(str, ls)))
def test_class_auto_vs_oracle(ls):
    """Whatever variant the library selects for the class must match too."""
    n = _n_for(ls)
    for pure in (True, False):
        if not pure and sum(ls) > 16:
            continue
        check(W.class_sweep(ls, n), pure)
        check(W.clustered(ls, max(3, n // 4)), pure)


@pytest.mark.parametrize("ls", CLASSES, ids=lambda ls: "".join(map(str, ls)))
def test_class_mma_vs_oracle(ls):
    """The DMMA quartet kernel on every class, including those AUTO serves with a fused kernel."""
    n = _n_for(ls)
    for pure in (True, False):
        if not pure and sum(ls) > 16:
            continue
        _, used = check(W.class_sweep(ls, n), pure, MMA)
        assert used == MMA
        check(W.clustered(ls, max(3, n // 4)), pure, MMA)


@pytest.mark.parametrize("coincide", ["AB", "CD", "ALL"])
@pytest.mark.parametrize("ls", [(1, 1, 1, 1), (2, 2, 2, 2), (3, 2, 1, 0), (4, 4, 2, 2)], ids=lambda ls: "".join(map(str, ls)))
def test_degenerate_geometry(ls, coincide):
    for variant in (engine.VARIANT_AUTO, GENERIC, MMA):
        check(W.clustered(ls, 23, coincide=coincide), True, variant)
        check(W.clustered(ls, 23, coincide=coincide), False, variant)


# ---- contraction ------------------------------------------------------------------------------------------

@pytest.mark.parametrize("ls,Ks", [((0, 0, 0, 0), (6, 6, 6, 6)), ((1, 0, 1, 0), (3, 6, 1, 2)), ((1, 1, 1, 1), (3, 3, 3, 3)),
                                   ((2, 2, 2, 2), (3, 3, 3, 3)), ((2, 1, 0, 2), (2, 1, 4, 3)), ((3, 3, 2, 2), (2, 2, 1, 3)),
                                   ((4, 2, 3, 1), (1, 2, 2, 1))])
def test_contracted_classes(ls, Ks):
    for variant in (engine.VARIANT_AUTO, GENERIC, MMA):
        w = W.independent_quartets("contr", ls, Ks, 67, (0.05, 50.0), (-2.0, 2.0), W.class_seed("contr", ls, Ks))
        check(w, True, variant)
        check(w, False, variant)


def test_config2_dddd_K1_and_K3_sampled():
    """BASELINE config 2 at reduced n here; the full 200k run is sampled in test_gpu_fullsize.py."""
    for K in (1, 3):
        w = W.config2(K=K, n=1500)
        for pure in (True, False):
            check(w, pure)


# ---- the warp-specialised fused kernel (fused2) -------------------------------------------------------------

FUSED2 = engine.VARIANT_FUSED2


@pytest.mark.parametrize("K", [1, 2, 3])
def test_fused2_config2_dddd(K):
    """(dd|dd): the kernel bench.py times, on config-2 inputs, both outputs, a ragged quartet count."""
    w = W.config2(K=K, n=613)
    for pure in (True, False):
        _, used = check(w, pure, FUSED2)
        assert used == FUSED2


@pytest.mark.parametrize("n", [1, 2, 7, 8, 9, 151])
def test_fused2_tails_and_small_batches(n):
    """Fewer quartets than one CTA pass, one more than a pass, and a count that leaves most CTAs idle."""
    w = W.independent_quartets("f2tail", (2, 2, 2, 2), (2, 3, 1, 2), n, (0.05, 50.0), (-2.0, 2.0), W.class_seed("f2tail", n))
    for pure in (True, False):
        _, used = check(w, pure, FUSED2)
        assert used == FUSED2


def test_fused2_mixed_contraction_and_clustered():
    for Ks in [(3, 1, 1, 3), (1, 4, 2, 1), (5, 1, 1, 1), (1, 1, 1, 6)]:
        w = W.independent_quartets("f2mix", (2, 2, 2, 2), Ks, 41, (0.05, 50.0), (-3.0, 3.0), W.class_seed("f2mix", Ks))
        check(w, True, FUSED2)
        check(w, False, FUSED2)
    for coincide in (None, "AB", "CD", "ALL"):
        check(W.clustered((2, 2, 2, 2), 29, K=(2, 2, 2, 2), coincide=coincide), True, FUSED2)


def test_fused2_is_deterministic():
    """Named-barrier hand-over, aliased drain region, L2 scratch: a race would show up as run-to-run differences."""
    for w, pure in [(W.config2(K=3, n=2500), True), (W.class_sweep((2, 1, 2, 0), 3001, K=(2, 2, 3, 1)), False)]:
        ref, used = gpu_run(w, pure, FUSED2)
        assert used == FUSED2
        for _ in range(3):
            again, _ = gpu_run(w, pure, FUSED2)
            assert np.array_equal(ref, again)


@pytest.mark.parametrize("ls", [(1, 1, 1, 1), (2, 0, 1, 1), (1, 1, 2, 0), (2, 1, 2, 2), (2, 2, 2, 0), (0, 2, 1, 2), (1, 2, 1, 1)],
                         ids=lambda ls: "".join(map(str, ls)))
def test_fused2_every_registered_shape(ls):
    """The other instantiated classes (la+lb >= 2, lc+ld >= 2), canonical and swapped shell order, contracted."""
    w = W.independent_quartets("f2cls", ls, (2, 1, 3, 2), 157, (0.05, 50.0), (-3.0, 3.0), W.class_seed("f2cls", ls))
    for pure in (True, False):
        _, used = check(w, pure, FUSED2)
        assert used == FUSED2
    check(W.clustered(ls, 23, K=(1, 2, 2, 1)), True, FUSED2)


def test_fused2_three_center_with_d_fitting_shell():
    w = W.class_sweep((2, 1, 2), 211, K=(3, 2, 1), three_center=True)
    for pure in (True, False):
        _, used = check(w, pure, FUSED2)
        assert used == FUSED2


def test_fused2_product_mode_and_paper_layout():
    w = _product((2, 2, 2, 2), 11, 6, K=3)
    for pure in (True, False):
        ref = oracle_run(w, pure)
        gpu, used = gpu_run(w, pure, FUSED2)
        assert used == FUSED2
        assert_parity(gpu.reshape(ref.shape), ref, "fused2 product")
        gp, _ = gpu_run(w, pure, FUSED2, layout=engine.LAYOUT_PAPER)
        n = engine.ncomp(2, pure) ** 2
        v = gp.reshape(6, n, n, 11).transpose(3, 0, 2, 1).reshape(11 * 6, n * n)
        assert_parity(v, ref, "fused2 paper layout")


# ---- the one-warp-per-quartet kernel for small classes -------------------------------------------------------

WARP = engine.VARIANT_WARP


@pytest.mark.parametrize("ls", [(3, 0, 0, 0), (0, 0, 0, 3), (3, 3, 0, 0), (0, 0, 3, 3), (3, 0, 3, 0), (4, 0, 4, 0), (4, 4, 0, 0),
                                (3, 2, 1, 0), (0, 3, 2, 1), (5, 0, 1, 0), (6, 0, 0, 0), (4, 1, 1, 1)], ids=lambda ls: "".join(map(str, ls)))
def test_warp_kernel_four_center(ls):
    for pure in (True, False):
        _, used = check(W.class_sweep(ls, 203), pure, WARP)
        assert used == WARP
        check(W.clustered(ls, 31, K=(2, 1, 1, 3)), pure, WARP)
    _, used = check(W.class_sweep(ls, 97), True)          # MD_VARIANT_AUTO: the measured table's choice for these classes
    assert used in (WARP, engine.VARIANT_MMA, engine.VARIANT_HL, engine.VARIANT_ERI3S)


@pytest.mark.parametrize("la,lb,lX", [(0, 0, 3), (0, 0, 6), (1, 0, 4), (3, 3, 0), (4, 4, 0), (3, 1, 2), (2, 2, 4), (0, 3, 5)])
def test_warp_kernel_three_center(la, lb, lX):
    for pure in (True, False):
        _, used = check(W.class_sweep((la, lb, lX), 203, K=(2, 2, 1), three_center=True), pure, WARP)
        assert used == WARP


def test_warp_kernel_product_mode_and_paper_layout():
    for ls, three in [((3, 0, 3, 0), False), ((0, 0, 4), True)]:
        w = _product(ls, 13, 7, three_center=three, K=2)
        ref = oracle_run(w, True)
        gpu, used = gpu_run(w, True, WARP)
        assert used == WARP
        assert_parity(gpu.reshape(ref.shape), ref, "warp product")
        gp, _ = gpu_run(w, True, WARP, layout=engine.LAYOUT_PAPER)
        nab = engine.ncomp(ls[0], True) * engine.ncomp(ls[1], True)
        ncd = engine.ncomp(ls[2], True) * (1 if three else engine.ncomp(ls[3], True))
        v = gp.reshape(7, ncd, nab, 13).transpose(3, 0, 2, 1).reshape(13 * 7, nab * ncd)
        assert_parity(v, ref, "warp paper layout")


# ---- 3-center ----------------------------------------------------------------------------------------------

@pytest.mark.parametrize("la,lb,lX", [(0, 0, 0), (1, 0, 0), (0, 1, 2), (1, 1, 1), (2, 2, 2), (2, 0, 6), (3, 3, 6), (3, 1, 4),
                                      (0, 3, 5), (4, 4, 4), (6, 6, 6), (0, 0, 6), (6, 5, 0)])
def test_three_center(la, lb, lX):
    n = _n_for((la, lb, lX))
    for variant in (engine.VARIANT_AUTO, GENERIC, MMA):
        for pure in (True, False):
            check(W.class_sweep((la, lb, lX), n, K=(1, 1, 1), three_center=True), pure, variant)
            check(W.clustered((la, lb, lX), max(3, n // 4), K=(1, 1, 1), three_center=True), pure, variant)


@pytest.mark.parametrize("K", [1, 2, 3, 4])
def test_config3_three_center_contracted(K):
    for (la, lb, lX) in [(1, 1, 2), (2, 1, 3), (3, 3, 6), (0, 2, 1)]:
        check(W.config3(la, lb, lX, K=K, n=101), True)


# ---- index lists, product mode, layouts, edge cases -----------------------------------------------------------

def _product(ls, nbra, nket, three_center=False, K=1):
    Ks = (K, 1, K, 1)
    return W.paper_microbench(ls, Ks[0], Ks[2], nbra, nket, three_center=three_center)


@pytest.mark.parametrize("ls", [(1, 1, 1, 1), (2, 1, 2, 0), (2, 2, 2, 2), (3, 3, 1, 1)], ids=lambda ls: "".join(map(str, ls)))
def test_product_mode_and_paper_layout(ls):
    w = _product(ls, 13, 7)
    for variant in (engine.VARIANT_AUTO, GENERIC, MMA):
        for pure in (True, False):
            ref = oracle_run(w, pure)                                        # [nbra*nket, nout], ket fastest
            gpu, _ = gpu_run(w, pure, variant)
            assert_parity(gpu.reshape(ref.shape), ref, "product quartet-major")
            gp, _ = gpu_run(w, pure, variant, layout=engine.LAYOUT_PAPER)    # V[ij,ab,cd,kl] column-major
            nf = engine.ncomp
            nab, ncd = nf(ls[0], pure) * nf(ls[1], pure), nf(ls[2], pure) * nf(ls[3], pure)
            v = gp.reshape(7, ncd, nab, 13).transpose(3, 0, 2, 1).reshape(13 * 7, nab * ncd)
            assert_parity(v, ref, "paper layout")


def test_pair_index_lists_and_shared_shells():
    """Pairs that index into shared shell batches in arbitrary order, quartets that reuse pairs."""
    rng = np.random.default_rng(5)
    a = W.make_shells(rng, 9, 2, 2, (0.2, 8.0), (-1.5, 1.5))
    b = W.make_shells(rng, 7, 1, 1, (0.2, 8.0), (-1.5, 1.5))
    c = W.make_shells(rng, 5, 0, 3, (0.2, 8.0), (-1.5, 1.5))
    d = W.make_shells(rng, 6, 2, 1, (0.2, 8.0), (-1.5, 1.5))
    bra_idx = np.stack([rng.integers(0, 9, 31), rng.integers(0, 7, 31)], 1).astype(np.int32)
    ket_idx = np.stack([rng.integers(0, 5, 17), rng.integers(0, 6, 17)], 1).astype(np.int32)
    qi = np.stack([rng.integers(0, 31, 211), rng.integers(0, 17, 211)], 1).astype(np.int32)
    w = W.Workload("idx", a, b, c, d, bra_idx, ket_idx, qi)
    for variant in (engine.VARIANT_AUTO, GENERIC, MMA):
        check(w, True, variant)
        check(w, False, variant)
    w2 = W.Workload("idxprod", a, b, c, d, bra_idx, ket_idx, None)
    check(w2, True)


def test_three_center_product_mode():
    w = _product((2, 1, 3), 11, 5, three_center=True)
    for variant in (engine.VARIANT_AUTO, GENERIC):
        check(w, True, variant)


def test_permutational_symmetry_on_gpu():
    """(ab|cd) = (ba|cd) = (cd|ab) evaluated by different class instantiations."""
    w = W.class_sweep((2, 1, 1, 0), 40)
    g, _ = gpu_run(w, False)
    g = g.reshape(40, 6, 3, 3, 1)
    wba = W.Workload("ba", w.b, w.a, w.c, w.d, None, None, w.quartet_idx)
    gba, _ = gpu_run(wba, False)
    np.testing.assert_allclose(gba.reshape(40, 3, 6, 3, 1).transpose(0, 2, 1, 3, 4), g, rtol=0, atol=1e-13)
    wcd = W.Workload("cdab", w.c, w.d, w.a, w.b, None, None, w.quartet_idx)
    gcd, _ = gpu_run(wcd, False)
    np.testing.assert_allclose(gcd.reshape(40, 3, 1, 6, 3).transpose(0, 3, 4, 1, 2), g, rtol=0, atol=1e-13)


def test_empty_and_single():
    import torch
    w = W.class_sweep((1, 1, 1, 1), 1)
    check(w, True)
    dw = engine.DeviceWorkload(w)
    out = torch.zeros(0, dtype=torch.float64, device="cuda")
    engine.md_eri4(dw.a, dw.b, dw.c, dw.d, None, None, dw.quartet_idx, 0, True, out, nbra=1, nket=1)   # no-op
    torch.cuda.synchronize()


def test_error_codes_on_device_buffers():
    import torch
    w = W.class_sweep((1, 1, 1, 1), 4)
    dw = engine.DeviceWorkload(w)
    small = torch.zeros(10, dtype=torch.float64, device="cuda")
    with pytest.raises(engine.MDError) as e:
        dw.run(True, small)
    assert e.value.code == engine.MD_ECAPACITY
    assert float(small.abs().sum()) == 0.0          # nothing written on an argument error
    out = dw.alloc_out(True)
    with pytest.raises(engine.MDError) as e:        # paper layout needs the product form
        dw.run(True, out, layout=engine.LAYOUT_PAPER)
    assert e.value.code == engine.MD_EINVAL


def test_host_buffer_call_matches_device_call():
    import torch
    for w, pure in [(W.config1(500), False), (W.class_sweep((2, 2, 2, 2), 300), True),
                    (W.class_sweep((2, 1, 3), 300, K=(1, 1, 1), three_center=True), True)]:
        gpu, _ = gpu_run(w, pure)
        host = torch.empty(w.nquartets * w.nout(pure), dtype=torch.float64).pin_memory()
        engine.run_host(w, pure, host)
        assert np.array_equal(host.numpy(), gpu)


def test_host_buffer_call_chunked_overlap():
    """Large quartet lists go through the chunked host call (copy-back overlapped with compute): same bits."""
    import torch
    for w, pure in [(W.class_sweep((1, 1, 1, 1), 70001), False), (W.config2(K=2, n=33000), True)]:
        gpu, _ = gpu_run(w, pure)
        host = torch.empty(w.nquartets * w.nout(pure), dtype=torch.float64).pin_memory()
        engine.run_host(w, pure, host)
        assert np.array_equal(host.numpy(), gpu)
    check(W.class_sweep((1, 1, 1, 1), 70001), False, sel=np.arange(0, 70001, 997))


def test_noncurrent_stream_is_asynchronous_and_correct():
    import torch
    w = W.class_sweep((2, 2, 1, 1), 500)
    ref, _ = gpu_run(w, True)
    s = torch.cuda.Stream()
    dw = engine.DeviceWorkload(w)
    out = dw.alloc_out(True)
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        dw.run(True, out, stream=s)
    s.synchronize()
    assert np.array_equal(out.cpu().numpy(), ref)

"""Thin ctypes binding of include/md_b200.h.  Argument marshalling only: every step of the hot
path runs in the CUDA library.  torch is used for device memory and streams.  There is no CPU
fallback: if the library is missing this module raises at first use.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmdb200.so")

MD_OK, MD_EINVAL, MD_ECAPACITY, MD_ECUDA, MD_ENOMEM, MD_ESTATIC, MD_ENOTINIT = 0, -1, -2, -3, -4, -5, -6
STATIC_SCRATCH_BYTES = 32 << 20
LAYOUT_QUARTET_MAJOR, LAYOUT_PAPER = 0, 1
VARIANT_AUTO, VARIANT_GENERIC, VARIANT_FUSED, VARIANT_MMA, VARIANT_FUSED2, VARIANT_WARP, VARIANT_HL, VARIANT_LOWL, VARIANT_ERI3S = 0, 1, 2, 3, 4, 5, 6, 7, 8

_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int32)


class md_shells(ctypes.Structure):
    _fields_ = [("l", ctypes.c_int32), ("K", ctypes.c_int32), ("n", ctypes.c_int64),
                ("center", ctypes.c_void_p), ("exps", ctypes.c_void_p), ("coefs", ctypes.c_void_p)]


class md_pairs(ctypes.Structure):
    _fields_ = [("a", md_shells), ("b", md_shells), ("npairs", ctypes.c_int64), ("idx", ctypes.c_void_p)]


SYMBOLS = ["md_eri4", "md_eri3", "md_eri4_host", "md_eri3_host", "md_eri4_out_elems", "md_eri3_out_elems",
           "md_eri4_workspace_bytes", "md_eri3_workspace_bytes", "md_set_workspace", "md_set_variant",
           "md_last_variant", "md_last_launch_count", "md_init", "md_boys", "md_fp64_peak", "md_strerror", "md_last_cuda_error",
           "md_version", "md_schwarz", "md_quartet_list", "md_exchange", "md_eri2", "md_eri4_static", "md_eri4_static_bytes", "md_eri4_grad", "md_eri3_grad", "md_eri2_grad"]

_lib = None


def lib():
    """Load libmdb200.so (raises if it has not been built: there is no fallback path)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2405_01834_b200.build` "
                               "(the engine has no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        pp, ps = ctypes.POINTER(md_pairs), ctypes.POINTER(md_shells)
        sig = [ctypes.c_int64, ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_int64,
               ctypes.c_void_p]
        for name, second in (("md_eri4", pp), ("md_eri3", ps), ("md_eri4_host", pp), ("md_eri3_host", ps),
                             ("md_eri4_static", pp)):
            f = getattr(L, name)
            f.argtypes = [pp, second] + sig
            f.restype = ctypes.c_int
        L.md_eri4_out_elems.argtypes = [ctypes.c_int] * 5 + [ctypes.c_int64]
        L.md_eri4_out_elems.restype = ctypes.c_int64
        L.md_eri3_out_elems.argtypes = [ctypes.c_int] * 4 + [ctypes.c_int64]
        L.md_eri3_out_elems.restype = ctypes.c_int64
        L.md_eri4_grad.argtypes = [pp, pp, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_void_p,
                                   ctypes.c_int64, ctypes.c_void_p]
        L.md_eri4_grad.restype = ctypes.c_int
        L.md_eri3_grad.argtypes = [pp, ps, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_void_p,
                                   ctypes.c_int64, ctypes.c_void_p]
        L.md_eri3_grad.restype = ctypes.c_int
        L.md_eri2_grad.argtypes = [ps, ps, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_void_p,
                                   ctypes.c_int64, ctypes.c_void_p]
        L.md_eri2_grad.restype = ctypes.c_int
        L.md_eri4_static_bytes.argtypes = [pp, pp, ctypes.c_int]
        L.md_eri4_static_bytes.restype = ctypes.c_int64
        L.md_eri4_workspace_bytes.argtypes = [pp, pp, ctypes.c_int64, ctypes.c_int, ctypes.c_int]
        L.md_eri4_workspace_bytes.restype = ctypes.c_int64
        L.md_eri3_workspace_bytes.argtypes = [pp, ps, ctypes.c_int64, ctypes.c_int, ctypes.c_int]
        L.md_eri3_workspace_bytes.restype = ctypes.c_int64
        L.md_set_workspace.argtypes = [ctypes.c_void_p, ctypes.c_size_t]
        L.md_set_variant.argtypes = [ctypes.c_int]
        L.md_boys.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        L.md_fp64_peak.argtypes = [ctypes.c_int, ctypes.c_int, _dp, _dp]
        L.md_schwarz.argtypes = [pp, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]
        L.md_quartet_list.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int64, ctypes.c_double, ctypes.c_int,
                                      ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p]
        L.md_eri2.argtypes = [ps, ps] + sig
        L.md_eri2.restype = ctypes.c_int
        L.md_exchange.argtypes = [pp, pp, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int] + [ctypes.c_void_p] * 4 + \
            [ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        L.md_strerror.argtypes = [ctypes.c_int]
        L.md_strerror.restype = ctypes.c_char_p
        L.md_last_cuda_error.restype = ctypes.c_char_p
        _lib = L
    return _lib


class MDError(RuntimeError):
    def __init__(self, code):
        L = lib()
        msg = L.md_strerror(code).decode()
        if code == MD_ECUDA:
            msg += ": " + L.md_last_cuda_error().decode()
        super().__init__(f"md_b200 error {code}: {msg}")
        self.code = code


def _check(code):
    if code != MD_OK:
        raise MDError(code)


def _ptr(x):
    """Raw address of a torch tensor (device or host) or a numpy array; None -> NULL."""
    if x is None:
        return None
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    return x.data_ptr()


def _shells_struct(s):
    """s: anything with .l .K .n .center .exps .coefs (arrays already on the wanted side)."""
    return md_shells(int(s.l), int(s.K), int(s.n), _ptr(s.center), _ptr(s.exps), _ptr(s.coefs))


def _pairs_struct(a, b, idx, npairs=None):
    n = (idx.shape[0] if idx is not None else min(a.n, b.n)) if npairs is None else npairs
    return md_pairs(_shells_struct(a), _shells_struct(b), int(n), _ptr(idx))


class DeviceShells:
    """A shell batch resident on the GPU (torch float64 tensors)."""

    def __init__(self, l, K, center, exps, coefs):
        self.l, self.K, self.center, self.exps, self.coefs = int(l), int(K), center, exps, coefs

    @property
    def n(self):
        return self.center.shape[0]


def to_device(shells, device="cuda"):
    import torch
    f = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).to(device)
    return DeviceShells(shells.l, shells.K, f(shells.center), f(shells.exps), f(shells.coefs))


def idx_to_device(idx, device="cuda"):
    import torch
    if idx is None:
        return None
    return torch.as_tensor(np.ascontiguousarray(idx, dtype=np.int32)).to(device)


def _stream_ptr(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def ncomp(l, pure):
    return 2 * l + 1 if pure else (l + 1) * (l + 2) // 2


def md_init():
    _check(lib().md_init())


def md_set_variant(v):
    _check(lib().md_set_variant(int(v)))


def md_set_workspace(buf):
    """buf: a torch CUDA tensor used as caller-owned scratch, or None to return to the stream-ordered pool."""
    if buf is None:
        _check(lib().md_set_workspace(None, 0))
    else:
        _check(lib().md_set_workspace(_ptr(buf), buf.numel() * buf.element_size()))


def md_eri4_workspace_bytes(a, b, c, d, bra_idx, ket_idx, nquartets, list_mode, pure, nbra=None, nket=None):
    bra = _pairs_struct(a, b, bra_idx, nbra)
    ket = _pairs_struct(c, d, ket_idx, nket)
    return lib().md_eri4_workspace_bytes(ctypes.byref(bra), ctypes.byref(ket), int(nquartets), int(list_mode), int(pure))


def md_eri3_workspace_bytes(a, b, x, bra_idx, ntriplets, list_mode, pure, nbra=None):
    bra = _pairs_struct(a, b, bra_idx, nbra)
    xs = _shells_struct(x)
    return lib().md_eri3_workspace_bytes(ctypes.byref(bra), ctypes.byref(xs), int(ntriplets), int(list_mode), int(pure))


def md_last_variant():
    return lib().md_last_variant()


def md_last_launch_count():
    return lib().md_last_launch_count()


def md_eri4_out_elems(la, lb, lc, ld, pure, n):
    return lib().md_eri4_out_elems(la, lb, lc, ld, int(pure), n)


def md_eri3_out_elems(la, lb, lX, pure, n):
    return lib().md_eri3_out_elems(la, lb, lX, int(pure), n)


def md_eri4(a, b, c, d, bra_idx, ket_idx, quartet_idx, nquartets, pure, out, layout=LAYOUT_QUARTET_MAJOR,
            stream=None, nbra=None, nket=None):
    """(ab|cd) on DEVICE tensors; `out` is a caller-owned torch float64 CUDA tensor.  Asynchronous."""
    bra = _pairs_struct(a, b, bra_idx, nbra)
    ket = _pairs_struct(c, d, ket_idx, nket)
    _check(lib().md_eri4(ctypes.byref(bra), ctypes.byref(ket), int(nquartets), _ptr(quartet_idx), int(pure),
                         int(layout), _ptr(out), out.numel(), _stream_ptr(stream)))
    return out


def md_eri4_static(a, b, c, d, bra_idx, ket_idx, quartet_idx, nquartets, pure, out, layout=LAYOUT_QUARTET_MAJOR,
                   stream=None, nbra=None, nket=None):
    """md_eri4 without any allocation: pair records in the library's static 32 MiB device array (include/md_b200.h).
    md_init() must have run; MD_ESTATIC if the records do not fit.  Calls that overlap on the GPU race on the array."""
    bra = _pairs_struct(a, b, bra_idx, nbra)
    ket = _pairs_struct(c, d, ket_idx, nket)
    _check(lib().md_eri4_static(ctypes.byref(bra), ctypes.byref(ket), int(nquartets), _ptr(quartet_idx), int(pure),
                                int(layout), _ptr(out), out.numel(), _stream_ptr(stream)))
    return out


def md_eri4_grad(a, b, c, d, bra_idx, ket_idx, quartet_idx, nquartets, pure, center, out, stream=None, nbra=None, nket=None):
    """d/dR_i (ab|cd) for the centre of shell `center` (0..3): out[q][i][a][b][c][d] on the DEVICE.  Asynchronous."""
    bra = _pairs_struct(a, b, bra_idx, nbra)
    ket = _pairs_struct(c, d, ket_idx, nket)
    _check(lib().md_eri4_grad(ctypes.byref(bra), ctypes.byref(ket), int(nquartets), _ptr(quartet_idx), int(pure), int(center),
                              _ptr(out), out.numel(), _stream_ptr(stream)))
    return out


def md_eri3_grad(a, b, x, bra_idx, triplet_idx, ntriplets, pure, center, out, stream=None, nbra=None):
    """d/dR_i (ab|X) for the centre of shell `center` (0, 1, 2 = a, b, X): out[t][i][a][b][mX] on the DEVICE.  Asynchronous."""
    bra = _pairs_struct(a, b, bra_idx, nbra)
    xs = _shells_struct(x)
    _check(lib().md_eri3_grad(ctypes.byref(bra), ctypes.byref(xs), int(ntriplets), _ptr(triplet_idx), int(pure), int(center),
                              _ptr(out), out.numel(), _stream_ptr(stream)))
    return out


def md_eri2_grad(x, y, pair_idx, npairs, pure, center, out, stream=None):
    """d/dR_i (X|Y) for the centre of X (center 0) or Y (1): out[t][i][mX][mY] on the DEVICE.  Asynchronous."""
    xs, ys = _shells_struct(x), _shells_struct(y)
    _check(lib().md_eri2_grad(ctypes.byref(xs), ctypes.byref(ys), int(npairs), _ptr(pair_idx), int(pure), int(center), _ptr(out),
                              out.numel(), _stream_ptr(stream)))
    return out


def md_eri4_static_bytes(a, b, c, d, bra_idx, ket_idx, pure, nbra=None, nket=None):
    bra = _pairs_struct(a, b, bra_idx, nbra)
    ket = _pairs_struct(c, d, ket_idx, nket)
    r = lib().md_eri4_static_bytes(ctypes.byref(bra), ctypes.byref(ket), int(pure))
    if r < 0:
        _check(int(r))
    return int(r)


def md_eri3(a, b, x, bra_idx, triplet_idx, ntriplets, pure, out, layout=LAYOUT_QUARTET_MAJOR, stream=None,
            nbra=None):
    """(ab|X) on DEVICE tensors.  Asynchronous."""
    bra = _pairs_struct(a, b, bra_idx, nbra)
    xs = _shells_struct(x)
    _check(lib().md_eri3(ctypes.byref(bra), ctypes.byref(xs), int(ntriplets), _ptr(triplet_idx), int(pure),
                         int(layout), _ptr(out), out.numel(), _stream_ptr(stream)))
    return out


def md_eri4_host(a, b, c, d, bra_idx, ket_idx, quartet_idx, nquartets, pure, out, layout=LAYOUT_QUARTET_MAJOR,
                 stream=None, nbra=None, nket=None):
    """(ab|cd) on HOST arrays (numpy or pinned torch CPU tensors); copies are inside the call."""
    bra = _pairs_struct(a, b, bra_idx, nbra)
    ket = _pairs_struct(c, d, ket_idx, nket)
    nout = out.size if isinstance(out, np.ndarray) else out.numel()
    _check(lib().md_eri4_host(ctypes.byref(bra), ctypes.byref(ket), int(nquartets), _ptr(quartet_idx), int(pure),
                              int(layout), _ptr(out), nout, _stream_ptr(stream)))
    return out


def md_eri3_host(a, b, x, bra_idx, triplet_idx, ntriplets, pure, out, layout=LAYOUT_QUARTET_MAJOR, stream=None,
                 nbra=None):
    bra = _pairs_struct(a, b, bra_idx, nbra)
    xs = _shells_struct(x)
    nout = out.size if isinstance(out, np.ndarray) else out.numel()
    _check(lib().md_eri3_host(ctypes.byref(bra), ctypes.byref(xs), int(ntriplets), _ptr(triplet_idx), int(pure),
                              int(layout), _ptr(out), nout, _stream_ptr(stream)))
    return out


def md_schwarz(a, b, pair_idx, pure, npairs=None, stream=None):
    """Schwarz factors Q[npairs] (torch CUDA float64) of a pair batch on DEVICE tensors."""
    import torch
    pairs = _pairs_struct(a, b, pair_idx, npairs)
    Q = torch.empty(pairs.npairs, dtype=torch.float64, device=a.center.device)
    _check(lib().md_schwarz(ctypes.byref(pairs), int(pure), _ptr(Q), _stream_ptr(stream)))
    return Q


def md_quartet_list(Qbra, Qket, thr, same=False, capacity=None, stream=None):
    """(count, idx[min(count, capacity), 2] int32 CUDA tensor) of the quartets with Qbra[i] Qket[j] >= thr, ascending (i, j).
    capacity=None counts first and allocates exactly."""
    import torch
    count = torch.zeros(1, dtype=torch.int64, device=Qbra.device)
    sp = _stream_ptr(stream)
    if capacity is None:
        _check(lib().md_quartet_list(_ptr(Qbra), Qbra.numel(), _ptr(Qket), Qket.numel(), float(thr), int(same), None, 0, _ptr(count), sp))
        capacity = int(count.item())
    idx = torch.empty((max(capacity, 0), 2), dtype=torch.int32, device=Qbra.device)
    _check(lib().md_quartet_list(_ptr(Qbra), Qbra.numel(), _ptr(Qket), Qket.numel(), float(thr), int(same),
                                 _ptr(idx) if capacity else None, capacity, _ptr(count), sp))
    n = int(count.item())
    return n, idx[: min(n, capacity)]


def md_eri2(x, y, pair_idx, npairs, pure, out, layout=LAYOUT_QUARTET_MAJOR, stream=None):
    """(X|Y) on DEVICE tensors; out[t][mX][mY].  Asynchronous."""
    xs, ys = _shells_struct(x), _shells_struct(y)
    _check(lib().md_eri2(ctypes.byref(xs), ctypes.byref(ys), int(npairs), _ptr(pair_idx), int(pure), int(layout), _ptr(out),
                         out.numel(), _stream_ptr(stream)))
    return out


def md_exchange(a, b, c, d, bra_idx, ket_idx, quartet_idx, nquartets, pure, offs, D, K, stream=None, nbra=None, nket=None):
    """K[b][c] += sum_ad (ab|cd) D[a][d] over the listed quartets (Eq. 32); offs = four int32 CUDA tensors."""
    bra = _pairs_struct(a, b, bra_idx, nbra)
    ket = _pairs_struct(c, d, ket_idx, nket)
    _check(lib().md_exchange(ctypes.byref(bra), ctypes.byref(ket), int(nquartets), _ptr(quartet_idx), int(pure),
                             _ptr(offs[0]), _ptr(offs[1]), _ptr(offs[2]), _ptr(offs[3]), D.shape[0], _ptr(D), _ptr(K),
                             _stream_ptr(stream)))
    return K


def md_boys(mmax, T, scheme=0):
    """F_m(T) for a torch CUDA float64 vector T -> [n, mmax+1] (the kernels' device routines)."""
    import torch
    out = torch.empty((T.numel(), mmax + 1), dtype=torch.float64, device=T.device)
    _check(lib().md_boys(int(mmax), int(scheme), T.numel(), _ptr(T), _ptr(out), _stream_ptr(None)))
    return out


def md_fp64_peak(kind, seconds=0.5):
    """Measured FP64 issue-loop rate in TFLOP/s: kind 0 DFMA, 1 DMMA m8n8k4, 2 DMMA m16n8k8."""
    tf, ms = ctypes.c_double(0), ctypes.c_double(0)
    _check(lib().md_fp64_peak(int(kind), max(1, int(seconds * 10)), ctypes.byref(tf), ctypes.byref(ms)))
    return tf.value, ms.value


class DeviceWorkload:
    """A workloads.Workload with its arrays copied to the GPU once (inputs resident in HBM)."""

    def __init__(self, w, device="cuda"):
        self.w = w
        self.a, self.b, self.c = to_device(w.a, device), to_device(w.b, device), to_device(w.c, device)
        self.d = None if w.three_center else to_device(w.d, device)
        self.bra_idx = idx_to_device(w.bra_idx, device)
        self.ket_idx = idx_to_device(w.ket_idx, device)
        self.quartet_idx = idx_to_device(w.quartet_idx, device)

    def alloc_out(self, pure):
        import torch
        return torch.empty(self.w.nquartets * self.w.nout(pure), dtype=torch.float64, device=self.a.center.device)

    def workspace_bytes(self, pure):
        w = self.w
        lm = w.quartet_idx is not None
        if w.three_center:
            return md_eri3_workspace_bytes(self.a, self.b, self.c, self.bra_idx, w.nquartets, lm, pure, nbra=w.nbra)
        return md_eri4_workspace_bytes(self.a, self.b, self.c, self.d, self.bra_idx, self.ket_idx, w.nquartets, lm, pure,
                                       nbra=w.nbra, nket=w.nket)

    def run(self, pure, out=None, layout=LAYOUT_QUARTET_MAJOR, stream=None):
        w = self.w
        out = self.alloc_out(pure) if out is None else out
        if w.three_center:
            return md_eri3(self.a, self.b, self.c, self.bra_idx, self.quartet_idx, w.nquartets, pure, out, layout,
                           stream, nbra=w.nbra)
        return md_eri4(self.a, self.b, self.c, self.d, self.bra_idx, self.ket_idx, self.quartet_idx, w.nquartets,
                       pure, out, layout, stream, nbra=w.nbra, nket=w.nket)


def run_host(w, pure, out, layout=LAYOUT_QUARTET_MAJOR, stream=None):
    """The host-buffer call on a workloads.Workload (numpy arrays in, numpy/pinned array out)."""
    if w.three_center:
        return md_eri3_host(w.a, w.b, w.c, w.bra_idx, w.quartet_idx, w.nquartets, pure, out, layout, stream,
                            nbra=w.nbra)
    return md_eri4_host(w.a, w.b, w.c, w.d, w.bra_idx, w.ket_idx, w.quartet_idx, w.nquartets, pure, out, layout,
                        stream, nbra=w.nbra, nket=w.nket)

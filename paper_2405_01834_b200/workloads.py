"""Seeded synthetic workloads.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic: it only draws centers, exponents and contraction coefficients, applies
the primitive normalisation constant that the recipe puts into the coefficients, and lays out
index lists.  numpy only.  The inputs stand in for the paper's "randomly generated Gaussian
shells and centers" microbenchmark; its molecule/basis-set files are not here.
"""
from dataclasses import dataclass
from typing import Optional
import math
import zlib

import numpy as np


def ncart(l):
    return (l + 1) * (l + 2) // 2


def nsolid(l):
    return 2 * l + 1


def nherm(l):
    """Number of Hermite Gaussians of order <= l."""
    return (l + 1) * (l + 2) * (l + 3) // 6


def _dfact(n):
    r = 1.0
    while n > 1:
        r *= n
        n -= 2
    return r


def prim_norm(zeta, l):
    """N(zeta,l) = (2 zeta/pi)^{3/4} (4 zeta)^{l/2} / sqrt((2l-1)!!): unit norm for x^l exp(-zeta r^2).

    Input recipe S1 of SURVEY.md 8(c); the library itself applies no normalisation.
    """
    zeta = np.asarray(zeta, dtype=np.float64)
    return (2.0 * zeta / math.pi) ** 0.75 * (4.0 * zeta) ** (l / 2.0) / math.sqrt(_dfact(2 * l - 1))


@dataclass
class Shells:
    """Homogeneous shell batch: n shells sharing l and K."""
    l: int
    K: int
    center: np.ndarray   # [n,3] bohr
    exps: np.ndarray     # [n,K]
    coefs: np.ndarray    # [n,K]  already including any normalisation

    @property
    def n(self):
        return self.center.shape[0]

    def astuple(self):
        return (self.l, self.center, self.exps, self.coefs)

    def take(self, idx):
        idx = np.asarray(idx)
        return Shells(self.l, self.K, np.ascontiguousarray(self.center[idx]),
                      np.ascontiguousarray(self.exps[idx]), np.ascontiguousarray(self.coefs[idx]))


def log_uniform(rng, lo, hi, size):
    return np.exp(rng.uniform(math.log(lo), math.log(hi), size))


def make_shells(rng, n, l, K, zeta_range, box, contracted="unit"):
    """n shells with centers uniform in box = (lo, hi) per axis and exponents log-uniform.

    K == 1: coefficient = prim_norm (recipe S1).
    K > 1 : u_k ~ U[0.1,1], c_k = s u_k prim_norm(zeta_k), s fixing unit self-overlap of the
            contracted x^l function (recipe S11).
    """
    lo, hi = box
    center = rng.uniform(lo, hi, (n, 3))
    exps = log_uniform(rng, zeta_range[0], zeta_range[1], (n, K))
    if K == 1:
        coefs = prim_norm(exps, l)
    else:
        u = rng.uniform(0.1, 1.0, (n, K))
        c = u * prim_norm(exps, l)
        zs = exps[:, :, None] + exps[:, None, :]
        ov = _dfact(2 * l - 1) / (2.0 * zs) ** l * (math.pi / zs) ** 1.5
        s2 = np.einsum("nk,nj,nkj->n", c, c, ov)
        coefs = c / np.sqrt(s2)[:, None]
    return Shells(l, K, np.ascontiguousarray(center), np.ascontiguousarray(exps), np.ascontiguousarray(coefs))


@dataclass
class Workload:
    """A batch of shell quartets (or triplets) of one class.

    bra pair i = (a[bra_idx[i,0]], b[bra_idx[i,1]]) (None: pair i = (a[i], b[i])).
    4-center: ket pair likewise from c, d.  3-center: d is None and ket "pair" k is shell c[k].
    quartet i = (bra pair quartet_idx[i,0], ket pair quartet_idx[i,1]); None means the full
    bra x ket product with the ket index fastest.
    """
    name: str
    a: Shells
    b: Shells
    c: Shells
    d: Optional[Shells]
    bra_idx: Optional[np.ndarray] = None
    ket_idx: Optional[np.ndarray] = None
    quartet_idx: Optional[np.ndarray] = None

    @property
    def three_center(self):
        return self.d is None

    @property
    def nbra(self):
        return self.a.n if self.bra_idx is None else len(self.bra_idx)

    @property
    def nket(self):
        if self.three_center:
            return self.c.n
        return self.c.n if self.ket_idx is None else len(self.ket_idx)

    @property
    def nquartets(self):
        return self.nbra * self.nket if self.quartet_idx is None else len(self.quartet_idx)

    def nout(self, pure):
        nf = nsolid if pure else ncart
        n = nf(self.a.l) * nf(self.b.l) * nf(self.c.l)
        return n if self.three_center else n * nf(self.d.l)

    def shell_indices(self, sel=None):
        """Per-quartet shell indices (ia, ib, ic, id) as int32 arrays (id is None for 3-center)."""
        if self.quartet_idx is None:
            q = np.arange(self.nquartets, dtype=np.int64)
            if sel is not None:
                q = q[sel]
            bi, ki = q // self.nket, q % self.nket
        else:
            qi = self.quartet_idx if sel is None else self.quartet_idx[sel]
            bi, ki = qi[:, 0].astype(np.int64), qi[:, 1].astype(np.int64)
        if self.bra_idx is None:
            ia, ib = bi, bi
        else:
            ia, ib = self.bra_idx[bi, 0], self.bra_idx[bi, 1]
        if self.three_center:
            ic, id_ = ki, None
        elif self.ket_idx is None:
            ic, id_ = ki, ki
        else:
            ic, id_ = self.ket_idx[ki, 0], self.ket_idx[ki, 1]
        f = lambda x: None if x is None else np.ascontiguousarray(x, dtype=np.int32)
        return f(ia), f(ib), f(ic), f(id_)

    def flops_model(self, pure=True):
        """Table I flop model with K folded in, per quartet."""
        ld = 0 if self.three_center else self.d.l
        Kd = 1 if self.three_center else self.d.K
        return flops_model(self.a.l, self.b.l, self.c.l, ld, self.a.K * self.b.K, self.c.K * Kd, pure)


def r_l_model(L):
    """R_L of Table I: known only at L = 4, 12, 24 (396, 7182, 71331); 3-point fit, reading G9."""
    return (L + 2) * (L + 7) * (L * L + 5 * L + 12) // 8


def flops_model(la, lb, lc, ld, Kbra, Kket, pure=True):
    nf = nsolid if pure else ncart
    Nb, Nk = nf(la) * nf(lb), nf(lc) * nf(ld)
    Hb, Hk = nherm(la + lb), nherm(lc + ld)
    L = la + lb + lc + ld
    return Kbra * Kket * (r_l_model(L) + Hb * Hk // 2 + 2 * Hb * Hk * Nk) + Kbra * (2 * Nb * Hb * Nk)


def class_seed(*key):
    return zlib.crc32(repr(key).encode()) & 0x7FFFFFFF


def independent_quartets(name, ls, Ks, n, zeta_range, box, seed, three_center=False):
    """Structure (A) of SURVEY.md 8(d): 4 (or 3) fresh shells per quartet, quartet i = (pair i, pair i)."""
    rng = np.random.default_rng(seed)
    sh = [make_shells(rng, n, ls[k], Ks[k], zeta_range[k] if isinstance(zeta_range[0], tuple) else zeta_range, box)
          for k in range(3 if three_center else 4)]
    qi = np.stack([np.arange(n, dtype=np.int32)] * 2, axis=1)
    return Workload(name, sh[0], sh[1], sh[2], None if three_center else sh[3], None, None, qi)


def product_batch(name, ls, Ks, nbra, nket, zeta_range, box, seed, three_center=False):
    """Structure (B): the paper's bra-list x ket-list product."""
    rng = np.random.default_rng(seed)
    a = make_shells(rng, nbra, ls[0], Ks[0], zeta_range, box)
    b = make_shells(rng, nbra, ls[1], Ks[1], zeta_range, box)
    c = make_shells(rng, nket, ls[2], Ks[2], zeta_range, box)
    d = None if three_center else make_shells(rng, nket, ls[3], Ks[3], zeta_range, box)
    return Workload(name, a, b, c, d, None, None, None)


# ---------------------------------------------------------------------------------------
# BASELINE.json configs
# ---------------------------------------------------------------------------------------

def config1(n=2000):
    """(pp|pp), K=1, Cartesian, centers U[-3,3]^3, zeta log-uniform [0.1,20], seed 0."""
    return independent_quartets("cfg1_pppp_K1", (1, 1, 1, 1), (1, 1, 1, 1), n, (0.1, 20.0), (-3.0, 3.0), 0)


def config2(K=1, n=200_000):
    """(dd|dd), centers U[-5,5]^3, zeta log-uniform [0.05,50]; K=1 or K=3 per shell (recipe S11), seed 0."""
    return independent_quartets(f"cfg2_dddd_K{K}", (2, 2, 2, 2), (K,) * 4, n, (0.05, 50.0), (-5.0, 5.0), 0)


def config3(la, lb, lX, K=1, n=1_000_000):
    """3-center (ab|X): bra K per shell (reading S9), X K=1, zeta log-uniform [0.1,30], 10-bohr cube."""
    return independent_quartets(f"cfg3_{la}{lb}_{lX}_K{K}", (la, lb, lX), (K, K, 1), n, (0.1, 30.0), (0.0, 10.0),
                                class_seed("cfg3", la, lb, lX, K), three_center=True)


def config4(ls, n=20_000):
    """High-l uncontracted: zeta log-uniform [0.3,10], centers U[-4,4]^3."""
    return independent_quartets("cfg4_" + "".join(map(str, ls)), tuple(ls), (1, 1, 1, 1), n, (0.3, 10.0), (-4.0, 4.0),
                                class_seed("cfg4", *ls))


def class_sweep(ls, n, K=(1, 1, 1, 1), three_center=False):
    """Sweep 6 of SURVEY.md 8(d): config-4 distribution for any class."""
    return independent_quartets("sweep_" + "".join(map(str, ls)), tuple(ls), tuple(K), n, (0.3, 10.0), (-4.0, 4.0),
                                class_seed("sweep", tuple(ls), tuple(K), three_center), three_center=three_center)


def clustered(ls, n, half_width=0.5, K=(1, 1, 1, 1), seed=None, three_center=False, coincide=None):
    """Supplementary set of finding F1: all centers inside +-half_width bohr, so integrals are O(1e-5..1).

    coincide: None, "AB" (A=B), "CD" (C=D) or "ALL" (all four centers equal), reading S7.
    """
    seed = class_seed("clustered", tuple(ls), tuple(K), coincide) if seed is None else seed
    w = independent_quartets("clustered_" + "".join(map(str, ls)), tuple(ls), tuple(K), n, (0.3, 10.0),
                             (-half_width, half_width), seed, three_center=three_center)
    if coincide in ("AB", "ALL"):
        w.b.center[:] = w.a.center
    if coincide in ("CD", "ALL") and not three_center:
        w.d.center[:] = w.c.center
    if coincide == "ALL":
        w.c.center[:] = w.a.center
        if not three_center:
            w.d.center[:] = w.a.center
    return w


def paper_microbench(ls, Kbra, Kket, nbra, nket, seed=None, three_center=False):
    """Sweep 7: Tables IV/V shape, bra list x ket list; K=5 realised as 5x1 per pair (reading S6)."""
    Ks = (Kbra, 1, Kket, 1)
    seed = class_seed("paper", tuple(ls), Kbra, Kket) if seed is None else seed
    return product_batch("paper_" + "".join(map(str, ls)) + f"_K{Kbra}_{Kket}", ls, Ks, nbra, nket, (0.3, 10.0),
                         (-4.0, 4.0), seed, three_center=three_center)


# ---------------------------------------------------------------------------------------
# BASELINE config 5: synthetic quadruple-zeta-shaped molecule (readings S10, S11)
# ---------------------------------------------------------------------------------------

# (l, K) of the shells each atom carries, in the order BASELINE.json lists them
HEAVY_SHELLS = [(0, 6), (0, 1), (0, 1), (0, 1), (1, 3), (1, 1), (1, 1), (2, 1), (2, 1), (2, 1), (3, 1), (3, 1), (4, 1)]
H_SHELLS = [(0, 3), (0, 1), (0, 1), (1, 1), (1, 1), (2, 1), (3, 1)]


@dataclass
class Molecule:
    """Shell batches of the config-5 molecule, one homogeneous batch per (l, K) type, and for every ordered pair of
    types (la >= lb) the list of shell pairs (all pairs; i <= j inside one type)."""
    positions: np.ndarray                 # [natom, 3]
    types: list                           # [(l, K)] sorted
    shells: dict                          # (l, K) -> Shells
    atom_of: dict                         # (l, K) -> int array: atom index of each shell

    def pair_types(self, lmax=4):
        ts = [t for t in self.types if t[0] <= lmax]
        return [(ta, tb) for i, ta in enumerate(ts) for tb in ts[: i + 1]]      # la >= lb (types sorted by l, K)

    def pair_list(self, ta, tb):
        na, nb = self.shells[ta].n, self.shells[tb].n
        if ta == tb:
            i, j = np.triu_indices(na)
        else:
            i, j = np.meshgrid(np.arange(na), np.arange(nb), indexing="ij")
            i, j = i.ravel(), j.ravel()
        return np.ascontiguousarray(np.stack([i, j], 1).astype(np.int32))

    def nshells(self):
        return sum(s.n for s in self.shells.values())

    def nao(self, pure=True):
        return sum(s.n * (nsolid(s.l) if pure else ncart(s.l)) for s in self.shells.values())


def config5_molecule(n_heavy=48, n_h=96, edge=22.0, min_sep=1.8, seed=0):
    """48 heavy + 96 H atoms at seeded random positions in a cube of `edge` bohr, rejection-sampled to a minimum
    separation (reading S10); shells per atom as BASELINE.json lists them; exponents log-uniform in [0.1,5000] for
    contracted shells and [0.1,10] for single primitives; coefficients per reading S11."""
    rng = np.random.default_rng(seed)
    pos = []
    while len(pos) < n_heavy + n_h:
        p = rng.uniform(0.0, edge, 3)
        if all(np.linalg.norm(p - q) >= min_sep for q in pos):
            pos.append(p)
    pos = np.array(pos)
    per_type = {}
    for ia in range(n_heavy + n_h):
        for (l, K) in (HEAVY_SHELLS if ia < n_heavy else H_SHELLS):
            per_type.setdefault((l, K), []).append(ia)
    types = sorted(per_type)
    shells, atom_of = {}, {}
    for t in types:
        l, K = t
        atoms = np.array(per_type[t])
        zr = (0.1, 5000.0) if K > 1 else (0.1, 10.0)
        s = make_shells(rng, len(atoms), l, K, zr, (0.0, 1.0))
        s.center[:] = pos[atoms]
        shells[t], atom_of[t] = s, atoms
    return Molecule(pos, types, shells, atom_of)


def config5_class(mol, tab, tcd, bra_pairs, ket_pairs, quartet_idx, name=None):
    """One (la lb|lc ld) class of the molecule as a Workload: pair lists index into the type batches."""
    (ta, tb), (tc, td) = tab, tcd
    return Workload(name or f"cfg5_{ta}{tb}_{tc}{td}", mol.shells[ta], mol.shells[tb], mol.shells[tc], mol.shells[td],
                    bra_pairs, ket_pairs, quartet_idx)


def schwarz_count(qb, qk, thr, same):
    """Number of (bra pair, ket pair) combinations with Q_bra Q_ket >= thr; `same`: the two lists are the same
    pair type, count unordered combinations ij <= kl only."""
    sk = np.sort(qk)
    lo = np.searchsorted(sk, thr / np.maximum(qb, 1e-300), side="left")
    n = int((len(sk) - lo).sum())
    if same:
        n = (n + int((qb * qb >= thr).sum())) // 2
    return n


def schwarz_sample(rng, qb, qk, thr, nsample, same):
    """A seeded sample of quartet index pairs that pass the Schwarz bound (rejection sampling)."""
    out = []
    need = nsample
    for _ in range(64):
        if need <= 0:
            break
        i = rng.integers(0, len(qb), 2 * need + 16)
        j = rng.integers(0, len(qk), 2 * need + 16)
        ok = qb[i] * qk[j] >= thr
        if same:
            ok &= i <= j
        sel = np.nonzero(ok)[0][:need]
        out.append(np.stack([i[sel], j[sel]], 1))
        need -= len(sel)
    if not out:
        return np.zeros((0, 2), np.int32)
    return np.ascontiguousarray(np.concatenate(out).astype(np.int32))

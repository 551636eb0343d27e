"""Seeded synthetic shell sets and pair lists for the five BASELINE.json configs.

This module holds NONE of the method's arithmetic (no Boys, E, R, recurrences, contractions).  It only draws
the inputs -- centres, exponents, contraction coefficients, pair lists -- and applies the normalisation the
caller of an integral library is responsible for (the library applies coefficients
verbatim to unnormalised primitives).  Both the CUDA path and the CPU oracle receive exactly these arrays;
neither imports the other.

Recipe (the paper does not state its benchmark geometry, so these seeded
shells stand in for its per-class microbenchmarks): ``numpy.random.Generator(PCG64(seed))``; per shell set the
draw order is centres ``uniform(0, box, (n,3))``, exponents ``exp(uniform(ln lo, ln hi, n))``, then (K > 1)
coefficients ``uniform(0.1, 1, (n,K))``; pair lists from ``rng.permutation`` afterwards.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

L_LETTERS = "spdfghik"


@dataclass
class ShellSet:
    """Shell table in the layout of ``md4_set_shells`` (include/md4.h)."""

    centers: np.ndarray          # [nshell, 3] float64, bohr
    l: np.ndarray                # [nshell] int32
    prim_offset: np.ndarray      # [nshell+1] int32 (CSR)
    exponents: np.ndarray        # [nprim] float64
    coefficients: np.ndarray     # [nprim] float64, normalisation folded in

    @property
    def nshell(self) -> int:
        return int(self.l.shape[0])


@dataclass
class Workload:
    name: str
    shells: ShellSet
    bra_ij: np.ndarray           # [nbra, 2] int32
    ket_ij: np.ndarray           # [nket, 2] int32
    lclass: tuple                # (la, lb, lc, ld)
    kclass: tuple                # (Ka, Kb, Kc, Kd)
    seed: int
    meta: dict = field(default_factory=dict)

    @property
    def nquartets(self) -> int:
        return int(self.bra_ij.shape[0]) * int(self.ket_ij.shape[0])


def _self_overlap_radial(l: int, z: float) -> float:
    """Int S_lm(r)^2 exp(-z r^2) d3r for Racah-normalised S_lm: (4 pi/(2l+1)) Gamma(l+3/2) / (2 z^(l+3/2))."""
    return (4.0 * math.pi / (2 * l + 1)) * math.gamma(l + 1.5) / (2.0 * z ** (l + 1.5))


def normalise(l: int, exps: np.ndarray, coefs: np.ndarray) -> np.ndarray:
    """Coefficients of a unit-norm contracted solid-harmonic shell over unnormalised primitives (Q10):
    c_k <- c_k N_l(zeta_k), then divide by sqrt(sum_jk c_j c_k <j|k>)."""
    c = np.array([ck / math.sqrt(_self_overlap_radial(l, 2.0 * zk)) for ck, zk in zip(coefs, exps)])
    s = 0.0
    for cj, zj in zip(c, exps):
        for ck, zk in zip(c, exps):
            s += cj * ck * _self_overlap_radial(l, zj + zk)
    return c / math.sqrt(s)


def make_shells(rng: np.random.Generator, n: int, l, box: float, lo: float, hi: float, K: int = 1,
                ratio: float = 3.0) -> ShellSet:
    """n shells; K == 1: exponents log-uniform in [lo, hi]; K > 1: zeta_k = zeta_0 ratio^k with zeta_0
    log-uniform in [lo, hi] and coefficients uniform in [0.1, 1] before normalisation."""
    ls = np.full(n, l, dtype=np.int32) if np.isscalar(l) else np.asarray(l, dtype=np.int32)
    centers = rng.uniform(0.0, box, size=(n, 3))
    z0 = np.exp(rng.uniform(math.log(lo), math.log(hi), size=n))
    raw = rng.uniform(0.1, 1.0, size=(n, K)) if K > 1 else np.ones((n, 1))
    exps = z0[:, None] * ratio ** np.arange(K)[None, :]
    coefs = np.stack([normalise(int(ls[i]), exps[i], raw[i]) for i in range(n)])
    return ShellSet(centers=np.ascontiguousarray(centers), l=ls,
                    prim_offset=(np.arange(n + 1) * K).astype(np.int32),
                    exponents=np.ascontiguousarray(exps.reshape(-1)),
                    coefficients=np.ascontiguousarray(coefs.reshape(-1)))


def _pairs_from_flat(flat: np.ndarray, n: int) -> np.ndarray:
    return np.stack([flat // n, flat % n], axis=1).astype(np.int32)


def config1() -> Workload:
    """(gg|gg) K=1: 16 shells, box 6, exponents in [0.1, 20], seed 0; bra = [(0,1)], ket = all 256 ordered
    pairs i-major (includes i = j, both orders and the bra pair itself, T = 0)."""
    rng = np.random.Generator(np.random.PCG64(0))
    sh = make_shells(rng, 16, 4, 6.0, 0.1, 20.0)
    ket = _pairs_from_flat(np.arange(256), 16)
    return Workload("cfg1 (gg|gg) K=1", sh, np.array([[0, 1]], dtype=np.int32), ket, (4, 4, 4, 4), (1, 1, 1, 1), 0)


def _perm_config(name, seed, n, l, box, lo, hi, npair, K=1) -> Workload:
    rng = np.random.Generator(np.random.PCG64(seed))
    sh = make_shells(rng, n, l, box, lo, hi, K=K)
    bra = _pairs_from_flat(rng.permutation(n * n)[:npair], n)
    ket = _pairs_from_flat(rng.permutation(n * n)[:npair], n)
    return Workload(name, sh, bra, ket, (l,) * 4, (K,) * 4, seed)


def config2() -> Workload:
    """(hh|hh) K=1: 64 shells, box 10, [0.05, 50], seed 1; 64 bra x 64 ket pairs = 4096 quartets."""
    return _perm_config("cfg2 (hh|hh) K=1", 1, 64, 5, 10.0, 0.05, 50.0, 64)


def config3() -> Workload:
    """(ii|ii) K=1 (headline): 128 shells, box 12, [0.05, 50], seed 2; 128 x 128 = 16384 quartets."""
    return _perm_config("cfg3 (ii|ii) K=1", 2, 128, 6, 12.0, 0.05, 50.0, 128)


def config4() -> Workload:
    """(ii|ii) K=5 per shell (625 primitive quartets): 32 shells, box 12, zeta_0 in [0.05, 1], ratio 3,
    seed 3; 32 x 32 = 1024 quartets."""
    return _perm_config("cfg4 (ii|ii) K=5/shell", 3, 32, 6, 12.0, 0.05, 1.0, 32, K=5)


def sweep_classes():
    """The 21 classes (la lb|lc ld), l in {4,5,6}, la >= lb, lc >= ld, bra >= ket (pairs ordered
    lexicographically by (la, lb))."""
    prs = [(a, b) for a in (4, 5, 6) for b in (4, 5, 6) if a >= b]
    return [(a, b, c, d) for (a, b) in prs for (c, d) in prs if (a, b) >= (c, d)]


def config5(class_index: int, K: int = 1, nper: int = 8, seed_offset: int = 0) -> Workload:
    """One class of the mixed sweep: nper shells per role a,b,c,d (box 10), bra = all nper x nper (a_i,b_j),
    ket = all (c_i,d_j); K = 1: exponents in [0.05, 50]; K = 3: zeta_0 in [0.05, 50/9], ratio 3;
    seed 1000 + class index."""
    la, lb, lc, ld = sweep_classes()[class_index]
    seed = 1000 + class_index + seed_offset   # seed_offset: other ranks of a multi-GPU bench draw their own shells
    rng = np.random.Generator(np.random.PCG64(seed))
    ls = np.repeat(np.array([la, lb, lc, ld], dtype=np.int32), nper)
    hi = 50.0 if K == 1 else 50.0 / 9.0
    sh = make_shells(rng, 4 * nper, ls, 10.0, 0.05, hi, K=K)
    bra = np.array([[i, nper + j] for i in range(nper) for j in range(nper)], dtype=np.int32)
    ket = np.array([[2 * nper + i, 3 * nper + j] for i in range(nper) for j in range(nper)], dtype=np.int32)
    name = f"cfg5 ({L_LETTERS[la]}{L_LETTERS[lb]}|{L_LETTERS[lc]}{L_LETTERS[ld]}) K={K}/shell"
    return Workload(name, sh, bra, ket, (la, lb, lc, ld), (K,) * 4, seed)


def small_workload(lclass, kclass=(1, 1, 1, 1), nbra=3, nket=3, seed=7, box=4.0, lo=0.2, hi=5.0) -> Workload:
    """Small generic case for tests: one shell set per role, ragged pair lists allowed."""
    la, lb, lc, ld = lclass
    rng = np.random.Generator(np.random.PCG64(seed))
    n = max(nbra, nket, 2)
    sets = []
    for l, K in zip(lclass, kclass):
        sets.append(make_shells(rng, n, l, box, lo, hi, K=K))
    centers = np.concatenate([s.centers for s in sets])
    ls = np.concatenate([s.l for s in sets])
    exps = np.concatenate([s.exponents for s in sets])
    coefs = np.concatenate([s.coefficients for s in sets])
    counts = np.concatenate([np.diff(s.prim_offset) for s in sets])
    off = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    sh = ShellSet(centers, ls.astype(np.int32), off, exps, coefs)
    bra = np.array([[i % n, n + (i * 7 + 1) % n] for i in range(nbra)], dtype=np.int32).reshape(-1, 2)
    ket = np.array([[2 * n + (j * 3 + 1) % n, 3 * n + j % n] for j in range(nket)], dtype=np.int32).reshape(-1, 2)
    return Workload(f"small {lclass} K={kclass}", sh, bra, ket, tuple(lclass), tuple(kclass), seed)


# ---- sizes used by the FLOP / byte accounting -----------------------
def n_solid(l: int) -> int:
    return 2 * l + 1


def n_hermite(n: int) -> int:
    return (n + 1) * (n + 2) * (n + 3) // 6


def class_flops(lclass, kclass) -> int:
    """Algorithmic FLOPs per shell quartet, matrix operations only, bra transformed first:
    K_bra K_ket 2 N_ab N_p N_q + K_ket 2 N_ab N_q N_cd."""
    la, lb, lc, ld = lclass
    ka, kb, kc, kd = kclass
    nab, ncd = n_solid(la) * n_solid(lb), n_solid(lc) * n_solid(ld)
    np_, nq = n_hermite(la + lb), n_hermite(lc + ld)
    return ka * kb * kc * kd * 2 * nab * np_ * nq + kc * kd * 2 * nab * nq * ncd


def class_out_doubles(lclass) -> int:
    la, lb, lc, ld = lclass
    return n_solid(la) * n_solid(lb) * n_solid(lc) * n_solid(ld)

"""CPU oracle for (ab|cd) -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Thin ctypes front end of ``oracle/eri_oracle.c`` (Obara-Saika / Head-Gordon-Pople evaluator),
built twice from the same source: ``liberi_oracle_q.so`` evaluates in IEEE binary128 and is the parity
reference; ``liberi_oracle.so`` evaluates in x87 long double (the precision BASELINE.json names) and serves the
cheap pins and the timed CPU baseline.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with ``paper_2307_03452_b200``
and never imports it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "eri_oracle.c")
_LIB = os.path.join(_HERE, "liberi_oracle.so")
_LIBQ = os.path.join(_HERE, "liberi_oracle_q.so")
_lib = None
_libq = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no fast-math: long-double arithmetic must stay IEEE/x87 exact)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm", "-lpthread"]
        subprocess.run(cmd, check=True)
    return _LIB


def build_quad(force: bool = False) -> str:
    """Audit build of the same source in binary128 (libquadmath); used only to measure the rounding
    error of the long-double build."""
    if force or not os.path.exists(_LIBQ) or os.path.getmtime(_LIBQ) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=gnu11", "-DORACLE_QUAD", "-fPIC", "-shared", "-o", _LIBQ, _SRC,
               "-lquadmath", "-lm", "-lpthread"]
        subprocess.run(cmd, check=True)
    return _LIBQ


def _load(quad: bool = False):
    global _lib, _libq
    if quad:
        if _libq is None:
            build_quad()
            _libq = _bind(ctypes.CDLL(_LIBQ))
        return _libq
    if _lib is None:
        build()
        _lib = _bind(ctypes.CDLL(_LIB))
    return _lib


def _bind(lib):
    if True:
        ld_p = ctypes.POINTER(ctypes.c_longdouble)
        d_p = ctypes.POINTER(ctypes.c_double)
        i_p = ctypes.POINTER(ctypes.c_int)
        lib.oracle_boys.argtypes = [ctypes.c_int, ctypes.c_longdouble, ld_p]
        lib.oracle_boys.restype = None
        lib.oracle_set_kernel.argtypes = [ctypes.c_int, ctypes.c_double]
        lib.oracle_set_kernel.restype = ctypes.c_int
        lib.oracle_kernel_seeds.argtypes = [ctypes.c_int, ctypes.c_longdouble, ctypes.c_longdouble, ld_p]
        lib.oracle_kernel_seeds.restype = None
        lib.oracle_solid_coeff.argtypes = [ctypes.c_int, ld_p]
        lib.oracle_solid_coeff.restype = None
        lib.oracle_cart_pos.argtypes = [ctypes.c_int] * 3
        lib.oracle_cart_pos.restype = ctypes.c_int
        lib.oracle_quartet_ld.argtypes = [d_p, i_p, i_p, d_p, d_p] + [ctypes.c_int] * 5 + [ld_p]
        lib.oracle_quartet_ld.restype = ctypes.c_int
        lib.oracle_compute.argtypes = [ctypes.c_int, d_p, i_p, i_p, d_p, d_p, ctypes.c_int, i_p, ctypes.c_int, i_p,
                                       i_p, ctypes.c_int, d_p, ctypes.c_int, ctypes.c_int]
        lib.oracle_compute.restype = ctypes.c_int
    return lib


def _ld(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_longdouble))


def _d(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _i(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int))


def boys(mmax: int, T) -> np.ndarray:
    """F_m(T), m = 0..mmax, as a numpy longdouble array (Eq.11).  T is taken as a C double
    (ctypes converts through Python float), evaluated in long double."""
    out = np.zeros(mmax + 1, dtype=np.longdouble)
    _load().oracle_boys(int(mmax), ctypes.c_longdouble(float(T)), _ld(out))
    return out


KERNELS = {"coulomb": 0, "erf": 1, "erfc": 2}


def set_kernel(kind: str = "coulomb", omega: float = 0.0) -> None:
    """Interaction kernel of every later call, in BOTH builds: 1/r ("coulomb"), erf(omega r)/r or erfc(omega r)/r
    (ref. 21: only the seeds [0]^(m) change, see eri_oracle.c)."""
    for quad in (False, True):
        rc = _load(quad).oracle_set_kernel(KERNELS[kind], float(omega))
        if rc:
            raise ValueError(f"bad kernel {kind!r}, omega = {omega}")


def kernel_seeds(mmax: int, rho: float, T: float) -> np.ndarray:
    """G_m(rho, T), m = 0..mmax, for the current kernel (long-double build)."""
    out = np.zeros(mmax + 1, dtype=np.longdouble)
    _load().oracle_kernel_seeds(int(mmax), ctypes.c_longdouble(float(rho)), ctypes.c_longdouble(float(T)), _ld(out))
    return out


def solid_coeff(l: int) -> np.ndarray:
    """C[m+l, k]: coefficient of the k-th Cartesian monomial of degree l in S_lm."""
    nc = (l + 1) * (l + 2) // 2
    out = np.zeros((2 * l + 1, nc), dtype=np.longdouble)
    _load().oracle_solid_coeff(int(l), _ld(out))
    return out


def cart_pos(x: int, y: int, z: int) -> int:
    return _load().oracle_cart_pos(int(x), int(y), int(z))


def cart_list(l: int):
    """Cartesian exponent triples of degree l in the oracle's order."""
    lst = [None] * ((l + 1) * (l + 2) // 2)
    for x in range(l + 1):
        for y in range(l + 1 - x):
            lst[cart_pos(x, y, l - x - y)] = (x, y, l - x - y)
    return lst


class Shells:
    """Shell table in the layout of md4_set_shells (include/md4.h)."""

    def __init__(self, centers, l, prim_offset, exponents, coefficients):
        self.centers = np.ascontiguousarray(centers, dtype=np.float64).reshape(-1, 3)
        self.l = np.ascontiguousarray(l, dtype=np.int32)
        self.prim_offset = np.ascontiguousarray(prim_offset, dtype=np.int32)
        self.exponents = np.ascontiguousarray(exponents, dtype=np.float64)
        self.coefficients = np.ascontiguousarray(coefficients, dtype=np.float64)
        assert self.centers.shape[0] == self.l.shape[0] == self.prim_offset.shape[0] - 1
        assert self.exponents.shape[0] == self.coefficients.shape[0] == self.prim_offset[-1]


def quartet(sh: Shells, ia: int, ib: int, ic: int, id_: int, solid: bool = True, quad: bool = False) -> np.ndarray:
    """One contracted shell quartet in long double; shape (na, nb, nc, nd).
    quad=True evaluates in binary128 (audit build) and rounds to long double."""
    ls = [int(sh.l[k]) for k in (ia, ib, ic, id_)]
    dims = [2 * l + 1 if solid else (l + 1) * (l + 2) // 2 for l in ls]
    out = np.zeros(dims, dtype=np.longdouble)
    rc = _load(quad).oracle_quartet_ld(_d(sh.centers), _i(sh.l), _i(sh.prim_offset), _d(sh.exponents),
                                   _d(sh.coefficients), ia, ib, ic, id_, 1 if solid else 0, _ld(out))
    if rc:
        raise RuntimeError(f"oracle_quartet_ld failed rc={rc}")
    return out


def compute(sh: Shells, bra_ij, ket_ij, subset=None, nthreads: int | None = None, precision: str = "quad",
            nslice: int = 1) -> np.ndarray:
    """Batch in the md4_compute layout, float64: out[i_bra, j_ket, ma, mb, mc, md]
    (or out[k, ma, mb, mc, md] for the flat quartet indices i*nket+j listed in ``subset``).

    precision: "quad" (default, the parity reference: IEEE binary128 build) or "ld" (x87 long-double build,
    8x faster, loses up to ~1e-10 relative on tight high-l shells -- see the header of eri_oracle.c).
    nslice > 1 spreads the primitive loop of each quartet over threads (heavily contracted quartets)."""
    assert precision in ("quad", "ld")
    bra = np.ascontiguousarray(bra_ij, dtype=np.int32).reshape(-1, 2)
    ket = np.ascontiguousarray(ket_ij, dtype=np.int32).reshape(-1, 2)
    if nthreads is None:
        nthreads = os.cpu_count() or 1
    if bra.shape[0] == 0 or ket.shape[0] == 0:
        return np.zeros((bra.shape[0], ket.shape[0], 0), dtype=np.float64)
    dims = [2 * int(sh.l[k]) + 1 for k in (bra[0, 0], bra[0, 1], ket[0, 0], ket[0, 1])]
    if subset is None:
        out = np.zeros([bra.shape[0], ket.shape[0]] + dims, dtype=np.float64)
        sub_p, nsub = None, 0
    else:
        sub = np.ascontiguousarray(subset, dtype=np.int32)
        out = np.zeros([sub.shape[0]] + dims, dtype=np.float64)
        sub_p, nsub = _i(sub), sub.shape[0]
    rc = _load(precision == "quad").oracle_compute(sh.l.shape[0], _d(sh.centers), _i(sh.l), _i(sh.prim_offset), _d(sh.exponents),
                                _d(sh.coefficients), bra.shape[0], _i(bra), ket.shape[0], _i(ket), sub_p, nsub,
                                _d(out), int(nthreads), int(nslice))
    if rc:
        raise RuntimeError(f"oracle_compute failed rc={rc}")
    return out


def ao_offsets(sh: Shells) -> np.ndarray:
    """First AO (solid-harmonic function) of every shell and the total: shells in table order, 2l+1 functions each,
    m = -l..+l ascending -- the AO order md4_compute_jk uses (include/md4.h)."""
    return np.concatenate([[0], np.cumsum(2 * sh.l.astype(np.int64) + 1)])


def digest_jk(sh: Shells, bra_ij, ket_ij, D, **kw):
    """Direct digestion of a (bra list x ket list) batch into Coulomb- and exchange-type matrices ("computing
    Fock matrix elements directly", :249), written out as its definition: for EVERY listed quartet
    (bra pair (a,b), ket pair (c,d)), exactly

        J[a, b] += sum_{cd} (ab|cd) D[c, d]          K[a, c] += sum_{bd} (ab|cd) D[b, d]

    over the AO blocks of the four shells; nothing else (no permutational images, no factors: the caller lists what it
    wants).  Integrals from compute() (binary128 by default, rounded to double), contraction and accumulation in long
    double.  Returns (J, K) as long-double [nbf, nbf] arrays."""
    off = ao_offsets(sh)
    nbf = int(off[-1])
    Dl = np.asarray(D, dtype=np.longdouble).reshape(nbf, nbf)
    bra = np.ascontiguousarray(bra_ij, dtype=np.int32).reshape(-1, 2)
    ket = np.ascontiguousarray(ket_ij, dtype=np.int32).reshape(-1, 2)
    J = np.zeros((nbf, nbf), dtype=np.longdouble)
    K = np.zeros((nbf, nbf), dtype=np.longdouble)
    if bra.shape[0] == 0 or ket.shape[0] == 0:
        return J, K
    eri = compute(sh, bra, ket, **kw).astype(np.longdouble)      # [i, j, ma, mb, mc, md]
    for i, (a, b) in enumerate(bra):
        sa, sb = slice(off[a], off[a + 1]), slice(off[b], off[b + 1])
        for j, (c, d) in enumerate(ket):
            sc, sd = slice(off[c], off[c + 1]), slice(off[d], off[d + 1])
            g = eri[i, j]
            for ma in range(g.shape[0]):
                for mb in range(g.shape[1]):
                    J[off[a] + ma, off[b] + mb] += (g[ma, mb] * Dl[sc, sd]).sum()
                    for mc in range(g.shape[2]):
                        K[off[a] + ma, off[c] + mc] += (g[ma, mb, mc, :] * Dl[off[b] + mb, sd]).sum()
    return J, K

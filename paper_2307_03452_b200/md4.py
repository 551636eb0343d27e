"""Thin ctypes binding of libmd4 (include/md4.h): same names, argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; there is no CPU fallback -- if the
library is missing or no CUDA device is present the calls fail loudly.  torch is used only for device
memory and streams (``out`` tensors, ``torch.cuda.current_stream()``).
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmd4.so")

MD4_OK, MD4_EINVAL, MD4_EUNSUPPORTED, MD4_ESTATE, MD4_ENOMEM, MD4_ECUDA = range(6)
KERNELS = {"coulomb": 0, "erf": 1, "erfc": 2}   # md4_kernel of include/md4.h
STATUS_NAMES = ["MD4_OK", "MD4_EINVAL", "MD4_EUNSUPPORTED", "MD4_ESTATE", "MD4_ENOMEM", "MD4_ECUDA"]

#: every symbol include/md4.h declares (tests check the library exports exactly these)
SYMBOLS = [
    "md4_create", "md4_destroy", "md4_last_error", "md4_set_shells", "md4_build_pairs", "md4_free_pairs",
    "md4_stream_wait_pairs", "md4_set_kernel", "md4_num_ao", "md4_compute_jk", "md4_compute_jk_host",
    "md4_pairs_count", "md4_pairs_class", "md4_output_size", "md4_compute", "md4_compute_host", "md4_compute_static", "md4_trim",
    "md4_launch_count", "md4_flops_per_quartet", "md4_debug_boys", "md4_debug_solid_coeff",
    "md4_debug_hermite_r", "md4_debug_pair_h", "md4_debug_work_items",
]

_lib = None


class Md4Error(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{STATUS_NAMES[status] if 0 <= status < 6 else status}: {msg}")
        self.status = status


def load():
    """dlopen libmd4.so (built by ``python -m paper_2307_03452_b200.build``); raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} not found: build it with `python -m paper_2307_03452_b200.build` "
                           "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, ip, dp = ctypes.c_void_p, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_double)
    lib.md4_create.argtypes = [ctypes.POINTER(vp), ctypes.c_int]
    lib.md4_create.restype = ctypes.c_int
    lib.md4_destroy.argtypes = [vp]
    lib.md4_destroy.restype = None
    lib.md4_last_error.argtypes = [vp]
    lib.md4_last_error.restype = ctypes.c_char_p
    lib.md4_set_shells.argtypes = [vp, ctypes.c_int, dp, ip, ip, dp, dp]
    lib.md4_set_shells.restype = ctypes.c_int
    lib.md4_build_pairs.argtypes = [vp, ctypes.c_int, ip, ctypes.POINTER(vp)]
    lib.md4_build_pairs.restype = ctypes.c_int
    lib.md4_free_pairs.argtypes = [vp, vp]
    lib.md4_free_pairs.restype = None
    lib.md4_set_kernel.argtypes = [vp, ctypes.c_int, ctypes.c_double]
    lib.md4_set_kernel.restype = ctypes.c_int
    lib.md4_stream_wait_pairs.argtypes = [vp, vp, vp]
    lib.md4_stream_wait_pairs.restype = ctypes.c_int
    lib.md4_pairs_count.argtypes = [vp]
    lib.md4_pairs_count.restype = ctypes.c_int
    lib.md4_pairs_class.argtypes = [vp, ip]
    lib.md4_pairs_class.restype = ctypes.c_int
    lib.md4_output_size.argtypes = [vp, vp, ctypes.POINTER(ctypes.c_size_t)]
    lib.md4_output_size.restype = ctypes.c_int
    lib.md4_compute.argtypes = [vp, vp, vp, vp, ctypes.c_size_t, vp]
    lib.md4_compute.restype = ctypes.c_int
    lib.md4_compute_host.argtypes = [vp, vp, vp, vp, ctypes.c_size_t, vp]
    lib.md4_compute_static.argtypes = [vp, vp, vp, vp, ctypes.c_size_t, vp]
    lib.md4_compute_static.restype = ctypes.c_int
    lib.md4_trim.argtypes = [vp]
    lib.md4_trim.restype = ctypes.c_int
    lib.md4_compute_host.restype = ctypes.c_int
    lib.md4_num_ao.argtypes = [vp, ip]
    lib.md4_num_ao.restype = ctypes.c_int
    lib.md4_compute_jk.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    lib.md4_compute_jk.restype = ctypes.c_int
    lib.md4_compute_jk_host.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    lib.md4_compute_jk_host.restype = ctypes.c_int
    lib.md4_launch_count.argtypes = [vp]
    lib.md4_launch_count.restype = ctypes.c_longlong
    lib.md4_flops_per_quartet.argtypes = [vp, vp]
    lib.md4_flops_per_quartet.restype = ctypes.c_double
    lib.md4_debug_boys.argtypes = [vp, ctypes.c_int, ctypes.c_int, dp, dp]
    lib.md4_debug_boys.restype = ctypes.c_int
    lib.md4_debug_solid_coeff.argtypes = [vp, ctypes.c_int, dp]
    lib.md4_debug_solid_coeff.restype = ctypes.c_int
    lib.md4_debug_hermite_r.argtypes = [vp, ctypes.c_int, dp, dp]
    lib.md4_debug_hermite_r.restype = ctypes.c_int
    lib.md4_debug_pair_h.argtypes = [vp, vp, ctypes.c_int, ctypes.c_int, dp, dp]
    lib.md4_debug_pair_h.restype = ctypes.c_int
    lib.md4_debug_work_items.argtypes = [ctypes.c_int, ctypes.c_int, ip]
    lib.md4_debug_work_items.restype = ctypes.c_int
    _lib = lib
    return lib


def work_items(li: int, lj: int):
    """(number of items, first row block per item, row blocks per item) of a bra class; host logic, no GPU."""
    out = (ctypes.c_int * 7)()
    st = load().md4_debug_work_items(li, lj, out)
    if st != 0:
        raise Md4Error(st, "md4_debug_work_items")
    n = out[0]
    return n, list(out[1:1 + n]), list(out[4:4 + n])


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _ip(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int))


class PairList:
    """Handle of a device-resident shell-pair list (md4_pairs*)."""

    def __init__(self, engine: "Engine", handle):
        self.engine = engine
        self.handle = handle

    def __len__(self) -> int:
        return load().md4_pairs_count(self.handle)

    @property
    def klass(self):
        info = np.zeros(4, dtype=np.int32)
        self.engine._check(load().md4_pairs_class(self.handle, _ip(info)))
        return tuple(int(x) for x in info)

    def free(self):
        if self.handle is not None and self.engine.handle is not None:
            load().md4_free_pairs(self.engine.handle, self.handle)
        self.handle = None


class Engine:
    """md4_ctx*: one per CUDA device."""

    def __init__(self, device: int = 0):
        lib = load()
        h = ctypes.c_void_p()
        st = lib.md4_create(ctypes.byref(h), int(device))
        if st != MD4_OK:
            raise Md4Error(st, (lib.md4_last_error(None) or b"").decode())
        self.handle = h
        self.device = int(device)

    # -- plumbing
    def _check(self, st: int):
        if st != MD4_OK:
            raise Md4Error(st, (load().md4_last_error(self.handle) or b"").decode())

    def close(self):
        if self.handle is not None:
            load().md4_destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def last_error(self) -> str:
        return (load().md4_last_error(self.handle) or b"").decode()

    # -- the ABI calls
    def set_shells(self, centers, l, prim_offset, exponents, coefficients):
        c = np.ascontiguousarray(centers, dtype=np.float64).reshape(-1)
        li = np.ascontiguousarray(l, dtype=np.int32)
        off = np.ascontiguousarray(prim_offset, dtype=np.int32)
        ex = np.ascontiguousarray(exponents, dtype=np.float64)
        co = np.ascontiguousarray(coefficients, dtype=np.float64)
        self._check(load().md4_set_shells(self.handle, int(li.shape[0]), _dp(c), _ip(li), _ip(off), _dp(ex), _dp(co)))

    def set_kernel(self, kind: str = "coulomb", omega: float = 0.0):
        """Interaction kernel of later compute calls: "coulomb" (1/r12), "erf" or "erfc" (attenuated with omega)."""
        self._check(load().md4_set_kernel(self.handle, KERNELS[kind], float(omega)))

    def build_pairs(self, ij) -> PairList:
        a = np.ascontiguousarray(ij, dtype=np.int32).reshape(-1, 2)
        h = ctypes.c_void_p()
        self._check(load().md4_build_pairs(self.handle, int(a.shape[0]), _ip(a), ctypes.byref(h)))
        return PairList(self, h)

    def stream_wait_pairs(self, pairs: PairList, stream: int):
        self._check(load().md4_stream_wait_pairs(self.handle, pairs.handle, ctypes.c_void_p(stream)))

    def output_size(self, bra: PairList, ket: PairList) -> int:
        n = ctypes.c_size_t()
        self._check(load().md4_output_size(bra.handle, ket.handle, ctypes.byref(n)))
        return int(n.value)

    def output_shape(self, bra: PairList, ket: PairList):
        la, lb, _, _ = bra.klass
        lc, ld, _, _ = ket.klass
        return (len(bra), len(ket), 2 * la + 1, 2 * lb + 1, 2 * lc + 1, 2 * ld + 1)

    def compute(self, bra: PairList, ket: PairList, out=None, stream=None):
        """Enqueue md4_compute on ``stream`` (default: torch's current stream) into the torch CUDA tensor
        ``out`` (allocated if None).  Asynchronous; returns ``out`` shaped [nbra, nket, ma, mb, mc, md]."""
        import torch

        n = self.output_size(bra, ket)
        if out is None:
            out = torch.empty(n, dtype=torch.float64, device=f"cuda:{self.device}")
        if out.dtype != torch.float64 or not out.is_cuda or not out.is_contiguous():
            raise ValueError("out must be a contiguous float64 CUDA tensor")
        if stream is None:
            stream = torch.cuda.current_stream(self.device).cuda_stream
        self._check(load().md4_compute(self.handle, bra.handle, ket.handle, ctypes.c_void_p(out.data_ptr()),
                                       out.numel(), ctypes.c_void_p(stream)))
        return out.view(-1)[:n].view(self.output_shape(bra, ket)) if n else out.view(-1)[:0]

    def trim(self):
        """Return the idle blocks of the context's pool to the driver (md4_trim)."""
        self._check(load().md4_trim(self.handle))

    def compute_static(self, bra: PairList, ket: PairList, out, stream=None):
        """Enqueue md4_compute_static (no device allocation: the [ab|q~] scratch of contracted bras is the library's static
        32 MiB device array, md4.h) into the caller's contiguous float64 CUDA tensor ``out``; returns it shaped like compute."""
        import torch

        n = self.output_size(bra, ket)
        if out.dtype != torch.float64 or not out.is_cuda or not out.is_contiguous():
            raise ValueError("out must be a contiguous float64 CUDA tensor")
        if stream is None:
            stream = torch.cuda.current_stream(self.device).cuda_stream
        self._check(load().md4_compute_static(self.handle, bra.handle, ket.handle, ctypes.c_void_p(out.data_ptr()),
                                              out.numel(), ctypes.c_void_p(stream)))
        return out.view(-1)[:n].view(self.output_shape(bra, ket)) if n else out.view(-1)[:0]

    def compute_ptr(self, bra: PairList, ket: PairList, d_ptr: int, capacity: int, stream: int = 0):
        self._check(load().md4_compute(self.handle, bra.handle, ket.handle, ctypes.c_void_p(d_ptr), int(capacity),
                                       ctypes.c_void_p(stream)))

    def compute_host(self, bra: PairList, ket: PairList, out: np.ndarray | None = None, stream: int = 0):
        n = self.output_size(bra, ket)
        if out is None:
            out = np.empty(n, dtype=np.float64)
        self._check(load().md4_compute_host(self.handle, bra.handle, ket.handle, ctypes.c_void_p(out.ctypes.data),
                                            out.size, ctypes.c_void_p(stream)))
        return out.reshape(-1)[:n].reshape(self.output_shape(bra, ket))

    def num_ao(self) -> int:
        n = ctypes.c_int()
        self._check(load().md4_num_ao(self.handle, ctypes.byref(n)))
        return int(n.value)

    def compute_jk(self, bra: PairList, ket: PairList, D, J=None, K=None, stream=None):
        """Enqueue md4_compute_jk: J[a,b] += sum_cd (ab|cd) D[c,d], K[a,c] += sum_bd (ab|cd) D[b,d] on [nbf, nbf] float64 CUDA
        tensors (J / K are accumulated into; pass None to skip one)."""
        import torch

        def ptr(t):
            if t is None:
                return ctypes.c_void_p(0)
            if t.dtype != torch.float64 or not t.is_cuda or not t.is_contiguous():
                raise ValueError("D, J, K must be contiguous float64 CUDA tensors")
            return ctypes.c_void_p(t.data_ptr())

        if stream is None:
            stream = torch.cuda.current_stream(self.device).cuda_stream
        self._check(load().md4_compute_jk(self.handle, bra.handle, ket.handle, ptr(D), ptr(J), ptr(K), ctypes.c_void_p(stream)))

    def compute_jk_host(self, bra: PairList, ket: PairList, D: np.ndarray, J: np.ndarray | None = None,
                        K: np.ndarray | None = None, stream: int = 0):
        """md4_compute_jk_host on float64 numpy matrices (J / K accumulated in place)."""
        def ptr(x):
            if x is None:
                return ctypes.c_void_p(0)
            if x.dtype != np.float64 or not x.flags.c_contiguous:
                raise ValueError("D, J, K must be C-contiguous float64 arrays")
            return ctypes.c_void_p(x.ctypes.data)

        self._check(load().md4_compute_jk_host(self.handle, bra.handle, ket.handle, ptr(D), ptr(J), ptr(K), ctypes.c_void_p(stream)))

    def launch_count(self) -> int:
        return int(load().md4_launch_count(self.handle))

    def flops_per_quartet(self, bra: PairList, ket: PairList) -> float:
        return float(load().md4_flops_per_quartet(bra.handle, ket.handle))

    # -- stage-level debug access
    def debug_boys(self, mmax: int, T) -> np.ndarray:
        t = np.ascontiguousarray(T, dtype=np.float64).reshape(-1)
        out = np.zeros((t.shape[0], mmax + 1), dtype=np.float64)
        self._check(load().md4_debug_boys(self.handle, int(mmax), int(t.shape[0]), _dp(t), _dp(out)))
        return out

    def debug_solid_coeff(self, l: int) -> np.ndarray:
        out = np.zeros((2 * l + 1, (l + 1) * (l + 2) // 2), dtype=np.float64)
        self._check(load().md4_debug_solid_coeff(self.handle, int(l), _dp(out)))
        return out

    def debug_hermite_r(self, L: int, zp, P, zq, Q) -> np.ndarray:
        pq = np.array([zp, *P, zq, *Q], dtype=np.float64)
        out = np.zeros((L + 1, L + 1, L + 1), dtype=np.float64)
        self._check(load().md4_debug_hermite_r(self.handle, int(L), _dp(pq), _dp(out)))
        return out

    def debug_pair_h(self, pairs: PairList, ipair: int, iprim: int = 0):
        li, lj, _, _ = pairs.klass
        nab = (2 * li + 1) * (2 * lj + 1)
        lb = li + lj
        nh = (lb + 1) * (lb + 2) * (lb + 3) // 6
        out = np.zeros((nab, nh), dtype=np.float64)
        scal = np.zeros(5, dtype=np.float64)
        self._check(load().md4_debug_pair_h(self.handle, pairs.handle, int(ipair), int(iprim), _dp(out), _dp(scal)))
        return out, scal

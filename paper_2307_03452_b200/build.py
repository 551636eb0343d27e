"""Build libmd4.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo snapshot).

    python -m paper_2307_03452_b200.build [--force]
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmd4.so")
OBJ = os.path.join(HERE, "build")
SOURCES = ["md4_api.cu", "md4_pairs.cu", "md4_eri.cu", "md4_eri_small.cu", "md4_tables.cpp"]
HEADERS = ["md4_internal.h", "md4_device.cuh", os.path.join("..", "..", "include", "md4.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", shutil.which("nvcc")):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found")


HASHFILE = os.path.join(OBJ, "libmd4.srchash")


def source_hash() -> str:
    """sha256 over the contents of every source and header of libmd4 plus the compiler flags (16 hex digits).  The
    build records it beside the library; bench.py keys the committed ncu traffic figure on it (profiles/*.json), so a
    figure captured on another build is never reported."""
    import hashlib

    h = hashlib.sha256()
    for rel in sorted(SOURCES + HEADERS):
        with open(os.path.join(CSRC, rel), "rb") as f:
            h.update(rel.replace(os.sep, "/").encode() + b"\0" + f.read() + b"\0")
    h.update(" ".join(NVCC_FLAGS).encode())
    return h.hexdigest()[:16]


def _stale() -> bool:
    """Content-based (file times do not survive a repository snapshot): the library is current if the hash recorded
    when it was linked equals the hash of the sources now."""
    if not os.path.exists(LIB) or not os.path.exists(HASHFILE):
        return True
    try:
        return open(HASHFILE).read().strip() != source_hash()
    except OSError:
        return True


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = _nvcc()
    os.makedirs(OBJ, exist_ok=True)

    def compile_one(src):
        obj = os.path.join(OBJ, os.path.splitext(src)[0] + ".o")
        cmd = [nvcc] + NVCC_FLAGS + os.environ.get("MD4_NVCC_EXTRA", "").split() + ["-x", "cu", "-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        with open(obj + ".log", "w") as f:
            f.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}:\n{r.stdout}\n{r.stderr}")
        if verbose:
            print(r.stderr)
        return obj

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    # link under a temporary name and rename: a process that finds libmd4.so never sees a half-written file
    tmp = f"{LIB}.{os.getpid()}.tmp"
    cmd = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp] + objs
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        if os.path.exists(tmp):
            os.unlink(tmp)
        raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    if os.path.exists(HASHFILE):
        os.unlink(HASHFILE)
    os.replace(tmp, LIB)
    with open(HASHFILE + ".tmp", "w") as f:
        f.write(source_hash() + "\n")
    os.replace(HASHFILE + ".tmp", HASHFILE)
    return LIB


def ensure_built() -> str:
    """Compile libmd4.so if it is missing or older than its sources (a checkout has no build artefacts; an edited
    csrc/ must never run as a stale binary); never a fallback for the kernels."""
    return build()


def wait_until_built(timeout_s: float = 600.0) -> str:
    """For the local ranks > 0 of a multi-process launch: wait until rank 0's ensure_built() has left a library that is
    newer than every source (the rename in build() makes its appearance atomic)."""
    import time

    t0 = time.time()
    while _stale():
        if time.time() - t0 > timeout_s:
            raise RuntimeError("libmd4.so was not built in time by local rank 0")
        time.sleep(0.25)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))

"""CPU-side checks of the boundary: libmd4.so builds for sm_100a, loads, and exports every symbol that
include/md4.h declares; the product path fails loudly without a CUDA device (no CPU fallback); the product
package never imports the oracle.  No compute calls here."""
import ctypes
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "md4.h")


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(md4_[a-z_0-9]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    from paper_2307_03452_b200 import build

    path = build.build()
    assert os.path.exists(path)
    return ctypes.CDLL(path)


def test_header_and_binding_agree():
    from paper_2307_03452_b200 import md4

    assert _declared() == sorted(md4.SYMBOLS)


def test_library_exports_every_declared_symbol(lib):
    for name in _declared():
        assert hasattr(lib, name), f"libmd4.so does not export {name}"


def test_library_is_sm100a_with_fp64_mma():
    """The built library carries sm_100a SASS and the contraction uses the FP64 tensor pipe (DMMA)."""
    from paper_2307_03452_b200 import build

    path = build.build()
    r = subprocess.run(["cuobjdump", "-lelf", path], capture_output=True, text=True)
    assert "sm_100a" in r.stdout, r.stdout + r.stderr
    r = subprocess.run(["cuobjdump", "-sass", path], capture_output=True, text=True)
    assert "DMMA.8x8x4" in r.stdout


def test_no_cpu_fallback_without_gpu(lib):
    import torch

    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2307_03452_b200 import md4

    with pytest.raises(md4.Md4Error) as ei:
        md4.Engine(0)
    assert ei.value.status in (md4.MD4_ECUDA, md4.MD4_EINVAL)
    assert md4.load().md4_last_error(None)


def test_null_handles_are_rejected(lib):
    lib.md4_set_shells.restype = ctypes.c_int
    assert lib.md4_set_shells(None, 0, None, None, None, None, None) == 1
    assert lib.md4_pairs_count(None) == -1
    lib.md4_flops_per_quartet.restype = ctypes.c_double
    assert lib.md4_flops_per_quartet(None, None) == 0.0
    lib.md4_destroy(None)
    lib.md4_free_pairs(None, None)
    assert lib.md4_create(None, 0) == 1


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2307_03452_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "eri_oracle" not in txt, f
    code = "import sys; import paper_2307_03452_b200.md4, paper_2307_03452_b200.inputs; assert 'oracle' not in sys.modules"
    subprocess.run([sys.executable, "-c", code], check=True, cwd=ROOT)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "libmd4" not in txt and "import paper_2307_03452_b200" not in txt


def test_work_item_split_follows_the_sub_partition_rule(lib):
    """Host logic of md4_compute (no GPU): rows of a bra class -> work items of <= 11 eight-row blocks.  An item of n
    blocks costs ceil(n/4) block-times (FP64 tensor pipe per SM sub-partition, profiles/r1_fp64_peak.txt): the split
    must cover every row block exactly once and reach the minimum ceil(nrb/4); bras with an l = 7 shell (up to 29 row
    blocks) take three items."""
    from paper_2307_03452_b200 import md4

    expect = {(6, 6): [11, 11], (6, 5): [10, 8], (5, 5): [8, 8], (6, 4): [8, 7], (5, 4): [7, 6], (4, 4): [11], (2, 2): [4],
              (7, 7): [11, 10, 8], (7, 6): [9, 8, 8], (7, 4): [9, 8]}
    for li in range(8):
        for lj in range(li + 1):
            nrb = ((2 * li + 1) * (2 * lj + 1) + 7) // 8
            n, row0, nrows = md4.work_items(li, lj)
            assert sum(nrows) == nrb and all(1 <= r <= 11 for r in nrows)
            assert row0 == [sum(nrows[:i]) for i in range(n)]
            assert n == (1 if nrb <= 11 else 2 if nrb <= 22 else 3)
            assert sum((r + 3) // 4 for r in nrows) == (nrb + 3) // 4
            if (li, lj) in expect:
                assert nrows == expect[(li, lj)], (li, lj, nrows)

"""md4_compute_static (include/md4.h): the fused kernel with its [ab|q~] scratch in the library's file-scope
`static __device__` array, for callers that cannot allocate device memory.  Checked against the existing path
(md4_compute, the context's own scratch) on the same lists, two calls in a row, within the per-quartet bar of the
parity tests (1e-10 of max|integral|).  Collected last on purpose (file name): the suite runs with pytest -x."""
import numpy as np
import pytest

from paper_2307_03452_b200 import inputs

pytestmark = pytest.mark.gpu

TOL = 1e-10   # the bar of tests/test_gpu_parity.py


@pytest.fixture(scope="module")
def eng():
    import torch
    from paper_2307_03452_b200 import md4

    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    e = md4.Engine(0)
    yield e
    e.close()


def _lists(eng, wl):
    s = wl.shells
    eng.set_shells(s.centers, s.l, s.prim_offset, s.exponents, s.coefficients)
    return eng.build_pairs(wl.bra_ij), eng.build_pairs(wl.ket_ij)


def _rel_err_per_quartet(got, ref):
    g = got.reshape(got.shape[0] * got.shape[1], -1)
    r = ref.reshape(g.shape)
    assert np.all(np.isfinite(g))
    mx = np.abs(r).max(axis=1)
    assert np.all(mx > 0)
    return np.abs(g - r).max(axis=1) / mx


# contracted bras (the scratch is used; 14 x 14 = 196 quartets > 148 CTAs, so slabs are reused within a launch),
# one class per consumer-warp layout that fits the 32 MiB, and an uncontracted class (no scratch at all)
CASES = [
    ((4, 4, 4, 4), (2, 2, 1, 1), 14, 14),
    ((5, 4, 4, 4), (3, 1, 2, 1), 14, 14),
    ((6, 6, 5, 5), (2, 1, 1, 1), 13, 12),
    ((2, 1, 2, 0), (3, 2, 2, 2), 20, 17),
    ((6, 6, 6, 6), (1, 1, 1, 1), 6, 5),
]


@pytest.mark.parametrize("lclass,kclass,nbra,nket", CASES)
def test_static_scratch_matches_existing_path_twice(eng, lclass, kclass, nbra, nket):
    import torch

    wl = inputs.small_workload(lclass, kclass, nbra=nbra, nket=nket, seed=23)
    bra, ket = _lists(eng, wl)
    ref = eng.compute(bra, ket)
    torch.cuda.synchronize()
    ref = ref.cpu().numpy()
    out = torch.empty(ref.size, dtype=torch.float64, device="cuda:0")
    for call in range(2):
        out.fill_(float("nan"))   # every element must be rewritten by the call
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info(0)[0]
        got = eng.compute_static(bra, ket, out)
        torch.cuda.synchronize()
        if call == 1:   # (the first launch of a kernel may load its module)
            assert torch.cuda.mem_get_info(0)[0] == free_before, "md4_compute_static changed the free device memory"
        err = _rel_err_per_quartet(got.cpu().numpy(), ref)
        assert err.max() <= TOL, f"call {call}: max rel err {err.max():.3e} (quartet {int(err.argmax())})"
    bra.free(); ket.free()


def test_static_scratch_after_other_contents(eng):
    """The array keeps the last call's contents: a call of another class in between must not change the result."""
    import torch

    wa = inputs.small_workload((4, 4, 4, 4), (2, 2, 1, 1), nbra=14, nket=14, seed=29)
    bra, ket = _lists(eng, wa)
    ref = eng.compute(bra, ket)
    out = torch.empty(ref.numel(), dtype=torch.float64, device="cuda:0")
    first = eng.compute_static(bra, ket, out).clone()
    # same shell set, other lists: (gg| bra against itself as ket, then the original pair again
    other = torch.empty(eng.output_size(bra, bra), dtype=torch.float64, device="cuda:0")
    eng.compute_static(bra, bra, other)
    second = eng.compute_static(bra, ket, out)
    torch.cuda.synchronize()
    r = ref.cpu().numpy()
    for got in (first, second):
        assert _rel_err_per_quartet(got.cpu().numpy(), r).max() <= TOL
    bra.free(); ket.free()


def test_static_scratch_rejects_classes_beyond_the_maximum(eng):
    """(ii|ii) with a contracted bra needs 148 x 11 x 57 x 512 bytes = 47.5 MB > 32 MiB: clear error, nothing written."""
    import torch
    from paper_2307_03452_b200 import md4

    wl = inputs.small_workload((6, 6, 6, 6), (2, 1, 1, 1), nbra=2, nket=2, seed=31)
    bra, ket = _lists(eng, wl)
    out = torch.full((eng.output_size(bra, ket),), -7.0, dtype=torch.float64, device="cuda:0")
    with pytest.raises(md4.Md4Error) as ei:
        eng.compute_static(bra, ket, out)
    assert ei.value.status == md4.MD4_EUNSUPPORTED
    assert "static scratch holds 33554432" in str(ei.value) and "MD4_STATIC_SCRATCH_BYTES" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((out == -7.0).all())
    # the existing path takes the same lists
    ref = eng.compute(bra, ket)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(ref).all())
    bra.free(); ket.free()

"""Pins for the CPU oracle (oracle/eri_oracle.c): each test checks it against something OTHER than itself --
printed reference values, closed forms, exact invariants, a textbook recurrence, and a brute-force quadrature
that uses neither the Boys function nor any recurrence (SURVEY.md 8(c) "What pins the oracle").  CPU only."""
import math
import os

import numpy as np
import pytest

import oracle
import refquad

GOLD = os.path.join(os.path.dirname(__file__), "golden")
CENT = [[0, 0, 0], [0, 0, 1], [0, 1, 0], [1, 0, 0.5]]
ZETA = [1.0, 0.5, 0.75, 1.25]


def _example(ls):
    return oracle.Shells(CENT, ls, [0, 1, 2, 3, 4], ZETA, [1, 1, 1, 1])


def _rand_shells(rng, ls, K=(1, 1, 1, 1), box=2.5, lo=0.3, hi=3.0):
    cent = rng.uniform(0, box, (4, 3))
    off = np.concatenate([[0], np.cumsum(K)])
    ex = np.exp(rng.uniform(math.log(lo), math.log(hi), off[-1]))
    co = rng.uniform(0.3, 1.0, off[-1])
    return oracle.Shells(cent, ls, off, ex, co)


# ---------------------------------------------------------------- Boys function (Eq.11)
def test_boys_printed_values():
    for line in open(os.path.join(GOLD, "boys_values.txt")):
        if line.startswith("#") or not line.strip():
            continue
        m, T, ref = line.split()
        got = oracle.boys(24, float(T))[int(m)]      # all printed T are exact doubles
        assert abs(got - np.longdouble(ref)) <= 3e-18 * abs(np.longdouble(ref)), (m, T)   # printed to 19 digits; a few long-double ulps


def test_boys_vs_incomplete_gamma():
    """F_m(T) = gamma(m+1/2, T) / (2 T^(m+1/2)) evaluated by mpmath at 40 digits (library routine, not ours)."""
    import mpmath as mp

    mp.mp.dps = 40
    for T in ["1e-6", "0.01", "0.37", "1", "7.3", "33", "80", "119.99", "120.01", "250", "2000", "19000"]:
        F = oracle.boys(32, float(T))
        for m in (0, 1, 5, 12, 17, 24, 32):
            Tm = mp.mpf(float(T))      # the binding passes T as a C double: use exactly that value
            ref = mp.gammainc(m + mp.mpf(1) / 2, 0, Tm) / (2 * Tm ** (m + mp.mpf(1) / 2))
            got = mp.mpf(np.format_float_scientific(F[m], precision=25, unique=False))
            assert abs(got - ref) <= mp.mpf("2e-18") * ref, (T, m, got, ref)


def test_boys_closed_forms_and_recursion():
    for T in (0.3, 2.0, 17.0, 64.0):
        F = oracle.boys(10, np.longdouble(T))
        f0 = 0.5 * math.sqrt(math.pi / T) * math.erf(math.sqrt(T))            # F_0 = 1/2 sqrt(pi/T) erf(sqrt T)
        assert abs(float(F[0]) - f0) <= 4e-16 * f0
        for m in range(10):                                                   # (2m+1) F_m = 2T F_{m+1} + e^-T
            lhs = (2 * m + 1) * F[m]
            rhs = 2 * np.longdouble(T) * F[m + 1] + np.exp(-np.longdouble(T))
            assert abs(lhs - rhs) <= 1e-17 * abs(lhs)
    F = oracle.boys(24, np.longdouble(0))
    for m in range(25):
        assert abs(F[m] - np.longdouble(1) / (2 * m + 1)) < 1e-19                # F_m(0) = 1/(2m+1)


# ---------------------------------------------------------------- solid harmonics
@pytest.fixture(scope="module")
def recurrence_S():
    return refquad.solid_harmonics_recurrence(6)


def test_solid_coeff_vs_textbook_recurrence(recurrence_S):
    """Closed-form table of the oracle == polynomials built by the l-recurrence (different route), l = 0..6."""
    S, syms = recurrence_S
    for l in range(7):
        ref = refquad.solid_coeff_table(l, oracle.cart_list(l), S, syms)
        got = oracle.solid_coeff(l)
        assert np.abs(got - ref).max() <= 2e-18 * np.abs(ref).max(), l


def test_solid_printed_low_l():
    """S_11 = x, S_1-1 = y, S_10 = z, S_22 = sqrt3/2 (x^2-y^2), S_2-2 = sqrt3 xy, S_20 = z^2 - x^2/2 - y^2/2."""
    c1 = oracle.solid_coeff(1).astype(float)
    pos = {c: i for i, c in enumerate(oracle.cart_list(1))}
    assert c1[2, pos[(1, 0, 0)]] == 1 and c1[0, pos[(0, 1, 0)]] == 1 and c1[1, pos[(0, 0, 1)]] == 1
    assert np.count_nonzero(c1) == 3
    c2 = oracle.solid_coeff(2).astype(float)
    pos = {c: i for i, c in enumerate(oracle.cart_list(2))}
    assert np.isclose(c2[4, pos[(2, 0, 0)]], math.sqrt(3) / 2) and np.isclose(c2[4, pos[(0, 2, 0)]], -math.sqrt(3) / 2)
    assert np.isclose(c2[0, pos[(1, 1, 0)]], math.sqrt(3))
    assert np.isclose(c2[2, pos[(0, 0, 2)]], 1) and np.isclose(c2[2, pos[(2, 0, 0)]], -0.5) and np.isclose(c2[2, pos[(0, 2, 0)]], -0.5)


def test_solid_harmonic_and_unsold():
    """Laplacian S_lm = 0 (harmonic) and sum_m S_lm^2 = r^(2l) (Unsold), l = 1..6, on random points."""
    rng = np.random.default_rng(5)
    pts = rng.normal(size=(20, 3))
    for l in range(1, 7):
        C = oracle.solid_coeff(l).astype(float)
        cl = oracle.cart_list(l)
        val = np.array([[sum(C[m, k] * x ** a * y ** b * z ** c for k, (a, b, c) in enumerate(cl)) for m in range(2 * l + 1)]
                        for (x, y, z) in pts])
        r2 = (pts ** 2).sum(1)
        assert np.allclose((val ** 2).sum(1), r2 ** l, rtol=1e-12)
        # Laplacian of each monomial, exactly on coefficients
        for m in range(2 * l + 1):
            lap = {}
            for k, (a, b, c) in enumerate(cl):
                for (e, f) in (((a - 2, b, c), a * (a - 1)), ((a, b - 2, c), b * (b - 1)), ((a, b, c - 2), c * (c - 1))):
                    if f:
                        lap[e] = lap.get(e, 0.0) + f * C[m, k]
            assert all(abs(v) < 1e-12 * np.abs(C[m]).max() * l * l for v in lap.values()), (l, m)


# ---------------------------------------------------------------- integrals
def test_ssss_closed_form():
    """(ss|ss) = K_ab K_cd 2 pi^(5/2) / (p q sqrt(p+q)) F_0(T), F_0 via erf."""
    rng = np.random.default_rng(11)
    for _ in range(10):
        sh = _rand_shells(rng, [0, 0, 0, 0])
        za, zb, zc, zd = sh.exponents
        A, B, C, D = sh.centers
        p, q = za + zb, zc + zd
        P, Q = (za * A + zb * B) / p, (zc * C + zd * D) / q
        T = p * q / (p + q) * ((P - Q) ** 2).sum()
        F0 = 0.5 * math.sqrt(math.pi / T) * math.erf(math.sqrt(T))
        ref = (math.exp(-za * zb / p * ((A - B) ** 2).sum() - zc * zd / q * ((C - D) ** 2).sum())
               * 2 * math.pi ** 2.5 / (p * q * math.sqrt(p + q)) * F0 * np.prod(sh.coefficients))
        got = float(oracle.quartet(sh, 0, 1, 2, 3)[0, 0, 0, 0])
        assert abs(got - ref) <= 1e-14 * abs(ref)


def test_worked_example_golden():
    """The printed values of SURVEY.md 8(c) item 4 (40-digit, two routes)."""
    cache = {}
    for line in open(os.path.join(GOLD, "worked_example.txt")):
        if line.startswith("#") or not line.strip():
            continue
        kind, l, i, j, k, m, ref = line.split()
        l, idx, ref = int(l), [int(i), int(j), int(k), int(m)], np.longdouble(ref)
        if kind == "solid":
            q = cache.setdefault(("s", l), oracle.quartet(_example([l] * 4), 0, 1, 2, 3))
            got = q[tuple(x + l for x in idx)]
        elif kind == "cart":
            q = cache.setdefault(("c", l), oracle.quartet(_example([1] * 4), 0, 1, 2, 3, solid=False))
            ax = [(1, 0, 0), (0, 1, 0), (0, 0, 1)]
            got = q[tuple(oracle.cart_pos(*ax[x]) for x in idx)]
        else:  # cartp: (p_i s|ss)
            q = cache.setdefault(("p",), oracle.quartet(_example([1, 0, 0, 0]), 0, 1, 2, 3, solid=False))
            ax = [(1, 0, 0), (0, 1, 0), (0, 0, 1)]
            got = q[oracle.cart_pos(*ax[idx[0]]), 0, 0, 0]
        # long-double OS/HGP loses digits with l (measured against the binary128 audit build); 1e-13 still
        # separates any formula error (O(1)) from rounding.
        tol = {0: 2e-18, 1: 2e-18, 2: 1e-16, 4: 1e-14, 6: 1e-13}[l]
        assert abs(got - ref) <= tol * abs(ref), (line, got)


@pytest.mark.parametrize("ls", [(0, 0, 0, 0), (1, 0, 1, 0), (1, 1, 1, 1), (2, 1, 1, 2), (2, 2, 2, 2), (3, 1, 2, 0), (4, 4, 4, 4)])
def test_vs_bruteforce_quadrature(ls):
    """Every Cartesian component of a primitive quartet against the Gauss-Hermite x Gauss-Legendre quadrature."""
    rng = np.random.default_rng(100 + sum(ls))
    sh = _rand_shells(rng, list(ls), box=1.5, lo=0.4, hi=2.0)
    sh.coefficients[:] = 1.0
    cls = [oracle.cart_list(l) for l in ls]
    ref = refquad.eri_cart_quadrature(ls, sh.exponents, sh.centers, cls)
    got = oracle.quartet(sh, 0, 1, 2, 3, solid=False).astype(float)
    assert np.abs(got - ref).max() <= 5e-13 * np.abs(ref).max()


@pytest.mark.slow
def test_iiii_vs_bruteforce_quadrature():
    ls = (6, 6, 6, 6)
    cls = [oracle.cart_list(6)] * 4
    ref = refquad.eri_cart_quadrature(ls, ZETA, CENT, cls)
    got = oracle.quartet(_example([6] * 4), 0, 1, 2, 3, solid=False).astype(float)
    assert np.abs(got - ref).max() <= 5e-13 * np.abs(ref).max()


def test_solid_block_vs_quadrature_and_independent_transform(recurrence_S):
    """Solid-harmonic (dd|pd) block == quadrature Cartesians transformed with the RECURRENCE table."""
    S, syms = recurrence_S
    ls = (2, 2, 1, 2)
    rng = np.random.default_rng(3)
    sh = _rand_shells(rng, list(ls), box=1.5, lo=0.4, hi=2.0)
    cls = [oracle.cart_list(l) for l in ls]
    cart = refquad.eri_cart_quadrature(ls, sh.exponents, sh.centers, cls) * np.prod(sh.coefficients)
    Cs = [refquad.solid_coeff_table(l, cl, S, syms).astype(float) for l, cl in zip(ls, cls)]
    ref = np.einsum("ai,bj,ck,dl,ijkl->abcd", *Cs, cart)
    got = oracle.quartet(sh, 0, 1, 2, 3).astype(float)
    assert np.abs(got - ref).max() <= 5e-13 * np.abs(ref).max()


def test_contraction_is_sum_of_primitives():
    rng = np.random.default_rng(21)
    K = (2, 3, 1, 2)
    sh = _rand_shells(rng, [2, 1, 1, 0], K=K)
    tot = oracle.quartet(sh, 0, 1, 2, 3)
    acc = np.zeros_like(tot)
    off = sh.prim_offset
    for ka in range(K[0]):
        for kb in range(K[1]):
            for kc in range(K[2]):
                for kd in range(K[3]):
                    idx = [off[0] + ka, off[1] + kb, off[2] + kc, off[3] + kd]
                    one = oracle.Shells(sh.centers, sh.l, [0, 1, 2, 3, 4], sh.exponents[idx], sh.coefficients[idx])
                    acc += oracle.quartet(one, 0, 1, 2, 3)
    assert np.abs(acc - tot).max() <= 1e-17 * np.abs(tot).max()


@pytest.mark.parametrize("ls", [(2, 1, 3, 0), (4, 3, 2, 1), (5, 4, 4, 4)])
def test_eightfold_symmetry(ls):
    """(ab|cd) = (ba|cd) = (ab|dc) = (cd|ab) with the m indices permuted."""
    rng = np.random.default_rng(31 + sum(ls))
    sh = _rand_shells(rng, list(ls), K=(2, 1, 1, 2))
    q = oracle.quartet(sh, 0, 1, 2, 3)
    tol = 1e-12 * np.abs(q).max()   # different recursion paths; rounding only
    assert np.abs(oracle.quartet(sh, 1, 0, 2, 3) - q.transpose(1, 0, 2, 3)).max() <= tol
    assert np.abs(oracle.quartet(sh, 0, 1, 3, 2) - q.transpose(0, 1, 3, 2)).max() <= tol
    assert np.abs(oracle.quartet(sh, 2, 3, 0, 1) - q.transpose(2, 3, 0, 1)).max() <= tol
    assert np.abs(oracle.quartet(sh, 3, 2, 1, 0) - q.transpose(3, 2, 1, 0)).max() <= tol


def test_translation_invariance():
    rng = np.random.default_rng(41)
    sh = _rand_shells(rng, [3, 2, 4, 1], K=(1, 2, 1, 1))
    q = oracle.quartet(sh, 0, 1, 2, 3)
    sh2 = oracle.Shells(sh.centers + np.array([0.7, -1.3, 2.1]), sh.l, sh.prim_offset, sh.exponents, sh.coefficients)
    assert np.abs(oracle.quartet(sh2, 0, 1, 2, 3) - q).max() <= 1e-13 * np.abs(q).max()


def test_rotation_norm_invariance():
    """Real solid harmonics of fixed l transform orthogonally under rotation -> Frobenius norm of a quartet is
    invariant under a common rotation of all centres (pins the S_lm tables at l = 4..6)."""
    rng = np.random.default_rng(51)
    A = rng.normal(size=(3, 3))
    Rm, _ = np.linalg.qr(A)
    if np.linalg.det(Rm) < 0:
        Rm[:, 0] *= -1
    for ls in ((4, 4, 4, 4), (6, 5, 4, 6)):
        sh = _rand_shells(rng, list(ls))
        q = oracle.quartet(sh, 0, 1, 2, 3)
        sh2 = oracle.Shells(sh.centers @ Rm.T, sh.l, sh.prim_offset, sh.exponents, sh.coefficients)
        q2 = oracle.quartet(sh2, 0, 1, 2, 3)
        n1, n2 = np.sqrt((q ** 2).sum()), np.sqrt((q2 ** 2).sum())
        assert abs(n1 - n2) <= 1e-12 * n1
        assert np.abs(q - q2).max() > 1e-3 * np.abs(q).max()    # the rotation really changed the components


def test_scaling_relation():
    """Centres x lam, exponents x lam^-2 multiplies unnormalised integrals by lam^(la+lb+lc+ld+5)."""
    rng = np.random.default_rng(61)
    ls = [3, 2, 2, 1]
    sh = _rand_shells(rng, ls)
    lam = 1.7
    sh2 = oracle.Shells(sh.centers * lam, sh.l, sh.prim_offset, sh.exponents / lam ** 2, sh.coefficients)
    q, q2 = oracle.quartet(sh, 0, 1, 2, 3), oracle.quartet(sh2, 0, 1, 2, 3)
    assert np.abs(q2 - q * np.longdouble(lam) ** (sum(ls) + 5)).max() <= 1e-13 * np.abs(q2).max()


def test_one_centre_selection_rule():
    """A = B = C = D, s shells on a and b: (ss|lm, l'm') is diagonal, and for l = l' independent of m."""
    c = [[0.3, -0.2, 0.5]] * 4
    for l, lp in ((3, 3), (4, 4), (2, 4), (3, 5)):
        sh = oracle.Shells(c, [0, 0, l, lp], [0, 1, 2, 3, 4], [0.8, 1.1, 0.6, 1.4], [1, 1, 1, 1])
        q = oracle.quartet(sh, 0, 1, 2, 3)[0, 0]
        scale = np.abs(oracle.quartet(oracle.Shells(c, [0, 0, l, l], [0, 1, 2, 3, 4], [0.8, 1.1, 0.6, 1.4], [1] * 4), 0, 1, 2, 3)).max()
        if l == lp:
            d = np.diag(q)
            assert np.abs(q - np.diag(d)).max() <= 1e-16 * scale
            assert np.abs(d - d[0]).max() <= 1e-16 * scale and abs(d[0]) > 0
        else:
            assert np.abs(q).max() <= 1e-16 * scale


def test_paper_size_statements():
    """Counts printed in the paper against the generator's size helpers."""
    from paper_2307_03452_b200 import inputs as I

    vals = {ln.split()[0]: float(ln.split()[1]) for ln in open(os.path.join(GOLD, "paper_sizes.txt")) if not ln.startswith("#")}
    assert I.n_hermite(6) == vals["n_hermite_lbra6"] and I.n_hermite(6) ** 2 * 8 == vals["ffff_2index_bytes"]
    assert I.n_hermite(12) == vals["n_hermite_L12"] and I.n_hermite(12) * 8 == vals["ffff_1index_bytes"]
    assert I.n_hermite(6) * 49 == vals["H_f_elems"] and I.n_hermite(6) * 49 * 8 == vals["H_f_bytes"]
    assert 3 * 5 ** 4 * 9 * 8 == vals["rys_gggg_bytes"]

    def intensity(l):   # PAPER.md:151 Eq.19
        nab = ncd = I.n_solid(l) ** 2
        np_ = nq = I.n_hermite(2 * l)
        return 0.25 * nab * nq * (np_ + ncd) / (2 * np_ * nq + nab * (np_ + 2 * nq + ncd) + ncd * nq)

    assert round(intensity(6), 1) == vals["intensity_iiii"] and round(intensity(3), 1) == vals["intensity_ffff"]
    # FLOP count of SURVEY.md 8(d)
    assert I.class_flops((6, 6, 6, 6), (1, 1, 1, 1)) == 95964960
    assert I.class_flops((6, 6, 6, 6), (5, 5, 5, 5)) == 44383794000
    assert I.class_flops((4, 4, 4, 4), (1, 1, 1, 1)) == 6575580


# ------------------------------------------------- hard geometries: tight/diffuse pairs far from their partners
def _config1_shells():
    from paper_2307_03452_b200 import inputs as I

    wl = I.config1()
    s = wl.shells
    return oracle.Shells(s.centers, s.l, s.prim_offset, s.exponents, s.coefficients)


def test_hard_geometry_vs_40_digit_md():
    """BASELINE config 1, bra (0,1) x ket (5,4): zeta = (0.156, 8.24 | 0.136, 10.4), |CD| = 6.5 bohr, T = 215.
    With the horizontal recurrence always moving momentum from the first to the second centre the long-double
    oracle was wrong by 4e-3 here.  Reference: the paper's MD form at 40 digits (tests/mpmd.py), a third route."""
    import mpmd

    sh = _config1_shells()
    rows = [(0, 0), (4, 4), (8, 1), (3, 7), (6, 2)]
    ref = mpmd.mp_quartet_rows(sh, 0, 1, 5, 4, rows)
    for quad, tol in ((True, 1e-15), (False, 1e-11)):
        q = oracle.quartet(sh, 0, 1, 5, 4, quad=quad).astype(np.float64)
        got = np.stack([q[a, b] for a, b in rows])
        assert np.abs(got - ref).max() <= tol * np.abs(q).max(), (quad, np.abs(got - ref).max() / np.abs(q).max())


def test_building_centre_choice_is_symmetric():
    """(ab|cd) = (ba|cd) = (cd|ab) on a hard geometry, in both builds; equal exponents (tie) included."""
    cent = [[0, 0, 0], [0, 0, 5.0], [4.0, 1.0, 0], [4.0, 1.0, 0.7]]
    for zs in ([0.12, 9.0, 11.0, 0.2], [0.5, 0.5, 3.0, 3.0]):
        sh = oracle.Shells(cent, [4, 3, 3, 4], [0, 1, 2, 3, 4], zs, [1, 1, 1, 1])
        for quad, tol in ((True, 1e-25), (False, 1e-12)):
            q = oracle.quartet(sh, 0, 1, 2, 3, quad=quad)
            mx = np.abs(q).max()
            assert np.abs(oracle.quartet(sh, 2, 3, 0, 1, quad=quad) - q.transpose(2, 3, 0, 1)).max() <= max(tol, 2e-18) * mx
            assert np.abs(oracle.quartet(sh, 1, 0, 3, 2, quad=quad) - q.transpose(1, 0, 3, 2)).max() <= max(tol, 2e-18) * mx


def test_batch_driver_slices_and_precisions():
    """oracle.compute: primitive slices add up to the unsliced result; binary128 and long-double builds agree on a
    benign contracted geometry; subset addressing."""
    rng = np.random.default_rng(77)
    sh = _rand_shells(rng, [2, 1, 2, 1], K=(3, 2, 2, 3))
    bra, ket = np.array([[0, 1], [1, 0]], dtype=np.int32), np.array([[2, 3]], dtype=np.int32)
    sh2 = oracle.Shells(np.concatenate([sh.centers]), sh.l, sh.prim_offset, sh.exponents, sh.coefficients)
    # bra pair (1,0) has (l1,l0) = (1,2): lists must share a class, so use two lists of one pair each
    for b in (bra[:1], bra[1:]):
        full = oracle.compute(sh2, b, ket, nthreads=2)
        sliced = oracle.compute(sh2, b, ket, nthreads=3, nslice=5)
        ld = oracle.compute(sh2, b, ket, nthreads=2, precision="ld")
        assert np.abs(full - sliced).max() <= 1e-16 * np.abs(full).max()
        assert np.abs(full - ld).max() <= 1e-15 * np.abs(full).max()
        one = oracle.quartet(sh2, int(b[0, 0]), int(b[0, 1]), 2, 3, quad=True).astype(np.float64)
        assert np.array_equal(full[0, 0], one)
        sub = oracle.compute(sh2, b, ket, subset=[0], nthreads=1)
        assert np.array_equal(sub[0], full[0, 0])


def test_batch_driver_addressing_on_ragged_lists():
    """oracle.compute writes out[i_bra][j_ket] (the md4_compute layout, include/md4.h): a 2 x 3 list with distinct
    shells on every pair, each slot against its own oracle.quartet call (the per-quartet routine is what the other
    pins check); an i/j transposition or a wrong stride in the batch driver would fail here.  Also the subset form
    out[k] = quartet subset[k] in the caller's order, and sliced primitive loops on the same lists."""
    rng = np.random.default_rng(78)
    n = 6
    cent = rng.uniform(0, 2.5, (n, 3))
    ls = np.array([2, 2, 2, 1, 1, 1], dtype=np.int32)           # bra pairs (d,p), ket pairs (p,d)
    K = [1, 2, 1, 2, 1, 1]                                      # shells 1 and 3 (unused) shift the primitive offsets
    off = np.concatenate([[0], np.cumsum(K)]).astype(np.int32)
    ex = np.exp(rng.uniform(math.log(0.3), math.log(3.0), off[-1]))
    co = rng.uniform(0.3, 1.0, off[-1])
    sh = oracle.Shells(cent, ls, off, ex, co)
    bra = np.array([[0, 4], [2, 5]], dtype=np.int32)           # both (l=2,K=1 | l=1,K=1)
    ket = np.array([[4, 0], [5, 2], [4, 2]], dtype=np.int32)   # all (l=1,K=1 | l=2,K=1), three different pairs
    full = oracle.compute(sh, bra, ket, nthreads=3)
    assert full.shape == (2, 3, 5, 3, 3, 5)
    for i, (a, b) in enumerate(bra):
        for j, (c, d) in enumerate(ket):
            one = oracle.quartet(sh, int(a), int(b), int(c), int(d), quad=True).astype(np.float64)
            assert np.array_equal(full[i, j], one), (i, j)
    # the six quartets are pairwise different, so a transposed or shifted slot cannot pass by accident
    flat = full.reshape(6, -1)
    for x in range(6):
        for y in range(x + 1, 6):
            assert np.abs(flat[x] - flat[y]).max() > 1e-6 * np.abs(flat[x]).max()
    order = [5, 0, 3]
    sub = oracle.compute(sh, bra, ket, subset=order, nthreads=2)
    for k, f in enumerate(order):
        assert np.array_equal(sub[k], full[f // 3, f % 3])
    sliced = oracle.compute(sh, bra, ket, subset=order, nthreads=4, nslice=3)
    assert np.abs(sliced - sub).max() <= 1e-16 * np.abs(sub).max()


# ------------------------------------------------ non-Coulomb kernels (ref. 21)
@pytest.fixture
def coulomb_after():
    yield
    oracle.set_kernel("coulomb")


def test_kernel_seeds_vs_truncated_boys_integral(coulomb_after):
    """G_m = Int_0^s y^2m exp(-T y^2) dy (erf), Int_s^1 (erfc), s^2 = omega^2/(omega^2 + rho): mpmath quadrature of the
    defining integral at 30 digits (library routine) against the oracle's s^(2m+1) F_m(s^2 T) form."""
    import mpmath as mp

    mp.mp.dps = 30
    for omega, rho, T in [(0.3, 0.7, 0.0), (0.3, 0.7, 2.5), (1.1, 0.05, 40.0), (0.2, 25.0, 130.0), (5.0, 1.0, 9.0)]:
        s = mp.sqrt(mp.mpf(omega) ** 2 / (mp.mpf(omega) ** 2 + mp.mpf(rho)))
        for kind, (lo, hi) in (("erf", (0, s)), ("erfc", (s, 1))):
            oracle.set_kernel(kind, omega)
            G = oracle.kernel_seeds(12, rho, T)
            for m in (0, 1, 5, 12):
                ref = mp.quad(lambda y: y ** (2 * m) * mp.exp(-mp.mpf(T) * y * y), [lo, hi])
                got = mp.mpf(np.format_float_scientific(G[m], precision=25, unique=False))
                # a few long-double ulps of the value, plus (erfc is a difference) of the full Boys integral it is cut from
                full = mp.quad(lambda y: y ** (2 * m) * mp.exp(-mp.mpf(T) * y * y), [0, 1])
                assert abs(got - ref) <= mp.mpf("1e-17") * abs(ref) + mp.mpf("5e-19") * full, (kind, omega, rho, T, m)


@pytest.mark.parametrize("kind", ["erf", "erfc"])
@pytest.mark.parametrize("ls", [(0, 0, 0, 0), (1, 1, 1, 1), (2, 1, 0, 2)])
def test_attenuated_kernels_vs_bruteforce_quadrature(coulomb_after, kind, ls):
    """(ab|cd) with erf(omega r12)/r12 and erfc(omega r12)/r12 against the brute-force quadrature of refquad.py with the
    u-integral of 1/r12 = (2/sqrt pi) Int exp(-u^2 r12^2) du cut at omega: uses neither Boys nor any recurrence."""
    rng = np.random.default_rng(91)
    sh = _rand_shells(rng, list(ls))
    omega = 0.6
    oracle.set_kernel(kind, omega)
    got = oracle.quartet(sh, 0, 1, 2, 3, solid=False).astype(np.float64) / np.prod(sh.coefficients)
    cls = [oracle.cart_list(l) for l in ls]
    ref = refquad.eri_cart_quadrature(ls, sh.exponents, sh.centers, cls, kernel=kind, omega=omega, ngl=160)
    assert np.abs(got - ref).max() <= 2e-12 * np.abs(ref).max(), np.abs(got - ref).max() / np.abs(ref).max()


def test_attenuated_kernels_sum_and_limits(coulomb_after):
    """erf + erfc = Coulomb element by element; omega -> infinity: erf -> Coulomb, erfc -> 0; omega -> 0: erf -> 0
    like omega (2/sqrt pi) omega times the overlap-type integral, checked as a ratio of two small omegas."""
    rng = np.random.default_rng(92)
    sh = _rand_shells(rng, [3, 2, 2, 1], K=(2, 1, 1, 2))
    oracle.set_kernel("coulomb")
    c = oracle.quartet(sh, 0, 1, 2, 3, quad=True)
    oracle.set_kernel("erf", 0.45)
    e = oracle.quartet(sh, 0, 1, 2, 3, quad=True)
    oracle.set_kernel("erfc", 0.45)
    ec = oracle.quartet(sh, 0, 1, 2, 3, quad=True)
    scale = np.abs(c).max()
    assert np.abs(e + ec - c).max() <= 1e-17 * scale
    assert np.abs(e).max() > 1e-3 * scale and np.abs(ec).max() > 1e-3 * scale      # both parts matter at this omega
    oracle.set_kernel("erf", 1e6)
    assert np.abs(oracle.quartet(sh, 0, 1, 2, 3, quad=True) - c).max() <= 1e-10 * scale
    oracle.set_kernel("erf", 1e-5)
    a = oracle.quartet(sh, 0, 1, 2, 3, quad=True)
    oracle.set_kernel("erf", 2e-5)
    b = oracle.quartet(sh, 0, 1, 2, 3, quad=True)
    big = np.abs(a) > 1e-3 * np.abs(a).max()
    assert np.abs(b[big] / a[big] - 2.0).max() <= 1e-6      # next order: omega^2 r12^2


# ------------------------------------------------ direct digestion
def test_digest_jk_hand_computed_s_shells():
    """Four s shells, bra list [(0,1),(2,0)], ket list [(2,3),(1,1)]: J and K by hand from the closed form
    (ss|ss) = K_ab K_cd 2 pi^{5/2}/(p q sqrt(p+q)) F_0(T), F_0 = sqrt(pi/T) erf(sqrt T)/2 (math.erf), summed quartet by
    quartet in this test -- not by the oracle's contraction code."""
    rng = np.random.default_rng(5)
    cent = rng.uniform(0, 2.0, (4, 3))
    ex = np.array([0.8, 1.3, 0.5, 2.1])
    co = np.array([0.7, 1.1, 0.9, 0.6])
    sh = oracle.Shells(cent, [0, 0, 0, 0], [0, 1, 2, 3, 4], ex, co)
    D = rng.uniform(-1, 1, (4, 4))
    bra, ket = [(0, 1), (2, 0)], [(2, 3), (1, 1)]

    def ssss(a, b, c, d):
        p, q = ex[a] + ex[b], ex[c] + ex[d]
        P = (ex[a] * cent[a] + ex[b] * cent[b]) / p
        Q = (ex[c] * cent[c] + ex[d] * cent[d]) / q
        kab = math.exp(-ex[a] * ex[b] / p * ((cent[a] - cent[b]) ** 2).sum())
        kcd = math.exp(-ex[c] * ex[d] / q * ((cent[c] - cent[d]) ** 2).sum())
        T = p * q / (p + q) * ((P - Q) ** 2).sum()
        f0 = 1.0 if T == 0 else 0.5 * math.sqrt(math.pi / T) * math.erf(math.sqrt(T))
        return co[a] * co[b] * co[c] * co[d] * kab * kcd * 2 * math.pi ** 2.5 / (p * q * math.sqrt(p + q)) * f0

    Jh, Kh = np.zeros((4, 4)), np.zeros((4, 4))
    for a, b in bra:
        for c, d in ket:
            v = ssss(a, b, c, d)
            Jh[a, b] += v * D[c, d]
            Kh[a, c] += v * D[b, d]
    J, K = oracle.digest_jk(sh, bra, ket, D)
    assert np.abs(J.astype(float) - Jh).max() <= 1e-14 * np.abs(Jh).max()
    assert np.abs(K.astype(float) - Kh).max() <= 1e-14 * np.abs(Kh).max()
    assert np.count_nonzero(Jh) == 2 and np.count_nonzero(Kh) == 4      # only the listed blocks are touched


def test_digest_jk_index_roles_with_unit_densities():
    """(dp|pd)-type shells with a density that is 1 in ONE element: J then is one (c,d) slice of the quartet and K one
    (b,d) slice, taken here straight from oracle.quartet -- a swapped pair of indices in the contraction would fail."""
    rng = np.random.default_rng(6)
    sh = _rand_shells(rng, [2, 1, 1, 2])
    off = oracle.ao_offsets(sh)
    g = oracle.quartet(sh, 0, 1, 2, 3, quad=True).astype(np.float64)      # [5, 3, 3, 5]
    nbf = int(off[-1])
    mc, md, mb = 2, 3, 1
    D = np.zeros((nbf, nbf)); D[off[2] + mc, off[3] + md] = 1.0
    J, K = oracle.digest_jk(sh, [(0, 1)], [(2, 3)], D)
    assert np.array_equal(J[off[0]:off[1], off[1]:off[2]].astype(float), g[:, :, mc, md]) and np.abs(K).max() == 0
    D = np.zeros((nbf, nbf)); D[off[1] + mb, off[3] + md] = 1.0
    J, K = oracle.digest_jk(sh, [(0, 1)], [(2, 3)], D)
    assert np.array_equal(K[off[0]:off[1], off[2]:off[3]].astype(float), g[:, mb, :, md]) and np.abs(J).max() == 0

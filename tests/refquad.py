"""Independent references used ONLY to pin the oracle (tests, CPU).

1. ``eri_cart_quadrature``: brute-force quadrature of a primitive Cartesian (ab|cd) block that uses neither the
   Boys function, nor Hermite E/R recurrences, nor Obara-Saika (SURVEY.md 8(c) "pins" item 3):
       1/r12 = (2/sqrt(pi)) Int_0^inf exp(-u^2 r12^2) du,
   so [ab|cd] = (2/sqrt(pi)) Int du  prod_{i=x,y,z} I_i(u), with I_i(u) the 2-D integral over (x1, x2) of
   polynomial x exp(-quadratic form), done EXACTLY by tensor Gauss-Hermite after completing the square
   (M = [[p+u^2, -u^2], [-u^2, q+u^2]], Cholesky, affine map), and the u-integral by Gauss-Legendre in
   t in (0,1), u^2 = rho t^2 / (1 - t^2).
2. ``solid_harmonics_recurrence``: real solid harmonics S_lm (Racah normalisation) as exact sympy polynomials
   built by the textbook recurrences in l (a different route from the closed form the oracle uses).
"""
from __future__ import annotations

import math

import numpy as np


def _axis_integrals(la, lb, lc, ld, za, zb, zc, zd, A, B, C, D, u2, ngh):
    """I(u)[nt, a, b, c, d] for one Cartesian axis; A,B,C,D scalars; u2 array [nt]."""
    p, q = za + zb, zc + zd
    P, Q = (za * A + zb * B) / p, (zc * C + zd * D) / q
    kab = math.exp(-za * zb / p * (A - B) ** 2)
    kcd = math.exp(-zc * zd / q * (C - D) ** 2)
    d = P - Q
    x, w = np.polynomial.hermite.hermgauss(ngh)          # weight exp(-x^2)
    nt = u2.shape[0]
    out = np.zeros((nt, la + 1, lb + 1, lc + 1, ld + 1))
    for it in range(nt):
        s = u2[it]
        M = np.array([[p + s, -s], [-s, q + s]])
        # exponent: -(y^T M y + 2 s d (y1 - y2) + s d^2), y = (x1-P, x2-Q); centre y0 solves M y0 = -s d (1,-1)
        y0 = np.linalg.solve(M, -s * d * np.array([1.0, -1.0]))
        const = s * d * d - y0 @ M @ y0
        Lc = np.linalg.cholesky(M)                       # M = Lc Lc^T ; w = Lc^T z ; z = Lc^-T w
        LinvT = np.linalg.inv(Lc).T
        W1, W2 = np.meshgrid(x, x, indexing="ij")
        Z1 = LinvT[0, 0] * W1 + LinvT[0, 1] * W2
        Z2 = LinvT[1, 0] * W1 + LinvT[1, 1] * W2
        X1 = P + y0[0] + Z1
        X2 = Q + y0[1] + Z2
        wt = np.outer(w, w) * math.exp(-const) / abs(np.linalg.det(Lc)) * kab * kcd
        pa = np.stack([(X1 - A) ** k for k in range(la + 1)]).reshape(la + 1, -1)
        pb = np.stack([(X1 - B) ** k for k in range(lb + 1)]).reshape(lb + 1, -1)
        pc = np.stack([(X2 - C) ** k for k in range(lc + 1)]).reshape(lc + 1, -1)
        pd = np.stack([(X2 - D) ** k for k in range(ld + 1)]).reshape(ld + 1, -1)
        fab = (pa[:, None, :] * pb[None, :, :]).reshape(-1, pa.shape[1]) * wt.reshape(1, -1)
        fcd = (pc[:, None, :] * pd[None, :, :]).reshape(-1, pa.shape[1])
        out[it] = (fab @ fcd.T).reshape(la + 1, lb + 1, lc + 1, ld + 1)
    return out


def eri_cart_quadrature(ls, zs, centers, cart_lists, ngl=120, ngh=None, kernel="coulomb", omega=None):
    """Unnormalised primitive Cartesian block [a b|c d]: array [na, nb, nc, nd] in the order of ``cart_lists``
    (four lists of (x,y,z) exponent triples).  kernel: "coulomb" 1/r12; "erf": erf(omega r12)/r12 = (2/sqrt(pi))
    Int_0^omega exp(-u^2 r12^2) du, i.e. the same u-integral cut at u = omega (t <= omega/sqrt(rho + omega^2));
    "erfc": the rest of the u-range."""
    la, lb, lc, ld = ls
    za, zb, zc, zd = zs
    A, B, C, D = [np.asarray(c, dtype=float) for c in centers]
    if ngh is None:
        ngh = (la + lb + lc + ld) // 2 + 4
    p, q = za + zb, zc + zd
    rho = p * q / (p + q)
    t, wt = np.polynomial.legendre.leggauss(ngl)
    t0, t1 = 0.0, 1.0
    if kernel != "coulomb":
        tc = omega / math.sqrt(rho + omega * omega)
        t0, t1 = (0.0, tc) if kernel == "erf" else (tc, 1.0)
    t = t0 + (t1 - t0) * 0.5 * (t + 1.0)
    wt = (t1 - t0) * 0.5 * wt
    u2 = rho * t * t / (1.0 - t * t)
    dudt = math.sqrt(rho) * (1.0 - t * t) ** -1.5
    I = [_axis_integrals(la, lb, lc, ld, za, zb, zc, zd, A[i], B[i], C[i], D[i], u2, ngh) for i in range(3)]
    ca, cb, cc, cd = [np.array(cl) for cl in cart_lists]
    out = np.zeros((len(ca), len(cb), len(cc), len(cd)))
    ix = np.ix_
    for it in range(ngl):
        g = np.ones_like(out)
        for i in range(3):
            g = g * I[i][it][ix(ca[:, i], cb[:, i], cc[:, i], cd[:, i])]
        out += (2.0 / math.sqrt(math.pi)) * wt[it] * dudt[it] * g
    return out


def solid_harmonics_recurrence(lmax):
    """dict (l, m) -> sympy polynomial in x, y, z for the Racah-normalised real solid harmonics, by recurrence:
       S_00 = 1
       S_{l+1, l+1}  = sqrt(2^{d_l0} (2l+1)/(2l+2)) (x S_{l,l} - (1-d_l0) y S_{l,-l})
       S_{l+1,-l-1}  = sqrt(2^{d_l0} (2l+1)/(2l+2)) (y S_{l,l} + (1-d_l0) x S_{l,-l})
       S_{l+1, m}    = [(2l+1) z S_{l,m} - sqrt((l+m)(l-m)) r^2 S_{l-1,m}] / sqrt((l+m+1)(l-m+1)),  |m| <= l
    (Helgaker, Jorgensen, Olsen, Molecular Electronic-Structure Theory, sec. 6.4.2)."""
    import sympy as sp

    x, y, z = sp.symbols("x y z")
    r2 = x * x + y * y + z * z
    S = {(0, 0): sp.Integer(1)}
    for l in range(lmax):
        d0 = 1 if l == 0 else 0
        f = sp.sqrt(sp.Rational(2 ** d0 * (2 * l + 1), 2 * l + 2))
        S[(l + 1, l + 1)] = sp.expand(f * (x * S[(l, l)] - (1 - d0) * y * S[(l, -l)]))
        S[(l + 1, -l - 1)] = sp.expand(f * (y * S[(l, l)] + (1 - d0) * x * S[(l, -l)]))
        for m in range(-l, l + 1):
            prev = S[(l - 1, m)] if abs(m) <= l - 1 else 0
            S[(l + 1, m)] = sp.expand(((2 * l + 1) * z * S[(l, m)] - sp.sqrt((l + m) * (l - m)) * r2 * prev)
                                      / sp.sqrt((l + m + 1) * (l - m + 1)))
    return S, (x, y, z)


def solid_coeff_table(l, cart_list, S=None, syms=None, prec=30):
    """C[m+l][k] from the recurrence polynomials as mpmath/float values in the order of cart_list."""
    import sympy as sp

    if S is None:
        S, syms = solid_harmonics_recurrence(l)
    x, y, z = syms
    tab = np.zeros((2 * l + 1, len(cart_list)), dtype=np.longdouble)
    for m in range(-l, l + 1):
        poly = sp.Poly(S[(l, m)], x, y, z)
        for k, (ex, ey, ez) in enumerate(cart_list):
            c = poly.coeff_monomial(x ** ex * y ** ey * z ** ez)
            tab[m + l, k] = np.longdouble(str(sp.N(c, prec)))
    return tab

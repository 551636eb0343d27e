"""40-digit (mpmath) McMurchie-Davidson reference, written out from the paper's equations: test infrastructure.

mp_R  : Hermite Coulomb tensor R^{(0)}_{tuv} by Eq.10-13, Boys function from mpmath's incomplete
        gamma (a library routine).
mp_H  : H = c_a c_b C_la (x) C_lb E for one primitive pair, E by Eq.4-5, Eq.16
        with the oracle's solid-harmonic table.
mp_quartet : (ab|cd) of one uncontracted shell quartet by Eq.6-8 + Eq.14-15 at 40 digits -- a third route,
        independent of the OS/HGP recurrences of the oracle and of the CUDA kernels (which it shares no code with).
Used by tests only.
"""
import numpy as np

import oracle


def mp_R_dict(L, zp, P, zq, Q, kernel="coulomb", omega=None):
    """{(t,u,v): R^{(0)}_{tuv}} as mpmath numbers, t+u+v <= L; prefactor 2 pi^{5/2}/(zp zq sqrt(zp+zq)) included.
    kernel "erf" / "erfc": seeds from the truncated Boys integral Int y^2m exp(-T y^2) dy over [0, s] / [s, 1],
    s^2 = omega^2/(omega^2 + rho), by mpmath quadrature of that definition (ref. 21)."""
    import mpmath as mp

    mp.mp.dps = 40
    zp, zq = mp.mpf(zp), mp.mpf(zq)
    X = [mp.mpf(a) - mp.mpf(b) for a, b in zip(P, Q)]
    rho = zp * zq / (zp + zq)
    T = rho * sum(x * x for x in X)
    pref = 2 * mp.pi ** mp.mpf(2.5) / (zp * zq * mp.sqrt(zp + zq))

    def F(m):
        if kernel != "coulomb":
            s = mp.sqrt(mp.mpf(omega) ** 2 / (mp.mpf(omega) ** 2 + rho))
            lo, hi = (0, s) if kernel == "erf" else (s, 1)
            return mp.quad(lambda y: y ** (2 * m) * mp.exp(-T * y * y), [lo, hi])
        if T == 0:
            return mp.mpf(1) / (2 * m + 1)
        return mp.gammainc(m + mp.mpf(1) / 2, 0, T) / (2 * T ** (m + mp.mpf(1) / 2))

    # R[m][(t,u,v)], Helgaker-style: R^m_{t+1} = t R^{m+1}_{t-1} + X R^{m+1}_t  (Eq.13)
    R = {}
    for m in range(L + 1):
        R[(m, 0, 0, 0)] = pref * (-2 * rho) ** m * F(m)
    for n in range(1, L + 1):
        for t in range(n + 1):
            for u in range(n - t + 1):
                v = n - t - u
                for m in range(L - n + 1):
                    if t > 0:
                        val = X[0] * R[(m + 1, t - 1, u, v)] + ((t - 1) * R[(m + 1, t - 2, u, v)] if t > 1 else 0)
                    elif u > 0:
                        val = X[1] * R[(m + 1, t, u - 1, v)] + ((u - 1) * R[(m + 1, t, u - 2, v)] if u > 1 else 0)
                    else:
                        val = X[2] * R[(m + 1, t, u, v - 1)] + ((v - 1) * R[(m + 1, t, u, v - 2)] if v > 1 else 0)
                    R[(m, t, u, v)] = val
    return {k[1:]: val for k, val in R.items() if k[0] == 0}


def mp_R(L, zp, P, zq, Q, kernel="coulomb", omega=None):
    """R^{(0)}_{tuv} as a float array [L+1]^3 (entries with t+u+v > L are 0)."""
    R = mp_R_dict(L, zp, [float(x) for x in P], zq, [float(x) for x in Q], kernel, omega)
    out = np.zeros((L + 1,) * 3)
    for (t, u, v), val in R.items():
        out[t, u, v] = float(val)
    return out


def mp_H(sh, i, j, ka, kb):
    """H = c_a c_b C_la (x) C_lb E for one primitive pair, 40-digit E by Eq.4-5, oracle's solid tables."""
    import mpmath as mp

    mp.mp.dps = 40
    li, lj = int(sh.l[i]), int(sh.l[j])
    za = mp.mpf(float(sh.exponents[sh.prim_offset[i] + ka])); zb = mp.mpf(float(sh.exponents[sh.prim_offset[j] + kb]))
    ca = mp.mpf(float(sh.coefficients[sh.prim_offset[i] + ka])); cb = mp.mpf(float(sh.coefficients[sh.prim_offset[j] + kb]))
    A = [mp.mpf(float(x)) for x in sh.centers[i]]; B = [mp.mpf(float(x)) for x in sh.centers[j]]
    p = za + zb
    P = [(za * a + zb * b) / p for a, b in zip(A, B)]
    E = []
    for ax in range(3):
        e = {(0, 0, 0): mp.mpf(1)}
        g = lambda a_, b_, t_: e.get((a_, b_, t_), mp.mpf(0))
        for a_ in range(li):
            for t in range(a_ + 2):
                e[(a_ + 1, 0, t)] = g(a_, 0, t - 1) / (2 * p) + (P[ax] - A[ax]) * g(a_, 0, t) + (t + 1) * g(a_, 0, t + 1)
        for a_ in range(li + 1):
            for b_ in range(lj):
                for t in range(a_ + b_ + 2):
                    e[(a_, b_ + 1, t)] = g(a_, b_, t - 1) / (2 * p) + (P[ax] - B[ax]) * g(a_, b_, t) + (t + 1) * g(a_, b_, t + 1)
        E.append(e)
    Ca, Cb = oracle.solid_coeff(li), oracle.solid_coeff(lj)
    carta, cartb = oracle.cart_list(li), oracle.cart_list(lj)
    lb = li + lj
    herm = [(t, u, n - t - u) for n in range(lb + 1) for t in range(n, -1, -1) for u in range(n - t, -1, -1)]
    Ecart = np.zeros((len(carta), len(cartb), len(herm)), dtype=object)
    for ia, a in enumerate(carta):
        for ib, b in enumerate(cartb):
            for ih, (t, u, v) in enumerate(herm):
                Ecart[ia, ib, ih] = (E[0].get((a[0], b[0], t), 0) * E[1].get((a[1], b[1], u), 0) * E[2].get((a[2], b[2], v), 0))
    Ecart = np.array(Ecart, dtype=np.longdouble)
    H = np.einsum("ma,nb,abh->mnh", Ca, Cb, Ecart) * np.longdouble(float(ca * cb))
    mu = za * zb / p
    lnK = -mu * sum((a - b) ** 2 for a, b in zip(A, B))
    return H.reshape(-1, len(herm)).astype(np.float64), float(p), [float(x) for x in P], float(lnK)




def _mp_E_axis(la, lb, p, XPA, XPB):
    """(E_i)^t_{ab}, a <= la, b <= lb, by Eq.4-5, seed 1."""
    import mpmath as mp

    e = {(0, 0, 0): mp.mpf(1)}
    g = lambda a_, b_, t_: e.get((a_, b_, t_), mp.mpf(0))
    for a_ in range(la):
        for t in range(a_ + 2):
            e[(a_ + 1, 0, t)] = g(a_, 0, t - 1) / (2 * p) + XPA * g(a_, 0, t) + (t + 1) * g(a_, 0, t + 1)
    for a_ in range(la + 1):
        for b_ in range(lb):
            for t in range(a_ + b_ + 2):
                e[(a_, b_ + 1, t)] = g(a_, b_, t - 1) / (2 * p) + XPB * g(a_, b_, t) + (t + 1) * g(a_, b_, t + 1)
    return e


def _mp_solid_table(l, S, syms):
    """C[m+l][cartesian triple] at 40 digits from the exact sympy recurrence polynomials of tests/refquad.py."""
    import mpmath as mp
    import sympy as sp

    x, y, z = syms
    tab = []
    for m in range(-l, l + 1):
        poly = sp.Poly(S[(l, m)], x, y, z)
        tab.append({mono: mp.mpf(str(sp.N(c, 45))) for mono, c in zip(poly.monoms(), poly.coeffs())})
    return tab


def _mp_pair_H(sh, i, j, S, syms):
    """Rows (ma, mb) -> {hermite (t,u,v): H}, K_ab c_a c_b folded in; zeta_p; P (all mpmath, 40 digits)."""
    import mpmath as mp

    mp.mp.dps = 40
    li, lj = int(sh.l[i]), int(sh.l[j])
    assert sh.prim_offset[i + 1] - sh.prim_offset[i] == 1 and sh.prim_offset[j + 1] - sh.prim_offset[j] == 1
    za, zb = mp.mpf(float(sh.exponents[sh.prim_offset[i]])), mp.mpf(float(sh.exponents[sh.prim_offset[j]]))
    w = mp.mpf(float(sh.coefficients[sh.prim_offset[i]])) * mp.mpf(float(sh.coefficients[sh.prim_offset[j]]))
    A = [mp.mpf(float(x)) for x in sh.centers[i]]; B = [mp.mpf(float(x)) for x in sh.centers[j]]
    p = za + zb
    P = [(za * a + zb * b) / p for a, b in zip(A, B)]
    w *= mp.exp(-za * zb / p * sum((a - b) ** 2 for a, b in zip(A, B)))
    E = [_mp_E_axis(li, lj, p, P[k] - A[k], P[k] - B[k]) for k in range(3)]
    Ca, Cb = _mp_solid_table(li, S, syms), _mp_solid_table(lj, S, syms)
    lb = li + lj
    herm = [(t, u, n - t - u) for n in range(lb + 1) for t in range(n, -1, -1) for u in range(n - t, -1, -1)]
    rows = {}
    for ma in range(2 * li + 1):
        for mb in range(2 * lj + 1):
            row = {}
            for (ax, ay, az), ca in Ca[ma].items():
                for (bx, by, bz), cb in Cb[mb].items():
                    c = w * ca * cb
                    for (t, u, v) in herm:
                        if t > ax + bx or u > ay + by or v > az + bz:
                            continue
                        row[(t, u, v)] = row.get((t, u, v), 0) + c * E[0][(ax, bx, t)] * E[1][(ay, by, u)] * E[2][(az, bz, v)]
            rows[(ma, mb)] = row
    return rows, p, P


def mp_quartet_rows(sh, ia, ib, ic, id_, bra_rows):
    """(ab|cd)[(ma,mb) in bra_rows, mc, md] of one UNCONTRACTED shell quartet at 40 digits, by the paper's matrix
    McMurchie-Davidson form: Eq.6-8 + Eq.14-16.  Returns a float array [len(bra_rows), 2lc+1, 2ld+1]."""
    import mpmath as mp
    import refquad

    mp.mp.dps = 40
    lmax = int(max(sh.l[k] for k in (ia, ib, ic, id_)))
    S, syms = refquad.solid_harmonics_recurrence(max(lmax, 1))
    Hab, p, P = _mp_pair_H(sh, ia, ib, S, syms)
    Hcd, q, Q = _mp_pair_H(sh, ic, id_, S, syms)
    L = int(sh.l[ia] + sh.l[ib] + sh.l[ic] + sh.l[id_])
    R = mp_R_dict(L, p, P, q, Q)
    lc, ld = int(sh.l[ic]), int(sh.l[id_])
    out = np.zeros((len(bra_rows), 2 * lc + 1, 2 * ld + 1))
    for r, key in enumerate(bra_rows):
        hab = Hab[tuple(key)]
        # [ab|q~] = sum_p~ H_ab[p~] (-1)^{|q~|} R[p~+q~]   (Eq.8, Eq.14)
        herm_q = set()
        for row in Hcd.values():
            herm_q.update(row.keys())
        abq = {}
        for (t2, u2, v2) in herm_q:
            sgn = -1 if (t2 + u2 + v2) & 1 else 1
            abq[(t2, u2, v2)] = sgn * sum(h * R[(t + t2, u + u2, v + v2)] for (t, u, v), h in hab.items())
        for mc in range(2 * lc + 1):
            for md in range(2 * ld + 1):
                out[r, mc, md] = float(sum(h * abq[k] for k, h in Hcd[(mc, md)].items()))   # Eq.15
    return out

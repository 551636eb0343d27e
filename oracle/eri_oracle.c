/*
 * eri_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, extended-precision CPU evaluator of contracted 4-center 2-electron repulsion integrals
 * (ab|cd) over real-solid-harmonic Gaussian shells.  It is the parity oracle for the CUDA path of
 * this repository and shares no code, header, table or constant with it.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * What it computes (definition of the result; PAPER.md:49 Eq.1, :70 Eq.6, :109-113 Eq.16):
 *   (ab|cd)_{ma mb mc md} = sum_{ka kb kc kd} c_ka c_kb c_kc c_kd
 *        * Int Int chi^ka_{la ma}(r) chi^kb_{lb mb}(r) |r-r'|^-1 chi^kc_{lc mc}(r') chi^kd_{ld md}(r') d3r d3r'
 *   chi^k_{lm}(r) = S_lm(r-A) exp(-zeta_k |r-A|^2),  S_lm = real solid harmonic, Racah normalisation,
 *   coefficients applied verbatim to UNNORMALISED primitives.
 *
 * How (a different exact algorithm from the paper's matrix McMurchie-Davidson form, so that agreement
 * means something): Obara-Saika vertical recurrence + Head-Gordon-Pople horizontal recurrence, which
 * the paper cites as the reference CPU method (PAPER.md:19, :281-282 refs 18-19, :224 "OSHGP") but does
 * not print; the recurrences below are restated from those references and are pinned by the tests in
 * tests/test_oracle_*.py (closed form (ss|ss), Boys values, symmetries, scaling, one-centre rule,
 * brute-force quadrature that uses neither Boys nor any recurrence, and the worked example of
 * SURVEY.md 8(c) item 4).  No function in this file is "parity unpinned".
 *
 * Steps per shell quartet (SURVEY.md 8(c) "Oracle algorithm" 1-6):
 *   1. per primitive quartet: p, q, P, Q, W, rho, T, K_ab, K_cd
 *   2. seeds [00|00]^(m) = c_a c_b c_c c_d K_ab K_cd 2 pi^{5/2} / (p q sqrt(p+q)) F_m(T), m = 0..L
 *   3. vertical recurrence -> [e0|f0]^(m)
 *   4. contraction of the m = 0 values
 *   5. horizontal recurrence on contracted integrals
 *   6. 4-index Cartesian -> solid-harmonic transform
 * Step 5 moves momentum away from the centre with the larger exponent, chosen per primitive pair (see
 * quartet_cart): with a fixed direction the long-double result was wrong by 4e-3 on BASELINE config 1.
 *
 * Arithmetic type `real`.  Default build (liberi_oracle.so): long double (x87 80-bit on x86-64), the
 * precision BASELINE.json names; it serves the pins and the timed CPU baseline.  -DORACLE_QUAD build
 * (liberi_oracle_q.so): the same source in IEEE binary128 (libquadmath) -- THE PARITY REFERENCE.
 * Why: step 6 projects Cartesian integrals onto solid harmonics; for a tight shell of high l far from its
 * partner distribution the pure-l part is ~(s/R)^l of the Cartesian values (s = Gaussian width, R =
 * distance), e.g. 1e-8..1e-9 for l = 6, and those digits are lost whatever the order of the steps.
 * Measured on BASELINE config 3 (seeded sample of 10 quartets): long double vs binary128 differ by up to
 * 7.6e-11 of max|integral| -- too close to the 1e-10 parity bar -- so parity is taken against binary128
 * (error < 1e-24 by the same estimate).  Interfaces stay double / long double.
 */
#include <math.h>
#include <pthread.h>
#include <stdlib.h>
#include <string.h>

#ifdef ORACLE_QUAD
/* binary128 build (liberi_oracle_q.so): the parity reference, see the header. */
#include <quadmath.h>
typedef __float128 real;
#define R_EXP expq
#define R_SQRT sqrtq
#define R_ACOS acosq
#define R_POW powq
#else
typedef long double real;
#define R_EXP expl
#define R_SQRT sqrtl
#define R_ACOS acosl
#define R_POW powl
#endif

#define ORACLE_LMAX 8               /* per-shell l accepted by the oracle */
#define ORACLE_LTOT (4 * ORACLE_LMAX)
#define ORACLE_NCUM(n) (((n) * ((n) + 1) * ((n) + 2)) / 6) /* # Cartesian triples of degree < n */

/* ------------------------------------------------------------------------------------------------
 * Cartesian bookkeeping.  Triples (x,y,z) of degree n = x+y+z are ordered with x descending, then y
 * descending; the cumulative index over all degrees < n is n(n+1)(n+2)/6 (the pyramidal number of
 * PAPER.md:130).
 * ---------------------------------------------------------------------------------------------- */
static int cart_index(int x, int y, int z)
{
    int n = x + y + z, r = n - x;
    return ORACLE_NCUM(n) + r * (r + 1) / 2 + z;
}

#define ORACLE_NC_MAX ORACLE_NCUM(2 * ORACLE_LMAX + 1)
static int g_cx[ORACLE_NC_MAX], g_cy[ORACLE_NC_MAX], g_cz[ORACLE_NC_MAX];
static pthread_once_t g_once = PTHREAD_ONCE_INIT;

static void init_tables(void)
{
    for (int n = 0; n <= 2 * ORACLE_LMAX; ++n)
        for (int x = n; x >= 0; --x)
            for (int y = n - x; y >= 0; --y) {
                int z = n - x - y, i = cart_index(x, y, z);
                g_cx[i] = x; g_cy[i] = y; g_cz[i] = z;
            }
}

static int comp(int idx, int axis) { return axis == 0 ? g_cx[idx] : axis == 1 ? g_cy[idx] : g_cz[idx]; }
static int lower(int idx, int axis) /* index of the triple with one quantum less along axis */
{
    int x = g_cx[idx] - (axis == 0), y = g_cy[idx] - (axis == 1), z = g_cz[idx] - (axis == 2);
    return cart_index(x, y, z);
}
static int raise(int idx, int axis)
{
    int x = g_cx[idx] + (axis == 0), y = g_cy[idx] + (axis == 1), z = g_cz[idx] + (axis == 2);
    return cart_index(x, y, z);
}
static int first_axis(int idx) { return g_cx[idx] > 0 ? 0 : g_cy[idx] > 0 ? 1 : 2; }

/* ------------------------------------------------------------------------------------------------
 * Boys function F_m(T) = int_0^1 y^{2m} exp(-T y^2) dy, m = 0..mmax  (Eq.11).
 * The paper does not say how to evaluate it.  Oracle method:
 *   T <= 120 : F_M(T) = e^{-T} sum_{k>=0} (2T)^k / [(2M+1)(2M+3)...(2M+2k+1)]   (all terms positive),
 *              then downward F_m = (2T F_{m+1} + e^{-T}) / (2m+1);
 *   T  > 120 : F_m = Gamma(m+1/2) / (2 T^{m+1/2})  (complementary part < 1e-26 relative for m <= 32).
 * Pinned in tests against mpmath's incomplete gamma, erf closed form, F_m(0)=1/(2m+1) and the printed
 * 50-digit values of SURVEY.md Q11.
 * ---------------------------------------------------------------------------------------------- */
static void boys_real(int mmax, real T, real *F)
{
    if (T > 120.0L) {
        /* Gamma(m+1/2) = (2m-1)!! sqrt(pi) / 2^m */
        real g = R_SQRT(R_ACOS(-1.0L)); /* Gamma(1/2) */
        real tp = R_SQRT(T);            /* T^{m+1/2} */
        for (int m = 0; m <= mmax; ++m) {
            F[m] = g / (2.0L * tp);
            g *= (m + 0.5L);
            tp *= T;
        }
        return;
    }
    real eT = R_EXP(-T);
    real term = (real)1.0L / (2 * mmax + 1), sum = term;
    for (int k = 1; k < 4000; ++k) {
        term *= 2.0L * T / (2 * mmax + 2 * k + 1);
        sum += term;
        if (term < 1e-40L * sum) break;
    }
    F[mmax] = eT * sum;
    for (int m = mmax - 1; m >= 0; --m) F[m] = (2.0L * T * F[m + 1] + eT) / (2 * m + 1);
}

/* ------------------------------------------------------------------------------------------------
 * Interaction kernel g(r12) ("[0]^(m) is related to the Boys function (or similar quantities for
 * non-Coulomb integrals, ref. 21)").  Ref. 21 (Ahlrichs 2006) shows that for g(r) = Int w(u) exp(-u^2 r^2) du the
 * Obara-Saika recurrences are unchanged and only the seeds change: with y^2 = u^2/(rho + u^2),
 *     [00|00]^(m) = prefactor * G_m,   G_m = Int_0^1 w~(y) y^{2m} exp(-T y^2) dy.
 *   Coulomb 1/r:            w~ = 1 on [0,1]          G_m = F_m(T)
 *   erf(omega r)/r:         w~ = 1 on [0,s], else 0   G_m = s^{2m+1} F_m(s^2 T),  s^2 = omega^2/(omega^2 + rho)
 *   erfc(omega r)/r:        the difference            G_m = F_m(T) - s^{2m+1} F_m(s^2 T)
 * (substitute y = s y' in the truncated integral).  Process-wide setting, read when a quartet starts.
 * Pinned in tests/test_oracle_pins.py: G_m against mpmath quadrature of the truncated integral, (ab|cd) against the
 * brute-force quadrature of tests/refquad.py with the u-integral cut at omega, erf + erfc = Coulomb, omega -> infinity.
 * ---------------------------------------------------------------------------------------------- */
static int g_kernel_kind = 0;          /* 0 Coulomb, 1 erf-attenuated, 2 erfc-attenuated */
static double g_kernel_omega = 0.0;
int oracle_set_kernel(int kind, double omega)
{
    if (kind < 0 || kind > 2 || (kind != 0 && !(omega > 0.0))) return 1;
    g_kernel_kind = kind; g_kernel_omega = omega;
    return 0;
}

/* G_m, m = 0..mmax, for the current kernel */
static void kernel_seeds(int mmax, real rho, real T, real *G)
{
    boys_real(mmax, T, G);
    if (g_kernel_kind == 0) return;
    real w2 = (real)g_kernel_omega * (real)g_kernel_omega;
    real s2 = w2 / (w2 + rho), sp = R_SQRT(s2);      /* sp = s^{2m+1} */
    real *H = (real *)malloc(sizeof(real) * (mmax + 1));
    boys_real(mmax, s2 * T, H);
    for (int m = 0; m <= mmax; ++m) {
        real att = sp * H[m];
        G[m] = g_kernel_kind == 1 ? att : G[m] - att;
        sp *= s2;
    }
    free(H);
}

void oracle_kernel_seeds(int mmax, long double rho, long double T, long double *G)
{
    real *tmp = (real *)malloc(sizeof(real) * (mmax + 1));
    kernel_seeds(mmax, (real)rho, (real)T, tmp);
    for (int m = 0; m <= mmax; ++m) G[m] = (long double)tmp[m];
    free(tmp);
}

void oracle_boys(int mmax, long double T, long double *F)
{
    real *tmp = (real *)malloc(sizeof(real) * (mmax + 1));
    boys_real(mmax, (real)T, tmp);
    for (int m = 0; m <= mmax; ++m) F[m] = (long double)tmp[m];
    free(tmp);
}

/* ------------------------------------------------------------------------------------------------
 * Real solid harmonics, Racah normalisation (Helgaker-Jorgensen-Olsen sec. 6.4; the
 * paper defers these coefficients to its ref. 40):
 *   S_lm = N_lm sum_{t=0}^{[(l-|m|)/2]} sum_{u=0}^{t} sum_{v} C^{lm}_{tuv}
 *              x^{2t+|m|-2(u+v)} y^{2(u+v)} z^{l-2t-|m|},
 *   v = v_m, v_m+1, ... with 2v <= |m|,  v_m = 0 (m >= 0) or 1/2 (m < 0),
 *   C^{lm}_{tuv} = (-1)^{t+v-v_m} 4^{-t} binom(l,t) binom(l-t,|m|+t) binom(t,u) binom(|m|,2v),
 *   N_lm = 1/(2^{|m|} l!) sqrt( 2 (l+|m|)! (l-|m|)! / 2^{delta_m0} ).
 * Output C[(m+l) * ncart + k], k = position of (x,y,z) inside degree l in the ordering above.
 * ---------------------------------------------------------------------------------------------- */
static real binom(int n, int k)
{
    if (k < 0 || k > n) return 0.0L;
    real r = 1.0L;
    for (int i = 1; i <= k; ++i) r = r * (n - k + i) / i;
    return r;
}
static real factorial(int n) { real r = 1.0L; for (int i = 2; i <= n; ++i) r *= i; return r; }

static void solid_coeff_real(int l, real *C)
{
    pthread_once(&g_once, init_tables);
    int nc = (l + 1) * (l + 2) / 2, base = ORACLE_NCUM(l);
    for (int i = 0; i < (2 * l + 1) * nc; ++i) C[i] = 0.0L;
    for (int m = -l; m <= l; ++m) {
        int am = m < 0 ? -m : m;
        real N = R_SQRT(2.0L * factorial(l + am) * factorial(l - am) / (m == 0 ? 2.0L : 1.0L)) /
                 (R_POW(2.0L, am) * factorial(l));
        int w0 = m < 0 ? 1 : 0; /* w = 2v */
        for (int t = 0; 2 * t <= l - am; ++t)
            for (int u = 0; u <= t; ++u)
                for (int w = w0; w <= am; w += 2) {
                    int sgn = ((t + (w - w0) / 2) & 1) ? -1 : 1;
                    real c = sgn * R_POW(0.25L, t) * binom(l, t) * binom(l - t, am + t) * binom(t, u) * binom(am, w);
                    int ex = 2 * t + am - 2 * u - w, ey = 2 * u + w, ez = l - 2 * t - am;
                    C[(m + l) * nc + cart_index(ex, ey, ez) - base] += N * c;
                }
    }
}

void oracle_solid_coeff(int l, long double *C)
{
    int n = (2 * l + 1) * (l + 1) * (l + 2) / 2;
    real *tmp = (real *)malloc(sizeof(real) * n);
    solid_coeff_real(l, tmp);
    for (int i = 0; i < n; ++i) C[i] = (long double)tmp[i];
    free(tmp);
}

/* position of Cartesian (x,y,z) inside its degree, exported so tests can address Cartesian outputs */
int oracle_cart_pos(int x, int y, int z) { return cart_index(x, y, z) - ORACLE_NCUM(x + y + z); }

/* ------------------------------------------------------------------------------------------------
 * One contracted shell quartet, Cartesian components: out[a][b][c][d], a over the (la+1)(la+2)/2
 * Cartesian functions of degree la in the ordering above, etc.  Steps 1-5.
 * ---------------------------------------------------------------------------------------------- */
typedef struct {
    const double *center;     /* [3] */
    int l, nprim;
    const double *exps, *coefs;
} shell_t;

/* quartet_cart_dir: the part of the contraction whose primitive pairs have zeta_a >= zeta_b (zeta_a > zeta_b
 * if strict_bra) and zeta_c >= zeta_d (zeta_c > zeta_d if strict_ket).  The vertical recurrence builds
 * all momentum on the FIRST centre of each pair (A and C), the horizontal one moves it to the second.
 * *nused = number of primitive quartets that passed the filter (0: out is not written).
 * slice/nslice: only primitive quartets number slice, slice+nslice, ... of the four-fold loop are summed
 * (the integral is linear in them; the batch driver adds the partial sums), nslice = 1 for everything.  */
static int quartet_cart_dir(const shell_t *sa, const shell_t *sb, const shell_t *sc, const shell_t *sd,
                            int strict_bra, int strict_ket, int slice, int nslice, real *out, int *nused)
{
    pthread_once(&g_once, init_tables);
    *nused = 0;
    int prim_counter = 0;   /* primitive quartets are dealt round-robin to nslice independent partial sums */
    const int la = sa->l, lb = sb->l, lc = sc->l, ld = sd->l;
    const int lbra = la + lb, lket = lc + ld, L = lbra + lket;
    const int ne = ORACLE_NCUM(lbra + 1), nf = ORACLE_NCUM(lket + 1), nm = L + 1;
    const real pi = R_ACOS(-1.0L);
    real A[3], B[3], C[3], D[3];
    for (int i = 0; i < 3; ++i) { A[i] = sa->center[i]; B[i] = sb->center[i]; C[i] = sc->center[i]; D[i] = sd->center[i]; }
    real AB2 = 0, CD2 = 0;
    for (int i = 0; i < 3; ++i) { AB2 += (A[i] - B[i]) * (A[i] - B[i]); CD2 += (C[i] - D[i]) * (C[i] - D[i]); }

    real *V = (real *)malloc(sizeof(real) * (size_t)ne * nf * nm);      /* [f][e][m] primitive */
    real *G = (real *)calloc((size_t)ne * nf, sizeof(real));            /* contracted (e0|f0)   */
    real *F = (real *)malloc(sizeof(real) * nm);
    if (!V || !G || !F) { free(V); free(G); free(F); return 1; }
#define VV(e, f, m) V[((size_t)(f) * ne + (e)) * nm + (m)]

    for (int ka = 0; ka < sa->nprim; ++ka)
    for (int kb = 0; kb < sb->nprim; ++kb)
    for (int kc = 0; kc < sc->nprim; ++kc)
    for (int kd = 0; kd < sd->nprim; ++kd) {
        /* step 1 */
        real za = sa->exps[ka], zb = sb->exps[kb], zc = sc->exps[kc], zd = sd->exps[kd];
        if ((prim_counter++ % nslice) != slice) continue;
        if (strict_bra ? !(za > zb) : !(za >= zb)) continue;
        if (strict_ket ? !(zc > zd) : !(zc >= zd)) continue;
        ++*nused;
        real p = za + zb, q = zc + zd, rho = p * q / (p + q);
        real P[3], Q[3], W[3], PA[3], QC[3], WP[3], WQ[3], PQ2 = 0;
        for (int i = 0; i < 3; ++i) {
            P[i] = (za * A[i] + zb * B[i]) / p;
            Q[i] = (zc * C[i] + zd * D[i]) / q;
            W[i] = (p * P[i] + q * Q[i]) / (p + q);
            PA[i] = P[i] - A[i]; QC[i] = Q[i] - C[i]; WP[i] = W[i] - P[i]; WQ[i] = W[i] - Q[i];
            PQ2 += (P[i] - Q[i]) * (P[i] - Q[i]);
        }
        real T = rho * PQ2;
        real Kab = R_EXP(-za * zb / p * AB2), Kcd = R_EXP(-zc * zd / q * CD2);
        /* step 2 */
        real pref = (real)sa->coefs[ka] * sb->coefs[kb] * sc->coefs[kc] * sd->coefs[kd] * Kab * Kcd *
                    2.0L * R_POW(pi, 2.5L) / (p * q * R_SQRT(p + q));
        kernel_seeds(L, rho, T, F);     /* F_m(T) for the Coulomb kernel */
        for (int m = 0; m <= L; ++m) VV(0, 0, m) = pref * F[m];
        /* step 3a: [e+1_i,0|00]^(m) = PA_i [e0|00]^(m) + WP_i [e0|00]^(m+1)
         *                            + e_i/(2p) ( [e-1_i,0|00]^(m) - rho/p [e-1_i,0|00]^(m+1) )           */
        for (int e1 = 1; e1 < ne; ++e1) {
            int i = first_axis(e1), e = lower(e1, i), ei = comp(e, i);
            int deg = g_cx[e1] + g_cy[e1] + g_cz[e1];
            int em = ei > 0 ? lower(e, i) : 0;
            for (int m = 0; m <= L - deg; ++m) {
                real v = PA[i] * VV(e, 0, m) + WP[i] * VV(e, 0, m + 1);
                if (ei > 0) v += ei / (2.0L * p) * (VV(em, 0, m) - rho / p * VV(em, 0, m + 1));
                VV(e1, 0, m) = v;
            }
        }
        /* step 3b: [e0|f+1_i,0]^(m) = QC_i [e0|f0]^(m) + WQ_i [e0|f0]^(m+1)
         *                            + f_i/(2q) ( [e0|f-1_i,0]^(m) - rho/q [e0|f-1_i,0]^(m+1) )
         *                            + e_i/(2(p+q)) [e-1_i,0|f0]^(m+1)                                    */
        for (int f1 = 1; f1 < nf; ++f1) {
            int i = first_axis(f1), f = lower(f1, i), fi = comp(f, i);
            int fdeg = g_cx[f1] + g_cy[f1] + g_cz[f1];
            int fm = fi > 0 ? lower(f, i) : 0;
            for (int e = 0; e < ne; ++e) {
                int edeg = g_cx[e] + g_cy[e] + g_cz[e], ei = comp(e, i);
                int em = ei > 0 ? lower(e, i) : 0;
                for (int m = 0; m <= L - edeg - fdeg; ++m) {
                    real v = QC[i] * VV(e, f, m) + WQ[i] * VV(e, f, m + 1);
                    if (fi > 0) v += fi / (2.0L * q) * (VV(e, fm, m) - rho / q * VV(e, fm, m + 1));
                    if (ei > 0) v += ei / (2.0L * (p + q)) * VV(em, f, m + 1);
                    VV(e, f1, m) = v;
                }
            }
        }
        /* step 4 */
        for (int e = ORACLE_NCUM(la); e < ne; ++e)
            for (int f = ORACLE_NCUM(lc); f < nf; ++f) G[(size_t)e * nf + f] += VV(e, f, 0);
    }
#undef VV
    free(V); free(F);
    if (*nused == 0) { free(G); return 0; }

    /* step 5a, bra: (a,b+1_i| = (a+1_i,b| + (A_i-B_i)(a,b|, one ket index f at a time.
     * X[a*nbc + b], a over all degrees <= lbra, b over all degrees <= lb; keep |a| = la, |b| = lb.      */
    const int nbc = ORACLE_NCUM(lb + 1), ndc = ORACLE_NCUM(ld + 1);
    const int na = (la + 1) * (la + 2) / 2, nb = (lb + 1) * (lb + 2) / 2, nc = (lc + 1) * (lc + 2) / 2,
              nd = (ld + 1) * (ld + 2) / 2;
    real *X = (real *)calloc((size_t)ne * nbc, sizeof(real));
    real *Y = (real *)calloc((size_t)na * nb * nf, sizeof(real));       /* Y[ab][f] */
    if (!X || !Y) { free(G); free(X); free(Y); return 1; }
    for (int f = ORACLE_NCUM(lc); f < nf; ++f) {
        for (int a = 0; a < ne; ++a) X[(size_t)a * nbc + 0] = G[(size_t)a * nf + f];
        for (int b1 = 1; b1 < nbc; ++b1) {
            int i = first_axis(b1), b = lower(b1, i), bdeg = g_cx[b1] + g_cy[b1] + g_cz[b1];
            for (int a = ORACLE_NCUM(la); a < ORACLE_NCUM(lbra - bdeg + 1); ++a)
                X[(size_t)a * nbc + b1] = X[(size_t)raise(a, i) * nbc + b] + (A[i] - B[i]) * X[(size_t)a * nbc + b];
        }
        for (int a = 0; a < na; ++a)
            for (int b = 0; b < nb; ++b)
                Y[((size_t)a * nb + b) * nf + f] = X[(size_t)(ORACLE_NCUM(la) + a) * nbc + (ORACLE_NCUM(lb) + b)];
    }
    free(X); free(G);
    /* step 5b, ket: (ab|c,d+1_i) = (ab|c+1_i,d) + (C_i-D_i)(ab|c,d)                                      */
    real *Z = (real *)calloc((size_t)nf * ndc, sizeof(real));
    for (int ab = 0; ab < na * nb; ++ab) {
        for (int c = 0; c < nf; ++c) Z[(size_t)c * ndc + 0] = Y[(size_t)ab * nf + c];
        for (int d1 = 1; d1 < ndc; ++d1) {
            int i = first_axis(d1), d = lower(d1, i), ddeg = g_cx[d1] + g_cy[d1] + g_cz[d1];
            for (int c = ORACLE_NCUM(lc); c < ORACLE_NCUM(lket - ddeg + 1); ++c) {
                int cp = raise(c, i);
                Z[(size_t)c * ndc + d1] = Z[(size_t)cp * ndc + d] + (C[i] - D[i]) * Z[(size_t)c * ndc + d];
            }
        }
        for (int c = 0; c < nc; ++c)
            for (int d = 0; d < nd; ++d)
                out[((size_t)ab * nc + c) * nd + d] = Z[(size_t)(ORACLE_NCUM(lc) + c) * ndc + (ORACLE_NCUM(ld) + d)];
    }
    free(Y); free(Z);
    return 0;
}

/* One contracted shell quartet, Cartesian components out[a][b][c][d] (steps 1-5).
 *
 * Direction of the horizontal recurrence.  (a,b+1_i| = (a+1_i,b| + (A_i-B_i)(a,b| rebuilds x_B^lb from
 * powers of x_A; when the product Gaussian sits near B (zeta_b >> zeta_a, |P-A| ~ |AB|) the wanted value
 * is small and the terms are of size |AB|^(la+lb): digits are lost (measured on BASELINE config 1:
 * 4e-3 relative against the binary128 build of this file when A is always the building centre).
 * The defining integral is symmetric, (ab|cd) = (ba|cd) = (ab|dc), so each primitive pair may build on
 * either centre.  Here every primitive pair builds on its centre with the LARGER exponent, for which
 * |P-A| <= |AB|/2 and the terms of the transfer are at most 3^lb times the result: the contraction is
 * split into the four groups (zeta_a >= zeta_b | zeta_a < zeta_b) x (zeta_c >= zeta_d | zeta_c < zeta_d),
 * each group goes through steps 1-5 with its own building centres, the swapped groups are transposed
 * back, and the four Cartesian results are added.  Same recurrences, same result, no digits lost
 * (reading R3).                                                                            */
static int quartet_cart(const shell_t *sa, const shell_t *sb, const shell_t *sc, const shell_t *sd, int slice,
                        int nslice, real *out)
{
    const int na = (sa->l + 1) * (sa->l + 2) / 2, nb = (sb->l + 1) * (sb->l + 2) / 2,
              nc = (sc->l + 1) * (sc->l + 2) / 2, nd = (sd->l + 1) * (sd->l + 2) / 2;
    const size_t n = (size_t)na * nb * nc * nd;
    real *tmp = (real *)malloc(sizeof(real) * n);
    if (!tmp) return 1;
    for (size_t t = 0; t < n; ++t) out[t] = 0;
    for (int swb = 0; swb < 2; ++swb)
        for (int swk = 0; swk < 2; ++swk) {
            int used = 0;
            int rc = quartet_cart_dir(swb ? sb : sa, swb ? sa : sb, swk ? sd : sc, swk ? sc : sd, swb, swk, slice, nslice,
                                      tmp, &used);
            if (rc) { free(tmp); return rc; }
            if (!used) continue;
            /* tmp is [x0][x1][y0][y1] with (x0,x1) = (b,a) if swb and (y0,y1) = (d,c) if swk */
            for (int a = 0; a < na; ++a)
                for (int b = 0; b < nb; ++b)
                    for (int c = 0; c < nc; ++c)
                        for (int d = 0; d < nd; ++d) {
                            size_t bra = swb ? (size_t)b * na + a : (size_t)a * nb + b;
                            size_t ket = swk ? (size_t)d * nc + c : (size_t)c * nd + d;
                            out[(((size_t)a * nb + b) * nc + c) * nd + d] += tmp[bra * ((size_t)nc * nd) + ket];
                        }
        }
    free(tmp);
    return 0;
}

/* step 6: transform one index of a 4-index array from Cartesian to solid harmonics.
 * in [n0][ncart][n2] -> out [n0][nsph][n2]                                                             */
static void transform_index(const real *in, real *out, int n0, int l, int n2)
{
    int ncart = (l + 1) * (l + 2) / 2, ns = 2 * l + 1;
    real *C = (real *)malloc(sizeof(real) * ns * ncart);
    solid_coeff_real(l, C);
    for (int i0 = 0; i0 < n0; ++i0)
        for (int m = 0; m < ns; ++m)
            for (int i2 = 0; i2 < n2; ++i2) {
                real s = 0;
                for (int k = 0; k < ncart; ++k) s += C[m * ncart + k] * in[((size_t)i0 * ncart + k) * n2 + i2];
                out[((size_t)i0 * ns + m) * n2 + i2] = s;
            }
    free(C);
}

static int quartet_solid(const shell_t *sa, const shell_t *sb, const shell_t *sc, const shell_t *sd, int slice,
                         int nslice, real *out)
{
    int l[4] = {sa->l, sb->l, sc->l, sd->l}, ncart[4], ns[4];
    size_t big = 1;
    for (int i = 0; i < 4; ++i) { ncart[i] = (l[i] + 1) * (l[i] + 2) / 2; ns[i] = 2 * l[i] + 1; big *= ncart[i]; }
    real *t0 = (real *)malloc(sizeof(real) * big), *t1 = (real *)malloc(sizeof(real) * big);
    if (!t0 || !t1) { free(t0); free(t1); return 1; }
    int rc = quartet_cart(sa, sb, sc, sd, slice, nslice, t0);
    if (!rc) {
        transform_index(t0, t1, 1, l[0], ncart[1] * ncart[2] * ncart[3]);
        transform_index(t1, t0, ns[0], l[1], ncart[2] * ncart[3]);
        transform_index(t0, t1, ns[0] * ns[1], l[2], ncart[3]);
        transform_index(t1, out, ns[0] * ns[1] * ns[2], l[3], 1);
    }
    free(t0); free(t1);
    return rc;
}

/* ------------------------------------------------------------------------------------------------
 * Public entry points (C ABI, host pointers only).
 * ---------------------------------------------------------------------------------------------- */
static int make_shell(shell_t *s, int idx, const double *centers, const int *l, const int *prim_offset,
                      const double *exps, const double *coefs)
{
    s->center = centers + 3 * idx;
    s->l = l[idx];
    s->nprim = prim_offset[idx + 1] - prim_offset[idx];
    s->exps = exps + prim_offset[idx];
    s->coefs = coefs + prim_offset[idx];
    return (s->l < 0 || s->l > ORACLE_LMAX || s->nprim < 1);
}

/* One quartet of shells (ia ib|ic id) from a shell table in the md4_set_shells layout
 * (include/md4.h).  solid != 0: out[ma][mb][mc][md], m = -l..l ascending; solid == 0: Cartesian
 * components in the ordering of oracle_cart_pos.  out is long double.  Returns 0 on success.          */
int oracle_quartet_ld(const double *centers, const int *l, const int *prim_offset, const double *exps,
                      const double *coefs, int ia, int ib, int ic, int id, int solid, long double *out)
{
    shell_t s[4];
    int idx[4] = {ia, ib, ic, id};
    for (int i = 0; i < 4; ++i)
        if (make_shell(&s[i], idx[i], centers, l, prim_offset, exps, coefs)) return 2;
    size_t n = 1;
    for (int i = 0; i < 4; ++i) n *= solid ? (size_t)(2 * s[i].l + 1) : (size_t)((s[i].l + 1) * (s[i].l + 2) / 2);
    real *tmp = (real *)malloc(sizeof(real) * n);
    if (!tmp) return 1;
    int rc = solid ? quartet_solid(&s[0], &s[1], &s[2], &s[3], 0, 1, tmp)
                   : quartet_cart(&s[0], &s[1], &s[2], &s[3], 0, 1, tmp);
    for (size_t t = 0; t < n; ++t) out[t] = (long double)tmp[t];
    free(tmp);
    return rc;
}

typedef struct {
    const double *centers; const int *l, *prim_offset; const double *exps, *coefs;
    int nbra; const int *bra_ij; int nket; const int *ket_ij;
    double *out; size_t per_quartet;
    const int *subset; int nsubset;         /* optional list of flat quartet indices i*nket+j */
    int nslice; real *acc;                  /* nslice > 1: partial sums over primitive slices, added in acc */
    int next; pthread_mutex_t mu; int rc;
} job_t;

static void *worker(void *arg)
{
    job_t *J = (job_t *)arg;
    real *buf = (real *)malloc(sizeof(real) * J->per_quartet);
    int total = (J->subset ? J->nsubset : J->nbra * J->nket) * J->nslice;
    for (;;) {
        pthread_mutex_lock(&J->mu);
        int job = J->next++;
        pthread_mutex_unlock(&J->mu);
        if (job >= total || !buf) break;
        int k = job / J->nslice, slice = job % J->nslice;
        int flat = J->subset ? J->subset[k] : k;
        int i = flat / J->nket, j = flat % J->nket;
        shell_t s[4];
        int idx[4] = {J->bra_ij[2 * i], J->bra_ij[2 * i + 1], J->ket_ij[2 * j], J->ket_ij[2 * j + 1]};
        int rc = 0;
        for (int t = 0; t < 4; ++t) rc |= make_shell(&s[t], idx[t], J->centers, J->l, J->prim_offset, J->exps, J->coefs);
        if (!rc) rc = quartet_solid(&s[0], &s[1], &s[2], &s[3], slice, J->nslice, buf);
        if (rc) { J->rc = rc ? rc : 2; break; }
        /* with a subset the k-th result goes to slot k, otherwise to slot i*nket+j */
        size_t slot = (size_t)(J->subset ? k : flat) * J->per_quartet;
        if (J->nslice == 1) {
            for (size_t t = 0; t < J->per_quartet; ++t) J->out[slot + t] = (double)buf[t];
        } else {
            pthread_mutex_lock(&J->mu);
            for (size_t t = 0; t < J->per_quartet; ++t) J->acc[slot + t] += buf[t];
            pthread_mutex_unlock(&J->mu);
        }
    }
    free(buf);
    return NULL;
}

/* Batch: out[i_bra][j_ket][ma][mb][mc][md] (the layout of md4_compute, include/md4.h), evaluated in `real`
 * and rounded to double once at the end.  All bra pairs must share (l_i,l_j), all ket pairs likewise.  If
 * subset != NULL only the listed flat quartet indices (i*nket + j) are computed and written densely:
 * out[k][ma][mb][mc][md].  nslice > 1 splits the primitive loop of every quartet into nslice partial sums
 * that run on different threads (for heavily contracted quartets); the partial sums are added in `real`. */
int oracle_compute(int nshell, const double *centers, const int *l, const int *prim_offset, const double *exps,
                   const double *coefs, int nbra, const int *bra_ij, int nket, const int *ket_ij,
                   const int *subset, int nsubset, double *out, int nthreads, int nslice)
{
    (void)nshell;
    if (nbra <= 0 || nket <= 0) return 0;
    job_t J;
    memset(&J, 0, sizeof J);
    J.centers = centers; J.l = l; J.prim_offset = prim_offset; J.exps = exps; J.coefs = coefs;
    J.nbra = nbra; J.bra_ij = bra_ij; J.nket = nket; J.ket_ij = ket_ij; J.out = out;
    J.subset = subset; J.nsubset = nsubset;
    J.nslice = nslice < 1 ? 1 : nslice;
    J.per_quartet = (size_t)(2 * l[bra_ij[0]] + 1) * (2 * l[bra_ij[1]] + 1) * (2 * l[ket_ij[0]] + 1) * (2 * l[ket_ij[1]] + 1);
    size_t nq = (size_t)(subset ? nsubset : nbra * nket);
    if (J.nslice > 1) {
        J.acc = (real *)malloc(sizeof(real) * nq * J.per_quartet);
        if (!J.acc) return 1;
        for (size_t t = 0; t < nq * J.per_quartet; ++t) J.acc[t] = 0;
    }
    pthread_mutex_init(&J.mu, NULL);
    if (nthreads < 1) nthreads = 1;
    if (nthreads > 256) nthreads = 256;
    pthread_t th[256];
    for (int t = 0; t < nthreads; ++t) pthread_create(&th[t], NULL, worker, &J);
    for (int t = 0; t < nthreads; ++t) pthread_join(th[t], NULL);
    pthread_mutex_destroy(&J.mu);
    if (J.nslice > 1) {
        if (!J.rc) for (size_t t = 0; t < nq * J.per_quartet; ++t) out[t] = (double)J.acc[t];
        free(J.acc);
    }
    return J.rc;
}

// md4_pairs.cu -- shell-pair precompute kernel (S:8(a) step a1; the paper's
// compute_hermite_gaussian_transform, Listing 2.1 lines 2-3).
// Per primitive pair: zeta_p, R_p, ln K_ab (S:8(c) Q2), the 1-D Hermite expansion tables
// (E_i)^t_{a_i b_i} by Eq.4-5, and H = c_a c_b C_la (x) C_lb E (Eq.16) as two
// half transforms in double-double arithmetic, rounded to FP64 and written in the 8x8-blocked layout of
// md4_internal.h.
#include "md4_internal.h"

namespace md4 {

namespace {
constexpr int NSMAX = 2 * LMAX + 1;    // 15
constexpr int PAIR_THREADS = 256;
constexpr int PAIR_SPLIT = 8;          // CTAs per primitive pair (each takes a range of Hermite column blocks)

// ---- double-double arithmetic (error-free transformations; __d*_rn blocks FMA contraction) ---------
// Why: H = C_la (x) C_lb E cancels the radial contaminants of the Cartesian Gaussians.  For a tight
// shell of high l far from its partner the surviving part is ~(2 zeta_p)^-l/2 of the terms (1e-6 for
// l = 6, zeta_p = 50) and it meets R values that are ~R^6/720 larger than the ones the leading part
// meets: in plain FP64 the error reached 3e-8 of max|integral| on BASELINE config 5 (bar 1e-10).
// E, the E products and both half transforms therefore run in double-double; H is rounded to FP64 at
// the end, every entry correct to ~1e-16 of ITSELF.
typedef double2 dd;  // x = hi, y = lo
__device__ __forceinline__ dd dd_two_sum(double a, double b) {
    const double s = __dadd_rn(a, b), bb = __dadd_rn(s, -a);
    return make_double2(s, __dadd_rn(__dadd_rn(a, -__dadd_rn(s, -bb)), __dadd_rn(b, -bb)));
}
__device__ __forceinline__ dd dd_quick(double a, double b) {
    const double s = __dadd_rn(a, b);
    return make_double2(s, __dadd_rn(b, -__dadd_rn(s, -a)));
}
__device__ __forceinline__ dd dd_add(dd a, dd b) {
    dd s = dd_two_sum(a.x, b.x);
    return dd_quick(s.x, __dadd_rn(s.y, __dadd_rn(a.y, b.y)));
}
__device__ __forceinline__ dd dd_mul(dd a, dd b) {
    const double p = __dmul_rn(a.x, b.x);
    double e = __fma_rn(a.x, b.x, -p);
    e = __fma_rn(a.x, b.y, e);
    e = __fma_rn(a.y, b.x, e);
    return dd_quick(p, e);
}
__device__ __forceinline__ dd dd_mul_d(dd a, double b) {
    const double p = __dmul_rn(a.x, b);
    double e = __fma_rn(a.x, b, -p);
    e = __fma_rn(a.y, b, e);
    return dd_quick(p, e);
}

struct PairKernelArgs {
    const double* centers;
    const int* off;
    const double* expo;
    const double* coef;
    const int* ij;
    const uint32_t* colb;     // bra-role column order for this l_pair (md4_internal.h)
    const int* b2k;           // bra column -> ket column
    const double *Ca, *CaLo;  // [(2li+1) * nc(li)] high / low parts
    const double *Cb, *CbLo;
    double* Hb;
    double* Hk;
    double* scal;
    int li, lj, Ki, Kj, nab, nrb, ncb;
    size_t hstrideb, hstridek;
};

// Shared memory of one CTA, sized for the class of the list (li, lj), not for MD4_LMAX: an (ii) list takes 87 kB (two
// CTAs per SM), a (gg) list 33 kB, a (kk) list 132 kB.  1-D tables E[axis][(ai * na1 + bi) * nt1 + t] with na1 =
// max(li, lj) + 1 and nt1 = li + lj + 1.
struct PairSmemLayout {
    int na1, nt1, esz;
    size_t oE, oCa, oCb, oY, oca, ocb, total;
    __host__ __device__ PairSmemLayout(int li, int lj) {
        na1 = (li > lj ? li : lj) + 1;
        nt1 = li + lj + 1;
        esz = na1 * na1 * nt1;
        const int nca = n_cart(li), ncb = n_cart(lj), nsa = 2 * li + 1, nsb = 2 * lj + 1;
        size_t o = 0;
        oE = o; o += (size_t)3 * esz * sizeof(dd);
        oCa = o; o += (size_t)nsa * nca * sizeof(dd);
        oCb = o; o += (size_t)nsb * ncb * sizeof(dd);
        oY = o; o += (size_t)nca * nsb * 8 * sizeof(dd);
        oca = o; o += (size_t)nca * 2;
        ocb = o; o += (size_t)ncb * 2;
        total = (o + 15) / 16 * 16;
    }
};

__global__ void __launch_bounds__(PAIR_THREADS) pair_h_kernel(PairKernelArgs a) {
    extern __shared__ __align__(16) unsigned char pair_smem_raw[];
    const PairSmemLayout lay(a.li, a.lj);
    const int NA1 = lay.na1, NT1 = lay.nt1, ESZ = lay.esz;
    struct {
        dd* E[3]; dd* Ca; dd* Cb; dd* Y;
        unsigned char (*ca)[2]; unsigned char (*cb)[2];
    } sm;
    for (int i = 0; i < 3; ++i) sm.E[i] = reinterpret_cast<dd*>(pair_smem_raw + lay.oE) + (size_t)i * ESZ;
    sm.Ca = reinterpret_cast<dd*>(pair_smem_raw + lay.oCa);
    sm.Cb = reinterpret_cast<dd*>(pair_smem_raw + lay.oCb);
    sm.Y = reinterpret_cast<dd*>(pair_smem_raw + lay.oY);
    sm.ca = reinterpret_cast<unsigned char (*)[2]>(pair_smem_raw + lay.oca);
    sm.cb = reinterpret_cast<unsigned char (*)[2]>(pair_smem_raw + lay.ocb);

    const int tid = threadIdx.x, nthr = blockDim.x;
    const int split = blockIdx.x % PAIR_SPLIT;
    const int ip = blockIdx.x / PAIR_SPLIT;
    const int kk = a.Ki * a.Kj;
    const int ipair = ip / kk, kab = ip % kk, ka = kab / a.Kj, kb = kab % a.Kj;
    const int si = a.ij[2 * ipair], sj = a.ij[2 * ipair + 1];
    const int li = a.li, lj = a.lj;
    const int nca = n_cart(li), ncbt = n_cart(lj), nsa = 2 * li + 1, nsb = 2 * lj + 1;

    const double za = a.expo[a.off[si] + ka], zb = a.expo[a.off[sj] + kb];
    const double zp = za + zb;
    double A[3], B[3], P[3], XPA[3], XPB[3];
    double ab2 = 0.0;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        A[i] = a.centers[3 * si + i];
        B[i] = a.centers[3 * sj + i];
        const double d = B[i] - A[i];
        P[i] = (za * A[i] + zb * B[i]) / zp;
        // P - A and P - B from the centre difference: each keeps full relative accuracy when P sits on a centre
        XPA[i] = (zb / zp) * d;
        XPB[i] = -(za / zp) * d;
        ab2 += d * d;
    }
    for (int i = tid; i < 3 * ESZ; i += nthr) sm.E[0][i] = make_double2(0.0, 0.0);   // the three tables are contiguous
    for (int i = tid; i < nsa * nca; i += nthr) sm.Ca[i] = make_double2(a.Ca[i], a.CaLo[i]);
    for (int i = tid; i < nsb * ncbt; i += nthr) sm.Cb[i] = make_double2(a.Cb[i], a.CbLo[i]);
    if (tid == 0) {
        int k = 0;
        for (int x = li; x >= 0; --x)
            for (int y = li - x; y >= 0; --y, ++k) { sm.ca[k][0] = x; sm.ca[k][1] = y; }
        k = 0;
        for (int x = lj; x >= 0; --x)
            for (int y = lj - x; y >= 0; --y, ++k) { sm.cb[k][0] = x; sm.cb[k][1] = y; }
        if (split == 0) {
            double* s = a.scal + (size_t)ip * 8;
            s[0] = zp; s[1] = P[0]; s[2] = P[1]; s[3] = P[2];
            s[4] = -(za * zb / zp) * ab2;  // ln K_ab; made relative to the pair maximum by pair_finalize_kernel
            s[5] = 0.0; s[6] = 0.0; s[7] = 0.0;
        }
    }
    __syncthreads();
    // 1-D tables (Eq.4: raise a at b = 0, Eq.5: raise b), seed (E_i)^0_00 = 1: warp i does axis i,
    // lane t does Hermite order t; one step of the recurrence per __syncwarp.
    const int warp = tid >> 5, lane = tid & 31;
    if (warp < 3) {
        dd* E = sm.E[0] + (size_t)warp * ESZ;
        const double xpa = XPA[warp], xpb = XPB[warp], h = 0.5 / zp;
        if (lane == 0) E[0] = make_double2(1.0, 0.0);
        __syncwarp();
        for (int ai = 0; ai < li; ++ai) {
            const dd* e = E + (ai * NA1) * NT1;
            const int t = lane;
            if (t <= ai + 1) {
                dd v = dd_mul_d(e[t], xpa);
                if (t < ai) v = dd_add(v, dd_mul_d(e[t + 1], (double)(t + 1)));  // (E)^t_ab = 0 for t > a+b
                if (t > 0) v = dd_add(v, dd_mul_d(e[t - 1], h));
                E[((ai + 1) * NA1) * NT1 + t] = v;
            }
            __syncwarp();
        }
        for (int bi = 0; bi < lj; ++bi) {
            // all a_i in parallel: lanes (ai, t) flattened
            for (int idx = lane; idx < (li + 1) * NT1; idx += 32) {
                const int ai = idx / NT1, t = idx % NT1;
                if (t <= ai + bi + 1) {
                    const dd* e = E + (ai * NA1 + bi) * NT1;
                    dd v = dd_mul_d(e[t], xpb);
                    if (t < ai + bi) v = dd_add(v, dd_mul_d(e[t + 1], (double)(t + 1)));
                    if (t > 0) v = dd_add(v, dd_mul_d(e[t - 1], h));
                    E[(ai * NA1 + bi + 1) * NT1 + t] = v;
                }
            }
            __syncwarp();
        }
    }
    __syncthreads();
    const double wgt = a.coef[a.off[si] + ka] * a.coef[a.off[sj] + kb];
    const int jb0 = (int)((long long)split * a.ncb / PAIR_SPLIT), jb1 = (int)((long long)(split + 1) * a.ncb / PAIR_SPLIT);
    for (int jb = jb0; jb < jb1; ++jb) {
        // half transform over b: Y[ac][mb][pp] = sum_bc Cb[mb][bc] Ex Ey Ez.  One thread per (ac, pp) keeps the
        // 2 lb + 1 sums in registers, so each product Ex Ey Ez is formed once; zero coefficients of the (sparse)
        // solid-harmonic table are skipped (the test is uniform over the warp: mb and bc do not depend on the lane)
        for (int idx = tid; idx < nca * 8; idx += nthr) {
            const int pp = idx & 7, ac = idx >> 3;
            const int col = jb * 8 + pp;
            dd acc[NSMAX];
#pragma unroll
            for (int mb = 0; mb < NSMAX; ++mb) acc[mb] = make_double2(0.0, 0.0);
            const uint32_t w = a.colb[col];
            if (!(w & COL_PAD)) {
                const int t = w & 255, u = (w >> 8) & 255, v = (w >> 16) & 255;
                const int ax = sm.ca[ac][0], ay = sm.ca[ac][1], az = li - ax - ay;
                for (int bc = 0; bc < ncbt; ++bc) {
                    const int bx = sm.cb[bc][0], by = sm.cb[bc][1], bz = lj - bx - by;
                    if (t > ax + bx || u > ay + by || v > az + bz) continue;
                    const dd e3 = dd_mul(dd_mul(sm.E[0][(ax * NA1 + bx) * NT1 + t], sm.E[1][(ay * NA1 + by) * NT1 + u]),
                                         sm.E[2][(az * NA1 + bz) * NT1 + v]);
#pragma unroll
                    for (int mb = 0; mb < NSMAX; ++mb) {
                        if (mb < nsb) {
                            const dd cb = sm.Cb[mb * ncbt + bc];
                            if (cb.x != 0.0) acc[mb] = dd_add(acc[mb], dd_mul(cb, e3));
                        }
                    }
                }
            }
#pragma unroll
            for (int mb = 0; mb < NSMAX; ++mb)
                if (mb < nsb) sm.Y[(ac * nsb + mb) * 8 + pp] = acc[mb];
        }
        __syncthreads();
        // half transform over a, contraction weight, blocked store
        // (both role copies: the bra-order block here, the same number at its ket-order column there)
        double* Hp = a.Hb + (size_t)ip * a.hstrideb + (size_t)jb * a.nrb * 64;
        double* Hq = a.Hk + (size_t)ip * a.hstridek;
        for (int idx = tid; idx < a.nab * 8; idx += nthr) {
            const int pp = idx & 7, row = idx >> 3;
            const int ma = row / nsb, mb = row % nsb;
            dd acc = make_double2(0.0, 0.0);
            for (int ac = 0; ac < nca; ++ac) {
                const dd ca = sm.Ca[ma * nca + ac];
                if (ca.x != 0.0) acc = dd_add(acc, dd_mul(ca, sm.Y[(ac * nsb + mb) * 8 + pp]));
            }
            const double h = wgt * acc.x + wgt * acc.y;
            Hp[(row >> 3) * 64 + (row & 7) * 8 + pp] = h;
            const int ck = a.b2k[jb * 8 + pp];
            if (ck >= 0) Hq[((size_t)(ck >> 3) * a.nrb + (row >> 3)) * 64 + (row & 7) * 8 + (ck & 7)] = h;
        }
        __syncthreads();
    }
}

__global__ void pair_finalize_kernel(double* scal, double* pairmax, int npair, int kk) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= npair) return;
    double m = -1.0e300;
    for (int k = 0; k < kk; ++k) m = fmax(m, scal[((size_t)i * kk + k) * 8 + 4]);
    pairmax[i] = m;
    for (int k = 0; k < kk; ++k) scal[((size_t)i * kk + k) * 8 + 4] -= m;
}
}  // namespace

cudaError_t launch_pair_kernel(md4_ctx* ctx, const PairListDev& pl, cudaStream_t st) {
    if (pl.npair == 0) return cudaSuccess;
    const int kk = pl.Ki * pl.Kj;
    const size_t nprim = (size_t)pl.npair * kk;
    cudaError_t e = cudaMemsetAsync(pl.Hb, 0, nprim * pl.hstrideb * sizeof(double), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(pl.Hk, 0, nprim * pl.hstridek * sizeof(double), st);
    if (e != cudaSuccess) return e;
    PairKernelArgs a;
    a.centers = ctx->d_centers; a.off = ctx->d_off; a.expo = ctx->d_exp; a.coef = ctx->d_coef;
    a.ij = pl.ij; a.colb = ctx->tab.colb[pl.lsum]; a.b2k = ctx->tab.b2k[pl.lsum];
    a.Ca = ctx->tab.solid[pl.li]; a.CaLo = ctx->tab.solid_lo[pl.li];
    a.Cb = ctx->tab.solid[pl.lj]; a.CbLo = ctx->tab.solid_lo[pl.lj];
    a.Hb = pl.Hb; a.Hk = pl.Hk; a.scal = pl.scal;
    a.li = pl.li; a.lj = pl.lj; a.Ki = pl.Ki; a.Kj = pl.Kj;
    a.nab = pl.nab; a.nrb = pl.nrb; a.ncb = pl.ncbb; a.hstrideb = pl.hstrideb; a.hstridek = pl.hstridek;
    const size_t nblk = nprim * PAIR_SPLIT;
    if (nblk > 2147483647ull) return cudaErrorInvalidValue;
    if (ctx->configured.insert(reinterpret_cast<const void*>(pair_h_kernel)).second) {
        e = cudaFuncSetAttribute(pair_h_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PairSmemLayout(LMAX, LMAX).total);
        if (e != cudaSuccess) { ctx->configured.erase(reinterpret_cast<const void*>(pair_h_kernel)); return e; }
    }
    pair_h_kernel<<<(unsigned)nblk, PAIR_THREADS, PairSmemLayout(pl.li, pl.lj).total, st>>>(a);
    ctx->launches++;
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    pair_finalize_kernel<<<(pl.npair + 127) / 128, 128, 0, st>>>(pl.scal, pl.pairmax, pl.npair, kk);
    ctx->launches++;
    return cudaGetLastError();
}

}  // namespace md4

// md4_pairs.cu -- shell-pair precompute kernel (S:8(a) step a1; the paper's
// compute_hermite_gaussian_transform, Listing 2.1 lines 2-3).
// Per primitive pair: zeta_p, R_p, ln K_ab (S:8(c) Q2), the 1-D Hermite expansion tables
// (E_i)^t_{a_i b_i} by Eq.4-5, and H = c_a c_b C_la (x) C_lb E (Eq.16) as two
// half transforms, written in the 8x8-blocked layout of md4_internal.h.
#include "md4_internal.h"

namespace md4 {

namespace {
constexpr int NA1 = LMAX + 1;          // a_i = 0..6
constexpr int NT1 = 2 * LMAX + 1;      // t = 0..12
constexpr int ESZ = NA1 * NA1 * NT1;   // 637 per axis
constexpr int NCMAX = (LMAX + 1) * (LMAX + 2) / 2;  // 28
constexpr int NSMAX = 2 * LMAX + 1;    // 13

struct PairKernelArgs {
    const double* centers;
    const int* off;
    const double* expo;
    const double* coef;
    const int* ij;
    const uint32_t* tuv;
    const double* Ca;  // [(2li+1) * nc(li)]
    const double* Cb;
    double* H;
    double* scal;
    int li, lj, Ki, Kj, nab, nrb, nherm, ncb;
    size_t hstride;
};

__global__ void __launch_bounds__(256) pair_h_kernel(PairKernelArgs a) {
    __shared__ double sE[3][ESZ];
    __shared__ double sCa[NSMAX * NCMAX];
    __shared__ double sCb[NSMAX * NCMAX];
    __shared__ double sY[NCMAX * NSMAX * 8];
    __shared__ unsigned char sca[NCMAX][2], scb[NCMAX][2];

    const int tid = threadIdx.x, nthr = blockDim.x;
    const int jb = blockIdx.x % a.ncb;
    const int ip = blockIdx.x / a.ncb;
    const int kk = a.Ki * a.Kj;
    const int ipair = ip / kk, kab = ip % kk, ka = kab / a.Kj, kb = kab % a.Kj;
    const int si = a.ij[2 * ipair], sj = a.ij[2 * ipair + 1];
    const int li = a.li, lj = a.lj;
    const int nca = n_cart(li), ncbt = n_cart(lj), nsa = 2 * li + 1, nsb = 2 * lj + 1;

    const double za = a.expo[a.off[si] + ka], zb = a.expo[a.off[sj] + kb];
    const double zp = za + zb;
    double A[3], B[3], P[3];
    double ab2 = 0.0;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        A[i] = a.centers[3 * si + i];
        B[i] = a.centers[3 * sj + i];
        P[i] = (za * A[i] + zb * B[i]) / zp;
        ab2 += (A[i] - B[i]) * (A[i] - B[i]);
    }
    for (int i = tid; i < 3 * ESZ; i += nthr) (&sE[0][0])[i] = 0.0;
    for (int i = tid; i < nsa * nca; i += nthr) sCa[i] = a.Ca[i];
    for (int i = tid; i < nsb * ncbt; i += nthr) sCb[i] = a.Cb[i];
    if (tid == 0) {
        int k = 0;
        for (int x = li; x >= 0; --x)
            for (int y = li - x; y >= 0; --y, ++k) { sca[k][0] = x; sca[k][1] = y; }
        k = 0;
        for (int x = lj; x >= 0; --x)
            for (int y = lj - x; y >= 0; --y, ++k) { scb[k][0] = x; scb[k][1] = y; }
        if (jb == 0) {
            double* s = a.scal + (size_t)ip * 8;
            s[0] = zp; s[1] = P[0]; s[2] = P[1]; s[3] = P[2];
            s[4] = -(za * zb / zp) * ab2;  // ln K_ab; made relative to the pair maximum by pair_finalize_kernel
            s[5] = 0.0; s[6] = 0.0; s[7] = 0.0;
        }
    }
    __syncthreads();
    // 1-D tables, one thread per axis (Eq.4: raise a at b = 0, Eq.5: raise b), seed (E_i)^0_00 = 1.
    if (tid < 3) {
        double* E = sE[tid];
        const double xpa = P[tid] - A[tid], xpb = P[tid] - B[tid], h = 0.5 / zp;
        E[0] = 1.0;
        for (int ai = 0; ai < li; ++ai)
            for (int t = 0; t <= ai + 1; ++t) {
                const double* e = E + (ai * NA1) * NT1;
                double v = xpa * e[t];
                if (t < ai) v += (t + 1) * e[t + 1];  // (E)^t_ab = 0 for t > a+b
                if (t > 0) v += h * e[t - 1];
                E[((ai + 1) * NA1) * NT1 + t] = v;
            }
        for (int ai = 0; ai <= li; ++ai)
            for (int bi = 0; bi < lj; ++bi)
                for (int t = 0; t <= ai + bi + 1; ++t) {
                    const double* e = E + (ai * NA1 + bi) * NT1;
                    double v = xpb * e[t];
                    if (t < ai + bi) v += (t + 1) * e[t + 1];
                    if (t > 0) v += h * e[t - 1];
                    E[(ai * NA1 + bi + 1) * NT1 + t] = v;
                }
    }
    __syncthreads();
    // half transform over b: Y[ac][mb][pp] = sum_bc Cb[mb][bc] Ex Ey Ez
    for (int idx = tid; idx < nca * nsb * 8; idx += nthr) {
        const int pp = idx & 7, mb = (idx >> 3) % nsb, ac = (idx >> 3) / nsb;
        const int col = jb * 8 + pp;
        double acc = 0.0;
        if (col < a.nherm) {
            const uint32_t w = a.tuv[col];
            const int t = w & 255, u = (w >> 8) & 255, v = (w >> 16) & 255;
            const int ax = sca[ac][0], ay = sca[ac][1], az = li - ax - ay;
            for (int bc = 0; bc < ncbt; ++bc) {
                const int bx = scb[bc][0], by = scb[bc][1], bz = lj - bx - by;
                if (t > ax + bx || u > ay + by || v > az + bz) continue;
                acc += sCb[mb * ncbt + bc] * (sE[0][(ax * NA1 + bx) * NT1 + t] * sE[1][(ay * NA1 + by) * NT1 + u] *
                                              sE[2][(az * NA1 + bz) * NT1 + v]);
            }
        }
        sY[idx] = acc;
    }
    __syncthreads();
    // half transform over a, contraction weight, blocked store
    const double wgt = a.coef[a.off[si] + ka] * a.coef[a.off[sj] + kb];
    double* Hp = a.H + (size_t)ip * a.hstride + (size_t)jb * a.nrb * 64;
    for (int idx = tid; idx < a.nab * 8; idx += nthr) {
        const int pp = idx & 7, row = idx >> 3;
        const int ma = row / nsb, mb = row % nsb;
        double acc = 0.0;
        for (int ac = 0; ac < nca; ++ac) acc += sCa[ma * nca + ac] * sY[(ac * nsb + mb) * 8 + pp];
        Hp[(row >> 3) * 64 + (row & 7) * 8 + pp] = wgt * acc;
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
    cudaError_t e = cudaMemsetAsync(pl.H, 0, nprim * pl.hstride * sizeof(double), st);
    if (e != cudaSuccess) return e;
    PairKernelArgs a;
    a.centers = ctx->d_centers; a.off = ctx->d_off; a.expo = ctx->d_exp; a.coef = ctx->d_coef;
    a.ij = pl.ij; a.tuv = ctx->tab.tuv; a.Ca = ctx->tab.solid[pl.li]; a.Cb = ctx->tab.solid[pl.lj];
    a.H = pl.H; a.scal = pl.scal;
    a.li = pl.li; a.lj = pl.lj; a.Ki = pl.Ki; a.Kj = pl.Kj;
    a.nab = pl.nab; a.nrb = pl.nrb; a.nherm = pl.nherm; a.ncb = pl.ncb; a.hstride = pl.hstride;
    const size_t nblk = nprim * pl.ncb;
    if (nblk > 2147483647ull) return cudaErrorInvalidValue;
    pair_h_kernel<<<(unsigned)nblk, 256, 0, st>>>(a);
    ctx->launches++;
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    pair_finalize_kernel<<<(pl.npair + 127) / 128, 128, 0, st>>>(pl.scal, pl.pairmax, pl.npair, kk);
    ctx->launches++;
    return cudaGetLastError();
}

}  // namespace md4

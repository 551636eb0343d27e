// md4_eri.cu -- the fused (ab|cd) kernel: S:8(a) steps a2-a9 in one launch.
//
// One CTA works on (one shell quartet) x (a group of 8-row blocks of the bra index ab); one warp owns
// one 8-row block.  Per primitive quartet the CTA builds the Hermite Coulomb tensor R (Eq.10-13) in
// shared memory; then every warp, independently,
//   GEMM1 (Eq.14/17):  T[8 x 8*NQT] = H_ab[8 rows, :] . G[:, q~ chunk],
//          A fragments straight from global/L2 (each H_ab row block is used by exactly one warp),
//          B fragments gathered from shared memory: G[p~,q~] = (-1)^{|q~|} R[p~+q~] (Eq.8) read at
//          address(p~) + address(q~) in the additive layout -- the 2-index integrals never exist in HBM
//          (the paper writes them out), and not in shared memory either;
//   GEMM2 (Eq.15/18):  out[8 x Ncd] += T . H_cd[:, chunk]^T, A fragments = the C fragments of
//          GEMM1 re-used in registers (the two DMMA k-steps of an 8-column block take the even and the
//          odd columns, which is exactly what a lane holds), B fragments from global through L1.
// Both contractions run on the FP64 tensor pipe (mma.sync m8n8k4 f64 -> SASS DMMA.8x8x4; tcgen05 has
// no f64 kind on sm_100a, S: facts table).  (ab|cd) accumulates in registers over all primitive
// quartets (Listing 2.1) and is written once.
#include "md4_device.cuh"

namespace md4 {

namespace {

struct EriArgs {
    const double* Hb; const double* sb; const double* pmb; size_t hsb;
    const double* Hk; const double* sk; const double* pmk; size_t hsk;
    int Kb, Kk, nbra, nket;
    int nab, ncd, nrb_ab, nrb_cd, ncb_p, ncb_q, nherm_p, nherm_q;
    int L, S, wpc, ncta_per_q;
    long long nitems;
    const uint32_t* rtab; const uint32_t* tuv; const double* boys;
    double* out;
};

__host__ __device__ inline size_t align16(size_t x) { return (x + 15) & ~(size_t)15; }

struct SmemLayout {
    size_t ra, rc0, rc1, ss, ap, aq, sg, total;
    __host__ __device__ SmemLayout(int L, int ncb_p, int ncb_q) {
        const int S = L + 1;
        size_t o = 0;
        ra = o; o += align16((size_t)S * S * S * 8);
        rc0 = o; o += align16((size_t)n_hermite(L) * 8);
        rc1 = o; o += align16((size_t)n_hermite(L) * 8);
        ss = o; o += 32 * 8;
        ap = o; o += align16((size_t)ncb_p * 8 * 4);
        aq = o; o += align16((size_t)ncb_q * 8 * 4);
        sg = o; o += align16((size_t)ncb_q * 4);
        total = o;
    }
};

template <int NT_CD, int NQT, int MAXW>
__global__ void __launch_bounds__(MAXW * 32, 1) eri_kernel(const EriArgs a) {
    extern __shared__ __align__(16) unsigned char smem[];
    const SmemLayout lay(a.L, a.ncb_p, a.ncb_q);
    double* Ra = reinterpret_cast<double*>(smem + lay.ra);
    double* Rc0 = reinterpret_cast<double*>(smem + lay.rc0);
    double* Rc1 = reinterpret_cast<double*>(smem + lay.rc1);
    double* sS = reinterpret_cast<double*>(smem + lay.ss);
    int* ap = reinterpret_cast<int*>(smem + lay.ap);   // byte offset of p~ in Ra, per H_ab column
    int* aq = reinterpret_cast<int*>(smem + lay.aq);   // byte offset of q~ in Ra, per H_cd column
    unsigned* sg = reinterpret_cast<unsigned*>(smem + lay.sg);  // per q~ block: bit c set if |q~| odd

    const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5;
    const int S = a.S, L = a.L;

    // per-class gather tables (padding columns point at R_000: finite value times a zero of H)
    for (int c = tid; c < a.ncb_p * 8; c += nthr) {
        int off = 0;
        if (c < a.nherm_p) { const uint32_t q = __ldg(a.tuv + c); off = (((q & 255) * S + ((q >> 8) & 255)) * S + ((q >> 16) & 255)) * 8; }
        ap[c] = off;
    }
    for (int c = tid; c < a.ncb_q * 8; c += nthr) {
        int off = 0;
        if (c < a.nherm_q) { const uint32_t q = __ldg(a.tuv + c); off = (((q & 255) * S + ((q >> 8) & 255)) * S + ((q >> 16) & 255)) * 8; }
        aq[c] = off;
    }
    for (int b = tid; b < a.ncb_q; b += nthr) {
        unsigned m = 0;
        for (int c = 0; c < 8; ++c) {
            const int col = b * 8 + c;
            if (col < a.nherm_q) { const uint32_t q = __ldg(a.tuv + col); m |= (((q & 255) + ((q >> 8) & 255) + ((q >> 16) & 255)) & 1u) << c; }
        }
        sg[b] = m;
    }
    __syncthreads();

    const int nchunk = (a.ncb_q + NQT - 1) / NQT;
    const unsigned char* RaB = reinterpret_cast<const unsigned char*>(Ra);
    const int k4 = lane & 3, n8 = lane >> 2;

    for (long long item = blockIdx.x; item < a.nitems; item += gridDim.x) {
        const long long quartet = item / a.ncta_per_q;
        const int ms = (int)(item % a.ncta_per_q);
        const int ib = (int)(quartet / a.nket), jk = (int)(quartet % a.nket);
        const int mbk = ms * a.wpc + warp;       // 8-row block of ab owned by this warp
        const bool active = (warp < a.wpc) && (mbk < a.nrb_ab);

        double2 acc[NT_CD];
#pragma unroll
        for (int i = 0; i < NT_CD; ++i) acc[i] = make_double2(0.0, 0.0);

        for (int kq = 0; kq < a.Kk; ++kq) {
            const double* sq = a.sk + ((size_t)jk * a.Kk + kq) * 8;
            const double* Hq = a.Hk + ((size_t)jk * a.Kk + kq) * a.hsk;
            for (int kp = 0; kp < a.Kb; ++kp) {
                const double* sp = a.sb + ((size_t)ib * a.Kb + kp) * 8;
                const double* Hp = a.Hb + ((size_t)ib * a.Kb + kp) * a.hsb;
                __syncthreads();  // every warp is done with the previous R
                hermite_r_block(Ra, Rc0, Rc1, sS, a.rtab, a.tuv, a.boys, L, S, __ldg(sp), __ldg(sp + 1),
                                __ldg(sp + 2), __ldg(sp + 3), __ldg(sq), __ldg(sq + 1), __ldg(sq + 2),
                                __ldg(sq + 3), exp(__ldg(sp + 4) + __ldg(sq + 4)), tid, nthr);
                if (!active) continue;
                const double* Ablk = Hp + (size_t)mbk * 64 + lane * 2;
                const size_t astride = (size_t)a.nrb_ab * 64;
                for (int ch = 0; ch < nchunk; ++ch) {
                    const int j0 = (int)((long long)ch * a.ncb_q / nchunk);
                    const int nq = (int)((long long)(ch + 1) * a.ncb_q / nchunk) - j0;
                    double2 T[NQT];
                    int aqr[NQT];
#pragma unroll
                    for (int n = 0; n < NQT; ++n) {
                        T[n] = make_double2(0.0, 0.0);
                        aqr[n] = (n < nq) ? aq[(j0 + n) * 8 + n8] : 0;
                    }
                    // ---- GEMM1: T = H_ab[8 rows] . G[:, chunk]
#pragma unroll 2
                    for (int jb = 0; jb < a.ncb_p; ++jb) {
                        const double2 av = __ldg(reinterpret_cast<const double2*>(Ablk + (size_t)jb * astride));
                        const int2 app = *reinterpret_cast<const int2*>(ap + jb * 8 + k4 * 2);
#pragma unroll
                        for (int n = 0; n < NQT; ++n) {
                            if (n < nq) {
                                const double b0 = *reinterpret_cast<const double*>(RaB + app.x + aqr[n]);
                                const double b1 = *reinterpret_cast<const double*>(RaB + app.y + aqr[n]);
                                dmma884(T[n].x, T[n].y, av.x, b0);
                                dmma884(T[n].x, T[n].y, av.y, b1);
                            }
                        }
                    }
                    // ---- sign of Eq.8 and GEMM2: acc += T . H_cd[:, chunk]^T
#pragma unroll
                    for (int n = 0; n < NQT; ++n) {
                        if (n < nq) {
                            const unsigned m = sg[j0 + n] >> (2 * k4);
                            const double tx = (m & 1u) ? -T[n].x : T[n].x;
                            const double ty = (m & 2u) ? -T[n].y : T[n].y;
                            const double* Bblk = Hq + ((size_t)(j0 + n) * a.nrb_cd) * 64 + lane * 2;
#pragma unroll
                            for (int nb = 0; nb < NT_CD; ++nb) {
                                if (nb < a.nrb_cd) {
                                    const double2 bv = __ldg(reinterpret_cast<const double2*>(Bblk + nb * 64));
                                    dmma884(acc[nb].x, acc[nb].y, tx, bv.x);
                                    dmma884(acc[nb].x, acc[nb].y, ty, bv.y);
                                }
                            }
                        }
                    }
                }
            }
        }
        // ---- epilogue: common factor K_ab K_cd of the pair maxima, applied in two halves so that
        // results near the bottom of the FP64 range are still correctly rounded
        if (active) {
            const double f = exp(0.5 * (__ldg(a.pmb + ib) + __ldg(a.pmk + jk)));
            const int row = mbk * 8 + n8;
            if (row < a.nab) {
                double* o = a.out + (size_t)quartet * a.nab * a.ncd + (size_t)row * a.ncd;
#pragma unroll
                for (int nb = 0; nb < NT_CD; ++nb) {
                    const int col = nb * 8 + 2 * k4;
                    if (col < a.ncd) o[col] = (acc[nb].x * f) * f;
                    if (col + 1 < a.ncd) o[col + 1] = (acc[nb].y * f) * f;
                }
            }
        }
    }
}

template <int NT_CD, int NQT, int MAXW>
md4_status launch_one(md4_ctx* ctx, const EriArgs& a, cudaStream_t st) {
    const SmemLayout lay(a.L, a.ncb_p, a.ncb_q);
    if (lay.total > (size_t)ctx->smem_optin) {
        ctx->err = "md4_compute: shared memory needed exceeds the device limit";
        return MD4_EUNSUPPORTED;
    }
    auto kern = eri_kernel<NT_CD, NQT, MAXW>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)lay.total);
    if (e != cudaSuccess) { ctx->err = std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e); return MD4_ECUDA; }
    long long grid = a.nitems < (long long)ctx->num_sms ? a.nitems : (long long)ctx->num_sms;
    kern<<<(unsigned)grid, a.wpc * 32, lay.total, st>>>(a);
    ctx->launches++;
    e = cudaGetLastError();
    if (e != cudaSuccess) { ctx->err = std::string("eri_kernel launch: ") + cudaGetErrorString(e); return MD4_ECUDA; }
    return MD4_OK;
}

template <int NT_CD>
md4_status launch_w(md4_ctx* ctx, const EriArgs& a, cudaStream_t st) {
    if (a.wpc <= 8) return launch_one<NT_CD, 8, 8>(ctx, a, st);
    return launch_one<NT_CD, 8, 12>(ctx, a, st);
}

}  // namespace

md4_status launch_eri(md4_ctx* ctx, const PairListDev& bra, const PairListDev& ket, double* d_out,
                      cudaStream_t st) {
    EriArgs a;
    a.Hb = bra.H; a.sb = bra.scal; a.pmb = bra.pairmax; a.hsb = bra.hstride;
    a.Hk = ket.H; a.sk = ket.scal; a.pmk = ket.pairmax; a.hsk = ket.hstride;
    a.Kb = bra.Ki * bra.Kj; a.Kk = ket.Ki * ket.Kj; a.nbra = bra.npair; a.nket = ket.npair;
    a.nab = bra.nab; a.ncd = ket.nab; a.nrb_ab = bra.nrb; a.nrb_cd = ket.nrb;
    a.ncb_p = bra.ncb; a.ncb_q = ket.ncb; a.nherm_p = bra.nherm; a.nherm_q = ket.nherm;
    a.L = bra.lsum + ket.lsum; a.S = a.L + 1;
    // warps per CTA = 8-row blocks per CTA; a quartet is split over ncta_per_q CTAs
    a.ncta_per_q = (a.nrb_ab + 11) / 12;
    a.wpc = (a.nrb_ab + a.ncta_per_q - 1) / a.ncta_per_q;
    a.nitems = (long long)a.nbra * a.nket * a.ncta_per_q;
    a.rtab = ctx->tab.rtab; a.tuv = ctx->tab.tuv; a.boys = ctx->tab.boys;
    a.out = d_out;
    const int nt = a.nrb_cd;
    if (nt <= 2) return launch_w<2>(ctx, a, st);
    if (nt <= 4) return launch_w<4>(ctx, a, st);
    if (nt <= 7) return launch_w<7>(ctx, a, st);
    if (nt <= 11) return launch_w<11>(ctx, a, st);
    if (nt <= 13) return launch_w<13>(ctx, a, st);
    if (nt <= 16) return launch_w<16>(ctx, a, st);
    if (nt <= 18) return launch_w<18>(ctx, a, st);
    if (nt <= 22) return launch_w<22>(ctx, a, st);
    ctx->err = "md4_compute: ket class too large";
    return MD4_EUNSUPPORTED;
}

// ---- stage-level debug kernels ---------------------------------------------------------------------
namespace {
__global__ void debug_boys_kernel(const double* tab, int mmax, int n, const double* T, double* out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n * (mmax + 1)) return;
    out[i] = boys_one(tab, i % (mmax + 1), T[i / (mmax + 1)]);
}

__global__ void debug_r_kernel(const uint32_t* rtab, const uint32_t* tuv, const double* boys, int L, const double* pq,
                               double* out) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int S = L + 1;
    double* Ra = reinterpret_cast<double*>(smem);
    double* Rc0 = Ra + S * S * S;
    double* Rc1 = Rc0 + n_hermite(L);
    double* sS = Rc1 + n_hermite(L);
    for (int i = threadIdx.x; i < S * S * S; i += blockDim.x) Ra[i] = 0.0;
    __syncthreads();
    hermite_r_block(Ra, Rc0, Rc1, sS, rtab, tuv, boys, L, S, pq[0], pq[1], pq[2], pq[3], pq[4], pq[5], pq[6], pq[7],
                    1.0, threadIdx.x, blockDim.x);
    __syncthreads();
    for (int i = threadIdx.x; i < S * S * S; i += blockDim.x) out[i] = Ra[i];
}
}  // namespace

cudaError_t launch_debug_boys(md4_ctx* ctx, int mmax, int n, const double* d_T, double* d_out) {
    const int tot = n * (mmax + 1);
    debug_boys_kernel<<<(tot + 127) / 128, 128>>>(ctx->tab.boys, mmax, n, d_T, d_out);
    ctx->launches++;
    return cudaGetLastError();
}

cudaError_t launch_debug_r(md4_ctx* ctx, int L, const double* d_pq, double* d_out) {
    const int S = L + 1;
    const size_t sm = ((size_t)S * S * S + 2 * (size_t)n_hermite(L) + 32) * 8;
    cudaError_t e = cudaFuncSetAttribute(debug_r_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) return e;
    debug_r_kernel<<<1, 256, sm>>>(ctx->tab.rtab, ctx->tab.tuv, ctx->tab.boys, L, d_pq, d_out);
    ctx->launches++;
    return cudaGetLastError();
}

}  // namespace md4

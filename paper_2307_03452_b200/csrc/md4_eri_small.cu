// md4_eri_small.cu -- (ab|cd) for LOW angular momenta (S:8(f) item 1: the (dd|dd), (ff|ff) rows of the paper's Table 1,
// P:216-222): uncontracted classes with at most 7 eight-row blocks on either side and L = l_a+l_b+l_c+l_d <= 12.
//
// A quartet of such a class is a few hundred to a few thousand DMMAs -- microseconds of tensor work.  The fused kernel
// of md4_eri.cu spends far longer than that per quartet on what surrounds the contractions: two block barriers, the
// scatter of R, the round trip of the H_cd ring and the first H_ab fragments from L2 (measured: 4.8 % of the FP64 peak
// for (dd|dd), 26 % for (ff|ff)).  Here ONE WARP computes a whole quartet on its own, with no block-level
// synchronisation at all, and the SM hides the latencies of one warp behind the other 8-24 warps it holds:
//   a2-a4  the warp builds R of its quartet in its own shared-memory slab (hermite_r_warp: Boys, seeds, Eq.13 in place,
//          P:85-97) and scatters it into an additive layout of its own, addr(t,u,v) = t (L+1)^2 + u (L+1) + v;
//   a5-a6  per 8-row block of ab: T[8 x N_q~] = H_ab[rows, :] . G, G[p~,q~] = (-1)^{|q~|} R[p~+q~] gathered at
//          addr(p~) + addr(q~) (Eq.8; Eq.14/17), A fragments from L1/L2 (the warps of a CTA share the bra pair);
//   a7     (ab|cd)[rows, :] = (sign . T) . H_cd^T (Eq.15/18) with B fragments straight from L1/L2, C fragments of GEMM1
//          re-used as A fragments in registers as in md4_eri.cu;
//   a9     the 8 x N_cd block is scaled and stored; next row block.
// Same H layouts, column orders and tables as the fused kernel (md4_internal.h); both contractions on DMMA.8x8x4.
#include "md4_device.cuh"

namespace md4 {

namespace {

constexpr int SM_LMAX = 12;          // highest L
constexpr int SM_NQ = 12;            // q~ / p~ column blocks, at most (84 Hermite functions for l_pair = 6, 96 columns with padding)
constexpr int SM_NCD = 7;            // 8-column blocks of cd, at most

struct SmallArgs {
    const double* Hb; const double* sb; const double* pmb; size_t hsb;
    const double* Hk; const double* sk; const double* pmk; size_t hsk;
    int nbra, nket, nab, ncd, nrb_ab, nrb_cd, ncb_p, ncb_q, L;
    long long nquartets;
    const uint32_t* rtab; const double* boys;
    KernelSpec ks;
    const uint32_t* colp; const uint32_t* colq; const uint32_t* tuv;
    double* out;
};

// per-CTA tables | per-warp slabs: additive R (L+1)^3 | graded R n_h(L) + L | seeds 32
struct SmallSmem {
    size_t ap, aq, sg, ad, slab0, slab, ra, ga, ss, total;
    __host__ __device__ SmallSmem(int L, int ncb_p, int ncb_q, int nwarps) {
        size_t o = 0;
        ap = o; o += (size_t)(ncb_p + 1) * 8 * 4;
        aq = o; o += (size_t)ncb_q * 8 * 4;
        sg = o; o += (size_t)((ncb_q + 3) / 4 * 4) * 4;
        ad = o; o += (size_t)((n_hermite(L) + 7) / 8 * 8) * 2;
        o = (o + 127) / 128 * 128;
        slab0 = o;
        size_t s = 0;
        ra = s; s += (size_t)(L + 1) * (L + 1) * (L + 1) * 8;
        ga = s; s += (size_t)((r_graded_alloc(L) + 1) / 2 * 2) * 8;
        ss = s; s += 32 * 8;
        slab = (s + 127) / 128 * 128;
        total = slab0 + slab * nwarps;
    }
};

__device__ __forceinline__ double2 ldg2s(const double* p) { return __ldg(reinterpret_cast<const double2*>(p)); }

// NQ / NCD: q~ (p~) column blocks and cd blocks, at most; NW: warps (quartets in flight) per CTA
template <int NQ, int NCD, int NW>
__global__ void __launch_bounds__(NW * 32) eri_small_kernel(const SmallArgs a) {
    extern __shared__ __align__(128) unsigned char smem[];
    const SmallSmem lay(a.L, a.ncb_p, a.ncb_q, NW);
    int* ap = reinterpret_cast<int*>(smem + lay.ap);
    int* aq = reinterpret_cast<int*>(smem + lay.aq);
    unsigned* sg = reinterpret_cast<unsigned*>(smem + lay.sg);
    uint16_t* sad = reinterpret_cast<uint16_t*>(smem + lay.ad);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int L = a.L, S1 = L + 1, S2 = S1 * S1;
    unsigned char* slab = smem + lay.slab0 + lay.slab * warp;
    double* Ra = reinterpret_cast<double*>(slab + lay.ra);
    double* GA = reinterpret_cast<double*>(slab + lay.ga);
    double* sS = reinterpret_cast<double*>(slab + lay.ss);

    // tables shared by the CTA: byte offsets of the p~ / q~ columns in the additive layout, sign bits (Eq.8), and the
    // additive address of every graded ordinal
    for (int c = tid; c < (a.ncb_p + 1) * 8; c += blockDim.x) {
        const uint32_t q = c < a.ncb_p * 8 ? __ldg(a.colp + c) : 0u;
        ap[c] = (q & COL_PAD) ? 0 : (int)(((q & 255) * S2 + ((q >> 8) & 255) * S1 + ((q >> 16) & 255)) * 8);
    }
    for (int c = tid; c < a.ncb_q * 8; c += blockDim.x) {
        const uint32_t q = __ldg(a.colq + c);
        aq[c] = (q & COL_PAD) ? 0 : (int)(((q & 255) * S2 + ((q >> 8) & 255) * S1 + ((q >> 16) & 255)) * 8);
    }
    for (int b = tid; b < a.ncb_q; b += blockDim.x) {
        unsigned m = 0;
        for (int c = 0; c < 8; ++c) {
            const uint32_t q = __ldg(a.colq + b * 8 + c);
            if (!(q & COL_PAD)) m |= (((q & 255) + ((q >> 8) & 255) + ((q >> 16) & 255)) & 1u) << c;
        }
        sg[b] = m;
    }
    for (int e = tid; e < n_hermite(L); e += blockDim.x) {
        const uint32_t q = __ldg(a.tuv + e);
        sad[e] = (uint16_t)((q & 255) * S2 + ((q >> 8) & 255) * S1 + ((q >> 16) & 255));
    }
    // the slab's additive array: only addresses with t+u+v <= L are ever written; a padding column reads address 0
    // (R_000, finite) against a zero of H, sums t+u+v > L never occur
    for (int i = lane; i < S1 * S2; i += 32) Ra[i] = 0.0;
    __syncthreads();

    const int k4 = lane & 3, n8 = lane >> 2;
    const uint32_t ra32 = smem_u32(Ra);
    const uint32_t ap32 = smem_u32(ap) + (uint32_t)k4 * 8u;
    const uint32_t aq32 = smem_u32(aq) + (uint32_t)n8 * 4u;
    const size_t astride = (size_t)a.nrb_ab * 64, bstride = (size_t)a.nrb_cd * 64;
    const long long gw = (long long)blockIdx.x * NW + warp, nw = (long long)gridDim.x * NW;

    for (long long qt = gw; qt < a.nquartets; qt += nw) {
        const int ib = (int)(qt / a.nket), jk = (int)(qt % a.nket);
        // ---- a2-a4: R of this quartet, graded order in place, then the additive layout
        {
            const double* sp = a.sb + (size_t)ib * 8;
            const double* sq = a.sk + (size_t)jk * 8;
            hermite_r_warp(GA, sS, a.rtab, a.boys, a.ks, L, __ldg(sp), __ldg(sp + 1), __ldg(sp + 2), __ldg(sp + 3), __ldg(sq),
                           __ldg(sq + 1), __ldg(sq + 2), __ldg(sq + 3), exp(__ldg(sp + 4) + __ldg(sq + 4)), lane, [] {});
            __syncwarp();
            for (int e = lane; e < n_hermite(L); e += 32) Ra[sad[e]] = GA[e];
            __syncwarp();
        }
        const double f = exp(0.5 * (__ldg(a.pmb + ib) + __ldg(a.pmk + jk)));
        const double* Hp = a.Hb + (size_t)ib * a.hsb + lane * 2;
        const double* Hq = a.Hk + (size_t)jk * a.hsk + lane * 2;
        uint32_t aqr[NQ];
#pragma unroll
        for (int n = 0; n < NQ; ++n) aqr[n] = ra32 + (n < a.ncb_q ? lds_u32(aq32 + (uint32_t)n * 32u) : 0u);
        for (int rb = 0; rb < a.nrb_ab; ++rb) {
            // ---- a5-a6 GEMM1: T = H_ab[rows of rb, :] . G
            double2 T[NQ];
#pragma unroll
            for (int n = 0; n < NQ; ++n) T[n] = make_double2(0.0, 0.0);
            const double* Ab = Hp + (size_t)rb * 64;
            double2 an = ldg2s(Ab), an2 = ldg2s(Ab + (size_t)min(1, a.ncb_p - 1) * astride);
            for (int jb = 0; jb < a.ncb_p; ++jb) {
                const double2 av = an;
                an = an2;
                an2 = ldg2s(Ab + (size_t)min(jb + 2, a.ncb_p - 1) * astride);
                const int2 app = lds_v2s32(ap32 + (uint32_t)jb * 32u);
                double b[NQ];
#pragma unroll
                for (int n = 0; n < NQ; ++n)
                    if (n < a.ncb_q) b[n] = lds_f64((uint32_t)app.x + aqr[n]);
#pragma unroll
                for (int n = 0; n < NQ; ++n)
                    if (n < a.ncb_q) dmma884(T[n].x, T[n].y, av.x, b[n]);
#pragma unroll
                for (int n = 0; n < NQ; ++n)
                    if (n < a.ncb_q) b[n] = lds_f64((uint32_t)app.y + aqr[n]);
#pragma unroll
                for (int n = 0; n < NQ; ++n)
                    if (n < a.ncb_q) dmma884(T[n].x, T[n].y, av.y, b[n]);
            }
            // ---- a7 GEMM2: (ab|cd)[rows, :] = (sign . T) . H_cd^T
            double2 acc[NCD];
#pragma unroll
            for (int i = 0; i < NCD; ++i) acc[i] = make_double2(0.0, 0.0);
            double2 bv[NCD];
#pragma unroll
            for (int i = 0; i < NCD; ++i)
                if (i < a.nrb_cd) bv[i] = ldg2s(Hq + (size_t)i * 64);
#pragma unroll
            for (int n = 0; n < NQ; ++n) {
                if (n < a.ncb_q) {
                    const uint32_t m = sg[n] >> (2 * k4);
                    const double tx = (m & 1u) ? -T[n].x : T[n].x;
                    const double ty = (m & 2u) ? -T[n].y : T[n].y;
                    // the B fragments of the next q~ block are requested before this block's DMMAs are issued
                    const double* Bn = Hq + (size_t)min(n + 1, a.ncb_q - 1) * bstride;
                    double2 bw[NCD];
#pragma unroll
                    for (int i = 0; i < NCD; ++i)
                        if (i < a.nrb_cd) bw[i] = ldg2s(Bn + (size_t)i * 64);
#pragma unroll
                    for (int i = 0; i < NCD; ++i)
                        if (i < a.nrb_cd) dmma884(acc[i].x, acc[i].y, tx, bv[i].x);
#pragma unroll
                    for (int i = 0; i < NCD; ++i)
                        if (i < a.nrb_cd) dmma884(acc[i].x, acc[i].y, ty, bv[i].y);
#pragma unroll
                    for (int i = 0; i < NCD; ++i) bv[i] = bw[i];
                }
            }
            // ---- a9: scale by K_ab K_cd of the pair (in two halves, as in md4_eri.cu) and store the 8 x N_cd block
            const int row = rb * 8 + n8;
            if (row < a.nab) {
                double* o = a.out + ((size_t)qt * a.nab + row) * a.ncd;
#pragma unroll
                for (int i = 0; i < NCD; ++i) {
                    const int col = i * 8 + 2 * k4;
                    if (col < a.ncd) __stcs(o + col, (acc[i].x * f) * f);
                    if (col + 1 < a.ncd) __stcs(o + col + 1, (acc[i].y * f) * f);
                }
            }
        }
        __syncwarp();   // every lane is done with Ra / GA before the next quartet's build overwrites them
    }
}

template <int NQ, int NCD, int NW>
md4_status launch_small_one(md4_ctx* ctx, SmallArgs& a, cudaStream_t st) {
    const SmallSmem lay(a.L, a.ncb_p, a.ncb_q, NW);
    if (lay.total > (size_t)ctx->smem_optin) { ctx->err = "md4_compute: small-class kernel needs too much shared memory"; return MD4_EUNSUPPORTED; }
    auto kern = eri_small_kernel<NQ, NCD, NW>;
    cudaError_t e = cudaSuccess;
    if (ctx->configured.insert(reinterpret_cast<const void*>(kern)).second) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, ctx->smem_optin);
        if (e != cudaSuccess) { ctx->configured.erase(reinterpret_cast<const void*>(kern)); ctx->err = std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e); return MD4_ECUDA; }
    }
    // resident CTAs per SM (shared memory and registers decide): the grid is persistent, one quartet per warp at a time
    int per_sm = 1;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, NW * 32, lay.total);
    if (e != cudaSuccess || per_sm < 1) { (void)cudaGetLastError(); per_sm = 1; }
    const long long want = (a.nquartets + NW - 1) / NW;
    const long long slots = (long long)ctx->num_sms * per_sm;
    const long long grid = want < slots ? want : slots;
    kern<<<(unsigned)grid, NW * 32, lay.total, st>>>(a);
    ctx->launches++;
    e = cudaGetLastError();
    if (e != cudaSuccess) { ctx->err = std::string("eri_small_kernel launch: ") + cudaGetErrorString(e); return MD4_ECUDA; }
    return MD4_OK;
}

}  // namespace

bool small_class_eligible(const PairListDev& bra, const PairListDev& ket) {
    return bra.Ki * bra.Kj == 1 && ket.Ki * ket.Kj == 1 && bra.nrb <= SM_NCD && ket.nrb <= SM_NCD && bra.ncbb <= SM_NQ &&
           ket.ncbk <= SM_NQ && bra.lsum + ket.lsum <= SM_LMAX;
}

md4_status launch_eri_small(md4_ctx* ctx, const PairListDev& bra, const PairListDev& ket, double* d_out, cudaStream_t st) {
    SmallArgs a;
    a.Hb = bra.Hb; a.sb = bra.scal; a.pmb = bra.pairmax; a.hsb = bra.hstrideb;
    a.Hk = ket.Hk; a.sk = ket.scal; a.pmk = ket.pairmax; a.hsk = ket.hstridek;
    a.nbra = bra.npair; a.nket = ket.npair;
    a.nab = bra.nab; a.ncd = ket.nab; a.nrb_ab = bra.nrb; a.nrb_cd = ket.nrb;
    a.ncb_p = bra.ncbb; a.ncb_q = ket.ncbk;
    a.L = bra.lsum + ket.lsum;
    a.nquartets = (long long)a.nbra * a.nket;
    a.rtab = ctx->tab.rtab; a.boys = ctx->tab.boys; a.tuv = ctx->tab.tuv;
    a.ks = ctx->kernel;
    a.colp = ctx->tab.colb[bra.lsum]; a.colq = ctx->tab.colk[ket.lsum];
    a.out = d_out;
    // up to (dd|dd): 6 column blocks, 4 blocks of cd, L = 8 (7.6 kB per warp): 16 warps per CTA at <= 128 registers;
    // up to (ff|ff): L = 12 (21.5 kB per warp): 8 warps per CTA
    if (a.ncb_q <= 6 && a.ncb_p <= 6 && a.nrb_cd <= 4 && a.L <= 8) return launch_small_one<6, 4, 16>(ctx, a, st);
    return launch_small_one<SM_NQ, SM_NCD, 8>(ctx, a, st);
}

}  // namespace md4

// md4_eri.cu -- the fused (ab|cd) kernel: S:8(a) steps a2-a9 in one launch.
//
// One CTA works on (one shell quartet) x (a group of 8-row blocks of the bra index ab); one consumer warp
// owns one 8-row block, one extra warp is the producer of the H_cd ring AND the builder of the Hermite
// Coulomb tensor R (Eq.10-13): while the consumers contract primitive quartet i it builds R of primitive
// quartet i+1 in graded order in its own shared-memory buffers (hermite_r_warp); between two primitive
// quartets all threads scatter that array into the additive layout (two barriers, ~1 % of the time; the
// recurrence itself is off the critical path).  Per primitive quartet every consumer warp, independently,
//   GEMM1 (Eq.14/17):  T[8 x 8*NQT] = H_ab[8 rows, :] . G[:, q~ chunk],
//          A fragments straight from global/L2, software-prefetched two k-blocks ahead (each H_ab row
//          block is used by exactly one warp),
//          B fragments gathered from shared memory: G[p~,q~] = (-1)^{|q~|} R[p~+q~] (Eq.8) read at
//          address(p~) + address(q~) in the additive layout -- the 2-index integrals never exist in HBM
//          (the paper writes them out), and not in shared memory either.  The column orders of
//          H_ab / H_cd make this gather free of bank conflicts (md4_internal.h "Column orders");
//   GEMM2 (Eq.15/18):  out[8 x Ncd] += T . H_cd[:, chunk]^T, A fragments = the C fragments of
//          GEMM1 re-used in registers (the two DMMA k-steps of an 8-column block take the even and the
//          odd columns, which is exactly what a lane holds), B fragments from a shared-memory ring of
//          H_cd column blocks that the producer warp fills with 1-D bulk copies (TMA) and all consumer
//          warps of the CTA share (full/empty mbarriers per stage).
// Both contractions run on the FP64 tensor pipe (mma.sync m8n8k4 f64 -> SASS DMMA.8x8x4; tcgen05 has
// no f64 kind on sm_100a, S: facts table).  (ab|cd) accumulates in registers over all primitive
// quartets (Listing 2.1) and is written once.
#include "md4_device.cuh"
#include <mutex>
#include <string>

namespace md4 {

namespace {

constexpr int MAX_STAGES = 16;

// Kernel instantiations by MAXW: 12 = bras with 10-11 row blocks per item (gg, ih, ii: three consumer warps per
// sub-partition) + 1 producer warp; 10 = bras with 8 row blocks per item (hh, ig: two consumer warps per sub-partition) + 4
// warps that build R, one per sub-partition; 11 = bras with 10 row blocks per item (ih: 10 + 8) under kets of at most 16
// column blocks + 2 builder warps, which sit on the two sub-partitions with two consumer warps ((ih|hg) 64.7 -> 67.7 %,
// (ih|ig) 68.3 -> 70.1 %; under ih kets one producer is as good: 73.5 %); 9 = bras with up to 7 (hg: 7 + 6 under ih / ii kets) + 1 producer warp, which
// then sits on the sub-partition with one consumer warp; 16 = bras of 12-15 row blocks (hg, ig) as ONE item under kets of
// at most 16 column blocks, 128 registers (see launch_eri_with); 8 / 4 = small classes, 2 / 3 CTAs per SM.  Registers are allocated per 4 warps, so
// the 12 warps of MAXW = 10 cost no more than 9 (168 registers either way).
// Why 4 builders: one producer warp took 6 % from the two consumer warps it shared a sub-partition with, and the other six
// waited for those two at the block barrier; spread over the four sub-partitions the same work costs every warp 1.5 %
// ((hh|gg) 2.90 -> 2.52 ms, (hh|hg) 3.80 -> 3.48, (ig|ig) 4.75 -> 4.53).
__host__ __device__ constexpr int builder_warps(int maxw) { return maxw == 10 ? 4 : (maxw == 11 ? 2 : 1); }
__host__ __device__ constexpr int cta_warps_max(int maxw) { return (maxw == 10 || maxw == 11) ? 12 : maxw; }

// How many k-blocks ahead GEMM1 loads its H_ab fragments (16 bytes per lane and k-block, from L2), per kernel
// instantiation; nt = 8-column blocks of the ket.  Measured on the 21 classes of cfg5 (K = 1) with depths 1, 2, 4, 5 in
// every slot; every extra k-block costs 4 registers and 4 moves per k-block, and the differences are 0-9 % (e.g. (ih|ih)
// 7.91 / 8.17 / 8.02 / 8.17 ms, (hh|hh) with four builders 4.70 / 5.03 / 4.62 / - ms).
__host__ __device__ constexpr int pf_depth(int maxw, int nt) {
    if (maxw == 16) return 2;   // wide items at 128 registers: 1 / 2 / 3 / 5 measured, (ig|ig) 4.11 / 4.04 / 4.10 / 4.17 ms
    if (maxw == 10) return nt == 11 ? 1 : ((nt == 13 || nt == 15 || nt == 16) ? 4 : 2);
    if (maxw <= 9) return (nt == 11 || nt == 13) ? 4 : 2;
    return (nt == 15 || nt == 16) ? 5 : (nt == 18 ? 1 : 2);
}

struct EriArgs {
    const double* Hb; const double* sb; const double* pmb; size_t hsb;
    const double* Hk; const double* sk; const double* pmk; size_t hsk;
    int Kb, Kk, nbra, nket;
    int nab, ncd, nrb_ab, nrb_cd, ncb_p, ncb_q;
    int L, wpc, ncta_per_q, nst;
    int row0[3], nrows[3];   // 8-row blocks of ab of the ncta_per_q work items of one quartet (plan_items)
    long long nquartets;
    int qmajor;   // 1: a CTA takes whole quartets (items of unequal size); 0: the items of a quartet go to neighbouring CTAs
    int tb;       // bra pairs per strip of the quartet order (quartet_pairs)
    const uint32_t* rtab; const uint32_t* tuv; const double* boys;
    KernelSpec ks;   // interaction kernel (md4_set_kernel)
    double* tacc;   // [grid][wpc][ncb_q][32][2] partial [ab|q~] of contracted bras
    const uint32_t* colp; const uint32_t* colq;   // bra-order columns of the bra class, ket-order columns of the ket class
    double* out;
    // direct digestion (md4_compute_jk): instead of storing (ab|cd), J[a,b] += sum_cd (ab|cd) D[c,d] and
    // K[a,c] += sum_bd (ab|cd) D[b,d] on AO matrices [nbf x nbf]; aob / aok = AO offsets of the shells of every pair
    int digest, nbf, nsb, nsd;        // nsb = 2 l_b + 1, nsd = 2 l_d + 1
    const int* aob; const int* aok;
    const double* D; double* J; double* K;
};

__host__ __device__ inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Shared memory: R in the additive layout | H_cd ring | graded R of the next primitive quartet (GA) | seeds | gather offsets of the p~ and q~ columns | sign bits | Eq.13 table |
// additive address per graded ordinal | mbarriers.
struct SmemLayout {
    size_t ra, un, ga, ss, ap, aq, sg, rt, ad, bars, dg, total, stage_bytes;
    // digest: D_cd of the ket pair (padded to whole column blocks), D_bd, column -> (mc, md)
    static constexpr int DG_TILE = (2 * LMAX + 1) * (2 * LMAX + 1);
    __host__ __device__ SmemLayout(int L, int ncb_p, int ncb_q, int nrb_cd, int nst, int digest = 0) {
        size_t o = 0;
        ra = o; o += align_up((size_t)r_alloc(L) * 8, 128);
        stage_bytes = (size_t)nrb_cd * 64 * 8;
        un = o; o += align_up(stage_bytes * nst, 128);
        ga = o; o += align_up((size_t)r_graded_alloc(L) * 8, 16);
        ss = o; o += 32 * 8;
        ap = o; o += align_up((size_t)(ncb_p + 1) * 8 * 4, 16);   // one block of slack: the k-loop prefetches
        aq = o; o += align_up((size_t)ncb_q * 8 * 4, 16);
        sg = o; o += align_up((size_t)ncb_q * 4, 16);
        rt = o; o += align_up((size_t)n_hermite(L) * 4, 16);   // Eq.13 table
        ad = o; o += align_up((size_t)n_hermite(L) * 2, 16);   // additive address per graded ordinal
        bars = o; o += 2 * MAX_STAGES * 8;
        dg = o;
        if (digest) o += (size_t)nrb_cd * 64 + DG_TILE * 8 + align_up((size_t)nrb_cd * 8 * 2, 16);
        total = o;
    }
};

__device__ __forceinline__ double2 ldg2(const double* p) { return __ldg(reinterpret_cast<const double2*>(p)); }

// Order in which the persistent grid walks the quartets: the bra list is cut into strips of tb pairs and a strip is walked
// ket-major, so the ~74 quartets the 148 CTAs work on at any time are tb bra pairs x 2-3 ket pairs: their H matrices
// (0.6 MB each for ii) stay in L2 while they are in use, every H_cd is read from HBM once per strip and every H_ab once.
// (Walking the flat list [bra][ket] put one bra and 74 different kets in flight and re-read H_cd from HBM 28 times over:
// 8.6 GB per cfg3 launch against 0.3 GB of pair data, profiles/r1_eri_kernel_ncu.md.)
__device__ __forceinline__ void quartet_pairs(const EriArgs& a, long long q, int& ib, int& jk) {
    const long long per_strip = (long long)a.tb * a.nket;
    const int strip = (int)(q / per_strip);
    const int r = (int)(q - strip * per_strip);
    const int b0 = strip * a.tb;
    const int hb = min(a.tb, a.nbra - b0);
    jk = r / hb;
    ib = b0 + r % hb;
}

// Position in the H_cd ring; every warp of the CTA (producer, consumers with and without rows) steps
// through the same sequence of column blocks, so the positions stay equal without communication.
struct RingPos {
    uint32_t s, ph;
    __device__ __forceinline__ void advance(uint32_t nst) {
        if (++s == nst) { s = 0; ph ^= 1u; }
    }
};

// All shared-memory operands of the consumer loop are addressed by 32-bit shared addresses.
struct ConsumerCtx {
    const double* Ablk;    // this lane's A fragment pair of k-block 0 of the warp's 8-row block of H_ab
    size_t astride;        // doubles between k-blocks of H_ab
    uint32_t ra32;         // R in the additive layout
    uint32_t ap32;         // ap + k4*2 (this lane's pair of p~ offsets in k-block 0)
    uint32_t aq32;         // aq + n8 (this lane's q~ offset in q-block 0)
    uint32_t sg32;         // sign bits per q-block
    uint32_t ring32;       // ring + lane*16 bytes (this lane's B fragment pair of GEMM2)
    uint32_t full32, empty32;
    uint32_t stage_bytes, nst;
    int ncb_p, nrb_cd, k4, lane;
    double* tacc;          // this lane's slot of the [ab|q~] scratch of its warp (q-block 0), contracted bras only
};

// One chunk of NQ q~ blocks for one warp: T = H_ab[8 rows] . G[:, chunk] (GEMM1), then
// acc += (sign . T) . H_cd[:, chunk]^T (GEMM2) against the ring.  PRED: q-blocks n >= nq are skipped
// (general classes); otherwise nq == NQ.  EXACT: nrb_cd == NT_CD.
template <int NQ, int NT_CD, bool EXACT, bool PRED, int PF>
__device__ __forceinline__ void consume_chunk(double2 (&acc)[NT_CD], const ConsumerCtx& c, int j0, int nq, RingPos& rp,
                                              bool load_t, bool last_kp) {
    double2 T[NQ];
    uint32_t aqr[NQ];
#pragma unroll
    for (int n = 0; n < NQ; ++n) {
        // [ab|q~] accumulates over the bra primitives (Listing 2.1 line 7): from the second one on the
        // accumulators start from the sum so far, kept in an L2-resident scratch in fragment layout
        T[n] = (load_t && (!PRED || n < nq)) ? *reinterpret_cast<const double2*>(c.tacc + (size_t)(j0 + n) * 64)
                                             : make_double2(0.0, 0.0);
        aqr[n] = c.ra32 + ((!PRED || n < nq) ? lds_u32(c.aq32 + (uint32_t)(j0 + n) * 32u) : 0u);
    }
    // ---- GEMM1: the B operand is G[p~,q~] = +-R[p~+q~] read at address(p~) + address(q~) (Eq.8)
    // H_ab fragments come from L2 (~1 us), PF k-blocks ahead (pf_depth above).
    // The address of the fragment PF k-blocks ahead is a running pointer (2 instructions per k-block; indexing it as
    // Ablk[(jb + PF) * astride] compiled to a 64-bit multiply-add chain of 7 and cost 3 % of the kernel: three warps per
    // sub-partition issue ~4 instructions per 16-clock DMMA each, the issue port is the second bottleneck).  The load stays
    // predicated: unconditional loads (into slack behind the list) save 4 moves per k-block but make the assembler hoist
    // them and spill accumulators (measured: 55.2-57.3 ms against 54.7 on cfg3).
    double2 af[PF];
#pragma unroll
    for (int i = 0; i < PF; ++i) af[i] = i < c.ncb_p ? ldg2(c.Ablk + (size_t)i * c.astride) : make_double2(0.0, 0.0);
    const double* apf = c.Ablk + (size_t)PF * c.astride;
    uint32_t app32 = c.ap32;
    int2 apn = lds_v2s32(app32);
    for (int jb = 0; jb < c.ncb_p; ++jb) {
        const double2 av = af[0];
#pragma unroll
        for (int i = 0; i + 1 < PF; ++i) af[i] = af[i + 1];
        if (jb + PF < c.ncb_p) af[PF - 1] = ldg2(apf);
        apf += c.astride;
        const int2 app = apn;
        app32 += 32u;
        apn = lds_v2s32(app32);   // the ap array has one block of slack
        double b[NQ];
#pragma unroll
        for (int n = 0; n < NQ; ++n)
            if (!PRED || n < nq) b[n] = lds_f64((uint32_t)app.x + aqr[n]);
#pragma unroll
        for (int n = 0; n < NQ; ++n)
            if (!PRED || n < nq) dmma884(T[n].x, T[n].y, av.x, b[n]);
#pragma unroll
        for (int n = 0; n < NQ; ++n)
            if (!PRED || n < nq) b[n] = lds_f64((uint32_t)app.y + aqr[n]);
#pragma unroll
        for (int n = 0; n < NQ; ++n)
            if (!PRED || n < nq) dmma884(T[n].x, T[n].y, av.y, b[n]);
    }
    if (!last_kp) {
        // more bra primitives to come: park the partial [ab|q~]; the ket transform runs once per ket primitive
#pragma unroll
        for (int n = 0; n < NQ; ++n)
            if (!PRED || n < nq) *reinterpret_cast<double2*>(c.tacc + (size_t)(j0 + n) * 64) = T[n];
        return;
    }
    // ---- sign of Eq.8 and GEMM2: acc += T . H_cd[:, chunk]^T
#pragma unroll
    for (int n = 0; n < NQ; ++n) {
        if (!PRED || n < nq) {
            const uint32_t m = lds_u32(c.sg32 + (uint32_t)(j0 + n) * 4u) >> (2 * c.k4);
            const double tx = (m & 1u) ? -T[n].x : T[n].x;
            const double ty = (m & 2u) ? -T[n].y : T[n].y;
            mbar_wait32(c.full32 + rp.s * 8u, rp.ph);
            const uint32_t bb = c.ring32 + rp.s * c.stage_bytes;
            constexpr int G = 4;   // B fragment pairs in flight
            int landed = 0;        // OR of a word of every B fragment of the stage: unknown to the assembler, see the release below
#pragma unroll
            for (int nb0 = 0; nb0 < NT_CD; nb0 += G) {
                double2 bv[G];
#pragma unroll
                for (int g = 0; g < G; ++g)
                    if (nb0 + g < NT_CD && (EXACT || nb0 + g < c.nrb_cd)) bv[g] = lds_v2f64(bb + (uint32_t)(nb0 + g) * 512u);
#pragma unroll
                for (int g = 0; g < G; ++g)
                    if (nb0 + g < NT_CD && (EXACT || nb0 + g < c.nrb_cd)) dmma884(acc[nb0 + g].x, acc[nb0 + g].y, tx, bv[g].x);
#pragma unroll
                for (int g = 0; g < G; ++g)
                    if (nb0 + g < NT_CD && (EXACT || nb0 + g < c.nrb_cd)) dmma884(acc[nb0 + g].x, acc[nb0 + g].y, ty, bv[g].y);
#pragma unroll
                for (int g = 0; g < G; ++g)
                    if (nb0 + g < NT_CD && (EXACT || nb0 + g < c.nrb_cd)) landed |= __double2loint(bv[g].y);
            }
            __syncwarp();
            // release the stage.  The arrive takes `landed` as an input, a value that depends on every B fragment of the
            // stage: it cannot be scheduled before all loads of the stage have delivered their data.  (Without it ptxas
            // places the arrive right behind the ISSUE of the last LDS; the producer may then refill the stage while
            // loads of it are still in flight -- the write-after-read race of DESIGN.md 6.1.)
            if (c.lane == 0) mbar_arrive32_dep(c.empty32 + rp.s * 8u, landed);
            rp.advance(c.nst);
        }
    }
}

template <int NT_CD, int NQT, int MAXW, bool EXACT, int MINB>
__global__ void __launch_bounds__(cta_warps_max(MAXW) * 32, MINB) eri_kernel(const EriArgs a) {
    extern __shared__ __align__(128) unsigned char smem[];
    const SmemLayout lay(a.L, a.ncb_p, a.ncb_q, a.nrb_cd, a.nst, a.digest);
    double* Ra = reinterpret_cast<double*>(smem + lay.ra);
    double* GA = reinterpret_cast<double*>(smem + lay.ga);
    double* sS = reinterpret_cast<double*>(smem + lay.ss);
    int* ap = reinterpret_cast<int*>(smem + lay.ap);   // byte offset of p~ in Ra, per H_ab column
    int* aq = reinterpret_cast<int*>(smem + lay.aq);   // byte offset of q~ in Ra, per H_cd column
    unsigned* sg = reinterpret_cast<unsigned*>(smem + lay.sg);  // per q~ block: bit c set if |q~| odd
    uint32_t* srt = reinterpret_cast<uint32_t*>(smem + lay.rt);
    uint16_t* sad = reinterpret_cast<uint16_t*>(smem + lay.ad);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + lay.bars);
    uint64_t* empty = full + MAX_STAGES;
    double* sDcd = reinterpret_cast<double*>(smem + lay.dg);          // [nrb_cd * 8]
    double* sDbd = sDcd + a.nrb_cd * 8;                               // [nsb * nsd]
    uint16_t* cmap = reinterpret_cast<uint16_t*>(sDbd + SmemLayout::DG_TILE);   // column of cd -> mc << 8 | md

    const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5;
    const int L = a.L;
    const int stage_doubles = a.nrb_cd * 64;

    // R array zeroed once: the scatter always writes the same addresses, everything else (only ever
    // read through padding columns, times a zero of H) stays 0
    for (int i = tid; i < r_alloc(L); i += nthr) Ra[i] = 0.0;
    r_tables_to_smem(srt, sad, a.rtab, a.tuv, L, tid, nthr);
    for (int c = tid; c < (a.ncb_p + 1) * 8; c += nthr) {
        const uint32_t q = c < a.ncb_p * 8 ? __ldg(a.colp + c) : 0u;
        ap[c] = r_addr(q & 255, (q >> 8) & 255, (q >> 16) & 255) * 8;
    }
    for (int c = tid; c < a.ncb_q * 8; c += nthr) {
        const uint32_t q = __ldg(a.colq + c);
        aq[c] = r_addr(q & 255, (q >> 8) & 255, (q >> 16) & 255) * 8;
    }
    for (int b = tid; b < a.ncb_q; b += nthr) {
        unsigned m = 0;
        for (int c = 0; c < 8; ++c) {
            const uint32_t q = __ldg(a.colq + b * 8 + c);
            if (!(q & COL_PAD)) m |= (((q & 255) + ((q >> 8) & 255) + ((q >> 16) & 255)) & 1u) << c;
        }
        sg[b] = m;
    }
    if (a.digest) {
        for (int c = tid; c < a.nrb_cd * 8; c += nthr) cmap[c] = (uint16_t)(c < a.ncd ? ((c / a.nsd) << 8) | (c % a.nsd) : 0);
    }
    if (tid == 0) {
        for (int s = 0; s < a.nst; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, (uint32_t)a.wpc); }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();

    const int nchunk = (a.ncb_q + NQT - 1) / NQT;
    constexpr int PF = pf_depth(MAXW, NT_CD);
    ConsumerCtx cc;
    cc.astride = (size_t)a.nrb_ab * 64;
    cc.ra32 = smem_u32(Ra);
    cc.k4 = lane & 3;
    cc.lane = lane;
    cc.ap32 = smem_u32(ap) + (uint32_t)cc.k4 * 8u;
    cc.aq32 = smem_u32(aq) + (uint32_t)(lane >> 2) * 4u;
    cc.sg32 = smem_u32(sg);
    cc.ring32 = smem_u32(smem + lay.un) + (uint32_t)lane * 16u;
    cc.full32 = smem_u32(full);
    cc.empty32 = smem_u32(empty);
    cc.stage_bytes = (uint32_t)lay.stage_bytes;
    cc.nst = (uint32_t)a.nst;
    cc.ncb_p = a.ncb_p;
    cc.nrb_cd = a.nrb_cd;
    cc.tacc = a.tacc + (((size_t)blockIdx.x * a.wpc + (warp < a.wpc ? warp : 0)) * a.ncb_q * 32 + lane) * 2;
    const uint32_t ringbase32 = smem_u32(smem + lay.un);
    RingPos rp{0u, 0u};  // same sequence in every warp
    const bool producer = (warp == a.wpc);
    constexpr int NBW = builder_warps(MAXW);
    const bool helper = NBW > 1 && warp > a.wpc;   // further R-builder warps (a.nbw - 1 of them), one per sub-partition

    // builds R of primitive quartet (it, q, p) into GA; poll() is called between batches
    auto build_r = [&](long long it, int q, int p, auto poll) {
        int ib, jk;
        quartet_pairs(a, it, ib, jk);
        const double* sp = a.sb + ((size_t)ib * a.Kb + p) * 8;
        const double* sq = a.sk + ((size_t)jk * a.Kk + q) * 8;
        hermite_r_warp<NBW * 32>(GA, sS, srt, a.boys, a.ks, L, __ldg(sp), __ldg(sp + 1), __ldg(sp + 2), __ldg(sp + 3), __ldg(sq),
                       __ldg(sq + 1), __ldg(sq + 2), __ldg(sq + 3), exp(__ldg(sp + 4) + __ldg(sq + 4)), (warp - a.wpc) * 32 + lane, poll);
    };

    // primitive quartets of this CTA in order: (quartet, item of the quartet, kq, kp), kp fastest.  A CTA takes
    // whole quartets, so that every CTA gets the same mix of item sizes
    // (equal items: neighbouring CTAs share a quartet, which halves the number of H_cd matrices in flight in L2)
    long long quartet = a.qmajor ? (long long)blockIdx.x : (long long)(blockIdx.x / a.ncta_per_q);
    int ms = a.qmajor ? 0 : (int)(blockIdx.x % a.ncta_per_q);
    int kq = 0, kp = 0;
    bool have = quartet < a.nquartets;
    if (have && (producer || helper)) build_r(quartet, 0, 0, [] {});

    double2 acc[NT_CD];
    while (have) {
        long long nquartet = quartet;
        int nms = ms, nkq = kq, nkp = kp + 1;
        if (nkp == a.Kb) {
            nkp = 0;
            if (++nkq == a.Kk) {
                nkq = 0;
                if (a.qmajor) {
                    if (++nms == a.ncta_per_q) { nms = 0; nquartet += gridDim.x; }
                } else {
                    const long long g = quartet * a.ncta_per_q + ms + gridDim.x;
                    nquartet = g / a.ncta_per_q;
                    nms = (int)(g % a.ncta_per_q);
                }
            }
        }
        const bool nhave = nquartet < a.nquartets;
        const bool item_ends = (nquartet != quartet) || (nms != ms);

        int ib, jk;
        quartet_pairs(a, quartet, ib, jk);
        const int mbk = (ms == 0 ? a.row0[0] : (ms == 1 ? a.row0[1] : a.row0[2])) + warp;   // 8-row block of ab owned by this warp
        const bool active = !producer && warp < (ms == 0 ? a.nrows[0] : (ms == 1 ? a.nrows[1] : a.nrows[2]));
        if (kq == 0 && kp == 0) {
#pragma unroll
            for (int i = 0; i < NT_CD; ++i) acc[i] = make_double2(0.0, 0.0);
        }
        __syncthreads();  // consumers are done with R of the previous primitive quartet, the builder with GA
        r_scatter(Ra, GA, sad, L, tid, nthr);
        if (a.digest && kq == 0 && kp == 0) {
            // a new item: the density blocks of this quartet are staged, D_cd (for J) and D_bd (for K)
            const int ao_b = __ldg(a.aob + 2 * ib + 1), ao_c = __ldg(a.aok + 2 * jk), ao_d = __ldg(a.aok + 2 * jk + 1);
            for (int c = tid; c < a.nrb_cd * 8; c += nthr)
                sDcd[c] = c < a.ncd ? __ldg(a.D + (size_t)(ao_c + c / a.nsd) * a.nbf + ao_d + c % a.nsd) : 0.0;
            for (int e = tid; e < a.nsb * a.nsd; e += nthr)
                sDbd[e] = __ldg(a.D + (size_t)(ao_b + e / a.nsd) * a.nbf + ao_d + e % a.nsd);
        }
        __syncthreads();

        const bool last_kp = (kp == a.Kb - 1);   // the ket transform (and the ring) run with the last bra primitive only
        if (producer) {
            // ---- stream H_cd of this ket primitive through the ring, one column block per stage, and build
            // R of the next primitive quartet in between
            const double* Hq = a.Hk + ((size_t)jk * a.Kk + kq) * a.hsk;
            int jq = last_kp ? 0 : a.ncb_q;
            auto issue = [&] {
                mbar_expect_tx32(cc.full32 + rp.s * 8u, cc.stage_bytes);
                bulk_g2s32(ringbase32 + rp.s * cc.stage_bytes, Hq + (size_t)jq * stage_doubles, cc.stage_bytes,
                           cc.full32 + rp.s * 8u);
                rp.advance(cc.nst);
                ++jq;
            };
            auto poll = [&] {
                if (lane == 0)
                    while (jq < a.ncb_q && mbar_test32(cc.empty32 + rp.s * 8u, rp.ph ^ 1u)) issue();
            };
            poll();
            if (nhave) build_r(nquartet, nkq, nkp, poll);
            if (lane == 0)
                while (jq < a.ncb_q) {
                    mbar_wait32(cc.empty32 + rp.s * 8u, rp.ph ^ 1u);
                    issue();
                }
            rp.s = __shfl_sync(0xffffffffu, rp.s, 0);
            rp.ph = __shfl_sync(0xffffffffu, rp.ph, 0);
        } else if (NBW > 1 && helper) {
            if (nhave) build_r(nquartet, nkq, nkp, [] {});
        } else if (!active) {
            // a warp without rows still takes part in the ring protocol
            for (int jq = last_kp ? 0 : a.ncb_q; jq < a.ncb_q; ++jq) {
                mbar_wait32(cc.full32 + rp.s * 8u, rp.ph);
                __syncwarp();
                if (lane == 0) mbar_arrive32(cc.empty32 + rp.s * 8u);
                rp.advance(cc.nst);
            }
        } else {
            const double* Hp = a.Hb + ((size_t)ib * a.Kb + kp) * a.hsb;
            cc.Ablk = Hp + (size_t)mbk * 64 + lane * 2;
            for (int ch = 0; ch < nchunk; ++ch) {
                const int j0 = ch * a.ncb_q / nchunk;
                const int nq = (ch + 1) * a.ncb_q / nchunk - j0;
                if (nq == NQT) consume_chunk<NQT, NT_CD, EXACT, false, PF>(acc, cc, j0, nq, rp, kp > 0, last_kp);
                else if (nq == NQT - 1) consume_chunk<NQT - 1, NT_CD, EXACT, false, PF>(acc, cc, j0, nq, rp, kp > 0, last_kp);
                else consume_chunk<NQT - 2, NT_CD, EXACT, true, PF>(acc, cc, j0, nq, rp, kp > 0, last_kp);
            }
            // ---- epilogue after the last primitive quartet of the item: common factor K_ab K_cd of the pair
            // maxima, applied in two halves so that results near the bottom of the FP64 range are still
            // correctly rounded
            if (item_ends && a.digest) {
                // ---- direct digestion: the row's (ab|cd) values meet D_cd (Coulomb-type J, one number per
                // row after a reduction over the four lanes of the row) and D_bd (exchange-type K, summed per (ma, mc) by a
                // small DMMA and a segmented reduction over the rows); nothing is stored per quartet
                const double f = exp(0.5 * (__ldg(a.pmb + ib) + __ldg(a.pmk + jk)));
                const int nrow = lane >> 2;
                const int row = mbk * 8 + nrow;
                const bool rowok = row < a.nab;
                const int ma = row / a.nsb, mb = rowok ? row % a.nsb : 0;   // rows of the padding have ma >= 2 l_a + 1 and zero values
                const int nsc = a.ncd / a.nsd;
                double js = 0.0;
                double2 S0 = make_double2(0.0, 0.0), S1 = make_double2(0.0, 0.0);   // S[row][mc]: mc = 2 k4 (+1), 8 + 2 k4 (+1)
#pragma unroll
                for (int nb = 0; nb < NT_CD; ++nb) {
                    if (!EXACT && nb >= a.nrb_cd) break;
                    const int col = nb * 8 + 2 * cc.k4;
                    const double vx = rowok ? (acc[nb].x * f) * f : 0.0, vy = rowok ? (acc[nb].y * f) * f : 0.0;
                    js = fma(vx, sDcd[col], fma(vy, sDcd[col + 1], js));
                    if (a.K) {
                        // K: weight every value with D[b, d], then sum the md index on the tensor pipe: S += W . B with
                        // B[column][mc] = 1 where the column belongs to mc.  W is in C-fragment layout, which is the
                        // A-fragment layout of the two k-steps (as in GEMM2); lane (k4, nrow) makes B[k = k4][n = nrow]
                        // from the column -> (mc, md) map of its own two columns.
                        const int wx = cmap[col], wy = cmap[col + 1];
                        const double ax = vx * sDbd[mb * a.nsd + (wx & 255)], ay = vy * sDbd[mb * a.nsd + (wy & 255)];
                        const int mcx = wx >> 8, mcy = wy >> 8;
                        dmma884(S0.x, S0.y, ax, mcx == nrow ? 1.0 : 0.0);
                        dmma884(S0.x, S0.y, ay, mcy == nrow ? 1.0 : 0.0);
                        if (nsc > 8) {
                            dmma884(S1.x, S1.y, ax, mcx == nrow + 8 ? 1.0 : 0.0);
                            dmma884(S1.x, S1.y, ay, mcy == nrow + 8 ? 1.0 : 0.0);
                        }
                    }
                }
                js += __shfl_xor_sync(0xffffffffu, js, 1);
                js += __shfl_xor_sync(0xffffffffu, js, 2);
                const int ao_a = __ldg(a.aob + 2 * ib);
                if (a.J && rowok && cc.k4 == 0)
                    atomicAdd(a.J + (size_t)(ao_a + ma) * a.nbf + __ldg(a.aob + 2 * ib + 1) + mb, js);
                if (a.K) {
                    // sum over the rows that share ma (rows are sorted by ma: segmented suffix sums by doubling), then the
                    // first row of every segment adds its four (ma, mc) sums to the AO matrix
                    double v[4] = {S0.x, S0.y, S1.x, S1.y};
#pragma unroll
                    for (int d = 1; d < 8; d *= 2) {
                        const int ma_o = __shfl_down_sync(0xffffffffu, ma, 4 * d);
                        const bool take = nrow + d < 8 && ma_o == ma;
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            const double o = __shfl_down_sync(0xffffffffu, v[i], 4 * d);
                            if (take) v[i] += o;
                        }
                    }
                    const int ma_p = __shfl_up_sync(0xffffffffu, ma, 4);
                    const bool head = nrow == 0 || ma_p != ma;
                    if (head && rowok) {
                        double* Kr = a.K + (size_t)(ao_a + ma) * a.nbf + __ldg(a.aok + 2 * jk);
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            const int mc = (i >> 1) * 8 + 2 * cc.k4 + (i & 1);
                            if (mc < nsc && v[i] != 0.0) atomicAdd(Kr + mc, v[i]);
                        }
                    }
                }
            } else if (item_ends) {
                const double f = exp(0.5 * (__ldg(a.pmb + ib) + __ldg(a.pmk + jk)));
                const int row = mbk * 8 + (lane >> 2);
                // (a9) 16-byte streaming stores (st.global.cs.v2.f64: the 3.7 GB output stream must not evict H from L2).
                // A lane holds columns (c, c+1), c = 8 nb + 2 k4, of its row; rows start at element (quartet Nab + row) Ncd of
                // the output, which is odd for every other row when Ncd is odd: there the aligned pairs are (c+1, c+2), whose
                // second element comes from the neighbouring lane (one shuffle per block).  One store instruction per block
                // serves both kinds of rows (address and values selected per lane).
                const size_t e0 = ((size_t)ib * a.nket + jk) * a.nab * a.ncd + (size_t)(row < a.nab ? row : 0) * a.ncd;
                double* o = a.out + e0;
                const int odd = (int)((reinterpret_cast<uintptr_t>(o) >> 3) & 1);   // d_out itself need only be 8-byte aligned
                const bool rowok = row < a.nab;
                const double f2x = (acc[0].x * f) * f;
                if (rowok && odd && cc.k4 == 0) __stcs(o, f2x);   // first element of a row that starts on an odd element
#pragma unroll
                for (int nb = 0; nb < NT_CD; ++nb) {
                    const double vx = (acc[nb].x * f) * f, vy = (acc[nb].y * f) * f;
                    // the x value of column c+2: from lane k4+1 (same block) or, for k4 = 3, from the row's lane 0, next block
                    double sv = vx;
                    if (nb + 1 < NT_CD && cc.k4 == 0) sv = (acc[nb + 1].x * f) * f;
                    const double nx = __shfl_sync(0xffffffffu, sv, (lane & ~3) | ((cc.k4 + 1) & 3));
                    const int c = nb * 8 + 2 * cc.k4 + odd;   // first column of this lane's aligned pair
                    const double p0 = odd ? vy : vx, p1 = odd ? nx : vy;
                    if (rowok) {
                        if (c + 1 < a.ncd) __stcs(reinterpret_cast<double2*>(o + c), make_double2(p0, p1));
                        else if (c < a.ncd) __stcs(o + c, p0);
                    }
                }
            }
        }
        quartet = nquartet; ms = nms; kq = nkq; kp = nkp; have = nhave;
    }
}

// Splits the nrb_ab eight-row blocks of a quartet into work items of at most 11 blocks (one consumer warp
// each).  The FP64 tensor pipe is per SM sub-partition (profiles/r1_fp64_peak.txt) and warp w runs on
// sub-partition w % 4, so an item of n blocks takes ceil(n/4) block-times: the split minimises their sum
// (18 blocks: 10 + 8 -> 3 + 2, not 9 + 9 -> 3 + 3), then the number of consumer warps.
void plan_items(EriArgs& a) {
    const int n = a.nrb_ab;
    for (int t = 0; t < 3; ++t) { a.row0[t] = 0; a.nrows[t] = 0; }
    if (n <= 11) { a.ncta_per_q = 1; a.nrows[0] = n; a.wpc = n; return; }
    // two items if they can hold the rows (n <= 22), else three (l = 7 bras: up to 29 row blocks)
    const int k = n <= 22 ? 2 : 3;
    int best = 1 << 30, b1 = 0, b2 = 0;
    for (int n1 = 1; n1 <= 11; ++n1)
        for (int n2 = (k == 2 ? n - n1 : 1); n2 <= (k == 2 ? n - n1 : 11); ++n2) {
            const int n3 = n - n1 - n2;
            if (n2 < 1 || n2 > n1 || n3 < 0 || n3 > n2 || n3 > 11 || (k == 3 && n3 < 1)) continue;
            const int cost = ((n1 + 3) / 4 + (n2 + 3) / 4 + (n3 + 3) / 4) * 16 + n1;
            if (cost < best) { best = cost; b1 = n1; b2 = n2; }
        }
    a.ncta_per_q = k;
    a.nrows[0] = b1; a.row0[1] = b1; a.nrows[1] = b2;
    if (k == 3) { a.row0[2] = b1 + b2; a.nrows[2] = n - b1 - b2; }
    a.wpc = b1;
}

// MINB CTAs per SM: small classes (few row blocks, small R) are latency-bound per work item -- two barriers, TMA
// and L2 round trips around a few dozen DMMAs -- so two or three CTAs share an SM there.
template <int NT_CD, int NQT, int MAXW, bool EXACT, int MINB>
md4_status launch_one(md4_ctx* ctx, EriArgs& a, cudaStream_t st) {
    // shared memory per CTA: the SM's 228 kB less 1 kB reserved per resident CTA
    const size_t budget = MINB == 1 ? (size_t)ctx->smem_optin : (size_t)(ctx->smem_optin + 1024) / MINB - 1024;
    // ring depth: whatever shared memory is left after R, at least 2 stages, at most MAX_STAGES
    int nst = 2;
    for (int s = MAX_STAGES; s >= 2; --s)
        if (SmemLayout(a.L, a.ncb_p, a.ncb_q, a.nrb_cd, s, a.digest).total <= budget) { nst = s; break; }
    if (nst > a.ncb_q) nst = a.ncb_q < 2 ? 2 : a.ncb_q;
    a.nst = nst;
    const SmemLayout lay(a.L, a.ncb_p, a.ncb_q, a.nrb_cd, nst, a.digest);
    if (lay.total > budget) {
        if (MINB > 1) return launch_one<NT_CD, NQT, MAXW, EXACT, 1>(ctx, a, st);
        ctx->err = "md4_compute: shared memory needed exceeds the device limit";
        return MD4_EUNSUPPORTED;
    }
    auto kern = eri_kernel<NT_CD, NQT, MAXW, EXACT, MINB>;
    cudaError_t e = cudaSuccess;
    // the shared-memory opt-in is a per-function attribute: set it once per context to the device maximum (never to a
    // class-dependent value, which two contexts on one device could interleave), then launch with what the class needs
    if (ctx->configured.insert(reinterpret_cast<const void*>(kern)).second) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, ctx->smem_optin);
        if (e != cudaSuccess) { ctx->configured.erase(reinterpret_cast<const void*>(kern)); ctx->err = std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e); return MD4_ECUDA; }
    }
    const long long nwork = a.qmajor ? a.nquartets : a.nquartets * a.ncta_per_q;
    const long long slots = (long long)ctx->num_sms * MINB;
    long long grid = nwork < slots ? nwork : slots;
    kern<<<(unsigned)grid, (a.wpc + builder_warps(MAXW)) * 32, lay.total, st>>>(a);
    ctx->launches++;
    e = cudaGetLastError();
    if (e != cudaSuccess) { ctx->err = std::string("eri_kernel launch: ") + cudaGetErrorString(e); return MD4_ECUDA; }
    return MD4_OK;
}

template <int NT_CD, bool EXACT>
md4_status launch_w(md4_ctx* ctx, EriArgs& a, cudaStream_t st) {
    if constexpr (NT_CD == 11 || NT_CD == 13 || NT_CD == 15 || NT_CD == 16) {
        if (a.wpc > 11) return launch_one<NT_CD, 8, 16, EXACT, 1>(ctx, a, st);
    }
    if (a.wpc <= 7) return launch_one<NT_CD, 8, 9, EXACT, 1>(ctx, a, st);
    if (a.wpc == 8) return launch_one<NT_CD, 8, 10, EXACT, 1>(ctx, a, st);
    if constexpr (NT_CD == 11 || NT_CD == 13 || NT_CD == 15 || NT_CD == 16) {
        if (a.wpc == 10) return launch_one<NT_CD, 8, 11, EXACT, 1>(ctx, a, st);
    }
    return launch_one<NT_CD, 8, 12, EXACT, 1>(ctx, a, st);
}

// small classes: at most 7 row blocks of ab (8 warps) and of cd
template <int NT_CD>
md4_status launch_small(md4_ctx* ctx, EriArgs& a, cudaStream_t st) {
    if (a.wpc + 1 <= 4) return launch_one<NT_CD, 8, 4, false, 3>(ctx, a, st);
    if (a.wpc + 1 <= 8) return launch_one<NT_CD, 8, 8, false, 2>(ctx, a, st);
    return launch_w<NT_CD, false>(ctx, a, st);
}

}  // namespace

void plan_items_host(int nrb_ab, int* nitems, int* row0, int* nrows) {
    EriArgs a;
    a.nrb_ab = nrb_ab;
    plan_items(a);
    *nitems = a.ncta_per_q;
    for (int t = 0; t < 3; ++t) { row0[t] = a.row0[t]; nrows[t] = a.nrows[t]; }
}

// tacc: the [ab|q~] scratch of contracted bras; tacc_cap: its size in bytes, checked against what the launch can touch
// (0: the context's own scratch, sized for every class at md4_create)
static md4_status launch_eri_with(md4_ctx* ctx, const PairListDev& bra, const PairListDev& ket, double* d_out,
                                  cudaStream_t st, const DigestArgs* dg, double* tacc, size_t tacc_cap) {
    // uncontracted low-l classes: one warp per quartet, no block-level synchronisation (md4_eri_small.cu)
    if (!dg && small_class_eligible(bra, ket)) return launch_eri_small(ctx, bra, ket, d_out, st);
    EriArgs a;
    a.digest = dg ? 1 : 0;
    a.nbf = dg ? dg->nbf : 0;
    a.nsb = n_solid(bra.lj); a.nsd = n_solid(ket.lj);
    a.aob = bra.ao; a.aok = ket.ao;
    a.D = dg ? dg->D : nullptr; a.J = dg ? dg->J : nullptr; a.K = dg ? dg->K : nullptr;
    a.Hb = bra.Hb; a.sb = bra.scal; a.pmb = bra.pairmax; a.hsb = bra.hstrideb;
    a.Hk = ket.Hk; a.sk = ket.scal; a.pmk = ket.pairmax; a.hsk = ket.hstridek;
    a.Kb = bra.Ki * bra.Kj; a.Kk = ket.Ki * ket.Kj; a.nbra = bra.npair; a.nket = ket.npair;
    a.nab = bra.nab; a.ncd = ket.nab; a.nrb_ab = bra.nrb; a.nrb_cd = ket.nrb;
    a.ncb_p = bra.ncbb; a.ncb_q = ket.ncbk;
    a.L = bra.lsum + ket.lsum;
    if (a.L > LTOT || ket.lsum > LKET_MAX || ket.nrb > 22) {
        ctx->err = "md4_compute: class beyond MD4_LSUM_MAX (needs l_a+l_b+l_c+l_d <= 24, l_c+l_d <= 12, (2l_c+1)(2l_d+1) <= 176)";
        return MD4_EUNSUPPORTED;
    }
    plan_items(a);
    // Kets of at most 16 column blocks (gg, hg, hh, ig) need 44-64 accumulator registers: the kernel then runs at 128
    // registers (with 0.2-3 kB of spills) and a CTA can hold 16 warps.  Bras of 12-15 row blocks (hg: 13, ig: 15) become ONE
    // item with a consumer warp per row block (instantiation MAXW = 16): the same number of block-times (13: 2 + 2 -> 4,
    // 15: 2 + 2 -> 4) but 3-4 warps per sub-partition instead of 2 to hide the gather latency, and R is built once per
    // quartet instead of once per item.  (hg|hg) 53.7 -> 60.1 %, (ig|hg) 62.8 -> 72.4 %, (ig|ig) 65.4 -> 71.3 % of peak.
    // 20 warps at 96 registers for hh bras (16 row blocks) were measured too: 52-56 % against 64-67 %.
    if ((a.nrb_cd == 11 || a.nrb_cd == 13 || a.nrb_cd == 15 || a.nrb_cd == 16) && a.nrb_ab >= 12 && a.nrb_ab <= 15) {
        a.ncta_per_q = 1; a.wpc = a.nrb_ab;
        a.row0[0] = 0; a.nrows[0] = a.nrb_ab; a.row0[1] = a.row0[2] = 0; a.nrows[1] = a.nrows[2] = 0;
    }
    a.nquartets = (long long)a.nbra * a.nket;
    a.qmajor = (a.ncta_per_q >= 2 && a.nrows[0] != a.nrows[a.ncta_per_q - 1]) ? 1 : 0;
    // strip height: the H matrices of a strip's bra pairs (K_bra matrices each) should stay L2-resident next to the kets
    // in flight: <= 16 MB per strip.  Measured on cfg3 / cfg5 (ii|ii) K=3: flat order 58.0 / 923 ms, 32-pair strips
    // 57.8 / 962 ms (a contracted strip of 32 is 185 MB), this rule 57.8 / 923 ms.
    {
        const double bytes_per_bra = (double)a.Kb * (double)a.hsb * sizeof(double);
        int tb = (int)(16.0 * 1024 * 1024 / bytes_per_bra);
        a.tb = tb < 1 ? 1 : (tb > 32 ? 32 : tb);
    }
    a.nst = 2;
    a.rtab = ctx->tab.rtab; a.tuv = ctx->tab.tuv; a.boys = ctx->tab.boys;
    a.ks = ctx->kernel;
    a.colp = ctx->tab.colb[bra.lsum]; a.colq = ctx->tab.colk[ket.lsum];
    a.out = d_out;
    a.tacc = tacc;
    const int nt = a.nrb_cd;
    if (tacc_cap && a.Kb > 1) {
        // one slab of wpc x ncb_q fragment blocks (512 bytes each) per CTA; resident CTAs per SM as in launch_small
        const int minb = nt <= 7 ? (a.wpc + 1 <= 4 ? 3 : (a.wpc + 1 <= 8 ? 2 : 1)) : 1;
        const size_t need = (size_t)ctx->num_sms * minb * a.wpc * a.ncb_q * 64 * sizeof(double);
        if (need > tacc_cap) {
            ctx->err = "md4_compute_static: this contracted bra class needs " + std::to_string(need) +
                       " bytes of [ab|q~] scratch, the static scratch holds " + std::to_string(tacc_cap) +
                       " (MD4_STATIC_SCRATCH_BYTES); use md4_compute";
            return MD4_EUNSUPPORTED;
        }
    }
    // exact instantiations for the ket classes of l >= 4 shells (N_cd = 81, 99, 117, 121, 143, 169); the
    // others (no product of two odd numbers <= 13 falls in 14, 17, 19-21 row blocks) run predicated
    if (nt == 11) return launch_w<11, true>(ctx, a, st);
    if (nt == 13) return launch_w<13, true>(ctx, a, st);
    if (nt == 15) return launch_w<15, true>(ctx, a, st);
    if (nt == 16) return launch_w<16, true>(ctx, a, st);
    if (nt == 18) return launch_w<18, true>(ctx, a, st);
    if (nt == 22) return launch_w<22, true>(ctx, a, st);
    if (nt <= 2) return launch_small<2>(ctx, a, st);
    if (nt <= 4) return launch_small<4>(ctx, a, st);
    if (nt <= 7) return launch_small<7>(ctx, a, st);
    if (nt <= 12) return launch_w<12, false>(ctx, a, st);
    if (nt <= 22) return launch_w<22, false>(ctx, a, st);   // kets with an l = 7 shell: 15 x 9 = 135 (17 blocks), 15 x 11 = 165 (21)
    ctx->err = "md4_compute: ket class too large";
    return MD4_EUNSUPPORTED;
}

md4_status launch_eri(md4_ctx* ctx, const PairListDev& bra, const PairListDev& ket, double* d_out,
                      cudaStream_t st, const DigestArgs* dg) {
    return launch_eri_with(ctx, bra, ket, d_out, st, dg, ctx->d_tacc, 0);
}

// ---- md4_compute_static: the fused kernel with its [ab|q~] scratch in a file-scope device array ---------------------
// For callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  The array is
// part of the library image: every GPU that loads libmd4.so holds MD4_STATIC_SCRATCH_BYTES until the process exits.  All
// calls on a device share it, whatever the context; it keeps the last call's contents.  Nothing in it has to start at
// zero: a CTA stores the partial [ab|q~] of a bra primitive before it loads it for the next one (consume_chunk), so there
// is nothing to clear -- but two launches with contracted bras that overlap on the GPU race on it.
namespace {
static __device__ __align__(256) double md4_static_tacc[MD4_STATIC_SCRATCH_BYTES / sizeof(double)];
constexpr int STATIC_MAX_DEVICES = 64;
double* g_static_tacc[STATIC_MAX_DEVICES] = {};   // device address of the array, per device ordinal (looked up once)
std::mutex g_static_mu;
}  // namespace

md4_status launch_eri_static(md4_ctx* ctx, const PairListDev& bra, const PairListDev& ket, double* d_out, cudaStream_t st) {
    // In host code `md4_static_tacc` is a host-side stand-in, not a device address: ask the runtime for the address on
    // the current device (the caller has made ctx->device current) and pass that to the kernel.
    if (ctx->device < 0 || ctx->device >= STATIC_MAX_DEVICES) {
        ctx->err = "md4_compute_static: device ordinal beyond 63";
        return MD4_EUNSUPPORTED;
    }
    double* tacc = nullptr;
    {
        std::lock_guard<std::mutex> lk(g_static_mu);
        if (!g_static_tacc[ctx->device]) {
            void* p = nullptr;
            const cudaError_t e = cudaGetSymbolAddress(&p, md4_static_tacc);
            if (e != cudaSuccess) {
                ctx->err = std::string("md4_compute_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e);
                return MD4_ECUDA;
            }
            g_static_tacc[ctx->device] = static_cast<double*>(p);
        }
        tacc = g_static_tacc[ctx->device];
    }
    return launch_eri_with(ctx, bra, ket, d_out, st, nullptr, tacc, (size_t)MD4_STATIC_SCRATCH_BYTES);
}

// ---- stage-level debug kernels ---------------------------------------------------------------------
namespace {
__global__ void debug_boys_kernel(const double* tab, int mmax, int n, const double* T, double* out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n * (mmax + 1)) return;
    out[i] = boys_one(tab, i % (mmax + 1), T[i / (mmax + 1)]);
}

// out: dense [(L+1)^3] array, out[(t*(L+1)+u)*(L+1)+v] = R_{tuv} for t+u+v <= L, 0 elsewhere; one warp
__global__ void debug_r_kernel(const uint32_t* rtab, const uint32_t* tuv, const double* boys, KernelSpec ks, int L,
                               const double* pq, double* out) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int S = L + 1;
    double* Ra = reinterpret_cast<double*>(smem);
    double* GA = Ra + r_alloc(L);
    double* sS = GA + 2 * n_hermite(L);
    uint32_t* srt = reinterpret_cast<uint32_t*>(sS + 32);
    uint16_t* sad = reinterpret_cast<uint16_t*>(srt + n_hermite(L));
    for (int i = threadIdx.x; i < r_alloc(L); i += blockDim.x) Ra[i] = 0.0;
    r_tables_to_smem(srt, sad, rtab, tuv, L, threadIdx.x, blockDim.x);
    __syncthreads();
    hermite_r_warp(GA, sS, srt, boys, ks, L, pq[0], pq[1], pq[2], pq[3], pq[4], pq[5], pq[6], pq[7], 1.0, threadIdx.x, [] {});
    __syncthreads();
    r_scatter(Ra, GA, sad, L, threadIdx.x, blockDim.x);
    __syncthreads();
    for (int i = threadIdx.x; i < S * S * S; i += blockDim.x) {
        const int t = i / (S * S), u = (i / S) % S, v = i % S;
        out[i] = (t + u + v <= L) ? Ra[r_addr(t, u, v)] : 0.0;
    }
}
}  // namespace

cudaError_t launch_debug_boys(md4_ctx* ctx, int mmax, int n, const double* d_T, double* d_out) {
    const int tot = n * (mmax + 1);
    debug_boys_kernel<<<(tot + 127) / 128, 128>>>(ctx->tab.boys, mmax, n, d_T, d_out);
    ctx->launches++;
    return cudaGetLastError();
}

cudaError_t launch_debug_r(md4_ctx* ctx, int L, const double* d_pq, double* d_out) {
    const size_t sm = ((size_t)r_alloc(L) + 2 * (size_t)n_hermite(L) + 32) * 8 + (size_t)n_hermite(L) * 6 + 16;
    cudaError_t e = cudaFuncSetAttribute(debug_r_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, ctx->smem_optin);
    if (e != cudaSuccess) return e;
    debug_r_kernel<<<1, 32, sm>>>(ctx->tab.rtab, ctx->tab.tuv, ctx->tab.boys, ctx->kernel, L, d_pq, d_out);
    ctx->launches++;
    return cudaGetLastError();
}

}  // namespace md4

// md4_device.cuh -- device functions shared by the compute kernel and the stage-level debug kernels:
// Boys function (Eq.11), seeds [0]^(m) (Eq.10, Eq.12) and the Hermite Coulomb tensor
// recurrence Eq.13 level by level in shared memory (after Listing 3.1).
#pragma once
#include "md4_internal.h"

namespace md4 {

// F_m(T): table of F_{m..m+7}(T_j) at the nearest node T_j = j/16 and a 7th-order Taylor step
// F_m(T) = sum_k F_{m+k}(T_j) (T_j - T)^k / k!  (remainder <= (1/32)^8/8! = 2.3e-17 relative);
// T >= 100: F_m = (2m-1)!!/(2T)^m sqrt(pi/T)/2 (relative error < 1e-19 for m <= 24; S:8(c) Q11).
__device__ __forceinline__ double boys_one(const double* __restrict__ tab, int m, double T) {
    if (T < (double)BOYS_TMAX) {
        const int j = (int)(T * BOYS_INV_DELTA + 0.5);
        const double d = (double)j * (1.0 / BOYS_INV_DELTA) - T;
        const double* f = tab + (size_t)j * BOYS_STRIDE + m;
        double r = __ldg(f + 7) * (1.0 / 5040.0);
        r = fma(r, d, __ldg(f + 6) * (1.0 / 720.0));
        r = fma(r, d, __ldg(f + 5) * (1.0 / 120.0));
        r = fma(r, d, __ldg(f + 4) * (1.0 / 24.0));
        r = fma(r, d, __ldg(f + 3) * (1.0 / 6.0));
        r = fma(r, d, __ldg(f + 2) * 0.5);
        r = fma(r, d, __ldg(f + 1));
        r = fma(r, d, __ldg(f));
        return r;
    }
    const double inv = 0.5 / T;
    double r = 0.5 * sqrt(3.14159265358979323846 / T);
    for (int k = 0; k < m; ++k) r *= (2 * k + 1) * inv;
    return r;
}

// Shared-memory copies of the Eq.13 table and of the additive address of every graded ordinal: the table is
// m-independent, so it is read from shared memory at every level instead of from global memory.
__device__ __forceinline__ void r_tables_to_smem(uint32_t* srt, uint16_t* sad, const uint32_t* __restrict__ rtab,
                                                 const uint32_t* __restrict__ tuv, int L, int tid, int nthr) {
    for (int e = tid; e < n_hermite(L); e += nthr) {
        srt[e] = __ldg(rtab + e);
        const uint32_t q = __ldg(tuv + e);
        sad[e] = (uint16_t)r_addr(q & 255, (q >> 8) & 255, (q >> 16) & 255);
    }
}

// Interaction kernel g(r12) ("[0]^(m) is related to the Boys function (or similar quantities for non-Coulomb
// integrals, ref. 21)"; S:8(f) item 3).  For g(r) = Int w(u) exp(-u^2 r^2) du only the seeds of Eq.10 change:
//   [0]^(m) = (-2 rho)^m prefactor G_m,  G_m = ka F_m(T) + kb s^(2m+1) F_m(s^2 T),  s^2 = omega^2 / (omega^2 + rho):
//   1/r: (ka, kb) = (1, 0);  erf(omega r)/r: (0, 1);  erfc(omega r)/r: (1, -1).  Everything downstream (Eq.13, the two
// contractions) is unchanged.
__device__ __forceinline__ double kernel_seed(const double* __restrict__ boys, const KernelSpec& ks, int m, double rho, double T) {
    double G = ks.ka != 0.0 ? ks.ka * boys_one(boys, m, T) : 0.0;
    if (ks.kb != 0.0) {
        const double s2 = ks.omega2 / (ks.omega2 + rho);
        double sp = sqrt(s2);
        for (int k = 0; k < m; ++k) sp *= s2;
        G = fma(ks.kb * sp, boys_one(boys, m, s2 * T), G);
    }
    return G;
}

// ---- Hermite Coulomb tensor, built by ONE warp in graded order, in place ---------------------------
// hermite_r_warp computes R^{(0)}_{tuv}, t+u+v <= L, of one primitive quartet into G[graded ordinal]
// (G: n_hermite(L) + L doubles, sS: 32 doubles; shared memory).  As in Listing 3.1 one array
// serves all levels: level l = 1..L holds [r]^(L-l), |r| <= l, at G[(L-l) + ord(r)], i.e. every level is
// shifted down by one slot, and is computed from level l-1 by Eq.13.  The slot a value is written to held
// the level l-1 value of the PREVIOUS ordinal, which only elements with an equal or higher ordinal read:
// batches of 32*B elements are therefore processed from the top down, all loads of a batch before its
// stores (__syncwarp) -- one warp needs no block barrier (the paper uses two per level).
// In the fused kernel the producer warp runs this for the NEXT primitive quartet while the consumer warps
// contract the current one, calling poll() between batches so that the H_cd ring keeps being refilled;
// r_scatter() then moves G into the additive layout (md4_internal.h) with all threads.  scale multiplies
// every value (K_ab K_cd relative to the pair maxima; 1 in the debug kernel).
__host__ __device__ inline int r_graded_alloc(int L) { return n_hermite(L) + L; }

// GS = 32 (one warp, `gtid` = lane) or a multiple of 32: then the builder warps of the fused kernel share the elements of
// every batch (thread gtid of gsize) and meet at named barrier 1 where the one-warp version has a __syncwarp; the batches
// are gsize * B elements.  The argument above holds between warps as well: a warp that runs ahead into the next (lower)
// batch only loads elements of lower ordinals than anything the batch above stores over.
template <int GS>
__device__ __forceinline__ void r_group_sync() {
    if constexpr (GS == 32) __syncwarp();
    else asm volatile("bar.sync 1, %0;\n" ::"n"(GS) : "memory");
}

template <int GS = 32, class Poll>
__device__ __forceinline__ void hermite_r_warp(double* G, double* sS, const uint32_t* srt,
                                               const double* __restrict__ boys, const KernelSpec& ks, int L, double zp, double Px,
                                               double Py, double Pz, double zq, double Qx, double Qy, double Qz,
                                               double scale, int gtid, Poll poll) {
    constexpr int gsize = GS;
    const double X0 = Px - Qx, X1 = Py - Qy, X2 = Pz - Qz;
    {
        const double zs = zp + zq;
        const double rho = zp * zq / zs;
        const double T = rho * (X0 * X0 + X1 * X1 + X2 * X2);
        // 2 pi^{5/2} = 34.98683665524972497
        const double pref = scale * 34.986836655249724970 / (zp * zq * sqrt(zs));
        if (gtid <= L) {
            const double F = kernel_seed(boys, ks, gtid, rho, T);
            double pw = pref;
            const double m2r = -2.0 * rho;
            for (int k = 0; k < gtid; ++k) pw *= m2r;
            sS[gtid] = pw * F;
        }
    }
    r_group_sync<GS>();
    if (gtid == 0) G[L] = sS[L];   // level 0: [0]^(L)
    r_group_sync<GS>();
    constexpr int B = 4;  // independent elements in flight per thread
    for (int l = 1; l <= L; ++l) {
        const int n = n_hermite(l);
        const double* src = G + (L - l + 1);
        double* dst = G + (L - l);
        const int nbatch = (n + gsize * B - 1) / (gsize * B);
        for (int bt = nbatch - 1; bt >= 0; --bt) {
            const int e0 = bt * gsize * B + gtid;
            uint32_t w[B];
#pragma unroll
            for (int k = 0; k < B; ++k) {
                const int e = e0 + k * gsize;
                w[k] = srt[e < n ? e : n - 1];
            }
            double val[B];
#pragma unroll
            for (int k = 0; k < B; ++k) {
                const int ax = (w[k] >> 29) & 3;
                const double x = ax == 0 ? X0 : (ax == 1 ? X1 : X2);
                val[k] = fma((double)((w[k] >> 24) & 31), src[w[k] & 4095], x * src[(w[k] >> 12) & 4095]);
            }
            r_group_sync<GS>();   // every load of the batch precedes its stores
#pragma unroll
            for (int k = 0; k < B; ++k) {
                const int e = e0 + k * gsize;
                if (e == 0) val[k] = sS[L - l];
                if (e < n) dst[e] = val[k];
            }
            poll();
        }
        r_group_sync<GS>();
    }
}

// G (graded order) -> Ra (additive layout); all nthr threads, caller synchronises before and after
__device__ __forceinline__ void r_scatter(double* Ra, const double* GA, const uint16_t* sad, int L, int tid, int nthr) {
    for (int e = tid; e < n_hermite(L); e += nthr) Ra[sad[e]] = GA[e];
}

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// ---- mbarrier / bulk-copy (TMA 1-D) primitives for the H_cd ring of the fused kernel -----------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
// shared-memory loads by 32-bit shared address.  Written as PTX so that the address arithmetic stays 32-bit
// (one IADD per load) and the compiler does not re-derive the shared window base at every access.
__device__ __forceinline__ double lds_f64(uint32_t addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];\n" : "=d"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ double2 lds_v2f64(uint32_t addr) {
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];\n" : "=d"(v.x), "=d"(v.y) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ int2 lds_v2s32(uint32_t addr) {
    int2 v;
    asm volatile("ld.shared.v2.s32 {%0,%1}, [%2];\n" : "=r"(v.x), "=r"(v.y) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t lds_u32(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];\n" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
// mbarrier operations by 32-bit shared address (same semantics as the pointer forms above)
__device__ __forceinline__ void mbar_arrive32(uint32_t bar) {
    asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.shared::cta.b64 st, [%0];\n}\n" ::"r"(bar) : "memory");
}
// arrive that carries a data dependency on `dep`: it is predicated on dep != 0 AND on dep == 0 (two instructions, one of
// which executes), so the assembler can neither drop `dep` nor schedule the arrive before `dep` has been computed.
// Used to keep the release of a ring stage behind the completion of every load of the stage (md4_eri.cu).
__device__ __forceinline__ void mbar_arrive32_dep(uint32_t bar, int dep) {
    asm volatile(
        "{\n .reg .b64 st;\n .reg .pred p;\n setp.ne.s32 p, %1, 0;\n"
        " @p mbarrier.arrive.shared::cta.b64 st, [%0];\n"
        " @!p mbarrier.arrive.shared::cta.b64 st, [%0];\n}\n" ::"r"(bar), "r"(dep) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx32(uint32_t bar, uint32_t bytes) {
    asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n}\n" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait32(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n .reg .pred p;\n"
        "W_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        " @p bra D_%=;\n bra W_%=;\n"
        "D_%=:\n}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ bool mbar_test32(uint32_t bar, uint32_t parity) {   // non-blocking
    uint32_t ok;
    asm volatile("{\n .reg .pred p;\n mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void bulk_g2s32(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar) : "memory");
}

}  // namespace md4

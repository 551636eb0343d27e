// md4_internal.h -- declarations shared by the translation units of libmd4 (never by the oracle).
// Citations: P:n = PAPER.md line n, S:8(x) = SURVEY.md section 8(x).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>
#include <set>
#include <map>

#include "../../include/md4.h"

namespace md4 {

constexpr int LMAX = MD4_LMAX;          // per shell
constexpr int LTOT = MD4_LSUM_MAX;      // highest Hermite order L = la+lb+lc+ld the fused kernel takes: R in the additive
                                        // layout (121 kB at L = 24) must fit shared memory next to the ring; l = 7 shells are
                                        // accepted in classes up to this L (S:8(f) item 4)
constexpr int LKET_MAX = 12;            // highest l_c + l_d: 57 q~ column blocks (TACC_QBLOCKS), <= 22 accumulator tiles per lane
constexpr int NR_MAX = (LTOT + 1) * (LTOT + 2) * (LTOT + 3) / 6;  // 2925

// Boys table: nodes T_j = j / BOYS_INV_DELTA, j = 0..BOYS_NODES-1, values F_m(T_j) for m = 0..BOYS_STRIDE-1.
constexpr int BOYS_INV_DELTA = 16;
constexpr int BOYS_TMAX = 100;          // above: asymptotic form (relative error < 1e-19 for m <= 24, S:8(c) Q11)
constexpr int BOYS_NODES = BOYS_TMAX * BOYS_INV_DELTA + 1;
constexpr int BOYS_TAYLOR = 8;          // terms k = 0..7
constexpr int BOYS_STRIDE = LTOT + BOYS_TAYLOR;  // 32

__host__ __device__ inline int n_hermite(int n) { return (n + 1) * (n + 2) * (n + 3) / 6; }
__host__ __device__ inline int n_cart(int l) { return (l + 1) * (l + 2) / 2; }
__host__ __device__ inline int n_solid(int l) { return 2 * l + 1; }

// Graded Hermite ordinal (all |r| <= n first, needed by the in-place-style level recurrence):
// degree ascending, then t descending, then u descending.
__host__ __device__ inline int herm_ord(int t, int u, int v) {
    int n = t + u + v;
    int w = n - t;
    return n * (n + 1) * (n + 2) / 6 + w * (w + 1) / 2 + (w - u);
}

// ---- additive layout of the Hermite Coulomb tensor in shared memory -------------------------------
// R_{tuv} lives at r_addr(t,u,v) = t*RS2 + u*RS1 + v, so that address(p~ + q~) = address(p~) +
// address(q~) and the 2-index integrals [p~|q~] = +-R_{p~+q~} (Eq.8) are a pure gather.  The
// strides are the same for every class (the column order of H depends on them): RS1 > 24, RS2 > 24*RS1
// keep the map injective on t+u+v <= 24, and their residues mod 16 (10 and 7) were chosen so that the
// Hermite indices of every l_pair = 8..12 split almost evenly over the sixteen 8-byte bank pairs
// (DESIGN.md "Conflict-free gather").
constexpr int RS1 = 26;
constexpr int RS2 = 631;
__host__ __device__ inline int r_addr(int t, int u, int v) { return t * RS2 + u * RS1 + v; }
__host__ __device__ inline int r_alloc(int L) { return L * RS2 + 32; }  // doubles; +32: padding columns read addresses 0..15 past the largest p~
constexpr int LPAIR = 2 * LMAX;          // highest l_a + l_b of a shell pair
constexpr int TACC_WARPS = 22;            // consumer warps per SM of the fused kernel, at most (11 per CTA; small classes: 3 CTAs x 3, 2 x 7)
constexpr int TACC_QBLOCKS = 64;         // q~ column blocks, at most (57 for l_pair = 12)
constexpr uint32_t COL_PAD = 1u << 31;   // flag of a padding column in the column tables

// Constant device tables, built once per context (md4_tables.cpp).
struct DeviceTables {
    const uint32_t* colb[LPAIR + 1];   // bra-role column order of H for l_pair: packed t | u<<8 | v<<16 | COL_PAD
    const uint32_t* colk[LPAIR + 1];   // ket-role column order
    const int* b2k[LPAIR + 1];         // bra column -> ket column of the same (t,u,v), -1 for padding
    const uint32_t* rtab;    // [NR_MAX] packed {idx0:12, idx1:12, C:5, axis:2} of Eq.13
    const uint32_t* tuv;     // [NR_MAX] packed t | u << 8 | v << 16 in graded order
    const double* boys;      // [BOYS_NODES * BOYS_STRIDE]
    const double* solid[LMAX + 1];     // [(2l+1) * n_cart(l)]  high parts
    const double* solid_lo[LMAX + 1];  // low parts of the double-double coefficients
};

struct HostTables {
    std::vector<uint32_t> rtab, tuv;
    std::vector<uint32_t> colb[LPAIR + 1], colk[LPAIR + 1];   // sizes are multiples of 8
    std::vector<int> b2k[LPAIR + 1], g2b[LPAIR + 1];          // g2b: graded ordinal -> bra column
    std::vector<double> boys;
    std::vector<double> solid[LMAX + 1], solid_lo[LMAX + 1];
};
void build_host_tables(HostTables& t);  // md4_tables.cpp

// H matrices are stored in 8x8 blocks, once per role (two copies, same numbers, different column order):
//   Hb (bra role, columns in colb order, ncbb blocks), Hk (ket role, colk order, ncbk blocks);
// element (row, col) of primitive pair ip lives at
//   H?[ip * hstride? + ((col/8) * nrb + row/8) * 64 + (row%8) * 8 + col%8],
// rows = solid-harmonic pair index ma*(2lj+1)+mb padded to nrb*8, cols padded to whole blocks, padding = 0.
// One block is exactly the A fragment pair (bra role: GEMM1) or the B fragment pair (ket role: GEMM2)
// of two DMMA.8x8x4 k-steps for a warp (lane*2 + {0,1}).
// Column orders (md4_tables.cpp build_orders): within a bra block the even columns and the odd columns
// are the two k-steps, and the four p~ of a k-step sit in four consecutive 8-byte bank pairs {4g..4g+3}
// of the additive R layout; within a ket block columns 0-3 and 4-7 (the two half warps of a B-fragment
// gather) have bank pairs {c, c+4, c+8, c+12}.  The 16 lanes of a half warp then read 16 different bank
// pairs: the gather of Eq.8 is free of shared-memory bank conflicts.
struct PairListDev {
    int npair, li, lj, Ki, Kj;
    int lsum, nab, nrb, nherm;
    int ncbb, ncbk;      // column blocks in bra / ket order
    size_t hstrideb, hstridek;   // doubles per primitive pair
    double* Hb;          // [npair*Ki*Kj * hstrideb]
    double* Hk;          // [npair*Ki*Kj * hstridek]
    double* scal;        // [npair*Ki*Kj * 8]: zeta_p, Px, Py, Pz, lnK - pairmax, 0, 0, 0
    double* pairmax;     // [npair] max over primitives of ln K_ab
    int* ij;             // [npair*2]
    int* ao;             // [npair*2] first AO (solid-harmonic function) of shells i and j in the shell set the list was built from
    int nbf;             // number of AOs of that shell set
};

// direct digestion (md4_compute_jk): AO-basis density in, Coulomb- / exchange-type matrices out (either may be null)
struct DigestArgs {
    int nbf;
    const double* D;
    double* J;
    double* K;
};

// Interaction kernel (md4_device.cuh kernel_seed): G_m = ka F_m(T) + kb s^(2m+1) F_m(s^2 T), s^2 = omega2/(omega2 + rho)
struct KernelSpec {
    double ka, kb, omega2;
};

// One device allocation that the context may hand from a released pair list to the next one of (about) that size.
// ev (may be null) completes when the last kernel that touches the block has finished; whoever reuses the block
// makes its first writer wait for it (stream-ordered, the host never blocks).
struct PoolBlock {
    void* p = nullptr;
    size_t bytes = 0;     // true size of the allocation
    cudaEvent_t ev = nullptr;
};

}  // namespace md4

struct md4_pairs {
    md4_ctx* ctx;
    md4::PairListDev d;          // views into `block`
    md4::PoolBlock block;        // the list's single device allocation: Hb | Hk | scal | pairmax | ij
    cudaEvent_t ready = nullptr;     // the pair kernel that fills the list has finished (recorded on ctx->build_stream)
    cudaEvent_t last_use = nullptr;  // the last md4_compute that reads the list has finished (recorded on its stream)
    bool used = false;
};

struct md4_ctx {
    int device;
    std::string err;
    md4::DeviceTables tab;
    std::vector<void*> table_allocs;
    // shells (device)
    int nshell = 0, nprim = 0;
    // one device block (grows only) centres | exponents | coefficients | l | offsets, filled through a pinned staging
    // buffer by a stream-ordered copy on build_stream, so replacing the shell set never synchronises the device
    void* d_shell_block = nullptr;
    size_t shell_block_bytes = 0;
    void* h_shell_stage = nullptr;
    size_t shell_stage_bytes = 0;
    cudaEvent_t shell_done = nullptr;
    double* d_centers = nullptr;
    int* d_l = nullptr;
    int* d_off = nullptr;
    double* d_exp = nullptr;
    double* d_coef = nullptr;
    std::vector<int> h_l, h_off, h_ao;   // h_ao: first AO of every shell, h_ao[nshell] = number of AOs
    std::set<md4_pairs*> lists;
    // released pair-list blocks kept for the next md4_build_pairs (workspaces grow only, S:8(b)): a batch loop that
    // builds and frees pair lists every step then never reaches cudaMalloc/cudaFree (both synchronise the device)
    std::multimap<size_t, md4::PoolBlock> pool;
    size_t pool_bytes = 0, pool_max_bytes = 0;
    cudaStream_t build_stream = nullptr;   // pair kernels run here; md4_compute waits for the lists' `ready` events
    // pinned staging for the index lists of md4_build_pairs (the caller's array is copied during the call, the
    // transfer to the device is stream-ordered): a slot is reused once its previous transfer has completed
    static constexpr int NSTAGE = 4;
    int* h_stage[NSTAGE] = {};
    size_t stage_ints[NSTAGE] = {};
    cudaEvent_t stage_done[NSTAGE] = {};
    int stage_next = 0;
    std::set<const void*> configured;      // kernels whose shared-memory opt-in has been set on this device
    double* d_tacc = nullptr;     // partial [ab|q~] of contracted bras, one slab per CTA of the fused kernel (md4_eri.cu)
    cudaEvent_t tacc_free = nullptr;       // completes when the last launch that uses d_tacc has finished
    bool tacc_used = false;
    double* d_scratch = nullptr;  // md4_compute_host staging
    size_t scratch_doubles = 0;
    static constexpr int NSLICE_EV = 8;   // md4_compute_host: bra slices whose D2H copy overlaps the next slice's kernel
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t slice_ev[NSLICE_EV] = {};
    md4::KernelSpec kernel = {1.0, 0.0, 1.0};   // interaction kernel of md4_compute: 1/r12 unless md4_set_kernel changed it
    long long launches = 0;
    int num_sms = 0;
    int smem_optin = 0;
    md4::HostTables htab;
};

namespace md4 {
// md4_pairs.cu
cudaError_t launch_pair_kernel(md4_ctx* ctx, const PairListDev& pl, cudaStream_t st);
// md4_eri.cu
md4_status launch_eri(md4_ctx* ctx, const PairListDev& bra, const PairListDev& ket, double* d_out,
                      cudaStream_t st, const DigestArgs* dg = nullptr);
// same, with the [ab|q~] scratch of contracted bras in the library's file-scope device array (md4_compute_static)
md4_status launch_eri_static(md4_ctx* ctx, const PairListDev& bra, const PairListDev& ket, double* d_out, cudaStream_t st);
void plan_items_host(int nrb_ab, int* nitems, int* row0, int* nrows);   // the work-item split of md4_compute (host logic)
// md4_eri_small.cu: uncontracted low-l classes, one warp per quartet
bool small_class_eligible(const PairListDev& bra, const PairListDev& ket);
md4_status launch_eri_small(md4_ctx* ctx, const PairListDev& bra, const PairListDev& ket, double* d_out, cudaStream_t st);
cudaError_t launch_debug_boys(md4_ctx* ctx, int mmax, int n, const double* d_T, double* d_out);
cudaError_t launch_debug_r(md4_ctx* ctx, int L, const double* d_pq, double* d_out);
}  // namespace md4

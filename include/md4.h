/*
 * md4.h -- C ABI of libmd4: B200-native (sm_100a) FP64 evaluator of 4-center 2-electron repulsion
 * integrals (ab|cd) over contracted real-solid-harmonic Gaussian shells, matrix form of the
 * McMurchie-Davidson scheme ("MD4", arXiv:2307.03452).
 *
 * Citations: P:n = line n of the paper text, S:8(x) = SURVEY.md section 8(x).
 *
 * The engine follows P:200 (section 3): "an engine object is constructed from the given bra and ket
 * basis sets and the integrals are computed asynchronously for the given bra and ket index pair
 * lists"; every pair in a list has the same (l_i, l_j) and the same contraction orders (K_i, K_j);
 * there is no screening: every listed quartet is computed.
 *
 * Definition of the result (Eq.1, Eq.6, Eq.16, S:8(c)):
 *   (ab|cd)_{ma mb mc md} = sum_{ka kb kc kd} c_ka c_kb c_kc c_kd
 *        Int Int chi^ka_{la ma}(r) chi^kb_{lb mb}(r) |r-r'|^-1 chi^kc_{lc mc}(r') chi^kd_{ld md}(r') d3r d3r'
 *   chi^k_{lm}(r) = S_lm(r-A) exp(-zeta_k |r-A|^2), S_lm the real solid harmonics in Racah
 *   normalisation (S_11 = x, S_1-1 = y, S_10 = z, S_20 = z^2 - x^2/2 - y^2/2), m = -l..+l ascending.
 *   Coefficients are applied verbatim to UNNORMALISED primitives: no hidden normalisation.
 *
 * Memory: every pointer argument says HOST or DEVICE.  Host arrays are copied during the call; the
 * caller may free them on return.  The output buffer is a caller-owned DEVICE buffer.
 * Errors: every entry point returns md4_status (or writes nothing and returns NULL/void where noted);
 * nothing throws or aborts across the ABI.  md4_last_error() gives a human-readable reason.
 * Threading: a context is not thread-safe (one host thread at a time); distinct contexts are independent.
 * Stream ordering: no entry point except md4_compute_host, md4_destroy and the md4_debug_* calls waits for
 * the device.  md4_set_shells and md4_build_pairs enqueue their copies and the pair kernel on an internal
 * stream of the context; md4_compute makes the caller's stream wait (on the device) for the pair kernels of
 * both lists.  md4_compute may be called on several streams of one context: launches whose bra list is
 * contracted share one scratch buffer of the context and are therefore ordered one after the other by an
 * internal event (each launch is a persistent grid that fills the GPU, so nothing is lost); all other
 * launches are independent.  md4_free_pairs never synchronises: the list's memory is handed to the next
 * md4_build_pairs together with the event of its last reader.
 */
#ifndef MD4_H
#define MD4_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MD4_LMAX 7 /* highest per-shell angular momentum accepted (k functions; "can be extended") */
#define MD4_LSUM_MAX 24 /* md4_compute needs l_a + l_b + l_c + l_d <= 24 (Hermite tensor R in shared memory), l_c + l_d <= 12
                           and (2l_c+1)(2l_d+1) <= 176: every class of l <= 6 shells, and l = 7 shells with lighter partners */

typedef struct md4_ctx md4_ctx;     /* opaque engine, one per CUDA device                     */
typedef struct md4_pairs md4_pairs; /* opaque shell-pair list (device resident), owned by ctx  */

typedef enum {
    MD4_OK = 0,
    MD4_EINVAL = 1,       /* bad argument: null pointer, index out of range, class mix, zeta <= 0 */
    MD4_EUNSUPPORTED = 2, /* l > MD4_LMAX, or a quartet class beyond MD4_LSUM_MAX                          */
    MD4_ESTATE = 3,       /* call order: pairs before shells, pairs of another context             */
    MD4_ENOMEM = 4,       /* host or device allocation failed                                      */
    MD4_ECUDA = 5         /* CUDA runtime error; text in md4_last_error                            */
} md4_status;

/* Create an engine on CUDA device `cuda_device`.  Builds the constant device tables: Hermite
 * ordinals and the R-recurrence table (Listing 3.1), Cartesian->solid-harmonic coefficients
 * (Eq.16) and the Boys interpolation table (Eq.11).  *out is NULL on failure. */
md4_status md4_create(md4_ctx** out, int cuda_device);

/* Free the engine, its shells, every pair list still alive and all workspaces.  NULL is a no-op. */
void md4_destroy(md4_ctx* ctx);

/* Text of the last failure on this context (ctx-owned, valid until the next call on ctx; never freed
 * by the caller).  With ctx == NULL returns the text of the last failed md4_create on this thread. */
const char* md4_last_error(const md4_ctx* ctx);

/* Upload shells exactly as the paper states the problem (Eq.1): centre, l, primitive
 * exponents, contraction coefficients.  Replaces any previous shell set; existing pair lists stay
 * valid (they hold their own data).
 *   centers_xyz   HOST [nshell*3]  bohr
 *   l             HOST [nshell]    0..MD4_LMAX (7; see MD4_LSUM_MAX for the classes md4_compute accepts)
 *   prim_offset   HOST [nshell+1]  CSR offsets into exponents/coefficients, prim_offset[0] = 0, increasing
 *   exponents     HOST [nprim]     > 0, finite
 *   coefficients  HOST [nprim]     finite, applied verbatim
 * nshell == 0 is accepted (clears the shell set). */
md4_status md4_set_shells(md4_ctx* ctx, int nshell, const double* centers_xyz, const int* l,
                          const int* prim_offset, const double* exponents, const double* coefficients);

/* Interaction kernel g(r12) of every later md4_compute / md4_compute_host / md4_debug_hermite_r on this context
 * (Eq.10: the seed [0]^(m) "is related to the Boys function F_m(x) (or similar quantities for non-Coulomb
 * integrals)", ref. 21; S:8(f) item 3).  Only the seeds change: G_m = F_m(T) for the Coulomb kernel,
 * s^(2m+1) F_m(s^2 T) with s^2 = omega^2/(omega^2 + rho) for erf(omega r12)/r12, and their difference for
 * erfc(omega r12)/r12; the recurrence Eq.13 and both contractions are the same.  omega (1/bohr) must be > 0 and finite
 * for the attenuated kernels and is ignored for MD4_KERNEL_COULOMB.  Pair lists are kernel-independent.  A launch uses
 * the kernel that is set when it is enqueued. */
typedef enum { MD4_KERNEL_COULOMB = 0, MD4_KERNEL_ERF = 1, MD4_KERNEL_ERFC = 2 } md4_kernel;
md4_status md4_set_kernel(md4_ctx* ctx, int kind, double omega);

/* Shell-pair precompute (S:8(a) a1; Eq.3-5, Eq.16, Listing 2.1 lines 2-3):
 * for every listed ordered pair (i,j) and every primitive pair (ka,kb) computes zeta_p, R_p,
 * ln K_ab = -zeta_a zeta_b/zeta_p |AB|^2 and the matrix H (solid-harmonic pair index x Hermite index)
 * = c_ka c_kb * C_la (x) C_lb * E, on the device.  All pairs must share (l_i, l_j, K_i, K_j), else
 * MD4_EINVAL.  A list is role-agnostic: the same list may serve as bra and as ket.
 *   ij   HOST [npair*2]  shell indices (i0,j0,i1,j1,...)
 * npair == 0 gives a valid empty list.  *out is NULL on failure.  The call validates, copies ij and
 * enqueues the pair kernel on the context's internal stream; it does not wait for the kernel (it blocks only
 * when it is several builds ahead of the device).  Device memory comes from the context's pool of released
 * lists when a block of about that size is there (at most max(4 GB, 1/8 of the device memory) are kept idle -- a batch
 * loop that frees a step's lists before building the next step's gets them all back without cudaMalloc; env
 * MD4_POOL_MAX_MB overrides; md4_trim returns the idle blocks to the driver). */
md4_status md4_build_pairs(md4_ctx* ctx, int npair, const int* ij, md4_pairs** out);

/* Release one pair list (also done by md4_destroy).  NULL is a no-op.  Does not synchronise: launches that still
 * read the list finish first, on the device, before its memory is overwritten by a later md4_build_pairs. */
void md4_free_pairs(md4_ctx* ctx, md4_pairs* pairs);

/* Return every idle block of the context's pool to the driver (cudaFree; waits for the launches that still read them).
 * For callers whose own allocator runs short of device memory; the pool refills as lists are released. */
md4_status md4_trim(md4_ctx* ctx);

/* Make cuda_stream wait, on the device, until the pair kernel of `pairs` has finished (the call itself returns at
 * once).  md4_compute does this for both of its lists; the call is for a caller that orders its own work -- or its
 * timing events, as bench.py does -- behind md4_build_pairs. */
md4_status md4_stream_wait_pairs(md4_ctx* ctx, const md4_pairs* pairs, void* cuda_stream);

/* Shape queries of a pair list; return -1 for NULL. */
int md4_pairs_count(const md4_pairs* pairs);
/* info[0..3] = l_i, l_j, K_i, K_j (HOST [4]). */
md4_status md4_pairs_class(const md4_pairs* pairs, int* info);

/* Number of doubles md4_compute writes: npair_bra * npair_ket * (2la+1)(2lb+1)(2lc+1)(2ld+1). */
md4_status md4_output_size(const md4_pairs* bra, const md4_pairs* ket, size_t* n_doubles);

/* Compute every quartet of (bra list) x (ket list) (S:8(a) a2-a9; Eq.6-15, P:115-128 Listing
 * 2.1): Boys F_m(T) -> Hermite Coulomb tensor R by the recurrence Eq.13 in shared memory -> bra
 * transform [ab|q~] = sum_p~ H_ab [p~|q~] -> ket transform (ab|cd) = sum_q~ [ab|q~] H_cd, accumulated
 * over primitive quartets, FP64 throughout.
 *   d_out   DEVICE, 8-byte aligned, capacity_doubles >= md4_output_size; fully OVERWRITTEN with
 *           out[i_bra][j_ket][ma][mb][mc][md], row-major, md fastest, m = -l..+l ascending.
 *   cuda_stream  the caller's cudaStream_t (NULL = default stream).  The call only enqueues work on
 *           that stream and returns: no device synchronisation, no allocation.  The stream first waits for
 *           the pair kernels of both lists (and, for a contracted bra, for the previous such launch of this
 *           context, see "Stream ordering" above).
 * On any error nothing is enqueued.  Empty lists: MD4_OK, nothing written. */
md4_status md4_compute(md4_ctx* ctx, const md4_pairs* bra, const md4_pairs* ket, double* d_out,
                       size_t capacity_doubles, void* cuda_stream);

/* md4_compute for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): same arguments, same result (bit for bit the same kernel), but the one scratch the
 * fused kernel uses -- the partial sums [ab|q~] of CONTRACTED bras (Listing 2.1 line 7), parked between bra
 * primitives -- lives in a file-scope `static __device__` array of MD4_STATIC_SCRATCH_BYTES inside the library instead
 * of the context's own buffer.  The call itself (and everything it calls) allocates nothing on the device: no
 * cudaMalloc, cudaFree or allocating library routine; the pair lists are inputs built beforehand (md4_build_pairs).
 *   - Every GPU that loads libmd4.so holds the array (32 MiB) until the process exits.
 *   - A contracted bra class whose launch needs more (num_SMs x resident CTAs x consumer warps x q~ column blocks x 512
 *     bytes: e.g. (ii|ii), (ih|ih) at K > 1 on 148 SMs) is rejected with MD4_EUNSUPPORTED and a message that names both
 *     numbers; nothing is enqueued.  Uncontracted bras (K_a = K_b = 1) use no scratch and are never rejected for size.
 *   - All calls on a device share the array, across contexts and streams, and it keeps the last call's contents.  The
 *     kernel writes every slot before it reads it, so nothing needs clearing between calls -- but two calls with
 *     contracted bras that OVERLAP on the GPU (different streams, different contexts, different host threads) race on
 *     it and give wrong integrals: the caller serialises them (one stream, or events).  md4_compute does not use the
 *     array and may overlap with one md4_compute_static.
 * Other errors, ordering against the pair builds and the output layout as for md4_compute. */
#define MD4_STATIC_SCRATCH_BYTES (32u * 1024u * 1024u)
md4_status md4_compute_static(md4_ctx* ctx, const md4_pairs* bra, const md4_pairs* ket, double* d_out,
                              size_t capacity_doubles, void* cuda_stream);

/* Same through HOST buffers (the end-to-end path bench.py's "e2e" times): copies the result to
 * h_out [capacity_doubles] (HOST) through an internal device buffer that grows on demand, and
 * synchronises before returning.  Large batches are computed in slices of the bra list; the copy of a slice
 * (internal copy stream) overlaps the kernel of the next one, so with a pinned h_out the call takes
 * max(compute, PCIe transfer) rather than their sum.  Pageable h_out works, without the overlap. */
md4_status md4_compute_host(md4_ctx* ctx, const md4_pairs* bra, const md4_pairs* ket, double* h_out,
                            size_t capacity_doubles, void* cuda_stream);

/* ---- direct digestion (S:8(f) item 2; "computing Fock matrix elements directly", P:249 exchange matrix) ------
 * AO order: the shells of md4_set_shells in table order, 2l+1 real solid harmonics each, m = -l..+l ascending;
 * md4_num_ao gives their number nbf for the current shell set.  A pair list remembers the AO offsets of its shells
 * (of the shell set it was built from). */
md4_status md4_num_ao(const md4_ctx* ctx, int* nbf);

/* For EVERY quartet of (bra list) x (ket list) -- bra pair (a,b), ket pair (c,d) -- exactly
 *     J[a,b] += sum_{cd} (ab|cd) D[c,d]          K[a,c] += sum_{bd} (ab|cd) D[b,d]
 * over the AO blocks of the four shells, and nothing else: no permutational images, no factors (the caller lists the
 * quartets it wants and scales D).  The integrals are contracted with the density blocks in the epilogue of the fused
 * kernel and are never written out: per quartet 8 Nab Ncd bytes of output stream become a few hundred atomic adds.
 *   d_D      DEVICE [nbf*nbf] row-major, read only
 *   d_J, d_K DEVICE [nbf*nbf] row-major, ACCUMULATED into (+=, double atomics: the order of the additions, hence the
 *            last bits, may differ from run to run); either may be NULL (not computed), not both
 * Same stream semantics as md4_compute (enqueue only).  Empty lists: MD4_OK, nothing touched.  Uses the current
 * interaction kernel (md4_set_kernel). */
md4_status md4_compute_jk(md4_ctx* ctx, const md4_pairs* bra, const md4_pairs* ket, const double* d_D,
                          double* d_J, double* d_K, void* cuda_stream);

/* Same through HOST matrices (the end-to-end path of bench.py's "e2e_digest"): copies D and the starting values of
 * J / K to the device, runs md4_compute_jk, copies J / K back and synchronises.  3 nbf^2 doubles cross the bus instead
 * of Nab Ncd doubles per quartet. */
md4_status md4_compute_jk_host(md4_ctx* ctx, const md4_pairs* bra, const md4_pairs* ket, const double* h_D,
                               double* h_J, double* h_K, void* cuda_stream);

/* Number of kernel launches this context has enqueued so far (bench.py's "gpu_launches"). */
long long md4_launch_count(const md4_ctx* ctx);

/* Algorithmic FLOPs per shell quartet for bra x ket, matrix operations only, bra transformed first
 * (Eq.17-18): Kbra Kket 2 Nab Np Nq + Kket 2 Nab Nq Ncd.  0 for NULL. */
double md4_flops_per_quartet(const md4_pairs* bra, const md4_pairs* ket);

/* ---- stage-level access for the parity tests (S:4 test layer 3) --------------------------------- */

/* How md4_compute splits the (2li+1)(2lj+1) rows of a bra class into work items of 8-row blocks, one consumer warp
 * per block (host logic only, no device needed): out7 HOST [7] = number of items per quartet (1 to 3), first row
 * block of item 0..2, row blocks of item 0..2.  The FP64 tensor pipe of sm_100a is per SM sub-partition, so an item
 * of n blocks costs ceil(n/4) block-times; the split minimises their sum.  (One exception is not reported here: under a
 * ket of at most 16 eight-column blocks -- gg, hg, hh, ig -- a bra of 12 to 15 row blocks runs as ONE item of 12-15
 * consumer warps at 128 registers.) */
md4_status md4_debug_work_items(int li, int lj, int* out7);

/* Boys function F_m(T), m = 0..mmax (mmax <= 4*MD4_LMAX), evaluated on the device by the same device
 * function the compute kernel uses (table + Taylor, asymptotic above T_max).
 *   T HOST [n], out HOST [n*(mmax+1)] */
md4_status md4_debug_boys(md4_ctx* ctx, int mmax, int n, const double* T, double* out);

/* Cartesian->solid coefficient table of the library for one l: out HOST [(2l+1) * (l+1)(l+2)/2],
 * row m+l, Cartesian triples ordered x descending then y descending. */
md4_status md4_debug_solid_coeff(md4_ctx* ctx, int l, double* out);

/* Hermite Coulomb tensor R^{(0)}_{tuv}, t+u+v <= L (L <= 4*MD4_LMAX), for one primitive quartet given
 * by (zeta_p, P, zeta_q, Q); prefactor 2 pi^{5/2}/(zeta_p zeta_q sqrt(zeta_p+zeta_q)) included, no K_ab.
 * pq HOST [8] = zeta_p, Px, Py, Pz, zeta_q, Qx, Qy, Qz; out HOST [(L+1)^3] indexed t*(L+1)^2+u*(L+1)+v
 * (entries with t+u+v > L are set to 0). */
md4_status md4_debug_hermite_r(md4_ctx* ctx, int L, const double* pq, double* out);

/* H matrix of primitive pair `iprim` (ka*Kj+kb) of pair `ipair`: out HOST [Nab * Np] row-major,
 * Nab = (2li+1)(2lj+1), Np = (lbra+1)(lbra+2)(lbra+3)/6, Hermite index ordered by degree t+u+v, then t
 * descending, then u descending; also scal HOST [5] = zeta_p, Px, Py, Pz, ln K_ab. */
md4_status md4_debug_pair_h(md4_ctx* ctx, const md4_pairs* pairs, int ipair, int iprim, double* out,
                            double* scal);

#ifdef __cplusplus
}
#endif
#endif /* MD4_H */

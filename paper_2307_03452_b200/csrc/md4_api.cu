// md4_api.cu -- the C ABI of include/md4.h: context, shells, pair lists, compute dispatch.
// Host logic only; every step of the hot path runs in the kernels of md4_pairs.cu / md4_eri.cu.
#include <cmath>
#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <new>

#include "md4_internal.h"

using namespace md4;

namespace {
thread_local std::string g_create_err;

template <class T>
cudaError_t upload(std::vector<void*>* keep, const T* h, size_t n, T** d) {
    *d = nullptr;
    cudaError_t e = cudaMalloc((void**)d, (n ? n : 1) * sizeof(T));
    if (e != cudaSuccess) return e;
    if (keep) keep->push_back(*d);
    if (n) e = cudaMemcpy(*d, h, n * sizeof(T), cudaMemcpyHostToDevice);
    return e;
}

md4_status fail(md4_ctx* ctx, md4_status s, const std::string& msg) {
    if (ctx) ctx->err = msg;
    return s;
}
md4_status cuda_fail(md4_ctx* ctx, const char* what, cudaError_t e) {
    (void)cudaGetLastError();
    return fail(ctx, e == cudaErrorMemoryAllocation ? MD4_ENOMEM : MD4_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

// forget the shell set (the device block is kept for the next one); release: the context is going away
void free_shells(md4_ctx* c, bool release = false) {
    c->d_centers = nullptr; c->d_l = nullptr; c->d_off = nullptr; c->d_exp = nullptr; c->d_coef = nullptr;
    c->nshell = 0; c->nprim = 0; c->h_l.clear(); c->h_off.clear(); c->h_ao.clear();
    if (release) {
        cudaFree(c->d_shell_block); c->d_shell_block = nullptr; c->shell_block_bytes = 0;
        if (c->h_shell_stage) cudaFreeHost(c->h_shell_stage);
        c->h_shell_stage = nullptr; c->shell_stage_bytes = 0;
        if (c->shell_done) cudaEventDestroy(c->shell_done);
        c->shell_done = nullptr;
    }
}

// ---- pool of pair-list blocks --------------------------------------------------------------------------
// A released list's block goes here together with the event of its last reader; the next md4_build_pairs of about
// that size takes it and makes its pair kernel wait for that event on the device.  Nothing here blocks the host.
constexpr size_t POOL_MIN_BYTES = (size_t)64 << 10;          // smaller blocks go straight to cudaMalloc/cudaFree
constexpr size_t POOL_MAX_FLOOR = (size_t)4 << 30;           // bytes kept idle at most: max(this, 1/8 of the device memory); env MD4_POOL_MAX_MB overrides

void pool_release(md4_ctx* c) {
    for (auto& kv : c->pool) {
        if (kv.second.ev) { cudaEventSynchronize(kv.second.ev); cudaEventDestroy(kv.second.ev); }
        cudaFree(kv.second.p);
    }
    c->pool.clear(); c->pool_bytes = 0;
}

// cudaMalloc for anything the context owns: on out-of-memory the idle pool is released and the call retried once
cudaError_t ctx_malloc(md4_ctx* c, void** out, size_t bytes) {
    *out = nullptr;
    cudaError_t e = cudaMalloc(out, bytes ? bytes : 8);
    if (e == cudaErrorMemoryAllocation && !c->pool.empty()) {
        (void)cudaGetLastError();
        pool_release(c);
        e = cudaMalloc(out, bytes ? bytes : 8);
    }
    return e;
}

cudaError_t pool_alloc(md4_ctx* c, size_t bytes, PoolBlock* out) {
    *out = PoolBlock();
    if (bytes >= POOL_MIN_BYTES) {
        auto it = c->pool.lower_bound(bytes);
        if (it != c->pool.end() && it->first <= bytes + bytes / 4) {
            *out = it->second;
            c->pool_bytes -= it->second.bytes;
            c->pool.erase(it);
            return cudaSuccess;
        }
    }
    cudaError_t e = ctx_malloc(c, &out->p, bytes);
    if (e == cudaSuccess) out->bytes = bytes ? bytes : 8;
    return e;
}

// c == nullptr: the context is going away (everything has been synchronised), free for real.  A block that would push
// the pool over its cap evicts the smallest idle blocks first (a sweep over many classes otherwise fills the pool with
// small blocks and then frees -- and re-allocates -- the big ones on every step).
void pool_free(md4_ctx* c, PoolBlock blk) {
    if (!blk.p) { if (blk.ev) cudaEventDestroy(blk.ev); return; }
    if (c && blk.bytes >= POOL_MIN_BYTES && blk.bytes <= c->pool_max_bytes) {
        while (c->pool_bytes + blk.bytes > c->pool_max_bytes && !c->pool.empty()) {
            auto it = c->pool.begin();
            if (it->second.ev) { cudaEventSynchronize(it->second.ev); cudaEventDestroy(it->second.ev); }
            cudaFree(it->second.p);
            c->pool_bytes -= it->second.bytes;
            c->pool.erase(it);
        }
        c->pool.emplace(blk.bytes, blk);
        c->pool_bytes += blk.bytes;
    } else {
        if (blk.ev) { cudaEventSynchronize(blk.ev); cudaEventDestroy(blk.ev); }
        cudaFree(blk.p);
    }
}

// to_pool: the block may be handed to the next list (with the event of its last reader)
void free_pair_storage(md4_pairs* p, bool to_pool) {
    PoolBlock blk = p->block;
    // the block is free once the list's own pair kernel and its last reader are done; both events are recorded in
    // stream order after each other's work only if a compute ran, so keep the later one: last_use if used, else ready
    blk.ev = p->used ? p->last_use : p->ready;
    cudaEvent_t other = p->used ? p->ready : p->last_use;
    if (other) cudaEventDestroy(other);
    pool_free(to_pool ? p->ctx : nullptr, blk);
    delete p;
}

struct DeviceGuard {
    int prev = -1;
    bool ok;
    explicit DeviceGuard(int dev) {
        ok = cudaGetDevice(&prev) == cudaSuccess && cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};
}  // namespace

extern "C" {

md4_status md4_create(md4_ctx** out, int cuda_device) {
    if (!out) { g_create_err = "md4_create: out is NULL"; return MD4_EINVAL; }
    *out = nullptr;
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess) { (void)cudaGetLastError(); g_create_err = std::string("md4_create: no CUDA device: ") + cudaGetErrorString(e); return MD4_ECUDA; }
    if (cuda_device < 0 || cuda_device >= ndev) { g_create_err = "md4_create: cuda_device out of range"; return MD4_EINVAL; }
    md4_ctx* c = new (std::nothrow) md4_ctx();
    if (!c) { g_create_err = "md4_create: out of host memory"; return MD4_ENOMEM; }
    c->device = cuda_device;
    DeviceGuard g(cuda_device);
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, cuda_device);
    if (e != cudaSuccess) { g_create_err = std::string("md4_create: ") + cudaGetErrorString(e); delete c; return MD4_ECUDA; }
    if (prop.major < 10) { g_create_err = "md4_create: libmd4 is built for sm_100a (B200) only"; delete c; return MD4_EUNSUPPORTED; }
    c->num_sms = prop.multiProcessorCount;
    c->smem_optin = (int)prop.sharedMemPerBlockOptin;
    build_host_tables(c->htab);
    uint32_t *d_rtab = nullptr, *d_tuv = nullptr;
    double* d_boys = nullptr;
    e = upload(&c->table_allocs, c->htab.rtab.data(), c->htab.rtab.size(), &d_rtab);
    if (e == cudaSuccess) e = upload(&c->table_allocs, c->htab.tuv.data(), c->htab.tuv.size(), &d_tuv);
    if (e == cudaSuccess) e = upload(&c->table_allocs, c->htab.boys.data(), c->htab.boys.size(), &d_boys);
    c->tab.rtab = d_rtab; c->tab.tuv = d_tuv; c->tab.boys = d_boys;
    for (int lp = 0; lp <= LPAIR && e == cudaSuccess; ++lp) {
        uint32_t* dc = nullptr;
        int* di = nullptr;
        e = upload(&c->table_allocs, c->htab.colb[lp].data(), c->htab.colb[lp].size(), &dc);
        c->tab.colb[lp] = dc;
        if (e == cudaSuccess) { e = upload(&c->table_allocs, c->htab.colk[lp].data(), c->htab.colk[lp].size(), &dc); c->tab.colk[lp] = dc; }
        if (e == cudaSuccess) { e = upload(&c->table_allocs, c->htab.b2k[lp].data(), c->htab.b2k[lp].size(), &di); c->tab.b2k[lp] = di; }
    }
    for (int l = 0; l <= LMAX && e == cudaSuccess; ++l) {
        double* d = nullptr;
        e = upload(&c->table_allocs, c->htab.solid[l].data(), c->htab.solid[l].size(), &d);
        c->tab.solid[l] = d;
        if (e == cudaSuccess) {
            e = upload(&c->table_allocs, c->htab.solid_lo[l].data(), c->htab.solid_lo[l].size(), &d);
            c->tab.solid_lo[l] = d;
        }
    }
    if (e == cudaSuccess) {
        // partial [ab|q~] of contracted bras: one slab per CTA of the persistent fused kernel (L2 resident)
        void* t = nullptr;
        e = cudaMalloc(&t, (size_t)c->num_sms * TACC_WARPS * TACC_QBLOCKS * 64 * sizeof(double));
        if (e == cudaSuccess) { c->table_allocs.push_back(t); c->d_tacc = static_cast<double*>(t); }
    }
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->build_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->tacc_free, cudaEventDisableTiming);
    // a batch loop frees all lists of a step before it builds the next step's: the idle pool must hold a step's working set
    // (13 GB for the 42 batches of cfg5), or every big list goes through cudaFree + cudaMalloc, each a device-wide sync
    c->pool_max_bytes = std::max(POOL_MAX_FLOOR, (size_t)prop.totalGlobalMem / 8);
    if (const char* env = std::getenv("MD4_POOL_MAX_MB")) {
        const long long mb = std::atoll(env);
        if (mb >= 0) c->pool_max_bytes = (size_t)mb << 20;
    }
    if (e != cudaSuccess) {
        g_create_err = std::string("md4_create: table upload: ") + cudaGetErrorString(e);
        for (void* p : c->table_allocs) cudaFree(p);
        if (c->build_stream) cudaStreamDestroy(c->build_stream);
        if (c->tacc_free) cudaEventDestroy(c->tacc_free);
        delete c;
        return e == cudaErrorMemoryAllocation ? MD4_ENOMEM : MD4_ECUDA;
    }
    *out = c;
    return MD4_OK;
}

void md4_destroy(md4_ctx* ctx) {
    if (!ctx) return;
    DeviceGuard g(ctx->device);
    cudaDeviceSynchronize();
    for (md4_pairs* p : ctx->lists) free_pair_storage(p, false);
    ctx->lists.clear();
    pool_release(ctx);
    free_shells(ctx, true);
    cudaFree(ctx->d_scratch);
    if (ctx->copy_stream) {
        for (int i = 0; i < md4_ctx::NSLICE_EV; ++i) cudaEventDestroy(ctx->slice_ev[i]);
        cudaStreamDestroy(ctx->copy_stream);
    }
    for (void* p : ctx->table_allocs) cudaFree(p);
    if (ctx->build_stream) cudaStreamDestroy(ctx->build_stream);
    if (ctx->tacc_free) cudaEventDestroy(ctx->tacc_free);
    for (int i = 0; i < md4_ctx::NSTAGE; ++i) {
        if (ctx->stage_done[i]) cudaEventDestroy(ctx->stage_done[i]);
        if (ctx->h_stage[i]) cudaFreeHost(ctx->h_stage[i]);
    }
    delete ctx;
}

const char* md4_last_error(const md4_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

md4_status md4_set_shells(md4_ctx* ctx, int nshell, const double* centers_xyz, const int* l, const int* prim_offset,
                          const double* exponents, const double* coefficients) {
    if (!ctx) return MD4_EINVAL;
    if (nshell < 0) return fail(ctx, MD4_EINVAL, "md4_set_shells: nshell < 0");
    if (nshell > 0 && (!centers_xyz || !l || !prim_offset || !exponents || !coefficients))
        return fail(ctx, MD4_EINVAL, "md4_set_shells: null array");
    int nprim = 0;
    if (nshell > 0) {
        if (prim_offset[0] != 0) return fail(ctx, MD4_EINVAL, "md4_set_shells: prim_offset[0] != 0");
        for (int i = 0; i < nshell; ++i) {
            if (l[i] < 0) return fail(ctx, MD4_EINVAL, "md4_set_shells: l < 0");
            if (l[i] > LMAX) return fail(ctx, MD4_EUNSUPPORTED, "md4_set_shells: l > MD4_LMAX");
            if (prim_offset[i + 1] <= prim_offset[i]) return fail(ctx, MD4_EINVAL, "md4_set_shells: shell without primitives");
            for (int k = 0; k < 3; ++k)
                if (!std::isfinite(centers_xyz[3 * i + k])) return fail(ctx, MD4_EINVAL, "md4_set_shells: centre not finite");
        }
        nprim = prim_offset[nshell];
        for (int k = 0; k < nprim; ++k) {
            if (!(exponents[k] > 0.0) || !std::isfinite(exponents[k])) return fail(ctx, MD4_EINVAL, "md4_set_shells: exponent must be > 0 and finite");
            if (!std::isfinite(coefficients[k])) return fail(ctx, MD4_EINVAL, "md4_set_shells: coefficient not finite");
        }
    }
    DeviceGuard g(ctx->device);
    free_shells(ctx);
    if (nshell == 0) return MD4_OK;
    auto up = [](size_t x) { return (x + 255) / 256 * 256; };
    const size_t oC = 0, oE = oC + up((size_t)nshell * 3 * sizeof(double)), oK = oE + up((size_t)nprim * sizeof(double)),
                 oL = oK + up((size_t)nprim * sizeof(double)), oO = oL + up((size_t)nshell * sizeof(int)),
                 total = oO + up(((size_t)nshell + 1) * sizeof(int));
    cudaError_t e = cudaSuccess;
    if (!ctx->shell_done) e = cudaEventCreateWithFlags(&ctx->shell_done, cudaEventDisableTiming);
    else e = cudaEventSynchronize(ctx->shell_done);          // the staging buffer is free again
    if (e == cudaSuccess && ctx->shell_stage_bytes < total) {
        if (ctx->h_shell_stage) cudaFreeHost(ctx->h_shell_stage);
        ctx->h_shell_stage = nullptr; ctx->shell_stage_bytes = 0;
        e = cudaMallocHost(&ctx->h_shell_stage, total);
        if (e == cudaSuccess) ctx->shell_stage_bytes = total;
    }
    if (e == cudaSuccess && ctx->shell_block_bytes < total) {
        cudaFree(ctx->d_shell_block);                         // rare (the block only grows); waits for pending pair kernels
        ctx->d_shell_block = nullptr; ctx->shell_block_bytes = 0;
        e = ctx_malloc(ctx, &ctx->d_shell_block, total);
        if (e == cudaSuccess) ctx->shell_block_bytes = total;
    }
    if (e == cudaSuccess) {
        char* h = static_cast<char*>(ctx->h_shell_stage);
        std::memcpy(h + oC, centers_xyz, (size_t)nshell * 3 * sizeof(double));
        std::memcpy(h + oE, exponents, (size_t)nprim * sizeof(double));
        std::memcpy(h + oK, coefficients, (size_t)nprim * sizeof(double));
        std::memcpy(h + oL, l, (size_t)nshell * sizeof(int));
        std::memcpy(h + oO, prim_offset, ((size_t)nshell + 1) * sizeof(int));
        // stream-ordered behind the pair kernels that still read the previous shell set
        e = cudaMemcpyAsync(ctx->d_shell_block, h, total, cudaMemcpyHostToDevice, ctx->build_stream);
    }
    if (e == cudaSuccess) e = cudaEventRecord(ctx->shell_done, ctx->build_stream);
    if (e != cudaSuccess) return cuda_fail(ctx, "md4_set_shells", e);
    char* dbase = static_cast<char*>(ctx->d_shell_block);
    ctx->d_centers = reinterpret_cast<double*>(dbase + oC);
    ctx->d_exp = reinterpret_cast<double*>(dbase + oE);
    ctx->d_coef = reinterpret_cast<double*>(dbase + oK);
    ctx->d_l = reinterpret_cast<int*>(dbase + oL);
    ctx->d_off = reinterpret_cast<int*>(dbase + oO);
    ctx->nshell = nshell; ctx->nprim = nprim;
    ctx->h_l.assign(l, l + nshell);
    ctx->h_off.assign(prim_offset, prim_offset + nshell + 1);
    ctx->h_ao.assign((size_t)nshell + 1, 0);
    for (int i = 0; i < nshell; ++i) ctx->h_ao[i + 1] = ctx->h_ao[i] + n_solid(l[i]);
    return MD4_OK;
}

md4_status md4_set_kernel(md4_ctx* ctx, int kind, double omega) {
    if (!ctx) return MD4_EINVAL;
    if (kind == MD4_KERNEL_COULOMB) { ctx->kernel = {1.0, 0.0, 1.0}; return MD4_OK; }
    if (kind != MD4_KERNEL_ERF && kind != MD4_KERNEL_ERFC) return fail(ctx, MD4_EINVAL, "md4_set_kernel: unknown kernel");
    if (!(omega > 0.0) || !std::isfinite(omega) || !std::isfinite(omega * omega))
        return fail(ctx, MD4_EINVAL, "md4_set_kernel: omega must be > 0 and finite");
    if (kind == MD4_KERNEL_ERF) ctx->kernel = {0.0, 1.0, omega * omega};
    else ctx->kernel = {1.0, -1.0, omega * omega};
    return MD4_OK;
}

md4_status md4_build_pairs(md4_ctx* ctx, int npair, const int* ij, md4_pairs** out) {
    if (!ctx) return MD4_EINVAL;
    if (!out) return fail(ctx, MD4_EINVAL, "md4_build_pairs: out is NULL");
    *out = nullptr;
    if (npair < 0) return fail(ctx, MD4_EINVAL, "md4_build_pairs: npair < 0");
    if (npair > 0 && !ij) return fail(ctx, MD4_EINVAL, "md4_build_pairs: ij is NULL");
    if (npair > 0 && ctx->nshell == 0) return fail(ctx, MD4_ESTATE, "md4_build_pairs: no shells uploaded");
    PairListDev d;
    std::memset(&d, 0, sizeof(d));
    d.npair = npair;
    d.Ki = d.Kj = 1;
    for (int p = 0; p < npair; ++p) {
        const int i = ij[2 * p], j = ij[2 * p + 1];
        if (i < 0 || j < 0 || i >= ctx->nshell || j >= ctx->nshell) return fail(ctx, MD4_EINVAL, "md4_build_pairs: shell index out of range");
        const int li = ctx->h_l[i], lj = ctx->h_l[j];
        const int Ki = ctx->h_off[i + 1] - ctx->h_off[i], Kj = ctx->h_off[j + 1] - ctx->h_off[j];
        if (p == 0) { d.li = li; d.lj = lj; d.Ki = Ki; d.Kj = Kj; }
        else if (li != d.li || lj != d.lj || Ki != d.Ki || Kj != d.Kj)
            return fail(ctx, MD4_EINVAL, "md4_build_pairs: pairs of one list must share (l_i, l_j, K_i, K_j) (P:200)");
    }
    d.lsum = d.li + d.lj;
    d.nab = n_solid(d.li) * n_solid(d.lj);
    d.nrb = (d.nab + 7) / 8;
    d.nherm = n_hermite(d.lsum);
    d.ncbb = (int)ctx->htab.colb[d.lsum].size() / 8;
    d.ncbk = (int)ctx->htab.colk[d.lsum].size() / 8;
    d.hstrideb = (size_t)d.ncbb * d.nrb * 64;
    d.hstridek = (size_t)d.ncbk * d.nrb * 64;
    md4_pairs* pl = new (std::nothrow) md4_pairs();
    if (!pl) return fail(ctx, MD4_ENOMEM, "md4_build_pairs: out of host memory");
    pl->ctx = ctx;
    pl->d = d;
    if (npair > 0) {
        DeviceGuard g(ctx->device);
        // one block per list: Hb | Hk | scal | pairmax | ij (every part 256-byte aligned)
        const size_t nprim = (size_t)npair * d.Ki * d.Kj;
        auto up = [](size_t x) { return (x + 255) / 256 * 256; };
        const size_t oHb = 0, oHk = oHb + up(nprim * d.hstrideb * sizeof(double)), oSc = oHk + up(nprim * d.hstridek * sizeof(double)),
                     oPm = oSc + up(nprim * 8 * sizeof(double)), oIj = oPm + up((size_t)npair * sizeof(double)),
                     total = oIj + up((size_t)npair * 4 * sizeof(int));   // ij, then the AO offsets of the same shells
        cudaError_t e = pool_alloc(ctx, total, &pl->block);
        if (e == cudaSuccess) {
            char* base = static_cast<char*>(pl->block.p);
            pl->d.Hb = reinterpret_cast<double*>(base + oHb);
            pl->d.Hk = reinterpret_cast<double*>(base + oHk);
            pl->d.scal = reinterpret_cast<double*>(base + oSc);
            pl->d.pairmax = reinterpret_cast<double*>(base + oPm);
            pl->d.ij = reinterpret_cast<int*>(base + oIj);
            pl->d.ao = pl->d.ij + 2 * (size_t)npair;
            pl->d.nbf = ctx->h_ao[ctx->nshell];
            e = cudaEventCreateWithFlags(&pl->ready, cudaEventDisableTiming);
        }
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&pl->last_use, cudaEventDisableTiming);
        // a recycled block: its previous readers finish before the pair kernel overwrites it (device-side wait)
        if (e == cudaSuccess && pl->block.ev) {
            e = cudaStreamWaitEvent(ctx->build_stream, pl->block.ev, 0);
            cudaEventDestroy(pl->block.ev);
            pl->block.ev = nullptr;
        }
        // ij is copied to pinned staging before the call returns (the caller may free it); transfer and kernel are only
        // enqueued: md4_compute waits for `ready` on the device.  The host blocks only if all NSTAGE staging slots
        // still wait for their transfers, i.e. when it is that many builds ahead of the device
        if (e == cudaSuccess) {
            const int sl = ctx->stage_next;
            ctx->stage_next = (sl + 1) % md4_ctx::NSTAGE;
            const size_t n = (size_t)npair * 4;
            if (ctx->stage_done[sl]) e = cudaEventSynchronize(ctx->stage_done[sl]);
            else e = cudaEventCreateWithFlags(&ctx->stage_done[sl], cudaEventDisableTiming);
            if (e == cudaSuccess && ctx->stage_ints[sl] < n) {
                if (ctx->h_stage[sl]) cudaFreeHost(ctx->h_stage[sl]);
                ctx->h_stage[sl] = nullptr; ctx->stage_ints[sl] = 0;
                const size_t cap = n < 4096 ? 4096 : n;
                e = cudaMallocHost((void**)&ctx->h_stage[sl], cap * sizeof(int));
                if (e == cudaSuccess) ctx->stage_ints[sl] = cap;
            }
            if (e == cudaSuccess) {
                std::memcpy(ctx->h_stage[sl], ij, (size_t)npair * 2 * sizeof(int));
                for (size_t t = 0; t < (size_t)npair * 2; ++t) ctx->h_stage[sl][(size_t)npair * 2 + t] = ctx->h_ao[ij[t]];
                e = cudaMemcpyAsync(pl->d.ij, ctx->h_stage[sl], n * sizeof(int), cudaMemcpyHostToDevice, ctx->build_stream);
            }
            if (e == cudaSuccess) e = cudaEventRecord(ctx->stage_done[sl], ctx->build_stream);
        }
        if (e == cudaSuccess) e = launch_pair_kernel(ctx, pl->d, ctx->build_stream);
        if (e == cudaSuccess) e = cudaEventRecord(pl->ready, ctx->build_stream);
        if (e != cudaSuccess) {
            cudaStreamSynchronize(ctx->build_stream);
            free_pair_storage(pl, false);
            return cuda_fail(ctx, "md4_build_pairs", e);
        }
    }
    ctx->lists.insert(pl);
    *out = pl;
    return MD4_OK;
}

void md4_free_pairs(md4_ctx* ctx, md4_pairs* pairs) {
    if (!ctx || !pairs) return;
    auto it = ctx->lists.find(pairs);
    if (it == ctx->lists.end()) return;
    ctx->lists.erase(it);
    DeviceGuard g(ctx->device);
    // no synchronisation: the block keeps the event of its last reader, and whoever gets the block next waits for it
    // on the device (pool_alloc / md4_build_pairs); blocks too small for the pool wait for that event on the host
    free_pair_storage(pairs, true);
}

md4_status md4_stream_wait_pairs(md4_ctx* ctx, const md4_pairs* pairs, void* cuda_stream) {
    if (!ctx) return MD4_EINVAL;
    if (!pairs) return fail(ctx, MD4_EINVAL, "md4_stream_wait_pairs: pair list is NULL");
    if (pairs->ctx != ctx || !ctx->lists.count(const_cast<md4_pairs*>(pairs)))
        return fail(ctx, MD4_ESTATE, "md4_stream_wait_pairs: pair list does not belong to this context");
    if (!pairs->ready) return MD4_OK;   // empty list: nothing was enqueued
    DeviceGuard g(ctx->device);
    cudaError_t e = cudaStreamWaitEvent((cudaStream_t)cuda_stream, pairs->ready, 0);
    if (e != cudaSuccess) return cuda_fail(ctx, "md4_stream_wait_pairs", e);
    return MD4_OK;
}

int md4_pairs_count(const md4_pairs* pairs) { return pairs ? pairs->d.npair : -1; }

md4_status md4_pairs_class(const md4_pairs* pairs, int* info) {
    if (!pairs || !info) return MD4_EINVAL;
    info[0] = pairs->d.li; info[1] = pairs->d.lj; info[2] = pairs->d.Ki; info[3] = pairs->d.Kj;
    return MD4_OK;
}

md4_status md4_output_size(const md4_pairs* bra, const md4_pairs* ket, size_t* n_doubles) {
    if (!bra || !ket || !n_doubles) return MD4_EINVAL;
    *n_doubles = (size_t)bra->d.npair * ket->d.npair * bra->d.nab * ket->d.nab;
    return MD4_OK;
}

double md4_flops_per_quartet(const md4_pairs* bra, const md4_pairs* ket) {
    if (!bra || !ket) return 0.0;
    const double kb = (double)bra->d.Ki * bra->d.Kj, kk = (double)ket->d.Ki * ket->d.Kj;
    return kb * kk * 2.0 * bra->d.nab * bra->d.nherm * ket->d.nherm + kk * 2.0 * bra->d.nab * ket->d.nherm * ket->d.nab;
}

long long md4_launch_count(const md4_ctx* ctx) { return ctx ? ctx->launches : 0; }

static md4_status check_compute(md4_ctx* ctx, const md4_pairs* bra, const md4_pairs* ket, const void* out, size_t cap,
                                size_t* need) {
    if (!ctx) return MD4_EINVAL;
    if (!bra || !ket) return fail(ctx, MD4_EINVAL, "md4_compute: pair list is NULL");
    if (bra->ctx != ctx || ket->ctx != ctx || !ctx->lists.count(const_cast<md4_pairs*>(bra)) ||
        !ctx->lists.count(const_cast<md4_pairs*>(ket)))
        return fail(ctx, MD4_ESTATE, "md4_compute: pair list does not belong to this context");
    md4_output_size(bra, ket, need);
    if (*need == 0) return MD4_OK;
    if (!out) return fail(ctx, MD4_EINVAL, "md4_compute: output pointer is NULL");
    if (((uintptr_t)out & 7) != 0) return fail(ctx, MD4_EINVAL, "md4_compute: output pointer not 8-byte aligned");
    if (cap < *need) return fail(ctx, MD4_EINVAL, "md4_compute: output capacity too small");
    return MD4_OK;
}

// Stream ordering around a launch (all device-side, the host never blocks): the launch waits for the pair kernels of
// both lists; a launch with a contracted bra also waits for the previous user of the context's [ab|q~] scratch, so
// two md4_compute calls on different streams of one context cannot race on it (they run one after the other -- each
// is a persistent grid that fills the GPU anyway); afterwards both lists remember the launch as their last reader.
static cudaError_t order_before(md4_ctx* ctx, const md4_pairs* bra, const md4_pairs* ket, cudaStream_t st) {
    cudaError_t e = cudaStreamWaitEvent(st, bra->ready, 0);
    if (e == cudaSuccess && ket != bra) e = cudaStreamWaitEvent(st, ket->ready, 0);
    if (e == cudaSuccess && bra->d.Ki * bra->d.Kj > 1 && ctx->tacc_used) e = cudaStreamWaitEvent(st, ctx->tacc_free, 0);
    return e;
}
static cudaError_t order_after(md4_ctx* ctx, const md4_pairs* bra, const md4_pairs* ket, cudaStream_t st) {
    md4_pairs* b = const_cast<md4_pairs*>(bra);
    md4_pairs* k = const_cast<md4_pairs*>(ket);
    cudaError_t e = cudaSuccess;
    if (bra->d.Ki * bra->d.Kj > 1) { e = cudaEventRecord(ctx->tacc_free, st); ctx->tacc_used = true; }
    // a list read from several streams must outlive all of them: chain the new record behind the old one
    if (e == cudaSuccess && b->used) e = cudaStreamWaitEvent(st, b->last_use, 0);
    if (e == cudaSuccess) { e = cudaEventRecord(b->last_use, st); b->used = true; }
    if (e == cudaSuccess && k != b) {
        if (k->used) e = cudaStreamWaitEvent(st, k->last_use, 0);
        if (e == cudaSuccess) { e = cudaEventRecord(k->last_use, st); k->used = true; }
    }
    return e;
}

md4_status md4_compute(md4_ctx* ctx, const md4_pairs* bra, const md4_pairs* ket, double* d_out, size_t capacity_doubles,
                       void* cuda_stream) {
    size_t need = 0;
    md4_status s = check_compute(ctx, bra, ket, d_out, capacity_doubles, &need);
    if (s != MD4_OK || need == 0) return s;
    DeviceGuard g(ctx->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e = order_before(ctx, bra, ket, st);
    if (e != cudaSuccess) return cuda_fail(ctx, "md4_compute", e);
    s = launch_eri(ctx, bra->d, ket->d, d_out, st);
    if (s != MD4_OK) return s;
    e = order_after(ctx, bra, ket, st);
    if (e != cudaSuccess) return cuda_fail(ctx, "md4_compute", e);
    return MD4_OK;
}

md4_status md4_trim(md4_ctx* ctx) {
    if (!ctx) return MD4_EINVAL;
    DeviceGuard g(ctx->device);
    pool_release(ctx);
    return MD4_OK;
}

// md4_compute with the [ab|q~] scratch in the library's static device array (md4_eri.cu: launch_eri_static).  Ordering:
// the launch waits for the pair kernels of both lists and the lists remember it as their last reader, as in
// md4_compute; the static scratch itself is NOT ordered (shared by every context on the device, md4.h).
md4_status md4_compute_static(md4_ctx* ctx, const md4_pairs* bra, const md4_pairs* ket, double* d_out,
                              size_t capacity_doubles, void* cuda_stream) {
    size_t need = 0;
    md4_status s = check_compute(ctx, bra, ket, d_out, capacity_doubles, &need);
    if (s != MD4_OK || need == 0) return s;
    DeviceGuard g(ctx->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaStreamWaitEvent(st, bra->ready, 0);
    if (e == cudaSuccess && ket != bra) e = cudaStreamWaitEvent(st, ket->ready, 0);
    if (e != cudaSuccess) return cuda_fail(ctx, "md4_compute_static", e);
    s = launch_eri_static(ctx, bra->d, ket->d, d_out, st);
    if (s != MD4_OK) return s;
    md4_pairs* b = const_cast<md4_pairs*>(bra);
    md4_pairs* k = const_cast<md4_pairs*>(ket);
    if (b->used) e = cudaStreamWaitEvent(st, b->last_use, 0);
    if (e == cudaSuccess) { e = cudaEventRecord(b->last_use, st); b->used = true; }
    if (e == cudaSuccess && k != b) {
        if (k->used) e = cudaStreamWaitEvent(st, k->last_use, 0);
        if (e == cudaSuccess) { e = cudaEventRecord(k->last_use, st); k->used = true; }
    }
    if (e != cudaSuccess) return cuda_fail(ctx, "md4_compute_static", e);
    return MD4_OK;
}

md4_status md4_compute_host(md4_ctx* ctx, const md4_pairs* bra, const md4_pairs* ket, double* h_out,
                            size_t capacity_doubles, void* cuda_stream) {
    size_t need = 0;
    md4_status s = check_compute(ctx, bra, ket, h_out, capacity_doubles, &need);
    if (s != MD4_OK || need == 0) return s;
    DeviceGuard g(ctx->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (ctx->scratch_doubles < need) {
        cudaFree(ctx->d_scratch);
        ctx->d_scratch = nullptr; ctx->scratch_doubles = 0;
        void* t = nullptr;
        cudaError_t e = ctx_malloc(ctx, &t, need * sizeof(double));
        if (e != cudaSuccess) return cuda_fail(ctx, "md4_compute_host", e);
        ctx->d_scratch = static_cast<double*>(t);
        ctx->scratch_doubles = need;
    }
    // The bra list is cut into slices: the copy of slice i to the host (copy stream) runs under the kernel of
    // slice i+1 (caller's stream).  out is bra-major, so a slice is one contiguous range of it.  With a pinned
    // h_out the call is bound by max(compute, PCIe) instead of their sum.
    if (!ctx->copy_stream) {
        cudaError_t e = cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking);
        for (int i = 0; i < md4_ctx::NSLICE_EV && e == cudaSuccess; ++i) e = cudaEventCreateWithFlags(&ctx->slice_ev[i], cudaEventDisableTiming);
        if (e != cudaSuccess) return cuda_fail(ctx, "md4_compute_host", e);
    }
    const size_t per_bra = need / (size_t)bra->d.npair;
    int nslice = 1;
    if (need * sizeof(double) >= ((size_t)64 << 20)) nslice = bra->d.npair < md4_ctx::NSLICE_EV ? bra->d.npair : md4_ctx::NSLICE_EV;
    const int kk = bra->d.Ki * bra->d.Kj;
    cudaError_t e = order_before(ctx, bra, ket, st);
    for (int i = 0; i < nslice && e == cudaSuccess; ++i) {
        const int b0 = (int)((long long)bra->d.npair * i / nslice), b1 = (int)((long long)bra->d.npair * (i + 1) / nslice);
        if (b1 == b0) continue;
        PairListDev sub = bra->d;
        sub.npair = b1 - b0;
        sub.Hb += (size_t)b0 * kk * sub.hstrideb;
        sub.Hk += (size_t)b0 * kk * sub.hstridek;
        sub.scal += (size_t)b0 * kk * 8;
        sub.pairmax += b0;
        sub.ij += 2 * (size_t)b0;
        sub.ao += 2 * (size_t)b0;
        double* d_slice = ctx->d_scratch + (size_t)b0 * per_bra;
        s = launch_eri(ctx, sub, ket->d, d_slice, st);
        if (s != MD4_OK) { cudaStreamSynchronize(st); cudaStreamSynchronize(ctx->copy_stream); return s; }
        e = cudaEventRecord(ctx->slice_ev[i], st);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->copy_stream, ctx->slice_ev[i], 0);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(h_out + (size_t)b0 * per_bra, d_slice, (size_t)(b1 - b0) * per_bra * sizeof(double),
                                cudaMemcpyDeviceToHost, ctx->copy_stream);
    }
    if (e == cudaSuccess) e = order_after(ctx, bra, ket, st);
    cudaError_t e2 = cudaStreamSynchronize(st);
    cudaError_t e3 = cudaStreamSynchronize(ctx->copy_stream);
    if (e == cudaSuccess) e = e2 != cudaSuccess ? e2 : e3;
    if (e != cudaSuccess) return cuda_fail(ctx, "md4_compute_host", e);
    return MD4_OK;
}

md4_status md4_num_ao(const md4_ctx* ctx, int* nbf) {
    if (!ctx || !nbf) return MD4_EINVAL;
    *nbf = ctx->nshell ? ctx->h_ao[ctx->nshell] : 0;
    return MD4_OK;
}

static md4_status check_jk(md4_ctx* ctx, const md4_pairs* bra, const md4_pairs* ket, const void* D, const void* J, const void* K,
                           bool* empty) {
    if (!ctx) return MD4_EINVAL;
    if (!bra || !ket) return fail(ctx, MD4_EINVAL, "md4_compute_jk: pair list is NULL");
    if (bra->ctx != ctx || ket->ctx != ctx || !ctx->lists.count(const_cast<md4_pairs*>(bra)) ||
        !ctx->lists.count(const_cast<md4_pairs*>(ket)))
        return fail(ctx, MD4_ESTATE, "md4_compute_jk: pair list does not belong to this context");
    *empty = bra->d.npair == 0 || ket->d.npair == 0;
    if (*empty) return MD4_OK;
    if (!D) return fail(ctx, MD4_EINVAL, "md4_compute_jk: density pointer is NULL");
    if (!J && !K) return fail(ctx, MD4_EINVAL, "md4_compute_jk: J and K are both NULL");
    if (bra->d.nbf != ket->d.nbf) return fail(ctx, MD4_ESTATE, "md4_compute_jk: the two lists were built from shell sets of different size");
    if ((((uintptr_t)D) | ((uintptr_t)J) | ((uintptr_t)K)) & 7) return fail(ctx, MD4_EINVAL, "md4_compute_jk: pointer not 8-byte aligned");
    return MD4_OK;
}

md4_status md4_compute_jk(md4_ctx* ctx, const md4_pairs* bra, const md4_pairs* ket, const double* d_D, double* d_J, double* d_K,
                          void* cuda_stream) {
    bool empty = false;
    md4_status s = check_jk(ctx, bra, ket, d_D, d_J, d_K, &empty);
    if (s != MD4_OK || empty) return s;
    DeviceGuard g(ctx->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e = order_before(ctx, bra, ket, st);
    if (e != cudaSuccess) return cuda_fail(ctx, "md4_compute_jk", e);
    DigestArgs dg{bra->d.nbf, d_D, d_J, d_K};
    s = launch_eri(ctx, bra->d, ket->d, nullptr, st, &dg);
    if (s != MD4_OK) return s;
    e = order_after(ctx, bra, ket, st);
    if (e != cudaSuccess) return cuda_fail(ctx, "md4_compute_jk", e);
    return MD4_OK;
}

md4_status md4_compute_jk_host(md4_ctx* ctx, const md4_pairs* bra, const md4_pairs* ket, const double* h_D, double* h_J, double* h_K,
                               void* cuda_stream) {
    bool empty = false;
    md4_status s = check_jk(ctx, bra, ket, h_D, h_J, h_K, &empty);
    if (s != MD4_OK || empty) return s;
    DeviceGuard g(ctx->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t n2 = (size_t)bra->d.nbf * bra->d.nbf;
    const size_t need = 3 * n2;   // D | J | K
    if (ctx->scratch_doubles < need) {
        cudaFree(ctx->d_scratch);
        ctx->d_scratch = nullptr; ctx->scratch_doubles = 0;
        void* t = nullptr;
        cudaError_t e = ctx_malloc(ctx, &t, need * sizeof(double));
        if (e != cudaSuccess) return cuda_fail(ctx, "md4_compute_jk_host", e);
        ctx->d_scratch = static_cast<double*>(t);
        ctx->scratch_doubles = need;
    }
    double *dD = ctx->d_scratch, *dJ = dD + n2, *dK = dJ + n2;
    cudaError_t e = cudaMemcpyAsync(dD, h_D, n2 * sizeof(double), cudaMemcpyHostToDevice, st);
    // J and K ACCUMULATE (+=): the host values are the starting point
    if (e == cudaSuccess && h_J) e = cudaMemcpyAsync(dJ, h_J, n2 * sizeof(double), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess && h_K) e = cudaMemcpyAsync(dK, h_K, n2 * sizeof(double), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(ctx, "md4_compute_jk_host", e);
    s = md4_compute_jk(ctx, bra, ket, dD, h_J ? dJ : nullptr, h_K ? dK : nullptr, cuda_stream);
    if (s != MD4_OK) { cudaStreamSynchronize(st); return s; }
    if (h_J) e = cudaMemcpyAsync(h_J, dJ, n2 * sizeof(double), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && h_K) e = cudaMemcpyAsync(h_K, dK, n2 * sizeof(double), cudaMemcpyDeviceToHost, st);
    cudaError_t e2 = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = e2;
    if (e != cudaSuccess) return cuda_fail(ctx, "md4_compute_jk_host", e);
    return MD4_OK;
}

md4_status md4_debug_work_items(int li, int lj, int* out7) {
    if (li < 0 || lj < 0 || li > LMAX || lj > LMAX || !out7) return MD4_EINVAL;
    const int nrb = (n_solid(li) * n_solid(lj) + 7) / 8;
    plan_items_host(nrb, out7, out7 + 1, out7 + 4);
    return MD4_OK;
}

md4_status md4_debug_boys(md4_ctx* ctx, int mmax, int n, const double* T, double* out) {
    if (!ctx) return MD4_EINVAL;
    if (mmax < 0 || mmax > LTOT || n < 0 || (n > 0 && (!T || !out))) return fail(ctx, MD4_EINVAL, "md4_debug_boys: bad argument");
    if (n == 0) return MD4_OK;
    for (int i = 0; i < n; ++i)
        if (!(T[i] >= 0.0) || !std::isfinite(T[i])) return fail(ctx, MD4_EINVAL, "md4_debug_boys: T must be >= 0 and finite");
    DeviceGuard g(ctx->device);
    double *dT = nullptr, *dO = nullptr;
    const size_t no = (size_t)n * (mmax + 1);
    cudaError_t e = cudaMalloc((void**)&dT, n * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void**)&dO, no * sizeof(double));
    if (e == cudaSuccess) e = cudaMemcpy(dT, T, n * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = launch_debug_boys(ctx, mmax, n, dT, dO);
    if (e == cudaSuccess) e = cudaMemcpy(out, dO, no * sizeof(double), cudaMemcpyDeviceToHost);
    cudaFree(dT); cudaFree(dO);
    if (e != cudaSuccess) return cuda_fail(ctx, "md4_debug_boys", e);
    return MD4_OK;
}

md4_status md4_debug_solid_coeff(md4_ctx* ctx, int l, double* out) {
    if (!ctx) return MD4_EINVAL;
    if (l < 0 || l > LMAX || !out) return fail(ctx, MD4_EINVAL, "md4_debug_solid_coeff: bad argument");
    DeviceGuard g(ctx->device);
    cudaError_t e = cudaMemcpy(out, ctx->tab.solid[l], (size_t)n_solid(l) * n_cart(l) * sizeof(double), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return cuda_fail(ctx, "md4_debug_solid_coeff", e);
    return MD4_OK;
}

md4_status md4_debug_hermite_r(md4_ctx* ctx, int L, const double* pq, double* out) {
    if (!ctx) return MD4_EINVAL;
    if (L < 0 || L > LTOT || !pq || !out) return fail(ctx, MD4_EINVAL, "md4_debug_hermite_r: bad argument");
    if (!(pq[0] > 0.0) || !(pq[4] > 0.0)) return fail(ctx, MD4_EINVAL, "md4_debug_hermite_r: exponents must be > 0");
    DeviceGuard g(ctx->device);
    const size_t no = (size_t)(L + 1) * (L + 1) * (L + 1);
    double *dP = nullptr, *dO = nullptr;
    cudaError_t e = cudaMalloc((void**)&dP, 8 * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void**)&dO, no * sizeof(double));
    if (e == cudaSuccess) e = cudaMemcpy(dP, pq, 8 * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = launch_debug_r(ctx, L, dP, dO);
    if (e == cudaSuccess) e = cudaMemcpy(out, dO, no * sizeof(double), cudaMemcpyDeviceToHost);
    cudaFree(dP); cudaFree(dO);
    if (e != cudaSuccess) return cuda_fail(ctx, "md4_debug_hermite_r", e);
    return MD4_OK;
}

md4_status md4_debug_pair_h(md4_ctx* ctx, const md4_pairs* pairs, int ipair, int iprim, double* out, double* scal) {
    if (!ctx) return MD4_EINVAL;
    if (!pairs || !out || !scal) return fail(ctx, MD4_EINVAL, "md4_debug_pair_h: null argument");
    if (!ctx->lists.count(const_cast<md4_pairs*>(pairs))) return fail(ctx, MD4_ESTATE, "md4_debug_pair_h: foreign pair list");
    const PairListDev& d = pairs->d;
    const int kk = d.Ki * d.Kj;
    if (ipair < 0 || ipair >= d.npair || iprim < 0 || iprim >= kk) return fail(ctx, MD4_EINVAL, "md4_debug_pair_h: index out of range");
    DeviceGuard g(ctx->device);
    if (pairs->ready) cudaEventSynchronize(pairs->ready);   // the pair kernel runs asynchronously on the build stream
    std::vector<double> blk(d.hstrideb), blk2(d.hstridek);
    double s8[8], pm = 0.0;
    const size_t ip = (size_t)ipair * kk + iprim;
    cudaError_t e = cudaMemcpy(blk.data(), d.Hb + ip * d.hstrideb, d.hstrideb * sizeof(double), cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(blk2.data(), d.Hk + ip * d.hstridek, d.hstridek * sizeof(double), cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(s8, d.scal + ip * 8, sizeof(s8), cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(&pm, d.pairmax + ipair, sizeof(double), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return cuda_fail(ctx, "md4_debug_pair_h", e);
    // out in graded Hermite order; the ket-role copy must hold the same numbers
    const std::vector<int>& g2b = ctx->htab.g2b[d.lsum];
    const std::vector<int>& b2k = ctx->htab.b2k[d.lsum];
    for (int r = 0; r < d.nab; ++r)
        for (int c = 0; c < d.nherm; ++c) {
            const int cb = g2b[c], ck = b2k[cb];
            const double vb = blk[((size_t)(cb >> 3) * d.nrb + (r >> 3)) * 64 + (r & 7) * 8 + (cb & 7)];
            const double vk = blk2[((size_t)(ck >> 3) * d.nrb + (r >> 3)) * 64 + (r & 7) * 8 + (ck & 7)];
            if (vb != vk && !(vb != vb && vk != vk)) return fail(ctx, MD4_ECUDA, "md4_debug_pair_h: bra-role and ket-role copies of H differ");
            out[(size_t)r * d.nherm + c] = vb;
        }
    scal[0] = s8[0]; scal[1] = s8[1]; scal[2] = s8[2]; scal[3] = s8[3]; scal[4] = s8[4] + pm;
    return MD4_OK;
}

}  // extern "C"

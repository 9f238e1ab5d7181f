// shaken.cu -- host side of libshaken: the C ABI of include/shaken.h.
//
// The host does three things: (a1) turns (J, q) into six integer thresholds per chain (PAPER.md:174 heat-bath
// rule on the integer scale), (a4) drives the step loop -- two kernel launches per full step, eq. (15) then
// eq. (16) (Alg. 3 :411-433) -- and (a9) moves int64 records and spins across the boundary.
// Every arithmetic step of the path runs in the kernels of kernels.cuh.  No CPU fallback exists.
#include "../../include/shaken.h"

#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <mutex>
#include <new>
#include <vector>

#include "kernels.cuh"

using namespace shaken;

struct shaken_ctx {
    int L = 0;
    int n_chains = 0;
    uint64_t seed = 0;
    uint32_t flags = 0;
    bool packed = false;

    void *d_sigma = nullptr, *d_tau = nullptr;
    bool own_spins = false;
    long long *d_rec = nullptr;
    int64_t rec_cap = 0;          // in records
    bool own_rec = false;
    bool rec_bound = false;
    int64_t n_rec = 0;
    uint32_t *d_tab = nullptr;    // [n_chains][8] per-chain tables for shaken_run_grid
    unsigned long long *d_bad = nullptr;
    uint2 *d_xch = nullptr;       // band path: hand-over rows xtop, xbot ([2][n_bands][L/4] {word, stamp} each)
    size_t xch_bytes = 0;
    uint32_t xch_stamp = 0;       // last stamp written into d_xch
    int coop = -1;                // cooperative launch supported (-1: not queried yet)
    bool no_cluster = false;      // a cluster launch failed once: small chains stay on one SM each
    mutable uint32_t pw_attr_done = 0;   // per-warp strip kernels whose dynamic shared-memory limit has been raised (launch_half)
    bool no_flow = false;         // test hook: bands of <= 7 rows use the two-phase band kernel instead of the data-flow one
    bool band_refuse_next = false;   // test hook: treat the next cooperative launch as refused (exercises the fall-back)
    void *d_stage = nullptr;      // staging for packed <-> int8 conversion
    size_t stage_bytes = 0;

    cudaStream_t stream = nullptr;
    uint64_t step = 0;
    uint32_t chain0 = 0;
    bool have_sigma = false, have_tau = false;   // the layer holds defined +-1 content (init, set_spins, adopt, or a run)
    int num_sms = 0;
    int variant = 0;
    int group = 1;                // coupling group size (shaken_set_coupling)
    long long *d_coal = nullptr;  // [n_chains / group] coalescence times, -1 = not yet; followed by the difference stamps
    bool perwarp = false;         // strip kernels: per-warp task lists for this run (many small chains)
    int64_t launches = 0;
    // row-slab sharding of one lattice (shaken_create_slab; kernel_slab.cuh)
    bool slab = false;
    int n_rows = 0;               // rows of this slab
    uint32_t row0 = 0;            // global index of its row 0
    void *d_sigma_alloc = nullptr, *d_tau_alloc = nullptr;   // allocations (sigma: rows -1 .. n_rows, tau: rows 0 .. n_rows)
    uint2 *d_inbox = nullptr;     // [2 sides][2 parities][L/4] {word, stamp}
    uint2 *peer_below = nullptr, *peer_above = nullptr;      // the neighbours' inboxes (peer-mapped device pointers)
    void *ipc_below = nullptr, *ipc_above = nullptr;         // ... when opened from IPC handles (closed on destroy)
    uint32_t xstamp = 0;          // exchanges done (every rank counts the same)
    bool published = false;       // the current sigma edge rows are in the neighbours' inboxes
    long long *slab_pending = nullptr;   // record whose C_x, C_y wait for the neighbour's row (closed lazily)
    char err[512] = {0};
};

static thread_local char g_err[512] = {0};

static int fail(shaken_ctx *c, int code, const char *fmt, ...)
{
    char *dst = c ? c->err : g_err;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 512, fmt, ap);
    va_end(ap);
    return code;
}

#define CU(call)                                                                                          \
    do {                                                                                                  \
        cudaError_t e_ = (call);                                                                          \
        if (e_ != cudaSuccess) return fail(ctx, SHAKEN_ECUDA, "%s: %s", #call, cudaGetErrorString(e_));   \
    } while (0)

// ---------------------------------------------------------------------------------------------------
// (a1) thresholds.  P(+|h) = e^h / (2 cosh h) = 1 / (1 + e^{-2h})  (Alg. 3 "exp(h)/2cosh(h)").
// ---------------------------------------------------------------------------------------------------
static uint32_t threshold_nonneg(double a)
{
    const double p = 1.0 / (1.0 + exp(-2.0 * a));
    double v = floor(ldexp(p, 32) + 0.5);
    if (v < 2147483648.0) v = 2147483648.0;
    if (v > 4294967295.0) v = 4294967295.0;
    return (uint32_t)v;
}

static uint32_t threshold_of_field(double h)
{
    if (h >= 0.0) return threshold_nonneg(h);
    return (uint32_t)(4294967296.0 - (double)threshold_nonneg(-h));
}

extern "C" int shaken_thresholds(double J, double q, uint32_t out[6])
{
    if (!out || !isfinite(J) || !isfinite(q)) return fail(nullptr, SHAKEN_EINVAL, "shaken_thresholds: bad argument");
    for (int k = 0; k < 3; ++k)
        for (int c = 0; c < 2; ++c) {
            const double h = (double)(2 * k - 2) * J + (double)(2 * c - 1) * q;   // eq. (14)
            out[2 * k + c] = threshold_of_field(h);
        }
    return SHAKEN_OK;
}

// table as the kernels read it: natural order T[2k + c], padded to 8 words
static void kernel_table(double J, double q, uint32_t tab[8])
{
    shaken_thresholds(J, q, tab);
    tab[6] = tab[7] = 0;
}

// ---------------------------------------------------------------------------------------------------
// context
// ---------------------------------------------------------------------------------------------------
extern "C" const char *shaken_version(void) { return "libshaken 0.1 (sm_100a)"; }

extern "C" const char *shaken_last_error(const shaken_ctx *ctx) { return ctx ? ctx->err : g_err; }

extern "C" int shaken_create(shaken_ctx **out, int32_t L, int32_t n_chains, uint64_t seed, uint32_t flags)
{
    if (!out) return fail(nullptr, SHAKEN_EINVAL, "shaken_create: out is NULL");
    *out = nullptr;
    if (flags != SHAKEN_INT8 && flags != SHAKEN_PACKED) return fail(nullptr, SHAKEN_EINVAL, "shaken_create: unknown flags %u", flags);
    const bool packed = flags == SHAKEN_PACKED;
    const int mult = packed ? 32 : 16;
    if (L < 16 || L > 65536 || L % mult != 0)
        return fail(nullptr, SHAKEN_EINVAL, "shaken_create: L=%d must be a multiple of %d in [16, 65536]", L, mult);
    if (n_chains < 1 || (double)n_chains * (double)L * (double)L >= 1099511627776.0)
        return fail(nullptr, SHAKEN_EINVAL, "shaken_create: n_chains=%d out of range", n_chains);
    shaken_ctx *c = new (std::nothrow) shaken_ctx();
    if (!c) return fail(nullptr, SHAKEN_ENOMEM, "shaken_create: out of host memory");
    c->L = L;
    c->n_chains = n_chains;
    c->seed = seed;
    c->flags = flags;
    c->packed = packed;
    *out = c;
    return SHAKEN_OK;
}

extern "C" int shaken_destroy(shaken_ctx *ctx)
{
    if (!ctx) return SHAKEN_OK;
    if (ctx->have_sigma || ctx->have_tau || ctx->d_rec || ctx->d_tab) cudaStreamSynchronize(ctx->stream);
    if (ctx->slab) {
        if (ctx->ipc_below) cudaIpcCloseMemHandle(ctx->ipc_below);
        if (ctx->ipc_above && ctx->ipc_above != ctx->ipc_below) cudaIpcCloseMemHandle(ctx->ipc_above);
        cudaFree(ctx->d_sigma_alloc);
        cudaFree(ctx->d_tau_alloc);
        cudaFree(ctx->d_inbox);
    } else if (ctx->own_spins) { cudaFree(ctx->d_sigma); cudaFree(ctx->d_tau); }
    if (ctx->own_rec) cudaFree(ctx->d_rec);
    cudaFree(ctx->d_tab);
    cudaFree(ctx->d_bad);
    cudaFree(ctx->d_stage);
    cudaFree(ctx->d_xch);
    cudaFree(ctx->d_coal);
    delete ctx;
    return SHAKEN_OK;
}

extern "C" size_t shaken_spin_bytes(const shaken_ctx *ctx)
{
    if (!ctx) return 0;
    if (ctx->slab) return (size_t)ctx->n_rows * (size_t)ctx->L;
    const size_t n = (size_t)ctx->n_chains * (size_t)ctx->L * (size_t)ctx->L;
    return ctx->packed ? n / 8 : n;
}

extern "C" size_t shaken_record_bytes(const shaken_ctx *ctx)
{
    return ctx ? (size_t)ctx->n_chains * SHAKEN_N_OBS * sizeof(int64_t) : 0;
}

static int ensure_device(shaken_ctx *ctx)
{
    if (ctx->num_sms) return SHAKEN_OK;
    int dev = 0;
    CU(cudaGetDevice(&dev));
    int sms = 0;
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    ctx->num_sms = sms;
    CU(cudaMalloc(&ctx->d_bad, sizeof(unsigned long long)));
    return SHAKEN_OK;
}

static int ensure_spins(shaken_ctx *ctx)
{
    int rc = ensure_device(ctx);
    if (rc) return rc;
    if (ctx->d_sigma && ctx->d_tau) return SHAKEN_OK;
    if (ctx->slab) {
        // sigma holds rows -1 .. n_rows, tau rows 0 .. n_rows (the halo rows live in the arrays, kernel_slab.cuh)
        const size_t row = (size_t)ctx->L, sb = (size_t)(ctx->n_rows + 2) * row, tb = (size_t)(ctx->n_rows + 1) * row;
        void *a = nullptr, *b = nullptr;
        if (cudaMalloc(&a, sb) != cudaSuccess || cudaMalloc(&b, tb) != cudaSuccess) {
            cudaFree(a);
            cudaGetLastError();
            return fail(ctx, SHAKEN_ENOMEM, "cudaMalloc of %zu + %zu slab bytes failed", sb, tb);
        }
        ctx->d_sigma_alloc = a;
        ctx->d_tau_alloc = b;
        ctx->d_sigma = (uint8_t *)a + row;
        ctx->d_tau = b;
        ctx->own_spins = true;
        CU(cudaMemsetAsync(a, 0x01, sb, ctx->stream));
        CU(cudaMemsetAsync(b, 0x01, tb, ctx->stream));
        return SHAKEN_OK;
    }
    const size_t nb = shaken_spin_bytes(ctx);
    void *a = nullptr, *b = nullptr;
    if (cudaMalloc(&a, nb) != cudaSuccess || cudaMalloc(&b, nb) != cudaSuccess) {
        cudaFree(a);
        cudaGetLastError();
        return fail(ctx, SHAKEN_ENOMEM, "cudaMalloc of 2 x %zu bytes failed", nb);
    }
    ctx->d_sigma = a;
    ctx->d_tau = b;
    ctx->own_spins = true;
    // defined content before any init: all +1
    CU(cudaMemsetAsync(a, ctx->packed ? 0xFF : 0x01, nb, ctx->stream));
    CU(cudaMemsetAsync(b, ctx->packed ? 0xFF : 0x01, nb, ctx->stream));
    return SHAKEN_OK;
}

extern "C" int shaken_bind(shaken_ctx *ctx, void *d_sigma, void *d_tau, void *d_records, size_t rec_bytes, void *cuda_stream)
{
    if (!ctx) return fail(nullptr, SHAKEN_EINVAL, "shaken_bind: ctx is NULL");
    if (ctx->slab) return fail(ctx, SHAKEN_ESTATE, "shaken_bind: a slab context owns its buffers (use shaken_set_stream)");
    if (!d_sigma || !d_tau || ((uintptr_t)d_sigma & 15) || ((uintptr_t)d_tau & 15) || d_sigma == d_tau)
        return fail(ctx, SHAKEN_EINVAL, "shaken_bind: sigma/tau must be distinct, non-NULL, 16-byte aligned device pointers");
    if ((d_records == nullptr) != (rec_bytes == 0) || ((uintptr_t)d_records & 7))
        return fail(ctx, SHAKEN_EINVAL, "shaken_bind: records pointer / size mismatch or misaligned");
    int rc = ensure_device(ctx);
    if (rc) return rc;
    if (ctx->have_sigma || ctx->have_tau || ctx->d_rec) CU(cudaStreamSynchronize(ctx->stream));
    if (ctx->own_spins) { cudaFree(ctx->d_sigma); cudaFree(ctx->d_tau); ctx->own_spins = false; }
    if (ctx->own_rec) { cudaFree(ctx->d_rec); ctx->own_rec = false; }
    ctx->d_sigma = d_sigma;
    ctx->d_tau = d_tau;
    ctx->stream = (cudaStream_t)cuda_stream;
    ctx->d_rec = (long long *)d_records;
    ctx->rec_cap = d_records ? (int64_t)(rec_bytes / shaken_record_bytes(ctx)) : 0;
    ctx->rec_bound = d_records != nullptr;
    ctx->n_rec = 0;
    ctx->have_sigma = ctx->have_tau = false;   // content unknown until shaken_init / shaken_set_spins / shaken_adopt_spins
    if (d_records) CU(cudaMemsetAsync(d_records, 0, (size_t)ctx->rec_cap * shaken_record_bytes(ctx), ctx->stream));
    return SHAKEN_OK;
}

static int grow_records(shaken_ctx *ctx, int64_t need)
{
    if (need <= ctx->rec_cap) return SHAKEN_OK;
    if (ctx->rec_bound) return fail(ctx, SHAKEN_ENOSPC, "bound record buffer holds %lld records, %lld needed", (long long)ctx->rec_cap, (long long)need);
    int rc = ensure_device(ctx);
    if (rc) return rc;
    int64_t cap = ctx->rec_cap ? ctx->rec_cap : 64;
    while (cap < need) cap *= 2;
    const size_t rb = shaken_record_bytes(ctx);
    long long *p = nullptr;
    if (cudaMalloc(&p, (size_t)cap * rb) != cudaSuccess) {
        cudaGetLastError();
        return fail(ctx, SHAKEN_ENOMEM, "cudaMalloc of %zu record bytes failed", (size_t)cap * rb);
    }
    CU(cudaMemsetAsync(p, 0, (size_t)cap * rb, ctx->stream));
    if (ctx->d_rec && ctx->n_rec > 0)
        CU(cudaMemcpyAsync(p, ctx->d_rec, (size_t)ctx->n_rec * rb, cudaMemcpyDeviceToDevice, ctx->stream));
    if (ctx->d_rec) {
        CU(cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->d_rec);
    }
    ctx->d_rec = p;
    ctx->rec_cap = cap;
    ctx->own_rec = true;
    return SHAKEN_OK;
}

extern "C" int shaken_reserve_records(shaken_ctx *ctx, int64_t max_records)
{
    if (!ctx || max_records < 0) return fail(ctx, SHAKEN_EINVAL, "shaken_reserve_records: bad argument");
    if (ctx->rec_bound) return fail(ctx, SHAKEN_ESTATE, "shaken_reserve_records: record buffer is bound");
    return grow_records(ctx, max_records);
}

extern "C" int64_t shaken_num_records(const shaken_ctx *ctx) { return ctx ? ctx->n_rec : SHAKEN_EINVAL; }

extern "C" int shaken_clear_records(shaken_ctx *ctx)
{
    if (!ctx) return fail(nullptr, SHAKEN_EINVAL, "shaken_clear_records: ctx is NULL");
    if (ctx->d_rec && ctx->n_rec > 0)
        CU(cudaMemsetAsync(ctx->d_rec, 0, (size_t)ctx->n_rec * shaken_record_bytes(ctx), ctx->stream));
    ctx->n_rec = 0;
    ctx->slab_pending = nullptr;   // (a slab's last record may still have been waiting for its bond sums)
    return SHAKEN_OK;
}

extern "C" int shaken_get_step(const shaken_ctx *ctx, uint64_t *step)
{
    if (!ctx || !step) return SHAKEN_EINVAL;
    *step = ctx->step;
    return SHAKEN_OK;
}

extern "C" int shaken_set_step(shaken_ctx *ctx, uint64_t step)
{
    if (!ctx) return SHAKEN_EINVAL;
    ctx->step = step;
    if (ctx->d_coal) {   // difference stamps are step indices: forget them (coalescence times already found stay)
        const size_t ng = (size_t)(ctx->n_chains / ctx->group);
        CU(cudaMemsetAsync(ctx->d_coal + ng, 0, ng * sizeof(long long), ctx->stream));
    }
    return SHAKEN_OK;
}

extern "C" int shaken_set_chain_offset(shaken_ctx *ctx, uint32_t first_chain)
{
    if (!ctx) return fail(nullptr, SHAKEN_EINVAL, "shaken_set_chain_offset: ctx is NULL");
    if ((uint64_t)first_chain + (uint64_t)ctx->n_chains > 4294967296ull)
        return fail(ctx, SHAKEN_EINVAL, "shaken_set_chain_offset: first_chain + n_chains exceeds 2^32");
    ctx->chain0 = first_chain;
    return SHAKEN_OK;
}

extern "C" int shaken_synchronize(shaken_ctx *ctx)
{
    if (!ctx) return fail(nullptr, SHAKEN_EINVAL, "shaken_synchronize: ctx is NULL");
    CU(cudaStreamSynchronize(ctx->stream));
    return SHAKEN_OK;
}

extern "C" int64_t shaken_launch_count(const shaken_ctx *ctx) { return ctx ? ctx->launches : SHAKEN_EINVAL; }

extern "C" int shaken_set_variant(shaken_ctx *ctx, int variant)
{
    if (!ctx || (variant != 0 && variant != SHAKEN_VARIANT_STRIPS && variant != SHAKEN_VARIANT_PERWARP))
        return fail(ctx, SHAKEN_EINVAL, "shaken_set_variant: unknown variant %d", variant);
    ctx->variant = variant;
    return SHAKEN_OK;
}

// ---------------------------------------------------------------------------------------------------
// coupled chains and coalescence times
// ---------------------------------------------------------------------------------------------------
static int reset_coalescence(shaken_ctx *ctx)
{
    if (!ctx->d_coal) return SHAKEN_OK;
    const size_t ng = (size_t)(ctx->n_chains / ctx->group);
    CU(cudaMemsetAsync(ctx->d_coal, 0xFF, ng * sizeof(long long), ctx->stream));          // -1
    CU(cudaMemsetAsync(ctx->d_coal + ng, 0, ng * sizeof(long long), ctx->stream));        // stamps
    return SHAKEN_OK;
}

extern "C" int shaken_set_coupling(shaken_ctx *ctx, int32_t group)
{
    if (!ctx) return fail(nullptr, SHAKEN_EINVAL, "shaken_set_coupling: ctx is NULL");
    if (group < 1 || ctx->n_chains % group != 0)
        return fail(ctx, SHAKEN_EINVAL, "shaken_set_coupling: group=%d must be >= 1 and divide n_chains=%d", group, ctx->n_chains);
    if (ctx->d_coal) {
        CU(cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->d_coal);
        ctx->d_coal = nullptr;
    }
    ctx->group = group;
    if (group > 1) {
        int rc = ensure_device(ctx);
        if (rc) return rc;
        const size_t ng = (size_t)(ctx->n_chains / group);
        if (cudaMalloc(&ctx->d_coal, 2 * ng * sizeof(long long)) != cudaSuccess) {
            cudaGetLastError();
            ctx->group = 1;
            return fail(ctx, SHAKEN_ENOMEM, "cudaMalloc of the coalescence times failed");
        }
        return reset_coalescence(ctx);
    }
    return SHAKEN_OK;
}

extern "C" int64_t shaken_coalescence(shaken_ctx *ctx, int64_t *out, int64_t max_groups)
{
    if (!ctx || max_groups < 0) return fail(ctx, SHAKEN_EINVAL, "shaken_coalescence: bad argument");
    if (ctx->group <= 1) return 0;
    const int64_t ng = ctx->n_chains / ctx->group, n = ng < max_groups ? ng : max_groups;
    if (n > 0) {
        if (!out) return fail(ctx, SHAKEN_EINVAL, "shaken_coalescence: out is NULL");
        cudaError_t e = cudaMemcpyAsync(out, ctx->d_coal, (size_t)n * sizeof(int64_t), cudaMemcpyDeviceToHost, ctx->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
        if (e != cudaSuccess) return fail(ctx, SHAKEN_ECUDA, "shaken_coalescence: %s", cudaGetErrorString(e));
    }
    return n;
}

static int slab_close_record(shaken_ctx *ctx);

static int grid_for(const shaken_ctx *ctx, long long work_items, int per_thread_items = 1)
{
    long long blocks = (work_items + (long long)256 * per_thread_items - 1) / ((long long)256 * per_thread_items);
    const long long cap = (long long)ctx->num_sms * 16;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    return (int)blocks;
}

// ---------------------------------------------------------------------------------------------------
// (a2) init
// ---------------------------------------------------------------------------------------------------
extern "C" int shaken_init(shaken_ctx *ctx, int mode)
{
    if (!ctx) return fail(nullptr, SHAKEN_EINVAL, "shaken_init: ctx is NULL");
    if (mode != SHAKEN_INIT_UP && mode != SHAKEN_INIT_DOWN && mode != SHAKEN_INIT_IID && mode != SHAKEN_INIT_SANDWICH)
        return fail(ctx, SHAKEN_EINVAL, "shaken_init: mode %d is not +1, -1, 0 or 2", mode);
    if (ctx->slab && mode == SHAKEN_INIT_SANDWICH) return fail(ctx, SHAKEN_EINVAL, "shaken_init: a slab context holds one chain");
    int rc = ensure_spins(ctx);
    if (rc) return rc;
    const size_t nb = shaken_spin_bytes(ctx);
    ctx->published = false;
    ctx->slab_pending = nullptr;
    if (mode == SHAKEN_INIT_IID) {
        const uint32_t k0 = (uint32_t)ctx->seed, k1 = (uint32_t)(ctx->seed >> 32);
        const long long sites = (long long)ctx->L * (ctx->slab ? ctx->n_rows : ctx->L);
        if (ctx->packed) {
            const long long wpc = sites / 32;
            init_iid_pk<<<grid_for(ctx, wpc * ctx->n_chains), 256, 0, ctx->stream>>>((uint32_t *)ctx->d_sigma, (uint32_t *)ctx->d_tau, ctx->n_chains, ctx->chain0, wpc, k0, k1);
        } else {
            const long long cpc = sites / 4;
            init_iid_i8<<<grid_for(ctx, cpc * ctx->n_chains), 256, 0, ctx->stream>>>((uint8_t *)ctx->d_sigma, (uint8_t *)ctx->d_tau, ctx->n_chains, ctx->chain0, cpc, k0, k1, ctx->slab ? ctx->row0 * (uint32_t)(ctx->L / 4) : 0u);
        }
        ctx->launches++;
        CU(cudaGetLastError());
    } else if (mode == SHAKEN_INIT_SANDWICH) {
        const long long n_vec = (long long)(nb / 16), vpc = n_vec / ctx->n_chains;
        const uint32_t plus = ctx->packed ? 0xFFFFFFFFu : 0x01010101u, minus = ctx->packed ? 0u : 0xFFFFFFFFu;
        init_sandwich<<<grid_for(ctx, n_vec), 256, 0, ctx->stream>>>((uint4 *)ctx->d_sigma, (uint4 *)ctx->d_tau, n_vec, vpc, ctx->group, plus, minus);
        ctx->launches++;
        CU(cudaGetLastError());
    } else {
        const int up = mode == SHAKEN_INIT_UP;
        const int byte = ctx->packed ? (up ? 0xFF : 0x00) : (up ? 0x01 : 0xFF);
        CU(cudaMemsetAsync(ctx->d_sigma, byte, nb, ctx->stream));
        CU(cudaMemsetAsync(ctx->d_tau, byte, nb, ctx->stream));
    }
    ctx->have_sigma = ctx->have_tau = true;
    ctx->step = 0;
    int rcc = reset_coalescence(ctx);
    if (rcc) return rcc;
    return shaken_clear_records(ctx);
}

// ---------------------------------------------------------------------------------------------------
// (a3)-(a8) the step loop
// ---------------------------------------------------------------------------------------------------
// launch with programmatic stream serialization (see kernels_common.cuh: wait_for_previous_kernel)
template <typename K, typename P>
static cudaError_t launch_pdl(K kernel, int grid, int threads, cudaStream_t stream, const P &p, size_t dyn_smem = 0)
{
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3((unsigned)threads);
    cfg.dynamicSmemBytes = dyn_smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, p);
}

template <int HALF, int FLAGS>
static cudaError_t launch_half(const shaken_ctx *ctx, const StepParams &p, int grid)
{
    // int8: block tasks (one threshold table per block; plain half-steps use the paired lookup) or per-warp task
    // lists (kernel_i8.cuh); results are identical
    cudaError_t e;
    if (ctx->packed) e = launch_pdl(half_step_pk<HALF, FLAGS>, grid, PK_THREADS, ctx->stream, p);
    else if (ctx->perwarp) {
        // per-warp paired tables (kernel_i8.cuh PWPAIR): 16 warps x 64 entries x 16 copies x 8 B = 128 KiB of dynamic shared memory
        constexpr size_t pw_smem = (FLAGS & F_NOUPDATE) ? 0 : (size_t)(I8_THREADS / 32) * 64 * 16 * sizeof(uint2);
        constexpr uint32_t bit = 1u << (HALF * 16 + FLAGS);           // one bit per instantiation; a context lives on one device
        static_assert(FLAGS < 16, "pw_attr_done holds 16 flag combinations per half-step");
        if (pw_smem && !(ctx->pw_attr_done & bit)) {
            e = cudaFuncSetAttribute(half_step_i8<HALF, FLAGS, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pw_smem);
            if (e != cudaSuccess) return e;
            ctx->pw_attr_done |= bit;
        }
        e = launch_pdl(half_step_i8<HALF, FLAGS, true>, grid, I8_THREADS, ctx->stream, p, pw_smem);
    }
    else e = launch_pdl(half_step_i8<HALF, FLAGS, false>, grid, I8_THREADS, ctx->stream, p);
    return e != cudaSuccess ? e : cudaGetLastError();
}

static int choose_rows_per_task(const shaken_ctx *ctx, int nseg, long long grid_cap, int wpb, double *score_out = nullptr)
{
    const int NR = ctx->slab ? ctx->n_rows : ctx->L;      // rows a launch redraws
    // Strip height R.  Tall strips amortise the halo row and the unprefetched loads at a strip's start; the persistent
    // grid walks block tasks (8 warp strips of one chain) round-robin, so the last wave should be full and so should
    // the warps of a block task.  Maximise
    //     fill * warp_use * machine * R / (R + 3)      (halo row + the unprefetched first rows of a strip)
    // fill = ntasks / (grid * waves), warp_use = strips per chain / (8 * block tasks per chain), machine = grid / cap.
    int best = 4;
    double best_score = -1.0;
    const int Rmax = NR < MAX_ROWS_PER_TASK ? NR : MAX_ROWS_PER_TASK;
    for (int R = Rmax; R >= (NR < 4 ? 1 : 4); --R) {
        const long long nrb = (NR + R - 1) / R;
        const long long tpc = nrb * nseg;
        const long long bpc = (tpc + wpb - 1) / wpb;
        const long long ntasks = (long long)ctx->n_chains * bpc;
        const long long grid = ntasks < grid_cap ? ntasks : grid_cap;
        const long long waves = (ntasks + grid - 1) / grid;
        const double fill = (double)ntasks / (double)(grid * waves);
        const double warp_use = (double)NR / (double)(nrb * R) * (double)tpc / (double)(bpc * wpb);
        const double machine = (double)grid / (double)grid_cap;
        const double score = fill * warp_use * machine * ((double)R / ((double)R + 3.0));
        if (score > best_score + 1e-9) { best_score = score; best = R; }
    }
    if (score_out) *score_out = best_score;
    return best;
}

// ---------------------------------------------------------------------------------------------------
// Band path (kernel_band.cuh, kernel_alt.cuh: alt_band_i8): mid-size lattices, few chains -- the whole run in ONE
// cooperative launch, row bands resident in shared memory.  Returns 0 when the run was launched (bookkeeping done),
// 1 when the path does not apply or the cooperative launch was refused (the strip kernels do the job then), < 0 on error.
// ---------------------------------------------------------------------------------------------------
static int try_band_launch(shaken_ctx *ctx, bool alternate, const uint32_t *gtab, const uint32_t utab[8], int64_t n_steps, int64_t obs_every, int64_t n_new)
{
    if (ctx->packed || ctx->variant != 0 || ctx->group != 1 || ctx->L <= SMALL_L_MAX || ctx->L > BAND_L_MAX || ctx->n_chains > ctx->num_sms) return 1;
    if (ctx->coop < 0) {
        int dev = 0, v = 0;
        CU(cudaGetDevice(&dev));
        CU(cudaDeviceGetAttribute(&v, cudaDevAttrCooperativeLaunch, dev));
        ctx->coop = v;
    }
    int bpc = ctx->num_sms / ctx->n_chains;
    if (bpc > ctx->L) bpc = ctx->L;
    int rpb = (ctx->L + bpc - 1) / bpc;
    if (alternate) rpb += rpb & 1;                                    // even: every band has at least two rows (L is even)
    bpc = (ctx->L + rpb - 1) / rpb;
    const int W = ctx->L / 4;
    const size_t smem = alternate ? alt_band_smem_bytes(ctx->L, rpb) : band_smem_bytes(ctx->L, rpb);
    const int n_bands = bpc * ctx->n_chains;
    // worth it while a half-step is short next to a launch; measured against the strip kernels: 3.6x at 512^2, 2.5x at
    // 1024^2, 2.2x at 2048^2 (the largest band that fits shared memory)
    const bool small_job = (double)ctx->n_chains * ctx->L * ctx->L <= 4.5e6;
    if (!ctx->coop || !small_job || smem > 160 * 1024) return 1;
    const int rows_out = alternate ? 2 : 1;                           // rows a band publishes per side and step
    const size_t xrow = (size_t)2 * n_bands * rows_out * W;           // uint2 elements per hand-over array (two parities)
    const size_t need = 2 * xrow * sizeof(uint2);
    if (ctx->xch_bytes < need) {
        cudaFree(ctx->d_xch);
        ctx->d_xch = nullptr;
        ctx->xch_bytes = 0;
        if (cudaMalloc(&ctx->d_xch, need) != cudaSuccess) {
            cudaGetLastError();
            return fail(ctx, SHAKEN_ENOMEM, "cudaMalloc of %zu exchange bytes failed", need);
        }
        ctx->xch_bytes = need;
        ctx->xch_stamp = 0xFFFFFFFFu;                                // forces the clearing below
    }
    // stamps must be new to the buffer: clear it when the 32-bit stamp space would wrap (or after allocation)
    if ((uint64_t)ctx->xch_stamp + (uint64_t)n_steps + 2ull >= 0xFFFFFFFFull) {
        if ((uint64_t)n_steps >= 0x7FFFFFF0ull) return fail(ctx, SHAKEN_EINVAL, "shaken_run: n_steps too large for one call");
        CU(cudaMemsetAsync(ctx->d_xch, 0, ctx->xch_bytes, ctx->stream));
        ctx->xch_stamp = 0;
    }
    BandParams bp;
    memset(&bp, 0, sizeof(bp));
    bp.sigma = (uint8_t *)ctx->d_sigma;
    bp.tau = (uint8_t *)ctx->d_tau;
    bp.L = ctx->L;
    bp.n_chains = ctx->n_chains;
    bp.chain0 = ctx->chain0;
    bp.t0 = ctx->step;
    bp.n_steps = n_steps;
    bp.obs_every = obs_every;
    bp.rec = ctx->d_rec ? ctx->d_rec + (size_t)ctx->n_rec * ctx->n_chains * SHAKEN_N_OBS : nullptr;
    bp.gtab = gtab;
    memcpy(bp.utab, utab, sizeof(bp.utab));
    make_step_keys(ctx->seed, 0, bp.keys);
    bp.bpc = bpc;
    bp.rows_per_band = rpb;
    bp.xtop = ctx->d_xch;
    bp.xbot = ctx->d_xch + xrow;
    bp.stamp0 = ctx->xch_stamp;
    bp.magicW = (uint32_t)(4294967296ull / (uint64_t)W) + 1u;
    bp.magicV = (uint32_t)(4294967296ull / (uint64_t)(W / 4)) + 1u;
    ctx->xch_stamp += (uint32_t)n_steps;                             // one stamp per full step
    // bands of at most 7 rows (cfg 2): the data-flow schedule (kernel_flow.cuh); taller bands: two phases per step
    const bool flow = !alternate && !ctx->no_flow && flow_applies(ctx->L, rpb);
    const void *kernel = alternate ? (const void *)alt_band_i8 : flow ? (const void *)band_flow_i8 : (const void *)band_run_i8;
    if (flow) bp.slot_group = flow_slot_groups(ctx->L, rpb);
    CU(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    void *args[] = {&bp};
    // the bands wait for one another, so they must all be resident: a cooperative launch either guarantees
    // that or fails up front (a smaller or shared GPU) -- then the strip kernels do the job
    const cudaError_t le = ctx->band_refuse_next ? cudaErrorCooperativeLaunchTooLarge
                                                 : cudaLaunchCooperativeKernel(kernel, dim3(n_bands), dim3(BAND_THREADS), args, smem, ctx->stream);
    ctx->band_refuse_next = false;
    if (le == cudaSuccess) {
        ctx->launches++;
        ctx->step += (uint64_t)n_steps;
        ctx->n_rec += n_new;
        if (!alternate) ctx->have_tau = true;
        return 0;
    }
    cudaGetLastError();
    ctx->xch_stamp -= (uint32_t)n_steps;
    if (le != cudaErrorCooperativeLaunchTooLarge && le != cudaErrorLaunchOutOfResources && le != cudaErrorNotSupported)
        return fail(ctx, SHAKEN_ECUDA, "band kernel launch: %s", cudaGetErrorString(le));
    return 1;
}

// ---------------------------------------------------------------------------------------------------
// shaken_run_static: the band path for callers that must not allocate.  The band kernels' only scratch memory -- the
// hand-over rows xtop / xbot -- is a file-scope device array instead of a cudaMalloc'ed buffer.  In HOST code the array's
// name is a host-side stand-in, not a device address: the address the kernels get comes from cudaGetSymbolAddress, looked
// up once per device (with that device current) in shaken_static_setup.
// ---------------------------------------------------------------------------------------------------
constexpr size_t STATIC_XCH_PAIRS = (size_t)SHAKEN_STATIC_SCRATCH_BYTES / sizeof(uint2);
static __device__ __align__(256) uint2 g_static_xch[STATIC_XCH_PAIRS];

struct StaticDevice {
    bool ready = false;
    uint2 *xch = nullptr;       // device address of g_static_xch on this device
    int num_sms = 0;
    int coop = 0;
};
constexpr int STATIC_MAX_DEVICES = 64;
static StaticDevice g_static_dev[STATIC_MAX_DEVICES];
static std::mutex g_static_mutex;

static int static_device(StaticDevice **out)
{
    shaken_ctx *ctx = nullptr;
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return fail(nullptr, SHAKEN_EINVAL, "shaken_static_setup: device ordinal %d not supported", dev);
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticDevice &d = g_static_dev[dev];
    if (!d.ready) {
        uint2 *ptr = nullptr;
        CU(cudaGetSymbolAddress((void **)&ptr, g_static_xch));
        if (!ptr) return fail(nullptr, SHAKEN_ECUDA, "shaken_static_setup: no device address for the scratch array");
        CU(cudaDeviceGetAttribute(&d.num_sms, cudaDevAttrMultiProcessorCount, dev));
        CU(cudaDeviceGetAttribute(&d.coop, cudaDevAttrCooperativeLaunch, dev));
        d.xch = ptr;
        d.ready = true;
    }
    *out = &d;
    return SHAKEN_OK;
}

extern "C" int shaken_static_setup(void)
{
    StaticDevice *d = nullptr;
    return static_device(&d);
}

extern "C" int shaken_run_static(void *sigma, void *tau, int32_t L, int32_t n_chains, uint64_t seed, uint64_t t0, double J, double q,
                                 int64_t n_steps, int64_t obs_every, int64_t *rec, int64_t max_records, void *cuda_stream)
{
    shaken_ctx *ctx = nullptr;                                        // (errors go to the thread's message buffer)
    if (!sigma || !tau || ((uintptr_t)sigma & 15) || ((uintptr_t)tau & 15))
        return fail(nullptr, SHAKEN_EINVAL, "shaken_run_static: sigma and tau must be non-NULL, 16-byte aligned device pointers");
    if (L <= SMALL_L_MAX || L > BAND_L_MAX || L % 16 != 0)
        return fail(nullptr, SHAKEN_EINVAL, "shaken_run_static: L=%d must be a multiple of 16 in (%d, %d]", L, SMALL_L_MAX, BAND_L_MAX);
    if (!isfinite(J) || !isfinite(q)) return fail(nullptr, SHAKEN_EINVAL, "shaken_run_static: non-finite coupling");
    if (n_steps < 0 || obs_every < 0 || max_records < 0) return fail(nullptr, SHAKEN_EINVAL, "shaken_run_static: negative count");
    if ((uint64_t)n_steps >= 0x7FFFFFF0ull) return fail(nullptr, SHAKEN_EINVAL, "shaken_run_static: n_steps too large for one call");
    StaticDevice *d = nullptr;
    int rc = static_device(&d);
    if (rc) return rc;
    if (n_chains < 1 || n_chains > d->num_sms)
        return fail(nullptr, SHAKEN_EINVAL, "shaken_run_static: n_chains=%d must lie in [1, %d] (one band per SM at least)", n_chains, d->num_sms);
    if (!d->coop) return fail(nullptr, SHAKEN_ECUDA, "shaken_run_static: the device has no cooperative launch");
    // bands as in the context path (try_band_launch)
    int bpc = d->num_sms / n_chains;
    if (bpc > L) bpc = L;
    const int rpb = (L + bpc - 1) / bpc;
    bpc = (L + rpb - 1) / rpb;
    const int W = L / 4;
    const int n_bands = bpc * n_chains;
    const size_t smem = band_smem_bytes(L, rpb);
    if (smem > 160 * 1024)
        return fail(nullptr, SHAKEN_EINVAL, "shaken_run_static: %d chains of %d^2 need bands of %d rows = %zu bytes of shared memory, beyond the maximum of %d",
                    n_chains, L, rpb, smem, 160 * 1024);
    const size_t xrow = (size_t)2 * n_bands * W;                      // uint2 elements per hand-over array (two parities)
    const size_t need = 2 * xrow * sizeof(uint2);
    if (need > (size_t)SHAKEN_STATIC_SCRATCH_BYTES)
        return fail(nullptr, SHAKEN_EINVAL, "shaken_run_static: %d bands of %d-spin rows need %zu bytes of hand-over scratch, beyond the static maximum of %d",
                    n_bands, L, need, SHAKEN_STATIC_SCRATCH_BYTES);
    int64_t n_new = 0;
    if (obs_every > 0) n_new = (int64_t)((t0 + (uint64_t)n_steps) / (uint64_t)obs_every - t0 / (uint64_t)obs_every);
    if (n_new > 0 && !rec) return fail(nullptr, SHAKEN_EINVAL, "shaken_run_static: rec is NULL but the run takes %lld records", (long long)n_new);
    if (n_new > max_records) return fail(nullptr, SHAKEN_ENOSPC, "shaken_run_static: the run takes %lld records, rec holds %lld", (long long)n_new, (long long)max_records);
    if (n_steps == 0) return SHAKEN_OK;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    // the array keeps the last call's contents: stamps must be new to it, so clear the part this call uses (stamp 0 = none)
    CU(cudaMemsetAsync(d->xch, 0, need, stream));
    if (n_new > 0) CU(cudaMemsetAsync(rec, 0, (size_t)n_new * n_chains * SHAKEN_N_OBS * sizeof(int64_t), stream));
    BandParams bp;
    memset(&bp, 0, sizeof(bp));
    bp.sigma = (uint8_t *)sigma;
    bp.tau = (uint8_t *)tau;
    bp.L = L;
    bp.n_chains = n_chains;
    bp.chain0 = 0;
    bp.t0 = t0;
    bp.n_steps = n_steps;
    bp.obs_every = obs_every;
    bp.rec = n_new > 0 ? (long long *)rec : nullptr;
    bp.gtab = nullptr;
    kernel_table(J, q, bp.utab);
    make_step_keys(seed, 0, bp.keys);
    bp.bpc = bpc;
    bp.rows_per_band = rpb;
    bp.xtop = d->xch;                                                 // the DEVICE address from cudaGetSymbolAddress
    bp.xbot = d->xch + xrow;
    bp.stamp0 = 0;
    bp.magicW = (uint32_t)(4294967296ull / (uint64_t)W) + 1u;
    bp.magicV = (uint32_t)(4294967296ull / (uint64_t)(W / 4)) + 1u;
    const void *kernel = flow_applies(L, rpb) ? (const void *)band_flow_i8 : (const void *)band_run_i8;
    bp.slot_group = flow_slot_groups(L, rpb);
    CU(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    void *args[] = {&bp};
    const cudaError_t le = cudaLaunchCooperativeKernel(kernel, dim3(n_bands), dim3(BAND_THREADS), args, smem, stream);
    if (le != cudaSuccess) {
        cudaGetLastError();
        return fail(nullptr, SHAKEN_ECUDA, "shaken_run_static: cooperative launch of %d bands: %s", n_bands, cudaGetErrorString(le));
    }
    return SHAKEN_OK;
}

// ---------------------------------------------------------------------------------------------------
// Row-slab sharding of one lattice (second bullet; kernel_slab.cuh)
// ---------------------------------------------------------------------------------------------------
extern "C" int shaken_create_slab(shaken_ctx **out, int32_t L, int32_t row0, int32_t n_rows, uint64_t seed)
{
    if (!out) return fail(nullptr, SHAKEN_EINVAL, "shaken_create_slab: out is NULL");
    *out = nullptr;
    if (L < 16 || L > 65536 || L % 16 != 0) return fail(nullptr, SHAKEN_EINVAL, "shaken_create_slab: L=%d must be a multiple of 16 in [16, 65536]", L);
    if (row0 < 0 || n_rows < 2 || row0 + n_rows > L)
        return fail(nullptr, SHAKEN_EINVAL, "shaken_create_slab: rows [%d, %d) must lie in [0, L) and be at least two", row0, row0 + n_rows);
    shaken_ctx *c = new (std::nothrow) shaken_ctx();
    if (!c) return fail(nullptr, SHAKEN_ENOMEM, "shaken_create_slab: out of host memory");
    c->L = L;
    c->n_chains = 1;
    c->seed = seed;
    c->flags = SHAKEN_INT8;
    c->slab = true;
    c->row0 = (uint32_t)row0;
    c->n_rows = n_rows;
    *out = c;
    return SHAKEN_OK;
}

extern "C" int shaken_set_stream(shaken_ctx *ctx, void *cuda_stream)
{
    if (!ctx) return fail(nullptr, SHAKEN_EINVAL, "shaken_set_stream: ctx is NULL");
    if (ctx->d_sigma || ctx->d_rec) CU(cudaStreamSynchronize(ctx->stream));
    ctx->stream = (cudaStream_t)cuda_stream;
    return SHAKEN_OK;
}

static int slab_ensure_inbox(shaken_ctx *ctx)
{
    if (ctx->d_inbox) return SHAKEN_OK;
    const size_t bytes = (size_t)4 * (ctx->L / 4) * sizeof(uint2);
    if (cudaMalloc(&ctx->d_inbox, bytes) != cudaSuccess) {
        cudaGetLastError();
        return fail(ctx, SHAKEN_ENOMEM, "cudaMalloc of the slab inbox failed");
    }
    CU(cudaMemset(ctx->d_inbox, 0, bytes));            // stamp 0 is never used by an exchange
    return SHAKEN_OK;
}

extern "C" int shaken_slab_inbox(shaken_ctx *ctx, void **d_inbox, size_t *bytes)
{
    if (!ctx || !ctx->slab || !d_inbox) return fail(ctx, SHAKEN_EINVAL, "shaken_slab_inbox: not a slab context or NULL argument");
    int rc = slab_ensure_inbox(ctx);
    if (rc) return rc;
    *d_inbox = ctx->d_inbox;
    if (bytes) *bytes = (size_t)4 * (ctx->L / 4) * sizeof(uint2);
    return SHAKEN_OK;
}

extern "C" int shaken_slab_connect(shaken_ctx *ctx, void *d_inbox_below, void *d_inbox_above)
{
    if (!ctx || !ctx->slab || !d_inbox_below || !d_inbox_above) return fail(ctx, SHAKEN_EINVAL, "shaken_slab_connect: not a slab context or NULL argument");
    int rc = slab_ensure_inbox(ctx);
    if (rc) return rc;
    ctx->peer_below = (uint2 *)d_inbox_below;
    ctx->peer_above = (uint2 *)d_inbox_above;
    ctx->published = false;
    return SHAKEN_OK;
}

extern "C" int shaken_slab_ipc_export(shaken_ctx *ctx, void *handle64)
{
    if (!ctx || !ctx->slab || !handle64) return fail(ctx, SHAKEN_EINVAL, "shaken_slab_ipc_export: not a slab context or NULL argument");
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "IPC handle size");
    int rc = slab_ensure_inbox(ctx);
    if (rc) return rc;
    cudaIpcMemHandle_t h;
    CU(cudaIpcGetMemHandle(&h, ctx->d_inbox));
    memcpy(handle64, &h, 64);
    return SHAKEN_OK;
}

extern "C" int shaken_slab_ipc_connect(shaken_ctx *ctx, const void *below_handle64, const void *above_handle64)
{
    if (!ctx || !ctx->slab || !below_handle64 || !above_handle64) return fail(ctx, SHAKEN_EINVAL, "shaken_slab_ipc_connect: not a slab context or NULL argument");
    cudaIpcMemHandle_t hb, ha;
    memcpy(&hb, below_handle64, 64);
    memcpy(&ha, above_handle64, 64);
    void *pb = nullptr, *pa = nullptr;
    CU(cudaIpcOpenMemHandle(&pb, hb, cudaIpcMemLazyEnablePeerAccess));
    if (memcmp(&hb, &ha, 64) == 0) pa = pb;             // two ranks: the same neighbour on both sides
    else if (cudaIpcOpenMemHandle(&pa, ha, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess) {
        const cudaError_t e = cudaGetLastError();
        cudaIpcCloseMemHandle(pb);
        return fail(ctx, SHAKEN_ECUDA, "cudaIpcOpenMemHandle (rank above): %s", cudaGetErrorString(e));
    }
    ctx->ipc_below = pb;
    ctx->ipc_above = pa;
    return shaken_slab_connect(ctx, pb, pa);
}

static void slab_params(shaken_ctx *ctx, SlabParams &sp, double J, double q, uint64_t t)
{
    memset(&sp, 0, sizeof(sp));
    sp.sigma = (uint8_t *)ctx->d_sigma;
    sp.tau = (uint8_t *)ctx->d_tau;
    sp.L = ctx->L;
    sp.n_rows = ctx->n_rows;
    sp.row0 = ctx->row0;
    sp.chain = ctx->chain0;
    sp.inbox = ctx->d_inbox;
    sp.to_below = ctx->peer_below;
    sp.to_above = ctx->peer_above;
    sp.stamp = ctx->xstamp;
    kernel_table(J, q, sp.utab);
    make_step_keys(ctx->seed, 2 * t, sp.keys);
}

static int slab_grid(const shaken_ctx *ctx, int items)
{
    int g = (items + SLAB_THREADS - 1) / SLAB_THREADS;
    return g < 1 ? 1 : (g > ctx->num_sms ? ctx->num_sms : g);
}

// store this slab's bottom and top sigma rows into the neighbours' inboxes (a new exchange: every rank counts alike)
static int slab_publish_now(shaken_ctx *ctx)
{
    if (ctx->xstamp == 0xFFFFFFFFu) return fail(ctx, SHAKEN_ESTATE, "slab exchange counter exhausted (2^32 - 1 exchanges)");
    ctx->xstamp++;
    SlabParams sp;
    slab_params(ctx, sp, 0.0, 0.0, 0);
    slab_publish<<<slab_grid(ctx, ctx->L / 4), SLAB_THREADS, 0, ctx->stream>>>(sp);
    CU(cudaGetLastError());
    ctx->launches++;
    ctx->published = true;
    return SHAKEN_OK;
}

extern "C" int shaken_slab_exchange(shaken_ctx *ctx)
{
    if (!ctx || !ctx->slab) return fail(ctx, SHAKEN_EINVAL, "shaken_slab_exchange: not a slab context");
    if (!ctx->peer_below || !ctx->peer_above) return fail(ctx, SHAKEN_ESTATE, "shaken_slab_exchange: not connected (shaken_slab_connect)");
    if (!ctx->have_sigma) return fail(ctx, SHAKEN_ESTATE, "shaken_slab_exchange: no sigma yet");
    int rc = ensure_device(ctx);
    if (rc) return rc;
    return ctx->published ? SHAKEN_OK : slab_publish_now(ctx);
}

// the record of the last step of a run still lacks C_x, C_y: they need the neighbour's new row below this slab
static int slab_close_record(shaken_ctx *ctx)
{
    if (!ctx->published) { int rc = slab_publish_now(ctx); if (rc) return rc; }
    SlabParams sp;
    slab_params(ctx, sp, 0.0, 0.0, 0);
    sp.redraw = 0;
    slab_edge<<<slab_grid(ctx, ctx->L / 16), SLAB_THREADS, 0, ctx->stream>>>(sp);
    CU(cudaGetLastError());
    StepParams p;
    memset(&p, 0, sizeof(p));
    p.L = ctx->L;
    p.nvec = ctx->L / 16;
    p.n_chains = 1;
    p.chain0 = ctx->chain0;
    p.group = 1;
    p.nseg = (p.nvec + 31) / 32;
    p.slab_rows = ctx->n_rows;
    p.row0 = ctx->row0;
    p.rows_per_task = choose_rows_per_task(ctx, p.nseg, ctx->num_sms, I8_THREADS / 32);
    p.nrb = (ctx->n_rows + p.rows_per_task - 1) / p.rows_per_task;
    p.ntasks = ((long long)p.nrb * p.nseg + I8_THREADS / 32 - 1) / (I8_THREADS / 32);
    p.src = ctx->d_sigma;
    p.rec_prev = ctx->slab_pending;
    ctx->perwarp = false;
    const int grid = (int)(p.ntasks < ctx->num_sms ? p.ntasks : ctx->num_sms);
    cudaError_t e = launch_half<0, F_BONDS | F_NOUPDATE>(ctx, p, grid);
    if (e != cudaSuccess) return fail(ctx, SHAKEN_ECUDA, "slab bond-sum launch: %s", cudaGetErrorString(e));
    ctx->launches += 2;
    ctx->slab_pending = nullptr;
    return SHAKEN_OK;
}

static int run_slab(shaken_ctx *ctx, double J, double q, int64_t n_steps, int64_t obs_every)
{
    if (!ctx->peer_below || !ctx->peer_above) return fail(ctx, SHAKEN_ESTATE, "shaken_run: slab not connected (shaken_slab_connect)");
    StepParams p;
    memset(&p, 0, sizeof(p));
    p.L = ctx->L;
    p.nvec = ctx->L / 16;
    p.n_chains = 1;
    p.chain0 = ctx->chain0;
    p.group = 1;
    p.nseg = (p.nvec + 31) / 32;
    p.slab_rows = ctx->n_rows;
    p.row0 = ctx->row0;
    const int wpb = I8_THREADS / 32;
    p.rows_per_task = choose_rows_per_task(ctx, p.nseg, ctx->num_sms, wpb);
    p.nrb = (ctx->n_rows + p.rows_per_task - 1) / p.rows_per_task;
    p.ntasks = ((long long)p.nrb * p.nseg + wpb - 1) / wpb;
    kernel_table(J, q, p.utab);
    ctx->perwarp = false;
    const int grid = (int)(p.ntasks < ctx->num_sms ? p.ntasks : ctx->num_sms);
    const size_t rec_stride = SHAKEN_N_OBS;
    ctx->have_tau = true;
    long long *pending = ctx->slab_pending;             // a record of an earlier call that still lacks C_x, C_y
    ctx->slab_pending = nullptr;
    for (int64_t s = 0; s < n_steps; ++s) {
        const uint64_t t = ctx->step;
        const bool rec = obs_every > 0 && (t + 1) % (uint64_t)obs_every == 0;
        long long *cur = rec ? ctx->d_rec + (size_t)ctx->n_rec * rec_stride : nullptr;
        // hand-over: the neighbours' edge rows of the current sigma into the arrays, tau row n_rows redrawn from them
        if (!ctx->published) { int rc = slab_publish_now(ctx); if (rc) return rc; }
        SlabParams sp;
        slab_params(ctx, sp, J, q, t);
        sp.redraw = 1;
        slab_edge<<<slab_grid(ctx, ctx->L / 16), SLAB_THREADS, 0, ctx->stream>>>(sp);
        CU(cudaGetLastError());
        cudaError_t e;
        p.src = ctx->d_sigma;
        p.dst = ctx->d_tau;
        p.rec_cur = cur;
        p.rec_prev = pending;
        make_step_keys(ctx->seed, 2 * t, p.keys);
        if (rec && pending) e = launch_half<0, F_OBS | F_BONDS>(ctx, p, grid);
        else if (rec) e = launch_half<0, F_OBS>(ctx, p, grid);
        else if (pending) e = launch_half<0, F_BONDS>(ctx, p, grid);
        else e = launch_half<0, 0>(ctx, p, grid);
        if (e != cudaSuccess) return fail(ctx, SHAKEN_ECUDA, "slab half-step 0 launch: %s", cudaGetErrorString(e));
        pending = nullptr;
        p.src = ctx->d_tau;
        p.dst = ctx->d_sigma;
        p.rec_prev = nullptr;
        make_step_keys(ctx->seed, 2 * t + 1, p.keys);
        if (rec) e = launch_half<1, F_OBS>(ctx, p, grid);
        else e = launch_half<1, 0>(ctx, p, grid);
        if (e != cudaSuccess) return fail(ctx, SHAKEN_ECUDA, "slab half-step 1 launch: %s", cudaGetErrorString(e));
        ctx->launches += 3;
        ctx->step = t + 1;
        ctx->published = false;
        { int rc = slab_publish_now(ctx); if (rc) return rc; }     // the neighbours' next half-step 0 waits for these rows
        if (rec) {
            pending = cur;
            ctx->n_rec++;
        }
    }
    ctx->slab_pending = pending;                        // closed by the next run or by shaken_observables
    return SHAKEN_OK;
}

static int run_impl(shaken_ctx *ctx, const double *J, const double *q, bool uniform, int64_t n_steps, int64_t obs_every)
{
    if (n_steps < 0 || obs_every < 0) return fail(ctx, SHAKEN_EINVAL, "shaken_run: negative count");
    const int nJ = uniform ? 1 : ctx->n_chains;
    for (int i = 0; i < nJ; ++i)
        if (!isfinite(J[i]) || !isfinite(q[i])) return fail(ctx, SHAKEN_EINVAL, "shaken_run: non-finite coupling for chain %d", i);
    if (!ctx->have_sigma || !ctx->d_sigma) return fail(ctx, SHAKEN_ESTATE, "shaken_run: no sigma yet (call shaken_init, shaken_set_spins or shaken_adopt_spins)");
    int rc = ensure_device(ctx);
    if (rc) return rc;
    if (n_steps == 0) return SHAKEN_OK;

    // records this run appends
    int64_t n_new = 0;
    if (obs_every > 0) n_new = (int64_t)((ctx->step + (uint64_t)n_steps) / (uint64_t)obs_every - ctx->step / (uint64_t)obs_every);
    if (n_new > 0) {
        rc = grow_records(ctx, ctx->n_rec + n_new);
        if (rc) return rc;
    }
    if (ctx->slab) return run_slab(ctx, J[0], q[0], n_steps, obs_every);

    StepParams p;
    memset(&p, 0, sizeof(p));
    p.L = ctx->L;
    p.nvec = ctx->packed ? ctx->L / 32 : ctx->L / 16;
    p.n_chains = ctx->n_chains;
    p.chain0 = ctx->chain0;
    p.group = ctx->group;
    p.nseg = (p.nvec + 31) / 32;
    const int resident = 1;                                   // resident blocks per SM (launch bounds)
    int wpb = ctx->packed ? PK_THREADS / 32 : I8_THREADS / 32;   // warps per block
    const long long cap = (long long)ctx->num_sms * resident;
    double score_block = 0.0;
    p.rows_per_task = choose_rows_per_task(ctx, p.nseg, cap, wpb, &score_block);
    p.nrb = (ctx->L + p.rows_per_task - 1) / p.rows_per_task;
    // block tasks: wpb consecutive warp strips of one chain
    p.ntasks = (long long)ctx->n_chains * (((long long)p.nrb * p.nseg + wpb - 1) / wpb);
    // many small chains: per-warp task lists (kernel_i8.cuh PERWARP).  Every warp gets a RANGE of the same number of
    // consecutive strip-rows (a strip-row = one row of one 32-vector column strip of one chain), so the launch is one full
    // wave whatever the chain size; a range is walked piece by piece, each piece paying the halo row and the two
    // unprefetched rows of a strip start.
    ctx->perwarp = false;
    if (!ctx->packed && (ctx->variant == SHAKEN_VARIANT_PERWARP || ctx->n_chains > 1)) {
        const long long S = (long long)ctx->n_chains * p.nseg * ctx->L;              // strip-rows per launch
        const long long warps = cap * wpb;
        long long waves = (S + warps * MAX_ROWS_PER_TASK - 1) / (warps * MAX_ROWS_PER_TASK);
        long long n_ranges = warps * waves;
        if (n_ranges > S) n_ranges = S;
        const long long len = (S + n_ranges - 1) / n_ranges;
        n_ranges = (S + len - 1) / len;
        const long long waves_r = (n_ranges + warps - 1) / warps;
        const double fill = (double)S / (double)(waves_r * warps * len);
        const double pieces = 1.0 + (double)len / (double)ctx->L;                     // strip starts per range, on average
        const double score_pw = fill * (double)len / ((double)len + 3.0 * pieces);
        // (launches with sums: block tasks keep their index bytes off the multiplier pipe, per-warp lists cannot: about 3 %)
        const bool mostly_plain = obs_every == 0 || obs_every > 4;
        if (ctx->variant == SHAKEN_VARIANT_PERWARP || score_pw * (mostly_plain ? 1.0 : 0.97) > score_block + 0.02) {
            ctx->perwarp = true;
            p.rows_total = S;
            p.range_len = (int)len;
            p.ntasks = n_ranges;
        }
    }

    if (uniform) {
        kernel_table(J[0], q[0], p.utab);
        p.gtab = nullptr;
    } else {
        if (!ctx->d_tab && cudaMalloc(&ctx->d_tab, (size_t)ctx->n_chains * 8 * sizeof(uint32_t)) != cudaSuccess) {
            cudaGetLastError();
            return fail(ctx, SHAKEN_ENOMEM, "cudaMalloc of the threshold tables failed");
        }
        std::vector<uint32_t> h((size_t)ctx->n_chains * 8);
        for (int i = 0; i < ctx->n_chains; ++i) kernel_table(J[i], q[i], &h[(size_t)i * 8]);
        // pageable source: the copy is staged before the call returns, so h may go out of scope
        CU(cudaMemcpyAsync(ctx->d_tab, h.data(), h.size() * sizeof(uint32_t), cudaMemcpyHostToDevice, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        p.gtab = ctx->d_tab;
    }

    // small-lattice path: one CTA per chain keeps both sublattices in shared memory for the whole run
    // (also mid-size chains, L <= 288, when there are enough of them to fill the machine: the strip kernels would leave
    // most lanes of a warp idle on rows narrower than 512 spins, and the band path is for few chains)
    const bool small_path = !ctx->packed && ctx->variant == 0 && ctx->group <= SMALL_GROUP_MAX &&
                            small_smem_bytes(ctx->L, ctx->group) <= 200 * 1024 &&
                            (ctx->L <= SMALL_L_MAX || (ctx->L <= SMALL_L_BATCH_MAX && 2 * (ctx->n_chains / ctx->group) >= ctx->num_sms));
    // A few small chains: one chain per CLUSTER of 8 SMs (kernel_cluster.cuh) instead of one per SM -- rows in the shared
    // memory of 8 CTAs, the neighbours' rows read through distributed shared memory, one cluster barrier per full step.
    // Which of the two is faster was measured at L = 32, 64, 128 for 19 ... 1024 chains: the cluster kernel (one word per thread:
    // short latency, less instruction-level parallelism) wins while the machine is not full -- up to about 110 / 95 / 58 chains
    // with records on every step, 80 / 74 / 30 without -- e.g. 37 chains of 64^2: 1.17 against 2.10 us per step.
    const int cluster_max_chains = max(ctx->num_sms / CLUSTER_CTAS, (obs_every == 1 || obs_every == 2 ? 128 : 100) - (9 * ctx->L) / 16);
    const bool cluster_path = small_path && ctx->group == 1 && ctx->L >= 32 && ctx->L <= SMALL_L_MAX && !ctx->no_cluster &&
                              ctx->n_chains <= cluster_max_chains;
    if (cluster_path) {
        SmallParams sp;
        memset(&sp, 0, sizeof(sp));
        sp.sigma = (uint8_t *)ctx->d_sigma;
        sp.tau = (uint8_t *)ctx->d_tau;
        sp.L = ctx->L;
        sp.n_chains = ctx->n_chains;
        sp.group = 1;
        sp.chain0 = ctx->chain0;
        sp.t0 = ctx->step;
        sp.n_steps = n_steps;
        sp.obs_every = obs_every;
        sp.rec = ctx->d_rec ? ctx->d_rec + (size_t)ctx->n_rec * ctx->n_chains * SHAKEN_N_OBS : nullptr;
        sp.gtab = p.gtab;
        memcpy(sp.utab, p.utab, sizeof(sp.utab));
        make_step_keys(ctx->seed, 0, sp.keys);
        const int threads = cluster_threads(ctx->L);
        cudaLaunchConfig_t cfg;
        memset(&cfg, 0, sizeof(cfg));
        cfg.gridDim = dim3((unsigned)(ctx->n_chains * CLUSTER_CTAS));
        cfg.blockDim = dim3((unsigned)threads);
        cfg.dynamicSmemBytes = cluster_smem_bytes(ctx->L);
        cfg.stream = ctx->stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = CLUSTER_CTAS;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        const cudaError_t le = cudaLaunchKernelEx(&cfg, cluster_run_i8, sp);
        if (le == cudaSuccess) {
            ctx->launches++;
            ctx->step += (uint64_t)n_steps;
            ctx->n_rec += n_new;
            ctx->have_tau = true;
            return SHAKEN_OK;
        }
        cudaGetLastError();
        ctx->no_cluster = true;                   // (a device or partition that cannot co-schedule the cluster: one chain per SM instead)
    }
    if (small_path) {
        SmallParams sp;
        memset(&sp, 0, sizeof(sp));
        sp.sigma = (uint8_t *)ctx->d_sigma;
        sp.tau = (uint8_t *)ctx->d_tau;
        sp.L = ctx->L;
        sp.n_chains = ctx->n_chains;
        sp.group = ctx->group;
        sp.coal = ctx->group > 1 ? ctx->d_coal : nullptr;
        sp.chain0 = ctx->chain0;
        sp.t0 = ctx->step;
        sp.n_steps = n_steps;
        sp.obs_every = obs_every;
        sp.rec = ctx->d_rec ? ctx->d_rec + (size_t)ctx->n_rec * ctx->n_chains * SHAKEN_N_OBS : nullptr;
        sp.gtab = p.gtab;
        memcpy(sp.utab, p.utab, sizeof(sp.utab));
        make_step_keys(ctx->seed, 0, sp.keys);
        const int nvecs = ctx->L * ctx->L / 16;             // one 16-byte vector per thread per trip
        const size_t smem = small_smem_bytes(ctx->L, ctx->group);
        // Block size.  Up to 256 vectors: one per thread.  Beyond: 512 threads, unless two CTAs fit an SM (shared memory) and
        // there are more CTAs than SMs -- then blocks of at most 256 threads, so that two or three resident CTAs hide each
        // other's block barriers (1024 chains of 128^2: 773 -> 840 site-updates/ns, 1600 of 208^2: 863 -> 922), a little
        // smaller where that fills the last trip much better (576 vectors at L = 96: 3 x 192 instead of 2 x 512: 553 -> 681).
        int threads = nvecs <= 256 ? ((nvecs + 31) / 32) * 32 : 512;
        if (nvecs > 256 && 2 * (smem + 2048) <= 220 * 1024 && ctx->n_chains / ctx->group > ctx->num_sms) {
            threads = 256;
            double best = (double)nvecs / (double)(((nvecs + 255) / 256) * 256);
            for (int t = 224; t >= 192; t -= 32) {
                const double eff = (double)nvecs / (double)(((nvecs + t - 1) / t) * t);
                if (eff > best * 1.05) { best = eff; threads = t; }
            }
        }
        if (threads <= 256) {
            if (smem > 40 * 1024) CU(cudaFuncSetAttribute(small_run_i8<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            small_run_i8<256><<<ctx->n_chains / ctx->group, threads, smem, ctx->stream>>>(sp);
        } else {
            if (smem > 40 * 1024) CU(cudaFuncSetAttribute(small_run_i8<512>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            small_run_i8<512><<<ctx->n_chains / ctx->group, threads, smem, ctx->stream>>>(sp);
        }
        CU(cudaGetLastError());
        ctx->launches++;
        ctx->step += (uint64_t)n_steps;
        ctx->n_rec += n_new;
        ctx->have_tau = true;
        return SHAKEN_OK;
    }

    // band path: mid-size lattices, few chains -- the whole run in one cooperative launch (kernel_band.cuh)
    {
        const int br = try_band_launch(ctx, false, p.gtab, p.utab, n_steps, obs_every, n_new);
        if (br <= 0) return br;                                       // 0: done, < 0: error, 1: not applicable / refused
    }

    const long long blocks_needed = ctx->perwarp ? (p.ntasks + I8_THREADS / 32 - 1) / (I8_THREADS / 32) : p.ntasks;   // (ranges / warps per block)
    const int grid = (int)(blocks_needed < cap ? blocks_needed : cap);
    const size_t rec_stride = (size_t)ctx->n_chains * SHAKEN_N_OBS;

    ctx->have_tau = true;           // half-step 0 redraws every tau from sigma alone
    // coupled chains: the comparison of a step's sigma rides on the NEXT half-step 0 (which reads exactly that sigma), the
    // bookkeeping on the half-step 1 after it; the last step of the call is closed by a read-only pass
    const bool coupled = ctx->group > 1;
    const long long ng = coupled ? ctx->n_chains / ctx->group : 0;
    p.coal = coupled ? ctx->d_coal : nullptr;
    p.diff = coupled ? reinterpret_cast<unsigned long long *>(ctx->d_coal + ng) : nullptr;
    bool cmp_due = false;           // sigma has changed since it was last compared
    auto half0 = [&](int flags) -> cudaError_t {
        switch (flags) {
            case 0: return launch_half<0, 0>(ctx, p, grid);
            case F_OBS: return launch_half<0, F_OBS>(ctx, p, grid);
            case F_BONDS: return launch_half<0, F_BONDS>(ctx, p, grid);
            case F_OBS | F_BONDS: return launch_half<0, F_OBS | F_BONDS>(ctx, p, grid);
            case F_COAL: return launch_half<0, F_COAL>(ctx, p, grid);
            case F_COAL | F_OBS: return launch_half<0, F_COAL | F_OBS>(ctx, p, grid);
            case F_COAL | F_BONDS: return launch_half<0, F_COAL | F_BONDS>(ctx, p, grid);
            case F_COAL | F_OBS | F_BONDS: return launch_half<0, F_COAL | F_OBS | F_BONDS>(ctx, p, grid);
            case F_NOUPDATE | F_BONDS: return launch_half<0, F_NOUPDATE | F_BONDS>(ctx, p, grid);
            case F_NOUPDATE | F_COAL: return launch_half<0, F_NOUPDATE | F_COAL>(ctx, p, grid);
            default: return launch_half<0, F_NOUPDATE | F_COAL | F_BONDS>(ctx, p, grid);
        }
    };
    long long *pending = nullptr;   // record that still lacks C_x, C_y
    for (int64_t s = 0; s < n_steps; ++s) {
        const uint64_t t = ctx->step;
        const bool rec = obs_every > 0 && (t + 1) % (uint64_t)obs_every == 0;
        long long *cur = rec ? ctx->d_rec + (size_t)ctx->n_rec * rec_stride : nullptr;
        cudaError_t e;
        // half-step 0: tau <- sigma  (eq. 15)
        p.src = ctx->d_sigma;
        p.dst = ctx->d_tau;
        p.rec_cur = cur;
        p.rec_prev = pending;
        p.cstamp = p.fin_stamp = (unsigned long long)t;             // sigma as it stands is the state after t steps
        p.do_fin = 0;
        make_step_keys(ctx->seed, 2 * t, p.keys);
        e = half0((rec ? F_OBS : 0) | (pending ? F_BONDS : 0) | (cmp_due ? F_COAL : 0));
        if (e != cudaSuccess) return fail(ctx, SHAKEN_ECUDA, "half-step 0 launch: %s", cudaGetErrorString(e));
        pending = nullptr;
        // half-step 1: sigma <- tau  (eq. 16)
        p.src = ctx->d_tau;
        p.dst = ctx->d_sigma;
        p.rec_prev = nullptr;
        p.do_fin = cmp_due ? 1 : 0;
        make_step_keys(ctx->seed, 2 * t + 1, p.keys);
        if (rec) e = launch_half<1, F_OBS>(ctx, p, grid);
        else e = launch_half<1, 0>(ctx, p, grid);
        if (e != cudaSuccess) return fail(ctx, SHAKEN_ECUDA, "half-step 1 launch: %s", cudaGetErrorString(e));
        ctx->launches += 2;
        ctx->step = t + 1;
        cmp_due = coupled;
        if (rec) {
            pending = cur;
            ctx->n_rec++;
        }
    }
    if (pending || cmp_due) {
        // the last step: its sigma-layer bond sums (if it was recorded) and its comparison (coupled chains) are taken by
        // a read-only pass over sigma
        p.src = ctx->d_sigma;
        p.dst = nullptr;
        p.rec_cur = nullptr;
        p.rec_prev = pending;
        p.cstamp = p.fin_stamp = (unsigned long long)ctx->step;
        p.do_fin = 0;
        cudaError_t e = half0(F_NOUPDATE | (pending ? F_BONDS : 0) | (cmp_due ? F_COAL : 0));
        if (e != cudaSuccess) return fail(ctx, SHAKEN_ECUDA, "closing read-only launch: %s", cudaGetErrorString(e));
        ctx->launches++;
        if (cmp_due) {
            coalesce_finalize<<<grid_for(ctx, ng), 256, 0, ctx->stream>>>(ctx->d_coal, p.diff, ng, (unsigned long long)ctx->step);
            CU(cudaGetLastError());
            ctx->launches++;
        }
    }
    return SHAKEN_OK;
}

extern "C" int shaken_run(shaken_ctx *ctx, double J, double q, int64_t n_steps, int64_t obs_every)
{
    if (!ctx) return fail(nullptr, SHAKEN_EINVAL, "shaken_run: ctx is NULL");
    return run_impl(ctx, &J, &q, true, n_steps, obs_every);
}

extern "C" int shaken_run_grid(shaken_ctx *ctx, const double *J, const double *q, int64_t n_steps, int64_t obs_every)
{
    if (!ctx) return fail(nullptr, SHAKEN_EINVAL, "shaken_run_grid: ctx is NULL");
    if (!J || !q) return fail(ctx, SHAKEN_EINVAL, "shaken_run_grid: J or q is NULL");
    return run_impl(ctx, J, q, false, n_steps, obs_every);
}

// ---------------------------------------------------------------------------------------------------
// alternate (even sites / odd sites) parallel heat bath on the square lattice
// ---------------------------------------------------------------------------------------------------
extern "C" int shaken_alt_thresholds(double J, uint32_t out[5])
{
    if (!out || !isfinite(J)) return fail(nullptr, SHAKEN_EINVAL, "shaken_alt_thresholds: bad argument");
    for (int k = 0; k < 5; ++k) out[k] = threshold_of_field((double)(2 * k - 4) * J);   // h = J * (sum of 4 neighbours)
    return SHAKEN_OK;
}

static int run_alt_impl(shaken_ctx *ctx, const double *J, bool uniform, int64_t n_steps, int64_t obs_every)
{
    if (n_steps < 0 || obs_every < 0) return fail(ctx, SHAKEN_EINVAL, "shaken_run_alternate: negative count");
    const int nJ = uniform ? 1 : ctx->n_chains;
    for (int i = 0; i < nJ; ++i)
        if (!isfinite(J[i])) return fail(ctx, SHAKEN_EINVAL, "shaken_run_alternate: non-finite coupling for chain %d", i);
    if (ctx->slab) return fail(ctx, SHAKEN_ESTATE, "shaken_run_alternate: not available on a slab context");
    if (!ctx->have_sigma || !ctx->d_sigma) return fail(ctx, SHAKEN_ESTATE, "shaken_run_alternate: no sigma yet (call shaken_init, shaken_set_spins or shaken_adopt_spins)");
    int rc = ensure_device(ctx);
    if (rc) return rc;
    if (n_steps == 0) return SHAKEN_OK;
    int64_t n_new = 0;
    if (obs_every > 0) n_new = (int64_t)((ctx->step + (uint64_t)n_steps) / (uint64_t)obs_every - ctx->step / (uint64_t)obs_every);
    if (n_new > 0) {
        rc = grow_records(ctx, ctx->n_rec + n_new);
        if (rc) return rc;
    }

    AltParams p;
    memset(&p, 0, sizeof(p));
    p.sigma = ctx->d_sigma;
    p.L = ctx->L;
    p.nvec = ctx->packed ? ctx->L / 32 : ctx->L / 16;
    p.n_chains = ctx->n_chains;
    p.chain0 = ctx->chain0;
    p.group = ctx->group;
    const bool strips = !ctx->packed && p.nvec >= 32;            // wide int8 rows: alt_strip_i8 walks column strips
    int R;
    if (strips) {
        const int nseg = (p.nvec + 31) / 32;
        // strip height: balance over the resident warps (2 blocks of 8 warps per SM) against the two halo rows per strip
        const double warps = (double)ctx->num_sms * 2 * (ALT_THREADS / 32);
        double best = -1.0;
        R = 2;
        for (int cand = 2; cand <= 256 && cand <= ctx->L; cand *= 2) {
            const double tasks = (double)ctx->n_chains * ((ctx->L + cand - 1) / cand) * nseg;
            const double waves = tasks / warps;
            const double score = (waves < 1.0 ? waves : waves / ceil(waves)) * cand / (cand + 2.0);
            if (score > best) { best = score; R = cand; }
        }
        p.nrb = (ctx->L + R - 1) / R;
        p.ntasks = (long long)ctx->n_chains * p.nrb * nseg;
    } else {
        R = 512 / p.nvec;                                        // about 16 vectors per lane and task
        if (R < 1) R = 1;
        if (R > ctx->L) R = ctx->L;
        p.nrb = (ctx->L + R - 1) / R;
        p.ntasks = (long long)ctx->n_chains * p.nrb;
    }
    p.rows_per_task = R;
    if (uniform) {
        shaken_alt_thresholds(J[0], p.utab);
        p.gtab = nullptr;
    } else {
        if (!ctx->d_tab && cudaMalloc(&ctx->d_tab, (size_t)ctx->n_chains * 8 * sizeof(uint32_t)) != cudaSuccess) {
            cudaGetLastError();
            return fail(ctx, SHAKEN_ENOMEM, "cudaMalloc of the threshold tables failed");
        }
        std::vector<uint32_t> h((size_t)ctx->n_chains * 8, 0u);
        for (int i = 0; i < ctx->n_chains; ++i) shaken_alt_thresholds(J[i], &h[(size_t)i * 8]);
        CU(cudaMemcpyAsync(ctx->d_tab, h.data(), h.size() * sizeof(uint32_t), cudaMemcpyHostToDevice, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        p.gtab = ctx->d_tab;
    }
    // small lattices: one CTA per coupling group, sigma in shared memory, the whole run in one launch
    // (also mid-size chains, L <= 288, when there are enough of them to fill the machine, as in run_impl)
    if (!ctx->packed && ctx->variant == 0 && ctx->group <= SMALL_GROUP_MAX && alt_small_smem_bytes(ctx->L, ctx->group) <= 200 * 1024 &&
        (ctx->L <= SMALL_L_MAX || (ctx->L <= SMALL_L_BATCH_MAX && 2 * (ctx->n_chains / ctx->group) >= ctx->num_sms))) {
        SmallParams sp;
        memset(&sp, 0, sizeof(sp));
        sp.sigma = (uint8_t *)ctx->d_sigma;
        sp.tau = nullptr;
        sp.L = ctx->L;
        sp.n_chains = ctx->n_chains;
        sp.group = ctx->group;
        sp.coal = ctx->group > 1 ? ctx->d_coal : nullptr;
        sp.chain0 = ctx->chain0;
        sp.t0 = ctx->step;
        sp.n_steps = n_steps;
        sp.obs_every = obs_every;
        sp.rec = ctx->d_rec ? ctx->d_rec + (size_t)ctx->n_rec * ctx->n_chains * SHAKEN_N_OBS : nullptr;
        sp.gtab = p.gtab;
        memcpy(sp.utab, p.utab, sizeof(sp.utab));
        make_step_keys(ctx->seed, 0, sp.keys);
        const int nvecs = ctx->L * ctx->L / 16;
        const int threads = nvecs >= 256 ? 256 : ((nvecs + 31) / 32) * 32;
        const size_t smem = alt_small_smem_bytes(ctx->L, ctx->group);
        if (smem > 40 * 1024) CU(cudaFuncSetAttribute(alt_small_i8, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        alt_small_i8<<<ctx->n_chains / ctx->group, threads, smem, ctx->stream>>>(sp);
        CU(cudaGetLastError());
        ctx->launches++;
        ctx->step += (uint64_t)n_steps;
        ctx->n_rec += n_new;
        return SHAKEN_OK;
    }

    // mid-size lattices, few chains: the whole run in one cooperative launch (kernel_alt.cuh: alt_band_i8)
    {
        const int br = try_band_launch(ctx, true, p.gtab, p.utab, n_steps, obs_every, n_new);
        if (br <= 0) return br;
    }

    const int wpb = ALT_THREADS / 32;
    long long blocks = (p.ntasks + wpb - 1) / wpb;
    const long long cap = (long long)ctx->num_sms * (strips ? 2 : 8);
    const int grid = (int)(blocks < cap ? blocks : cap);
    const size_t rec_stride = (size_t)ctx->n_chains * SHAKEN_N_OBS;

    for (int64_t s = 0; s < n_steps; ++s) {
        const uint64_t t = ctx->step;
        const bool rec = obs_every > 0 && (t + 1) % (uint64_t)obs_every == 0;
        p.rec = nullptr;
        cudaError_t le;
        make_step_keys(ctx->seed, 2 * t, p.keys);
        if (ctx->packed) le = launch_pdl(alt_half<0, false, true>, grid, ALT_THREADS, ctx->stream, p);
        else if (strips) le = launch_pdl(alt_strip_i8<0, false>, grid, ALT_THREADS, ctx->stream, p);
        else le = launch_pdl(alt_half<0, false, false>, grid, ALT_THREADS, ctx->stream, p);
        if (le != cudaSuccess) return fail(ctx, SHAKEN_ECUDA, "alternate half-step 0 launch: %s", cudaGetErrorString(le));
        make_step_keys(ctx->seed, 2 * t + 1, p.keys);
        if (rec) {
            p.rec = ctx->d_rec + (size_t)ctx->n_rec * rec_stride;
            if (ctx->packed) le = launch_pdl(alt_half<1, true, true>, grid, ALT_THREADS, ctx->stream, p);
            else if (strips) le = launch_pdl(alt_strip_i8<1, true>, grid, ALT_THREADS, ctx->stream, p);
            else le = launch_pdl(alt_half<1, true, false>, grid, ALT_THREADS, ctx->stream, p);
            ctx->n_rec++;
        } else {
            if (ctx->packed) le = launch_pdl(alt_half<1, false, true>, grid, ALT_THREADS, ctx->stream, p);
            else if (strips) le = launch_pdl(alt_strip_i8<1, false>, grid, ALT_THREADS, ctx->stream, p);
            else le = launch_pdl(alt_half<1, false, false>, grid, ALT_THREADS, ctx->stream, p);
        }
        if (le != cudaSuccess) return fail(ctx, SHAKEN_ECUDA, "alternate half-step 1 launch: %s", cudaGetErrorString(le));
        CU(cudaGetLastError());
        ctx->launches += 2;
        ctx->step = t + 1;
        if (ctx->group > 1) {
            const long long ng = ctx->n_chains / ctx->group;
            const long long vpc = (long long)(shaken_spin_bytes(ctx) / 16) / ctx->n_chains;
            unsigned long long *diff = reinterpret_cast<unsigned long long *>(ctx->d_coal + ng);
            coalesce_compare<<<grid_for(ctx, ng * (ctx->group - 1) * vpc), 256, 0, ctx->stream>>>((const uint4 *)ctx->d_sigma, vpc, ctx->group, ng, ctx->d_coal, diff, (unsigned long long)ctx->step);
            coalesce_finalize<<<grid_for(ctx, ng), 256, 0, ctx->stream>>>(ctx->d_coal, diff, ng, (unsigned long long)ctx->step);
            CU(cudaGetLastError());
            ctx->launches += 2;
        }
    }
    return SHAKEN_OK;
}

extern "C" int shaken_run_alternate(shaken_ctx *ctx, double J, int64_t n_steps, int64_t obs_every)
{
    if (!ctx) return fail(nullptr, SHAKEN_EINVAL, "shaken_run_alternate: ctx is NULL");
    return run_alt_impl(ctx, &J, true, n_steps, obs_every);
}

extern "C" int shaken_run_alternate_grid(shaken_ctx *ctx, const double *J, int64_t n_steps, int64_t obs_every)
{
    if (!ctx) return fail(nullptr, SHAKEN_EINVAL, "shaken_run_alternate_grid: ctx is NULL");
    if (!J) return fail(ctx, SHAKEN_EINVAL, "shaken_run_alternate_grid: J is NULL");
    return run_alt_impl(ctx, J, false, n_steps, obs_every);
}

// ---------------------------------------------------------------------------------------------------
// (a9) records and state I/O
// ---------------------------------------------------------------------------------------------------
extern "C" int64_t shaken_observables(shaken_ctx *ctx, int64_t *out, int64_t max_records)
{
    if (!ctx || max_records < 0) return fail(ctx, SHAKEN_EINVAL, "shaken_observables: bad argument");
    if (ctx->slab && ctx->slab_pending) {
        const int rc = slab_close_record(ctx);
        if (rc) return rc;
    }
    const int64_t n = ctx->n_rec < max_records ? ctx->n_rec : max_records;
    if (n > 0) {
        if (!out) return fail(ctx, SHAKEN_EINVAL, "shaken_observables: out is NULL");
        cudaError_t e = cudaMemcpyAsync(out, ctx->d_rec, (size_t)n * shaken_record_bytes(ctx), cudaMemcpyDeviceToHost, ctx->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
        if (e != cudaSuccess) return fail(ctx, SHAKEN_ECUDA, "shaken_observables: %s", cudaGetErrorString(e));
    } else {
        cudaError_t e = cudaStreamSynchronize(ctx->stream);
        if (e != cudaSuccess) return fail(ctx, SHAKEN_ECUDA, "shaken_observables: %s", cudaGetErrorString(e));
    }
    return n;
}

static int ensure_stage(shaken_ctx *ctx, size_t bytes)
{
    if (ctx->stage_bytes >= bytes) return SHAKEN_OK;
    cudaFree(ctx->d_stage);
    ctx->d_stage = nullptr;
    ctx->stage_bytes = 0;
    if (cudaMalloc(&ctx->d_stage, bytes) != cudaSuccess) {
        cudaGetLastError();
        return fail(ctx, SHAKEN_ENOMEM, "cudaMalloc of %zu staging bytes failed", bytes);
    }
    ctx->stage_bytes = bytes;
    return SHAKEN_OK;
}

static const size_t STAGE_SITES = (size_t)64 << 20;   // conversion chunk: 64 Mi spins

extern "C" int shaken_get_spins(shaken_ctx *ctx, int which, int8_t *host)
{
    if (!ctx || !host || (which != 0 && which != 1)) return fail(ctx, SHAKEN_EINVAL, "shaken_get_spins: bad argument");
    if (!(which ? ctx->have_tau : ctx->have_sigma) || !ctx->d_sigma)
        return fail(ctx, SHAKEN_ESTATE, "shaken_get_spins: %s has no defined content yet", which ? "tau" : "sigma");
    const size_t n = ctx->slab ? shaken_spin_bytes(ctx) : (size_t)ctx->n_chains * ctx->L * ctx->L;
    const void *src = which ? ctx->d_tau : ctx->d_sigma;
    if (!ctx->packed) {
        CU(cudaMemcpyAsync(host, src, n, cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        return SHAKEN_OK;
    }
    const size_t chunk = n < STAGE_SITES ? n : STAGE_SITES;
    int rc = ensure_stage(ctx, chunk);
    if (rc) return rc;
    for (size_t off = 0; off < n; off += chunk) {
        const size_t m = n - off < chunk ? n - off : chunk;
        unpack_words<<<grid_for(ctx, (long long)(m / 32)), 256, 0, ctx->stream>>>((const uint32_t *)src + off / 32, (uint8_t *)ctx->d_stage, (long long)(m / 32));
        ctx->launches++;
        CU(cudaGetLastError());
        CU(cudaMemcpyAsync(host + off, ctx->d_stage, m, cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
    }
    return SHAKEN_OK;
}

extern "C" int shaken_set_spins(shaken_ctx *ctx, int which, const int8_t *host)
{
    if (!ctx || !host || (which != 0 && which != 1)) return fail(ctx, SHAKEN_EINVAL, "shaken_set_spins: bad argument");
    int rc = ensure_spins(ctx);
    if (rc) return rc;
    const size_t n = ctx->slab ? shaken_spin_bytes(ctx) : (size_t)ctx->n_chains * ctx->L * ctx->L;
    void *dst = which ? ctx->d_tau : ctx->d_sigma;
    if (which == 0) {
        if (ctx->slab && ctx->slab_pending) {            // the last record's C_x, C_y are sums over the sigma about to be replaced
            rc = slab_close_record(ctx);
            if (rc) return rc;
        }
        ctx->published = false;
    }
    CU(cudaMemsetAsync(ctx->d_bad, 0, sizeof(unsigned long long), ctx->stream));
    if (!ctx->packed) {
        CU(cudaMemcpyAsync(dst, host, n, cudaMemcpyHostToDevice, ctx->stream));
        validate_bytes<<<grid_for(ctx, (long long)(n / 16)), 256, 0, ctx->stream>>>((const uint8_t *)dst, (long long)(n / 16), ctx->d_bad);
        ctx->launches++;
        CU(cudaGetLastError());
    } else {
        const size_t chunk = n < STAGE_SITES ? n : STAGE_SITES;
        rc = ensure_stage(ctx, chunk);
        if (rc) return rc;
        for (size_t off = 0; off < n; off += chunk) {
            const size_t m = n - off < chunk ? n - off : chunk;
            CU(cudaMemcpyAsync(ctx->d_stage, host + off, m, cudaMemcpyHostToDevice, ctx->stream));
            pack_words<<<grid_for(ctx, (long long)(m / 32)), 256, 0, ctx->stream>>>((const uint8_t *)ctx->d_stage, (uint32_t *)dst + off / 32, (long long)(m / 32), ctx->d_bad);
            ctx->launches++;
            CU(cudaGetLastError());
            CU(cudaStreamSynchronize(ctx->stream));   // the staging buffer is reused by the next chunk
        }
    }
    unsigned long long bad = 0;
    CU(cudaMemcpyAsync(&bad, ctx->d_bad, sizeof(bad), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    (which ? ctx->have_tau : ctx->have_sigma) = bad == 0;
    if (bad) return fail(ctx, SHAKEN_EINVAL, "shaken_set_spins: %llu values are neither +1 nor -1 (sublattice content is now unspecified)", bad);
    return SHAKEN_OK;
}

extern "C" int shaken_adopt_spins(shaken_ctx *ctx)
{
    if (!ctx) return fail(nullptr, SHAKEN_EINVAL, "shaken_adopt_spins: ctx is NULL");
    if (!ctx->d_sigma || !ctx->d_tau) return fail(ctx, SHAKEN_ESTATE, "shaken_adopt_spins: no buffers (call shaken_bind first)");
    int rc = ensure_device(ctx);
    if (rc) return rc;
    unsigned long long bad = 0;
    if (!ctx->packed) {   // every bit pattern is a valid packed word; int8 layers must hold 0x01 / 0xFF only
        const long long nvec = (long long)(shaken_spin_bytes(ctx) / 16);
        CU(cudaMemsetAsync(ctx->d_bad, 0, sizeof(unsigned long long), ctx->stream));
        validate_bytes<<<grid_for(ctx, nvec), 256, 0, ctx->stream>>>((const uint8_t *)ctx->d_sigma, nvec, ctx->d_bad);
        validate_bytes<<<grid_for(ctx, nvec), 256, 0, ctx->stream>>>((const uint8_t *)ctx->d_tau, nvec, ctx->d_bad);
        ctx->launches += 2;
        CU(cudaGetLastError());
        CU(cudaMemcpyAsync(&bad, ctx->d_bad, sizeof(bad), cudaMemcpyDeviceToHost, ctx->stream));
    }
    CU(cudaStreamSynchronize(ctx->stream));
    if (bad) return fail(ctx, SHAKEN_EINVAL, "shaken_adopt_spins: %llu bytes of the bound buffers are neither +1 nor -1", bad);
    ctx->have_sigma = ctx->have_tau = true;
    return SHAKEN_OK;
}

// ---------------------------------------------------------------------------------------------------
// diagonal correlations
// ---------------------------------------------------------------------------------------------------
extern "C" int shaken_diag_correlations(shaken_ctx *ctx, const int32_t *ells, int32_t n_ell, int64_t *out)
{
    if (!ctx || !ells || !out || n_ell < 1) return fail(ctx, SHAKEN_EINVAL, "shaken_diag_correlations: bad argument");
    if (ctx->slab) return fail(ctx, SHAKEN_ESTATE, "shaken_diag_correlations: not available on a slab context");
    if (!ctx->have_sigma || !ctx->d_sigma) return fail(ctx, SHAKEN_ESTATE, "shaken_diag_correlations: no sigma yet");
    for (int e = 0; e < n_ell; ++e)
        if (ells[e] < 0) return fail(ctx, SHAKEN_EINVAL, "shaken_diag_correlations: negative distance");
    int rc = ensure_device(ctx);
    if (rc) return rc;
    const size_t n = (size_t)ctx->n_chains * (size_t)n_ell * 2;
    long long *d = nullptr;
    if (cudaMalloc(&d, n * sizeof(long long)) != cudaSuccess) {
        cudaGetLastError();
        return fail(ctx, SHAKEN_ENOMEM, "cudaMalloc of %zu correlation sums failed", n);
    }
    cudaError_t err = cudaMemsetAsync(d, 0, n * sizeof(long long), ctx->stream);
    const int W = ctx->packed ? ctx->L / 32 : ctx->L / 4;
    long long bpc = ((long long)ctx->L * W + 255) / 256;
    const long long cap = (long long)ctx->num_sms * 8 / ctx->n_chains + 1;
    if (bpc > cap) bpc = cap;
    const dim3 grid((unsigned)bpc, (unsigned)(ctx->n_chains < 65535 ? ctx->n_chains : 65535));   // chains beyond gridDim.y: looped in the kernel
    for (int e = 0; e < n_ell && err == cudaSuccess; ++e) {
        const int l = ells[e] % ctx->L;
        if (ctx->packed) diag_corr<true><<<grid, 256, 0, ctx->stream>>>((const uint32_t *)ctx->d_sigma, ctx->L, ctx->n_chains, l, d, n_ell, e);
        else diag_corr<false><<<grid, 256, 0, ctx->stream>>>((const uint32_t *)ctx->d_sigma, ctx->L, ctx->n_chains, l, d, n_ell, e);
        ctx->launches++;
        err = cudaGetLastError();
    }
    if (err == cudaSuccess) err = cudaMemcpyAsync(out, d, n * sizeof(long long), cudaMemcpyDeviceToHost, ctx->stream);
    if (err == cudaSuccess) err = cudaStreamSynchronize(ctx->stream);
    cudaFree(d);
    if (err != cudaSuccess) return fail(ctx, SHAKEN_ECUDA, "shaken_diag_correlations: %s", cudaGetErrorString(err));
    return SHAKEN_OK;
}

// ---------------------------------------------------------------------------------------------------
// (a9) derived statistics of the recorded magnetisation, exact integer power sums
// ---------------------------------------------------------------------------------------------------
namespace {
// 256-bit unsigned integer, just enough for sums of M^4 (|M| <= 2^32) and products of two 128-bit sums
struct U256 {
    unsigned long long w[4] = {0, 0, 0, 0};   // little endian
    void add(const U256 &o)
    {
        unsigned __int128 c = 0;
        for (int i = 0; i < 4; ++i) { c += (unsigned __int128)w[i] + o.w[i]; w[i] = (unsigned long long)c; c >>= 64; }
    }
    bool sub(const U256 &o)                    // *this -= o; returns true if the result wrapped (o was larger)
    {
        __int128 b = 0;
        for (int i = 0; i < 4; ++i) { b += (__int128)w[i] - (__int128)o.w[i]; w[i] = (unsigned long long)b; b >>= 64; }
        return b != 0;
    }
    static U256 mul(unsigned __int128 a, unsigned __int128 b)
    {
        const unsigned long long x[2] = {(unsigned long long)a, (unsigned long long)(a >> 64)}, y[2] = {(unsigned long long)b, (unsigned long long)(b >> 64)};
        U256 r;
        for (int i = 0; i < 2; ++i) {
            unsigned __int128 c = 0;
            for (int j = 0; j < 2; ++j) { c += (unsigned __int128)x[i] * y[j] + r.w[i + j]; r.w[i + j] = (unsigned long long)c; c >>= 64; }
            r.w[i + 2] += (unsigned long long)c;
        }
        return r;
    }
    U256 times(unsigned long long k) const
    {
        U256 r;
        unsigned __int128 c = 0;
        for (int i = 0; i < 4; ++i) { c += (unsigned __int128)w[i] * k; r.w[i] = (unsigned long long)c; c >>= 64; }
        return r;
    }
    bool less(const U256 &o) const
    {
        for (int i = 3; i >= 0; --i) if (w[i] != o.w[i]) return w[i] < o.w[i];
        return false;
    }
    long double ld() const { return (((long double)w[3] * 18446744073709551616.0L + (long double)w[2]) * 18446744073709551616.0L + (long double)w[1]) * 18446744073709551616.0L + (long double)w[0]; }
};
}   // namespace

extern "C" int shaken_moments(const int64_t *M, int64_t n, int64_t stride, int64_t n_sites, double out[SHAKEN_N_MOMENTS])
{
    if (!M || !out || n < 1 || n >= (1ll << 31) || stride < 1 || n_sites < 1 || n_sites > (1ll << 32))
        return fail(nullptr, SHAKEN_EINVAL, "shaken_moments: bad argument");
    unsigned __int128 S2 = 0, Sa = 0;
    __int128 S1 = 0;
    U256 S4;
    for (int64_t i = 0; i < n; ++i) {
        const int64_t v = M[i * stride];
        const unsigned long long a = v < 0 ? 0ull - (unsigned long long)v : (unsigned long long)v;
        if (a > (unsigned long long)n_sites) return fail(nullptr, SHAKEN_EINVAL, "shaken_moments: |M| = %llu exceeds n_sites", a);
        const unsigned __int128 sq = (unsigned __int128)a * a;
        S1 += v;
        Sa += a;
        S2 += sq;
        S4.add(U256::mul(sq, sq));
    }
    const long double N = (long double)n_sites, dn = (long double)n;
    out[0] = (double)((long double)S1 / (dn * N));                     // <m>
    out[1] = (double)((long double)Sa / (dn * N));                     // <|m|>
    out[2] = (double)((long double)S2 / (dn * N * N));                 // <m^2>
    out[3] = (double)(S4.ld() / (dn * N * N * N * N));                 // <m^4>
    // Var m = (n S2 - S1^2) / (n^2 N^2): the difference is taken exactly (both terms < 2^127 for n < 2^31)
    const unsigned __int128 a1 = S1 < 0 ? (unsigned __int128)(-S1) : (unsigned __int128)S1;
    out[4] = (double)((long double)((unsigned __int128)n * S2 - a1 * a1) / (dn * dn * N * N));
    // Binder U = 1 - n S4 / (3 S2^2) = (3 S2^2 - n S4) / (3 S2^2), numerator exact in 256 bits
    if (S2 == 0) out[5] = NAN;
    else {
        U256 den = U256::mul(S2, S2).times(3ull), num = den;
        const U256 nS4 = S4.times((unsigned long long)n);
        if (den.less(nS4)) { U256 t = nS4; t.sub(den); out[5] = -(double)(t.ld() / den.ld()); }
        else { num.sub(nS4); out[5] = (double)(num.ld() / den.ld()); }
    }
    return SHAKEN_OK;
}

// ---------------------------------------------------------------------------------------------------
// measurement hook: the Philox-only ceiling (kernels.cuh: philox_rate)
// ---------------------------------------------------------------------------------------------------
extern "C" int shaken_selftest_philox_rate(int32_t blocks_per_sm, int32_t iters, int32_t reps, double *sites_per_ns)
{
    shaken_ctx *ctx = nullptr;
    if (!sites_per_ns || blocks_per_sm < 1 || blocks_per_sm > 8 || iters < 1 || iters > (1 << 20) || reps < 1)
        return fail(nullptr, SHAKEN_EINVAL, "shaken_selftest_philox_rate: bad argument");
    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if ((double)sms * blocks_per_sm * 256.0 * 4.0 * iters >= 4294967296.0)
        return fail(nullptr, SHAKEN_EINVAL, "shaken_selftest_philox_rate: counter range exceeds 2^32");
    StepKeys K;
    make_step_keys(3, 12345, K);
    uint32_t *d = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaError_t e = cudaMalloc(&d, 64);
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    double best = 0.0;
    for (int r = 0; r <= reps && e == cudaSuccess; ++r) {      // r = 0 warms up
        cudaEventRecord(e0, 0);
        philox_rate<<<sms * blocks_per_sm, 256>>>(d, K, iters);
        cudaEventRecord(e1, 0);
        e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        const double rate = (double)sms * blocks_per_sm * 256.0 * 16.0 * iters / ((double)ms * 1e6);
        if (r > 0 && e == cudaSuccess && rate > best) best = rate;
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(d);
    if (e != cudaSuccess) return fail(ctx, SHAKEN_ECUDA, "shaken_selftest_philox_rate: %s", cudaGetErrorString(e));
    *sites_per_ns = best;
    return SHAKEN_OK;
}

// ---------------------------------------------------------------------------------------------------
// test hook
// ---------------------------------------------------------------------------------------------------
extern "C" int shaken_test_band_hook(shaken_ctx *ctx, int what, uint32_t value)
{
    if (!ctx) return fail(nullptr, SHAKEN_EINVAL, "shaken_test_band_hook: ctx is NULL");
    if (what == 0) ctx->xch_stamp = value;              // next band launch starts its stamps here (wrap handling)
    else if (what == 1) ctx->band_refuse_next = value != 0;   // next cooperative launch counts as refused
    else if (what == 2) ctx->no_flow = value != 0;            // bands of <= 7 rows: two-phase kernel instead of the data-flow one
    else return fail(ctx, SHAKEN_EINVAL, "shaken_test_band_hook: unknown selector %d", what);
    return SHAKEN_OK;
}

extern "C" int shaken_philox_words(const uint32_t *ctr, const uint32_t *key, uint32_t *out, int64_t n)
{
    shaken_ctx *ctx = nullptr;
    if (!ctr || !key || !out || n < 0) return fail(nullptr, SHAKEN_EINVAL, "shaken_philox_words: bad argument");
    if (n == 0) return SHAKEN_OK;
    uint32_t *dc = nullptr, *dk = nullptr, *dout = nullptr;
    cudaError_t e = cudaMalloc(&dc, (size_t)n * 16);
    if (e == cudaSuccess) e = cudaMalloc(&dk, (size_t)n * 8);
    if (e == cudaSuccess) e = cudaMalloc(&dout, (size_t)n * 16);
    if (e == cudaSuccess) e = cudaMemcpy(dc, ctr, (size_t)n * 16, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(dk, key, (size_t)n * 8, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        long long blocks = (n + 255) / 256;
        if (blocks > 4096) blocks = 4096;
        philox_hook<<<(int)blocks, 256>>>(dc, dk, dout, (long long)n);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(out, dout, (size_t)n * 16, cudaMemcpyDeviceToHost);
    cudaFree(dc);
    cudaFree(dk);
    cudaFree(dout);
    if (e != cudaSuccess) return fail(ctx, SHAKEN_ECUDA, "shaken_philox_words: %s", cudaGetErrorString(e));
    return SHAKEN_OK;
}

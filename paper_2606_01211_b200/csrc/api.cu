// api.cu -- the C ABI of include/lwe.h: argument validation, context and workspace
// management, and stream-ordered dispatch to the kernels.  No arithmetic of the method
// happens on the host.
#include <new>
#include <string.h>

#include "lwe_internal.cuh"

using namespace lwe;

#include <nvtx3/nvToolsExt.h>

// NVTX range around every entry point (the paper's own tooling: Nsight Systems timelines with NVTX).
// Header-only NVTX3: without a tool attached a push / pop is one load and a branch.
struct NvtxScope {
    explicit NvtxScope(const char *name) { nvtxRangePushA(name); }
    ~NvtxScope() { nvtxRangePop(); }
};

struct lwe_ctx {
    Ctx c;
};

namespace lwe {

cudaError_t kernel_prepare(Ctx *c, const void *fn, size_t smem, int threads, int *occ)
{
    KernelCfg *k = nullptr;
    for (int i = 0; i < c->n_kcfg; i++)
        if (c->kcfg[i].fn == fn) { k = &c->kcfg[i]; break; }
    if (!k) {
        // first launch of this function by this context: opt in on the context's device
        cudaFuncAttributes fa;
        cudaError_t err = cudaFuncGetAttributes(&fa, fn);
        if (err != cudaSuccess) return err;
        const int limit = c->smem_optin - (int)fa.sharedSizeBytes;
        if (limit > 48 * 1024) {
            err = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, limit);
            if (err != cudaSuccess) return err;
        }
        // kernels that need a large dynamic shared memory are launched with the SM's maximal shared-memory carve-out:
        // the driver's default sized the generator kernels (2 x 64 KB per SM wanted) for ONE resident CTA (ncu:
        // launch__occupancy_limit_shared_mem = 1)
        // (decided by the first launch's request: every kernel here asks for the same order of dynamic shared memory on
        // all its launches; the small-smem streaming kernels keep the default carve-out and their L1)
        if (smem > 48 * 1024)
            cudaFuncSetAttribute(fn, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
        if ((int)smem > limit && (int)smem > 48 * 1024) return cudaErrorInvalidValue;
        if (c->n_kcfg >= kMaxKernelCfg) {
            // table full (more distinct kernels than kMaxKernelCfg: raise it): the function is configured, only the
            // cache is missing -- answer an occupancy question with an uncached query instead of failing
            if (occ) {
                int q = 0;
                err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&q, fn, threads, smem);
                if (err != cudaSuccess) return err;
                *occ = q < 1 ? 1 : q;
            }
            return cudaSuccess;
        }
        k = &c->kcfg[c->n_kcfg++];
        k->fn = fn;
        k->occ_threads = 0;
        k->occ_smem = 0;
        k->occ = 0;
    }
    if (occ) {
        if (!k->occ || k->occ_threads != threads || k->occ_smem != smem) {
            int q = 0;
            cudaError_t err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&q, fn, threads, smem);
            if (err != cudaSuccess) return err;
            k->occ = q < 1 ? 1 : q;
            k->occ_threads = threads;
            k->occ_smem = smem;
        }
        *occ = k->occ;
    }
    return cudaSuccess;
}

}  // namespace lwe

namespace {

bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

bool is_pow2(uint32_t x) { return x && !(x & (x - 1)); }

ModQ make_modq(uint32_t q)
{
    ModQ mq;
    mq.q = q;
    mq.mu = (uint32_t)((1ull << 32) / q);
    mq.T = q * (65536u / q);
    mq.half = q / 2;
    mq.pow2 = is_pow2(q) ? 1u : 0u;
    mq.mask = q - 1;
    mq.two32 = (uint32_t)((1ull << 32) % q);
    return mq;
}

template <class T>
cudaError_t dev_alloc(T **p, size_t count)
{
    return cudaMalloc(reinterpret_cast<void **>(p), count * sizeof(T) ? count * sizeof(T) : 16);
}

void free_all(Ctx *c)
{
    cudaFree(c->d_A16); cudaFree(c->d_exc_col_cnt); cudaFree(c->d_exc_col_rows); cudaFree(c->d_exc_row_cnt);
    cudaFree(c->d_exc_row_cols); cudaFree(c->d_exc_overflow);
    if (c->h_exc_overflow) cudaFreeHost(c->h_exc_overflow);
    cudaFree(c->d_Sx);
    cudaFree(c->d_Apanel);
    cudaFree(c->d_foflags); cudaFree(c->d_vprime); cudaFree(c->d_tile_locks);
    cudaFree(c->d_te0); cudaFree(c->d_Rexp); cudaFree(c->d_vacc); cudaFree(c->d_dacc); cudaFree(c->d_counters);
    cudaFree(c->d_hs); cudaFree(c->d_he); cudaFree(c->d_hb); cudaFree(c->d_hU); cudaFree(c->d_hv);
    cudaFree(c->d_hR); cudaFree(c->d_hmu); cudaFree(c->d_hmuout);
    if (c->s_in) cudaStreamDestroy(c->s_in);
    if (c->s_out) cudaStreamDestroy(c->s_out);
    if (c->ev_entry) cudaEventDestroy(c->ev_entry);
    if (c->ev_out) cudaEventDestroy(c->ev_out);
    if (c->ev_se) cudaEventDestroy(c->ev_se);
    if (c->ev_kg) cudaEventDestroy(c->ev_kg);
    for (int i = 0; i < kHostChunks; i++) {
        if (c->ev_in[i]) cudaEventDestroy(c->ev_in[i]);
        if (c->ev_done[i]) cudaEventDestroy(c->ev_done[i]);
    }
    if (c->ev) {
        for (int i = 0; i < 2 * kMaxProfEvents; i++)
            if (c->ev[i]) cudaEventDestroy(c->ev[i]);
        delete[] c->ev;
        c->ev = nullptr;
    }
    delete[] c->ev_kernel;
    c->ev_kernel = nullptr;
}

struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
        if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// exception-list capacity of a wide context: 4x the expected number of elements >= 2^16 per column (row) of a
// uniform A plus 16, rounded up to a power of two (q = 65537, m = 8192: expected 0.125, capacity 16)
uint32_t exc_capacity(uint32_t len, uint32_t q)
{
    const double mean = (double)len * (double)(q - 65536u) / (double)q;
    uint32_t want = (uint32_t)(4.0 * mean) + 16u, cap = 16u;
    while (cap < want) cap <<= 1;
    return cap;
}

#define CHECK_CTX(ctx) do { if (!(ctx)) return LWE_ERR_NULLPTR; } while (0)
// the uint16 entry points do not exist for a modulus that needs 17 bits, and vice versa
#define REQUIRE_NARROW(ctx) do { if ((ctx)->c.wide) return LWE_ERR_UNSUPPORTED; } while (0)
#define REQUIRE_WIDE(ctx) do { if (!(ctx)->c.wide) return LWE_ERR_UNSUPPORTED; } while (0)
#define REQUIRE_PTR(p) do { if (!(p)) return LWE_ERR_NULLPTR; } while (0)
#define REQUIRE_ALIGNED(p) do { if (!aligned16(p)) return LWE_ERR_ALIGN; } while (0)
#define LAUNCH(c, expr) do { cudaError_t _e = (expr); if (_e != cudaSuccess) { (c)->last_cuda_error = (int)_e; return LWE_ERR_CUDA; } } while (0)

}  // namespace

extern "C" {

const char *lwe_strerror(int code)
{
    switch (code) {
    case LWE_OK: return "ok";
    case LWE_ERR_PARAM: return "invalid parameter";
    case LWE_ERR_ALIGN: return "pointer or offset not aligned as the contract requires";
    case LWE_ERR_NULLPTR: return "required pointer is NULL";
    case LWE_ERR_CUDA: return "CUDA runtime error (see lwe_last_cuda_error)";
    case LWE_ERR_UNSUPPORTED: return "unsupported device or variant";
    default: return "unknown error code";
    }
}

int lwe_create(lwe_ctx **out, const lwe_params *p, int device)
{
    NvtxScope nvtx_("lwe_create");
    if (!out || !p) return LWE_ERR_NULLPTR;
    *out = nullptr;
    if (p->n == 0 || p->m == 0 || p->k == 0 || p->n % 8 || p->m % 8 || p->k % 8) return LWE_ERR_PARAM;
    if (p->q < 2 || p->q > 65536u + 1024u || p->eta < 1 || p->eta > 8 || p->max_batch < 1) return LWE_ERR_PARAM;
    if (p->k > 2048 || p->n > (1u << 20) || p->m > (1u << 20)) return LWE_ERR_PARAM;
    const bool wide = p->q > 65536u;
    if (wide && (p->k > 1024 || p->m > 262144u || p->n > 262144u || exc_capacity(p->m, p->q) > 1024u ||
                 exc_capacity(p->n, p->q) > 1024u))
        return LWE_ERR_UNSUPPORTED;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return LWE_ERR_UNSUPPORTED;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return LWE_ERR_CUDA;
    if (prop.major != 10) return LWE_ERR_UNSUPPORTED;          // sm_100a only: no fallback, no other backend

    DeviceGuard guard(device);
    if (!guard.ok) return LWE_ERR_CUDA;

    lwe_ctx *h = new (std::nothrow) lwe_ctx();
    if (!h) return LWE_ERR_CUDA;
    Ctx *c = &h->c;
    memset(c, 0, sizeof(*c));
    c->p = *p;
    c->mq = make_modq(p->q);
    c->device = device;
    c->sm_count = prop.multiProcessorCount;
    c->smem_optin = (int)prop.sharedMemPerBlockOptin;
    c->wide = wide ? 1u : 0u;

    const size_t B = p->max_batch, n = p->n, m = p->m, k = p->k;
    cudaError_t e = cudaSuccess;
    auto ok = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
    ok(dev_alloc(&c->d_te0, 256));
    ok(dev_alloc(&c->d_Rexp, m * k * B));
    if (keygen_tc_workspace_bytes(*p)) ok(dev_alloc(&c->d_Sx, keygen_tc_workspace_bytes(*p)));
    {
        // row panel of a regenerated A: <= 256 MiB, a multiple of 128 rows (one K block of the GEMM), >= 128.  Every
        // panel costs the GEMM a pass over U (read-add-write epilogue) and a fresh prologue / tail per tile: 64 MiB
        // panels made the 32-instance encaps at C4 1.80 ms, of which only 0.36 ms is the generator and 1.0 ms the GEMM
        size_t rows = ((size_t)256 << 20) / (2 * n) / 128 * 128;
        if (rows < 128) rows = 128;
        if (rows > 65536) rows = 65536;          // one tensor-core pass holds at most 65536 rows (32-bit byte-plane sums)
        if (rows > m) rows = m;
        c->panel_rows = c->panel_rows_alloc = (uint32_t)rows;
        ok(dev_alloc(&c->d_Apanel, rows * n));
    }
    ok(dev_alloc(&c->d_foflags, B));
    ok(dev_alloc(&c->d_vprime, B * k));
    ok(dev_alloc(&c->d_tile_locks, encaps_regen_lock_words(*p)));
    ok(dev_alloc(&c->d_vacc, k * B));
    ok(dev_alloc(&c->d_dacc, k * B));
    ok(dev_alloc(&c->d_counters, 8 + 2 * B));
    if (wide) {
        // the packed public matrix and its exception lists (lwe_wide_load_matrix); no lwe_kem_host staging
        c->exc_cap_col = exc_capacity(p->m, p->q);
        c->exc_cap_row = exc_capacity(p->n, p->q);
        ok(dev_alloc(&c->d_A16, m * n));
        ok(dev_alloc(&c->d_exc_col_cnt, n)); ok(dev_alloc(&c->d_exc_col_rows, n * c->exc_cap_col));
        ok(dev_alloc(&c->d_exc_row_cnt, m)); ok(dev_alloc(&c->d_exc_row_cols, m * c->exc_cap_row));
        ok(dev_alloc(&c->d_exc_overflow, 4));
        ok(cudaMallocHost(reinterpret_cast<void **>(&c->h_exc_overflow), 16));
    } else {
        ok(dev_alloc(&c->d_hs, B * n)); ok(dev_alloc(&c->d_he, B * m)); ok(dev_alloc(&c->d_hb, B * m));
        ok(dev_alloc(&c->d_hU, B * n * k)); ok(dev_alloc(&c->d_hv, B * k));
        ok(dev_alloc(&c->d_hR, B * m * k / 8)); ok(dev_alloc(&c->d_hmu, B * k / 8)); ok(dev_alloc(&c->d_hmuout, B * k / 8));
    }
    ok(cudaStreamCreateWithFlags(&c->s_in, cudaStreamNonBlocking));
    ok(cudaStreamCreateWithFlags(&c->s_out, cudaStreamNonBlocking));
    ok(cudaEventCreateWithFlags(&c->ev_entry, cudaEventDisableTiming));
    ok(cudaEventCreateWithFlags(&c->ev_out, cudaEventDisableTiming));
    ok(cudaEventCreateWithFlags(&c->ev_se, cudaEventDisableTiming));
    ok(cudaEventCreateWithFlags(&c->ev_kg, cudaEventDisableTiming));
    for (int i = 0; i < kHostChunks; i++) {
        ok(cudaEventCreateWithFlags(&c->ev_in[i], cudaEventDisableTiming));
        ok(cudaEventCreateWithFlags(&c->ev_done[i], cudaEventDisableTiming));
    }
    if (e == cudaSuccess) {
        uint32_t te0[256];
        aes_te0_host(te0);
        ok(cudaMemcpy(c->d_te0, te0, sizeof(te0), cudaMemcpyHostToDevice));
        ok(cudaMemset(c->d_vacc, 0, k * B * sizeof(unsigned long long)));
        ok(cudaMemset(c->d_dacc, 0, k * B * sizeof(unsigned long long)));
        ok(cudaMemset(c->d_counters, 0, (8 + 2 * B) * sizeof(unsigned int)));
        ok(cudaMemset(c->d_tile_locks, 0, encaps_regen_lock_words(*p) * sizeof(uint32_t)));
    }
    if (e != cudaSuccess) {
        free_all(c);
        delete h;
        return LWE_ERR_CUDA;
    }
    // TMA descriptor encoder, resolved through the runtime (no link-time libcuda dependency)
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPointByVersion("cuTensorMapEncodeTiled", &fn, 12000, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
        c->encode_tiled = fn;
    cudaGetLastError();
    *out = h;
    return LWE_OK;
}

void lwe_destroy(lwe_ctx *ctx)
{
    NvtxScope nvtx_("lwe_destroy");
    if (!ctx) return;
    DeviceGuard guard(ctx->c.device);
    cudaDeviceSynchronize();
    free_all(&ctx->c);
    delete ctx;
}

int lwe_last_cuda_error(const lwe_ctx *ctx) { return ctx ? ctx->c.last_cuda_error : 0; }
uint64_t lwe_launch_count(const lwe_ctx *ctx) { return ctx ? ctx->c.launches : 0; }

int lwe_set_option(lwe_ctx *ctx, int option, int64_t value)
{
    CHECK_CTX(ctx);
    if (option == LWE_OPT_ENCAPS_PATH) {
        if (value < 0 || value > 3) return LWE_ERR_PARAM;
        ctx->c.encaps_path = (int)value;
        return LWE_OK;
    }
    if (option == LWE_OPT_KEYGEN_PATH) {
        if (value < 0 || value > 2) return LWE_ERR_PARAM;
        ctx->c.keygen_path = (int)value;
        return LWE_OK;
    }
    if (option == LWE_OPT_PANEL_ROWS) {
        Ctx *c = &ctx->c;
        if (value == 0) { c->panel_rows = c->panel_rows_alloc; return LWE_OK; }
        if (value < 8 || value % 8 || value > (int64_t)c->panel_rows_alloc) return LWE_ERR_PARAM;
        c->panel_rows = (uint32_t)value;
        return LWE_OK;
    }
    if (option == LWE_OPT_R_OPERAND) {
        if (value < 0 || value > 1) return LWE_ERR_PARAM;
        ctx->c.r_operand = (int)value;
        return LWE_OK;
    }
    if (option == LWE_OPT_PDL) {
        if (value < 0 || value > 1) return LWE_ERR_PARAM;
        ctx->c.no_pdl = value ? 0 : 1;
        return LWE_OK;
    }
    if (option == LWE_OPT_V_PATH) {
        if (value < 0 || value > 1) return LWE_ERR_PARAM;
        ctx->c.v_path = (int)value;
        return LWE_OK;
    }
    if (option == LWE_OPT_REGEN_PATH) {
        if (value < 0 || value > 2) return LWE_ERR_PARAM;
        ctx->c.regen_path = (int)value;
        return LWE_OK;
    }
    if (option == LWE_OPT_PROFILE) {
        Ctx *c = &ctx->c;
        if (value < 0 || value > 1 + LWE_K_COUNT) return LWE_ERR_PARAM;
        if (value && !c->ev) {
            DeviceGuard guard(c->device);
            c->ev = new (std::nothrow) cudaEvent_t[2 * kMaxProfEvents]();
            c->ev_kernel = new (std::nothrow) uint8_t[kMaxProfEvents]();
            if (!c->ev || !c->ev_kernel) return LWE_ERR_CUDA;
            for (int i = 0; i < 2 * kMaxProfEvents; i++) LWE_CUDA_TRY(c, cudaEventCreate(&c->ev[i]));
        }
        c->profile = (int)value;
        return LWE_OK;
    }
    return LWE_ERR_PARAM;
}

int lwe_probe_int8_pipe(lwe_ctx *ctx, uint32_t iters, int signed_dense_b, uint64_t *h_ops, void *stream)
{
    NvtxScope nvtx_("lwe_probe_int8_pipe");
    CHECK_CTX(ctx);
    if (iters == 0 || iters > (1u << 24) || (signed_dense_b != 0 && signed_dense_b != 1)) return LWE_ERR_PARAM;
    Ctx *c = &ctx->c;
    DeviceGuard guard(c->device);
    LAUNCH(c, launch_probe_int8(c, iters, signed_dense_b, h_ops, (cudaStream_t)stream));
    return LWE_OK;
}

int lwe_profile_reset(lwe_ctx *ctx)
{
    CHECK_CTX(ctx);
    ctx->c.n_ev = 0;
    return LWE_OK;
}

int lwe_profile_read(lwe_ctx *ctx, int kernel_id, double *h_total_ms, uint64_t *h_launches)
{
    CHECK_CTX(ctx);
    if (kernel_id < 0 || kernel_id >= LWE_K_COUNT) return LWE_ERR_PARAM;
    Ctx *c = &ctx->c;
    DeviceGuard guard(c->device);
    double total = 0.0;
    uint64_t count = 0;
    for (int i = 0; i < c->n_ev; i++) {
        if (c->ev_kernel[i] != kernel_id) continue;
        LWE_CUDA_TRY(c, cudaEventSynchronize(c->ev[2 * i + 1]));
        float ms = 0.f;
        LWE_CUDA_TRY(c, cudaEventElapsedTime(&ms, c->ev[2 * i], c->ev[2 * i + 1]));
        total += ms;
        count++;
    }
    if (h_total_ms) *h_total_ms = total;
    if (h_launches) *h_launches = count;
    return LWE_OK;
}

int lwe_rng_fill(lwe_ctx *ctx, void *d_out, size_t nbytes, const uint8_t key[16], const uint8_t iv[16],
                 uint64_t byte_offset, void *stream)
{
    NvtxScope nvtx_("lwe_rng_fill");
    CHECK_CTX(ctx);
    REQUIRE_PTR(key); REQUIRE_PTR(iv);
    if (nbytes == 0) return LWE_OK;
    REQUIRE_PTR(d_out); REQUIRE_ALIGNED(d_out);
    Ctx *c = &ctx->c;
    DeviceGuard guard(c->device);
    AesKey k;
    aes128_expand_key_host(key, &k);
    uint64_t hi = 0, lo = 0;
    for (int i = 0; i < 8; i++) { hi = (hi << 8) | iv[i]; lo = (lo << 8) | iv[8 + i]; }
    LAUNCH(c, launch_rng_fill(c, (uint8_t *)d_out, nbytes, k, hi, lo, byte_offset, (cudaStream_t)stream));
    return LWE_OK;
}

static int sampler_args(lwe_ctx *ctx, const void *d_out, uint64_t first, uint64_t count, uint32_t tag,
                        uint32_t inst0, uint32_t n_inst)
{
    CHECK_CTX(ctx);
    if (tag == 0 || tag > 255) return LWE_ERR_PARAM;
    if ((uint64_t)inst0 + n_inst > (1ull << 32)) return LWE_ERR_PARAM;
    if (first % 8) return LWE_ERR_ALIGN;
    if (count == 0 || n_inst == 0) return LWE_OK;
    REQUIRE_PTR(d_out); REQUIRE_ALIGNED(d_out);
    return LWE_OK;
}

int lwe_sample_uniform(lwe_ctx *ctx, uint16_t *d_out, uint64_t first, uint64_t count, uint64_t seed,
                       uint32_t tag, uint32_t inst0, uint32_t n_inst, void *stream)
{
    NvtxScope nvtx_("lwe_sample_uniform");
    int rc = sampler_args(ctx, d_out, first, count, tag, inst0, n_inst);
    if (rc != LWE_OK) return rc;
    REQUIRE_NARROW(ctx);
    if (count == 0 || n_inst == 0) return rc;
    Ctx *c = &ctx->c;
    DeviceGuard guard(c->device);
    LAUNCH(c, launch_sample_uniform(c, d_out, first, count, seed_key_host(seed), tag, inst0, n_inst, (cudaStream_t)stream));
    return LWE_OK;
}

int lwe_sample_cbd(lwe_ctx *ctx, uint16_t *d_out, uint64_t first, uint64_t count, uint64_t seed,
                   uint32_t tag, uint32_t inst0, uint32_t n_inst, void *stream)
{
    NvtxScope nvtx_("lwe_sample_cbd");
    int rc = sampler_args(ctx, d_out, first, count, tag, inst0, n_inst);
    if (rc != LWE_OK) return rc;
    REQUIRE_NARROW(ctx);
    if (count == 0 || n_inst == 0) return rc;
    Ctx *c = &ctx->c;
    DeviceGuard guard(c->device);
    LAUNCH(c, launch_sample_cbd(c, d_out, first, count, seed_key_host(seed), tag, inst0, n_inst, (cudaStream_t)stream));
    return LWE_OK;
}

int lwe_sample_bits(lwe_ctx *ctx, uint8_t *d_out, uint64_t first_bit, uint64_t nbits, uint64_t seed,
                    uint32_t tag, uint32_t inst0, uint32_t n_inst, void *stream)
{
    NvtxScope nvtx_("lwe_sample_bits");
    int rc = sampler_args(ctx, d_out, first_bit, nbits, tag, inst0, n_inst);
    if (rc != LWE_OK || nbits == 0 || n_inst == 0) return rc;
    Ctx *c = &ctx->c;
    DeviceGuard guard(c->device);
    LAUNCH(c, launch_sample_bits(c, d_out, first_bit, nbits, seed_key_host(seed), tag, inst0, n_inst, (cudaStream_t)stream));
    return LWE_OK;
}

int lwe_sample_kem(lwe_ctx *ctx, uint16_t *d_s, uint16_t *d_e, uint8_t *d_Rbits, uint8_t *d_mubits, uint64_t seed,
                   uint32_t inst0, uint32_t n_inst, void *stream)
{
    NvtxScope nvtx_("lwe_sample_kem");
    CHECK_CTX(ctx);
    REQUIRE_NARROW(ctx);
    if ((uint64_t)inst0 + n_inst > (1ull << 32)) return LWE_ERR_PARAM;
    if (n_inst == 0) return LWE_OK;
    REQUIRE_PTR(d_s); REQUIRE_PTR(d_e); REQUIRE_PTR(d_Rbits); REQUIRE_PTR(d_mubits);
    REQUIRE_ALIGNED(d_s); REQUIRE_ALIGNED(d_e); REQUIRE_ALIGNED(d_Rbits); REQUIRE_ALIGNED(d_mubits);
    Ctx *c = &ctx->c;
    DeviceGuard guard(c->device);
    LAUNCH(c, launch_sample_kem(c, d_s, d_e, d_Rbits, d_mubits, seed_key_host(seed), inst0, n_inst, (cudaStream_t)stream));
    return LWE_OK;
}

int lwe_keygen(lwe_ctx *ctx, const uint16_t *d_A, uint64_t seed_A, const uint16_t *d_s, const uint16_t *d_e,
               uint16_t *d_b, uint32_t batch, void *stream)
{
    NvtxScope nvtx_("lwe_keygen");
    CHECK_CTX(ctx);
    REQUIRE_NARROW(ctx);
    Ctx *c = &ctx->c;
    if (batch == 0 || batch > c->p.max_batch) return LWE_ERR_PARAM;
    REQUIRE_PTR(d_s); REQUIRE_PTR(d_e); REQUIRE_PTR(d_b);
    REQUIRE_ALIGNED(d_A); REQUIRE_ALIGNED(d_s); REQUIRE_ALIGNED(d_e); REQUIRE_ALIGNED(d_b);
    bool tcp = d_A && keygen_tc_supported(c, batch) && (c->keygen_path == 2 || (c->keygen_path == 0 && batch >= 2));
    if (d_A && c->keygen_path == 2 && !tcp) return LWE_ERR_UNSUPPORTED;
    DeviceGuard guard(c->device);
    if (tcp) LAUNCH(c, launch_keygen_tc(c, d_A, d_s, d_e, d_b, batch, (cudaStream_t)stream));
    else if (d_A) LAUNCH(c, launch_keygen_stored(c, d_A, d_s, d_e, d_b, batch, (cudaStream_t)stream));
    else LAUNCH(c, launch_keygen_regen(c, seed_key_host(seed_A), d_s, d_e, d_b, batch, (cudaStream_t)stream));
    return LWE_OK;
}

// expand R (+ v) and run U = A^T R.  compare = false: write U (accumulating over the panels of a regenerated A);
// compare = true (stored A only): write nothing, compare with d_U and OR mismatches into c->d_foflags.
static int encaps_core(Ctx *c, const uint16_t *d_A, uint64_t seed_A, const uint16_t *d_b, const uint8_t *d_Rbits,
                       const uint8_t *d_mubits, uint16_t *d_U, uint16_t *d_v, uint32_t batch, bool compare, cudaStream_t st)
{
    bool tc = encaps_tc_supported(c, batch);
    if (c->encaps_path == 1) tc = false;
    if (c->encaps_path >= 2 && !tc) return LWE_ERR_UNSUPPORTED;
    // CTA pairs (cta_group::2) by default; path 2 keeps the single-CTA kernel selectable
    const bool pair = tc && c->encaps_path != 2 && encaps_tc2_supported(c, batch);
    if (c->encaps_path == 3 && !pair) return LWE_ERR_UNSUPPORTED;
    // one instance, A regenerated: generate the A tiles straight into the GEMM's shared-memory operand (N4)
    const bool fused = !d_A && !compare && tc && c->encaps_path != 1 && c->regen_path != 1 &&
                       encaps_regen_tc_supported(c, batch);
    if (!d_A && c->regen_path == 2 && !fused) return LWE_ERR_UNSUPPORTED;
    // CTA-pair GEMM with k % 128 == 0: the kernel expands its B tiles from the packed bits itself; the pass over R
    // here then only computes v (no expanded operand is written)
    const bool bits = pair && !fused && c->r_operand != 1 && encaps_tc2_bits_supported(c, batch);
    // ... and v comes from spare warps of that same kernel (LWE_OPT_V_PATH = 1: from the separate pass below)
    const bool v_fused = bits && c->v_path != 1 && encaps_tc2_v_fused_supported(c, batch);
    if (!v_fused)       // one pass over R's bits: v, and the expanded operand for the kernels that read one
        LAUNCH(c, launch_expand_R_and_v(c, d_b, d_Rbits, d_mubits, d_v, batch, tc && (fused || !bits), st));   // the fused regenerated-A kernel loads R through TMA
    if (fused) {
        LAUNCH(c, launch_encaps_regen_tc(c, seed_key_host(seed_A), d_U, st));
        return LWE_OK;
    }
    // Stored A: one pass over all m rows (m > 65536: passes of 65536 rows, the most a 32-bit byte-plane sum holds,
    // accumulated mod q).  d_A == NULL: A is regenerated from seed_A one row panel at a
    // time into the context's panel buffer (rows of A are contiguous ranges of the counter-indexed
    // stream) and the contraction is accumulated over the panels; A is never held in full.
    // Either way a pass is at most 65536 rows: the tcgen05 epilogue recombines lo + (hi << 8) in 32 bits, and a byte-plane
    // sum over more rows would wrap for a modulus that is not a power of two.
    const uint32_t m = c->p.m, cap = d_A ? m : c->panel_rows, step = cap < 65536u ? cap : 65536u;
    const AesKey keyA = d_A ? AesKey() : seed_key_host(seed_A);
    for (uint32_t row0 = 0; row0 < m; row0 += step) {
        const uint32_t rows = (m - row0 < step) ? (m - row0) : step;
        const uint16_t *panel = d_A ? d_A + (size_t)row0 * c->p.n : nullptr;
        if (!d_A) {
            LAUNCH(c, launch_sample_uniform(c, c->d_Apanel, (uint64_t)row0 * c->p.n, (uint64_t)rows * c->p.n, keyA,
                                            LWE_TAG_A, 0, 1, st));
            panel = c->d_Apanel;
        }
        const int mode = compare ? 2 : (row0 != 0 ? 1 : 0);
        if (pair) {
            const bool with_v = v_fused && row0 == 0;               // v spans all m rows: once, with the first panel
            LAUNCH(c, launch_encaps_tc2(c, panel, d_U, batch, row0, rows, mode, c->d_foflags, st, bits ? d_Rbits : nullptr,
                                        with_v ? d_b : nullptr, d_mubits, d_v));
        }
        else if (tc) LAUNCH(c, launch_encaps_tc(c, panel, d_U, batch, row0, rows, mode, c->d_foflags, st));
        else LAUNCH(c, launch_encaps_simt(c, panel, d_Rbits, d_U, batch, row0, rows, mode, c->d_foflags, st));
    }
    return LWE_OK;
}

int lwe_encaps(lwe_ctx *ctx, const uint16_t *d_A, uint64_t seed_A, const uint16_t *d_b, const uint8_t *d_Rbits,
               const uint8_t *d_mubits, uint16_t *d_U, uint16_t *d_v, uint32_t batch, void *stream)
{
    NvtxScope nvtx_("lwe_encaps");
    CHECK_CTX(ctx);
    REQUIRE_NARROW(ctx);
    Ctx *c = &ctx->c;
    if (batch == 0 || batch > c->p.max_batch) return LWE_ERR_PARAM;
    REQUIRE_PTR(d_b); REQUIRE_PTR(d_Rbits); REQUIRE_PTR(d_mubits); REQUIRE_PTR(d_U); REQUIRE_PTR(d_v);
    REQUIRE_ALIGNED(d_A); REQUIRE_ALIGNED(d_b); REQUIRE_ALIGNED(d_Rbits); REQUIRE_ALIGNED(d_mubits);
    REQUIRE_ALIGNED(d_U); REQUIRE_ALIGNED(d_v);
    DeviceGuard guard(c->device);
    return encaps_core(c, d_A, seed_A, d_b, d_Rbits, d_mubits, d_U, d_v, batch, false, (cudaStream_t)stream);
}

int lwe_decaps_fo(lwe_ctx *ctx, const uint16_t *d_A, const uint16_t *d_b, const uint16_t *d_U, const uint16_t *d_v,
                  const uint16_t *d_s, const uint8_t *d_Rbits, uint8_t *d_mubits_out, uint8_t *d_ok, uint32_t batch,
                  void *stream)
{
    NvtxScope nvtx_("lwe_decaps_fo");
    CHECK_CTX(ctx);
    REQUIRE_NARROW(ctx);
    Ctx *c = &ctx->c;
    if (batch == 0 || batch > c->p.max_batch) return LWE_ERR_PARAM;
    REQUIRE_PTR(d_A); REQUIRE_PTR(d_b); REQUIRE_PTR(d_U); REQUIRE_PTR(d_v); REQUIRE_PTR(d_s); REQUIRE_PTR(d_Rbits);
    REQUIRE_PTR(d_mubits_out); REQUIRE_PTR(d_ok);
    REQUIRE_ALIGNED(d_A); REQUIRE_ALIGNED(d_b); REQUIRE_ALIGNED(d_U); REQUIRE_ALIGNED(d_v); REQUIRE_ALIGNED(d_s);
    REQUIRE_ALIGNED(d_Rbits); REQUIRE_ALIGNED(d_mubits_out); REQUIRE_ALIGNED(d_ok);
    if (c->encaps_path >= 2 && !encaps_tc_supported(c, batch)) return LWE_ERR_UNSUPPORTED;
    if (c->p.m > 65536u) return LWE_ERR_UNSUPPORTED;     // the compare epilogue needs the whole sum in one pass
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    // Alg. 5: 1. m' <- Decrypt(sk, c)
    LAUNCH(c, launch_decaps(c, d_U, d_v, d_s, d_mubits_out, batch, st));
    // 2. c' <- Encrypt(pk, m') with the re-derived coins R; c' = (U', v') is never stored: v' goes to the
    //    workspace, U' is compared with U tile by tile in the GEMM epilogue
    LWE_CUDA_TRY(c, cudaMemsetAsync(c->d_foflags, 0, batch * sizeof(uint32_t), st));
    int rc = encaps_core(c, d_A, 0, d_b, d_Rbits, d_mubits_out, const_cast<uint16_t *>(d_U), c->d_vprime, batch, true, st);
    if (rc != LWE_OK) return rc;
    // 4. verdict c' == c per instance, on the device
    LAUNCH(c, launch_fo_verdict(c, d_v, c->d_vprime, c->d_foflags, d_ok, batch, st));
    return LWE_OK;
}

int lwe_decaps(lwe_ctx *ctx, const uint16_t *d_U, const uint16_t *d_v, const uint16_t *d_s,
               uint8_t *d_mubits_out, uint32_t batch, void *stream)
{
    NvtxScope nvtx_("lwe_decaps");
    CHECK_CTX(ctx);
    REQUIRE_NARROW(ctx);
    Ctx *c = &ctx->c;
    if (batch == 0 || batch > c->p.max_batch) return LWE_ERR_PARAM;
    REQUIRE_PTR(d_U); REQUIRE_PTR(d_v); REQUIRE_PTR(d_s); REQUIRE_PTR(d_mubits_out);
    REQUIRE_ALIGNED(d_U); REQUIRE_ALIGNED(d_v); REQUIRE_ALIGNED(d_s); REQUIRE_ALIGNED(d_mubits_out);
    DeviceGuard guard(c->device);
    LAUNCH(c, launch_decaps(c, d_U, d_v, d_s, d_mubits_out, batch, (cudaStream_t)stream));
    return LWE_OK;
}

static int gauss_args(lwe_ctx *ctx, const void *d_out, uint64_t first, uint64_t count, uint32_t tag, uint32_t inst0,
                      uint32_t n_inst, double sigma)
{
    int rc = sampler_args(ctx, d_out, first, count, tag, inst0, n_inst);
    if (rc != LWE_OK) return rc;
    if (!(sigma >= 0.5 && sigma <= 2.8)) return LWE_ERR_PARAM;   // the 24-entry table spans [-12, 12]: see lwe.h
    return LWE_OK;
}

int lwe_sample_gauss_s8(lwe_ctx *ctx, int8_t *d_out, uint64_t first, uint64_t count, uint64_t seed, uint32_t tag,
                        uint32_t inst0, uint32_t n_inst, double sigma, void *stream)
{
    NvtxScope nvtx_("lwe_sample_gauss_s8");
    int rc = gauss_args(ctx, d_out, first, count, tag, inst0, n_inst, sigma);
    if (rc != LWE_OK || count == 0 || n_inst == 0) return rc;
    Ctx *c = &ctx->c;
    DeviceGuard guard(c->device);
    LAUNCH(c, launch_sample_gauss(c, d_out, false, first, count, seed_key_host(seed), tag, inst0, n_inst, sigma,
                                  (cudaStream_t)stream));
    return LWE_OK;
}

int lwe_sample_gauss_u16(lwe_ctx *ctx, uint16_t *d_out, uint64_t first, uint64_t count, uint64_t seed, uint32_t tag,
                         uint32_t inst0, uint32_t n_inst, double sigma, void *stream)
{
    NvtxScope nvtx_("lwe_sample_gauss_u16");
    int rc = gauss_args(ctx, d_out, first, count, tag, inst0, n_inst, sigma);
    if (rc != LWE_OK) return rc;
    REQUIRE_NARROW(ctx);
    if (count == 0 || n_inst == 0) return rc;
    Ctx *c = &ctx->c;
    DeviceGuard guard(c->device);
    LAUNCH(c, launch_sample_gauss(c, d_out, true, first, count, seed_key_host(seed), tag, inst0, n_inst, sigma,
                                  (cudaStream_t)stream));
    return LWE_OK;
}

int lwe_sample_cuniform_s8(lwe_ctx *ctx, int8_t *d_out, uint64_t first, uint64_t count, uint64_t seed, uint32_t tag,
                           uint32_t inst0, uint32_t n_inst, uint32_t bound, void *stream)
{
    NvtxScope nvtx_("lwe_sample_cuniform_s8");
    CHECK_CTX(ctx);
    if (tag == 0 || tag > 255 || bound < 1 || bound > 127) return LWE_ERR_PARAM;
    if ((uint64_t)inst0 + n_inst > (1ull << 32)) return LWE_ERR_PARAM;
    if (count == 0 || n_inst == 0) return LWE_OK;
    REQUIRE_PTR(d_out); REQUIRE_ALIGNED(d_out);
    Ctx *c = &ctx->c;
    DeviceGuard guard(c->device);
    LAUNCH(c, launch_sample_cuniform(c, d_out, first, count, seed_key_host(seed), tag, inst0, n_inst, bound,
                                     (cudaStream_t)stream));
    return LWE_OK;
}

int lwe_sample_pke(lwe_ctx *ctx, void *d_s, void *d_e, int8_t *d_R, int8_t *d_E1, int8_t *d_e2, uint8_t *d_mubits,
                   uint64_t seed, uint32_t inst0, uint32_t n_inst, double sigma, uint32_t e2_bound, void *stream)
{
    NvtxScope nvtx_("lwe_sample_pke");
    CHECK_CTX(ctx);
    if (!(sigma >= 0.5 && sigma <= 2.8) || e2_bound < 1 || e2_bound > 127) return LWE_ERR_PARAM;
    if ((uint64_t)inst0 + n_inst > (1ull << 32)) return LWE_ERR_PARAM;
    if (n_inst == 0) return LWE_OK;
    REQUIRE_PTR(d_s); REQUIRE_PTR(d_e); REQUIRE_PTR(d_R); REQUIRE_PTR(d_E1); REQUIRE_PTR(d_e2); REQUIRE_PTR(d_mubits);
    REQUIRE_ALIGNED(d_s); REQUIRE_ALIGNED(d_e); REQUIRE_ALIGNED(d_R); REQUIRE_ALIGNED(d_E1); REQUIRE_ALIGNED(d_e2);
    REQUIRE_ALIGNED(d_mubits);
    Ctx *c = &ctx->c;
    DeviceGuard guard(c->device);
    LAUNCH(c, launch_sample_pke(c, d_s, d_e, d_R, d_E1, d_e2, d_mubits, seed_key_host(seed), inst0, n_inst, sigma, e2_bound,
                                (cudaStream_t)stream));
    return LWE_OK;
}

int lwe_encaps_pv(lwe_ctx *ctx, const uint16_t *d_A, const uint16_t *d_t, const int8_t *d_R, const int8_t *d_E1,
                  const int8_t *d_e2, const uint8_t *d_mubits, uint16_t *d_U, uint16_t *d_v, uint32_t batch, void *stream)
{
    NvtxScope nvtx_("lwe_encaps_pv");
    CHECK_CTX(ctx);
    REQUIRE_NARROW(ctx);
    Ctx *c = &ctx->c;
    if (batch == 0 || batch > c->p.max_batch) return LWE_ERR_PARAM;
    REQUIRE_PTR(d_A); REQUIRE_PTR(d_t); REQUIRE_PTR(d_R); REQUIRE_PTR(d_E1); REQUIRE_PTR(d_e2); REQUIRE_PTR(d_mubits);
    REQUIRE_PTR(d_U); REQUIRE_PTR(d_v);
    REQUIRE_ALIGNED(d_A); REQUIRE_ALIGNED(d_t); REQUIRE_ALIGNED(d_R); REQUIRE_ALIGNED(d_E1); REQUIRE_ALIGNED(d_e2);
    REQUIRE_ALIGNED(d_mubits); REQUIRE_ALIGNED(d_U); REQUIRE_ALIGNED(d_v);
    // tensor path: the CTA-pair GEMM; |lo/hi plane accumulator| <= 255 * 127 * m < 2^31 for m <= 65536
    bool tc = encaps_tc2_supported(c, batch) && c->encaps_path != 1 && c->p.m <= 65536u;
    if (c->encaps_path >= 2 && !tc) return LWE_ERR_UNSUPPORTED;
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    // k % 128 == 0: the GEMM reads R in place (no operand copy); the pass over R then only computes v
    const bool inplace = tc && c->r_operand != 1 && encaps_tc2_r_inplace_supported(c, batch);
    LAUNCH(c, launch_prep_R_pv_and_v(c, d_t, d_R, d_e2, d_mubits, d_v, batch, tc && !inplace, st));
    if (tc) LAUNCH(c, launch_encaps_tc2_pv(c, d_A, d_E1, d_U, batch, st, inplace ? d_R : nullptr));
    else LAUNCH(c, launch_encaps_pv_simt(c, d_A, d_R, d_E1, d_U, batch, st));
    return LWE_OK;
}

// ---------------------------------------------------------------------------------- wide contexts (q > 65536)

int lwe_sample_uniform_u32(lwe_ctx *ctx, uint32_t *d_out, uint64_t first, uint64_t count, uint64_t seed, uint32_t tag,
                           uint32_t inst0, uint32_t n_inst, void *stream)
{
    NvtxScope nvtx_("lwe_sample_uniform_u32");
    CHECK_CTX(ctx);
    REQUIRE_WIDE(ctx);
    if (tag == 0 || tag > 255) return LWE_ERR_PARAM;
    if ((uint64_t)inst0 + n_inst > (1ull << 32)) return LWE_ERR_PARAM;
    if (first % 4) return LWE_ERR_ALIGN;
    if (count == 0 || n_inst == 0) return LWE_OK;
    REQUIRE_PTR(d_out); REQUIRE_ALIGNED(d_out);
    Ctx *c = &ctx->c;
    DeviceGuard guard(c->device);
    LAUNCH(c, launch_sample_uniform32(c, d_out, first, count, seed_key_host(seed), tag, inst0, n_inst, (cudaStream_t)stream));
    return LWE_OK;
}

int lwe_sample_cbd_s8(lwe_ctx *ctx, int8_t *d_out, uint64_t first, uint64_t count, uint64_t seed, uint32_t tag,
                      uint32_t inst0, uint32_t n_inst, void *stream)
{
    NvtxScope nvtx_("lwe_sample_cbd_s8");
    int rc = sampler_args(ctx, d_out, first, count, tag, inst0, n_inst);
    if (rc != LWE_OK || count == 0 || n_inst == 0) return rc;
    Ctx *c = &ctx->c;
    DeviceGuard guard(c->device);
    LAUNCH(c, launch_sample_cbd_s8(c, d_out, first, count, seed_key_host(seed), tag, inst0, n_inst, (cudaStream_t)stream));
    return LWE_OK;
}

// pack rows of A given in panels; checks the exception lists afterwards (host synchronisation)
static int wide_finish_load(Ctx *c, cudaStream_t st)
{
    LWE_CUDA_TRY(c, cudaMemcpyAsync(c->h_exc_overflow, c->d_exc_overflow, sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
    LWE_CUDA_TRY(c, cudaStreamSynchronize(st));
    if (*c->h_exc_overflow) return (*c->h_exc_overflow & 2u) ? LWE_ERR_PARAM : LWE_ERR_UNSUPPORTED;
    c->A_loaded = 1;
    return LWE_OK;
}

static int wide_begin_load(Ctx *c, cudaStream_t st)
{
    c->A_loaded = 0;
    LWE_CUDA_TRY(c, cudaMemsetAsync(c->d_exc_col_cnt, 0, (size_t)c->p.n * sizeof(uint32_t), st));
    LWE_CUDA_TRY(c, cudaMemsetAsync(c->d_exc_row_cnt, 0, (size_t)c->p.m * sizeof(uint32_t), st));
    LWE_CUDA_TRY(c, cudaMemsetAsync(c->d_exc_overflow, 0, sizeof(uint32_t), st));
    return LWE_OK;
}

int lwe_wide_load_matrix(lwe_ctx *ctx, const uint32_t *d_A, void *stream)
{
    NvtxScope nvtx_("lwe_wide_load_matrix");
    CHECK_CTX(ctx);
    REQUIRE_WIDE(ctx);
    REQUIRE_PTR(d_A); REQUIRE_ALIGNED(d_A);
    Ctx *c = &ctx->c;
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    int rc = wide_begin_load(c, st);
    if (rc != LWE_OK) return rc;
    LAUNCH(c, launch_wide_pack(c, d_A, 0, c->p.m, st));
    return wide_finish_load(c, st);
}

int lwe_wide_load_matrix_seeded(lwe_ctx *ctx, uint64_t seed_A, void *stream)
{
    NvtxScope nvtx_("lwe_wide_load_matrix_seeded");
    CHECK_CTX(ctx);
    REQUIRE_WIDE(ctx);
    Ctx *c = &ctx->c;
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    int rc = wide_begin_load(c, st);
    if (rc != LWE_OK) return rc;
    // the uint32 A never exists in full: one row panel at a time through the context's panel buffer
    const AesKey key = seed_key_host(seed_A);
    uint32_t *panel = reinterpret_cast<uint32_t *>(c->d_Apanel);
    uint32_t step = c->panel_rows_alloc / 2;                   // the buffer holds panel_rows_alloc rows of uint16
    if (step < 1) step = 1;
    for (uint32_t row0 = 0; row0 < c->p.m; row0 += step) {
        const uint32_t rows = (c->p.m - row0 < step) ? (c->p.m - row0) : step;
        LAUNCH(c, launch_sample_uniform32(c, panel, (uint64_t)row0 * c->p.n, (uint64_t)rows * c->p.n, key, LWE_TAG_A, 0, 1, st));
        LAUNCH(c, launch_wide_pack(c, panel, row0, rows, st));
    }
    return wide_finish_load(c, st);
}

int lwe_wide_keygen(lwe_ctx *ctx, const int8_t *d_s, const int8_t *d_e, uint32_t *d_t, uint32_t batch, void *stream)
{
    NvtxScope nvtx_("lwe_wide_keygen");
    CHECK_CTX(ctx);
    REQUIRE_WIDE(ctx);
    Ctx *c = &ctx->c;
    if (batch == 0 || batch > c->p.max_batch) return LWE_ERR_PARAM;
    if (!c->A_loaded) return LWE_ERR_PARAM;
    REQUIRE_PTR(d_s); REQUIRE_PTR(d_e); REQUIRE_PTR(d_t);
    REQUIRE_ALIGNED(d_s); REQUIRE_ALIGNED(d_e); REQUIRE_ALIGNED(d_t);
    const bool tc = c->keygen_path != 1 && wide_keygen_tc_supported(c, batch);
    if (c->keygen_path == 2 && !tc) return LWE_ERR_UNSUPPORTED;
    DeviceGuard guard(c->device);
    if (tc) LAUNCH(c, launch_wide_keygen_tc(c, d_s, d_e, d_t, batch, (cudaStream_t)stream));
    else LAUNCH(c, launch_wide_keygen_simt(c, d_s, d_e, d_t, batch, (cudaStream_t)stream));
    return LWE_OK;
}

int lwe_wide_encaps(lwe_ctx *ctx, const uint32_t *d_t, const int8_t *d_R, const int8_t *d_E1, const int8_t *d_e2,
                    const uint8_t *d_mubits, uint32_t *d_U, uint32_t *d_v, uint32_t batch, void *stream)
{
    NvtxScope nvtx_("lwe_wide_encaps");
    CHECK_CTX(ctx);
    REQUIRE_WIDE(ctx);
    Ctx *c = &ctx->c;
    if (batch == 0 || batch > c->p.max_batch) return LWE_ERR_PARAM;
    if (!c->A_loaded) return LWE_ERR_PARAM;
    REQUIRE_PTR(d_t); REQUIRE_PTR(d_R); REQUIRE_PTR(d_E1); REQUIRE_PTR(d_e2); REQUIRE_PTR(d_mubits); REQUIRE_PTR(d_U);
    REQUIRE_PTR(d_v);
    REQUIRE_ALIGNED(d_t); REQUIRE_ALIGNED(d_R); REQUIRE_ALIGNED(d_E1); REQUIRE_ALIGNED(d_e2); REQUIRE_ALIGNED(d_mubits);
    REQUIRE_ALIGNED(d_U); REQUIRE_ALIGNED(d_v);
    const bool tc = encaps_tc2_supported(c, batch) && c->encaps_path != 1;
    if (c->encaps_path >= 2 && !tc) return LWE_ERR_UNSUPPORTED;
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    const bool inplace = tc && encaps_tc2_r_inplace_supported(c, batch);
    LAUNCH(c, launch_wide_v(c, d_t, d_R, d_e2, d_mubits, d_v, batch, tc && !inplace, st));
    if (tc) LAUNCH(c, launch_wide_encaps_tc2(c, d_R, d_E1, d_U, batch, st));
    else LAUNCH(c, launch_wide_encaps_simt(c, d_R, d_E1, d_U, batch, st));
    return LWE_OK;
}

int lwe_wide_decaps(lwe_ctx *ctx, const uint32_t *d_U, const uint32_t *d_v, const int8_t *d_s, uint8_t *d_mubits_out,
                    uint32_t batch, void *stream)
{
    NvtxScope nvtx_("lwe_wide_decaps");
    CHECK_CTX(ctx);
    REQUIRE_WIDE(ctx);
    Ctx *c = &ctx->c;
    if (batch == 0 || batch > c->p.max_batch) return LWE_ERR_PARAM;
    REQUIRE_PTR(d_U); REQUIRE_PTR(d_v); REQUIRE_PTR(d_s); REQUIRE_PTR(d_mubits_out);
    REQUIRE_ALIGNED(d_U); REQUIRE_ALIGNED(d_v); REQUIRE_ALIGNED(d_s); REQUIRE_ALIGNED(d_mubits_out);
    DeviceGuard guard(c->device);
    LAUNCH(c, launch_wide_decaps(c, d_U, d_v, d_s, d_mubits_out, batch, (cudaStream_t)stream));
    return LWE_OK;
}

int lwe_kem_host(lwe_ctx *ctx, const uint16_t *d_A, uint64_t seed_A, const uint16_t *h_s, const uint16_t *h_e,
                 const uint8_t *h_Rbits, const uint8_t *h_mubits, uint16_t *h_b, uint16_t *h_U, uint16_t *h_v,
                 uint8_t *h_mubits_out, uint32_t batch, void *stream)
{
    NvtxScope nvtx_("lwe_kem_host");
    CHECK_CTX(ctx);
    REQUIRE_NARROW(ctx);
    Ctx *c = &ctx->c;
    if (batch == 0 || batch > c->p.max_batch) return LWE_ERR_PARAM;
    REQUIRE_PTR(h_s); REQUIRE_PTR(h_e); REQUIRE_PTR(h_Rbits); REQUIRE_PTR(h_mubits);
    REQUIRE_PTR(h_b); REQUIRE_PTR(h_v); REQUIRE_PTR(h_mubits_out);
    REQUIRE_ALIGNED(d_A);
    REQUIRE_ALIGNED(h_s); REQUIRE_ALIGNED(h_e); REQUIRE_ALIGNED(h_Rbits); REQUIRE_ALIGNED(h_mubits);
    REQUIRE_ALIGNED(h_b); REQUIRE_ALIGNED(h_U); REQUIRE_ALIGNED(h_v); REQUIRE_ALIGNED(h_mubits_out);
    const size_t n = c->p.n, m = c->p.m, k = c->p.k;
    cudaStream_t st = (cudaStream_t)stream;
    DeviceGuard guard(c->device);
    // Software pipeline: the copy-in stream runs ahead of the compute stream (the caller's), the copy-out stream
    // behind it.  The call is bound by the copy-out of the ciphertexts (U: 2nk bytes per instance, 134 MB of the
    // 135 MB at C4), so the plan is made to START that copy as early as possible and never let it wait:
    //   * s, e and mu of every instance go in first (small), and KeyGen runs ONCE for the whole batch (A is read -- or
    //     regenerated -- once, not once per chunk);
    //   * Encrypt + Decrypt run chunk by chunk over R, with chunks of 1, 1, 2, 4, 8, ... instances: the first ciphertext
    //     is on its way back after one single-instance GEMM, and every later chunk is computed while the previous,
    //     smaller one is still on the bus.  (Equal chunks of 4 left the copy-out stream idle for the first chunk's
    //     compute and starved it in between: 46 GB/s of the link's 57.)
    // Chunk boundaries must be 16-byte aligned in every staging buffer (the packed-bit rows are the narrow ones: k/8
    // bytes of mu per instance); otherwise, and for a regenerated A (every Encrypt call regenerates all of A), fewer,
    // equal chunks are used.
    uint32_t c_t0[kHostChunks], c_g[kHostChunks], nchunks = 0;
    const bool row_aligned = ((k / 8) % 16 == 0) && ((m * k / 8) % 16 == 0);
    if (row_aligned && d_A) {
        uint32_t t0 = 0, g = 1;
        while (t0 < batch) {
            uint32_t take = (nchunks == (uint32_t)kHostChunks - 1) ? batch - t0 : (g < batch - t0 ? g : batch - t0);
            c_t0[nchunks] = t0; c_g[nchunks] = take; nchunks++;
            t0 += take;
            if (nchunks >= 2) g *= 2;
        }
    } else {
        uint32_t want = row_aligned ? (batch >= 16 ? 2u : 1u) : 1u;
        uint32_t per = (batch + want - 1) / want;
        if (((size_t)per * (k / 8)) % 16 || ((size_t)per * (m * k / 8)) % 16) per = batch;
        for (uint32_t t0 = 0; t0 < batch; t0 += per) {
            c_t0[nchunks] = t0; c_g[nchunks] = (batch - t0 < per) ? (batch - t0) : per; nchunks++;
        }
    }
    // Every failure from here on drains the three streams before returning: no copy to or from the caller's host
    // buffers may still be in flight when the call hands them back (lwe.h).
    auto drain = [&]() { cudaStreamSynchronize(c->s_in); cudaStreamSynchronize(st); cudaStreamSynchronize(c->s_out); };
#define KEM_HOST_TRY(expr)                                                                        \
    do {                                                                                          \
        cudaError_t _e = (expr);                                                                  \
        if (_e != cudaSuccess) { c->last_cuda_error = (int)_e; drain(); return LWE_ERR_CUDA; }    \
    } while (0)
    KEM_HOST_TRY(cudaEventRecord(c->ev_entry, st));
    KEM_HOST_TRY(cudaStreamWaitEvent(c->s_in, c->ev_entry, 0));      // staging buffers are free again
    KEM_HOST_TRY(cudaStreamWaitEvent(c->s_out, c->ev_entry, 0));
    KEM_HOST_TRY(cudaMemcpyAsync(c->d_hs, h_s, (size_t)batch * n * 2, cudaMemcpyHostToDevice, c->s_in));
    KEM_HOST_TRY(cudaMemcpyAsync(c->d_he, h_e, (size_t)batch * m * 2, cudaMemcpyHostToDevice, c->s_in));
    KEM_HOST_TRY(cudaMemcpyAsync(c->d_hmu, h_mubits, (size_t)batch * k / 8, cudaMemcpyHostToDevice, c->s_in));
    KEM_HOST_TRY(cudaEventRecord(c->ev_se, c->s_in));
    for (uint32_t ci = 0; ci < nchunks; ci++) {
        const size_t t0 = c_t0[ci], g = c_g[ci];
        KEM_HOST_TRY(cudaMemcpyAsync(c->d_hR + t0 * (m * k / 8), h_Rbits + t0 * (m * k / 8), g * m * k / 8,
                                        cudaMemcpyHostToDevice, c->s_in));
        KEM_HOST_TRY(cudaEventRecord(c->ev_in[ci], c->s_in));
    }
    KEM_HOST_TRY(cudaStreamWaitEvent(st, c->ev_se, 0));
    int rc = lwe_keygen(ctx, d_A, seed_A, c->d_hs, c->d_he, c->d_hb, batch, stream);
    if (rc != LWE_OK) { drain(); return rc; }
    KEM_HOST_TRY(cudaEventRecord(c->ev_kg, st));
    KEM_HOST_TRY(cudaStreamWaitEvent(c->s_out, c->ev_kg, 0));
    KEM_HOST_TRY(cudaMemcpyAsync(h_b, c->d_hb, (size_t)batch * m * 2, cudaMemcpyDeviceToHost, c->s_out));
    for (uint32_t ci = 0; ci < nchunks; ci++) {
        const size_t t0 = c_t0[ci];
        const uint32_t g = c_g[ci];
        KEM_HOST_TRY(cudaStreamWaitEvent(st, c->ev_in[ci], 0));
        rc = lwe_encaps(ctx, d_A, seed_A, c->d_hb + t0 * m, c->d_hR + t0 * (m * k / 8), c->d_hmu + t0 * (k / 8),
                        c->d_hU + t0 * n * k, c->d_hv + t0 * k, g, stream);
        if (rc != LWE_OK) { drain(); return rc; }
        KEM_HOST_TRY(cudaEventRecord(c->ev_done[ci], st));           // the chunk's ciphertext leaves before it is decrypted
        KEM_HOST_TRY(cudaStreamWaitEvent(c->s_out, c->ev_done[ci], 0));
        if (h_U)
            KEM_HOST_TRY(cudaMemcpyAsync(h_U + t0 * n * k, c->d_hU + t0 * n * k, (size_t)g * n * k * 2,
                                            cudaMemcpyDeviceToHost, c->s_out));
        rc = lwe_decaps(ctx, c->d_hU + t0 * n * k, c->d_hv + t0 * k, c->d_hs + t0 * n, c->d_hmuout + t0 * (k / 8), g, stream);
        if (rc != LWE_OK) { drain(); return rc; }
    }
    // the small outputs of every chunk in one copy each, behind the last chunk's Decrypt (a copy of a few hundred bytes
    // costs the copy engine as much as a megabyte of U)
    KEM_HOST_TRY(cudaEventRecord(c->ev_kg, st));
    KEM_HOST_TRY(cudaStreamWaitEvent(c->s_out, c->ev_kg, 0));
    KEM_HOST_TRY(cudaMemcpyAsync(h_v, c->d_hv, (size_t)batch * k * 2, cudaMemcpyDeviceToHost, c->s_out));
    KEM_HOST_TRY(cudaMemcpyAsync(h_mubits_out, c->d_hmuout, (size_t)batch * k / 8, cudaMemcpyDeviceToHost, c->s_out));
    KEM_HOST_TRY(cudaEventRecord(c->ev_out, c->s_out));
    KEM_HOST_TRY(cudaStreamWaitEvent(st, c->ev_out, 0));            // the caller's stream sees the whole call
    KEM_HOST_TRY(cudaStreamSynchronize(st));
    return LWE_OK;
}
#undef KEM_HOST_TRY

}  // extern "C"

// lwe_internal.cuh -- shared declarations of the CUDA path (context, launch helpers,
// modular arithmetic).  Product code: shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <cuda.h>
#include <stdint.h>
#include <stddef.h>

#include "../../include/lwe.h"

namespace lwe {

// ---------------------------------------------------------------------------------
// AES-128 round keys in the word convention the kernels use: word c of a 16-byte
// block is its bytes 4c..4c+3 loaded little-endian.
struct AesKey {
    uint32_t rk[44];
};

// Identifies one seeded stream family: key(seed) plus the upper 64 bits of the counter
// without the attempt / instance fields (S8(c) O3).
struct StreamId {
    AesKey key;
    uint32_t tag;
};

// mod-q helper constants.  mu = floor(2^32 / q) (exact 2^32/q for powers of two, which
// then needs q < 2^32: q = 65536 gives 65536).
struct ModQ {
    uint32_t q;
    uint32_t mu;        // floor(2^32 / q)
    uint32_t T;         // q * floor(65536 / q): rejection threshold of the uniform sampler
    uint32_t half;      // floor(q / 2)
    uint32_t pow2;      // 1 if q is a power of two
    uint32_t mask;      // q - 1 when pow2
    uint32_t two32;     // 2^32 mod q
};

__host__ __device__ __forceinline__ uint32_t mod_u32(uint32_t x, const ModQ &mq)
{
#ifdef __CUDA_ARCH__
    uint32_t qhat = __umulhi(x, mq.mu);
#else
    uint32_t qhat = (uint32_t)(((uint64_t)x * mq.mu) >> 32);
#endif
    uint32_t r = x - qhat * mq.q;          // in [0, 3q): Barrett with mu = floor(2^32/q)
    if (r >= mq.q) r -= mq.q;
    if (r >= mq.q) r -= mq.q;
    return r;
}

__host__ __device__ __forceinline__ uint32_t mod_u64(uint64_t x, const ModQ &mq)
{
    // x = hi*2^32 + lo = (hi mod q)(2^32 mod q) + lo (mod q): three 32-bit Barrett steps instead of a 64-bit
    // remainder (~100 instructions on the device).  (hi mod q)(2^32 mod q) < q^2 <= 2^32 fits 32 bits.
    if (mq.pow2) return (uint32_t)x & mq.mask;
    const uint32_t hi = (uint32_t)(x >> 32), lo = (uint32_t)x;
    const uint32_t t = mod_u32(hi, mq) * mq.two32;
    return mod_u32(mod_u32(t, mq) + mod_u32(lo, mq), mq);
}

// ---------------------------------------------------------------------------------
constexpr int kHostChunks = 8;        // lwe_kem_host splits a batch into at most this many chunks

// Per-context (hence per-device) launch state of one __global__ function: whether the opt-in to more than 48 KB
// of dynamic shared memory has been made ON THIS CONTEXT'S DEVICE (cudaFuncSetAttribute applies to the current
// device only) and the last occupancy answer.  Nothing of this kind is process-wide: a process may hold contexts
// on several GPUs.
struct KernelCfg {
    const void *fn;
    int occ_threads;
    size_t occ_smem;
    int occ;                          // resident CTAs per SM for (occ_threads, occ_smem); 0 = not asked yet
};
constexpr int kMaxKernelCfg = 96;

struct Ctx {
    lwe_params p;
    ModQ mq;
    int device;
    int sm_count;
    int smem_optin;                   // cudaDevAttrMaxSharedMemoryPerBlockOptin of the device
    KernelCfg kcfg[kMaxKernelCfg];
    int n_kcfg;
    int last_cuda_error;
    uint64_t launches;
    int encaps_path;                  // LWE_OPT_ENCAPS_PATH
    int keygen_path;                  // LWE_OPT_KEYGEN_PATH
    int regen_path;                   // LWE_OPT_REGEN_PATH
    int r_operand;                    // LWE_OPT_R_OPERAND
    int v_path;                       // LWE_OPT_V_PATH
    int no_pdl;                       // LWE_OPT_PDL = 0: programmatic dependent launch off

    // device tables
    uint32_t *d_te0;                  // 256-entry AES T-table (word = 2S | S<<8 | S<<16 | 3S<<24)

    // workspace (allocated once in lwe_create)
    uint8_t *d_Rexp;                  // [m][max_batch*k] u8 in {0,1}: B operand of the encaps GEMM
    uint8_t *d_Sx;                    // [4*max_batch rounded to 16][2n] u8: B operand of the batched keygen GEMM
    uint16_t *d_Apanel;               // [panel_rows][n]: one row panel of a regenerated A (encaps with d_A == NULL)
    uint32_t panel_rows;              // rows per panel in use (LWE_OPT_PANEL_ROWS), <= panel_rows_alloc
    uint32_t panel_rows_alloc;        // multiple of 128 (or m if smaller): panel_rows_alloc * n * 2 <= ~64 MiB
    unsigned long long *d_vacc;       // [max_batch*k] u64 partial sums of b^T R
    unsigned long long *d_dacc;       // [max_batch*k] u64 partial sums of U^T s
    unsigned int *d_counters;         // [8 + max_batch] self-resetting "last block" tickets
    uint32_t *d_foflags;              // [max_batch] mismatch flags of the FO re-encryption check
    uint16_t *d_vprime;               // [max_batch][k] re-encrypted v'
    uint32_t *d_tile_locks;           // [2 * n/64] per-tile lock + arrival count of the fused regenerated-A encaps
    // wide contexts (q > 65536: Table 1's q = 65537 rows): the public matrix held by the context, packed by
    // lwe_wide_load_matrix -- its low 16 bits as a uint16 matrix the tensor kernels read exactly like a narrow A, and the
    // few elements >= 2^16 as per-column and per-row exception lists (slot lists of fixed capacity)
    uint32_t wide;                    // 1 if q > 65536
    uint32_t A_loaded;                // lwe_wide_load_matrix has completed on this context
    uint16_t *d_A16;                  // [m][n] low 16 bits of A
    uint32_t exc_cap_col, exc_cap_row;// slots per column / per row
    uint32_t *d_exc_col_cnt;          // [n] elements >= 2^16 in column j (may exceed the capacity: overflow)
    uint32_t *d_exc_col_rows;         // [n][exc_cap_col] their row indices
    uint32_t *d_exc_row_cnt;          // [m]
    uint32_t *d_exc_row_cols;         // [m][exc_cap_row] their column indices
    uint32_t *d_exc_overflow;         // [1] set by the pack kernel when a slot list is full
    uint32_t *h_exc_overflow;         // pinned host copy read by lwe_wide_load_matrix
    // staging for lwe_kem_host
    uint16_t *d_hs, *d_he, *d_hb, *d_hU, *d_hv;
    uint8_t *d_hR, *d_hmu, *d_hmuout;
    // lwe_kem_host pipeline: copy-in / copy-out streams and the events that order them against the
    // caller's compute stream, one pair per chunk of instances
    cudaStream_t s_in, s_out;
    cudaEvent_t ev_entry, ev_out, ev_se, ev_kg, ev_in[kHostChunks], ev_done[kHostChunks];

    // driver entry point for TMA descriptors (resolved at create; no link-time libcuda)
    void *encode_tiled;

    // per-kernel device timing (LWE_OPT_PROFILE): event pairs recorded around launches
    int profile;
    int n_ev;                                              // pairs used so far
    cudaEvent_t *ev;                                       // [2 * kMaxProfEvents], created lazily
    uint8_t *ev_kernel;                                    // kernel id of each pair
};

constexpr int kMaxProfEvents = 8192;

// Brackets one kernel launch with CUDA events on the launching stream when profiling is on.
struct ProfScope {
    Ctx *c;
    cudaStream_t st;
    int slot;
    ProfScope(Ctx *c_, int kernel_id, cudaStream_t st_) : c(c_), st(st_), slot(-1)
    {
        if (!c->profile || !c->ev || c->n_ev >= kMaxProfEvents) return;
        if (c->profile >= 2 && c->profile - 2 != kernel_id) return;      // only one kernel is being timed
        slot = c->n_ev++;
        c->ev_kernel[slot] = (uint8_t)kernel_id;
        cudaEventRecord(c->ev[2 * slot], st);
    }
    ~ProfScope()
    {
        if (slot >= 0) cudaEventRecord(c->ev[2 * slot + 1], st);
    }
};

#define LWE_CUDA_TRY(ctx, expr)                                   \
    do {                                                          \
        cudaError_t _e = (expr);                                  \
        if (_e != cudaSuccess) {                                  \
            (ctx)->last_cuda_error = (int)_e;                     \
            return LWE_ERR_CUDA;                                  \
        }                                                         \
    } while (0)

// Before a launch of `fn` with `smem` bytes of dynamic shared memory: on first use by this context raise the
// function's dynamic shared-memory limit on the context's device to everything the device offers (a limit, not a
// reservation: contexts of different shapes sharing the function never lower it for each other).  If `occ` is not
// NULL it receives the resident CTAs per SM for (threads, smem), queried once per distinct pair (>= 1).
cudaError_t kernel_prepare(Ctx *c, const void *fn, size_t smem, int threads = 0, int *occ = nullptr);
template <class K>
inline cudaError_t kernel_prepare(Ctx *c, K fn, size_t smem, int threads = 0, int *occ = nullptr)
{
    return kernel_prepare(c, reinterpret_cast<const void *>(fn), smem, threads, occ);
}

// Programmatic dependent launch (the paper's goal of removing sync points, carried down to kernel boundaries).
// A kernel launched through launch_k may be scheduled while its predecessor in the stream still runs: everything it
// does before pdl_wait() -- barrier initialisation, TMEM allocation, tensor-map prefetch, the AES table fill -- overlaps
// the predecessor's tail and the launch latency; pdl_wait() returns once the predecessor has completed and its memory
// is visible, and NO access to memory another kernel may write or read for writing may precede it.  pdl_trigger()
// lets the successor be scheduled as soon as every CTA of this kernel has started.  Without the launch attribute
// (LWE_OPT_PDL = 0) both are no-ops.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// CONTRACT of launch_k: it attaches programmatic stream serialisation, so a kernel launched through it may START
// before its predecessor in the stream has finished.  Such a kernel MUST call pdl_wait() before its first access to
// global memory that any other kernel writes (or that it writes and another kernel reads) -- all of them do so right
// after their prologue -- and should call pdl_trigger() early.  A kernel without pdl_wait() must be launched with plain
// <<<>>> (full stream order), never moved to launch_k.  tests/test_gpu_stress.py runs the streaming kernels back to
// back with PDL on and off on reused buffers; the test cannot prove the absence of a race, the rule above does.
template <class... KArgs, class... Args>
inline cudaError_t launch_k(Ctx *c, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args &&...args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = c->no_pdl ? 0 : 1;
    c->launches++;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

// host-side key expansion (FIPS-197 5.2) into the kernels' word convention
void aes128_expand_key_host(const uint8_t key[16], AesKey *out);
void aes_te0_host(uint32_t te0[256]);
AesKey seed_key_host(uint64_t seed);

// kernel launchers (each returns a cudaError_t from the launch) --------------------
cudaError_t launch_rng_fill(Ctx *c, uint8_t *d_out, size_t nbytes, const AesKey &key,
                            uint64_t iv_hi, uint64_t iv_lo, uint64_t byte_offset, cudaStream_t st);
cudaError_t launch_sample_uniform(Ctx *c, uint16_t *d_out, uint64_t first, uint64_t count,
                                  const AesKey &key, uint32_t tag, uint32_t inst0, uint32_t n_inst,
                                  cudaStream_t st);
cudaError_t launch_sample_cbd(Ctx *c, uint16_t *d_out, uint64_t first, uint64_t count,
                              const AesKey &key, uint32_t tag, uint32_t inst0, uint32_t n_inst,
                              cudaStream_t st);
cudaError_t launch_sample_bits(Ctx *c, uint8_t *d_out, uint64_t first_bit, uint64_t nbits,
                               const AesKey &key, uint32_t tag, uint32_t inst0, uint32_t n_inst,
                               cudaStream_t st);
cudaError_t launch_sample_kem(Ctx *c, uint16_t *d_s, uint16_t *d_e, uint8_t *d_Rbits, uint8_t *d_mubits, const AesKey &key,
                              uint32_t inst0, uint32_t n_inst, cudaStream_t st);
cudaError_t launch_keygen_stored(Ctx *c, const uint16_t *d_A, const uint16_t *d_s, const uint16_t *d_e,
                                 uint16_t *d_b, uint32_t batch, cudaStream_t st);
size_t keygen_tc_workspace_bytes(const lwe_params &p);
bool keygen_tc_supported(const Ctx *c, uint32_t batch);
cudaError_t launch_keygen_tc(Ctx *c, const uint16_t *d_A, const uint16_t *d_s, const uint16_t *d_e, uint16_t *d_b,
                             uint32_t batch, cudaStream_t st);
cudaError_t launch_keygen_regen(Ctx *c, const AesKey &key, const uint16_t *d_s, const uint16_t *d_e,
                                uint16_t *d_b, uint32_t batch, cudaStream_t st);
cudaError_t launch_expand_R_and_v(Ctx *c, const uint16_t *d_b, const uint8_t *d_Rbits,
                                  const uint8_t *d_mubits, uint16_t *d_v, uint32_t batch,
                                  bool write_Rexp, cudaStream_t st);
// The three U = A^T R kernels take a ROW PANEL of A: d_A holds rows [row0, row0 + rows) of the m-row matrix
// (row0 = 0, rows = m for a stored A).  mode (EpiMode in tc_common.cuh): 0 = store U; 1 = add the residues
// already in d_U (panels after the first when A is regenerated panel by panel); 2 = write nothing, compare with
// d_U and OR a mismatch into d_flags[instance] (FO re-encryption check).
cudaError_t launch_encaps_simt(Ctx *c, const uint16_t *d_A, const uint8_t *d_Rbits, uint16_t *d_U,
                               uint32_t batch, uint32_t row0, uint32_t rows, int mode, uint32_t *d_flags, cudaStream_t st);
bool encaps_tc_supported(const Ctx *c, uint32_t batch);
cudaError_t launch_encaps_tc(Ctx *c, const uint16_t *d_A, uint16_t *d_U, uint32_t batch, uint32_t row0,
                             uint32_t rows, int mode, uint32_t *d_flags, cudaStream_t st);
bool encaps_tc2_supported(const Ctx *c, uint32_t batch);
// N4: A regenerated inside the GEMM's producer (one instance), encaps_regen_tc.cu
uint32_t encaps_regen_lock_words(const lwe_params &p);
bool encaps_regen_tc_supported(const Ctx *c, uint32_t batch);
cudaError_t launch_encaps_regen_tc(Ctx *c, const AesKey &key, uint16_t *d_U, cudaStream_t st);
// d_Rbits != NULL: the B operand is expanded from the packed bits inside the kernel (needs
// encaps_tc2_bits_supported); NULL: it is read from the expanded workspace c->d_Rexp.
// d_b != NULL (with d_Rbits; needs encaps_tc2_v_fused_supported): v = b^T R + mu floor(q/2) of all m rows is computed
// by spare warps of the same kernel and written to d_v (no separate pass over R's bits)
bool encaps_tc2_bits_supported(const Ctx *c, uint32_t batch);
bool encaps_tc2_v_fused_supported(const Ctx *c, uint32_t batch);
cudaError_t launch_encaps_tc2(Ctx *c, const uint16_t *d_A, uint16_t *d_U, uint32_t batch, uint32_t row0,
                              uint32_t rows, int mode, uint32_t *d_flags, cudaStream_t st,
                              const uint8_t *d_Rbits = nullptr, const uint16_t *d_b = nullptr,
                              const uint8_t *d_mubits = nullptr, uint16_t *d_v = nullptr);
// N2 (the paper's own PKE variant)
cudaError_t launch_sample_gauss(Ctx *c, void *d_out, bool as_u16, uint64_t first, uint64_t count, const AesKey &key,
                                uint32_t tag, uint32_t inst0, uint32_t n_inst, double sigma, cudaStream_t st);
cudaError_t launch_sample_pke(Ctx *c, void *d_s, void *d_e, int8_t *d_R, int8_t *d_E1, int8_t *d_e2, uint8_t *d_mubits,
                              const AesKey &key, uint32_t inst0, uint32_t n_inst, double sigma, uint32_t bound, cudaStream_t st);
cudaError_t launch_sample_cuniform(Ctx *c, int8_t *d_out, uint64_t first, uint64_t count, const AesKey &key, uint32_t tag,
                                   uint32_t inst0, uint32_t n_inst, uint32_t bound, cudaStream_t st);
cudaError_t launch_prep_R_pv_and_v(Ctx *c, const uint16_t *d_t, const int8_t *d_R, const int8_t *d_e2,
                                   const uint8_t *d_mubits, uint16_t *d_v, uint32_t batch, bool write_Rexp, cudaStream_t st);
// v alone for the int8 R (no operand copy), as a 16-byte-per-thread stream; wide: t, v are uint32 (else uint16)
bool pv_v_stream_supported(const Ctx *c);
cudaError_t launch_pv_v_stream(Ctx *c, const void *d_t, bool wide, const int8_t *d_R, const int8_t *d_e2, const uint8_t *d_mubits,
                               void *d_v, uint32_t batch, cudaStream_t st);
// d_R != NULL (needs k % 128 == 0): the B operand is read in place from the caller's int8 R [batch][m][k]; NULL: from
// the operand copy in c->d_Rexp
bool encaps_tc2_r_inplace_supported(const Ctx *c, uint32_t batch);
cudaError_t launch_encaps_tc2_pv(Ctx *c, const uint16_t *d_A, const int8_t *d_E1, uint16_t *d_U, uint32_t batch,
                                 cudaStream_t st, const int8_t *d_R = nullptr);
cudaError_t launch_encaps_pv_simt(Ctx *c, const uint16_t *d_A, const int8_t *d_R, const int8_t *d_E1, uint16_t *d_U,
                                  uint32_t batch, cudaStream_t st);
// wide path (q > 65536), wide.cu / rng_kernels.cu / keygen_tc.cu / encaps_tc2.cu
cudaError_t launch_sample_uniform32(Ctx *c, uint32_t *d_out, uint64_t first, uint64_t count, const AesKey &key, uint32_t tag,
                                    uint32_t inst0, uint32_t n_inst, cudaStream_t st);
cudaError_t launch_sample_cbd_s8(Ctx *c, int8_t *d_out, uint64_t first, uint64_t count, const AesKey &key, uint32_t tag,
                                 uint32_t inst0, uint32_t n_inst, cudaStream_t st);
cudaError_t launch_wide_pack(Ctx *c, const uint32_t *d_A, uint32_t row0, uint32_t rows, cudaStream_t st);
cudaError_t launch_wide_keygen_simt(Ctx *c, const int8_t *d_s, const int8_t *d_e, uint32_t *d_t, uint32_t batch, cudaStream_t st);
bool wide_keygen_tc_supported(const Ctx *c, uint32_t batch);
cudaError_t launch_wide_keygen_tc(Ctx *c, const int8_t *d_s, const int8_t *d_e, uint32_t *d_t, uint32_t batch, cudaStream_t st);
cudaError_t launch_wide_v(Ctx *c, const uint32_t *d_t, const int8_t *d_R, const int8_t *d_e2, const uint8_t *d_mubits,
                          uint32_t *d_v, uint32_t batch, bool write_Rexp, cudaStream_t st);
cudaError_t launch_wide_encaps_simt(Ctx *c, const int8_t *d_R, const int8_t *d_E1, uint32_t *d_U, uint32_t batch, cudaStream_t st);
cudaError_t launch_wide_encaps_tc2(Ctx *c, const int8_t *d_R, const int8_t *d_E1, uint32_t *d_U, uint32_t batch, cudaStream_t st);
cudaError_t launch_wide_decaps(Ctx *c, const uint32_t *d_U, const uint32_t *d_v, const int8_t *d_s, uint8_t *d_out,
                               uint32_t batch, cudaStream_t st);
cudaError_t launch_fo_verdict(Ctx *c, const uint16_t *d_v, const uint16_t *d_vprime, const uint32_t *d_flags,
                              uint8_t *d_ok, uint32_t batch, cudaStream_t st);
// measurement hook (probe_int8.cu): back-to-back tcgen05.mma kind::i8 on shared-memory-resident operands
cudaError_t launch_probe_int8(Ctx *c, uint32_t iters, int signed_dense_b, uint64_t *ops, cudaStream_t st);
cudaError_t launch_decaps(Ctx *c, const uint16_t *d_U, const uint16_t *d_v, const uint16_t *d_s,
                          uint8_t *d_out, uint32_t batch, cudaStream_t st);

}  // namespace lwe

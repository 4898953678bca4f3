/*
 * lwe.h -- C ABI of liblwe_b200: the data-parallel core of the plain-LWE KEM of
 * arxiv/paper_2606_01211, written for one NVIDIA B200 (sm_100a).
 *
 * Citations: P:Lnnn = PAPER.md line nnn; BJ = BASELINE.json; S8(x) = SURVEY.md
 * section 8(x); DESIGN.md section 3 = the readings taken where the paper is silent.
 *
 * Notation (S8): A in Z_q^{m x n} row-major uint16; s in Z_q^n; e, b in Z_q^m;
 * R in {0,1}^{m x k}; mu in {0,1}^k; U in Z_q^{n x k} row-major uint16; v in Z_q^k.
 * All vectors hold canonical representatives in [0, q).  Everything is integer
 * arithmetic; results are exact, so they do not depend on launch geometry.
 *
 * Conventions for every entry point
 *  - Pointers named d_* are DEVICE pointers (device of the context), caller-owned;
 *    h_* are HOST pointers (pinned memory recommended).  The library never frees or
 *    keeps them beyond the stream work it enqueues.  Inputs are never modified.
 *  - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *    Calls with d_* arguments only ENQUEUE work and return; they never synchronise
 *    the host (the paper's goal of removing sync points).
 *  - The context owns one workspace sized at creation from (m, k, max_batch); no
 *    call allocates ("allocate once").  A context must not be used from two
 *    streams at the same time.
 *  - Return value: LWE_OK or a negative lwe_status.  Arguments are validated before
 *    anything is launched: on an error nothing has been written.  No C++ exception
 *    crosses the ABI; nothing aborts.
 *  - Alignment: every d_* / h_* pointer must be 16-byte aligned (LWE_ERR_ALIGN).
 *  - There is no CPU fallback and no other backend: a device that is not compute
 *    capability 10.x gives LWE_ERR_UNSUPPORTED at lwe_create.
 */
#ifndef LWE_B200_H
#define LWE_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    LWE_OK = 0,
    LWE_ERR_PARAM = -1,       /* a size / modulus / range argument is invalid          */
    LWE_ERR_ALIGN = -2,       /* a pointer or offset violates the alignment contract    */
    LWE_ERR_NULLPTR = -3,     /* a required pointer is NULL                             */
    LWE_ERR_CUDA = -4,        /* the CUDA runtime reported an error (see lwe_last_cuda_error) */
    LWE_ERR_UNSUPPORTED = -5  /* not an sm_100 device, or a variant that is not built   */
} lwe_status;

/* Object tags of the seeded streams (S8(c) O3). */
enum { LWE_TAG_A = 1, LWE_TAG_S = 2, LWE_TAG_E = 3, LWE_TAG_R = 4, LWE_TAG_MU = 5,
       LWE_TAG_RG = 6, LWE_TAG_E1 = 7, LWE_TAG_E2 = 8 /* N2: Gaussian r, e1; centred-uniform e2 */ };

/* Problem shape.  n, m multiples of 8 (one AES block = 8 elements); k multiple of 8;
 * q in (1, 65536]; eta in [1, 8]; max_batch >= 1 = the largest `batch` any call
 * will pass (number of independent instances sharing one A, BJ configs[3]). */
typedef struct {
    uint32_t n, m, k, q, eta, max_batch;
} lwe_params;

typedef struct lwe_ctx lwe_ctx; /* opaque: tables, workspace, TMA descriptors */

/* Create / destroy a context on CUDA device `device`.  Allocates the workspace
 * (m*k*max_batch bytes for the expanded R operand, one row panel of A of at most
 * 64 MiB for the regenerated-A encaps, small accumulators, lwe_kem_host staging). */
int lwe_create(lwe_ctx **ctx, const lwe_params *p, int device);
void lwe_destroy(lwe_ctx *ctx);

const char *lwe_strerror(int code);
/* cudaError_t of the last LWE_ERR_CUDA on this context (0 if none). */
int lwe_last_cuda_error(const lwe_ctx *ctx);
/* Number of kernels this context has launched since creation (bench's gpu_launches). */
uint64_t lwe_launch_count(const lwe_ctx *ctx);

/* ---- a1: device-resident AES-128-CTR stream --------------------------------------
 * d_out[x] = byte (byte_offset + x) of KS(key, iv), 0 <= x < nbytes, where block j of
 * KS is AES-128_key((iv + j) mod 2^128), iv and the sum being 128-bit big-endian
 * integers (SP 800-38A CTR; equals `openssl aes-128-ctr` keystream).  Any offset is
 * reproducible: the result is a pure function of (key, iv, byte position).
 * P:L154-156 (device RNG, identical sequences on every GPU, one sub-seed per output
 * element); BJ north_star (1).  key, iv: HOST pointers, read before returning.
 * byte_offset and nbytes are arbitrary; d_out needs 16-byte alignment. */
int lwe_rng_fill(lwe_ctx *ctx, void *d_out, size_t nbytes, const uint8_t key[16],
                 const uint8_t iv[16], uint64_t byte_offset, void *stream);

/* ---- a2: samplers over the seeded streams (S8(c) O3-O6) --------------------------
 * Stream of object (seed, tag, attempt, inst): key = LE64(seed) || 0^8,
 * iv = BE64(tag*2^56 + attempt*2^32 + inst) || 0^8.  P:L154 (64-bit master seed).
 * Each call fills n_inst consecutive instances inst0 .. inst0+n_inst-1:
 * d_out[t][x] for instance inst0+t, element first+x; rows are `count` elements apart.
 *
 * uniform: element e: for attempt a = 0,1,..: c = LE16(stream bytes [2e, 2e+1] of
 *   attempt a); T = q*floor(65536/q); accept iff c < T; value c mod q.  Exactly
 *   uniform and O(1) random access.  BJ configs[2] ("uniform mod q by rejection").
 * cbd: w = LE16(stream bytes [2e,2e+1], attempt 0); x = popcount(w & M) -
 *   popcount((w >> 8) & M), M = 2^eta - 1; stored as x mod q.  P:L70.
 * bits: bit t of the stream = (byte floor(t/8) >> (t mod 8)) & 1; output packed the
 *   same way, ceil(nbits/8) bytes per instance, unused top bits zero.  first_bit must
 *   be a multiple of 8 (LWE_ERR_ALIGN).  P:L78 Alg.4 l.1; BJ configs (binary R).
 * `first` must be a multiple of 8 for uniform/cbd (one AES block = 8 elements). */
int lwe_sample_uniform(lwe_ctx *ctx, uint16_t *d_out, uint64_t first, uint64_t count,
                       uint64_t seed, uint32_t tag, uint32_t inst0, uint32_t n_inst, void *stream);
int lwe_sample_cbd(lwe_ctx *ctx, uint16_t *d_out, uint64_t first, uint64_t count,
                   uint64_t seed, uint32_t tag, uint32_t inst0, uint32_t n_inst, void *stream);
int lwe_sample_bits(lwe_ctx *ctx, uint8_t *d_out, uint64_t first_bit, uint64_t nbits,
                    uint64_t seed, uint32_t tag, uint32_t inst0, uint32_t n_inst, void *stream);

/* The four per-instance objects of n_inst KEM instances in ONE launch: exactly what
 *   lwe_sample_uniform(d_s, 0, n, seed, LWE_TAG_S, inst0, n_inst) + lwe_sample_cbd(d_e, 0, m, seed, LWE_TAG_E, ..)
 *   + lwe_sample_bits(d_Rbits, 0, m*k, seed, LWE_TAG_R, ..) + lwe_sample_bits(d_mubits, 0, k, seed, LWE_TAG_MU, ..)
 * write (n, m, k, q, eta of the context).  d_s [n_inst][n], d_e [n_inst][m], d_Rbits [n_inst][m*k/8],
 * d_mubits [n_inst][k/8].  No new semantics: it saves three kernel launches per batch ("only a seed crosses the
 * bus"). */
int lwe_sample_kem(lwe_ctx *ctx, uint16_t *d_s, uint16_t *d_e, uint8_t *d_Rbits, uint8_t *d_mubits, uint64_t seed,
                   uint32_t inst0, uint32_t n_inst, void *stream);

/* ---- a3 / a3': KeyGen ------------------------------------------------------------
 * d_b[t][i] = ( sum_{j<n} A[i][j] * d_s[t][j] + d_e[t][i] ) mod q,  0 <= t < batch.
 * P:L60 eq.(1).  d_A: m x n row-major, streamed from HBM: once per call for
 * batch >= 2 (all instances in one tensor-core GEMM, "many concurrent key
 * exchanges"), as one HBM-bound GEMV for batch 1.  d_A == NULL: A is never read; every element is regenerated
 * inside the kernel from (seed_A, LWE_TAG_A, inst 0) exactly as lwe_sample_uniform
 * would produce it (the paper's on-demand A).  batch <= max_batch. */
int lwe_keygen(lwe_ctx *ctx, const uint16_t *d_A, uint64_t seed_A,
               const uint16_t *d_s /*[batch][n]*/, const uint16_t *d_e /*[batch][m]*/,
               uint16_t *d_b /*[batch][m]*/, uint32_t batch, void *stream);

/* ---- a4 + a5: Encaps, all k bits of an instance in one contraction -----------------
 * d_U[t][j][c] = ( sum_{i<m} A[i][j] * R_t[i][c] ) mod q
 * d_v[t][c]    = ( sum_{i<m} d_b[t][i] * R_t[i][c] + mu_t[c]*floor(q/2) ) mod q
 * with R_t[i][c] = bit (i*k + c) of d_Rbits[t] and mu_t[c] = bit c of d_mubits[t]
 * (LSB-first).  Intra-operation batching, P:L130 item 3.
 * Runs as a u8 x u8 -> s32 tensor-core GEMM (tcgen05 kind::i8) over the byte planes
 * of A with a mod-q recombine epilogue; shapes the tensor path does not cover
 * (k % 16 != 0) use a CUDA-core kernel with identical results.
 * d_A == NULL: A is never read and never held in full: it is regenerated from
 * (seed_A, LWE_TAG_A, inst 0) one ROW PANEL at a time (rows of A are contiguous ranges
 * of the counter-indexed stream; a panel is <= 64 MiB of context workspace) and the
 * contraction is accumulated over the panels -- same U, bit for bit (
 * BJ configs[4] "stored and regenerated"). */
int lwe_encaps(lwe_ctx *ctx, const uint16_t *d_A, uint64_t seed_A,
               const uint16_t *d_b /*[batch][m]*/, const uint8_t *d_Rbits /*[batch][m*k/8]*/,
               const uint8_t *d_mubits /*[batch][k/8]*/, uint16_t *d_U /*[batch][n][k]*/,
               uint16_t *d_v /*[batch][k]*/, uint32_t batch, void *stream);

/* ---- a6: Decaps ------------------------------------------------------------------
 * d = ( d_v[t][c] - sum_{j<n} d_U[t][j][c] * d_s[t][j] ) mod q in [0,q);
 * bit = floor((4d + q) / (2q)) mod 2  (1 iff q/4 <= d < 3q/4); packed LSB-first into
 * d_mubits_out[t][k/8].  P:L174 ("mu = v - s.u (mod q)"), P:L68 (decoding threshold). */
int lwe_decaps(lwe_ctx *ctx, const uint16_t *d_U, const uint16_t *d_v, const uint16_t *d_s,
               uint8_t *d_mubits_out /*[batch][k/8]*/, uint32_t batch, void *stream);

/* ---- N3 (S8(f)): Decaps with the FO re-encryption check -----------------------------
 * Alg. 5 of the paper without its hashes: (1) m' = Decrypt(sk, c) exactly as
 * lwe_decaps, written to d_mubits_out; (2) c' = Encrypt(pk, m') with the re-derived coins d_Rbits
 * (the caller derives them as it did for Encaps -- in the paper through hashes that are outside this
 * library; in bench.py from (seed, LWE_TAG_R, inst)); (4) d_ok[t] = 1 iff c' == c, i.e. U' == U and
 * v' == v, else 0 (the caller then selects K or the implicit-rejection key, Alg. 5 l.5-7).
 * The verdict is formed on the device: c' is never materialised (U' is compared with d_U tile by tile
 * in the epilogue of the tensor-core GEMM, v' lives in the workspace) and nothing returns to the host
 * before it (the paper's decaps crosses the bus here).  The work done does not depend on
 * whether the ciphertext is valid.  d_A must be stored (NULL: LWE_ERR_NULLPTR).  d_ok: batch bytes. */
int lwe_decaps_fo(lwe_ctx *ctx, const uint16_t *d_A, const uint16_t *d_b /*[batch][m]*/,
                  const uint16_t *d_U /*[batch][n][k]*/, const uint16_t *d_v /*[batch][k]*/,
                  const uint16_t *d_s /*[batch][n]*/, const uint8_t *d_Rbits /*[batch][m*k/8]*/,
                  uint8_t *d_mubits_out /*[batch][k/8]*/, uint8_t *d_ok /*[batch]*/, uint32_t batch, void *stream);

/* ---- N2 (S8(f)): the paper's own PKE variant ------------------------------------------
 * P:L64 (KeyGen / Encrypt / Decrypt; Fig. 1 is an image whose text is lost), P:L70 (secret: binomial
 * eta = 3), Table 1 header P:L92 (Gaussian sigma for e, r, e1; centred uniform k for e2).  Readings
 * S20-S22 of DESIGN.md section 3.  With a context whose m = n (square A) and eta = 3:
 *   KeyGen : s = lwe_sample_cbd (tag S), e = lwe_sample_gauss_u16 (tag E), t = lwe_keygen(A, s, e)
 *   Encrypt: R = lwe_sample_gauss_s8 (tag RG, m*k per instance), E1 = lwe_sample_gauss_s8 (tag E1, n*k),
 *            e2 = lwe_sample_cuniform_s8 (tag E2, k), then lwe_encaps_pv
 *   Decrypt: lwe_decaps.
 * Moduli of Table 1 that fit uint16 (3329, 12289) are supported; 65537 needs a 17-bit residue type and is not.
 *
 * gauss: element e -> 16-bit stream word w as for cbd; z = -12 + #{ j : w >= C[j] } with the cumulative table
 *   C[j] = floor(65536 * Phi((j - 12 + 1/2) / sigma) + 1/2), j = 0..23, Phi(x) = erfc(-x / sqrt 2) / 2 evaluated in
 *   double on the host: the rounded Gaussian round(sigma N(0,1)) to 2^-16 per value.  0.5 <= sigma <= 8.
 *   _s8 stores z as int8, _u16 stores z mod q.  `first` multiple of 8.
 * cuniform: centred uniform on [-bound, bound], 1 <= bound <= 127: the rejection rule of uniform with modulus
 *   2*bound + 1 over the attempt streams, value (c mod (2 bound + 1)) - bound.  Any `first`. */
int lwe_sample_gauss_s8(lwe_ctx *ctx, int8_t *d_out, uint64_t first, uint64_t count, uint64_t seed, uint32_t tag,
                        uint32_t inst0, uint32_t n_inst, double sigma, void *stream);
int lwe_sample_gauss_u16(lwe_ctx *ctx, uint16_t *d_out, uint64_t first, uint64_t count, uint64_t seed, uint32_t tag,
                         uint32_t inst0, uint32_t n_inst, double sigma, void *stream);
int lwe_sample_cuniform_s8(lwe_ctx *ctx, int8_t *d_out, uint64_t first, uint64_t count, uint64_t seed, uint32_t tag,
                           uint32_t inst0, uint32_t n_inst, uint32_t bound, void *stream);
/* d_U[t][j][c] = ( sum_{i<m} A[i][j] * R_t[i][c] + E1_t[j][c] ) mod q
 * d_v[t][c]    = ( sum_{i<m} d_t[t][i] * R_t[i][c] + e2_t[c] + mu_t[c]*floor(q/2) ) mod q
 * with R_t = d_R[t] (int8 [m][k]), E1_t = d_E1[t] (int8 [n][k]), e2_t = d_e2[t] (int8 [k]).  Same tcgen05 kind::i8
 * GEMM as lwe_encaps with the B operand read as SIGNED int8 (no bit expansion: R is copied once into the operand
 * layout), signed byte-plane accumulators and E1 added in the recombine epilogue; |R| <= 127, m <= 65536.
 * d_A must be stored.  Shapes the tensor path does not take run on CUDA cores with identical results. */
int lwe_encaps_pv(lwe_ctx *ctx, const uint16_t *d_A, const uint16_t *d_t /*[batch][m]*/,
                  const int8_t *d_R /*[batch][m][k]*/, const int8_t *d_E1 /*[batch][n][k]*/,
                  const int8_t *d_e2 /*[batch][k]*/, const uint8_t *d_mubits /*[batch][k/8]*/,
                  uint16_t *d_U /*[batch][n][k]*/, uint16_t *d_v /*[batch][k]*/, uint32_t batch, void *stream);

/* ---- end-to-end with HOST buffers -----------------------------------------------
 * One full pass keygen -> encaps -> decaps for `batch` instances whose per-instance
 * inputs live in host memory: copies h_s, h_e, h_Rbits, h_mubits to the device,
 * runs the three steps against the device-resident public matrix d_A (or A regenerated
 * from seed_A if d_A == NULL), copies h_b, h_v, h_mubits_out (and h_U if not NULL) back,
 * and returns after synchronising `stream`.  Layouts as in the calls above. */
int lwe_kem_host(lwe_ctx *ctx, const uint16_t *d_A, uint64_t seed_A,
                 const uint16_t *h_s, const uint16_t *h_e, const uint8_t *h_Rbits,
                 const uint8_t *h_mubits, uint16_t *h_b, uint16_t *h_U /* may be NULL */,
                 uint16_t *h_v, uint8_t *h_mubits_out, uint32_t batch, void *stream);

/* ---- tuning / test / measurement hooks (no new semantics) --------------------------
 * LWE_OPT_ENCAPS_PATH: 0 = auto (tcgen05 GEMM on CTA pairs where the shape fits, else CUDA cores),
 *                      1 = force the CUDA-core kernel, 2 = force the single-CTA tcgen05 GEMM
 *                      (cta_group::1), 3 = force the CTA-pair tcgen05 GEMM (cta_group::2);
 *                      2 / 3 give LWE_ERR_UNSUPPORTED at call time if the shape does not fit.
 * LWE_OPT_PROFILE:     1 = bracket every kernel launch with a CUDA event pair on the
 *                      stream it is launched on (at most 8192 launches are kept between
 *                      resets; later ones are simply not timed); 2 + id = only launches of kernel LWE_K_<id>
 *                      (one pair per launch of that kernel, nothing around the others); 0 = off (default).
 * LWE_OPT_GEMV_VARIANT: keygen GEMV launch shape, 0 = auto; 1/2 = a warp per row with 4/8 loads in
 *                      flight per lane; 3/4 = a CTA per row with 4/2 loads per thread.  With A regenerated
 *                      (d_A == NULL) 1-4 select CTA size / AES blocks in flight instead.  Same result.
 * LWE_OPT_KEYGEN_PATH: stored-A keygen, 0 = auto (GEMV for batch 1, tensor-core skinny GEMM that reads A
 *                      once for batch >= 2), 1 = force one GEMV per instance, 2 = force the tcgen05 GEMM
 *                      (LWE_ERR_UNSUPPORTED if n > 32768 or the batch needs more than 256 operand columns:
 *                      2 per instance when q divides 2^16, else 3 for n <= 16384, else 4).
 * LWE_OPT_TUNE:        launch-shape knob of the tensor-core kernels for measurements (tile order, L2
 *                      eviction policy of the operand streams, ring depth); 0 = default.  Same result
 *                      for every value.
 * LWE_OPT_PANEL_ROWS:  rows of A regenerated per panel by lwe_encaps(d_A == NULL): a multiple of 8 in
 *                      [8, default]; 0 = default (<= 64 MiB of A per panel, a multiple of 128 rows).  Same
 *                      result for every value (tests use it to cross many panels at small sizes).
 * LWE_OPT_R_OPERAND:   how the CTA-pair GEMM gets its B operand, 0 = auto (k % 128 == 0: expanded from the packed bits of
 *                      R inside the kernel, nothing is written to HBM; otherwise from the expanded workspace),
 *                      1 = always expand R to a u8 matrix in the workspace first.  Same result for every value.
 * LWE_OPT_REGEN_PATH:  lwe_encaps(d_A == NULL), 0 = auto (one instance with k <= 256: A tiles generated straight into
 *                      the GEMM's shared-memory operand, A never touches HBM -- S8(f) N4; otherwise row panels),
 *                      1 = always row panels, 2 = force the fused kernel (LWE_ERR_UNSUPPORTED if batch > 1 or
 *                      k > 256 or the tensor path does not take the shape).  Same result for every value. */
enum { LWE_OPT_ENCAPS_PATH = 1, LWE_OPT_PROFILE = 2, LWE_OPT_GEMV_VARIANT = 3, LWE_OPT_KEYGEN_PATH = 4, LWE_OPT_TUNE = 5,
       LWE_OPT_PANEL_ROWS = 6, LWE_OPT_REGEN_PATH = 7, LWE_OPT_R_OPERAND = 8 };
int lwe_set_option(lwe_ctx *ctx, int option, int64_t value);

/* Kernel ids for lwe_profile_read (one per __global__ function of the library). */
enum {
    LWE_K_RNG_FILL = 0, LWE_K_SAMPLE_UNIFORM = 1, LWE_K_SAMPLE_CBD = 2, LWE_K_SAMPLE_BITS = 3,
    LWE_K_KEYGEN_STORED = 4, LWE_K_KEYGEN_REGEN = 5, LWE_K_EXPAND_R_V = 6, LWE_K_ENCAPS_TC = 7,
    LWE_K_ENCAPS_SIMT = 8, LWE_K_DECAPS = 9, LWE_K_KEYGEN_PREP = 10, LWE_K_KEYGEN_TC = 11, LWE_K_FO_VERDICT = 12,
    LWE_K_SAMPLE_GAUSS = 13, LWE_K_SAMPLE_CUNIFORM = 14, LWE_K_PREP_R_PV = 15, LWE_K_ENCAPS_REGEN_TC = 16, LWE_K_SAMPLE_KEM = 17, LWE_K_COUNT = 18
};
/* Sum of the device durations (milliseconds, CUDA events) and the number of timed launches
 * of kernel `kernel_id` since the last reset.  Waits for the recorded events to complete
 * (host synchronisation: call it outside any timed region).  h_total_ms / h_launches: HOST
 * pointers, either may be NULL.  lwe_profile_reset forgets all recorded pairs. */
int lwe_profile_read(lwe_ctx *ctx, int kernel_id, double *h_total_ms, uint64_t *h_launches);
int lwe_profile_reset(lwe_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* LWE_B200_H */

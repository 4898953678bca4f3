/*
 * lwe_oracle.h -- ORACLE. Test infrastructure, not the product.
 *
 * A plain, slow, obviously-correct CPU restatement of what the hot path of
 * arxiv/paper_2606_01211 ("GPU Acceleration of Learning With Errors KEMs Using
 * OpenACC") computes, in the Regev-style form BASELINE.json fixes.  It is the
 * definition written out: one `% q` after every multiply-add, byte-oriented
 * FIPS-197 AES, no tables shared with, and no code shared with, the CUDA path
 * under paper_2606_01211_b200/.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * Citations: P:Lnnn = /root/reference/PAPER.md line nnn; S8(c) Ok = SURVEY.md
 * section 8(c) definition Ok; BJ = BASELINE.json.  DESIGN.md section 3 lists every
 * reading taken where the paper is silent.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): FIPS-197 App. B / C.1 and
 * SP 800-38A F.5.1 known answers, 64-bit carry in the counter, an independent
 * AES (python `cryptography`/OpenSSL), closed-form CBD pmf, exhaustive rounding,
 * brute force with python big integers, linearity, unit-vector / one-hot
 * special cases, the noise identity  v - U^T s - mu*floor(q/2) = e^T R  and
 * decaps(encaps(mu)) == mu.  No function here is "parity unpinned"; the
 * conventions O3-O6 (seed->key, tags, bit order) are fixed by SURVEY 8(c) /
 * DESIGN.md and implemented twice, independently, here and in CUDA.
 *
 * All vectors hold canonical representatives in [0, q) as uint16_t (S13), q in (1, 65536]
 * (uint32_t and q < 2^31 in the *_w / *32 functions of the q = 65537 parameter sets, S23).
 * Everything is integer arithmetic.
 */
#ifndef LWE_ORACLE_H
#define LWE_ORACLE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Object tags of O3: which seeded object a stream belongs to. */
enum { ORC_TAG_A = 1, ORC_TAG_S = 2, ORC_TAG_E = 3, ORC_TAG_R = 4, ORC_TAG_MU = 5 };

/* O1. AES-128 block cipher, FIPS-197 (10 rounds). P:L154 (AES-based generator),
 * BJ north_star (1) (AES-128-CTR). */
void orc_aes128_encrypt_block(const uint8_t key[16], const uint8_t in[16], uint8_t out[16]);

/* O2. CTR keystream, SP 800-38A: block j = AES_key((iv + j) mod 2^128), iv and the
 * sum being 128-bit big-endian integers; out[x] = byte (byte_offset + x) of the
 * concatenated blocks. P:L154-156 ("identical sequences", "one sub-seed per output
 * element"); BJ north_star ("counter-indexed so any stream offset is reproducible"). */
void orc_ctr_bytes(const uint8_t key[16], const uint8_t iv[16],
                   uint64_t byte_offset, size_t nbytes, uint8_t *out);

/* O3. key(seed) = LE64(seed) || 0^8 ; iv(tag, attempt, inst) =
 * BE64(tag*2^56 + attempt*2^32 + inst) || 0^8.  P:L154 (64-bit master seed). */
void orc_seed_key(uint64_t seed, uint8_t key[16]);
void orc_object_iv(uint32_t tag, uint32_t attempt, uint32_t inst, uint8_t iv[16]);

/* O4. Uniform mod q by rejection, element t in [first, first+count):
 * for attempt a = 0,1,..: c = LE16(bytes [2t,2t+1] of KS(key(seed), iv(tag,a,inst)));
 * T = q*floor(65536/q); accept iff c < T; value c mod q.  BJ configs[2]. */
void orc_sample_uniform(uint16_t *out, uint64_t first, uint64_t count,
                        uint64_t seed, uint32_t tag, uint32_t inst, uint32_t q);

/* O4 on elements first + r*stride, 0 <= r < count (e.g. column j of the row-major m x n matrix A:
 * first = j, stride = n, count = m).  Same values orc_sample_uniform gives at those positions. */
void orc_sample_uniform_strided(uint16_t *out, uint64_t first, uint64_t stride, uint64_t count,
                                uint64_t seed, uint32_t tag, uint32_t inst, uint32_t q);

/* O5. Centred binomial eta in [1,8], element t: w = LE16(bytes [2t,2t+1] of
 * KS(key(seed), iv(tag,0,inst))); x = popcount(w & M) - popcount((w>>8) & M),
 * M = 2^eta - 1; stored as x mod q.  P:L70, P:L170, P:L320 (FIPS 203 CBD). */
void orc_sample_cbd(uint16_t *out, uint64_t first, uint64_t count,
                    uint64_t seed, uint32_t tag, uint32_t inst, uint32_t q, uint32_t eta);

/* O5 on one 16-bit stream word (what orc_sample_cbd applies to every word). */
uint16_t orc_cbd_from_word(uint32_t w, uint32_t q, uint32_t eta);

/* O6. Bits [first_bit, first_bit+nbits) of KS(key(seed), iv(tag,0,inst)), bit t =
 * (byte floor(t/8) >> (t mod 8)) & 1, written packed LSB-first starting at bit 0
 * of out[0].  P:L78 Alg.4 l.1; BJ configs (binary R, message bits). */
void orc_sample_bits(uint8_t *out, uint64_t first_bit, uint64_t nbits,
                     uint64_t seed, uint32_t tag, uint32_t inst);

/* O7. KeyGen: b_i = (sum_{j<n} A[i*n+j]*s[j] + e[i]) mod q, 0 <= i < m.
 * P:L60 eq.(1). */
void orc_keygen(const uint16_t *A, const uint16_t *s, const uint16_t *e, uint16_t *b,
                uint32_t m, uint32_t n, uint32_t q);

/* O8. Encaps, all k bits at once (intra-operation batching):
 * U[j*k+c] = (sum_{i<m} A[i*n+j]*R_ic) mod q ;
 * v[c]     = (sum_{i<m} b[i]*R_ic + mu_c*floor(q/2)) mod q ;
 * R_ic = bit (i*k+c) of Rbits, mu_c = bit c of mubits (LSB-first packing). */
void orc_encaps(const uint16_t *A, const uint16_t *b, const uint8_t *Rbits,
                const uint8_t *mubits, uint16_t *U, uint16_t *v,
                uint32_t m, uint32_t n, uint32_t k, uint32_t q);

/* O8 restricted to chosen rows of U (used at sizes where the full contraction is
 * impractical on a CPU): Urows[r*k+c] = U[rows[r]*k+c]. */
void orc_encaps_rows(const uint16_t *A, const uint8_t *Rbits, const uint32_t *rows,
                     uint32_t nrows, uint16_t *Urows,
                     uint32_t m, uint32_t n, uint32_t k, uint32_t q);

/* O8, v only. */
void orc_encaps_v(const uint16_t *b, const uint8_t *Rbits, const uint8_t *mubits,
                  uint16_t *v, uint32_t m, uint32_t k, uint32_t q);

/* O9. Decaps: d_c = (v[c] - sum_{j<n} U[j*k+c]*s[j]) mod q in [0,q);
 * bit_c = floor((4*d_c + q) / (2q)) mod 2; packed LSB-first into mubits_out[k/8].
 * If d_out != NULL it receives d_c.  P:L174; P:L68 ("decoding threshold"). */
void orc_decaps(const uint16_t *U, const uint16_t *v, const uint16_t *s,
                uint8_t *mubits_out, uint16_t *d_out,
                uint32_t n, uint32_t k, uint32_t q);

/* O9 rounding on one value d in [0,q): floor((4d + q)/(2q)) mod 2
 * (= 1 iff q/4 <= d < 3q/4). */
uint32_t orc_round_bit(uint32_t d, uint32_t q);

/* O11. Decaps with the FO re-encryption check, Alg. 5 lines 1, 2, 4 ("recomputes it
 * deterministically, and verifies its correctness through re-encryption"): m' = O9(U, v, s) -> mubits_out;
 * (U', v') = O8(A, b, Rbits, m'); returns 1 iff U' == U and v' == v, else 0.  The hashes of the FO transform
 * are not part of the hot path; Rbits are the re-derived encryption coins.
 * Pins: an honest ciphertext is accepted and decrypts to mu; ANY single-element change of (U, v) is rejected
 * whether or not it changes m' (tests/test_oracle_lwe.py). */
int orc_decaps_fo(const uint16_t *A, const uint16_t *b, const uint16_t *U, const uint16_t *v,
                  const uint16_t *s, const uint8_t *Rbits, uint8_t *mubits_out,
                  uint32_t m, uint32_t n, uint32_t k, uint32_t q);

/* ---- N2: the paper's own PKE variant.  P:L64 (KeyGen / Encrypt / Decrypt; Fig. 1 is an image whose
 * text is lost), P:L70 (secret ~ binomial eta = 3), Table 1 header P:L92 (Gaussian sigma for e, r, e1;
 * centred uniform k for e2).  Readings S20-S22 of DESIGN.md section 3:
 *   KeyGen  t = A s + e,  A in Z_q^{n x n}, s ~ CBD(3)^n (O5), e ~ D_sigma^n (O12)            -> O7 with m = n
 *   Encrypt (all k bits): R in Z^{n x k}, E1 in Z^{n x k} ~ D_sigma (O12), e2 in Z^k ~ U[-kappa, kappa] (O13)
 *           U = A^T R + E1,  v = t^T R + e2 + mu floor(q/2)                                  -> O14
 *   Decrypt = O9.
 * Object tags of the new streams. */
enum { ORC_TAG_RG = 6, ORC_TAG_E1 = 7, ORC_TAG_E2 = 8 };
#define ORC_GAUSS_TAU 12
#define ORC_GAUSS_CDT_LEN (2 * ORC_GAUSS_TAU)

/* O12. Rounded Gaussian z = round(sigma * N(0,1)) through a 16-bit cumulative table:
 * C[j] = floor(65536 * Phi((j - 12 + 1/2) / sigma) + 1/2), j = 0..23 (Phi = standard normal CDF, in double);
 * for the 16-bit stream word w of element t (as in O5): z = -12 + #{ j : w >= C[j] }.
 * So P(z) = (C[z+12] - C[z+11]) / 65536 with C[-1] = 0, C[24] = 65536: the rounded-Gaussian pmf
 * Phi((z+1/2)/sigma) - Phi((z-1/2)/sigma) to within 2^-16 per value.  The paper does not describe its sampler.
 * Pins: the table against an independent normal CDF and against numerical integration of the density; the
 * exhaustive histogram over all 65536 words; symmetry; mean 0 and variance sigma^2 + 1/12. */
void orc_gauss_cdt(double sigma, uint32_t cdt[ORC_GAUSS_CDT_LEN]);
int orc_gauss_from_word(uint32_t w, const uint32_t cdt[ORC_GAUSS_CDT_LEN]);
void orc_sample_gauss(int8_t *out_s8, uint16_t *out_u16, uint64_t first, uint64_t count,
                      uint64_t seed, uint32_t tag, uint32_t inst, double sigma, uint32_t q);

/* O13. Centred uniform on [-bound, bound] (Table 1 "centered uniform k (e2)"): O4's rejection rule with modulus
 * q' = 2*bound + 1 over the attempt streams, value (c mod q') - bound. */
void orc_sample_cuniform(int8_t *out, uint64_t first, uint64_t count,
                         uint64_t seed, uint32_t tag, uint32_t inst, uint32_t bound);

/* O14. Encrypt of the paper's PKE, all k bits at once:
 * U[j*k+c] = (sum_{i<m} A[i*n+j]*R[i*k+c] + E1[j*k+c]) mod q ;
 * v[c]     = (sum_{i<m} t[i]*R[i*k+c] + e2[c] + mu_c*floor(q/2)) mod q ;   R, E1, e2 signed (int8).
 * Pins: python big-integer brute force; reduces to O8 for R in {0,1}, E1 = 0, e2 = 0; the noise identity
 * v - U^T s - mu floor(q/2) = e^T R + e2 - s^T E1 (mod q); every bit recovered on Table 1's first parameter set. */
void orc_encaps_pv(const uint16_t *A, const uint16_t *t, const int8_t *R, const int8_t *E1, const int8_t *e2,
                   const uint8_t *mubits, uint16_t *U, uint16_t *v,
                   uint32_t m, uint32_t n, uint32_t k, uint32_t q);

/* ---- N2 on the q = 65537 rows of Table 1 (n = 8192 ... 131072): residues need 17 bits.
 * Readings S23-S25 of DESIGN.md section 3 (the paper says only "32-bit integers", and gives no sampler):
 *   S23  residues of a modulus q > 65536 are stored as uint32_t in [0, q);
 *   S24  uniform mod q on 32-bit stream words: O4 with the word size of the storage type (O4w below);
 *   S25  the small objects cross the boundary as signed int8: s ~ CBD(eta) in [-eta, eta] (O5s), e, R, E1 ~ D_sigma
 *        in [-12, 12] (O12), e2 in [-kappa, kappa] (O13).
 * The functions below take any 2 <= q < 2^31, so that for q <= 65536 they can be pinned against the uint16 ones.
 *
 * O4w. Uniform mod q by rejection on 32-bit words, element t: for attempt a = 0,1,..:
 *   c = LE32(bytes [4t, 4t+3] of KS(key(seed), iv(tag, a, inst))); T = q*floor(2^32/q); accept iff c < T; value c mod q.
 * Pins: the stream re-derived through OpenSSL with an independent walk over the attempt streams (a modulus with
 * 25 % rejection included); sub-range == slice; strided == gathered; chi-square uniformity at q = 65537. */
void orc_sample_uniform32(uint32_t *out, uint64_t first, uint64_t count,
                          uint64_t seed, uint32_t tag, uint32_t inst, uint32_t q);
void orc_sample_uniform32_strided(uint32_t *out, uint64_t first, uint64_t stride, uint64_t count,
                                  uint64_t seed, uint32_t tag, uint32_t inst, uint32_t q);

/* O5s. Centred binomial eta as a SIGNED value: x = popcount(w & M) - popcount((w >> 8) & M) of the element's 16-bit
 * stream word w exactly as O5, stored as int8 (no modulus involved).  Pin: x mod q == O5's residue, range, sign. */
void orc_sample_cbd_s8(int8_t *out, uint64_t first, uint64_t count,
                       uint64_t seed, uint32_t tag, uint32_t inst, uint32_t eta);

/* O7w. KeyGen of the paper's PKE with small signed secret and noise (eq.(1)):
 * t_i = (sum_{j<n} A[i*n+j]*s[j] + e[i]) mod q in [0, q), A uint32 residues, s, e int8.
 * Pins: python big-integer brute force (q = 65537, 65539, 100003); equals O7 for q <= 65536; A = 65536 everywhere
 * with q = 65537 gives t_i = e_i - sum_j s_j (2^16 = -1); linearity. */
void orc_keygen_w(const uint32_t *A, const int8_t *s, const int8_t *e, uint32_t *t,
                  uint32_t m, uint32_t n, uint32_t q);

/* O14w. Encrypt of the paper's PKE (O14) on uint32 residues:
 * U[j*k+c] = (sum_{i<m} A[i*n+j]*R[i*k+c] + E1[j*k+c]) mod q ;
 * v[c]     = (sum_{i<m} t[i]*R[i*k+c] + e2[c] + mu_c*floor(q/2)) mod q.
 * Pins: big-integer brute force; equals O14 for q <= 65536; the 2^16 = -1 special case; the noise identity
 * v - U^T s - mu floor(q/2) = e^T R + e2 - s^T E1 (mod q); every bit recovered on Table 1's n = 8192 row. */
void orc_encaps_pv_w(const uint32_t *A, const uint32_t *t, const int8_t *R, const int8_t *E1, const int8_t *e2,
                     const uint8_t *mubits, uint32_t *U, uint32_t *v,
                     uint32_t m, uint32_t n, uint32_t k, uint32_t q);

/* O9w. Decrypt on uint32 residues with the small signed secret:
 * d_c = (v[c] - sum_{j<n} U[j*k+c]*s[j]) mod q in [0, q); bit_c = floor((4 d_c + q) / (2q)) mod 2 (S12).
 * If d_out != NULL it receives d_c.  Pins: big-integer brute force; equals O9 for q <= 65536; exhaustive rounding
 * over all d for q = 65537. */
void orc_decaps_w(const uint32_t *U, const uint32_t *v, const int8_t *s,
                  uint8_t *mubits_out, uint32_t *d_out, uint32_t n, uint32_t k, uint32_t q);

/* Number of OpenMP threads the loops above will use (1 if built without OpenMP), and a setter so that the timed
 * CPU baseline can report a 1-thread and an all-core figure (the paper's OpenMP baseline).  Returns
 * the previous value; no effect without OpenMP.  Changes no arithmetic. */
int orc_num_threads(void);
int orc_set_num_threads(int threads);

#ifdef __cplusplus
}
#endif
#endif /* LWE_ORACLE_H */

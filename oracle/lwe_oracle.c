/*
 * lwe_oracle.c -- ORACLE. Test infrastructure, not the product (see lwe_oracle.h).
 *
 * Plain C11.  Everything follows the definitions of SURVEY.md 8(c) O1-O10 in the
 * order they are stated; there is no blocking, table trick or lazy reduction.
 * The only concession to run time is `#pragma omp parallel for` over independent
 * OUTPUT elements (rows of b, rows of U, columns of d), mirroring the paper's own
 * OpenMP baseline; it does not change any arithmetic.
 */
#include "lwe_oracle.h"

#include <stdlib.h>
#include <math.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------ O1: AES-128 */

/* GF(2^8) multiply modulo x^8 + x^4 + x^3 + x + 1 (FIPS-197 sec. 4.2). */
static uint8_t gf_mul(uint8_t a, uint8_t b)
{
    uint8_t p = 0;
    for (int bit = 0; bit < 8; bit++) {
        if (b & 1) p ^= a;
        uint8_t carry = (uint8_t)(a & 0x80);
        a = (uint8_t)(a << 1);
        if (carry) a ^= 0x1b;
        b >>= 1;
    }
    return p;
}

/* S-box built from its definition (FIPS-197 sec. 5.1.1): multiplicative inverse in
 * GF(2^8) (0 -> 0) followed by the affine map b ^ rotl(b,1..4) ^ 0x63. */
static uint8_t sbox_tab[256];
static int sbox_ready = 0;

static uint8_t rotl8(uint8_t x, int r) { return (uint8_t)((x << r) | (x >> (8 - r))); }

static void sbox_build(void)
{
    for (int x = 0; x < 256; x++) {
        uint8_t inv = 0;
        if (x != 0) {
            for (int y = 1; y < 256; y++) {
                if (gf_mul((uint8_t)x, (uint8_t)y) == 1) { inv = (uint8_t)y; break; }
            }
        }
        sbox_tab[x] = (uint8_t)(inv ^ rotl8(inv, 1) ^ rotl8(inv, 2) ^ rotl8(inv, 3) ^ rotl8(inv, 4) ^ 0x63);
    }
}

static void sbox_init(void)
{
    if (sbox_ready) return;
#ifdef _OPENMP
#pragma omp critical(orc_sbox_init)
#endif
    {
        if (!sbox_ready) {
            sbox_build();
            sbox_ready = 1;
        }
    }
}

/* Key expansion, FIPS-197 sec. 5.2, Nk = 4, Nr = 10: 44 words = 176 bytes. */
static void aes128_expand_key(const uint8_t key[16], uint8_t rk[176])
{
    memcpy(rk, key, 16);
    uint8_t rcon = 0x01;
    for (int w = 4; w < 44; w++) {
        uint8_t t[4];
        memcpy(t, rk + 4 * (w - 1), 4);
        if (w % 4 == 0) {
            /* RotWord, SubWord, xor Rcon */
            uint8_t t0 = t[0];
            t[0] = (uint8_t)(sbox_tab[t[1]] ^ rcon);
            t[1] = sbox_tab[t[2]];
            t[2] = sbox_tab[t[3]];
            t[3] = sbox_tab[t0];
            rcon = gf_mul(rcon, 2);
        }
        for (int x = 0; x < 4; x++) rk[4 * w + x] = (uint8_t)(rk[4 * (w - 4) + x] ^ t[x]);
    }
}

/* State byte (row r, column c) is st[r + 4c]; input byte order = state order
 * (FIPS-197 sec. 3.4). */
static void add_round_key(uint8_t st[16], const uint8_t *rk)
{
    for (int x = 0; x < 16; x++) st[x] ^= rk[x];
}

static void sub_bytes(uint8_t st[16])
{
    for (int x = 0; x < 16; x++) st[x] = sbox_tab[st[x]];
}

static void shift_rows(uint8_t st[16])
{
    uint8_t t[16];
    for (int r = 0; r < 4; r++)
        for (int c = 0; c < 4; c++)
            t[r + 4 * c] = st[r + 4 * ((c + r) % 4)];
    memcpy(st, t, 16);
}

static void mix_columns(uint8_t st[16])
{
    for (int c = 0; c < 4; c++) {
        uint8_t a0 = st[4 * c], a1 = st[4 * c + 1], a2 = st[4 * c + 2], a3 = st[4 * c + 3];
        st[4 * c + 0] = (uint8_t)(gf_mul(a0, 2) ^ gf_mul(a1, 3) ^ a2 ^ a3);
        st[4 * c + 1] = (uint8_t)(a0 ^ gf_mul(a1, 2) ^ gf_mul(a2, 3) ^ a3);
        st[4 * c + 2] = (uint8_t)(a0 ^ a1 ^ gf_mul(a2, 2) ^ gf_mul(a3, 3));
        st[4 * c + 3] = (uint8_t)(gf_mul(a0, 3) ^ a1 ^ a2 ^ gf_mul(a3, 2));
    }
}

static void aes128_encrypt_rk(const uint8_t rk[176], const uint8_t in[16], uint8_t out[16])
{
    uint8_t st[16];
    memcpy(st, in, 16);
    add_round_key(st, rk);
    for (int round = 1; round <= 9; round++) {
        sub_bytes(st);
        shift_rows(st);
        mix_columns(st);
        add_round_key(st, rk + 16 * round);
    }
    sub_bytes(st);
    shift_rows(st);
    add_round_key(st, rk + 160);
    memcpy(out, st, 16);
}

void orc_aes128_encrypt_block(const uint8_t key[16], const uint8_t in[16], uint8_t out[16])
{
    uint8_t rk[176];
    sbox_init();
    aes128_expand_key(key, rk);
    aes128_encrypt_rk(rk, in, out);
}

/* ------------------------------------------------------------------ O2: CTR */

/* ctr = (iv + j) mod 2^128, both 128-bit big-endian (byte 0 most significant). */
static void ctr_block_input(const uint8_t iv[16], uint64_t j, uint8_t ctr[16])
{
    unsigned carry = 0;
    for (int pos = 15; pos >= 0; pos--) {
        unsigned add = (pos >= 8) ? (unsigned)((j >> (8 * (15 - pos))) & 0xff) : 0u;
        unsigned sum = (unsigned)iv[pos] + add + carry;
        ctr[pos] = (uint8_t)(sum & 0xff);
        carry = sum >> 8;
    }
}

static void ctr_block(const uint8_t rk[176], const uint8_t iv[16], uint64_t j, uint8_t ks[16])
{
    uint8_t ctr[16];
    ctr_block_input(iv, j, ctr);
    aes128_encrypt_rk(rk, ctr, ks);
}

void orc_ctr_bytes(const uint8_t key[16], const uint8_t iv[16],
                   uint64_t byte_offset, size_t nbytes, uint8_t *out)
{
    uint8_t rk[176], ks[16];
    sbox_init();
    aes128_expand_key(key, rk);
    uint64_t have_block = UINT64_MAX;
    for (size_t x = 0; x < nbytes; x++) {
        uint64_t pos = byte_offset + x;
        uint64_t blk = pos / 16;
        if (blk != have_block) {
            ctr_block(rk, iv, blk, ks);
            have_block = blk;
        }
        out[x] = ks[pos % 16];
    }
}

/* ------------------------------------------------------------------ O3: seeded objects */

void orc_seed_key(uint64_t seed, uint8_t key[16])
{
    for (int x = 0; x < 8; x++) key[x] = (uint8_t)((seed >> (8 * x)) & 0xff); /* LE64 */
    for (int x = 8; x < 16; x++) key[x] = 0;
}

void orc_object_iv(uint32_t tag, uint32_t attempt, uint32_t inst, uint8_t iv[16])
{
    /* BE64(tag*2^56 + attempt*2^32 + inst), attempt < 2^24, tag < 2^8 */
    uint64_t hi = ((uint64_t)(tag & 0xff) << 56) | ((uint64_t)(attempt & 0xffffff) << 32) | (uint64_t)inst;
    for (int x = 0; x < 8; x++) iv[x] = (uint8_t)((hi >> (8 * (7 - x))) & 0xff);
    for (int x = 8; x < 16; x++) iv[x] = 0;
}

/* 16-bit little-endian word t of the stream of (seed, tag, attempt, inst). */
static uint16_t stream_word16(const uint8_t rk[176], uint32_t tag, uint32_t attempt, uint32_t inst, uint64_t t)
{
    uint8_t iv[16], ks[16];
    orc_object_iv(tag, attempt, inst, iv);
    ctr_block(rk, iv, (2 * t) / 16, ks);
    unsigned off = (unsigned)((2 * t) % 16);
    return (uint16_t)(ks[off] | ((unsigned)ks[off + 1] << 8));
}

/* ------------------------------------------------------------------ O4: uniform mod q */

void orc_sample_uniform(uint16_t *out, uint64_t first, uint64_t count,
                        uint64_t seed, uint32_t tag, uint32_t inst, uint32_t q)
{
    uint8_t key[16], rk[176];
    sbox_init();
    orc_seed_key(seed, key);
    aes128_expand_key(key, rk);
    const uint32_t T = q * (65536u / q);
    if (count == 0) return;
    /* walk the stream one 16-byte block (8 words) at a time so that the attempt-0
     * block is encrypted once, not once per word; later attempts are rare and are
     * fetched word by word. */
    const uint64_t blk_lo = first / 8, blk_hi = (first + count - 1) / 8;
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (uint64_t blk = blk_lo; blk <= blk_hi; blk++) {
        uint8_t iv[16], ks[16];
        orc_object_iv(tag, 0, inst, iv);
        ctr_block(rk, iv, blk, ks);
        for (unsigned w = 0; w < 8; w++) {
            uint64_t t = 8 * blk + w;
            if (t < first || t >= first + count) continue;
            uint32_t c = (uint32_t)ks[2 * w] | ((uint32_t)ks[2 * w + 1] << 8);
            for (uint32_t attempt = 1; c >= T; attempt++)
                c = stream_word16(rk, tag, attempt, inst, t);
            out[t - first] = (uint16_t)(c % q);
        }
    }
}

/* O4 on the elements first, first+stride, first+2*stride, ...: element by element, straight from
 * the definition (one stream word per attempt).  Used to draw a COLUMN of the row-major A
 * (first = j, stride = n) at sizes where A itself is too big to draw on a CPU. */
void orc_sample_uniform_strided(uint16_t *out, uint64_t first, uint64_t stride, uint64_t count,
                                uint64_t seed, uint32_t tag, uint32_t inst, uint32_t q)
{
    uint8_t key[16], rk[176];
    sbox_init();
    orc_seed_key(seed, key);
    aes128_expand_key(key, rk);
    const uint32_t T = q * (65536u / q);
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (uint64_t r = 0; r < count; r++) {
        const uint64_t t = first + r * stride;
        uint32_t c = stream_word16(rk, tag, 0, inst, t);
        for (uint32_t attempt = 1; c >= T; attempt++)
            c = stream_word16(rk, tag, attempt, inst, t);
        out[r] = (uint16_t)(c % q);
    }
}

/* ------------------------------------------------------------------ O5: CBD */

static int popcount16(unsigned w)
{
    int n = 0;
    for (int bit = 0; bit < 16; bit++) n += (int)((w >> bit) & 1u);
    return n;
}

uint16_t orc_cbd_from_word(uint32_t w, uint32_t q, uint32_t eta)
{
    const unsigned M = (1u << eta) - 1u;
    int val = popcount16(w & M) - popcount16((w >> 8) & M);            /* in [-eta, eta] */
    int64_t r = ((int64_t)val % (int64_t)q + (int64_t)q) % (int64_t)q;
    return (uint16_t)r;
}

void orc_sample_cbd(uint16_t *out, uint64_t first, uint64_t count,
                    uint64_t seed, uint32_t tag, uint32_t inst, uint32_t q, uint32_t eta)
{
    uint8_t key[16], rk[176];
    sbox_init();
    orc_seed_key(seed, key);
    aes128_expand_key(key, rk);
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (uint64_t x = 0; x < count; x++) {
        uint32_t w = stream_word16(rk, tag, 0, inst, first + x);
        out[x] = orc_cbd_from_word(w, q, eta);
    }
}

/* ------------------------------------------------------------------ O6: bits */

void orc_sample_bits(uint8_t *out, uint64_t first_bit, uint64_t nbits,
                     uint64_t seed, uint32_t tag, uint32_t inst)
{
    uint8_t key[16], iv[16];
    orc_seed_key(seed, key);
    orc_object_iv(tag, 0, inst, iv);
    memset(out, 0, (size_t)((nbits + 7) / 8));
    /* one keystream byte at a time; bit t of the stream -> bit (t - first_bit) of out */
    uint64_t byte_lo = first_bit / 8;
    uint64_t byte_hi = (first_bit + nbits + 7) / 8;      /* exclusive */
    size_t span = (size_t)(byte_hi - byte_lo);
    uint8_t *ks = (uint8_t *)malloc(span ? span : 1);
    orc_ctr_bytes(key, iv, byte_lo, span, ks);
    for (uint64_t x = 0; x < nbits; x++) {
        uint64_t t = first_bit + x;
        unsigned bit = (unsigned)((ks[t / 8 - byte_lo] >> (t % 8)) & 1u);
        out[x / 8] = (uint8_t)(out[x / 8] | (bit << (x % 8)));
    }
    free(ks);
}

/* ------------------------------------------------------------------ O7: keygen */

void orc_keygen(const uint16_t *A, const uint16_t *s, const uint16_t *e, uint16_t *b,
                uint32_t m, uint32_t n, uint32_t q)
{
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (uint32_t i = 0; i < m; i++) {
        uint64_t acc = 0;
        for (uint32_t j = 0; j < n; j++)
            acc = (acc + (uint64_t)A[(size_t)i * n + j] * (uint64_t)s[j]) % q;
        b[i] = (uint16_t)((acc + e[i]) % q);
    }
}

/* ------------------------------------------------------------------ O8: encaps */

static unsigned get_bit(const uint8_t *bits, uint64_t t)
{
    return (unsigned)((bits[t / 8] >> (t % 8)) & 1u);
}

/* Row j of U: U_jc = sum_i A_ij R_ic mod q, for all c. */
static void encaps_row(const uint16_t *A, const uint8_t *Rbits, uint32_t j, uint16_t *Urow,
                       uint32_t m, uint32_t n, uint32_t k, uint32_t q)
{
    for (uint32_t c = 0; c < k; c++) {
        uint64_t acc = 0;
        for (uint32_t i = 0; i < m; i++)
            acc = (acc + (uint64_t)A[(size_t)i * n + j] * get_bit(Rbits, (uint64_t)i * k + c)) % q;
        Urow[c] = (uint16_t)acc;
    }
}

void orc_encaps_v(const uint16_t *b, const uint8_t *Rbits, const uint8_t *mubits,
                  uint16_t *v, uint32_t m, uint32_t k, uint32_t q)
{
    for (uint32_t c = 0; c < k; c++) {
        uint64_t acc = 0;
        for (uint32_t i = 0; i < m; i++)
            acc = (acc + (uint64_t)b[i] * get_bit(Rbits, (uint64_t)i * k + c)) % q;
        acc = (acc + (uint64_t)get_bit(mubits, c) * (uint64_t)(q / 2)) % q;
        v[c] = (uint16_t)acc;
    }
}

void orc_encaps_rows(const uint16_t *A, const uint8_t *Rbits, const uint32_t *rows,
                     uint32_t nrows, uint16_t *Urows,
                     uint32_t m, uint32_t n, uint32_t k, uint32_t q)
{
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1)
#endif
    for (uint32_t r = 0; r < nrows; r++)
        encaps_row(A, Rbits, rows[r], Urows + (size_t)r * k, m, n, k, q);
}

void orc_encaps(const uint16_t *A, const uint16_t *b, const uint8_t *Rbits,
                const uint8_t *mubits, uint16_t *U, uint16_t *v,
                uint32_t m, uint32_t n, uint32_t k, uint32_t q)
{
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 4)
#endif
    for (uint32_t j = 0; j < n; j++)
        encaps_row(A, Rbits, j, U + (size_t)j * k, m, n, k, q);
    orc_encaps_v(b, Rbits, mubits, v, m, k, q);
}

/* ------------------------------------------------------------------ O9: decaps */

uint32_t orc_round_bit(uint32_t d, uint32_t q)
{
    /* round-half-up of 2d/q, mod 2 */
    return (uint32_t)(((4 * (uint64_t)d + q) / (2 * (uint64_t)q)) % 2);
}

void orc_decaps(const uint16_t *U, const uint16_t *v, const uint16_t *s,
                uint8_t *mubits_out, uint16_t *d_out,
                uint32_t n, uint32_t k, uint32_t q)
{
    uint8_t *bit = (uint8_t *)malloc(k ? k : 1);
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (uint32_t c = 0; c < k; c++) {
        uint64_t acc = 0;
        for (uint32_t j = 0; j < n; j++)
            acc = (acc + (uint64_t)U[(size_t)j * k + c] * (uint64_t)s[j]) % q;
        uint64_t d = ((uint64_t)v[c] + (uint64_t)q - acc) % q;       /* in [0,q) */
        if (d_out) d_out[c] = (uint16_t)d;
        bit[c] = (uint8_t)orc_round_bit((uint32_t)d, q);
    }
    memset(mubits_out, 0, (k + 7) / 8);
    for (uint32_t c = 0; c < k; c++)
        mubits_out[c / 8] = (uint8_t)(mubits_out[c / 8] | (bit[c] << (c % 8)));
    free(bit);
}

/* O11. Alg. 5 lines 1, 2, 4, in the paper's order: m' <- Decrypt(sk, c); c' <- Encrypt(pk, m') with the
 * re-derived coins R; verdict c' == c (every element of U and v).  The hashes of lines 3, 5, 7 are outside the
 * hot path. */
int orc_decaps_fo(const uint16_t *A, const uint16_t *b, const uint16_t *U, const uint16_t *v,
                  const uint16_t *s, const uint8_t *Rbits, uint8_t *mubits_out,
                  uint32_t m, uint32_t n, uint32_t k, uint32_t q)
{
    orc_decaps(U, v, s, mubits_out, NULL, n, k, q);                              /* 1: m' */
    uint16_t *U2 = (uint16_t *)malloc((size_t)n * k * sizeof(uint16_t) + 2);
    uint16_t *v2 = (uint16_t *)malloc((size_t)k * sizeof(uint16_t) + 2);
    orc_encaps(A, b, Rbits, mubits_out, U2, v2, m, n, k, q);                     /* 2: c' = (U', v') */
    int equal = 1;                                                               /* 4: c' == c ? */
    for (size_t x = 0; x < (size_t)n * k; x++) if (U2[x] != U[x]) equal = 0;
    for (uint32_t c = 0; c < k; c++) if (v2[c] != v[c]) equal = 0;
    free(U2);
    free(v2);
    return equal;
}

/* ================================================================== N2: the paper's own PKE variant
 * (Table 1 header P:L92: Gaussian sigma for e, r, e1; centred uniform for e2;
 * binomial eta = 3 for s; square A).  Readings S20-S22 of DESIGN.md section 3. */

/* O12. 16-bit CDT of the rounded Gaussian z = round(sigma * N(0,1)), support [-12, 12]:
 * C[j] = floor(65536 * Phi((j - 12 + 1/2) / sigma) + 1/2), j = 0..23, Phi the standard normal CDF. */
void orc_gauss_cdt(double sigma, uint32_t cdt[ORC_GAUSS_CDT_LEN])
{
    for (int j = 0; j < ORC_GAUSS_CDT_LEN; j++) {
        double x = ((double)j - (double)ORC_GAUSS_TAU + 0.5) / sigma;
        double Phi = 0.5 * erfc(-x / sqrt(2.0));
        cdt[j] = (uint32_t)floor(65536.0 * Phi + 0.5);
    }
}

/* z = -tau + #{ j : w >= C[j] } for a 16-bit stream word w */
int orc_gauss_from_word(uint32_t w, const uint32_t cdt[ORC_GAUSS_CDT_LEN])
{
    int z = -ORC_GAUSS_TAU;
    for (int j = 0; j < ORC_GAUSS_CDT_LEN; j++)
        if (w >= cdt[j]) z++;
    return z;
}

/* element t: w = LE16(bytes [2t, 2t+1] of KS(key(seed), iv(tag, 0, inst))); z as above.
 * out_s8 (if not NULL) receives z; out_u16 (if not NULL) receives z mod q in [0, q). */
void orc_sample_gauss(int8_t *out_s8, uint16_t *out_u16, uint64_t first, uint64_t count,
                      uint64_t seed, uint32_t tag, uint32_t inst, double sigma, uint32_t q)
{
    uint8_t key[16], rk[176];
    uint32_t cdt[ORC_GAUSS_CDT_LEN];
    sbox_init();
    orc_seed_key(seed, key);
    aes128_expand_key(key, rk);
    orc_gauss_cdt(sigma, cdt);
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (uint64_t x = 0; x < count; x++) {
        int z = orc_gauss_from_word(stream_word16(rk, tag, 0, inst, first + x), cdt);
        if (out_s8) out_s8[x] = (int8_t)z;
        if (out_u16) out_u16[x] = (uint16_t)((((int64_t)z % (int64_t)q) + (int64_t)q) % (int64_t)q);
    }
}

/* O13. Centred uniform on [-bound, bound]: rejection exactly as O4 with modulus q' = 2*bound + 1
 * (attempt streams), value (c mod q') - bound. */
void orc_sample_cuniform(int8_t *out, uint64_t first, uint64_t count,
                         uint64_t seed, uint32_t tag, uint32_t inst, uint32_t bound)
{
    uint8_t key[16], rk[176];
    sbox_init();
    orc_seed_key(seed, key);
    aes128_expand_key(key, rk);
    const uint32_t qq = 2 * bound + 1, T = qq * (65536u / qq);
    for (uint64_t x = 0; x < count; x++) {
        uint32_t c = stream_word16(rk, tag, 0, inst, first + x);
        for (uint32_t attempt = 1; c >= T; attempt++)
            c = stream_word16(rk, tag, attempt, inst, first + x);
        out[x] = (int8_t)((int)(c % qq) - (int)bound);
    }
}

static uint64_t mod_signed(int64_t x, uint32_t q)
{
    int64_t r = x % (int64_t)q;
    return (uint64_t)(r < 0 ? r + (int64_t)q : r);
}

/* O14. Encrypt of the paper's PKE for all k bits at once:
 * U[j*k+c] = (sum_i A[i*n+j]*R[i*k+c] + E1[j*k+c]) mod q
 * v[c]     = (sum_i t[i]*R[i*k+c] + e2[c] + mu_c*floor(q/2)) mod q        (R, E1, e2 small signed integers) */
void orc_encaps_pv(const uint16_t *A, const uint16_t *t, const int8_t *R, const int8_t *E1, const int8_t *e2,
                   const uint8_t *mubits, uint16_t *U, uint16_t *v,
                   uint32_t m, uint32_t n, uint32_t k, uint32_t q)
{
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (uint32_t j = 0; j < n; j++)
        for (uint32_t c = 0; c < k; c++) {
            uint64_t acc = 0;
            for (uint32_t i = 0; i < m; i++)
                acc = (acc + (uint64_t)A[(size_t)i * n + j] * mod_signed(R[(size_t)i * k + c], q)) % q;
            U[(size_t)j * k + c] = (uint16_t)((acc + mod_signed(E1[(size_t)j * k + c], q)) % q);
        }
    for (uint32_t c = 0; c < k; c++) {
        uint64_t acc = 0;
        for (uint32_t i = 0; i < m; i++)
            acc = (acc + (uint64_t)t[i] * mod_signed(R[(size_t)i * k + c], q)) % q;
        acc = (acc + mod_signed(e2[c], q)) % q;
        acc = (acc + (uint64_t)get_bit(mubits, c) * (q / 2)) % q;
        v[c] = (uint16_t)acc;
    }
}

/* ================================================================== N2 with q > 65536 (Table 1 rows n >= 8192,
 * P:L98-102): uint32 residues.  Readings S23-S25 of DESIGN.md section 3. */

/* 32-bit little-endian word t of the stream of (seed, tag, attempt, inst): bytes [4t, 4t+3]. */
static uint32_t stream_word32(const uint8_t rk[176], uint32_t tag, uint32_t attempt, uint32_t inst, uint64_t t)
{
    uint8_t iv[16], ks[16];
    orc_object_iv(tag, attempt, inst, iv);
    ctr_block(rk, iv, (4 * t) / 16, ks);
    unsigned off = (unsigned)((4 * t) % 16);
    return (uint32_t)ks[off] | ((uint32_t)ks[off + 1] << 8) | ((uint32_t)ks[off + 2] << 16) | ((uint32_t)ks[off + 3] << 24);
}

/* O4w, element by element, straight from the definition. */
void orc_sample_uniform32_strided(uint32_t *out, uint64_t first, uint64_t stride, uint64_t count,
                                  uint64_t seed, uint32_t tag, uint32_t inst, uint32_t q)
{
    uint8_t key[16], rk[176];
    sbox_init();
    orc_seed_key(seed, key);
    aes128_expand_key(key, rk);
    const uint64_t T = (uint64_t)q * ((1ull << 32) / q);        /* q * floor(2^32 / q) <= 2^32 */
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (uint64_t r = 0; r < count; r++) {
        const uint64_t t = first + r * stride;
        uint64_t c = stream_word32(rk, tag, 0, inst, t);
        for (uint32_t attempt = 1; c >= T; attempt++)
            c = stream_word32(rk, tag, attempt, inst, t);
        out[r] = (uint32_t)(c % q);
    }
}

/* O4w on a contiguous range: the same values, walking the stream one 16-byte block (4 words) at a time so that the
 * attempt-0 block is encrypted once, not once per word (as orc_sample_uniform does; cross-checked against the
 * element-wise function above in tests/test_oracle_wide.py). */
void orc_sample_uniform32(uint32_t *out, uint64_t first, uint64_t count,
                          uint64_t seed, uint32_t tag, uint32_t inst, uint32_t q)
{
    uint8_t key[16], rk[176];
    sbox_init();
    orc_seed_key(seed, key);
    aes128_expand_key(key, rk);
    const uint64_t T = (uint64_t)q * ((1ull << 32) / q);
    if (count == 0) return;
    const uint64_t blk_lo = first / 4, blk_hi = (first + count - 1) / 4;
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (uint64_t blk = blk_lo; blk <= blk_hi; blk++) {
        uint8_t iv[16], ks[16];
        orc_object_iv(tag, 0, inst, iv);
        ctr_block(rk, iv, blk, ks);
        for (unsigned w = 0; w < 4; w++) {
            uint64_t t = 4 * blk + w;
            if (t < first || t >= first + count) continue;
            uint64_t c = (uint64_t)ks[4 * w] | ((uint64_t)ks[4 * w + 1] << 8) | ((uint64_t)ks[4 * w + 2] << 16) |
                         ((uint64_t)ks[4 * w + 3] << 24);
            for (uint32_t attempt = 1; c >= T; attempt++)
                c = stream_word32(rk, tag, attempt, inst, t);
            out[t - first] = (uint32_t)(c % q);
        }
    }
}

/* O5s. */
void orc_sample_cbd_s8(int8_t *out, uint64_t first, uint64_t count,
                       uint64_t seed, uint32_t tag, uint32_t inst, uint32_t eta)
{
    uint8_t key[16], rk[176];
    sbox_init();
    orc_seed_key(seed, key);
    aes128_expand_key(key, rk);
    const unsigned M = (1u << eta) - 1u;
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (uint64_t x = 0; x < count; x++) {
        unsigned w = stream_word16(rk, tag, 0, inst, first + x);
        out[x] = (int8_t)(popcount16(w & M) - popcount16((w >> 8) & M));
    }
}

/* O7w. */
void orc_keygen_w(const uint32_t *A, const int8_t *s, const int8_t *e, uint32_t *t,
                  uint32_t m, uint32_t n, uint32_t q)
{
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (uint32_t i = 0; i < m; i++) {
        uint64_t acc = 0;
        for (uint32_t j = 0; j < n; j++)
            acc = (acc + (uint64_t)A[(size_t)i * n + j] * mod_signed(s[j], q)) % q;
        t[i] = (uint32_t)((acc + mod_signed(e[i], q)) % q);
    }
}

/* O14w. */
void orc_encaps_pv_w(const uint32_t *A, const uint32_t *t, const int8_t *R, const int8_t *E1, const int8_t *e2,
                     const uint8_t *mubits, uint32_t *U, uint32_t *v,
                     uint32_t m, uint32_t n, uint32_t k, uint32_t q)
{
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (uint32_t j = 0; j < n; j++)
        for (uint32_t c = 0; c < k; c++) {
            uint64_t acc = 0;
            for (uint32_t i = 0; i < m; i++)
                acc = (acc + (uint64_t)A[(size_t)i * n + j] * mod_signed(R[(size_t)i * k + c], q)) % q;
            U[(size_t)j * k + c] = (uint32_t)((acc + mod_signed(E1[(size_t)j * k + c], q)) % q);
        }
    for (uint32_t c = 0; c < k; c++) {
        uint64_t acc = 0;
        for (uint32_t i = 0; i < m; i++)
            acc = (acc + (uint64_t)t[i] * mod_signed(R[(size_t)i * k + c], q)) % q;
        acc = (acc + mod_signed(e2[c], q)) % q;
        acc = (acc + (uint64_t)get_bit(mubits, c) * (q / 2)) % q;
        v[c] = (uint32_t)acc;
    }
}

/* O9w. */
void orc_decaps_w(const uint32_t *U, const uint32_t *v, const int8_t *s,
                  uint8_t *mubits_out, uint32_t *d_out, uint32_t n, uint32_t k, uint32_t q)
{
    uint8_t *bit = (uint8_t *)malloc(k ? k : 1);
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (uint32_t c = 0; c < k; c++) {
        uint64_t acc = 0;
        for (uint32_t j = 0; j < n; j++)
            acc = (acc + (uint64_t)U[(size_t)j * k + c] * mod_signed(s[j], q)) % q;
        uint64_t d = ((uint64_t)v[c] + (uint64_t)q - acc) % q;       /* in [0,q) */
        if (d_out) d_out[c] = (uint32_t)d;
        bit[c] = (uint8_t)orc_round_bit((uint32_t)d, q);
    }
    memset(mubits_out, 0, (k + 7) / 8);
    for (uint32_t c = 0; c < k; c++)
        mubits_out[c / 8] = (uint8_t)(mubits_out[c / 8] | (bit[c] << (c % 8)));
    free(bit);
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

int orc_set_num_threads(int threads)
{
    int prev = orc_num_threads();
#ifdef _OPENMP
    if (threads >= 1) omp_set_num_threads(threads);
#else
    (void)threads;
#endif
    return prev;
}

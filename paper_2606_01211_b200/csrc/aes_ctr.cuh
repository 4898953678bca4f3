// aes_ctr.cuh -- device-side AES-128 for the counter-indexed stream (S8(a) a1).
//
// T-table formulation, built around what bounds it on sm_100: the integer-logic pipe
// (LOP3 / PRMT / SHF: 64 lanes/clk/SM, half the issue rate) and the shared-memory crossbar
// (one conflict-free 32-lane wavefront per clock and SM).
//
// Layout.  Two tables, T0 and T1 = rotl8(T0), each replicated once per shared-memory bank, in
// rows of 256 bytes: row x = [T0[x] x 32 lanes | T1[x] x 32 lanes].  Lane l reads T0[x] at byte
// x*256 + 4l and T1[x] at x*256 + 128 + 4l, so
//   * the 16 data-dependent lookups of a round never bank-conflict (1 wavefront each; a plain
//     1 KB table read at 32 random indices serialises ~3.5-way), and
//   * a lookup address is ONE instruction: PRMT puts state byte i into byte 1 of the lane's
//     constant offset word (byte 0 = 4l or 128 + 4l, bytes 2-3 = 0); the table base comes in
//     through the uniform-register operand of LDS [R + UR].  The usual extract-shift-add costs
//     two to three integer instructions per lookup.
//   * with T1 = rotl8(T0) only one rotation per column is left:
//       col = T0[a0] ^ T1[a1] ^ rk ^ rotl16(T0[a2] ^ T1[a3])
//     (rotl16(T1[x]) = rotl24(T0[x])): 4 PRMT + 4 LDS + 3 LOP3 + 1 PRMT = 12 instructions per
//     column and round, 8 of them on the integer pipe -- the single-table form needed 17 / 13.
// 64 KB of shared memory per CTA.
//
// Word convention: word c of a block = bytes 4c..4c+3 little-endian, i.e. state
// column c with row r in byte r.  FIPS-197: SubBytes+ShiftRows+MixColumns of column
// c = Te0[a(0,c)] ^ rotl8(Te0[a(1,c+1)]) ^ rotl16(Te0[a(2,c+2)]) ^ rotl24(Te0[a(3,c+3)]),
// Te0[x] = 2S | S<<8 | S<<16 | 3S<<24 with S = SubBytes(x).
#pragma once

#include "lwe_internal.cuh"

namespace lwe {

constexpr int kAesRowBytes = 256;
constexpr int kAesTableBytes = 256 * kAesRowBytes;     // 64 KB

// A lane's view of the table: base of the table and the lane's two offset words.
struct AesTab {
    const uint8_t *base;
    uint32_t o0, o1;       // 4*lane, 128 + 4*lane
};

// Fills the table (all NT threads of the CTA), synchronises, and returns the calling lane's view.
// NT = the CTA size, a compile-time constant: the ~16 loads of a thread are then issued back to back and the fill
// costs one memory latency.  With a run-time stride the loop stays rolled, every store waits for its own load, and
// 16 serial L2 latencies made ~7 of the ~10 us a sampler launch takes before its first AES block (measured: a sampler
// call of 8 elements, 10.2 us).
template <int NT>
__device__ __forceinline__ AesTab aes_table_to_smem(void *smem, const uint32_t *__restrict__ te0)
{
    uint32_t *w = reinterpret_cast<uint32_t *>(smem);
    constexpr int kWords = kAesTableBytes / 4, kIters = (kWords + NT - 1) / NT;
    uint32_t t[kIters];
#pragma unroll
    for (int it = 0; it < kIters; it++) {
        const int idx = threadIdx.x + it * NT;
        t[it] = (idx < kWords) ? __ldg(te0 + (idx >> 6)) : 0u;
    }
#pragma unroll
    for (int it = 0; it < kIters; it++) {
        const int idx = threadIdx.x + it * NT;
        if (idx < kWords) w[idx] = (idx & 32) ? __byte_perm(t[it], t[it], 0x2103) : t[it];   // second half of the row: rotl8
    }
    __syncthreads();
    AesTab tab;
    tab.base = reinterpret_cast<const uint8_t *>(smem);
    tab.o0 = (threadIdx.x & 31) * 4;
    tab.o1 = tab.o0 + 128;
    return tab;
}

__device__ __forceinline__ uint32_t rotl16(uint32_t x) { return __byte_perm(x, x, 0x1032); }

// Table word for state byte `kByte` of s: off = tab.o0 (T0) or tab.o1 (T1).
// PRMT selector: result = (off.byte0, s.byte[kByte], off.byte1 = 0, off.byte2 = 0).
template <int kByte>
__device__ __forceinline__ uint32_t te(const AesTab &tab, uint32_t s, uint32_t off)
{
    return *reinterpret_cast<const uint32_t *>(tab.base + __byte_perm(s, off, 0x6504 + 0x10 * kByte));
}

__device__ __forceinline__ void aes128_encrypt(const AesKey &k, const AesTab &tab,
                                               uint32_t s0, uint32_t s1, uint32_t s2, uint32_t s3,
                                               uint32_t &o0, uint32_t &o1, uint32_t &o2, uint32_t &o3)
{
    const uint32_t a = tab.o0, b = tab.o1;
    s0 ^= k.rk[0]; s1 ^= k.rk[1]; s2 ^= k.rk[2]; s3 ^= k.rk[3];
#pragma unroll
    for (int r = 1; r <= 9; r++) {
        uint32_t t0 = (te<0>(tab, s0, a) ^ te<1>(tab, s1, b) ^ k.rk[4 * r]) ^ rotl16(te<2>(tab, s2, a) ^ te<3>(tab, s3, b));
        uint32_t t1 = (te<0>(tab, s1, a) ^ te<1>(tab, s2, b) ^ k.rk[4 * r + 1]) ^ rotl16(te<2>(tab, s3, a) ^ te<3>(tab, s0, b));
        uint32_t t2 = (te<0>(tab, s2, a) ^ te<1>(tab, s3, b) ^ k.rk[4 * r + 2]) ^ rotl16(te<2>(tab, s0, a) ^ te<3>(tab, s1, b));
        uint32_t t3 = (te<0>(tab, s3, a) ^ te<1>(tab, s0, b) ^ k.rk[4 * r + 3]) ^ rotl16(te<2>(tab, s1, a) ^ te<3>(tab, s2, b));
        s0 = t0; s1 = t1; s2 = t2; s3 = t3;
    }
    // last round: SubBytes + ShiftRows only; S(x) is byte 1 of T0[x]
    {
        uint32_t w, x, y, z;
        w = te<0>(tab, s0, a); x = te<1>(tab, s1, a); y = te<2>(tab, s2, a); z = te<3>(tab, s3, a);
        o0 = __byte_perm(__byte_perm(w, x, 0x0051), __byte_perm(y, z, 0x0051), 0x5410) ^ k.rk[40];
        w = te<0>(tab, s1, a); x = te<1>(tab, s2, a); y = te<2>(tab, s3, a); z = te<3>(tab, s0, a);
        o1 = __byte_perm(__byte_perm(w, x, 0x0051), __byte_perm(y, z, 0x0051), 0x5410) ^ k.rk[41];
        w = te<0>(tab, s2, a); x = te<1>(tab, s3, a); y = te<2>(tab, s0, a); z = te<3>(tab, s1, a);
        o2 = __byte_perm(__byte_perm(w, x, 0x0051), __byte_perm(y, z, 0x0051), 0x5410) ^ k.rk[42];
        w = te<0>(tab, s3, a); x = te<1>(tab, s0, a); y = te<2>(tab, s1, a); z = te<3>(tab, s2, a);
        o3 = __byte_perm(__byte_perm(w, x, 0x0051), __byte_perm(y, z, 0x0051), 0x5410) ^ k.rk[43];
    }
}

__device__ __forceinline__ uint32_t bswap32(uint32_t x) { return __byte_perm(x, 0, 0x0123); }

// Keystream block whose 128-bit big-endian counter is (hi:lo).
__device__ __forceinline__ uint4 aes_ctr_block(const AesKey &k, const AesTab &tab, uint64_t hi, uint64_t lo)
{
    uint4 o;
    aes128_encrypt(k, tab, bswap32((uint32_t)(hi >> 32)), bswap32((uint32_t)hi),
                   bswap32((uint32_t)(lo >> 32)), bswap32((uint32_t)lo), o.x, o.y, o.z, o.w);
    return o;
}

// Upper 64 counter bits of a seeded object stream (S8(c) O3); the lower 64 bits are
// the block index.
__device__ __host__ __forceinline__ uint64_t object_iv_hi(uint32_t tag, uint32_t attempt, uint32_t inst)
{
    return ((uint64_t)(tag & 0xffu) << 56) | ((uint64_t)(attempt & 0xffffffu) << 32) | (uint64_t)inst;
}

// Rare path of the uniform sampler: at least one of the 8 candidates of `ks` was rejected (c >= T); draw the
// replacements from the attempt streams 1, 2, ... of the same block position (S8(c) O4).  Out of line so that
// its registers (8 candidates, a second AES state) do not weigh on the callers' hot loops.
static __device__ __noinline__ uint4 uniform_block_retry(const AesKey *kp, const uint8_t *tab_base, uint32_t T,
                                                  uint32_t tag, uint32_t inst, uint64_t blk, uint4 ks)
{
    AesTab tab;
    tab.base = tab_base;
    tab.o0 = (threadIdx.x & 31) * 4;
    tab.o1 = tab.o0 + 128;
    uint32_t c[8] = {ks.x & 0xffffu, ks.x >> 16, ks.y & 0xffffu, ks.y >> 16,
                     ks.z & 0xffffu, ks.z >> 16, ks.w & 0xffffu, ks.w >> 16};
    uint32_t pending = 0;
#pragma unroll
    for (int i = 0; i < 8; i++) pending |= (c[i] >= T) ? (1u << i) : 0u;
    for (uint32_t attempt = 1; pending; attempt++) {          // P(reject) = 1 - T/65536 per element and attempt
        uint4 kr = aes_ctr_block(*kp, tab, object_iv_hi(tag, attempt, inst), blk);
        uint32_t r[8] = {kr.x & 0xffffu, kr.x >> 16, kr.y & 0xffffu, kr.y >> 16,
                         kr.z & 0xffffu, kr.z >> 16, kr.w & 0xffffu, kr.w >> 16};
#pragma unroll
        for (int i = 0; i < 8; i++) {
            if (pending & (1u << i)) {
                c[i] = r[i];
                if (r[i] < T) pending &= ~(1u << i);
            }
        }
    }
    return make_uint4(c[0] | (c[1] << 16), c[2] | (c[3] << 16), c[4] | (c[5] << 16), c[6] | (c[7] << 16));
}

// 8 uniform-mod-q elements of block `blk` of object (tag, inst): rejection sampling
// over attempt streams (S8(c) O4).  Returns them packed two per word, low element
// first (for q = 2^16 this is the raw keystream block).
__device__ __forceinline__ uint4 uniform_block(const AesKey &k, const AesTab &tab, const ModQ &mq,
                                               uint32_t tag, uint32_t inst, uint64_t blk)
{
    uint4 ks = aes_ctr_block(k, tab, object_iv_hi(tag, 0, inst), blk);
    if (mq.q == 65536u) return ks;
    if (mq.T != 65536u) {
        // any 16-bit candidate >= T ?  (T <= 65535 here)
        const uint32_t T = mq.T;
        const bool rej = ((ks.x & 0xffffu) >= T) | ((ks.x >> 16) >= T) | ((ks.y & 0xffffu) >= T) | ((ks.y >> 16) >= T) |
                         ((ks.z & 0xffffu) >= T) | ((ks.z >> 16) >= T) | ((ks.w & 0xffffu) >= T) | ((ks.w >> 16) >= T);
        if (rej) ks = uniform_block_retry(&k, tab.base, T, tag, inst, blk, ks);
        if (T == mq.q) return ks;                               // accepted candidates are already < q
    }
    uint32_t w[4] = {ks.x, ks.y, ks.z, ks.w};
#pragma unroll
    for (int i = 0; i < 4; i++) w[i] = mod_u32(w[i] & 0xffffu, mq) | (mod_u32(w[i] >> 16, mq) << 16);
    return make_uint4(w[0], w[1], w[2], w[3]);
}

}  // namespace lwe

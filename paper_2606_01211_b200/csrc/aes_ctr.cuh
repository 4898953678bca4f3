// aes_ctr.cuh -- device-side AES-128 for the counter-indexed stream (S8(a) a1).
//
// T-table formulation (one 256-entry table Te0, the other three by byte rotation),
// with Te0 replicated once per shared-memory bank: lane l always reads word
// (x*32 + l), so the 16 data-dependent lookups of a round never bank-conflict
// (a 1 KB table read at 32 random indices would serialise ~3.5-way).  32 KB of
// shared memory per CTA buys a fixed 1 wavefront per lookup.
//
// Word convention: word c of a block = bytes 4c..4c+3 little-endian, i.e. state
// column c with row r in byte r.  FIPS-197: SubBytes+ShiftRows+MixColumns of column
// c = Te0[a(0,c)] ^ rotl8(Te0[a(1,c+1)]) ^ rotl16(Te0[a(2,c+2)]) ^ rotl24(Te0[a(3,c+3)]),
// Te0[x] = 2S | S<<8 | S<<16 | 3S<<24 with S = SubBytes(x).
#pragma once

#include "lwe_internal.cuh"

namespace lwe {

constexpr int kAesTableWords = 256 * 32;               // 32 KB
constexpr int kAesTableBytes = kAesTableWords * 4;

__device__ __forceinline__ void aes_table_to_smem(uint32_t *sT, const uint32_t *__restrict__ te0)
{
    for (int idx = threadIdx.x; idx < kAesTableWords; idx += blockDim.x) sT[idx] = __ldg(te0 + (idx >> 5));
    __syncthreads();
}

__device__ __forceinline__ uint32_t rotl8(uint32_t x) { return __byte_perm(x, x, 0x2103); }
__device__ __forceinline__ uint32_t rotl16(uint32_t x) { return __byte_perm(x, x, 0x1032); }
__device__ __forceinline__ uint32_t rotl24(uint32_t x) { return __byte_perm(x, x, 0x0321); }

// sTl = sT + lane: the calling lane's private bank column
__device__ __forceinline__ uint32_t te(const uint32_t *sTl, uint32_t byte) { return sTl[byte << 5]; }

__device__ __forceinline__ void aes128_encrypt(const AesKey &k, const uint32_t *sTl,
                                               uint32_t s0, uint32_t s1, uint32_t s2, uint32_t s3,
                                               uint32_t &o0, uint32_t &o1, uint32_t &o2, uint32_t &o3)
{
    s0 ^= k.rk[0]; s1 ^= k.rk[1]; s2 ^= k.rk[2]; s3 ^= k.rk[3];
#pragma unroll
    for (int r = 1; r <= 9; r++) {
        uint32_t t0 = te(sTl, s0 & 0xff) ^ rotl8(te(sTl, (s1 >> 8) & 0xff)) ^
                      rotl16(te(sTl, (s2 >> 16) & 0xff)) ^ rotl24(te(sTl, s3 >> 24)) ^ k.rk[4 * r];
        uint32_t t1 = te(sTl, s1 & 0xff) ^ rotl8(te(sTl, (s2 >> 8) & 0xff)) ^
                      rotl16(te(sTl, (s3 >> 16) & 0xff)) ^ rotl24(te(sTl, s0 >> 24)) ^ k.rk[4 * r + 1];
        uint32_t t2 = te(sTl, s2 & 0xff) ^ rotl8(te(sTl, (s3 >> 8) & 0xff)) ^
                      rotl16(te(sTl, (s0 >> 16) & 0xff)) ^ rotl24(te(sTl, s1 >> 24)) ^ k.rk[4 * r + 2];
        uint32_t t3 = te(sTl, s3 & 0xff) ^ rotl8(te(sTl, (s0 >> 8) & 0xff)) ^
                      rotl16(te(sTl, (s1 >> 16) & 0xff)) ^ rotl24(te(sTl, s2 >> 24)) ^ k.rk[4 * r + 3];
        s0 = t0; s1 = t1; s2 = t2; s3 = t3;
    }
    // last round: SubBytes + ShiftRows only; S(x) is byte 1 of Te0[x]
    {
        uint32_t a, b, c, d;
        a = te(sTl, s0 & 0xff); b = te(sTl, (s1 >> 8) & 0xff); c = te(sTl, (s2 >> 16) & 0xff); d = te(sTl, s3 >> 24);
        o0 = __byte_perm(__byte_perm(a, b, 0x0051), __byte_perm(c, d, 0x0051), 0x5410) ^ k.rk[40];
        a = te(sTl, s1 & 0xff); b = te(sTl, (s2 >> 8) & 0xff); c = te(sTl, (s3 >> 16) & 0xff); d = te(sTl, s0 >> 24);
        o1 = __byte_perm(__byte_perm(a, b, 0x0051), __byte_perm(c, d, 0x0051), 0x5410) ^ k.rk[41];
        a = te(sTl, s2 & 0xff); b = te(sTl, (s3 >> 8) & 0xff); c = te(sTl, (s0 >> 16) & 0xff); d = te(sTl, s1 >> 24);
        o2 = __byte_perm(__byte_perm(a, b, 0x0051), __byte_perm(c, d, 0x0051), 0x5410) ^ k.rk[42];
        a = te(sTl, s3 & 0xff); b = te(sTl, (s0 >> 8) & 0xff); c = te(sTl, (s1 >> 16) & 0xff); d = te(sTl, s2 >> 24);
        o3 = __byte_perm(__byte_perm(a, b, 0x0051), __byte_perm(c, d, 0x0051), 0x5410) ^ k.rk[43];
    }
}

__device__ __forceinline__ uint32_t bswap32(uint32_t x) { return __byte_perm(x, 0, 0x0123); }

// Keystream block whose 128-bit big-endian counter is (hi:lo).
__device__ __forceinline__ uint4 aes_ctr_block(const AesKey &k, const uint32_t *sTl, uint64_t hi, uint64_t lo)
{
    uint4 o;
    aes128_encrypt(k, sTl, bswap32((uint32_t)(hi >> 32)), bswap32((uint32_t)hi),
                   bswap32((uint32_t)(lo >> 32)), bswap32((uint32_t)lo), o.x, o.y, o.z, o.w);
    return o;
}

// Upper 64 counter bits of a seeded object stream (S8(c) O3); the lower 64 bits are
// the block index.
__device__ __host__ __forceinline__ uint64_t object_iv_hi(uint32_t tag, uint32_t attempt, uint32_t inst)
{
    return ((uint64_t)(tag & 0xffu) << 56) | ((uint64_t)(attempt & 0xffffffu) << 32) | (uint64_t)inst;
}

// 8 uniform-mod-q elements of block `blk` of object (tag, inst): rejection sampling
// over attempt streams (S8(c) O4).  Returns them packed two per word, low element
// first (for q = 2^16 this is the raw keystream block).
__device__ __forceinline__ uint4 uniform_block(const AesKey &k, const uint32_t *sTl, const ModQ &mq,
                                               uint32_t tag, uint32_t inst, uint64_t blk)
{
    uint4 ks = aes_ctr_block(k, sTl, object_iv_hi(tag, 0, inst), blk);
    if (mq.T == 65536u) {
        if (mq.q == 65536u) return ks;
        uint32_t w[4] = {ks.x, ks.y, ks.z, ks.w};
#pragma unroll
        for (int i = 0; i < 4; i++)
            w[i] = mod_u32(w[i] & 0xffffu, mq) | (mod_u32(w[i] >> 16, mq) << 16);
        return make_uint4(w[0], w[1], w[2], w[3]);
    }
    uint32_t c[8] = {ks.x & 0xffffu, ks.x >> 16, ks.y & 0xffffu, ks.y >> 16,
                     ks.z & 0xffffu, ks.z >> 16, ks.w & 0xffffu, ks.w >> 16};
    uint32_t pending = 0;
#pragma unroll
    for (int i = 0; i < 8; i++) pending |= (c[i] >= mq.T) ? (1u << i) : 0u;
    for (uint32_t attempt = 1; pending; attempt++) {          // rare: P(reject) = 1 - T/65536 per element
        uint4 kr = aes_ctr_block(k, sTl, object_iv_hi(tag, attempt, inst), blk);
        uint32_t r[8] = {kr.x & 0xffffu, kr.x >> 16, kr.y & 0xffffu, kr.y >> 16,
                         kr.z & 0xffffu, kr.z >> 16, kr.w & 0xffffu, kr.w >> 16};
#pragma unroll
        for (int i = 0; i < 8; i++) {
            if (pending & (1u << i)) {
                c[i] = r[i];
                if (r[i] < mq.T) pending &= ~(1u << i);
            }
        }
    }
#pragma unroll
    for (int i = 0; i < 8; i++) c[i] = mod_u32(c[i], mq);
    return make_uint4(c[0] | (c[1] << 16), c[2] | (c[3] << 16), c[4] | (c[5] << 16), c[6] | (c[7] << 16));
}

}  // namespace lwe

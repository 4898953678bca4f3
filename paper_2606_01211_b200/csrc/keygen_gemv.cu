// keygen_gemv.cu -- a3 / a3': b = A s + e mod q (eq.(1)).
//
// HBM-bound: A (2mn bytes) is read exactly once, 16 bytes per thread per load, fully
// coalesced; everything else is noise.  The paper's kernel gives one thread a whole
// row -- on B200 that is an uncoalesced stream; here a TEAM of threads
// (a warp for short rows, the whole CTA for long ones) owns a row, so that the
// work items are small (no tail) and each load instruction covers 512 B..4 KB of
// one row.
//
// Arithmetic: s is split into bytes once per CTA and kept in shared memory packed
// for dp2a: word p = s_lo[2p] | s_lo[2p+1]<<8 | s_hi[2p]<<16 | s_hi[2p+1]<<24.  One A
// word holds two u16 elements, so
//     acc_lo = dp2a.lo(Aword, sword, acc_lo)   (+= a0*s_lo0 + a1*s_lo1)
//     acc_hi = dp2a.hi(Aword, sword, acc_hi)   (+= a0*s_hi0 + a1*s_hi1)
// costs one instruction per element with no unpacking of A.  A.s = acc_lo + 256*acc_hi.
// Each dp2a adds < 2^25, so u32 accumulators are flushed into u64 every 128 steps
// (exact for any q); for q | 2^32 wrap-around is already exact and the flush is moot.
#include "aes_ctr.cuh"

namespace lwe {

constexpr int kGemvThreads = 256;
constexpr int kRedBytes = 256;           // per-warp u64 slots of the team reduction (<= 32 warps)
constexpr int kFlushEvery = 32;          // uint4 loads between flushes: 32*4 = 128 dp2a per accumulator

__device__ __forceinline__ uint4 ldg_stream(const uint4 *p)
{
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

__device__ __forceinline__ void dot8(uint4 a, uint4 sw, uint32_t &lo, uint32_t &hi)
{
    lo = __dp2a_lo(a.x, sw.x, lo); hi = __dp2a_hi(a.x, sw.x, hi);
    lo = __dp2a_lo(a.y, sw.y, lo); hi = __dp2a_hi(a.y, sw.y, hi);
    lo = __dp2a_lo(a.z, sw.z, lo); hi = __dp2a_hi(a.z, sw.z, hi);
    lo = __dp2a_lo(a.w, sw.w, lo); hi = __dp2a_hi(a.w, sw.w, hi);
}

// pack s (n u16) into the dp2a operand layout in shared memory
__device__ __forceinline__ void pack_s_to_smem(uint32_t *sS, const uint16_t *__restrict__ s, uint32_t n)
{
    const uint32_t *s32 = reinterpret_cast<const uint32_t *>(s);
    for (uint32_t p = threadIdx.x; p < n / 2; p += blockDim.x) {
        uint32_t w = __ldg(s32 + p);                    // s[2p] | s[2p+1] << 16
        sS[p] = __byte_perm(w, 0, 0x3120);              // (b0, b2, b1, b3)
    }
    __syncthreads();
}

// barrier over one row team: the whole CTA, or TPR threads on a named barrier of their own
template <int TPR, int NT>
__device__ __forceinline__ void team_sync(uint32_t team)
{
    if (TPR == NT) __syncthreads();
    else asm volatile("bar.sync %0, %1;" ::"r"(team + 1), "n"(TPR) : "memory");
}

template <int TPR, int NT>   // threads per row team: 32 (a warp) or a multiple of 32 dividing the CTA size NT
__device__ __forceinline__ uint64_t team_reduce(uint64_t v, uint64_t *sRed)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (TPR == 32) return v;
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31, team = threadIdx.x / TPR;
    team_sync<TPR, NT>(team);                           // previous row's readers are done
    if (lane == 0) sRed[warp] = v;
    team_sync<TPR, NT>(team);
    uint64_t t = 0;
#pragma unroll
    for (int w = 0; w < TPR / 32; w++) t += sRed[team * (TPR / 32) + w];
    return t;
}

// kRegen = false: A streamed from HBM.  kRegen = true: A never read, every 16-byte
// chunk (8 elements) is one AES-CTR block of object (seed_A, LWE_TAG_A, inst 0)
// (+ rejection attempts), S8(c) O4 -- the paper's on-demand A.
template <int TPR, bool kRegen, int UNR, int NT>
__global__ void __launch_bounds__(NT)
keygen_gemv_kernel(const uint16_t *__restrict__ A, const __grid_constant__ AesKey key, const uint32_t *__restrict__ te0,
                   const uint16_t *__restrict__ s, const uint16_t *__restrict__ e, uint16_t *__restrict__ b,
                   uint32_t m, uint32_t n, uint32_t batch, ModQ mq)
{
    extern __shared__ __align__(16) uint8_t smem_raw[];
    uint32_t *sS = reinterpret_cast<uint32_t *>(smem_raw);                // n/2 words
    uint64_t *sRed = reinterpret_cast<uint64_t *>(smem_raw + 2 * (size_t)n);  // one u64 per warp
    AesTab tab = {};
    pdl_trigger();
    if (kRegen) tab = aes_table_to_smem<NT>(smem_raw + 2 * (size_t)n + kRedBytes, te0);
    pdl_wait();

    constexpr int kTeams = NT / TPR;
    const uint32_t team = threadIdx.x / TPR, tl = threadIdx.x % TPR;
    const uint32_t chunks = n / 8;                       // 16-byte chunks per row
    const uint32_t row0 = blockIdx.x * kTeams + team;
    const uint32_t row_step = gridDim.x * kTeams;
    const uint4 *sS4 = reinterpret_cast<const uint4 *>(sS);

    for (uint32_t t = 0; t < batch; t++) {
        if (t) __syncthreads();
        pack_s_to_smem(sS, s + (size_t)t * n, n);
        if (!kRegen && TPR == 32) {
            // Stored A, a warp per row: software-pipelined in registers over the warp's whole sequence of (row, batch)
            // positions -- the loads of the next batch (of this row or of the warp's next row) are issued before the
            // current batch is consumed, so a lane always has UNR..2 UNR independent 16-byte loads in flight.  With
            // load-then-consume batches the pass sat at 5.4 TB/s; a pure load loop of the same shape reaches 6.4.
            uint4 a0[UNR], a1[UNR];
            // positions are (row, first chunk of the batch) with the chunk base WARP-UNIFORM (lane tl adds tl + u * 32 and
            // masks what lies past the row's end), so that all lanes move to the next row -- and meet in its shuffle
            // reduction -- together, whatever n is
            auto load = [&](uint4 (&a)[UNR], uint32_t i, uint32_t cb) {
                const uint4 *Arow = reinterpret_cast<const uint4 *>(A + (size_t)i * n);
#pragma unroll
                for (int u = 0; u < UNR; u++) {
                    const uint32_t c = cb + tl + u * TPR;
                    if (c < chunks) a[u] = ldg_stream(Arow + c);
                    else a[u] = make_uint4(0, 0, 0, 0);
                }
            };
            uint64_t sum_lo = 0, sum_hi = 0;
            uint32_t lo = 0, hi = 0, since = 0;
            // consumes the batch at (i, cb); `last` = it is the row's last batch: reduce and write b[i]
            auto consume = [&](const uint4 (&a)[UNR], uint32_t i, uint32_t cb, bool last) {
#pragma unroll
                for (int u = 0; u < UNR; u++) {
                    const uint32_t c = cb + tl + u * TPR;
                    const uint4 sw = (c < chunks) ? sS4[c] : make_uint4(0, 0, 0, 0);
                    dot8(a[u], sw, lo, hi);
                }
                since += UNR;
                if (!mq.pow2 && (since >= kFlushEvery || last)) {
                    sum_lo += lo; sum_hi += hi; lo = 0; hi = 0; since = 0;
                }
                if (!last) return;
                uint64_t total = mq.pow2 ? (uint64_t)(lo + (hi << 8)) : sum_lo + (sum_hi << 8);   // pow2: exact mod 2^32, q | 2^32
                total = team_reduce<TPR, NT>(total, sRed);
                if (tl == 0) {
                    const uint32_t ei = e[(size_t)t * m + i];
                    const uint32_t r = mq.pow2 ? (((uint32_t)total + ei) & mq.mask) : mod_u64(total + ei, mq);
                    b[(size_t)t * m + i] = (uint16_t)r;
                }
                sum_lo = sum_hi = 0; lo = hi = 0; since = 0;
            };
            constexpr uint32_t kStep = UNR * TPR;
            uint32_t ci = row0, cb = 0;                      // current position; the next one follows below
            if (ci < m) load(a0, ci, cb);
            while (ci < m) {
                uint32_t ni = ci, nb = cb + kStep;
                if (nb >= chunks) { ni = ci + row_step; nb = 0; }
                if (ni < m) load(a1, ni, nb);
                consume(a0, ci, cb, ni != ci);
                if (ni >= m) break;
                ci = ni; cb = nb;
                ni = ci; nb = cb + kStep;
                if (nb >= chunks) { ni = ci + row_step; nb = 0; }
                if (ni < m) load(a0, ni, nb);
                consume(a1, ci, cb, ni != ci);
                ci = ni; cb = nb;
            }
            continue;
        }
        // rows are visited team-uniformly; TPR == CTA needs every thread in the loop
        for (uint32_t i = row0; i < m; i += row_step) {
            uint64_t sum_lo = 0, sum_hi = 0;
            uint32_t lo = 0, hi = 0;
            const uint4 *Arow = reinterpret_cast<const uint4 *>(A + (size_t)i * n);
            uint32_t since = 0;
            for (uint32_t c0 = tl; c0 < chunks; c0 += UNR * TPR) {
                uint4 a[UNR];
#pragma unroll
                for (int u = 0; u < UNR; u++) {
                    uint32_t c = c0 + u * TPR;
                    if (c < chunks) {
                        if (kRegen) a[u] = uniform_block(key, tab, mq, LWE_TAG_A, 0, (uint64_t)i * chunks + c);
                        else a[u] = ldg_stream(Arow + c);
                    } else {
                        a[u] = make_uint4(0, 0, 0, 0);
                    }
                }
#pragma unroll
                for (int u = 0; u < UNR; u++) {
                    uint32_t c = c0 + u * TPR;
                    uint4 sw = (c < chunks) ? sS4[c] : make_uint4(0, 0, 0, 0);
                    dot8(a[u], sw, lo, hi);
                }
                since += UNR;
                if (!mq.pow2 && since >= kFlushEvery) {
                    sum_lo += lo; sum_hi += hi; lo = 0; hi = 0; since = 0;
                }
            }
            uint64_t total;
            if (mq.pow2) total = (uint64_t)(lo + (hi << 8));              // exact mod 2^32, q | 2^32
            else total = (sum_lo + lo) + ((sum_hi + hi) << 8);
            total = team_reduce<TPR, NT>(total, sRed);
            if (tl == 0) {
                uint32_t ei = e[(size_t)t * m + i];
                uint32_t r = mq.pow2 ? (((uint32_t)total + ei) & mq.mask) : mod_u64(total + ei, mq);
                b[(size_t)t * m + i] = (uint16_t)r;
            }
        }
    }
}

template <int TPR, bool kRegen, int UNR, int NT = kGemvThreads>
static cudaError_t launch_gemv(Ctx *c, const uint16_t *d_A, const AesKey &key, const uint16_t *d_s,
                               const uint16_t *d_e, uint16_t *d_b, uint32_t batch, cudaStream_t st)
{
    const uint32_t n = c->p.n, m = c->p.m;
    size_t smem = 2 * (size_t)n + kRedBytes + (kRegen ? kAesTableBytes : 0);
    auto kern = keygen_gemv_kernel<TPR, kRegen, UNR, NT>;
    // shared-memory opt-in and occupancy: once per (context, instantiation, smem size) -- host calls, not per launch
    int per_sm = 1;
    cudaError_t perr = kernel_prepare(c, kern, smem, NT, &per_sm);
    if (perr != cudaSuccess) return perr;
    constexpr int kTeams = NT / TPR;
    uint32_t grid = (uint32_t)(c->sm_count * per_sm);
    uint32_t need = (m + kTeams - 1) / kTeams;
    if (grid > need) grid = need;
    ProfScope prof(c, kRegen ? LWE_K_KEYGEN_REGEN : LWE_K_KEYGEN_STORED, st);
    return launch_k(c, kern, grid, NT, smem, st, d_A, key, c->d_te0, d_s, d_e, d_b, m, n, batch, c->mq);
}

cudaError_t launch_keygen_stored(Ctx *c, const uint16_t *d_A, const uint16_t *d_s, const uint16_t *d_e,
                                 uint16_t *d_b, uint32_t batch, cudaStream_t st)
{
    AesKey none = {};
    // measured on B200: a warp per row; 8 x 16 B in flight per lane once a row is at least 4 KB
    if (c->p.n >= 2048) return launch_gemv<32, false, 8>(c, d_A, none, d_s, d_e, d_b, batch, st);
    return launch_gemv<32, false, 4>(c, d_A, none, d_s, d_e, d_b, batch, st);
}

cudaError_t launch_keygen_regen(Ctx *c, const AesKey &key, const uint16_t *d_s, const uint16_t *d_e,
                                uint16_t *d_b, uint32_t batch, cudaStream_t st)
{
    // one 64 KB AES table and one copy of s per CTA: large CTAs (3 row teams of 256, or 32 warp teams) keep
    // 24-32 warps per SM behind a single table.  Measured on B200 (C4, GB/s of A regenerated): 768 threads x 2
    // blocks in flight 698, 1024 x 2 663; 4 in flight spills at <= 85 registers and halves the rate
    if (c->p.n >= 4096) return launch_gemv<256, true, 2, 768>(c, nullptr, key, d_s, d_e, d_b, batch, st);
    return launch_gemv<32, true, 2, 1024>(c, nullptr, key, d_s, d_e, d_b, batch, st);
}

}  // namespace lwe

// keygen_tc.cu -- a3 for a batch of instances sharing A: B = A S + E mod q on the tensor cores
// (eq.(1) for "many concurrent key exchanges"; BJ configs[3]; S8(f) N1).
//
// Why.  A GEMV per instance re-reads A from HBM once per instance (32 x 256 MiB at C4); the
// products for all instances of a batch form a skinny GEMM that reads A ONCE.  It needs
// ~1e14 MAC/s, far beyond the CUDA cores and trivial for tcgen05, so the kernel stays
// HBM-bound on the single pass over A -- the same roofline as one GEMV.
//
// Formulation (u8 x u8 -> s32, kind::i8).  A (m x n uint16, row-major) is read in place as the
// uint8 matrix A8 (m x 2n): k' = 2j is the low byte of A[i][j], k' = 2j+1 the high byte.  Here the
// contraction index k' is the FAST axis of A8: a K-major operand, the classic TMA/UMMA layout.
// Each instance t contributes CPI K-major u8 rows to the B operand Sx (built by keygen_prep_kernel):
//     col 0: Sx[2j] = lo(s_j), Sx[2j+1] = 0         -> D0  = sum lo(A) lo(s)
//     col 1: Sx[2j] = hi(s_j), Sx[2j+1] = lo(s_j)   -> D12 = sum lo(A) hi(s) + hi(A) lo(s)   (both 2^8 terms at once)
//     col 2: Sx[2j] = 0,       Sx[2j+1] = hi(s_j)   -> D3  = sum hi(A) hi(s)
// and  b[t][i] = (D0 + 2^8 D12 + 2^16 D3 + e[t][i]) mod q,  combined in 64 bits.
//   CPI = 2 when q divides 2^16: the 2^16 D3 term vanishes mod q and col 2 is not needed; the s32 accumulators
//           may then wrap mod 2^32 harmlessly (q | 2^32).
//   CPI = 3 otherwise while D12 <= 2 * 255^2 * n < 2^31, i.e. n <= 16384;
//   CPI = 4 for larger n: the two 2^8 terms in separate columns (hi, 0) and (0, lo), every D <= 255^2 n < 2^31 for
//           n <= 33025 (the path is taken for n <= 32768).
// The S operand is re-streamed from L2 by every strip, so its width is what loads the L2->SM path beside the
// single HBM pass over A: 4 columns per instance made that path carry 2x the A stream (0.68 of HBM); 2 make it 1.5x.
//
// Shape.  One CTA owns a 128-row strip of A over the whole contraction (no split-K, no atomics):
// tile 128 x N x 128 bytes of k' per stage, N = CPI*batch rounded up (<= 256), TMA-fed
// multi-stage ring sized to fill shared memory (192 KB in flight per SM hides HBM latency), two
// TMEM accumulators so the epilogue of strip t overlaps the main loop of strip t+1.
//   warp 0: TMA producer   warp 1: TMEM alloc + MMA issuer   warps 2-5: epilogue (one lane quarter each)
#include "tc_common.cuh"

namespace lwe {

namespace {

using namespace tc;

constexpr uint32_t kTileM = 128;          // rows of A per strip
constexpr uint32_t kTileK = 128;          // bytes of k' per stage (= 64 columns of A)
constexpr uint32_t kThreads = 192;
constexpr uint32_t kMaxStages = 8;
constexpr uint32_t kSmemBudget = 208 * 1024;      // ring; + one A tile of slack + alignment + barriers <= 227 KB

__global__ void __launch_bounds__(256)
keygen_prep_kernel(const uint16_t *__restrict__ s, uint16_t *__restrict__ Sx, uint32_t n, uint32_t batch,
                   uint32_t cpi)
{
    // Sx viewed as uint16[ncols][n]: word j of a row = bytes (2j, 2j+1)
    pdl_trigger();
    pdl_wait();
    const uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t col = blockIdx.y;
    if (j >= n) return;
    const uint32_t t = col / cpi, v = col - t * cpi;
    uint32_t w = 0;
    if (t < batch) {
        const uint32_t sj = s[(size_t)t * n + j];
        const uint32_t lo = sj & 0xffu, hi = sj >> 8;
        if (cpi == 4) w = (v == 0) ? lo : (v == 1) ? hi : (v == 2) ? (lo << 8) : (hi << 8);
        else w = (v == 0) ? lo : (v == 1) ? (hi | (lo << 8)) : (hi << 8);
    }
    Sx[(size_t)col * n + j] = (uint16_t)w;
}

// Wide path (q > 65536, wide.cu): the secret is a small SIGNED integer (int8), so two operand columns per instance
// suffice for any q:  col 0: Sx[2j] = s_j, Sx[2j+1] = 0 -> D_lo = sum lo(A16) s;  col 1: Sx[2j] = 0, Sx[2j+1] = s_j ->
// D_hi = sum hi(A16) s, with the B operand read as signed int8:  t = D_lo + 2^8 D_hi + 2^16 sum_{exceptions} s_j + e.
__global__ void __launch_bounds__(256)
keygen_prep_s8_kernel(const int8_t *__restrict__ s, uint16_t *__restrict__ Sx, uint32_t n, uint32_t batch)
{
    pdl_trigger();
    pdl_wait();
    const uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t col = blockIdx.y;
    if (j >= n) return;
    const uint32_t t = col >> 1;
    uint32_t w = 0;
    if (t < batch) {
        const uint32_t sj = (uint8_t)s[(size_t)t * n + j];
        w = (col & 1u) ? (sj << 8) : sj;
    }
    Sx[(size_t)col * n + j] = (uint16_t)w;
}

// what the wide epilogue needs beside the accumulators: the exception lists of the rows and the secrets themselves
struct KgWide {
    const uint32_t *row_cnt, *row_cols;
    uint32_t cap;
    const int8_t *s;
    // 32-bit reduction of the signed sums: bias / ebias are multiples of q above |D| <= 255 * 128 * n and above
    // |e - delta * corr| (corr = sum of the secrets at the row's exceptions), delta = q - 2^16 (2^16 = -delta mod q)
    uint32_t bias, ebias, delta;
    // n > 65536 (a signed byte-plane sum holds 255 * 128 * 65536 < 2^31): the columns of A are contracted in passes of
    // <= 65536; this launch covers one pass (its `n` argument = the columns of the pass), n_full = the row length of s;
    // from the second pass on (accum) the epilogue adds the residues already in t instead of e and the exception terms
    uint32_t n_full, accum;
};

// 8 * CPI accumulator columns (= 8 instances) of this warp's 32 TMEM lanes
template <uint32_t CPI>
__device__ __forceinline__ void tmem_ld_8inst(uint32_t taddr, uint32_t (&r)[8 * CPI])
{
#pragma unroll
    for (uint32_t g = 0; g < CPI; g++)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                     : "=r"(r[8 * g]), "=r"(r[8 * g + 1]), "=r"(r[8 * g + 2]), "=r"(r[8 * g + 3]), "=r"(r[8 * g + 4]),
                       "=r"(r[8 * g + 5]), "=r"(r[8 * g + 6]), "=r"(r[8 * g + 7])
                     : "r"(taddr + 8 * g));
}

// SLABS: 128-byte K slabs per pipeline stage.  A TMA box is at most 128 bytes wide under SWIZZLE_128B, i.e. 128
// separate 128-byte pieces of 128 different rows of A; loading SLABS adjacent boxes back to back makes every
// row piece SLABS*128 contiguous bytes for the memory system.
// kWide (CPI = 2): A is the low-16 matrix of a wide context, the B operand holds signed int8 secrets, e is int8, b is
// uint32, and the epilogue adds the 2^16-weighted exceptions of its row (see keygen_prep_s8_kernel).
template <uint32_t CPI, uint32_t SLABS, bool kWide = false>
__global__ void __launch_bounds__(kThreads, 1)
keygen_tc_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapS,
                 const void *__restrict__ e_, void *__restrict__ b_, uint32_t m, uint32_t n, uint32_t batch,
                 uint32_t N, uint32_t stages, ModQ mq, uint32_t rps, KgWide wd)
{
    static_assert(!kWide || CPI == 2, "the wide path uses two signed operand columns per instance");
    const uint16_t *e = static_cast<const uint16_t *>(e_);
    uint16_t *b = static_cast<uint16_t *>(b_);
    const int8_t *e8 = static_cast<const int8_t *>(e_);
    uint32_t *b32 = static_cast<uint32_t *>(b_);
    // rps = rows of A per strip (<= 128, a multiple of 8; the TMA box of A has rps rows) and an A slab of the ring
    // holds exactly those rows (rps * 128 bytes = whole 1 KB swizzle atoms).  The MMA is always M = 128: rows rps..127 of
    // the accumulator are computed from whatever follows the slab in shared memory (the next slab, the S tiles, the next
    // stage; the allocation ends with one A tile of slack for the last stage) and are never read back.  The ring is latency-bound (a stage is released only when its MMAs have completed), so what
    // a short strip does not use buys more stages: 6 instead of 4 at the wide n = 8192 shape (56-row strips).
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;
    const uint32_t kBytesA = rps * kTileK;
    const uint32_t bytes_slab = kBytesA + N * kTileK;
    const uint32_t bytes_stage = SLABS * bytes_slab;
    const uint32_t tx_stage = SLABS * (rps * kTileK + N * kTileK);          // bytes TMA delivers per stage
    const uint32_t bars = base + stages * bytes_stage;
    auto full_bar = [&](uint32_t s) { return bars + 8 * s; };
    auto empty_bar = [&](uint32_t s) { return bars + 8 * (kMaxStages + s); };
    auto tfull_bar = [&](uint32_t a) { return bars + 8 * (2 * kMaxStages + a); };
    auto tempty_bar = [&](uint32_t a) { return bars + 8 * (2 * kMaxStages + 2 + a); };
    const uint32_t tmem_slot = bars + 8 * (2 * kMaxStages + 4);
    volatile uint32_t *tmem_slot_ptr = reinterpret_cast<volatile uint32_t *>(smem_raw + (tmem_slot - raw));

    const uint32_t warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;   // warp-uniform
    const uint32_t strips = (m + rps - 1) / rps;
    const uint32_t k_blocks = (2 * n + SLABS * kTileK - 1) / (SLABS * kTileK);      // stages per strip
    const uint32_t acc_cols = (N <= 32) ? 32 : (N <= 64) ? 64 : (N <= 128) ? 128 : 256;   // per accumulator
    const uint32_t tmem_cols = 2 * acc_cols;

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&mapA) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&mapS) : "memory");
        for (uint32_t s = 0; s < stages; s++) {
            mbar_init(full_bar(s), 1);
            mbar_init(empty_bar(s), 1);
        }
        for (uint32_t a = 0; a < 2; a++) {
            mbar_init(tfull_bar(a), 1);
            mbar_init(tempty_bar(a), 4);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    pdl_trigger();
    if (warp == 1) tmem_alloc(tmem_slot, tmem_cols);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;
    pdl_wait();                          // everything above overlapped the previous kernel; its outputs are needed now

    // warp-convergent role loops, one elected lane around the issue (see encaps_tc2.cu)
    if (warp == 0) {
        uint32_t stage = 0, phase = 0;
        for (uint32_t t = blockIdx.x; t < strips; t += gridDim.x) {
            const int32_t row0 = (int32_t)(t * rps);
            for (uint32_t kb = 0; kb < k_blocks; kb++) {
                mbar_wait(empty_bar(stage), phase ^ 1);
                const uint32_t sa = base + stage * bytes_stage;
                const int32_t k0 = (int32_t)(kb * SLABS * kTileK);
                if (elect_one()) {
                    mbar_expect_tx(full_bar(stage), tx_stage);                   // out-of-range slabs arrive as zeros
#pragma unroll
                    for (uint32_t h = 0; h < SLABS; h++)                         // 128 rows x 128 bytes of k' each
                        tma_load_2d(sa + h * kBytesA, &mapA, full_bar(stage), k0 + (int32_t)(h * kTileK), row0);
#pragma unroll
                    for (uint32_t h = 0; h < SLABS; h++)                         // N rows x 128 bytes of k' each
                        tma_load_2d(sa + SLABS * kBytesA + h * N * kTileK, &mapS, full_bar(stage),
                                    k0 + (int32_t)(h * kTileK), 0);
                }
                __syncwarp();
                if (++stage == stages) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == 1) {
        const uint32_t idesc = instr_desc_u8(kTileM, N, false, false, kWide);   // both operands K-major; wide: signed S
        uint32_t stage = 0, phase = 0, it = 0;
        for (uint32_t t = blockIdx.x; t < strips; t += gridDim.x, it++) {
            const uint32_t acc = it & 1, acc_phase = (it >> 1) & 1;
            mbar_wait(tempty_bar(acc), acc_phase ^ 1);
            tc_fence_after();
            const uint32_t d_tmem = tmem_base + acc * acc_cols;
            for (uint32_t kb = 0; kb < k_blocks; kb++) {
                mbar_wait(full_bar(stage), phase);
                tc_fence_after();
                const uint32_t sa = base + stage * bytes_stage;
                if (elect_one()) {
                    // a K step is 32 bytes along the 128-byte swizzled row: advance the start address
#pragma unroll
                    for (uint32_t h = 0; h < SLABS; h++) {
                        uint64_t adesc = make_desc_k_sw128(sa + h * kBytesA, 1024);
                        uint64_t bdesc = make_desc_k_sw128(sa + SLABS * kBytesA + h * N * kTileK, 1024);
#pragma unroll
                        for (uint32_t ks = 0; ks < kTileK / kUmmaK; ks++) {
                            umma_i8(d_tmem, adesc, bdesc, idesc, (kb | h | ks) ? 1u : 0u);
                            adesc += kUmmaK >> 4;
                            bdesc += kUmmaK >> 4;
                        }
                    }
                    umma_commit(empty_bar(stage));
                    if (kb == k_blocks - 1) umma_commit(tfull_bar(acc));
                }
                __syncwarp();
                if (++stage == stages) { stage = 0; phase ^= 1; }
            }
        }
    } else {
        // epilogue: lane = row of the strip; 8 instances (8 * CPI accumulator columns) per step
        const uint32_t quarter = warp & 3;
        uint32_t it = 0;
        for (uint32_t t = blockIdx.x; t < strips; t += gridDim.x, it++) {
            const uint32_t acc = it & 1, acc_phase = (it >> 1) & 1;
            const uint32_t rin = quarter * 32 + lane;                    // row inside the strip
            const uint32_t i = t * rps + rin;
            const bool row_ok = rin < rps && i < m;
            // e of the first 32 instances is fetched while the main loop of this strip still runs: with one strip
            // per CTA nothing else hides the epilogue, and 4 rounds of dependent global loads were ~4 us of 56
            const bool accum = kWide && wd.accum;
            uint32_t epre[32];
#pragma unroll
            for (uint32_t x = 0; x < 32; x++)
                epre[x] = (row_ok && x < batch) ? (kWide ? (accum ? b32[(size_t)x * m + i] : (uint32_t)(int)__ldg(e8 + (size_t)x * m + i))
                                                         : (uint32_t)__ldg(e + (size_t)x * m + i)) : 0u;
            const uint32_t exc = (kWide && row_ok && !accum) ? min(__ldg(wd.row_cnt + i), wd.cap) : 0u;
            if (kWide) {
                // the 2^16-weighted elements of this row (about one row in eight has one): their secrets are folded into
                // the prefetched e here, 32 independent loads per exception, while the main loop still runs.  Inside the
                // instance loop below the same sum was a dependent load chain per instance (~0.7 us each with nothing to
                // hide it: 58 us for 32 instances against 32 us for 8, ncu)
                for (uint32_t y = 0; y < exc; y++) {
                    const uint32_t col = __ldg(wd.row_cols + (size_t)i * wd.cap + y);
#pragma unroll
                    for (uint32_t x = 0; x < 32; x++)
                        if (x < batch) epre[x] -= wd.delta * (uint32_t)(int)__ldg(wd.s + (size_t)x * wd.n_full + col);
                }
            }
            mbar_wait(tfull_bar(acc), acc_phase);
            tc_fence_after();
            const uint32_t taddr = tmem_base + ((quarter * 32) << 16) + acc * acc_cols;
#pragma unroll
            for (uint32_t i0 = 0; i0 < 128; i0 += 8) {
                if (i0 >= batch) break;
                uint32_t r[8 * CPI];
                tmem_ld_8inst<CPI>(taddr + i0 * CPI, r);
                tmem_ld_wait();
                if (row_ok) {
#pragma unroll
                    for (uint32_t x = 0; x < 8; x++) {
                        const uint32_t inst = i0 + x;
                        if (inst < batch) {
                            if (kWide) {
                                if (accum) {                             // a later column pass: add to the residue in t
                                    const uint32_t old = (i0 < 32) ? epre[(i0 + x) & 31] : b32[(size_t)inst * m + i];
                                    const uint32_t add = mod_u32(mod_u32(r[2 * x] + wd.bias, mq) + 256u * mod_u32(r[2 * x + 1] + wd.bias, mq), mq);
                                    const uint32_t sum = old + add;      // < 2q
                                    b32[(size_t)inst * m + i] = sum >= mq.q ? sum - mq.q : sum;
                                    continue;
                                }
                                int ei;
                                if (i0 < 32) {
                                    ei = (int)epre[(i0 + x) & 31];           // e minus the exception terms, prefetched
                                } else {
                                    ei = (int)e8[(size_t)inst * m + i];
                                    for (uint32_t y = 0; y < exc; y++)     // elements >= 2^16 of this row: rare
                                        ei -= (int)wd.delta * (int)wd.s[(size_t)inst * wd.n_full + wd.row_cols[(size_t)i * wd.cap + y]];
                                }
                                // three 32-bit Barrett steps on biased (non-negative) values; a 64-bit remainder per
                                // element (~150 instructions) made this epilogue, not HBM, the kernel's limit
                                // (ncu: 67 us for 136 MB, DRAM 25 %)
                                b32[(size_t)inst * m + i] =
                                    mod_u32(mod_u32(r[2 * x] + wd.bias, mq) + 256u * mod_u32(r[2 * x + 1] + wd.bias, mq) +
                                            ((uint32_t)ei + wd.ebias), mq);
                                continue;
                            }
                            const uint32_t ei = (i0 < 32) ? epre[(i0 + x) & 31] : (uint32_t)e[(size_t)inst * m + i];
                            uint32_t o;
                            if (CPI == 2) {
                                o = (r[2 * x] + (r[2 * x + 1] << 8) + ei) & mq.mask;     // q | 2^16: wrap-around is exact
                            } else {
                                uint64_t tot = (CPI == 3)
                                    ? (uint64_t)r[3 * x] + ((uint64_t)r[3 * x + 1] << 8) + ((uint64_t)r[3 * x + 2] << 16)
                                    : (uint64_t)r[4 * x] + (((uint64_t)r[4 * x + 1] + r[4 * x + 2]) << 8) +
                                          ((uint64_t)r[4 * x + 3] << 16);
                                o = mod_u64(tot + ei, mq);
                            }
                            b[(size_t)inst * m + i] = (uint16_t)o;
                        }
                    }
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tempty_bar(acc));
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, tmem_cols);
}

// columns of the B operand per instance (see the header comment)
uint32_t cols_per_inst(const lwe_params &p)
{
    const bool q_divides_2_16 = (p.q & (p.q - 1)) == 0;               // q <= 65536 always
    return q_divides_2_16 ? 2u : (p.n <= 16384 ? 3u : 4u);
}
// 8 instances per epilogue step and 16-column MMA granularity: whole groups of 8 instances
uint32_t padded_cols(uint32_t batch, uint32_t cpi) { return (((batch + 7u) & ~7u) * cpi + 15u) & ~15u; }

// Ring shape for strips of rps rows and N operand columns: slabs per stage as wide as leaves >= 3 stages in flight,
// then as many stages as fit.  Returns the dynamic shared-memory size (ring + the slack an M = 128 MMA may read past a
// short last slab + alignment + barriers).
uint32_t ring_shape(uint32_t rps, uint32_t N, uint32_t *slabs, uint32_t *stages)
{
    const uint32_t bytes_slab = rps * kTileK + N * kTileK;
    *slabs = (3 * 2 * bytes_slab <= kSmemBudget) ? 2 : 1;
    const uint32_t bytes_stage = *slabs * bytes_slab;
    *stages = kSmemBudget / bytes_stage;
    if (*stages > kMaxStages) *stages = kMaxStages;
    return *stages * bytes_stage + kTileM * kTileK + 1024 + 256;
}

}  // namespace

size_t keygen_tc_workspace_bytes(const lwe_params &p)
{
    if (p.q > 65536u) {                                                 // wide context: two signed columns per instance
        const uint32_t Nw = padded_cols(p.max_batch, 2);
        return (p.n <= 262144 && Nw <= 256) ? (size_t)Nw * 2 * p.n : 0;
    }
    const uint32_t N = padded_cols(p.max_batch, cols_per_inst(p));
    return (p.n <= 32768 && N <= 256) ? (size_t)N * 2 * p.n : 0;       // 0: the tensor-core keygen is not available
}

bool keygen_tc_supported(const Ctx *c, uint32_t batch)
{
    const lwe_params &p = c->p;
    const uint32_t cpi = cols_per_inst(p);
    return c->encode_tiled != nullptr && c->d_Sx != nullptr && p.n <= 32768 && padded_cols(batch, cpi) <= 256 &&
           padded_cols(p.max_batch, cpi) <= 256;
}

cudaError_t launch_keygen_tc(Ctx *c, const uint16_t *d_A, const uint16_t *d_s, const uint16_t *d_e, uint16_t *d_b,
                             uint32_t batch, cudaStream_t st)
{
    const lwe_params &p = c->p;
    const uint32_t cpi = cols_per_inst(p);
    const uint32_t N = padded_cols(batch, cpi);
    {
        ProfScope prof(c, LWE_K_KEYGEN_PREP, st);
        dim3 grid((p.n + 255) / 256, N);
        cudaError_t err = launch_k(c, keygen_prep_kernel, grid, 256, 0, st, d_s, reinterpret_cast<uint16_t *>(c->d_Sx), p.n,
                                   batch, cpi);
        if (err != cudaSuccess) return err;
    }
    CUtensorMap mapA, mapS;
    // rows per strip: as many strips as fill whole waves of SMs (C4: 16384 rows -> 147 strips of 112 rows instead of
    // 128 strips of 128 on 148 SMs; each SM keeps its whole shared memory in flight, so more SMs = more bandwidth)
    const uint32_t waves = (p.m + kTileM * (uint32_t)c->sm_count - 1) / (kTileM * (uint32_t)c->sm_count);
    uint32_t rps = ((p.m + waves * (uint32_t)c->sm_count - 1) / (waves * (uint32_t)c->sm_count) + 7u) & ~7u;
    if (rps > kTileM) rps = kTileM;
    if (rps < 8) rps = 8;
    if (!make_map_u8(c, &mapA, d_A, 2ull * p.n, p.m, rps)) return cudaErrorInvalidValue;
    if (!make_map_u8(c, &mapS, c->d_Sx, 2ull * p.n, N, N)) return cudaErrorInvalidValue;
    uint32_t slabs, stages;
    const uint32_t smem = ring_shape(rps, N, &slabs, &stages);
    typedef void (*Kern)(const CUtensorMap, const CUtensorMap, const void *, void *, uint32_t, uint32_t, uint32_t,
                         uint32_t, uint32_t, ModQ, uint32_t, KgWide);
    static const Kern table[3][2] = {{keygen_tc_kernel<2, 1>, keygen_tc_kernel<2, 2>},
                                     {keygen_tc_kernel<3, 1>, keygen_tc_kernel<3, 2>},
                                     {keygen_tc_kernel<4, 1>, keygen_tc_kernel<4, 2>}};
    Kern kern = table[cpi - 2][slabs - 1];
    cudaError_t perr = kernel_prepare(c, kern, smem);
    if (perr != cudaSuccess) return perr;
    const uint32_t strips = (p.m + rps - 1) / rps;
    const uint32_t grid = strips < (uint32_t)c->sm_count ? strips : (uint32_t)c->sm_count;
    ProfScope prof(c, LWE_K_KEYGEN_TC, st);
    return launch_k(c, kern, grid, kThreads, smem, st, mapA, mapS, d_e, d_b, p.m, p.n, batch, N, stages, c->mq, rps, KgWide{});
}

// ---- wide path: t = A s + e on uint32 residues, A = the context's packed matrix (wide.cu)
bool wide_keygen_tc_supported(const Ctx *c, uint32_t batch)
{
    // |D| <= 255 * 128 * n < 2^31 for n <= 65536: longer rows are contracted in column passes of 65536
    return c->encode_tiled != nullptr && c->d_Sx != nullptr && c->p.n <= 262144 && padded_cols(batch, 2) <= 256 &&
           padded_cols(c->p.max_batch, 2) <= 256;
}

cudaError_t launch_wide_keygen_tc(Ctx *c, const int8_t *d_s, const int8_t *d_e, uint32_t *d_t, uint32_t batch, cudaStream_t st)
{
    const lwe_params &p = c->p;
    const uint32_t N = padded_cols(batch, 2);
    {
        ProfScope prof(c, LWE_K_KEYGEN_PREP, st);
        dim3 grid((p.n + 255) / 256, N);
        cudaError_t err = launch_k(c, keygen_prep_s8_kernel, grid, 256, 0, st, d_s, reinterpret_cast<uint16_t *>(c->d_Sx),
                                   p.n, batch);
        if (err != cudaSuccess) return err;
    }
    const uint32_t waves = (p.m + kTileM * (uint32_t)c->sm_count - 1) / (kTileM * (uint32_t)c->sm_count);
    uint32_t rps = ((p.m + waves * (uint32_t)c->sm_count - 1) / (waves * (uint32_t)c->sm_count) + 7u) & ~7u;
    if (rps > kTileM) rps = kTileM;
    if (rps < 8) rps = 8;
    uint32_t slabs, stages;
    const uint32_t smem = ring_shape(rps, N, &slabs, &stages);
    auto kern = slabs == 2 ? keygen_tc_kernel<2, 2, true> : keygen_tc_kernel<2, 1, true>;
    cudaError_t perr = kernel_prepare(c, kern, smem);
    if (perr != cudaSuccess) return perr;
    const uint32_t strips = (p.m + rps - 1) / rps;
    const uint32_t grid = strips < (uint32_t)c->sm_count ? strips : (uint32_t)c->sm_count;
    const uint64_t q = p.q, delta = q - 65536u;
    // column passes of <= 65536 (Table 1's n = 131072 row: two): each a column range of A16 and of the operand rows,
    // mapped with the full row pitch; the first adds e and the exception terms, the later ones add to t
    const uint32_t step = p.n < 65536u ? p.n : 65536u;
    for (uint32_t col0 = 0; col0 < p.n; col0 += step) {
        const uint32_t cols = (p.n - col0 < step) ? (p.n - col0) : step;
        CUtensorMap mapA, mapS;
        if (!make_map_u8(c, &mapA, c->d_A16 + col0, 2ull * cols, p.m, rps, 2ull * p.n)) return cudaErrorInvalidValue;
        if (!make_map_u8(c, &mapS, c->d_Sx + 2ull * col0, 2ull * cols, N, N, 2ull * p.n)) return cudaErrorInvalidValue;
        const uint64_t plane_max = 255ull * 128ull * cols, e_max = 128ull + delta * 128ull * c->exc_cap_row;
        const KgWide wd = {c->d_exc_row_cnt, c->d_exc_row_cols, c->exc_cap_row, d_s,
                           (uint32_t)((plane_max + q - 1) / q * q), (uint32_t)((e_max + q - 1) / q * q), (uint32_t)delta,
                           p.n, col0 ? 1u : 0u};
        ProfScope prof(c, LWE_K_KEYGEN_TC, st);
        cudaError_t err = launch_k(c, kern, grid, kThreads, smem, st, mapA, mapS, d_e, d_t, p.m, cols, batch, N, stages, c->mq,
                                   rps, wd);
        if (err != cudaSuccess) return err;
    }
    return cudaSuccess;
}

}  // namespace lwe

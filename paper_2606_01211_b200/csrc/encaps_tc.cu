// encaps_tc.cu -- a4: U = A^T R mod q as a tcgen05 kind::i8 GEMM (BJ north_star (3);
// the bit-batched contraction of P:L136-148).
//
// Formulation.  The little-endian uint16 matrix A (m x n) is read, unchanged, as a
// uint8 matrix A8 (m x 2n): byte-column 2j is the low byte plane of column j, 2j+1 the
// high plane.  One GEMM  D[2n x N] = A8^T . Rexp  (u8 x u8 -> s32, N = batch*k, K = m)
// therefore yields acc_lo in even rows and acc_hi in odd rows with no split pass, and
//   U[j][c] = (D[2j][c] + 256*D[2j+1][c]) mod q.
// Bounds (m <= 65536): D <= 255*m < 2^31; D_lo + 256*D_hi <= 65535*m < 2^32.
//
// Operand major-ness.  The contraction index i is the SLOW axis of both A8 (row-major
// m x 2n) and Rexp (m x N): both operands are "MN-major".  tcgen05 accepts MN-major
// 8-bit operands (instruction-descriptor bits 15/16), and the canonical MN-major
// SWIZZLE_128B shared-memory layout (rows of 128 bytes along M/N, 8 K-rows per 1 KB
// atom) is exactly what a TMA box {128 bytes, K rows} with CU_TENSOR_MAP_SWIZZLE_128B
// writes -- so A is consumed in place: no transpose, no plane split, no second copy.
//
// Kernel shape (v1): persistent, one CTA per SM, cta_group::1, tile 128 (byte-rows
// of D = 64 columns of A) x 256 (= one instance when k = 256) x K_TILE 128 per stage,
// 4-stage TMA->smem ring, two 256-column TMEM accumulators so the epilogue of tile t
// overlaps the main loop of tile t+1.
//   warp 0 : TMA producer (1 lane)      warp 1 : TMEM alloc + MMA issuer (1 lane)
//   warps 2-5 : epilogue, one TMEM lane quarter each: tcgen05.ld -> pair lo/hi lanes by
//               shuffle -> mod q -> 32-byte stores into U[t][j][c]
#include "tc_common.cuh"

namespace lwe {

namespace {

using namespace tc;

constexpr uint32_t kTileM = 128;      // bytes of A8 row = 64 u16 columns of A
constexpr uint32_t kTileN = 256;
constexpr uint32_t kTileK = 128;      // rows of A / R per pipeline stage
constexpr uint32_t kStages = 4;
constexpr uint32_t kBytesA = kTileM * kTileK;              // 16 KB
constexpr uint32_t kBytesBHalf = 128 * kTileK;             // 16 KB per 128-column half
constexpr uint32_t kBytesStage = kBytesA + 2 * kBytesBHalf; // 48 KB
constexpr uint32_t kThreads = 192;
constexpr uint32_t kTmemCols = 512;
constexpr uint32_t kSmemBytes = kStages * kBytesStage + 1024 /*align*/ + 256 /*barriers*/;

constexpr uint32_t kInstrDesc = instr_desc_u8(kTileM, kTileN, true, true);     // both operands MN-major

struct TileSched {
    uint32_t m_tiles, n_tiles, total;
    __device__ __forceinline__ void coords(uint32_t t, uint32_t &mt, uint32_t &nt) const
    {
        // groups of 8 n-tiles; inside a group n varies fastest, then m: CTAs running at the
        // same time share A strips (L2) and the group's R panels stay L2-resident.
        const uint32_t g = 8;
        uint32_t per_group = m_tiles * g;
        uint32_t grp = t / per_group, r = t - grp * per_group;
        uint32_t width = (n_tiles - grp * g) < g ? (n_tiles - grp * g) : g;
        mt = r / width;
        nt = grp * g + (r - mt * width);
    }
};

template <int kMode>
__global__ void __launch_bounds__(kThreads, 1)
encaps_tc_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapR,
                 uint16_t *__restrict__ U, uint32_t *__restrict__ flags, uint32_t m, uint32_t n, uint32_t k,
                 uint32_t ncols_total, ModQ mq)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;                 // SWIZZLE_128B atoms need 1 KB alignment
    const uint32_t bars = base + kStages * kBytesStage;           // barrier block (8-byte aligned)
    // barrier layout: full[kStages], empty[kStages], tmem_full[2], tmem_empty[2], then the TMEM base word
    auto full_bar = [&](uint32_t s) { return bars + 8 * s; };
    auto empty_bar = [&](uint32_t s) { return bars + 8 * (kStages + s); };
    auto tfull_bar = [&](uint32_t a) { return bars + 8 * (2 * kStages + a); };
    auto tempty_bar = [&](uint32_t a) { return bars + 8 * (2 * kStages + 2 + a); };
    const uint32_t tmem_slot = bars + 8 * (2 * kStages + 4);
    volatile uint32_t *tmem_slot_ptr = reinterpret_cast<volatile uint32_t *>(smem_raw + (tmem_slot - raw));

    const uint32_t warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;   // warp-uniform

    TileSched sched;
    sched.m_tiles = (2 * n + kTileM - 1) / kTileM;
    sched.n_tiles = (ncols_total + kTileN - 1) / kTileN;
    sched.total = sched.m_tiles * sched.n_tiles;
    const uint32_t k_blocks = (m + kTileK - 1) / kTileK;

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&mapA) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&mapR) : "memory");
        for (uint32_t s = 0; s < kStages; s++) {
            mbar_init(full_bar(s), 1);
            mbar_init(empty_bar(s), 1);
        }
        for (uint32_t a = 0; a < 2; a++) {
            mbar_init(tfull_bar(a), 1);
            mbar_init(tempty_bar(a), 4);                            // one arrival per epilogue warp
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) tmem_alloc(tmem_slot, kTmemCols);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    // warp-convergent role loops, one elected lane around the issue (see encaps_tc2.cu)
    if (warp == 0) {
        // ===================== TMA producer =====================
        uint32_t stage = 0, phase = 0;
        for (uint32_t t = blockIdx.x; t < sched.total; t += gridDim.x) {
            uint32_t mt, nt;
            sched.coords(t, mt, nt);
            const int32_t a_col = (int32_t)(mt * kTileM), r_col = (int32_t)(nt * kTileN);
            for (uint32_t kb = 0; kb < k_blocks; kb++) {
                mbar_wait(empty_bar(stage), phase ^ 1);
                const uint32_t sa = base + stage * kBytesStage;
                const int32_t row = (int32_t)(kb * kTileK);
                if (elect_one()) {
                    mbar_expect_tx(full_bar(stage), kBytesStage);
                    tma_load_2d(sa, &mapA, full_bar(stage), a_col, row);
                    tma_load_2d(sa + kBytesA, &mapR, full_bar(stage), r_col, row);
                    tma_load_2d(sa + kBytesA + kBytesBHalf, &mapR, full_bar(stage), r_col + 128, row);
                }
                __syncwarp();
                if (++stage == kStages) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer =====================
        uint32_t stage = 0, phase = 0, it = 0;
        for (uint32_t t = blockIdx.x; t < sched.total; t += gridDim.x, it++) {
            const uint32_t acc = it & 1, acc_phase = (it >> 1) & 1;
            mbar_wait(tempty_bar(acc), acc_phase ^ 1);          // epilogue has drained this accumulator
            tc_fence_after();
            const uint32_t d_tmem = tmem_base + acc * kTileN;
            for (uint32_t kb = 0; kb < k_blocks; kb++) {
                mbar_wait(full_bar(stage), phase);
                tc_fence_after();
                const uint32_t sa = base + stage * kBytesStage;
                if (elect_one()) {
                    // K step = 32 rows of 128 bytes = 4 KB in both operands: one add on the address field
                    uint64_t adesc = make_desc_mn_sw128(sa, 0, 1024);
                    uint64_t bdesc = make_desc_mn_sw128(sa + kBytesA, kBytesBHalf, 1024);
#pragma unroll
                    for (uint32_t ks = 0; ks < kTileK / kUmmaK; ks++) {
                        umma_i8(d_tmem, adesc, bdesc, kInstrDesc, (kb | ks) ? 1u : 0u);
                        adesc += (kUmmaK * 128) >> 4;
                        bdesc += (kUmmaK * 128) >> 4;
                    }
                    umma_commit(empty_bar(stage));                  // smem slot free once these MMAs retire
                    if (kb == k_blocks - 1) umma_commit(tfull_bar(acc));
                }
                __syncwarp();
                if (++stage == kStages) { stage = 0; phase ^= 1; }
            }
        }
    } else {
        // ===================== epilogue (warps 2..5) =====================
        const uint32_t quarter = warp & 3;                          // TMEM lanes 32*quarter .. +31
        uint32_t it = 0;
        for (uint32_t t = blockIdx.x; t < sched.total; t += gridDim.x, it++) {
            uint32_t mt, nt;
            sched.coords(t, mt, nt);
            const uint32_t acc = it & 1, acc_phase = (it >> 1) & 1;
            mbar_wait(tfull_bar(acc), acc_phase);
            tc_fence_after();
            const uint32_t brow = mt * kTileM + quarter * 32 + lane;   // byte-row of D
            const uint32_t j = brow >> 1;                             // column of A / row of U
            const bool odd = lane & 1;
            const uint32_t taddr = tmem_base + ((quarter * 32) << 16) + acc * kTileN;
            MismatchAcc mism;
#pragma unroll 1
            for (uint32_t cb = 0; cb < kTileN; cb += 32) {
                uint32_t r[32];
                tmem_ld_32x32b_x32(taddr + cb, r);
                tmem_ld_wait();
                uint32_t o[16];
#pragma unroll
                for (int x = 0; x < 16; x++) {
                    uint32_t send = odd ? r[x] : r[16 + x];
                    uint32_t recv = __shfl_xor_sync(0xffffffffu, send, 1);
                    uint32_t val = odd ? (recv + (r[16 + x] << 8)) : (r[x] + (recv << 8));
                    o[x] = mq.pow2 ? (val & mq.mask) : mod_u32(val, mq);
                }
                const uint32_t col = nt * kTileN + cb + (odd ? 16u : 0u);   // first of my 16 columns
                if (j < n && col < ncols_total) {
                    const uint32_t inst = col / k, c = col - inst * k;
                    const bool bad = store_u16x16<kMode>(reinterpret_cast<uint4 *>(U + ((size_t)inst * n + j) * k + c), o, mq);
                    if (kMode == kEpiCompare) mism.note(flags, inst, bad);
                }
            }
            if (kMode == kEpiCompare) mism.flush_warp(flags);
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tempty_bar(acc));
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, kTmemCols);
}

}  // namespace

bool encaps_tc_supported(const Ctx *c, uint32_t batch)
{
    const lwe_params &p = c->p;
    // m is not limited here: the callers pass row panels of at most 65536 rows (a byte-plane sum <= 255 * 65536)
    return c->encode_tiled != nullptr && p.k % 16 == 0 && (2ull * p.n) % 16 == 0 && ((uint64_t)batch * p.k) % 16 == 0;
}

cudaError_t launch_encaps_tc(Ctx *c, const uint16_t *d_A, uint16_t *d_U, uint32_t batch, uint32_t row0, uint32_t rows,
                             int mode, uint32_t *d_flags, cudaStream_t st)
{
    const lwe_params &p = c->p;
    const uint32_t ncols = batch * p.k;
    CUtensorMap mapA, mapR;
    // d_A holds rows [row0, row0 + rows) of A (the whole matrix when row0 = 0, rows = m)
    if (!make_map_u8(c, &mapA, d_A, 2ull * p.n, rows, kTileK)) return cudaErrorInvalidValue;
    if (!make_map_u8(c, &mapR, c->d_Rexp + (size_t)row0 * ncols, ncols, rows, kTileK)) return cudaErrorInvalidValue;
    auto kern = mode == kEpiAccum ? encaps_tc_kernel<kEpiAccum>
              : mode == kEpiCompare ? encaps_tc_kernel<kEpiCompare> : encaps_tc_kernel<kEpiStore>;
    cudaError_t err = kernel_prepare(c, kern, kSmemBytes);
    if (err != cudaSuccess) return err;
    const uint32_t tiles = ((2 * p.n + kTileM - 1) / kTileM) * ((ncols + kTileN - 1) / kTileN);
    uint32_t grid = tiles < (uint32_t)c->sm_count ? tiles : (uint32_t)c->sm_count;
    ProfScope prof(c, LWE_K_ENCAPS_TC, st);
    kern<<<grid, kThreads, kSmemBytes, st>>>(mapA, mapR, d_U, d_flags, rows, p.n, p.k, ncols, c->mq);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace lwe

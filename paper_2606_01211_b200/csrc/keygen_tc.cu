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
// Each instance t contributes four K-major u8 rows to the B operand Sx (built by keygen_prep_kernel):
//     col 4t+0: Sx[2j] = lo(s_j), Sx[2j+1] = 0         -> D0 = sum lo(A) lo(s)
//     col 4t+1: Sx[2j] = hi(s_j), Sx[2j+1] = 0         -> D1 = sum lo(A) hi(s)
//     col 4t+2: Sx[2j] = 0,       Sx[2j+1] = lo(s_j)   -> D2 = sum hi(A) lo(s)
//     col 4t+3: Sx[2j] = 0,       Sx[2j+1] = hi(s_j)   -> D3 = sum hi(A) hi(s)
// and  b[t][i] = (D0 + 2^8 (D1 + D2) + 2^16 D3 + e[t][i]) mod q,  combined in 64 bits.
// Bounds: every D <= 255^2 n < 2^31 for n <= 33025 (the path is taken for n <= 32768).
//
// Shape.  One CTA owns a 128-row strip of A over the whole contraction (no split-K, no atomics):
// tile 128 x N x 128 bytes of k' per stage, N = 4*batch rounded up to 16 (<= 256), TMA-fed
// multi-stage ring sized to fill shared memory (192 KB in flight per SM hides HBM latency), two
// TMEM accumulators so the epilogue of strip t overlaps the main loop of strip t+1.
//   warp 0: TMA producer   warp 1: TMEM alloc + MMA issuer   warps 2-5: epilogue (one lane quarter each)
#include "tc_common.cuh"

namespace lwe {

namespace {

using namespace tc;

constexpr uint32_t kTileM = 128;          // rows of A per strip
constexpr uint32_t kTileK = 128;          // bytes of k' per stage (= 64 columns of A)
constexpr uint32_t kBytesA = kTileM * kTileK;
constexpr uint32_t kThreads = 192;
constexpr uint32_t kMaxStages = 8;
constexpr uint32_t kSmemBudget = 200 * 1024;

__global__ void __launch_bounds__(256)
keygen_prep_kernel(const uint16_t *__restrict__ s, uint16_t *__restrict__ Sx, uint32_t n, uint32_t batch,
                   uint32_t ncols)
{
    // Sx viewed as uint16[ncols][n]: word j of a row = bytes (2j, 2j+1)
    const uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t col = blockIdx.y;
    if (j >= n) return;
    const uint32_t t = col >> 2, v = col & 3;
    uint32_t w = 0;
    if (t < batch) {
        const uint32_t sj = s[(size_t)t * n + j];
        w = (v == 0) ? (sj & 0xffu) : (v == 1) ? (sj >> 8) : (v == 2) ? ((sj & 0xffu) << 8) : (sj & 0xff00u);
    }
    Sx[(size_t)col * n + j] = (uint16_t)w;
}

__global__ void __launch_bounds__(kThreads, 1)
keygen_tc_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapS,
                 const uint16_t *__restrict__ e, uint16_t *__restrict__ b, uint32_t m, uint32_t n, uint32_t batch,
                 uint32_t N, uint32_t stages, ModQ mq)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;
    const uint32_t bytes_stage = kBytesA + N * kTileK;
    const uint32_t bars = base + stages * bytes_stage;
    auto full_bar = [&](uint32_t s) { return bars + 8 * s; };
    auto empty_bar = [&](uint32_t s) { return bars + 8 * (kMaxStages + s); };
    auto tfull_bar = [&](uint32_t a) { return bars + 8 * (2 * kMaxStages + a); };
    auto tempty_bar = [&](uint32_t a) { return bars + 8 * (2 * kMaxStages + 2 + a); };
    const uint32_t tmem_slot = bars + 8 * (2 * kMaxStages + 4);
    volatile uint32_t *tmem_slot_ptr = reinterpret_cast<volatile uint32_t *>(smem_raw + (tmem_slot - raw));

    const uint32_t warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;   // warp-uniform
    const uint32_t strips = (m + kTileM - 1) / kTileM;
    const uint32_t k_blocks = (2 * n + kTileK - 1) / kTileK;
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
    if (warp == 1) tmem_alloc(tmem_slot, tmem_cols);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    // warp-convergent role loops, one elected lane around the issue (see encaps_tc2.cu)
    if (warp == 0) {
        uint32_t stage = 0, phase = 0;
        for (uint32_t t = blockIdx.x; t < strips; t += gridDim.x) {
            const int32_t row0 = (int32_t)(t * kTileM);
            for (uint32_t kb = 0; kb < k_blocks; kb++) {
                mbar_wait(empty_bar(stage), phase ^ 1);
                const uint32_t sa = base + stage * bytes_stage;
                const int32_t k0 = (int32_t)(kb * kTileK);
                if (elect_one()) {
                    mbar_expect_tx(full_bar(stage), bytes_stage);
                    tma_load_2d(sa, &mapA, full_bar(stage), k0, row0);          // 128 rows x 128 bytes of k'
                    tma_load_2d(sa + kBytesA, &mapS, full_bar(stage), k0, 0);   // N rows x 128 bytes of k'
                }
                __syncwarp();
                if (++stage == stages) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == 1) {
        const uint32_t idesc = instr_desc_u8(kTileM, N, false, false);      // both operands K-major
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
                    uint64_t adesc = make_desc_k_sw128(sa, 1024);
                    uint64_t bdesc = make_desc_k_sw128(sa + kBytesA, 1024);
#pragma unroll
                    for (uint32_t ks = 0; ks < kTileK / kUmmaK; ks++) {
                        umma_i8(d_tmem, adesc, bdesc, idesc, (kb | ks) ? 1u : 0u);
                        adesc += kUmmaK >> 4;
                        bdesc += kUmmaK >> 4;
                    }
                    umma_commit(empty_bar(stage));
                    if (kb == k_blocks - 1) umma_commit(tfull_bar(acc));
                }
                __syncwarp();
                if (++stage == stages) { stage = 0; phase ^= 1; }
            }
        }
    } else {
        // epilogue: lane = row of the strip; 32 accumulator columns = 8 instances per tcgen05.ld
        const uint32_t quarter = warp & 3;
        uint32_t it = 0;
        for (uint32_t t = blockIdx.x; t < strips; t += gridDim.x, it++) {
            const uint32_t acc = it & 1, acc_phase = (it >> 1) & 1;
            mbar_wait(tfull_bar(acc), acc_phase);
            tc_fence_after();
            const uint32_t i = t * kTileM + quarter * 32 + lane;
            const uint32_t taddr = tmem_base + ((quarter * 32) << 16) + acc * acc_cols;
#pragma unroll 1
            for (uint32_t cb = 0; cb < 4 * batch; cb += 32) {
                uint32_t r[32];
                tmem_ld_32x32b_x32(taddr + cb, r);
                tmem_ld_wait();
                if (i < m) {
#pragma unroll
                    for (uint32_t x = 0; x < 8; x++) {
                        const uint32_t inst = (cb >> 2) + x;
                        if (inst < batch) {
                            uint64_t tot = (uint64_t)r[4 * x] + (((uint64_t)r[4 * x + 1] + r[4 * x + 2]) << 8) +
                                           ((uint64_t)r[4 * x + 3] << 16) + e[(size_t)inst * m + i];
                            uint32_t o = mq.pow2 ? ((uint32_t)tot & mq.mask) : mod_u64(tot, mq);
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

uint32_t padded_cols(uint32_t batch) { return (4 * batch + 15u) & ~15u; }

}  // namespace

size_t keygen_tc_workspace_bytes(const lwe_params &p)
{
    return (size_t)padded_cols(p.max_batch) * 2 * p.n;
}

bool keygen_tc_supported(const Ctx *c, uint32_t batch)
{
    const lwe_params &p = c->p;
    return c->encode_tiled != nullptr && c->d_Sx != nullptr && p.n <= 32768 && padded_cols(batch) <= 256 &&
           padded_cols(p.max_batch) <= 256;
}

cudaError_t launch_keygen_tc(Ctx *c, const uint16_t *d_A, const uint16_t *d_s, const uint16_t *d_e, uint16_t *d_b,
                             uint32_t batch, cudaStream_t st)
{
    const lwe_params &p = c->p;
    const uint32_t N = padded_cols(batch);
    {
        ProfScope prof(c, LWE_K_KEYGEN_PREP, st);
        dim3 grid((p.n + 255) / 256, N);
        keygen_prep_kernel<<<grid, 256, 0, st>>>(d_s, reinterpret_cast<uint16_t *>(c->d_Sx), p.n, batch, N);
        c->launches++;
        cudaError_t err = cudaGetLastError();
        if (err != cudaSuccess) return err;
    }
    CUtensorMap mapA, mapS;
    if (!make_map_u8(c, &mapA, d_A, 2ull * p.n, p.m, kTileM)) return cudaErrorInvalidValue;
    if (!make_map_u8(c, &mapS, c->d_Sx, 2ull * p.n, N, N)) return cudaErrorInvalidValue;
    const uint32_t bytes_stage = kBytesA + N * kTileK;
    uint32_t stages = kSmemBudget / bytes_stage;
    if (stages > kMaxStages) stages = kMaxStages;
    const uint32_t smem = stages * bytes_stage + 1024 + 256;
    static int configured = 0;
    if (!configured) {
        cudaError_t err = cudaFuncSetAttribute(keygen_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                               (int)(kSmemBudget + 1024 + 256));
        if (err != cudaSuccess) return err;
        configured = 1;
    }
    const uint32_t strips = (p.m + kTileM - 1) / kTileM;
    const uint32_t grid = strips < (uint32_t)c->sm_count ? strips : (uint32_t)c->sm_count;
    ProfScope prof(c, LWE_K_KEYGEN_TC, st);
    keygen_tc_kernel<<<grid, kThreads, smem, st>>>(mapA, mapS, d_e, d_b, p.m, p.n, batch, N, stages, c->mq);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace lwe

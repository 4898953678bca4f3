// probe_int8.cu -- measurement hook: the int8 tensor pipe's own rate on this GPU (S8(d) "Denominators": a
// box-measured int8 peak to divide the encaps GEMM by).
//
// Every SM pair (cluster of two CTAs, as in encaps_tc2.cu) issues the product's own instruction --
// tcgen05.mma.cta_group::2.kind::i8, M = 256, N = 256, K = 32, MN-major SWIZZLE_128B operands, s32 accumulators in
// TMEM -- back to back on operand tiles that already sit in shared memory: no TMA, no global loads, no epilogue.
// Four K steps per 128-row stage and one tcgen05.commit per stage, exactly the product's cadence, over a ring of
// kStages resident stages and two alternating TMEM accumulators; the issuing thread runs at most kDepth commits
// ahead of the pipe.  Operand contents are pseudo-random bytes (the data the pipe toggles sets its power draw, and
// on a power-capped chip its clock): A = uniform u8 like the byte planes of a uniform A; B = {0,1} bytes (mode 0, the
// binary R of the KEM) or dense s8 (mode 1, the signed operand of the paper's own PKE / a library GEMM's data).
// Nothing is computed for anyone: the accumulators are never read.
#include "tc_common.cuh"

namespace lwe {

using namespace tc;

namespace {

constexpr uint32_t kStages = 4, kTileK = 128, kCtaM = 128, kHalfN = 128, kDepth = 8;
constexpr uint32_t kBytesA = kCtaM * kTileK, kBytesB = kHalfN * kTileK, kBytesStage = kBytesA + kBytesB;
constexpr uint32_t kSmem = kStages * kBytesStage + 1024 + 256;
constexpr uint32_t kThreads = 128;
constexpr uint32_t kDescU8 = instr_desc_u8(256, 256, true, true, false);
constexpr uint32_t kDescS8 = instr_desc_u8(256, 256, true, true, true);

__device__ __forceinline__ uint32_t mix(uint32_t x)
{
    x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
    return x;
}

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads, 1)
probe_int8_kernel(uint32_t iters, uint32_t signed_dense_b)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;
    const uint32_t bars = base + kStages * kBytesStage;
    auto done_bar = [&](uint32_t s) { return bars + 8 * s; };
    const uint32_t tmem_slot = bars + 8 * kDepth;
    volatile uint32_t *tmem_slot_ptr = reinterpret_cast<volatile uint32_t *>(smem_raw + (tmem_slot - raw));
    const uint32_t warp = threadIdx.x >> 5, rank = cluster_ctarank();

    // operand tiles: written once by the CTA's own threads (generic proxy), then fenced into the async proxy
    uint32_t *tiles = reinterpret_cast<uint32_t *>(smem_raw + (base - raw));
    for (uint32_t w = threadIdx.x; w < kStages * kBytesStage / 4; w += kThreads) {
        uint32_t r = mix(w * 2654435761u + blockIdx.x * 40503u + 1u);
        const bool is_b = (w * 4) % kBytesStage >= kBytesA;
        if (is_b && !signed_dense_b) r &= 0x01010101u;
        tiles[w] = r;
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    if (warp == 0 && (threadIdx.x & 31) == 0) {
        for (uint32_t s = 0; s < kDepth; s++) mbar_init(done_bar(s), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) tmem_alloc_pair(tmem_slot, 512);
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    if (warp == 1 && rank == 0) {
        const uint32_t idesc = signed_dense_b ? kDescS8 : kDescU8;
        uint32_t slot = 0, phase = 0, stage = 0;
        for (uint32_t it = 0; it < iters; it++) {
            if (it >= kDepth) mbar_wait(done_bar(slot), phase ^ 1);        // the commit issued kDepth stages ago
            const uint32_t sa = base + stage * kBytesStage;
            const uint32_t d_tmem = tmem_base + ((it >> 5) & 1) * 256;     // 32 stages (4096 rows of K) per accumulator
            if (elect_one()) {
                uint64_t adesc = make_desc_mn_sw128(sa, 0, 1024);
                uint64_t bdesc = make_desc_mn_sw128(sa + kBytesA, 0, 1024);
#pragma unroll
                for (uint32_t ks = 0; ks < kTileK / kUmmaK; ks++) {
                    umma_i8_pair(d_tmem, adesc, bdesc, idesc, ((it & 31) | ks) ? 1u : 0u);
                    adesc += (kUmmaK * 128) >> 4;
                    bdesc += (kUmmaK * 128) >> 4;
                }
                umma_commit_pair(done_bar(slot), 0x1);                     // arrives in the leader only
            }
            __syncwarp();
            if (++stage == kStages) stage = 0;
            if (++slot == kDepth) { slot = 0; phase ^= 1; }
        }
        // drain: the last commit on every barrier (its j-th completion is waited for with parity j & 1)
        for (uint32_t s = 0; s < kDepth && s < iters; s++) {
            const uint32_t commits = (iters - s + kDepth - 1) / kDepth;
            mbar_wait(done_bar(s), (commits - 1) & 1);
        }
        tc_fence_after();
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    if (warp == 1) tmem_dealloc_pair(tmem_base, 512);
}

}  // namespace

// ops of one launch = pairs * iters * 4 MMAs * 2 * 256 * 256 * 32
cudaError_t launch_probe_int8(Ctx *c, uint32_t iters, int signed_dense_b, uint64_t *ops, cudaStream_t st)
{
    cudaError_t e = kernel_prepare(c, probe_int8_kernel, kSmem);
    if (e != cudaSuccess) return e;
    const uint32_t pairs = (uint32_t)c->sm_count / 2;
    if (ops) *ops = (uint64_t)pairs * iters * (kTileK / kUmmaK) * 2ull * 256ull * 256ull * kUmmaK;
    probe_int8_kernel<<<2 * pairs, kThreads, kSmem, st>>>(iters, signed_dense_b ? 1u : 0u);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace lwe

// encaps_regen_tc.cu -- a4 with A never stored, S8(f) N4: the AES-CTR generator fused into the producer of the
// tcgen05 GEMM U = A^T R mod q ("on-demand matrix element generation"; BJ configs[4] "regenerated
// on the fly"; BJ north_star (1)+(3)).
//
// Why.  lwe_encaps(d_A == NULL) used to regenerate A one row panel at a time into HBM and run the stored-A GEMM on
// each panel: every byte of A was written to HBM once and read back once, and the generator and the tensor pipe
// took turns.  For one instance (N = k <= 256 columns) every A tile is consumed by exactly one MMA tile, so the
// tile can be generated straight into the shared-memory operand buffer: A never exists in HBM at all, and the
// MMAs, the R loads and the epilogue hide completely under the generator, which is what bounds the kernel
// (ALU/LDS: 160 table lookups per 16-byte block).
//
// Layout identity that makes this cheap.  The GEMM reads A in place as the u8 matrix A8 (m x 2n), an MN-major
// operand whose canonical SWIZZLE_128B tile is "rows of 128 bytes along M, 8 K-rows per 1 KB atom, 16-byte chunk
// c of row r stored at chunk c ^ (r & 7)" -- and 128 bytes of a row of A8 are exactly 8 consecutive AES-CTR
// blocks of the counter-indexed stream of A (S8(c) O3/O4: block index = (i n + j) / 8).  So one generator thread
// produces one 16-byte chunk and stores it with one st.shared.v4 at its swizzled position; what TMA would have
// written is reproduced bit for bit.
//
// Shape.  Persistent, one CTA per SM, cta_group::1, tile 128 byte-rows of D (= 64 columns of A) x 256 x kTileK.
//   warp 0        : TMA producer of the R tile (2 boxes of 128 columns), expect_tx on full[s]
//   warp 1        : TMEM alloc + MMA issuer
//   warps 2-5     : epilogue (one TMEM lane quarter each)
//   warps 6..6+G-1: generators; warp g owns rows 8g..8g+7 of the stage (kTileK = 8 G), two AES blocks in flight
//                   per thread; after its stores: fence.proxy.async (generic -> async proxy), one arrive on full[s]
// full[s] therefore counts 1 + G arrivals plus the R bytes.
//
// Balance.  n/64 tiles over 148 SMs leave a ragged last wave (C5: 512 tiles = 3.46 waves), and the kernel is
// compute-bound in the generator, so the contraction is split S ways (unit = tile x K range, S chosen on the host
// to fill the last wave: C5 S = 2 -> 6.92 waves).  The S partial results of a tile are residues mod q; they are
// combined in U itself under a per-tile lock: the first unit to finish stores, later ones add mod q (order-free:
// a sum of residues is the residue of the sum), the last resets the tile's counter.  No unit ever waits while
// holding a lock, and all CTAs are resident, so this cannot deadlock.
#include "aes_ctr.cuh"
#include "tc_common.cuh"

namespace lwe {

namespace {

using namespace tc;

constexpr uint32_t kTileM = 128;
constexpr uint32_t kTileN = 256;
constexpr uint32_t kTmemCols = 512;
constexpr uint32_t kInstrDesc = instr_desc_u8(kTileM, kTileN, true, true);

template <uint32_t G, uint32_t kStages>
struct RegenCfg {
    static constexpr uint32_t kTileK = 8 * G;
    static constexpr uint32_t kThreads = (6 + G) * 32;
    static constexpr uint32_t kBytesA = kTileM * kTileK;
    static constexpr uint32_t kBytesBHalf = 128 * kTileK;
    static constexpr uint32_t kBytesStage = kBytesA + 2 * kBytesBHalf;
    static constexpr uint32_t kSmemBytes = kStages * kBytesStage + kAesTableBytes + 1024 /*align*/ + 256 /*barriers*/;
};

__device__ __forceinline__ void epi_bar() { asm volatile("bar.sync 1, 128;" ::: "memory"); }

template <uint32_t G, uint32_t kStages>
__global__ void __launch_bounds__(RegenCfg<G, kStages>::kThreads, 1)
encaps_regen_tc_kernel(const __grid_constant__ CUtensorMap mapR, const __grid_constant__ AesKey key, const uint32_t *__restrict__ te0,
                       uint16_t *__restrict__ U, uint32_t *__restrict__ locks, uint32_t m, uint32_t n, uint32_t k,
                       uint32_t splits, ModQ mq)
{
    using Cfg = RegenCfg<G, kStages>;
    constexpr uint32_t kTileK = Cfg::kTileK, kBytesA = Cfg::kBytesA, kBytesBHalf = Cfg::kBytesBHalf,
                       kBytesStage = Cfg::kBytesStage;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;
    uint8_t *const gbase = smem_raw + (base - raw);                       // generic view of `base`
    const uint32_t tab_off = kStages * kBytesStage;
    const uint32_t bars = base + tab_off + kAesTableBytes;
    auto full_bar = [&](uint32_t s) { return bars + 8 * s; };
    auto empty_bar = [&](uint32_t s) { return bars + 8 * (kStages + s); };
    auto tfull_bar = [&](uint32_t a) { return bars + 8 * (2 * kStages + a); };
    auto tempty_bar = [&](uint32_t a) { return bars + 8 * (2 * kStages + 2 + a); };
    const uint32_t tmem_slot = bars + 8 * (2 * kStages + 4);
    volatile uint32_t *tmem_slot_ptr = reinterpret_cast<volatile uint32_t *>(gbase + (tmem_slot - base));
    volatile uint32_t *first_slot = reinterpret_cast<volatile uint32_t *>(gbase + (tmem_slot + 8 - base));

    const uint32_t warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;
    const uint32_t m_tiles = (2 * n + kTileM - 1) / kTileM;
    const uint32_t units = m_tiles * splits;
    const uint32_t k_blocks = (m + kTileK - 1) / kTileK;

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&mapR) : "memory");
        for (uint32_t s = 0; s < kStages; s++) {
            mbar_init(full_bar(s), 1 + G);
            mbar_init(empty_bar(s), 1);
        }
        for (uint32_t a = 0; a < 2; a++) {
            mbar_init(tfull_bar(a), 1);
            mbar_init(tempty_bar(a), 4);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) tmem_alloc(tmem_slot, kTmemCols);
    const AesTab tab = aes_table_to_smem<Cfg::kThreads>(gbase + tab_off, te0);          // all threads; ends with __syncthreads()
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    if (warp == 0) {
        // ===================== TMA producer of the R tile =====================
        uint32_t stage = 0, phase = 0;
        for (uint32_t u = blockIdx.x; u < units; u += gridDim.x) {
            const uint32_t split = u / m_tiles;
            const uint32_t kb0 = (uint32_t)((uint64_t)split * k_blocks / splits);
            const uint32_t kb1 = (uint32_t)((uint64_t)(split + 1) * k_blocks / splits);
            for (uint32_t kb = kb0; kb < kb1; kb++) {
                mbar_wait(empty_bar(stage), phase ^ 1);
                const uint32_t sb = base + stage * kBytesStage + kBytesA;
                const int32_t row = (int32_t)(kb * kTileK);
                if (elect_one()) {
                    mbar_expect_tx(full_bar(stage), 2 * kBytesBHalf);           // rows >= m arrive as zeros
                    tma_load_2d(sb, &mapR, full_bar(stage), 0, row);
                    tma_load_2d(sb + kBytesBHalf, &mapR, full_bar(stage), 128, row);
                }
                __syncwarp();
                if (++stage == kStages) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer =====================
        uint32_t stage = 0, phase = 0, it = 0;
        for (uint32_t u = blockIdx.x; u < units; u += gridDim.x, it++) {
            const uint32_t split = u / m_tiles;
            const uint32_t kb0 = (uint32_t)((uint64_t)split * k_blocks / splits);
            const uint32_t kb1 = (uint32_t)((uint64_t)(split + 1) * k_blocks / splits);
            const uint32_t acc = it & 1, acc_phase = (it >> 1) & 1;
            mbar_wait(tempty_bar(acc), acc_phase ^ 1);
            tc_fence_after();
            const uint32_t d_tmem = tmem_base + acc * kTileN;
            for (uint32_t kb = kb0; kb < kb1; kb++) {
                mbar_wait(full_bar(stage), phase);
                tc_fence_after();
                const uint32_t sa = base + stage * kBytesStage;
                if (elect_one()) {
                    uint64_t adesc = make_desc_mn_sw128(sa, 0, 1024);
                    uint64_t bdesc = make_desc_mn_sw128(sa + kBytesA, kBytesBHalf, 1024);
#pragma unroll
                    for (uint32_t ks = 0; ks < kTileK / kUmmaK; ks++) {
                        umma_i8(d_tmem, adesc, bdesc, kInstrDesc, (kb != kb0 || ks) ? 1u : 0u);
                        adesc += (kUmmaK * 128) >> 4;
                        bdesc += (kUmmaK * 128) >> 4;
                    }
                    umma_commit(empty_bar(stage));
                    if (kb == kb1 - 1) umma_commit(tfull_bar(acc));
                }
                __syncwarp();
                if (++stage == kStages) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp < 6) {
        // ===================== epilogue (warps 2..5) =====================
        const uint32_t quarter = warp & 3;
        const bool epi_leader = (warp == 2 && lane == 0);
        uint32_t *cnts = locks + m_tiles;
        uint32_t it = 0;
        for (uint32_t u = blockIdx.x; u < units; u += gridDim.x, it++) {
            const uint32_t split = u / m_tiles, mt = u - split * m_tiles;
            const uint32_t acc = it & 1, acc_phase = (it >> 1) & 1;
            mbar_wait(tfull_bar(acc), acc_phase);
            tc_fence_after();
            bool first = true;
            if (splits > 1) {
                // per-tile lock: the first unit of a tile to get here stores, the others add mod q
                if (epi_leader) {
                    while (atomicCAS(locks + mt, 0u, 1u) != 0u) __nanosleep(200);
                    __threadfence();
                    *first_slot = (*reinterpret_cast<volatile uint32_t *>(cnts + mt) == 0u) ? 1u : 0u;
                }
                epi_bar();
                first = *first_slot != 0u;
            }
            const uint32_t brow = mt * kTileM + quarter * 32 + lane;
            const uint32_t j = brow >> 1;
            const bool odd = lane & 1;
            const uint32_t taddr = tmem_base + ((quarter * 32) << 16) + acc * kTileN;
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
                const uint32_t col = cb + (odd ? 16u : 0u);
                if (j < n && col < k) {
                    uint4 *dst = reinterpret_cast<uint4 *>(U + (size_t)j * k + col);
                    if (!first) {
                        // written by another SM under the same lock: read past L1
                        const uint4 p0 = __ldcg(dst), p1 = __ldcg(dst + 1);
                        const uint32_t old[8] = {p0.x, p0.y, p0.z, p0.w, p1.x, p1.y, p1.z, p1.w};
#pragma unroll
                        for (int x = 0; x < 16; x++) {
                            uint32_t val = o[x] + ((x & 1) ? (old[x >> 1] >> 16) : (old[x >> 1] & 0xffffu));   // < 2q
                            o[x] = mq.pow2 ? (val & mq.mask) : (val >= mq.q ? val - mq.q : val);
                        }
                    }
                    dst[0] = make_uint4(o[0] | (o[1] << 16), o[2] | (o[3] << 16), o[4] | (o[5] << 16), o[6] | (o[7] << 16));
                    dst[1] = make_uint4(o[8] | (o[9] << 16), o[10] | (o[11] << 16), o[12] | (o[13] << 16), o[14] | (o[15] << 16));
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tempty_bar(acc));
            if (splits > 1) {
                __threadfence();                                        // my part of the tile is visible device-wide
                epi_bar();
                if (epi_leader) {
                    volatile uint32_t *cnt = reinterpret_cast<volatile uint32_t *>(cnts + mt);
                    const uint32_t done = *cnt + 1;
                    *cnt = (done == splits) ? 0u : done;                // self-resetting: ready for the next call
                    __threadfence();
                    atomicExch(locks + mt, 0u);
                }
            }
        }
    } else {
        // ===================== generators (warps 6 .. 6+G-1) =====================
        const uint32_t g = warp - 6;
        const uint32_t chunk = lane & 7, rsub = lane >> 3;
        const uint32_t chunks_per_row = n / 8;
        uint32_t stage = 0, phase = 0;
        for (uint32_t u = blockIdx.x; u < units; u += gridDim.x) {
            const uint32_t split = u / m_tiles, mt = u - split * m_tiles;
            const uint32_t kb0 = (uint32_t)((uint64_t)split * k_blocks / splits);
            const uint32_t kb1 = (uint32_t)((uint64_t)(split + 1) * k_blocks / splits);
            const uint32_t cglob = mt * 8 + chunk;                      // 16-byte chunk (= AES block) within a row of A
            const bool col_ok = cglob < chunks_per_row;
            for (uint32_t kb = kb0; kb < kb1; kb++) {
                mbar_wait(empty_bar(stage), phase ^ 1);
                uint8_t *sa = gbase + stage * kBytesStage;
                uint4 blk[2];
#pragma unroll
                for (int h = 0; h < 2; h++) {
                    const uint32_t r = g * 8 + rsub + 4 * h;
                    const uint32_t i = kb * kTileK + r;
                    blk[h] = (col_ok && i < m)
                        ? uniform_block(key, tab, mq, LWE_TAG_A, 0, (uint64_t)i * chunks_per_row + cglob)
                        : make_uint4(0, 0, 0, 0);
                }
#pragma unroll
                for (int h = 0; h < 2; h++) {
                    const uint32_t r = g * 8 + rsub + 4 * h;
                    *reinterpret_cast<uint4 *>(sa + r * 128 + ((chunk ^ (r & 7)) << 4)) = blk[h];
                }
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");    // generic stores -> tcgen05's proxy
                __syncwarp();
                if (lane == 0) mbar_arrive(full_bar(stage));
                if (++stage == kStages) { stage = 0; phase ^= 1; }
            }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, kTmemCols);
}

// S = number of K ranges per tile: minimise (waves of units) x (K blocks per unit)
uint32_t choose_splits(uint32_t m_tiles, uint32_t k_blocks, uint32_t ctas)
{
    uint32_t best = 1;
    uint64_t best_cost = ~0ull;
    for (uint32_t s = 1; s <= 16 && s * 4 <= k_blocks; s++) {
        const uint64_t waves = ((uint64_t)m_tiles * s + ctas - 1) / ctas;
        const uint64_t cost = waves * ((k_blocks + s - 1) / s) + s;     // + s: one epilogue pass per split
        if (cost < best_cost) { best_cost = cost; best = s; }
    }
    return best;
}

template <uint32_t G, uint32_t kStages>
cudaError_t launch_cfg(Ctx *c, const AesKey &key, uint16_t *d_U, cudaStream_t st)
{
    using Cfg = RegenCfg<G, kStages>;
    const lwe_params &p = c->p;
    CUtensorMap mapR;
    if (!make_map_u8(c, &mapR, c->d_Rexp, p.k, p.m, Cfg::kTileK)) return cudaErrorInvalidValue;
    auto kern = encaps_regen_tc_kernel<G, kStages>;
    cudaError_t perr = kernel_prepare(c, kern, Cfg::kSmemBytes);
    if (perr != cudaSuccess) return perr;
    const uint32_t m_tiles = (2 * p.n + kTileM - 1) / kTileM;
    const uint32_t k_blocks = (p.m + Cfg::kTileK - 1) / Cfg::kTileK;
    const uint32_t splits = choose_splits(m_tiles, k_blocks, (uint32_t)c->sm_count);
    const uint32_t units = m_tiles * splits;
    const uint32_t grid = units < (uint32_t)c->sm_count ? units : (uint32_t)c->sm_count;
    ProfScope prof(c, LWE_K_ENCAPS_REGEN_TC, st);
    kern<<<grid, Cfg::kThreads, Cfg::kSmemBytes, st>>>(mapR, key, c->d_te0, d_U, c->d_tile_locks, p.m, p.n, p.k, splits,
                                                       c->mq);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace

uint32_t encaps_regen_lock_words(const lwe_params &p) { return 2 * ((2 * p.n + kTileM - 1) / kTileM); }

// one instance (N = k <= 256 columns): every A tile feeds exactly one MMA tile
bool encaps_regen_tc_supported(const Ctx *c, uint32_t batch)
{
    return batch == 1 && c->p.k <= kTileN && c->p.m <= 65536u && c->d_tile_locks != nullptr && encaps_tc_supported(c, batch);
}

cudaError_t launch_encaps_regen_tc(Ctx *c, const AesKey &key, uint16_t *d_U, cudaStream_t st)
{
    // 24 generator warps (K block 192), 2-stage ring: measured best on B200 (16 warps x 3 stages: -6 %)
    return launch_cfg<24, 2>(c, key, d_U, st);
}

}  // namespace lwe

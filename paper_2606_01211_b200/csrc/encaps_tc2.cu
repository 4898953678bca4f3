// encaps_tc2.cu -- a4 on CTA pairs: the same GEMM as encaps_tc.cu (D[2n x N] = A8^T . Rexp,
// u8 x u8 -> s32, U = (D_even + 256 D_odd) mod q, BJ north_star (3)) issued as
// tcgen05.mma.cta_group::2.
//
// Why a second kernel.  With cta_group::1 every SM stages its own copy of the 256-column R tile:
// per 128-deep K block 16 KB of A and 32 KB of R cross L2 -> shared memory, and the tensor pipe
// reads 96 B/clk of shared memory while TMA writes another 96 B/clk.  A CTA pair on one TPC splits
// the N dimension of the B operand between its two SMs (each loads 128 of the 256 columns) while
// each keeps its own 128 rows of A: 32 KB per K block and SM instead of 48 KB, i.e. one third less
// L2->SM and shared-memory traffic for the same MMA rate.  ncu on the cta_group::1 kernel showed the
// tensor pipe 84 % active with DRAM at 20 %: the feed, not HBM, was the limit.
//
// Shape.  Persistent, grid = SM count, clusters of 2.  Pair tile: 256 byte-rows of D (= 128 columns
// of A) x 256 columns (= one instance at k = 256); each CTA owns 128 byte-rows, accumulated in its
// own TMEM (two 256-column accumulators, so the epilogue of tile t overlaps the MMAs of tile t+1).
// K block 128, 6-stage ring of 32 KB.
//   warp 0 : TMA producer (both CTAs; completion bytes of both land on the LEADER's full barrier)
//   warp 1 : TMEM alloc (both CTAs) + MMA issuer (leader CTA only, one lane)
//   warps 2-5 : epilogue on the CTA's own TMEM lanes, as in encaps_tc.cu
//   warps 6-13 (kBitsB, the default for k % 128 == 0): expanders -- the B tile is not loaded but built in shared
//               memory from R's packed bits (see the comment above the kernel); TMA then carries only A
// Barriers: full[s] lives on the leader (1 arrival + 64 KB of transaction bytes); empty[s] and
// tmem_full[a] exist in both CTAs and are signalled by multicast tcgen05.commit; tmem_empty[a]
// lives on the leader and collects the 8 epilogue warps of the pair.
#include "tc_common.cuh"

namespace lwe {

namespace {

using namespace tc;

constexpr uint32_t kCtaM = 128;                  // byte-rows of D per CTA
constexpr uint32_t kPairM = 2 * kCtaM;           // per pair
constexpr uint32_t kTileN = 256;
constexpr uint32_t kHalfN = kTileN / 2;          // columns of R staged by each CTA
constexpr uint32_t kThreads = 192;
constexpr uint32_t kExpGroups = 2;                  // expander groups per CTA (kBitsB): group j takes K blocks j, j+2, ..
constexpr uint32_t kExpWarps = 4 * kExpGroups;      // 4 warps = 128 threads = one K row each
constexpr uint32_t kVWarps = 2;                     // kBitsB: warps computing v = b^T R + mu floor(q/2) beside the GEMM
constexpr uint32_t kThreadsBits = kThreads + 32 * kExpWarps + 32 * kVWarps;
// the signed-R modes (N2) run EIGHT epilogue warps per CTA, two per TMEM lane quarter, each taking half of the tile's
// columns: their epilogue (two Barrett reductions, E1, the exception terms, 32-bit stores) costs ~40 instructions
// per element, and with four warps it -- not the tensor pipe -- set the pace (ncu: epilogue warps busy 81 % of the
// time, tensor pipe 65 %; profiles/r2_wide_gemm_*)
constexpr uint32_t kThreadsPv = kThreads + 128;
constexpr uint32_t kBitStages = 12;                 // ring of packed-bit tiles, deeper than the operand ring
constexpr uint32_t kBitTileBytes = 128 * 16;        // 128 K rows x 128 columns of bits
constexpr uint32_t kTmemCols = 512;

constexpr uint32_t kInstrDesc = instr_desc_u8(kPairM, kTileN, true, true);
constexpr uint32_t kInstrDescSignedB = instr_desc_u8(kPairM, kTileN, true, true, true);     // N2: R holds int8

struct PairSched {
    uint32_t m_tiles, n_tiles, total, g;
    __device__ __forceinline__ void coords(uint32_t t, uint32_t &mt, uint32_t &nt) const
    {
        // groups of g n-tiles, n fastest inside a group: pairs running together share A strips and
        // the group's R panels stay in L2 (same order as the cta_group::1 kernel)
        uint32_t per_group = m_tiles * g;
        uint32_t grp = t / per_group, r = t - grp * per_group;
        uint32_t width = (n_tiles - grp * g) < g ? (n_tiles - grp * g) : g;
        mt = r / width;
        nt = grp * g + (r - mt * width);
    }
};

template <uint32_t kStages, uint32_t kTileK>
struct PairCfg {
    static constexpr uint32_t kBytesA = kCtaM * kTileK;
    static constexpr uint32_t kBytesB = kHalfN * kTileK;
    static constexpr uint32_t kBytesStage = kBytesA + kBytesB;
    static constexpr uint32_t kSmemBytes = kStages * kBytesStage + 1024 /*align*/ + 256 /*barriers*/;
    // kBitsB: + a ring of packed-bit tiles (128 K rows x 16 bytes each) and its barriers
    // ... and the v warps' k <= 2048 column sums
    static constexpr uint32_t kSmemBytesBits = kSmemBytes + kBitStages * kBitTileBytes + 256 + 2048 * 4 + 16;
};

// kBitsB: the B operand is never expanded in HBM.  Eight extra warps per CTA (two groups taking alternate K blocks)
// read the packed bits of R (16 bytes = the 128 columns of one K row of this CTA's half tile per thread), spread them to {0,1} bytes and store
// them into the stage's B buffer in the swizzled layout TMA would have produced; the stage's full barrier then
// counts the arrivals of one group of each CTA (8 warps) beside the A bytes.  Needs k % 128 == 0 (a half tile lies inside
// one instance) and kTileK == 128 (one row per expander thread).  Against the expanded operand this removes the
// 128 MiB expanded-R write per batch and every DRAM / L2 re-read of it by the GEMM (16x fewer operand bytes).
// a5 inside the GEMM (kBitsB): v_c = sum_i b_i R_ic + mu_c floor(q/2) mod q (BJ north_star) is one more
// "row" of the same contraction, but its left operand b differs per instance, so it cannot ride the tensor pipe
// without computing batch x batch blocks for a diagonal.  Two spare warps per CTA compute it on the CUDA cores while
// the MMAs run: 2 instructions per bit of R, ~0.8 % of the SM's issue slots over the kernel's life, and the separate
// 29 us pass over R's bits (0.09 of HBM, 2.4 % of the step) disappears from the stream.
struct VArgs {
    const uint16_t *b;                 // [batch][m]; NULL: v is not computed by this launch
    const uint8_t *Rbits, *mubits;
    uint16_t *v;
    unsigned long long *acc;           // [batch][k] u64 partial sums, left zeroed
    unsigned int *tickets;             // [batch] self-resetting
    uint32_t m, batch, splits;         // rows per instance, instances, row ranges per instance
};

// Executed by the kVWarps * 32 threads `vt` = 0..63 of a CTA; the CTAs share the (instance, row range) units.
// The arithmetic of expand_R_and_v_w32_kernel (encaps_aux.cu): a thread owns one 32-bit word of R bits (32 columns)
// of a row; its 32 column sums sit in 16-bit lanes of 2 x 16 registers, one byte plane of b at a time.
__device__ __forceinline__ void v_warps_role(const VArgs &va, uint32_t vt, uint32_t k, const ModQ &mq, uint32_t *sSum,
                                             volatile uint32_t *sLast)
{
    constexpr uint32_t kVT = 32 * kVWarps;
    auto vbar = [&]() { asm volatile("bar.sync 1, %0;" ::"n"(kVT) : "memory"); };
    const uint32_t wpr = k / 32;                               // words per row: a power of two <= 64
    const uint32_t w = vt & (wpr - 1);
    const uint32_t rows_per_iter = kVT / wpr, rslot = vt / wpr;
    const uint32_t units = va.batch * va.splits;
    for (uint32_t u = blockIdx.x; u < units; u += gridDim.x) {
        const uint32_t t = u / va.splits, sidx = u - t * va.splits;
        const uint32_t per = ((va.m + va.splits - 1) / va.splits + rows_per_iter - 1) / rows_per_iter * rows_per_iter;
        const uint32_t ibeg = sidx * per, iend = min(va.m, ibeg + per);
        const uint32_t *Rt = reinterpret_cast<const uint32_t *>(va.Rbits + (size_t)t * va.m * (k / 8));
        const uint16_t *bt = va.b + (size_t)t * va.m;
        for (uint32_t c = vt; c < k; c += kVT) sSum[c] = 0;
        vbar();
        uint32_t aL[16], aH[16];
#pragma unroll
        for (int x = 0; x < 16; x++) { aL[x] = 0; aH[x] = 0; }
        auto flush = [&]() {
            uint32_t vals[32];
#pragma unroll
            for (int x = 0; x < 16; x++) {
                vals[x] = (aL[x] & 0xffffu) + ((aH[x] & 0xffffu) << 8);
                vals[x + 16] = (aL[x] >> 16) + ((aH[x] >> 16) << 8);
                aL[x] = 0; aH[x] = 0;
            }
            for (uint32_t off = wpr; off < 32; off <<= 1) {
#pragma unroll
                for (int x = 0; x < 32; x++) vals[x] += __shfl_xor_sync(0xffffffffu, vals[x], off);
            }
            if ((vt & 31) < wpr || wpr >= 32) {
#pragma unroll
                for (int x = 0; x < 32; x++)
                    if (vals[x]) atomicAdd(&sSum[x * wpr + w], vals[x]);
            }
        };
        constexpr int kUnroll = 4;
        constexpr uint32_t kFlushIters = 256 / kUnroll;       // <= 256 rows per thread between flushes (16-bit lanes)
        uint32_t iters = 0;
        for (uint32_t i0 = ibeg + rslot; i0 < iend; i0 += kUnroll * rows_per_iter) {
            uint32_t r[kUnroll], bi[kUnroll];
#pragma unroll
            for (int q = 0; q < kUnroll; q++) {
                const uint32_t i = i0 + q * rows_per_iter;
                r[q] = (i < iend) ? __ldg(Rt + (size_t)i * wpr + w) : 0u;
                bi[q] = (i < iend) ? (uint32_t)__ldg(bt + i) : 0u;
            }
#pragma unroll
            for (int q = 0; q < kUnroll; q++) {
                const uint32_t bl = bi[q] & 0xffu, bh = bi[q] >> 8;
#pragma unroll
                for (int x = 0; x < 16; x++) {
                    const uint32_t two = (r[q] >> x) & 0x00010001u;     // columns x (low lane) and x + 16 (high lane)
                    aL[x] += two * bl;
                    aH[x] += two * bh;
                }
            }
            if (++iters == kFlushIters) { flush(); iters = 0; }
        }
        flush();
        vbar();
        for (uint32_t c = vt; c < k; c += kVT) {
            const uint32_t sum = sSum[(c & 31u) * wpr + (c >> 5)];
            if (sum) atomicAdd(va.acc + (size_t)t * k + c, (unsigned long long)sum);
        }
        __threadfence();
        vbar();
        if (vt == 0) *sLast = (atomicAdd(va.tickets + t, 1u) == va.splits - 1) ? 1u : 0u;
        vbar();
        if (*sLast) {                                          // the last range of instance t: reduce mod q, write v
            __threadfence();
            for (uint32_t c = vt; c < k; c += kVT) {
                const unsigned long long sum = __ldcg(va.acc + (size_t)t * k + c);
                va.acc[(size_t)t * k + c] = 0;
                const uint32_t mu = (va.mubits[(size_t)t * (k / 8) + c / 8] >> (c % 8)) & 1u;
                va.v[(size_t)t * k + c] = (uint16_t)mod_u64(sum + (unsigned long long)mu * mq.half, mq);
            }
            if (vt == 0) va.tickets[t] = 0;
        }
        vbar();
    }
}

// The signed-R modes (N2) beside the accumulators.  r_inplace: the B operand is read IN PLACE from the caller's int8
// R [batch][m_full][k] (a half tile lies inside one instance when k % 128 == 0; rows of the next instance that a
// ragged last K block drags in meet zero-filled rows of A) -- no operand copy is made.  Wide contexts: the
// exception list of column j (rows i with A[i][j] >= 2^16) and R itself, for the 2^16 R[i][c] terms.
struct PvArgs {
    const int8_t *E1;
    uint32_t bias, e1bias, two_step;      // see launch_pair
    uint32_t r_inplace, m_full;
    const int8_t *R;
    const uint32_t *exc_cnt, *exc_rows;
    uint32_t exc_cap, delta;              // delta = q - 2^16: 2^16 = -delta (mod q)
    // wide contexts with m > 65536: the rows are contracted in passes of <= 65536 (a signed byte-plane sum holds no
    // more); this launch covers rows [row0, row0 + rows) -- only the exceptions in that range count -- and, from the
    // second pass on (accum), adds the residues already in U (E1 is added by the first pass only: E1 = NULL later)
    uint32_t row0, rows, accum;
};

template <uint32_t kStages, uint32_t kTileK, int kMode, bool kBitsB>
__global__ void __cluster_dims__(2, 1, 1)
__launch_bounds__(kBitsB ? kThreadsBits : ((kMode == kEpiStorePv || kMode == kEpiStorePvW) ? kThreadsPv : kThreads), 1)
encaps_tc2_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapR,
                  void *__restrict__ U_, uint32_t *__restrict__ flags, uint32_t m,
                  uint32_t n, uint32_t k,
                  uint32_t ncols_total, ModQ mq, uint32_t group_w, PvArgs pv,
                  const __grid_constant__ CUtensorMap mapBits, uint32_t bits_row0,
                  uint32_t bits_rows_per_inst, VArgs va)
{
    constexpr bool kPv = (kMode == kEpiStorePv || kMode == kEpiStorePvW);
    uint16_t *U = static_cast<uint16_t *>(U_);
    uint32_t *U32 = static_cast<uint32_t *>(U_);
    const int8_t *E1 = pv.E1;
    static_assert(!kBitsB || kTileK == 128, "one K row per expander thread");
    using Cfg = PairCfg<kStages, kTileK>;
    constexpr uint32_t kBytesA = Cfg::kBytesA, kBytesStage = Cfg::kBytesStage;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;
    const uint32_t bits_ring = base + kStages * kBytesStage;                        // kBitsB only
    const uint32_t bars = bits_ring + (kBitsB ? kBitStages * kBitTileBytes : 0u);
    auto bfull_bar = [&](uint32_t s) { return bars + 256 + 8 * s; };                // kBitsB only
    auto bempty_bar = [&](uint32_t s) { return bars + 256 + 8 * (kBitStages + s); };
    auto full_bar = [&](uint32_t s) { return bars + 8 * s; };
    auto empty_bar = [&](uint32_t s) { return bars + 8 * (kStages + s); };
    auto tfull_bar = [&](uint32_t a) { return bars + 8 * (2 * kStages + a); };
    auto tempty_bar = [&](uint32_t a) { return bars + 8 * (2 * kStages + 2 + a); };
    const uint32_t tmem_slot = bars + 8 * (2 * kStages + 4);
    volatile uint32_t *tmem_slot_ptr = reinterpret_cast<volatile uint32_t *>(smem_raw + (tmem_slot - raw));

    const uint32_t warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;   // warp-uniform
    const uint32_t rank = cluster_ctarank();                     // 0 = leader
    const uint32_t pair = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;

    PairSched sched;
    sched.g = group_w;
    sched.m_tiles = (2 * n + kPairM - 1) / kPairM;
    sched.n_tiles = (ncols_total + kTileN - 1) / kTileN;
    sched.total = sched.m_tiles * sched.n_tiles;
    const uint32_t k_blocks = (m + kTileK - 1) / kTileK;

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&mapA) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&mapR) : "memory");
        for (uint32_t s = 0; s < kStages; s++) {
            mbar_init(full_bar(s), kBitsB ? 1 + 2 * 4 : 1);       // the leader's expect_tx arrival (+ one expander group per CTA)
            mbar_init(empty_bar(s), 1);                           // one multicast commit
        }
        for (uint32_t a = 0; a < 2; a++) {
            mbar_init(tfull_bar(a), 1);
            mbar_init(tempty_bar(a), kPv ? 16 : 8);               // 4 (signed-R modes: 8) epilogue warps of each CTA
        }
        if (kBitsB) {
            asm volatile("prefetch.tensormap [%0];" ::"l"(&mapBits) : "memory");
            for (uint32_t s = 0; s < kBitStages; s++) {
                mbar_init(bfull_bar(s), 1);
                mbar_init(bempty_bar(s), 4);                      // one arrival per warp of the consuming group
            }
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    pdl_trigger();
    if (warp == 1) tmem_alloc_pair(tmem_slot, kTmemCols);
    tc_fence_before();
    cluster_sync_all();                                           // barriers of BOTH CTAs are initialised
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;
    pdl_wait();                          // the prologue above overlapped the previous kernel; its outputs are needed now

    // The producer and MMA roles run WARP-CONVERGENT loops and elect one lane only around the
    // instructions that must be issued once: inside a divergent `if (lane == 0)` region the compiler
    // cannot keep descriptors and barrier addresses in uniform registers and wraps every TMA / MMA /
    // commit in an ELECT + R2UR + vote loop (~130 SASS instructions per K block, which made the
    // issuing thread, not the tensor pipe, the bottleneck: ncu source page, profiles/r1b_*).
    if (warp == 0) {
        // ===================== TMA producer (both CTAs) =====================
        uint32_t stage = 0, phase = 0;
        for (uint32_t t = pair; t < sched.total; t += n_pairs) {
            uint32_t mt, nt;
            sched.coords(t, mt, nt);
            const int32_t a_col = (int32_t)(mt * kPairM + rank * kCtaM);
            int32_t r_col = (int32_t)(nt * kTileN + rank * kHalfN), r_row0 = 0;
            if (kPv && pv.r_inplace) {                     // this half tile inside R [batch][m_full][k]
                const uint32_t inst = (uint32_t)r_col / k;
                r_col -= (int32_t)(inst * k);
                r_row0 = (int32_t)(inst * pv.m_full + pv.row0);   // past the batch: out of range -> zeros
            }
            for (uint32_t kb = 0; kb < k_blocks; kb++) {
                mbar_wait(empty_bar(stage), phase ^ 1);
                const uint32_t sa = base + stage * kBytesStage;
                const uint32_t lead_full = map_to_cta(full_bar(stage), 0);
                const int32_t row = (int32_t)(kb * kTileK);
                if (elect_one()) {
                    if (rank == 0) mbar_expect_tx(full_bar(stage), 2 * (kBitsB ? kBytesA : kBytesStage));   // both CTAs' bytes
                    tma_load_2d_pair(sa, &mapA, lead_full, a_col, row);
                    if (!kBitsB) tma_load_2d_pair(sa + kBytesA, &mapR, lead_full, r_col, r_row0 + row);
                }
                __syncwarp();
                if (++stage == kStages) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer (leader CTA) =====================
        if (rank == 0) {
            uint32_t stage = 0, phase = 0, it = 0;
            for (uint32_t t = pair; t < sched.total; t += n_pairs, it++) {
                const uint32_t acc = it & 1, acc_phase = (it >> 1) & 1;
                mbar_wait(tempty_bar(acc), acc_phase ^ 1);          // both epilogues drained this accumulator
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + acc * kTileN;
                for (uint32_t kb = 0; kb < k_blocks; kb++) {
                    mbar_wait(full_bar(stage), phase);
                    tc_fence_after();
                    const uint32_t sa = base + stage * kBytesStage;
                    if (elect_one()) {
                        // descriptors differ only in the 14-bit start-address field: one add per MMA
                        uint64_t adesc = make_desc_mn_sw128(sa, 0, 1024);
                        uint64_t bdesc = make_desc_mn_sw128(sa + kBytesA, 0, 1024);
#pragma unroll
                        for (uint32_t ks = 0; ks < kTileK / kUmmaK; ks++) {
                            umma_i8_pair(d_tmem, adesc, bdesc, kPv ? kInstrDescSignedB : kInstrDesc,
                                         (kb | ks) ? 1u : 0u);
                            adesc += (kUmmaK * 128) >> 4;
                            bdesc += (kUmmaK * 128) >> 4;
                        }
                        umma_commit_pair(empty_bar(stage), 0x3);    // frees the slot in both CTAs
                        if (kb == k_blocks - 1) umma_commit_pair(tfull_bar(acc), 0x3);
                    }
                    __syncwarp();
                    if (++stage == kStages) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (kBitsB && warp >= 6 + kExpWarps) {
        // ===================== v warps (both CTAs): a5 on the CUDA cores beside the MMAs =====================
        if (va.b != nullptr) {
            uint32_t *sSum = reinterpret_cast<uint32_t *>(smem_raw + (bars + 512 - raw));
            v_warps_role(va, threadIdx.x - 32 * (6 + kExpWarps), k, mq, sSum, sSum + 2048);
        }
    } else if (kBitsB && warp >= 6) {
        // ===================== B-operand expanders (warps 6..13, both CTAs) =====================
        // The packed bits of this CTA's half tile (128 K rows x 16 bytes) arrive through their own, deeper TMA ring
        // (issued kBitStages - 1 K blocks ahead by warp 6), so that only the expansion itself -- not a global-memory
        // latency -- sits between "stage freed" and "stage full", in parallel with the A tile's TMA.
        // Two groups of 4 warps take alternate K blocks: a group has two stage periods for its load-expand-store-
        // fence-arrive chain (one was not enough: the chain, ~600 cycles, exceeds the 512-cycle MMA time of a stage).
        const uint32_t group = (warp - 6) >> 2;
        const uint32_t r = ((warp - 6) & 3) * 32 + lane;            // K row of the stage owned by this thread
        const uint32_t my_tiles = (sched.total > pair) ? (sched.total - pair + n_pairs - 1) / n_pairs : 0u;
        const uint32_t total_kb = my_tiles * k_blocks;              // K blocks this CTA streams
        // load cursor (runs ahead) -- only used by warp 6
        uint32_t lt = pair, lkb = 0, lg = 0, lrow = 0, lcol = 0;
        auto set_load_tile = [&]() {
            uint32_t mt, nt;
            sched.coords(lt, mt, nt);
            const uint32_t col0 = nt * kTileN + rank * kHalfN;
            const uint32_t inst = col0 / k;
            lrow = inst * bits_rows_per_inst + bits_row0;           // instances past the batch: out of range -> zeros
            lcol = (col0 - inst * k) / 8;
        };
        auto issue_load = [&]() {                                   // K block lg of the stream -> ring slot lg % kBitStages
            const uint32_t bs = lg % kBitStages, bphase = (lg / kBitStages) & 1;
            mbar_wait(bempty_bar(bs), bphase ^ 1);
            if (elect_one()) {
                mbar_expect_tx(bfull_bar(bs), kBitTileBytes);
                tma_load_2d(bits_ring + bs * kBitTileBytes, &mapBits, bfull_bar(bs), (int32_t)lcol,
                            (int32_t)(lrow + lkb * kTileK));
            }
            __syncwarp();
            lg++;
            if (++lkb == k_blocks) { lkb = 0; lt += n_pairs; if (lg < total_kb) set_load_tile(); }
        };
        if (warp == 6 && total_kb) set_load_tile();
        for (uint32_t g = group; g < total_kb; g += kExpGroups) {
            if (warp == 6)
                while (lg < total_kb && lg < g + kBitStages - 1) issue_load();
            const uint32_t bs = g % kBitStages, bphase = (g / kBitStages) & 1;
            const uint32_t stage = g % kStages, phase = (g / kStages) & 1;
            mbar_wait(bfull_bar(bs), bphase);
            uint32_t w[4];
            asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];"
                         : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]) : "r"(bits_ring + bs * kBitTileBytes + r * 16));
            __syncwarp();
            if (lane == 0) mbar_arrive(bempty_bar(bs));
            mbar_wait(empty_bar(stage), phase ^ 1);                 // the MMAs that read this B buffer have retired
            const uint32_t srow = base + stage * kBytesStage + kBytesA + r * 128;
#pragma unroll
            for (uint32_t c = 0; c < 8; c++) {                      // 16-byte chunk c = columns 16c .. 16c+15
                const uint32_t bits = w[c >> 1] >> (16 * (c & 1));
                uint32_t o[4];
#pragma unroll
                for (int h = 0; h < 4; h++) o[h] = (((bits >> (4 * h)) & 0xfu) * 0x00204081u) & 0x01010101u;
                asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};"
                             ::"r"(srow + ((c ^ (r & 7)) << 4)), "r"(o[0]), "r"(o[1]), "r"(o[2]), "r"(o[3]) : "memory");
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");        // generic stores -> the MMA's proxy
            __syncwarp();
            if (lane == 0) mbar_arrive_remote(map_to_cta(full_bar(stage), 0));
        }
    } else if (warp < 6 || (kPv && !kBitsB)) {
        // ===================== epilogue (warps 2..5, both CTAs; signed-R modes: warps 2..9) =====================
        const uint32_t quarter = warp & 3;                           // the TMEM lane quarter a warp may read
        const uint32_t cb_lo = (kPv && warp >= 6) ? kTileN / 2 : 0u; // warps 6..9 take the upper half of the columns
        const uint32_t cb_hi = (kPv && warp < 6) ? kTileN / 2 : kTileN;
        const uint32_t lead_tempty0 = map_to_cta(tempty_bar(0), 0), lead_tempty1 = map_to_cta(tempty_bar(1), 0);
        uint32_t it = 0;
        for (uint32_t t = pair; t < sched.total; t += n_pairs, it++) {
            uint32_t mt, nt;
            sched.coords(t, mt, nt);
            const uint32_t acc = it & 1, acc_phase = (it >> 1) & 1;
            const uint32_t brow = mt * kPairM + rank * kCtaM + quarter * 32 + lane;   // byte-row of D
            const uint32_t j = brow >> 1;
            const bool odd = lane & 1;
            const uint32_t taddr = tmem_base + ((quarter * 32) << 16) + acc * kTileN;
            MismatchAcc mism;
            // wide: number of elements >= 2^16 in column j of A (rare: ~m/65537 per column)
            const uint32_t exc = (kMode == kEpiStorePvW && j < n) ? min(__ldg(pv.exc_cnt + j), pv.exc_cap) : 0u;
            // one 32-column piece of the tile: this lane's 16 columns of row j
            auto do_chunk = [&](uint32_t cb, const uint4 &e1v) {
                uint32_t r[32];
                tmem_ld_32x32b_x32(taddr + cb, r);
                tmem_ld_wait();
                uint32_t o[16];
                const uint32_t col = nt * kTileN + cb + (odd ? 16u : 0u);
                const bool in_range = j < n && col < ncols_total;
                const uint32_t inst = col / k, c = col - inst * k;
                const uint32_t e1w[4] = {e1v.x, e1v.y, e1v.z, e1v.w};   // 16 int8 of E1[inst][j][c..c+15] (N2 only)
                // wide: corr[x] = sum over the exceptions i of column j of R[inst][i][c + x]
                int corr[16];
                if (kMode == kEpiStorePvW) {
#pragma unroll
                    for (int x = 0; x < 16; x++) corr[x] = 0;
                    const uint32_t cnt = in_range ? exc : 0u;
                    for (uint32_t y = 0; y < cnt; y++) {
                        const uint32_t i = __ldg(pv.exc_rows + (size_t)j * pv.exc_cap + y);
                        if (i - pv.row0 >= pv.rows) continue;                       // belongs to another row pass
                        const uint4 r4 = __ldg(reinterpret_cast<const uint4 *>(pv.R + ((size_t)inst * pv.m_full + i) * k + c));
                        const uint32_t rw[4] = {r4.x, r4.y, r4.z, r4.w};
#pragma unroll
                        for (int x = 0; x < 16; x++) corr[x] += (int)(int8_t)(rw[x >> 2] >> (8 * (x & 3)));
                    }
                }
                if (kPv) {
                    // signed planes: lo = sum lo(A) r, hi = sum hi(A) r; U = lo + 256 hi + e1 (- delta corr) mod q.
                    // General q: straight-line unsigned arithmetic (a branch per sign serialised the 16 elements:
                    // 0.65 ms instead of 0.17 ms at n = 4096).  pv.bias is a multiple of q >= 255 * 128 * rows, so
                    // plane + bias is the same residue in [0, 2^32); pv.e1bias likewise covers e1.  The kind of
                    // reduction is decided once per piece, not per element.
                    uint32_t lo[16], hi[16], e1[16];
#pragma unroll
                    for (int x = 0; x < 16; x++) {
                        const uint32_t recv = __shfl_xor_sync(0xffffffffu, odd ? r[x] : r[16 + x], 1);
                        lo[x] = odd ? recv : r[x];
                        hi[x] = odd ? r[16 + x] : recv;
                        int32_t ev = (int32_t)(int8_t)(e1w[x >> 2] >> (8 * (x & 3)));
                        if (kMode == kEpiStorePvW) ev -= (int32_t)pv.delta * corr[x];       // 2^16 = -delta (mod q)
                        e1[x] = (uint32_t)ev;
                    }
                    const uint32_t bias = pv.bias, e1bias = pv.e1bias;
                    if (mq.pow2) {
#pragma unroll
                        for (int x = 0; x < 16; x++) o[x] = (lo[x] + (hi[x] << 8) + e1[x]) & mq.mask;
                    } else if (pv.two_step) {   // (lo + bias) + 256 (hi mod q) + e1 stays below 2^32: one reduction less
#pragma unroll
                        for (int x = 0; x < 16; x++)
                            o[x] = mod_u32((lo[x] + bias) + 256u * mod_u32(hi[x] + bias, mq) + (e1[x] + e1bias), mq);
                    } else {
#pragma unroll
                        for (int x = 0; x < 16; x++)
                            o[x] = mod_u32(mod_u32(lo[x] + bias, mq) + 256u * mod_u32(hi[x] + bias, mq) + (e1[x] + e1bias), mq);
                    }
                } else {
#pragma unroll
                    for (int x = 0; x < 16; x++) {
                        uint32_t send = odd ? r[x] : r[16 + x];
                        uint32_t recv = __shfl_xor_sync(0xffffffffu, send, 1);
                        uint32_t val = odd ? (recv + (r[16 + x] << 8)) : (r[x] + (recv << 8));
                        o[x] = mq.pow2 ? (val & mq.mask) : mod_u32(val, mq);
                    }
                }
                if (in_range) {
                    if (kMode == kEpiStorePvW) {
                        uint4 *dst = reinterpret_cast<uint4 *>(U32 + ((size_t)inst * n + j) * k + c);
                        if (pv.accum) {                                             // a sum of residues is the residue of the sum
#pragma unroll
                            for (int x = 0; x < 4; x++) {
                                const uint4 old = dst[x];
                                const uint32_t ov[4] = {old.x, old.y, old.z, old.w};
#pragma unroll
                                for (int y = 0; y < 4; y++) {
                                    const uint32_t val = o[4 * x + y] + ov[y];      // < 2q
                                    o[4 * x + y] = val >= mq.q ? val - mq.q : val;
                                }
                            }
                        }
#pragma unroll
                        for (int x = 0; x < 4; x++) dst[x] = make_uint4(o[4 * x], o[4 * x + 1], o[4 * x + 2], o[4 * x + 3]);
                    } else {
                        const bool bad = store_u16x16<kMode>(reinterpret_cast<uint4 *>(U + ((size_t)inst * n + j) * k + c), o, mq);
                        if (kMode == kEpiCompare) mism.note(flags, inst, bad);
                    }
                }
            };
            if constexpr (kPv) {
                // E1 of the NEXT piece is fetched before the current one is processed, and the first before the
                // accumulator is ready: a dependent global load per piece after tfull made the epilogue (not the
                // tensor pipe) the limit at n = 8192 (0.71 ms instead of ~0.5).  The loop stays rolled: unrolled it
                // is 160 KB of code and thrashes the instruction cache (1.22 ms).
                auto e1_load = [&](uint32_t cb) {
                    const uint32_t col = nt * kTileN + cb + (odd ? 16u : 0u);
                    const uint32_t inst = col / k, c = col - inst * k;
                    return (E1 != nullptr && j < n && col < ncols_total)
                        ? __ldg(reinterpret_cast<const uint4 *>(E1 + ((size_t)inst * n + j) * k + c)) : make_uint4(0, 0, 0, 0);
                };
                uint4 e1cur = e1_load(cb_lo);
                mbar_wait(tfull_bar(acc), acc_phase);
                tc_fence_after();
#pragma unroll 1
                for (uint32_t cb = cb_lo; cb < cb_hi; cb += 32) {
                    const uint4 e1next = (cb + 32 < cb_hi) ? e1_load(cb + 32) : make_uint4(0, 0, 0, 0);
                    do_chunk(cb, e1cur);
                    e1cur = e1next;
                }
            } else {
                mbar_wait(tfull_bar(acc), acc_phase);
                tc_fence_after();
                const uint4 zero = make_uint4(0, 0, 0, 0);
#pragma unroll 1
                for (uint32_t cb = 0; cb < kTileN; cb += 32) do_chunk(cb, zero);
            }
            if (kMode == kEpiCompare) mism.flush_warp(flags);
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(acc ? lead_tempty1 : lead_tempty0);
        }
    }

    // no CTA of the pair may leave (or free TMEM) while its partner can still signal it or read its smem
    tc_fence_before();
    cluster_sync_all();
    if (warp == 1) tmem_dealloc_pair(tmem_base, kTmemCols);
}

}  // namespace

bool encaps_tc2_supported(const Ctx *c, uint32_t batch)
{
    return encaps_tc_supported(c, batch) && c->sm_count >= 2;
}

// signed-R modes: d_R = the caller's R [batch][m][k] (the wide epilogue reads its exception rows there); r_inplace:
// the B operand is read in place from it instead of from the copy in c->d_Rexp
template <uint32_t kStages, uint32_t kTileK, int kMode, bool kBitsB = false>
static cudaError_t launch_pair(Ctx *c, const uint16_t *d_A, void *d_U, uint32_t *d_flags, const int8_t *d_E1,
                               uint32_t batch, uint32_t row0, uint32_t rows, cudaStream_t st,
                               const uint8_t *d_Rbits = nullptr, const int8_t *d_R = nullptr, bool r_inplace = false,
                               const VArgs *vargs = nullptr)
{
    using Cfg = PairCfg<kStages, kTileK>;
    const lwe_params &p = c->p;
    const uint32_t ncols = batch * p.k;
    constexpr bool kPvMode = (kMode == kEpiStorePv || kMode == kEpiStorePvW);
    CUtensorMap mapA, mapR;
    // d_A holds rows [row0, row0 + rows) of A; the matching rows of the expanded R follow from row0
    if (!make_map_u8(c, &mapA, d_A, 2ull * p.n, rows, kTileK)) return cudaErrorInvalidValue;
    if (r_inplace) {
        if (!make_map_u8(c, &mapR, d_R, p.k, (uint64_t)batch * p.m, kTileK)) return cudaErrorInvalidValue;
    } else if (!make_map_u8(c, &mapR, c->d_Rexp + (size_t)row0 * ncols, ncols, rows, kTileK)) {
        return cudaErrorInvalidValue;
    }
    auto kern = encaps_tc2_kernel<kStages, kTileK, kMode, kBitsB>;
    const uint32_t smem_bytes = kBitsB ? Cfg::kSmemBytesBits : Cfg::kSmemBytes;
    cudaError_t err = kernel_prepare(c, kern, smem_bytes);
    if (err != cudaSuccess) return err;
    const uint32_t tiles = ((2 * p.n + kPairM - 1) / kPairM) * ((ncols + kTileN - 1) / kTileN);
    uint32_t pairs = (uint32_t)c->sm_count / 2;
    if (pairs > tiles) pairs = tiles;
    // tile order: groups of gw n-tiles run over every A strip before the next group starts, so A is re-streamed once per
    // group while the group's slice of the B operand stays in L2.  Bit operand: R is 16x smaller and stays in L2 by
    // itself, so all n-tiles of an A strip run together and A crosses HBM once (ncu at C4: 1.14 GB -> 0.30 GB read per
    // launch).  Byte operand (expanded u8, or the int8 R read in place): as many n-tiles as keep the group's slice at or
    // below 32 MiB, at least 8.  Measured on the signed-R GEMM, 32 instances (gw = 8 / 16 / 32): n = 8192, q = 65537
    // 0.644 / 0.630 / 0.673 ms (the whole 64 MB R beside 134 MB of A, 64 MB of E1 and 268 MB of U does not stay
    // resident), n = 4096 0.1587 / 0.1577 / 0.1559 ms.  The gain is small because that kernel is paced by the power cap,
    // not by HBM: the dense signed operand holds the chip at ~1.6 GHz (bench.py --phase int8_pipe_peak: u8 x s8
    // sustains 3.79 POP/s where u8 x {0,1} sustains 4.61).
    const uint32_t n_tiles_all = (ncols + kTileN - 1) / kTileN;
    uint32_t gw = n_tiles_all;
    if (!kBitsB) {
        const uint64_t slice = (uint64_t)rows * kTileN;                    // bytes of the B operand under one n-tile
        gw = (uint32_t)(((uint64_t)32 << 20) / (slice ? slice : 1));
        if (gw < 8u) gw = 8u;
        if (gw > n_tiles_all) gw = n_tiles_all;
    }
    ProfScope prof(c, LWE_K_ENCAPS_TC, st);
    // signed byte-plane sums of the N2 variant: |plane| <= 255 * 128 * rows; bias = the next multiple of q, so that
    // plane + bias is the same residue in [0, 2 bias] < 2^32 (rows <= 65536).  e1 (and, wide, e1 - delta * corr with
    // |corr| <= 128 * capacity) gets its own bias.  two_step: (lo + bias) + 256 (hi mod q) + (e1 + e1bias) < 2^32.
    PvArgs pv = {};
    const uint64_t plane_max = 255ull * 128ull * rows, q = p.q;
    const uint64_t delta = c->wide ? q - 65536u : 0u;
    const uint64_t e1_max = 128ull + delta * 128ull * c->exc_cap_col;
    pv.E1 = d_E1;
    pv.bias = (uint32_t)((plane_max + q - 1) / q * q);
    pv.e1bias = (uint32_t)((e1_max + q - 1) / q * q);
    pv.two_step = (2ull * pv.bias + 256ull * q + 2ull * pv.e1bias < (1ull << 32)) ? 1u : 0u;
    pv.r_inplace = r_inplace ? 1u : 0u;
    pv.m_full = p.m;
    pv.R = d_R;
    pv.exc_cnt = c->d_exc_col_cnt;
    pv.exc_rows = c->d_exc_col_rows;
    pv.exc_cap = c->exc_cap_col;
    pv.delta = (uint32_t)delta;
    pv.row0 = row0;
    pv.rows = rows;
    pv.accum = (kPvMode && row0 != 0) ? 1u : 0u;
    // packed bits of R as a byte matrix [batch * m][k / 8]; a bit tile = 128 rows x 16 bytes.  Rows of the panel
    // past `rows` meet zero-filled rows of A, rows past the last instance are zero-filled by TMA.
    CUtensorMap mapBits = mapR;
    if (kBitsB && !make_map_plain_u8(c, &mapBits, d_Rbits, p.k / 8, (uint64_t)batch * p.m, 16, kTileK))
        return cudaErrorInvalidValue;
    return launch_k(c, kern, 2 * pairs, kBitsB ? kThreadsBits : (kPvMode ? kThreadsPv : kThreads), smem_bytes, st,
                    mapA, mapR, d_U, d_flags, rows, p.n, p.k, ncols, c->mq, gw, pv, mapBits, row0, p.m,
                    vargs ? *vargs : VArgs{});
}

bool encaps_tc2_bits_supported(const Ctx *c, uint32_t batch)
{
    return encaps_tc2_supported(c, batch) && c->p.k % 128 == 0;
}

// a 128-column half tile must lie inside one instance's k columns
bool encaps_tc2_r_inplace_supported(const Ctx *c, uint32_t batch)
{
    return encaps_tc2_supported(c, batch) && c->p.k % 128 == 0;
}

// k = 32 * 2^j <= 2048: the v warps' word-column reduction needs a power-of-two number of words per row
bool encaps_tc2_v_fused_supported(const Ctx *c, uint32_t batch)
{
    const uint32_t wpr = c->p.k / 32;
    return encaps_tc2_bits_supported(c, batch) && c->p.k % 32 == 0 && (wpr & (wpr - 1)) == 0 && wpr <= 64;
}

cudaError_t launch_encaps_tc2(Ctx *c, const uint16_t *d_A, uint16_t *d_U, uint32_t batch, uint32_t row0, uint32_t rows,
                              int mode, uint32_t *d_flags, cudaStream_t st, const uint8_t *d_Rbits,
                              const uint16_t *d_b, const uint8_t *d_mubits, uint16_t *d_v)
{
    if (d_Rbits) {              // B operand expanded from the packed bits inside the kernel
        VArgs va = {};
        if (d_b) {              // ... and v computed by the kernel's spare warps (all m rows, whatever the panel)
            const uint32_t grid = 2 * min((uint32_t)c->sm_count / 2,
                                          ((2 * c->p.n + kPairM - 1) / kPairM) * ((batch * c->p.k + kTileN - 1) / kTileN));
            uint32_t splits = (grid + batch - 1) / batch;
            const uint32_t min_splits = (c->p.m + 65535u) / 65536u, max_splits = (c->p.m + 63u) / 64u;
            if (splits > max_splits) splits = max_splits;
            if (splits < min_splits) splits = min_splits;
            va = VArgs{d_b, d_Rbits, d_mubits, d_v, c->d_vacc, c->d_counters + 8 + c->p.max_batch, c->p.m, batch, splits};
        }
        if (mode == kEpiAccum) return launch_pair<6, 128, kEpiAccum, true>(c, d_A, d_U, nullptr, nullptr, batch, row0, rows, st, d_Rbits, nullptr, false, &va);
        if (mode == kEpiCompare) return launch_pair<6, 128, kEpiCompare, true>(c, d_A, d_U, d_flags, nullptr, batch, row0, rows, st, d_Rbits, nullptr, false, &va);
        return launch_pair<6, 128, kEpiStore, true>(c, d_A, d_U, nullptr, nullptr, batch, row0, rows, st, d_Rbits, nullptr, false, &va);
    }
    if (mode == kEpiAccum) return launch_pair<6, 128, kEpiAccum>(c, d_A, d_U, nullptr, nullptr, batch, row0, rows, st);
    if (mode == kEpiCompare) return launch_pair<6, 128, kEpiCompare>(c, d_A, d_U, d_flags, nullptr, batch, row0, rows, st);
    return launch_pair<6, 128, kEpiStore>(c, d_A, d_U, nullptr, nullptr, batch, row0, rows, st);
}

// N2: U = A^T R + E1 mod q; the int8 operand R is read in place (d_R) or from the copy in the context's operand buffer
cudaError_t launch_encaps_tc2_pv(Ctx *c, const uint16_t *d_A, const int8_t *d_E1, uint16_t *d_U, uint32_t batch,
                                 cudaStream_t st, const int8_t *d_R)
{
    return launch_pair<6, 128, kEpiStorePv>(c, d_A, d_U, nullptr, d_E1, batch, 0, c->p.m, st, nullptr, d_R, d_R != nullptr);
}

// N2 on a wide context: A = the packed low-16 matrix + exception lists, U uint32.  m > 65536: row passes of 65536
// (Table 1's n = 131072 row), the first adds E1, the later ones add the residues already in U.
cudaError_t launch_wide_encaps_tc2(Ctx *c, const int8_t *d_R, const int8_t *d_E1, uint32_t *d_U, uint32_t batch, cudaStream_t st)
{
    const uint32_t m = c->p.m, step = m < 65536u ? m : 65536u;
    for (uint32_t row0 = 0; row0 < m; row0 += step) {
        const uint32_t rows = (m - row0 < step) ? (m - row0) : step;
        cudaError_t err = launch_pair<6, 128, kEpiStorePvW>(c, c->d_A16 + (size_t)row0 * c->p.n, d_U, nullptr,
                                                            row0 == 0 ? d_E1 : nullptr, batch, row0, rows, st, nullptr, d_R,
                                                            encaps_tc2_r_inplace_supported(c, batch));
        if (err != cudaSuccess) return err;
    }
    return cudaSuccess;
}

}  // namespace lwe

// tc_common.cuh -- PTX wrappers shared by the tcgen05 kernels (encaps_tc.cu, keygen_tc.cu):
// mbarrier, TMA (cp.async.bulk.tensor), TMEM allocation, tcgen05.mma kind::i8 / commit / ld,
// shared-memory matrix descriptors and the host-side tensor-map helper.
#pragma once

#include "lwe_internal.cuh"

namespace lwe {
namespace tc {

constexpr uint32_t kUmmaK = 32;       // K per tcgen05.mma for 8-bit operands

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    // Watchdog: a protocol bug (wrong tx byte count, lost arrive) must surface as a launch
    // error, not as a hung GPU.  ~4 s at 2 GHz; only evaluated on the slow path.
    uint32_t done;
    long long t0 = 0;
    for (;;) {
        asm volatile(
            "{\n\t"
            ".reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t"
            "}" : "=r"(done) : "r"(bar), "r"(parity) : "memory");
        if (done) break;
        long long now = clock64();
        if (t0 == 0) t0 = now;
        else if (now - t0 > 8000000000ll) __trap();
    }
}
// true in exactly one lane of a fully converged warp; unlike `lane == 0` the compiler knows the region is
// entered by a single thread of a uniform warp and keeps its operands in uniform registers
__device__ __forceinline__ bool elect_one()
{
    uint32_t pred;
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "elect.sync _|p, 0xffffffff;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap *map, uint32_t bar, int32_t c0, int32_t c1)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1) : "memory");
}
__device__ __forceinline__ void tmem_alloc(uint32_t smem_dst, uint32_t ncols)
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols)
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void umma_i8(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t"
        "}" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld_32x32b_x32(uint32_t taddr, uint32_t (&r)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"
        "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
          "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
          "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// ---- CTA-pair (cta_group::2) variants: two CTAs of a cluster on one TPC share one MMA -------
__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
// shared::cluster address of the same shared-memory offset in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t map_to_cta(uint32_t saddr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// arrive on a barrier that may live in the peer CTA (address from map_to_cta)
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_bar)
{
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_bar) : "memory");
}
// the same with the default (CTA-scope release) semantics: for per-stage producer signals, where the data being
// published is shared memory already fenced into the async proxy.  The cluster-scope release above blocks the
// thread for ~1.5k cycles (measured: one per K block made the expander warps, not the tensor pipe, the limit).
__device__ __forceinline__ void mbar_arrive_remote(uint32_t cluster_bar)
{
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_bar) : "memory");
}
// TMA load whose completion bytes are credited to a barrier of the pair's leader CTA
__device__ __forceinline__ void tma_load_2d_pair(uint32_t dst, const CUtensorMap *map, uint32_t cluster_bar, int32_t c0,
                                                 int32_t c1)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(dst), "l"(map), "r"(cluster_bar), "r"(c0), "r"(c1) : "memory");
}
// executed by the same warp of BOTH CTAs of the pair
__device__ __forceinline__ void tmem_alloc_pair(uint32_t smem_dst, uint32_t ncols)
{
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc_pair(uint32_t taddr, uint32_t ncols)
{
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
// issued by one thread of the leader (even-ranked) CTA; D[256 x N] += A[256 x 32] B[32 x N], each CTA
// supplying its own 128 rows of A and its own N/2 columns of B from the same smem offsets
__device__ __forceinline__ void umma_i8_pair(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::i8 [%0], %1, %2, %3, p;\n\t"
        "}" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
// arrives on the barrier at this shared-memory offset in every CTA of `cta_mask`
__device__ __forceinline__ void umma_commit_pair(uint32_t bar, uint16_t cta_mask)
{
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                 ::"r"(bar), "h"(cta_mask) : "memory");
}

// Shared-memory matrix descriptor, MN-major, SWIZZLE_128B (sm_100 format, version 1):
// [0,14) start>>4 | [16,30) LBO>>4 (stride between 128-byte MN atoms) |
// [32,46) SBO>>4 (stride between 8-row K groups) | [46,48) version=1 | [61,64) layout=2.
__device__ __forceinline__ uint64_t make_desc_mn_sw128(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes)
{
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3ffffu) >> 4);
    d |= (uint64_t)((lbo_bytes >> 4) & 0x3fffu) << 16;
    d |= (uint64_t)((sbo_bytes >> 4) & 0x3fffu) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)2 << 61;
    return d;
}

// Same, K-major SWIZZLE_128B: rows of 128 bytes along K, 8 rows (M/N) per 1 KB atom; SBO = stride
// between 8-row groups; LBO is not used by swizzled K-major layouts.  A K step of 32 bytes inside
// the 128-byte row is taken by advancing the start address.
__device__ __forceinline__ uint64_t make_desc_k_sw128(uint32_t saddr, uint32_t sbo_bytes)
{
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3ffffu) >> 4);
    d |= (uint64_t)((sbo_bytes >> 4) & 0x3fffu) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)2 << 61;
    return d;
}

// Instruction descriptor for kind::i8: D = s32 (c_format 2 at [4,6)), A = B = u8 (format 0 at [7,10),
// [10,13)), A / B major-ness at bits 15 / 16 (1 = MN-major), N>>3 at [17,23), M>>4 at [24,29).
__host__ __device__ constexpr uint32_t instr_desc_u8(uint32_t M, uint32_t N, bool a_mn_major, bool b_mn_major,
                                                     bool b_signed = false)
{
    return (2u << 4) | ((b_signed ? 1u : 0u) << 10) | ((a_mn_major ? 1u : 0u) << 15) | ((b_mn_major ? 1u : 0u) << 16) |
           ((N >> 3) << 17) | ((M >> 4) << 24);
}

// What the U = A^T R kernels do with a finished 16-column piece of a row of U.
//   kEpiStore:   write it.
//   kEpiAccum:   add the residues already stored there (mod q) -- the contraction over the rows of A split into
//                panels (A regenerated panel by panel, encaps with d_A == NULL): a sum of residues mod q is the
//                residue of the sum.
//   kEpiCompare: write nothing; compare with what is stored there (the received ciphertext) and report a
//                mismatch -- the re-encryption check c' = c of the FO transform (Alg.5 l.2-4) without
//                ever materialising c'.
//   kEpiStorePv: the paper's own Encrypt (N2): the B operand is signed (Gaussian r), the accumulators are signed,
//                and E1[j][c] is added before the reduction: U = A^T R + E1 mod q.
//   kEpiStorePvW: the same on a wide context (q > 65536, wide.cu): A is the low-16 matrix, the elements >= 2^16 of
//                column j come from its exception list (2^16 R[i][c] each), U is written as uint32.
enum EpiMode { kEpiStore = 0, kEpiAccum = 1, kEpiCompare = 2, kEpiStorePv = 3, kEpiStorePvW = 4 };

template <int kMode>
__device__ __forceinline__ bool store_u16x16(uint4 *dst, uint32_t (&o)[16], const ModQ &mq)
{
    if (kMode == kEpiAccum || kMode == kEpiCompare) {
        const uint4 p0 = dst[0], p1 = dst[1];
        const uint32_t old[8] = {p0.x, p0.y, p0.z, p0.w, p1.x, p1.y, p1.z, p1.w};
        if (kMode == kEpiCompare) {
            uint32_t diff = 0;
#pragma unroll
            for (int x = 0; x < 8; x++) diff |= old[x] ^ (o[2 * x] | (o[2 * x + 1] << 16));
            return diff != 0;
        }
#pragma unroll
        for (int x = 0; x < 16; x++) {
            uint32_t val = o[x] + ((x & 1) ? (old[x >> 1] >> 16) : (old[x >> 1] & 0xffffu));   // < 2q
            o[x] = mq.pow2 ? (val & mq.mask) : (val >= mq.q ? val - mq.q : val);
        }
    }
    dst[0] = make_uint4(o[0] | (o[1] << 16), o[2] | (o[3] << 16), o[4] | (o[5] << 16), o[6] | (o[7] << 16));
    dst[1] = make_uint4(o[8] | (o[9] << 16), o[10] | (o[11] << 16), o[12] | (o[13] << 16), o[14] | (o[15] << 16));
    return false;
}

// kEpiCompare bookkeeping of one epilogue lane: mismatches are OR-ed per instance and flushed with ONE
// reduction per (lane, instance) -- issued whether or not anything differed, so the work done does not depend
// on the validity of the ciphertext ("constant-time decapsulation path").
struct MismatchAcc {
    uint32_t inst = 0xffffffffu, bad = 0;
    __device__ __forceinline__ void note(uint32_t *flags, uint32_t i, bool b)
    {
        if (i != inst) { flush(flags); inst = i; }
        bad |= b ? 1u : 0u;
    }
    __device__ __forceinline__ void flush(uint32_t *flags)
    {
        if (inst != 0xffffffffu) atomicOr(flags + inst, bad);
        bad = 0;
        inst = 0xffffffffu;
    }
    // end of a tile, whole warp converged: lanes holding the same instance share one reduction
    __device__ __forceinline__ void flush_warp(uint32_t *flags)
    {
        const uint32_t grp = __match_any_sync(0xffffffffu, inst);
        const uint32_t badmask = __ballot_sync(0xffffffffu, bad != 0);
        if (inst != 0xffffffffu && (threadIdx.x & 31) == (uint32_t)(__ffs(grp) - 1))
            atomicOr(flags + inst, (badmask & grp) ? 1u : 0u);
        bad = 0;
        inst = 0xffffffffu;
    }
};

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// u8 matrix [rows][width] row-major, box {128 bytes, box_rows}, SWIZZLE_128B, out-of-bounds -> 0
// pitch: bytes between rows (0 = width: a dense matrix); a larger pitch maps a column range of a wider matrix
inline bool make_map_u8(const Ctx *c, CUtensorMap *map, const void *ptr, uint64_t width, uint64_t rows,
                        uint32_t box_rows, uint64_t pitch = 0)
{
    if (!c->encode_tiled) return false;
    cuuint64_t dims[2] = {width, rows};
    cuuint64_t strides[1] = {pitch ? pitch : width};
    cuuint32_t box[2] = {128, box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = ((EncodeTiledFn)c->encode_tiled)(map, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void *>(ptr), dims,
                                                  strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                                  CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

// u8 matrix [rows][width] row-major, box {box_w bytes, box_rows}, no swizzle, out-of-bounds -> 0
inline bool make_map_plain_u8(const Ctx *c, CUtensorMap *map, const void *ptr, uint64_t width, uint64_t rows,
                              uint32_t box_w, uint32_t box_rows)
{
    if (!c->encode_tiled) return false;
    cuuint64_t dims[2] = {width, rows};
    cuuint64_t strides[1] = {width};
    cuuint32_t box[2] = {box_w, box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = ((EncodeTiledFn)c->encode_tiled)(map, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void *>(ptr), dims,
                                                  strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                                  CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

}  // namespace tc
}  // namespace lwe

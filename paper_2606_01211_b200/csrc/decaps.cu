// decaps.cu -- a6: d_c = v_c - sum_j U[j][c] s_j mod q, rounded to a bit.
//
// A column-sum of the n x k row-major U weighted by s: threads sit side by side on a
// row (8 columns = 16 bytes each, so a k = 256 row is one 512-byte coalesced read by a
// warp), rows are split over the CTAs of an instance, partial column sums meet in u64
// global accumulators, and the last CTA of the instance to finish (ticket counter)
// rounds and packs the k bits.  Accumulators and tickets are left zeroed for the next
// call.  Exact for any q: products < 2^32, sums < 2^48.
#include "lwe_internal.cuh"

namespace lwe {

constexpr int kDecThreads = 256;

__device__ __forceinline__ uint4 ldg_stream16(const uint4 *p)
{
    uint4 r;                                             // not volatile: read-only data, free to hoist
    asm("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
        : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

// acc += x * y with a 32 x 32 -> 64 bit multiply-add (one IMAD.WIDE)
__device__ __forceinline__ void mad_wide(unsigned long long &acc, uint32_t x, uint32_t y)
{
    asm("mad.wide.u32 %0, %1, %2, %0;" : "+l"(acc) : "r"(x), "r"(y));
}

__device__ __forceinline__ void accumulate_row(unsigned long long (&a)[8], const uint4 &u, uint32_t sj)
{
    mad_wide(a[0], u.x & 0xffffu, sj); mad_wide(a[1], u.x >> 16, sj);
    mad_wide(a[2], u.y & 0xffffu, sj); mad_wide(a[3], u.y >> 16, sj);
    mad_wide(a[4], u.z & 0xffffu, sj); mad_wide(a[5], u.z >> 16, sj);
    mad_wide(a[6], u.w & 0xffffu, sj); mad_wide(a[7], u.w >> 16, sj);
}

__global__ void __launch_bounds__(kDecThreads)
decaps_kernel(const uint16_t *__restrict__ U, const uint16_t *__restrict__ v, const uint16_t *__restrict__ s,
              uint8_t *__restrict__ out, unsigned long long *__restrict__ acc, unsigned int *__restrict__ tickets,
              uint32_t n, uint32_t k, ModQ mq)
{
    __shared__ uint32_t sLast;
    pdl_trigger();
    pdl_wait();
    const uint32_t t = blockIdx.y;                       // instance
    const uint32_t tpr = k / 8;                          // threads per row
    const uint32_t rows_per_iter = kDecThreads / tpr;    // >= 1 (k <= 2048 checked by the host)
    const uint32_t rslot = threadIdx.x / tpr, cg = threadIdx.x % tpr;
    const bool active = rslot < rows_per_iter;
    const uint16_t *Ut = U + (size_t)t * n * k;
    const uint16_t *st = s + (size_t)t * n;

    unsigned long long a[8];
#pragma unroll
    for (int x = 0; x < 8; x++) a[x] = 0;
    if (active) {
        // a CTA streams one contiguous range of rows; 8 independent 16-byte loads in flight per thread: the pass is
        // HBM-bound (2nk bytes of U) only with ~100 KB in flight per SM (4 loads per thread left it latency-bound at
        // 4.2 TB/s: ncu, round 2)
        constexpr int kUnroll = 8;
        const uint32_t per_cta = ((n + gridDim.x - 1) / gridDim.x + rows_per_iter - 1) / rows_per_iter * rows_per_iter;
        const uint32_t jbeg = blockIdx.x * per_cta, jend = min(n, jbeg + per_cta);
        const size_t row_u4 = k / 8;                      // uint4 per row
        uint32_t j = jbeg + rslot;
        const uint4 *up = reinterpret_cast<const uint4 *>(Ut) + (size_t)j * row_u4 + cg;
        const size_t ustep = (size_t)rows_per_iter * row_u4;
        for (; j + (kUnroll - 1) * rows_per_iter < jend; j += kUnroll * rows_per_iter, up += kUnroll * ustep) {
            uint4 u[kUnroll];
            uint32_t sj[kUnroll];
#pragma unroll
            for (int r = 0; r < kUnroll; r++) {
                u[r] = ldg_stream16(up + r * ustep);
                sj[r] = __ldg(st + j + r * rows_per_iter);
            }
#pragma unroll
            for (int r = 0; r < kUnroll; r++) accumulate_row(a, u[r], sj[r]);
        }
        for (; j < jend; j += rows_per_iter, up += ustep) accumulate_row(a, ldg_stream16(up), __ldg(st + j));
    }
    // sum the row slots of the CTA in shared memory, then one atomic per column per CTA.  Staged [row slot][column]:
    // a thread stores its 8 columns as 64 contiguous bytes and thread c then reads column c of every slot -- consecutive
    // 8-byte words across a warp in both phases (the earlier [x][thread] layout read 8 lanes from one bank: 660 k
    // conflicts per launch at C4, ncu)
    __shared__ __align__(16) unsigned long long sCol[kDecThreads * 8];
    {
        ulonglong2 *dst = reinterpret_cast<ulonglong2 *>(sCol + (size_t)threadIdx.x * 8);   // = [rslot][cg * 8 + x]
        dst[0] = make_ulonglong2(a[0], a[1]); dst[1] = make_ulonglong2(a[2], a[3]);
        dst[2] = make_ulonglong2(a[4], a[5]); dst[3] = make_ulonglong2(a[6], a[7]);
    }
    __syncthreads();
    for (uint32_t c = threadIdx.x; c < k; c += kDecThreads) {
        unsigned long long sum = 0;
        for (uint32_t rs = 0; rs < rows_per_iter; rs++) sum += sCol[(size_t)rs * k + c];
        if (sum) atomicAdd(acc + (size_t)t * k + c, sum);
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) sLast = (atomicAdd(tickets + t, 1u) == gridDim.x - 1) ? 1u : 0u;
    __syncthreads();
    if (!sLast) return;
    __threadfence();
    // finalize: one column per thread, a warp's 32 decisions packed by ballot (4 output bytes)
    for (uint32_t c0 = 0; c0 < k; c0 += kDecThreads) {
        const uint32_t c = c0 + threadIdx.x;
        uint32_t bit = 0;
        if (c < k) {
            unsigned long long sum = __ldcg(acc + (size_t)t * k + c);
            acc[(size_t)t * k + c] = 0;
            uint32_t us = mod_u64(sum, mq);
            uint32_t d = (uint32_t)v[(size_t)t * k + c] + mq.q - us;
            if (d >= mq.q) d -= mq.q;
            bit = (4u * d + mq.q) / (2u * mq.q) & 1u;            // d < q <= 65536: fits 32 bits
        }
        const uint32_t word = __ballot_sync(0xffffffffu, bit);
        if ((threadIdx.x & 31) == 0) {
            const uint32_t cw = c0 + (threadIdx.x & ~31u);          // first column of this warp
            for (uint32_t by = 0; by < 4 && cw + 8 * by < k; by++)
                out[(size_t)t * (k / 8) + cw / 8 + by] = (uint8_t)(word >> (8 * by));
        }
    }
    if (threadIdx.x == 0) tickets[t] = 0;
}

cudaError_t launch_decaps(Ctx *c, const uint16_t *d_U, const uint16_t *d_v, const uint16_t *d_s,
                          uint8_t *d_out, uint32_t batch, cudaStream_t st)
{
    const uint32_t n = c->p.n, k = c->p.k;
    const uint32_t rows_per_iter = kDecThreads / (k / 8);
    // exactly one wave of resident CTAs (a second, partial wave was the tail: 1184 CTAs on 740 slots ran at
    // 0.54 of HBM): as many row splits per instance as fit the SMs at the kernel's occupancy
    int per_sm = 1;
    cudaError_t perr = kernel_prepare(c, decaps_kernel, 0, kDecThreads, &per_sm);
    if (perr != cudaSuccess) return perr;
    uint32_t splits = (uint32_t)(per_sm * c->sm_count) / batch;
    uint32_t max_splits = (n + 4 * rows_per_iter - 1) / (4 * rows_per_iter);       // >= 4 row groups per CTA
    if (splits > max_splits) splits = max_splits;
    if (splits < 1) splits = 1;
    dim3 grid(splits, batch);
    ProfScope prof(c, LWE_K_DECAPS, st);
    return launch_k(c, decaps_kernel, grid, kDecThreads, 0, st, d_U, d_v, d_s, d_out, c->d_dacc, c->d_counters + 8, n, k, c->mq);
}

// FO verdict (Alg.5 l.4): ok[t] = 1 iff the re-encrypted ciphertext equals the received one, i.e. no
// U tile reported a mismatch (flags[t] == 0, set by the compare epilogue of the encaps GEMM) and v' == v.
// One warp per instance; the whole v row is always read (no early exit).
__global__ void __launch_bounds__(32)
fo_verdict_kernel(const uint16_t *__restrict__ v, const uint16_t *__restrict__ vprime, const uint32_t *__restrict__ flags,
                  uint8_t *__restrict__ ok, uint32_t k)
{
    const uint32_t t = blockIdx.x;
    uint32_t diff = 0;
    for (uint32_t c = threadIdx.x; c < k; c += 32) diff |= (uint32_t)(v[(size_t)t * k + c] ^ vprime[(size_t)t * k + c]);
    diff |= flags[t];
    const uint32_t any = __ballot_sync(0xffffffffu, diff != 0);
    if (threadIdx.x == 0) ok[t] = any ? 0 : 1;
}

cudaError_t launch_fo_verdict(Ctx *c, const uint16_t *d_v, const uint16_t *d_vprime, const uint32_t *d_flags,
                              uint8_t *d_ok, uint32_t batch, cudaStream_t st)
{
    ProfScope prof(c, LWE_K_FO_VERDICT, st);
    fo_verdict_kernel<<<batch, 32, 0, st>>>(d_v, d_vprime, d_flags, d_ok, c->p.k);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace lwe

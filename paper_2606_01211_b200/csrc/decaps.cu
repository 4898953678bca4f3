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

// Column accumulators of one thread (8 adjacent columns).  kAcc32 = false: u64 sums of the 32-bit products (exact for any
// q; one IMAD.WIDE and one unpack instruction per element).  kAcc32 = true (q a power of two): u32 sums that wrap mod 2^32 --
// exact mod q because q | 2^32 -- of products that keep the neighbouring column's bits above bit 15 (no mask: the low 16
// bits of u * s depend only on the low 16 bits of u), i.e. one IMAD per element and one shift per pair: half the issue slots.
template <bool kAcc32> struct ColAcc;
template <> struct ColAcc<false> {
    typedef unsigned long long T;
    static __device__ __forceinline__ void mad(T &acc, uint32_t x, uint32_t y) { asm("mad.wide.u32 %0, %1, %2, %0;" : "+l"(acc) : "r"(x), "r"(y)); }
    static __device__ __forceinline__ void row(T (&a)[8], const uint4 &u, uint32_t sj)
    {
        mad(a[0], u.x & 0xffffu, sj); mad(a[1], u.x >> 16, sj);
        mad(a[2], u.y & 0xffffu, sj); mad(a[3], u.y >> 16, sj);
        mad(a[4], u.z & 0xffffu, sj); mad(a[5], u.z >> 16, sj);
        mad(a[6], u.w & 0xffffu, sj); mad(a[7], u.w >> 16, sj);
    }
};
template <> struct ColAcc<true> {
    typedef uint32_t T;
    static __device__ __forceinline__ void row(T (&a)[8], const uint4 &u, uint32_t sj)
    {
        a[0] += u.x * sj; a[1] += (u.x >> 16) * sj; a[2] += u.y * sj; a[3] += (u.y >> 16) * sj;
        a[4] += u.z * sj; a[5] += (u.z >> 16) * sj; a[6] += u.w * sj; a[7] += (u.w >> 16) * sj;
    }
};

template <bool kAcc32>
__global__ void __launch_bounds__(kDecThreads)
decaps_kernel(const uint16_t *__restrict__ U, const uint16_t *__restrict__ v, const uint16_t *__restrict__ s,
              uint8_t *__restrict__ out, unsigned long long *__restrict__ acc, unsigned int *__restrict__ tickets,
              uint32_t n, uint32_t k, ModQ mq)
{
    typedef typename ColAcc<kAcc32>::T AccT;
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

    AccT a[8];
#pragma unroll
    for (int x = 0; x < 8; x++) a[x] = 0;
    if (active) {
        // A CTA streams one contiguous range of rows, software-pipelined in registers: the loads of the next batch of
        // kUnroll rows are issued before the current batch is consumed, so every thread has 4-8 independent 16-byte loads
        // in flight at all times (the pass is HBM-bound -- 2nk bytes of U -- only with ~100 KB in flight per SM; with
        // load-then-consume batches the kernel sat at 4.4 TB/s, a pure load loop of the same shape reaches 6.4).  Every
        // batch is a full one: a row past the end of the range re-reads the instance's first row (a valid address) with
        // s = 0, so that no thread ever walks a tail of single, latency-bound loads.
        constexpr int kUnroll = 4;
        const uint32_t per_cta = ((n + gridDim.x - 1) / gridDim.x + rows_per_iter - 1) / rows_per_iter * rows_per_iter;
        const uint32_t jbeg = blockIdx.x * per_cta, jend = min(n, jbeg + per_cta);
        const size_t row_u4 = k / 8;                      // uint4 per row
        uint32_t j = jbeg + rslot;
        const uint4 *up = reinterpret_cast<const uint4 *>(Ut) + (size_t)j * row_u4 + cg;
        const size_t ustep = (size_t)rows_per_iter * row_u4;
        const uint32_t jstep = kUnroll * rows_per_iter;
        uint4 u0[kUnroll], u1[kUnroll];
        uint32_t s0[kUnroll], s1[kUnroll];
        auto load = [&](uint4 (&uu)[kUnroll], uint32_t (&ss)[kUnroll]) {
#pragma unroll
            for (int r = 0; r < kUnroll; r++) {
                const bool in = j + r * rows_per_iter < jend;
                uu[r] = ldg_stream16(in ? up + r * ustep : reinterpret_cast<const uint4 *>(Ut) + cg);
                ss[r] = in ? (uint32_t)__ldg(st + j + r * rows_per_iter) : 0u;
            }
            j += jstep;
            up += kUnroll * ustep;
        };
        if (j < jend) {
            load(u0, s0);
            for (;;) {
                const bool more1 = j < jend;
                if (more1) load(u1, s1);
#pragma unroll
                for (int r = 0; r < kUnroll; r++) ColAcc<kAcc32>::row(a, u0[r], s0[r]);
                if (!more1) break;
                const bool more0 = j < jend;
                if (more0) load(u0, s0);
#pragma unroll
                for (int r = 0; r < kUnroll; r++) ColAcc<kAcc32>::row(a, u1[r], s1[r]);
                if (!more0) break;
            }
        }
    }
    // sum the row slots of the CTA in shared memory, then one atomic per column per CTA.  Staged [row slot][column]:
    // a thread stores its 8 columns contiguously and thread c then reads column c of every slot -- consecutive
    // words across a warp in both phases (the earlier [x][thread] layout read 8 lanes from one bank: 660 k
    // conflicts per launch at C4, ncu)
    __shared__ __align__(16) AccT sCol[kDecThreads * 8];
#pragma unroll
    for (int x = 0; x < 8; x++) sCol[(size_t)threadIdx.x * 8 + x] = a[x];   // = [rslot][cg * 8 + x], vectorised by the compiler
    __syncthreads();
    for (uint32_t c = threadIdx.x; c < k; c += kDecThreads) {
        AccT sum = 0;
        for (uint32_t rs = 0; rs < rows_per_iter; rs++) sum += sCol[(size_t)rs * k + c];
        // u32 sums (q | 2^32) are added into the low word of the u64 accumulator: a carry into the high word is harmless,
        // the finalize step reduces mod q
        if (sum) atomicAdd(acc + (size_t)t * k + c, (unsigned long long)sum);
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

template <bool kAcc32>
static cudaError_t launch_decaps_t(Ctx *c, const uint16_t *d_U, const uint16_t *d_v, const uint16_t *d_s,
                                   uint8_t *d_out, uint32_t batch, cudaStream_t st)
{
    const uint32_t n = c->p.n, k = c->p.k;
    const uint32_t rows_per_iter = kDecThreads / (k / 8);
    // exactly one wave of resident CTAs (a second, partial wave was the tail: 1184 CTAs on 740 slots ran at
    // 0.54 of HBM): as many row splits per instance as fit the SMs at the kernel's occupancy
    int per_sm = 1;
    cudaError_t perr = kernel_prepare(c, decaps_kernel<kAcc32>, 0, kDecThreads, &per_sm);
    if (perr != cudaSuccess) return perr;
    uint32_t splits = (uint32_t)(per_sm * c->sm_count) / batch;
    uint32_t max_splits = (n + 4 * rows_per_iter - 1) / (4 * rows_per_iter);       // >= 4 row groups per CTA
    if (splits > max_splits) splits = max_splits;
    if (splits < 1) splits = 1;
    dim3 grid(splits, batch);
    ProfScope prof(c, LWE_K_DECAPS, st);
    return launch_k(c, decaps_kernel<kAcc32>, grid, kDecThreads, 0, st, d_U, d_v, d_s, d_out, c->d_dacc, c->d_counters + 8, n, k, c->mq);
}

cudaError_t launch_decaps(Ctx *c, const uint16_t *d_U, const uint16_t *d_v, const uint16_t *d_s,
                          uint8_t *d_out, uint32_t batch, cudaStream_t st)
{
    return c->mq.pow2 ? launch_decaps_t<true>(c, d_U, d_v, d_s, d_out, batch, st)
                      : launch_decaps_t<false>(c, d_U, d_v, d_s, d_out, batch, st);
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

// decaps_static.cu -- lwe_decaps_static: Decaps (a6) for callers that must not allocate.
//
// Who this is for.  Every other entry point needs an lwe_ctx, and lwe_create() sizes a workspace with cudaMalloc.
// Some callers cannot do that: code running inside another framework's memory plan (a serving process whose caching
// allocator has already claimed the whole device, so a raw cudaMalloc fails or fragments its pool), a plug-in that is
// handed buffers and a stream and is forbidden to touch the allocator, or a latency-critical thread that must not take
// the driver's allocation lock (cudaMalloc / cudaFree synchronise the whole device).  For them the column accumulators
// and the "last CTA" tickets that lwe_decaps keeps in its context live here in ONE fixed array that is part of the
// library image: `static __device__`, so every GPU that loads the library carries its kStaticBytes (about 128 KiB)
// from module load until the process exits, whether or not this entry point is ever called.
//
// What follows from the array being shared and fixed:
//  * sizes are capped (LWE_STATIC_MAX_COLS accumulators = batch * k, LWE_STATIC_MAX_BATCH instances): larger calls get
//    LWE_ERR_UNSUPPORTED and nothing is launched;
//  * the array keeps whatever the previous call left in it, so each call first clears the part it will use (a
//    cudaMemsetAsync on the caller's stream, which does not allocate);
//  * all calls on one device use the same memory: two calls may not overlap on the GPU (different streams without an
//    ordering between them, or two host threads) -- they would add into each other's sums.  Calls on one stream are
//    ordered by the stream and are fine;
//  * in host code the array's name is only a handle for the runtime, not a device address.  The address is looked up
//    with cudaGetSymbolAddress once per device, with that device current, on the FIRST call made on that device; make
//    that first call outside any stream capture (the look-up may load the module).  Later calls only enqueue.
//
// The kernel is a variant of decaps_kernel (decaps.cu) with the same arithmetic -- u64 column sums of U[j][c] * s[j],
// exact for every q <= 65536 -- but it does not reset its scratch (the host clears it) and takes no part in the
// context's programmatic-dependent-launch chain.  No code path of the context-based calls is touched.
#include <mutex>

#include "lwe_internal.cuh"

namespace lwe {

constexpr int kStThreads = 256;
constexpr uint32_t kStaticMaxCols = LWE_STATIC_MAX_COLS;       // u64 accumulators: batch * k
constexpr uint32_t kStaticMaxBatch = LWE_STATIC_MAX_BATCH;     // u32 tickets
constexpr size_t kStaticWords = kStaticMaxCols + kStaticMaxBatch / 2;   // in unsigned long long
constexpr size_t kStaticBytes = kStaticWords * sizeof(unsigned long long);
constexpr int kStaticMaxDevices = 64;

// [0, kStaticMaxCols): column accumulators [instance][k]; then kStaticMaxBatch u32 tickets.
static __device__ __align__(256) unsigned long long g_decaps_static_scratch[kStaticWords];

__global__ void __launch_bounds__(kStThreads)
decaps_static_kernel(const uint16_t *__restrict__ U, const uint16_t *__restrict__ v, const uint16_t *__restrict__ s,
                     uint8_t *__restrict__ out, unsigned long long *__restrict__ acc, unsigned int *__restrict__ tickets,
                     uint32_t n, uint32_t k, ModQ mq)
{
    __shared__ uint32_t sLast;
    __shared__ __align__(16) unsigned long long sCol[kStThreads * 8];
    const uint32_t t = blockIdx.y;                       // instance
    const uint32_t tpr = k / 8;                          // threads per row of U (8 columns = 16 bytes each)
    const uint32_t rows_per_iter = kStThreads / tpr;     // >= 1: k <= 2048 checked by the host
    const uint32_t rslot = threadIdx.x / tpr, cg = threadIdx.x % tpr;
    const uint16_t *Ut = U + (size_t)t * n * k;
    const uint16_t *st = s + (size_t)t * n;

    unsigned long long a[8];
#pragma unroll
    for (int x = 0; x < 8; x++) a[x] = 0;
    if (rslot < rows_per_iter) {
        // this CTA's contiguous range of rows, four independent 16-byte loads in flight per thread
        const uint32_t per_cta = ((n + gridDim.x - 1) / gridDim.x + rows_per_iter - 1) / rows_per_iter * rows_per_iter;
        const uint32_t jbeg = blockIdx.x * per_cta, jend = min(n, jbeg + per_cta);
        const uint4 *Ur = reinterpret_cast<const uint4 *>(Ut);
        for (uint32_t j0 = jbeg + rslot; j0 < jend; j0 += 4 * rows_per_iter) {
            uint4 u[4];
            uint32_t sj[4];
#pragma unroll
            for (int r = 0; r < 4; r++) {
                const uint32_t j = j0 + r * rows_per_iter;
                const bool in = j < jend;
                u[r] = in ? __ldg(Ur + (size_t)j * tpr + cg) : make_uint4(0, 0, 0, 0);
                sj[r] = in ? (uint32_t)__ldg(st + j) : 0u;
            }
#pragma unroll
            for (int r = 0; r < 4; r++) {
                a[0] += (unsigned long long)(u[r].x & 0xffffu) * sj[r]; a[1] += (unsigned long long)(u[r].x >> 16) * sj[r];
                a[2] += (unsigned long long)(u[r].y & 0xffffu) * sj[r]; a[3] += (unsigned long long)(u[r].y >> 16) * sj[r];
                a[4] += (unsigned long long)(u[r].z & 0xffffu) * sj[r]; a[5] += (unsigned long long)(u[r].z >> 16) * sj[r];
                a[6] += (unsigned long long)(u[r].w & 0xffffu) * sj[r]; a[7] += (unsigned long long)(u[r].w >> 16) * sj[r];
            }
        }
    }
    // row slots of the CTA meet in shared memory ([row slot][column]), then one atomic per column per CTA
#pragma unroll
    for (int x = 0; x < 8; x++) sCol[(size_t)threadIdx.x * 8 + x] = a[x];
    __syncthreads();
    for (uint32_t c = threadIdx.x; c < k; c += kStThreads) {
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
    // the instance's last CTA: d = v - sum mod q, one column per thread, a warp's 32 decisions packed by ballot.
    // Nothing is reset here: the next call clears its own part of the scratch before it launches.
    for (uint32_t c0 = 0; c0 < k; c0 += kStThreads) {
        const uint32_t c = c0 + threadIdx.x;
        uint32_t bit = 0;
        if (c < k) {
            const uint32_t us = mod_u64(__ldcg(acc + (size_t)t * k + c), mq);
            uint32_t d = (uint32_t)v[(size_t)t * k + c] + mq.q - us;
            if (d >= mq.q) d -= mq.q;
            bit = (4u * d + mq.q) / (2u * mq.q) & 1u;    // 1 iff q/4 <= d < 3q/4
        }
        const uint32_t word = __ballot_sync(0xffffffffu, bit);
        if ((threadIdx.x & 31) == 0) {
            const uint32_t cw = c0 + (threadIdx.x & ~31u);
            for (uint32_t by = 0; by < 4 && cw + 8 * by < k; by++)
                out[(size_t)t * (k / 8) + cw / 8 + by] = (uint8_t)(word >> (8 * by));
        }
    }
}

// What the first call on a device finds out and every later call reuses.
struct StaticDev {
    bool ready;
    unsigned long long *scratch;      // device address of g_decaps_static_scratch ON THIS DEVICE
    int sm_count;
    int cc_major;
};
static StaticDev g_static_dev[kStaticMaxDevices];
static std::mutex g_static_mutex;

// Must run with `dev` current: cudaGetSymbolAddress answers for the current device's copy of the array.
static cudaError_t static_setup(int dev, StaticDev *out)
{
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticDev &d = g_static_dev[dev];
    if (!d.ready) {
        void *ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&ptr, g_decaps_static_scratch);
        if (e != cudaSuccess) return e;
        if (ptr == nullptr) return cudaErrorInvalidSymbol;
        if ((e = cudaDeviceGetAttribute(&d.sm_count, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
        if ((e = cudaDeviceGetAttribute(&d.cc_major, cudaDevAttrComputeCapabilityMajor, dev)) != cudaSuccess) return e;
        d.scratch = static_cast<unsigned long long *>(ptr);
        d.ready = true;
    }
    *out = d;
    return cudaSuccess;
}

}  // namespace lwe

using namespace lwe;

extern "C" int lwe_decaps_static(uint32_t n, uint32_t k, uint32_t q, const uint16_t *d_U, const uint16_t *d_v,
                                 const uint16_t *d_s, uint8_t *d_mubits_out, uint32_t batch, void *stream)
{
    if (n == 0 || k == 0 || k % 8 || k > 2048 || n > (1u << 20) || q < 2 || q > 65536u || batch == 0) return LWE_ERR_PARAM;
    if (!d_U || !d_v || !d_s || !d_mubits_out) return LWE_ERR_NULLPTR;
    if (((uintptr_t)d_U | (uintptr_t)d_v | (uintptr_t)d_s | (uintptr_t)d_mubits_out) & 15) return LWE_ERR_ALIGN;
    // the fixed array bounds what one call may ask for
    if (batch > kStaticMaxBatch || (uint64_t)batch * k > kStaticMaxCols) return LWE_ERR_UNSUPPORTED;

    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return LWE_ERR_CUDA;
    if (dev < 0 || dev >= kStaticMaxDevices) return LWE_ERR_UNSUPPORTED;
    StaticDev sd;
    if (static_setup(dev, &sd) != cudaSuccess) return LWE_ERR_CUDA;
    if (sd.cc_major != 10) return LWE_ERR_UNSUPPORTED;       // sm_100a code only, no other backend

    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long *acc = sd.scratch;
    unsigned int *tickets = reinterpret_cast<unsigned int *>(sd.scratch + kStaticMaxCols);
    // the array still holds the previous call's sums and tickets: clear the part this call uses, in stream order
    if (cudaMemsetAsync(acc, 0, (size_t)batch * k * sizeof(unsigned long long), st) != cudaSuccess) return LWE_ERR_CUDA;
    if (cudaMemsetAsync(tickets, 0, (size_t)batch * sizeof(unsigned int), st) != cudaSuccess) return LWE_ERR_CUDA;

    // one wave: as many row ranges per instance as fit the SMs at 4 CTAs each, at least 4 row groups per CTA
    const uint32_t rows_per_iter = kStThreads / (k / 8);
    uint32_t splits = (uint32_t)(4 * sd.sm_count) / batch;
    const uint32_t max_splits = (n + 4 * rows_per_iter - 1) / (4 * rows_per_iter);
    if (splits > max_splits) splits = max_splits;
    if (splits < 1) splits = 1;
    const uint32_t mod = q;
    ModQ mq;
    mq.q = mod;
    mq.mu = (uint32_t)((1ull << 32) / mod);
    mq.T = mod * (65536u / mod);
    mq.half = mod / 2;
    mq.pow2 = (mod & (mod - 1)) == 0 ? 1u : 0u;
    mq.mask = mod - 1;
    mq.two32 = (uint32_t)((1ull << 32) % mod);
    decaps_static_kernel<<<dim3(splits, batch), kStThreads, 0, st>>>(d_U, d_v, d_s, d_mubits_out, acc, tickets, n, k, mq);
    return cudaGetLastError() == cudaSuccess ? LWE_OK : LWE_ERR_CUDA;
}

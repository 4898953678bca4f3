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

__global__ void __launch_bounds__(kDecThreads)
decaps_kernel(const uint16_t *__restrict__ U, const uint16_t *__restrict__ v, const uint16_t *__restrict__ s,
              uint8_t *__restrict__ out, unsigned long long *__restrict__ acc, unsigned int *__restrict__ tickets,
              uint32_t n, uint32_t k, ModQ mq)
{
    __shared__ uint32_t sLast;
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
        for (uint32_t j = blockIdx.x * rows_per_iter + rslot; j < n; j += gridDim.x * rows_per_iter) {
            uint4 u = __ldg(reinterpret_cast<const uint4 *>(Ut + (size_t)j * k) + cg);
            uint32_t sj = __ldg(st + j);
            a[0] += (unsigned long long)((u.x & 0xffffu) * sj);
            a[1] += (unsigned long long)((u.x >> 16) * sj);
            a[2] += (unsigned long long)((u.y & 0xffffu) * sj);
            a[3] += (unsigned long long)((u.y >> 16) * sj);
            a[4] += (unsigned long long)((u.z & 0xffffu) * sj);
            a[5] += (unsigned long long)((u.z >> 16) * sj);
            a[6] += (unsigned long long)((u.w & 0xffffu) * sj);
            a[7] += (unsigned long long)((u.w >> 16) * sj);
        }
    }
    // sum the row slots of the CTA in shared memory, then one atomic per column per CTA
    __shared__ unsigned long long sCol[kDecThreads * 8];
#pragma unroll
    for (int x = 0; x < 8; x++) sCol[x * kDecThreads + threadIdx.x] = a[x];      // inactive threads hold zeros
    __syncthreads();
    for (uint32_t c = threadIdx.x; c < k; c += kDecThreads) {
        const uint32_t ccg = c >> 3, x = c & 7;
        unsigned long long sum = 0;
        for (uint32_t rs = 0; rs < rows_per_iter; rs++) sum += sCol[x * kDecThreads + rs * tpr + ccg];
        if (sum) atomicAdd(acc + (size_t)t * k + c, sum);
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) sLast = (atomicAdd(tickets + t, 1u) == gridDim.x - 1) ? 1u : 0u;
    __syncthreads();
    if (!sLast) return;
    __threadfence();
    // finalize: k columns, 8 per thread-iteration -> one output byte
    for (uint32_t byte = threadIdx.x; byte < k / 8; byte += kDecThreads) {
        uint32_t bits = 0;
        for (uint32_t x = 0; x < 8; x++) {
            uint32_t c = 8 * byte + x;
            unsigned long long sum = __ldcg(acc + (size_t)t * k + c);
            acc[(size_t)t * k + c] = 0;
            uint32_t us = mod_u64(sum, mq);
            uint32_t d = (uint32_t)v[(size_t)t * k + c] + mq.q - us;
            if (d >= mq.q) d -= mq.q;
            uint32_t bit = (uint32_t)(((4ull * d + mq.q) / (2ull * mq.q)) & 1ull);
            bits |= bit << x;
        }
        out[(size_t)t * (k / 8) + byte] = (uint8_t)bits;
    }
    if (threadIdx.x == 0) tickets[t] = 0;
}

cudaError_t launch_decaps(Ctx *c, const uint16_t *d_U, const uint16_t *d_v, const uint16_t *d_s,
                          uint8_t *d_out, uint32_t batch, cudaStream_t st)
{
    const uint32_t n = c->p.n, k = c->p.k;
    const uint32_t rows_per_iter = kDecThreads / (k / 8);
    uint32_t splits = (uint32_t)((4 * c->sm_count + batch - 1) / batch);
    uint32_t max_splits = (n + 4 * rows_per_iter - 1) / (4 * rows_per_iter);       // >= 4 row groups per CTA
    if (splits > max_splits) splits = max_splits;
    if (splits < 1) splits = 1;
    dim3 grid(splits, batch);
    ProfScope prof(c, LWE_K_DECAPS, st);
    decaps_kernel<<<grid, kDecThreads, 0, st>>>(d_U, d_v, d_s, d_out, c->d_dacc, c->d_counters + 8, n, k, c->mq);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace lwe

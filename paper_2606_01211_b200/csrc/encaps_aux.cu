// encaps_aux.cu -- the small parts of Encaps (S8(a) a4/a5):
//   * expand_R_and_v: one pass over the packed bits of R that (i) writes them as the
//     u8 {0,1} B-operand of the tensor-core GEMM, laid out [i][t*k + c] so that one
//     256-column GEMM tile is one instance, and (ii) accumulates
//     v_c = sum_i b_i R_ic + mu_c floor(q/2) mod q  (BJ north_star) on the fly,
//     so that R's bits are read from HBM once.
//   * encaps_simt: CUDA-core U = A^T R for shapes the tensor path does not take
//     (k % 16 != 0, tiny n) and as an in-library cross-check of the tcgen05 kernel.
#include "lwe_internal.cuh"

namespace lwe {

constexpr int kAuxThreads = 256;

// grid (row_splits, batch).  Thread = (row slot, column byte): 8 columns of one row.
__global__ void __launch_bounds__(kAuxThreads)
expand_R_and_v_kernel(const uint16_t *__restrict__ b, const uint8_t *__restrict__ Rbits,
                      const uint8_t *__restrict__ mubits, uint8_t *__restrict__ Rexp, uint16_t *__restrict__ v,
                      unsigned long long *__restrict__ acc, unsigned int *__restrict__ tickets,
                      uint32_t m, uint32_t k, uint32_t ld_exp, bool write_Rexp, ModQ mq)
{
    __shared__ uint32_t sLast;
    const uint32_t t = blockIdx.y;
    const uint32_t kb = k / 8;                           // bytes of R bits per row
    const uint32_t rows_per_iter = kAuxThreads / kb;     // >= 1 (k <= 2048)
    const uint32_t rslot = threadIdx.x / kb, cb = threadIdx.x % kb;
    const bool active = rslot < rows_per_iter;
    const uint8_t *Rt = Rbits + (size_t)t * m * kb;
    const uint16_t *bt = b + (size_t)t * m;

    uint32_t a[8];                                       // sum_i b_i R_ic <= 65535 * 65536 < 2^32
#pragma unroll
    for (int x = 0; x < 8; x++) a[x] = 0;
    if (active) {
        for (uint32_t i = blockIdx.x * rows_per_iter + rslot; i < m; i += gridDim.x * rows_per_iter) {
            uint32_t r = __ldg(Rt + (size_t)i * kb + cb);
            uint32_t bi = __ldg(bt + i);
            if (write_Rexp) {
                // bit x of r -> byte x of the 8-byte output: (nibble * 0x00204081) & 0x01010101
                uint32_t lo = ((r & 0xfu) * 0x00204081u) & 0x01010101u;
                uint32_t hi = ((r >> 4) * 0x00204081u) & 0x01010101u;
                *reinterpret_cast<uint2 *>(Rexp + (size_t)i * ld_exp + (size_t)t * k + 8 * cb) = make_uint2(lo, hi);
            }
#pragma unroll
            for (int x = 0; x < 8; x++) a[x] += ((r >> x) & 1u) ? bi : 0u;
        }
    }
    // Block-level sum over the row slots (a CTA's total still fits 32 bits: <= 65535 * m), then
    // ONE atomic per column per CTA instead of one per thread.
    __shared__ uint32_t sCol[kAuxThreads * 8];
#pragma unroll
    for (int x = 0; x < 8; x++) sCol[x * kAuxThreads + threadIdx.x] = active ? a[x] : 0u;
    __syncthreads();
    for (uint32_t c = threadIdx.x; c < k; c += kAuxThreads) {
        const uint32_t ccb = c >> 3, x = c & 7;
        uint32_t sum = 0;
        for (uint32_t rs = 0; rs < rows_per_iter; rs++) sum += sCol[x * kAuxThreads + rs * kb + ccb];
        if (sum) atomicAdd(acc + (size_t)t * k + c, (unsigned long long)sum);
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) sLast = (atomicAdd(tickets + t, 1u) == gridDim.x - 1) ? 1u : 0u;
    __syncthreads();
    if (!sLast) return;
    __threadfence();
    for (uint32_t c = threadIdx.x; c < k; c += kAuxThreads) {
        unsigned long long sum = __ldcg(acc + (size_t)t * k + c);
        acc[(size_t)t * k + c] = 0;
        uint32_t mu = (mubits[(size_t)t * kb + c / 8] >> (c % 8)) & 1u;
        v[(size_t)t * k + c] = (uint16_t)mod_u64(sum + (unsigned long long)mu * mq.half, mq);
    }
    if (threadIdx.x == 0) tickets[t] = 0;
}

// Fast path for k = 32 * 2^j: a thread owns one 32-bit word of R bits (32 columns) of a row, so a warp
// reads 128 contiguous bytes of bits and writes 32-byte pieces that tile whole 128-byte lines of Rexp
// (HBM-bound: 1 bit in, 1 byte out).  Its 32 column sums sit in registers over all the rows it visits;
// lanes and warps holding the same word column meet in shared memory, CTAs in the u64 global
// accumulators, and the last CTA of the instance (ticket) reduces mod q and writes v.
template <bool kWriteRexp>
__global__ void __launch_bounds__(kAuxThreads)
expand_R_and_v_w32_kernel(const uint16_t *__restrict__ b, const uint8_t *__restrict__ Rbits,
                          const uint8_t *__restrict__ mubits, uint8_t *__restrict__ Rexp, uint16_t *__restrict__ v,
                          unsigned long long *__restrict__ acc, unsigned int *__restrict__ tickets,
                          uint32_t m, uint32_t k, uint32_t ld_exp, ModQ mq)
{
    __shared__ uint32_t sLast;
    extern __shared__ uint32_t sSum[];                        // k column sums of this CTA (<= 65535 * m < 2^32)
    const uint32_t t = blockIdx.y;
    const uint32_t wpr = k / 32;                              // words per row, a power of two <= 64
    const uint32_t w = threadIdx.x & (wpr - 1);               // my word column
    const uint32_t rows_per_iter = kAuxThreads / wpr;
    const uint32_t rslot = threadIdx.x / wpr;
    const uint32_t *Rt = reinterpret_cast<const uint32_t *>(Rbits + (size_t)t * m * (k / 8));
    const uint16_t *bt = b + (size_t)t * m;
    for (uint32_t c = threadIdx.x; c < k; c += kAuxThreads) sSum[c] = 0;
    __syncthreads();

    // Column sums of b_i R_ic in 16-bit lanes, one byte plane of b at a time: register x holds the partial sums of
    // columns x and x + 16 of the thread's 32, sum <= 255 * (rows since the last flush) < 2^16 for <= 256 rows.
    // (r >> x) & 0x00010001 puts the two bits into the two lanes, one IMAD (fma pipe) per byte plane adds the row:
    // 2 instructions per column, against 3.4 for bit-test + predicated add on the alu pipe alone.
    uint32_t aL[16], aH[16];
#pragma unroll
    for (int x = 0; x < 16; x++) { aL[x] = 0; aH[x] = 0; }
    // unpack, add up the lanes of the warp that hold the same word column (lane mod wpr) by shuffle, and let one lane
    // per word column add into the CTA's sums, stored [x][w] so that those lanes hit different banks (32 same-address
    // shared atomics per thread, 4 lanes deep, had made this flush the longest part of the kernel)
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
        if ((threadIdx.x & 31) < wpr || wpr >= 32) {
#pragma unroll
            for (int x = 0; x < 32; x++)
                if (vals[x]) atomicAdd(&sSum[x * wpr + w], vals[x]);
        }
    };
    constexpr int kUnroll = 4;
    constexpr uint32_t kFlushIters = 256 / kUnroll;           // rows per thread between flushes <= 256
    // a CTA streams one contiguous range of rows
    const uint32_t step = rows_per_iter;
    const uint32_t per_cta = ((m + gridDim.x - 1) / gridDim.x + rows_per_iter - 1) / rows_per_iter * rows_per_iter;
    const uint32_t ibeg = blockIdx.x * per_cta, iend = min(m, ibeg + per_cta);
    uint32_t iters = 0;
    for (uint32_t i0 = ibeg + rslot; i0 < iend; i0 += kUnroll * step) {
        uint32_t r[kUnroll], bi[kUnroll];
#pragma unroll
        for (int u = 0; u < kUnroll; u++) {
            const uint32_t i = i0 + u * step;
            r[u] = (i < iend) ? __ldg(Rt + (size_t)i * wpr + w) : 0u;
            bi[u] = (i < iend) ? (uint32_t)__ldg(bt + i) : 0u;
        }
#pragma unroll
        for (int u = 0; u < kUnroll; u++) {
            const uint32_t i = i0 + u * step;
            if (kWriteRexp && i < iend) {
                // bit x of a nibble -> byte x of a word: (nibble * 0x00204081) & 0x01010101
                uint32_t o[8];
#pragma unroll
                for (int h = 0; h < 8; h++) o[h] = (((r[u] >> (4 * h)) & 0xfu) * 0x00204081u) & 0x01010101u;
                uint4 *dst = reinterpret_cast<uint4 *>(Rexp + (size_t)i * ld_exp + (size_t)t * k + 32 * w);
                dst[0] = make_uint4(o[0], o[1], o[2], o[3]);
                dst[1] = make_uint4(o[4], o[5], o[6], o[7]);
            }
            const uint32_t bl = bi[u] & 0xffu, bh = bi[u] >> 8;
#pragma unroll
            for (int x = 0; x < 16; x++) {
                const uint32_t two = (r[u] >> x) & 0x00010001u;     // columns x (low lane) and x + 16 (high lane)
                aL[x] += two * bl;
                aH[x] += two * bh;
            }
        }
        if (++iters == kFlushIters) { flush(); iters = 0; }
    }
    flush();
    __syncthreads();
    for (uint32_t c = threadIdx.x; c < k; c += kAuxThreads) {
        const uint32_t sum = sSum[(c & 31u) * wpr + (c >> 5)];
        if (sum) atomicAdd(acc + (size_t)t * k + c, (unsigned long long)sum);
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) sLast = (atomicAdd(tickets + t, 1u) == gridDim.x - 1) ? 1u : 0u;
    __syncthreads();
    if (!sLast) return;
    __threadfence();
    for (uint32_t c = threadIdx.x; c < k; c += kAuxThreads) {
        unsigned long long sum = __ldcg(acc + (size_t)t * k + c);
        acc[(size_t)t * k + c] = 0;
        uint32_t mu = (mubits[(size_t)t * (k / 8) + c / 8] >> (c % 8)) & 1u;
        v[(size_t)t * k + c] = (uint16_t)mod_u64(sum + (unsigned long long)mu * mq.half, mq);
    }
    if (threadIdx.x == 0) tickets[t] = 0;
}

cudaError_t launch_expand_R_and_v(Ctx *c, const uint16_t *d_b, const uint8_t *d_Rbits, const uint8_t *d_mubits,
                                  uint16_t *d_v, uint32_t batch, bool write_Rexp, cudaStream_t st)
{
    const uint32_t m = c->p.m, k = c->p.k;
    ProfScope prof(c, LWE_K_EXPAND_R_V, st);
    const uint32_t wpr = k / 32;
    if (k % 32 == 0 && (wpr & (wpr - 1)) == 0 && wpr <= 64) {
        const uint32_t rows_per_iter = kAuxThreads / wpr;
        const size_t smem = (size_t)k * sizeof(uint32_t);
        // exactly one wave of resident CTAs (608 CTAs on 296 slots left a third, nearly empty wave)
        int occ = 1;
        cudaError_t perr = write_Rexp ? kernel_prepare(c, expand_R_and_v_w32_kernel<true>, smem, kAuxThreads, &occ)
                                      : kernel_prepare(c, expand_R_and_v_w32_kernel<false>, smem, kAuxThreads, &occ);
        if (perr != cudaSuccess) return perr;
        uint32_t splits = (uint32_t)(occ * c->sm_count) / batch;
        uint32_t max_splits = (m + 4 * rows_per_iter - 1) / (4 * rows_per_iter);   // >= 4 rows per thread
        if (splits > max_splits) splits = max_splits;
        const uint32_t min_splits = (m + 65535u) / 65536u;       // a CTA's 32-bit column sums hold <= 65536 rows
        if (splits < min_splits) splits = min_splits;
        dim3 grid(splits, batch);
        if (write_Rexp)
            expand_R_and_v_w32_kernel<true><<<grid, kAuxThreads, smem, st>>>(
                d_b, d_Rbits, d_mubits, c->d_Rexp, d_v, c->d_vacc, c->d_counters + 8 + c->p.max_batch, m, k, batch * k, c->mq);
        else
            expand_R_and_v_w32_kernel<false><<<grid, kAuxThreads, smem, st>>>(
                d_b, d_Rbits, d_mubits, c->d_Rexp, d_v, c->d_vacc, c->d_counters + 8 + c->p.max_batch, m, k, batch * k, c->mq);
        c->launches++;
        return cudaGetLastError();
    }
    const uint32_t rows_per_iter = kAuxThreads / (k / 8);
    uint32_t splits = (uint32_t)((4 * c->sm_count + batch - 1) / batch);
    uint32_t max_splits = (m + 4 * rows_per_iter - 1) / (4 * rows_per_iter);   // >= 4 row groups per CTA
    if (splits > max_splits) splits = max_splits;
    const uint32_t min_splits = (m + 65535u) / 65536u;           // a thread's 32-bit column sums hold <= 65536 rows
    if (splits < min_splits) splits = min_splits;
    dim3 grid(splits, batch);
    expand_R_and_v_kernel<<<grid, kAuxThreads, 0, st>>>(d_b, d_Rbits, d_mubits, c->d_Rexp, d_v, c->d_vacc,
                                                        c->d_counters + 8 + c->p.max_batch, m, k,
                                                        batch * k, write_Rexp, c->mq);
    c->launches++;
    return cudaGetLastError();
}

// ------------------------------------------------------------------ CUDA-core U = A^T R
// grid (ceil(n/32), k/8, batch), block 32 x 8: thread (x, y) owns U[j = 32*bx + x][8 columns of
// byte by] over the row range y, y+8, ...; the 8 row-slices are summed through shared memory.
// A holds rows [row0, row0 + rows) of the m-row matrix (the whole of it when row0 = 0, rows = m);
// accumulate: add the residues already in U (row panels of a regenerated A, see tc_common.cuh).
__global__ void __launch_bounds__(256)
encaps_simt_kernel(const uint16_t *__restrict__ A, const uint8_t *__restrict__ Rbits, uint16_t *__restrict__ U,
                   uint32_t m, uint32_t n, uint32_t k, uint32_t row0, uint32_t rows, int mode, uint32_t *__restrict__ flags,
                   ModQ mq)
{
    __shared__ uint32_t sAcc[8][32][8];
    const uint32_t t = blockIdx.z, cb = blockIdx.y, kb = k / 8;
    const uint32_t j = blockIdx.x * 32 + threadIdx.x;
    const uint8_t *Rt = Rbits + ((size_t)t * m + row0) * kb;
    uint32_t a[8];
#pragma unroll
    for (int x = 0; x < 8; x++) a[x] = 0;
    if (j < n) {
        for (uint32_t i = threadIdx.y; i < rows; i += 8) {
            uint32_t aij = __ldg(A + (size_t)i * n + j);
            uint32_t r = __ldg(Rt + (size_t)i * kb + cb);
#pragma unroll
            for (int x = 0; x < 8; x++) a[x] += ((r >> x) & 1u) ? aij : 0u;   // <= 65535 * 65536 < 2^32
        }
    }
#pragma unroll
    for (int x = 0; x < 8; x++) sAcc[threadIdx.y][threadIdx.x][x] = a[x];
    __syncthreads();
    if (threadIdx.y == 0 && j < n) {
        uint32_t o[8];
#pragma unroll
        for (int x = 0; x < 8; x++) {
            unsigned long long sum = 0;
            for (int y = 0; y < 8; y++) sum += sAcc[y][threadIdx.x][x];
            o[x] = mod_u64(sum, mq);
        }
        uint4 *dst = reinterpret_cast<uint4 *>(U + ((size_t)t * n + j) * k + 8 * cb);
        if (mode == 2) {                                     // FO re-encryption check: compare, write nothing
            const uint4 p = *dst;
            const uint32_t diff = (p.x ^ (o[0] | (o[1] << 16))) | (p.y ^ (o[2] | (o[3] << 16))) |
                                  (p.z ^ (o[4] | (o[5] << 16))) | (p.w ^ (o[6] | (o[7] << 16)));
            atomicOr(flags + t, diff ? 1u : 0u);
            return;
        }
        if (mode == 1) {
            const uint4 p = *dst;
            const uint32_t old[4] = {p.x, p.y, p.z, p.w};
#pragma unroll
            for (int x = 0; x < 8; x++) {
                uint32_t val = o[x] + ((x & 1) ? (old[x >> 1] >> 16) : (old[x >> 1] & 0xffffu));
                o[x] = val >= mq.q ? val - mq.q : val;
            }
        }
        *dst = make_uint4(o[0] | (o[1] << 16), o[2] | (o[3] << 16), o[4] | (o[5] << 16), o[6] | (o[7] << 16));
    }
}

cudaError_t launch_encaps_simt(Ctx *c, const uint16_t *d_A, const uint8_t *d_Rbits, uint16_t *d_U,
                               uint32_t batch, uint32_t row0, uint32_t rows, int mode, uint32_t *d_flags, cudaStream_t st)
{
    const uint32_t m = c->p.m, n = c->p.n, k = c->p.k;
    dim3 grid((n + 31) / 32, k / 8, batch), block(32, 8);
    ProfScope prof(c, LWE_K_ENCAPS_SIMT, st);
    encaps_simt_kernel<<<grid, block, 0, st>>>(d_A, d_Rbits, d_U, m, n, k, row0, rows, mode, d_flags, c->mq);
    c->launches++;
    return cudaGetLastError();
}

// ------------------------------------------------------------------ N2: the paper's own Encrypt (Gaussian r)
// prep_R_pv_and_v: one pass over the int8 matrix R of every instance that (i) copies it into the GEMM's operand
// buffer laid out [i][t*k + c] (one 256-column tile = one instance, as for the binary R) and (ii) accumulates
// v_c = sum_i t_i R_ic + e2_c + mu_c floor(q/2) mod q (O14; Table 1 header P:L92).
// grid (row_splits, batch); thread = (row slot, 4 columns = one 32-bit word of int8).
__global__ void __launch_bounds__(kAuxThreads)
prep_R_pv_and_v_kernel(const uint16_t *__restrict__ tvec, const int8_t *__restrict__ R, const int8_t *__restrict__ e2,
                       const uint8_t *__restrict__ mubits, uint8_t *__restrict__ Rexp, uint16_t *__restrict__ v,
                       unsigned long long *__restrict__ acc, unsigned int *__restrict__ tickets,
                       uint32_t m, uint32_t k, uint32_t ld_exp, bool write_Rexp, ModQ mq)
{
    __shared__ uint32_t sLast;
    __shared__ unsigned long long sCol[4 * kAuxThreads];
    pdl_trigger();
    pdl_wait();
    const uint32_t t = blockIdx.y;
    const uint32_t wpr = k / 4;                          // words per row (k % 8 == 0)
    const uint32_t rows_per_iter = kAuxThreads / wpr ? kAuxThreads / wpr : 1;
    const uint32_t words_per_thread = (wpr + kAuxThreads - 1) / kAuxThreads;       // > 1 only for k > 1024
    const uint32_t rslot = threadIdx.x / wpr;
    const bool active = rslot < rows_per_iter;
    const int8_t *Rt = R + (size_t)t * m * k;
    const uint16_t *tt = tvec + (size_t)t * m;
    for (uint32_t wq = 0; wq < words_per_thread; wq++) {
        const uint32_t w = (threadIdx.x % wpr) + wq * kAuxThreads;
        long long a[4] = {0, 0, 0, 0};                   // |t_i r| < 2^16 * 2^7, summed over <= 2^20 rows
        if (active && w < wpr) {
            for (uint32_t i = blockIdx.x * rows_per_iter + rslot; i < m; i += gridDim.x * rows_per_iter) {
                const uint32_t r = __ldg(reinterpret_cast<const uint32_t *>(Rt + (size_t)i * k) + w);
                const int ti = (int)__ldg(tt + i);
                if (write_Rexp) *reinterpret_cast<uint32_t *>(Rexp + (size_t)i * ld_exp + (size_t)t * k + 4 * w) = r;
#pragma unroll
                for (int x = 0; x < 4; x++) a[x] += (long long)(ti * (int)(int8_t)(r >> (8 * x)));
            }
        }
        // block-level sum over the row slots, then one atomic per column per CTA (two's complement: u64 adds)
#pragma unroll
        for (int x = 0; x < 4; x++) sCol[x * kAuxThreads + threadIdx.x] = (active && w < wpr) ? (unsigned long long)a[x] : 0ull;
        __syncthreads();
        if (threadIdx.x < wpr && w < wpr) {
#pragma unroll
            for (int x = 0; x < 4; x++) {
                unsigned long long sum = 0;
                for (uint32_t rs = 0; rs < rows_per_iter; rs++) sum += sCol[x * kAuxThreads + rs * wpr + threadIdx.x];
                if (sum) atomicAdd(acc + (size_t)t * k + 4 * w + x, sum);
            }
        }
        __syncthreads();
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) sLast = (atomicAdd(tickets + t, 1u) == gridDim.x - 1) ? 1u : 0u;
    __syncthreads();
    if (!sLast) return;
    __threadfence();
    for (uint32_t c = threadIdx.x; c < k; c += kAuxThreads) {
        const long long sum = (long long)__ldcg(acc + (size_t)t * k + c);
        acc[(size_t)t * k + c] = 0;
        const uint32_t mu = (mubits[(size_t)t * (k / 8) + c / 8] >> (c % 8)) & 1u;
        long long tot = sum + (long long)e2[(size_t)t * k + c] + (long long)mu * mq.half;
        long long r = tot % (long long)mq.q;
        if (r < 0) r += mq.q;
        v[(size_t)t * k + c] = (uint16_t)r;
    }
    if (threadIdx.x == 0) tickets[t] = 0;
}

// v alone (the GEMM reads R in place, nothing to copy): a pure stream over the int8 R of every instance -- 16 columns
// (one 16-byte load) per thread, rows split over the CTAs of an instance, register-pipelined like decaps_kernel (the
// next four rows' loads are issued before the current four are consumed), s32 column sums per thread (|t_i r| < 2^24,
// the host keeps a thread's share below 96 rows), u64 partial sums across CTAs, last CTA of the instance finalizes.
// The one-word-per-thread loop above ran this pass at 0.9 TB/s (73 us for the 64 MB of Table 1's n = 8192 row).
// TT = uint16_t (narrow contexts) or uint32_t (wide contexts): type of t and v.
__device__ __forceinline__ uint4 ldg_stream16_aux(const uint4 *p)
{
    uint4 r;
    asm("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ void pv_row(int (&a)[16], const uint4 &u, int ti)
{
    const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
    for (int y = 0; y < 4; y++)
#pragma unroll
        for (int x = 0; x < 4; x++) a[4 * y + x] += ti * (int)(int8_t)(w[y] >> (8 * x));
}

template <class TT>
__global__ void __launch_bounds__(kAuxThreads)
pv_v_stream_kernel(const TT *__restrict__ tvec, const int8_t *__restrict__ R, const int8_t *__restrict__ e2,
                   const uint8_t *__restrict__ mubits, TT *__restrict__ v, unsigned long long *__restrict__ acc,
                   unsigned int *__restrict__ tickets, uint32_t m, uint32_t k, uint32_t q)
{
    __shared__ uint32_t sLast;
    __shared__ __align__(16) int sCol[kAuxThreads * 16];
    pdl_trigger();
    pdl_wait();
    const uint32_t t = blockIdx.y;
    const uint32_t tpr = k / 16;                         // threads per row: a power of two <= 256 (host)
    const uint32_t rpi = kAuxThreads / tpr;
    const uint32_t rslot = threadIdx.x / tpr, cg = threadIdx.x % tpr;
    const uint4 *Rt = reinterpret_cast<const uint4 *>(R + (size_t)t * m * k);
    const TT *tt = tvec + (size_t)t * m;
    int a[16];
#pragma unroll
    for (int x = 0; x < 16; x++) a[x] = 0;
    {
        constexpr int kUnroll = 4;
        const uint32_t per_cta = ((m + gridDim.x - 1) / gridDim.x + rpi - 1) / rpi * rpi;
        const uint32_t ibeg = blockIdx.x * per_cta, iend = min(m, ibeg + per_cta);
        uint32_t i = ibeg + rslot;
        const uint4 *up = Rt + (size_t)i * tpr + cg;
        const size_t ustep = (size_t)rpi * tpr;
        uint4 u0[kUnroll], u1[kUnroll];
        int t0[kUnroll], t1[kUnroll];
        auto load = [&](uint4 (&uu)[kUnroll], int (&ts)[kUnroll]) {
#pragma unroll
            for (int r = 0; r < kUnroll; r++) {
                const bool in = i + r * rpi < iend;          // a row past the range: a valid address, t = 0
                uu[r] = ldg_stream16_aux(in ? up + r * ustep : Rt + cg);
                ts[r] = in ? (int)__ldg(tt + i + r * rpi) : 0;
            }
            i += kUnroll * rpi;
            up += kUnroll * ustep;
        };
        if (i < iend) {
            load(u0, t0);
            for (;;) {
                const bool more1 = i < iend;
                if (more1) load(u1, t1);
#pragma unroll
                for (int r = 0; r < kUnroll; r++) pv_row(a, u0[r], t0[r]);
                if (!more1) break;
                const bool more0 = i < iend;
                if (more0) load(u0, t0);
#pragma unroll
                for (int r = 0; r < kUnroll; r++) pv_row(a, u1[r], t1[r]);
                if (!more0) break;
            }
        }
    }
    // [row slot][column]: a thread stores its 16 columns contiguously, thread c then reads column c of every slot
#pragma unroll
    for (int x = 0; x < 16; x++) sCol[(size_t)threadIdx.x * 16 + x] = a[x];
    __syncthreads();
    for (uint32_t c = threadIdx.x; c < k; c += kAuxThreads) {
        long long sum = 0;
        for (uint32_t rs = 0; rs < rpi; rs++) sum += (long long)sCol[(size_t)rs * k + c];
        if (sum) atomicAdd(acc + (size_t)t * k + c, (unsigned long long)sum);     // two's complement: u64 adds
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) sLast = (atomicAdd(tickets + t, 1u) == gridDim.x - 1) ? 1u : 0u;
    __syncthreads();
    if (!sLast) return;
    __threadfence();
    for (uint32_t c = threadIdx.x; c < k; c += kAuxThreads) {
        const long long sum = (long long)__ldcg(acc + (size_t)t * k + c);
        acc[(size_t)t * k + c] = 0;
        const uint32_t mu = (mubits[(size_t)t * (k / 8) + c / 8] >> (c % 8)) & 1u;
        long long r = (sum + (long long)e2[(size_t)t * k + c] + (long long)mu * (q / 2)) % (long long)q;
        if (r < 0) r += q;
        v[(size_t)t * k + c] = (TT)r;
    }
    if (threadIdx.x == 0) tickets[t] = 0;
}

bool pv_v_stream_supported(const Ctx *c)
{
    const uint32_t tpr = c->p.k / 16;
    return c->p.k % 16 == 0 && tpr >= 1 && tpr <= (uint32_t)kAuxThreads && (tpr & (tpr - 1)) == 0;
}

template <class TT>
static cudaError_t launch_pv_v_stream_t(Ctx *c, const TT *d_t, const int8_t *d_R, const int8_t *d_e2, const uint8_t *d_mubits,
                                        TT *d_v, uint32_t batch, cudaStream_t st)
{
    const uint32_t m = c->p.m, k = c->p.k;
    const uint32_t rpi = kAuxThreads / (k / 16);
    int per_sm = 1;
    cudaError_t perr = kernel_prepare(c, pv_v_stream_kernel<TT>, 0, kAuxThreads, &per_sm);
    if (perr != cudaSuccess) return perr;
    uint32_t splits = (uint32_t)(per_sm * c->sm_count) / batch;            // one wave of resident CTAs
    const uint32_t max_splits = (m + 4 * rpi - 1) / (4 * rpi);           // >= 4 row groups per CTA
    const uint32_t min_splits = (m + 96 * rpi - 1) / (96 * rpi);         // <= 96 rows per thread: s32 sums cannot overflow
    if (splits > max_splits) splits = max_splits;
    if (splits < min_splits) splits = min_splits;
    if (splits < 1) splits = 1;
    ProfScope prof(c, LWE_K_PREP_R_PV, st);
    return launch_k(c, pv_v_stream_kernel<TT>, dim3(splits, batch), kAuxThreads, 0, st, d_t, d_R, d_e2, d_mubits, d_v, c->d_vacc,
                    c->d_counters + 8 + c->p.max_batch, m, k, c->p.q);
}

cudaError_t launch_pv_v_stream(Ctx *c, const void *d_t, bool wide, const int8_t *d_R, const int8_t *d_e2, const uint8_t *d_mubits,
                               void *d_v, uint32_t batch, cudaStream_t st)
{
    if (wide)
        return launch_pv_v_stream_t<uint32_t>(c, static_cast<const uint32_t *>(d_t), d_R, d_e2, d_mubits,
                                              static_cast<uint32_t *>(d_v), batch, st);
    return launch_pv_v_stream_t<uint16_t>(c, static_cast<const uint16_t *>(d_t), d_R, d_e2, d_mubits,
                                          static_cast<uint16_t *>(d_v), batch, st);
}

cudaError_t launch_prep_R_pv_and_v(Ctx *c, const uint16_t *d_t, const int8_t *d_R, const int8_t *d_e2,
                                   const uint8_t *d_mubits, uint16_t *d_v, uint32_t batch, bool write_Rexp, cudaStream_t st)
{
    if (!write_Rexp && pv_v_stream_supported(c)) return launch_pv_v_stream(c, d_t, false, d_R, d_e2, d_mubits, d_v, batch, st);
    const uint32_t m = c->p.m, k = c->p.k;
    const uint32_t wpr = k / 4;
    const uint32_t rows_per_iter = kAuxThreads / wpr ? kAuxThreads / wpr : 1;
    uint32_t splits = (uint32_t)(4 * c->sm_count) / batch;
    uint32_t max_splits = (m + 4 * rows_per_iter - 1) / (4 * rows_per_iter);
    if (splits > max_splits) splits = max_splits;
    if (splits < 1) splits = 1;
    dim3 grid(splits, batch);
    ProfScope prof(c, LWE_K_PREP_R_PV, st);
    return launch_k(c, prep_R_pv_and_v_kernel, grid, kAuxThreads, 0, st, d_t, d_R, d_e2, d_mubits, c->d_Rexp, d_v, c->d_vacc,
                    c->d_counters + 8 + c->p.max_batch, m, k, batch * k, write_Rexp, c->mq);
}

// CUDA-core U = A^T R + E1 for the int8 R (shapes the tensor path does not take, and its cross-check).
// grid (ceil(n/32), k/8, batch), block 32 x 8 as encaps_simt_kernel.
__global__ void __launch_bounds__(256)
encaps_pv_simt_kernel(const uint16_t *__restrict__ A, const int8_t *__restrict__ R, const int8_t *__restrict__ E1,
                      uint16_t *__restrict__ U, uint32_t m, uint32_t n, uint32_t k, ModQ mq)
{
    __shared__ long long sAcc[8][32][8];
    const uint32_t t = blockIdx.z, cb = blockIdx.y;
    const uint32_t j = blockIdx.x * 32 + threadIdx.x;
    const int8_t *Rt = R + (size_t)t * m * k;
    long long a[8];
#pragma unroll
    for (int x = 0; x < 8; x++) a[x] = 0;
    if (j < n) {
        for (uint32_t i = threadIdx.y; i < m; i += 8) {
            const int aij = (int)__ldg(A + (size_t)i * n + j);
            const uint2 r = __ldg(reinterpret_cast<const uint2 *>(Rt + (size_t)i * k + 8 * cb));
#pragma unroll
            for (int x = 0; x < 4; x++) {
                a[x] += (long long)(aij * (int)(int8_t)(r.x >> (8 * x)));
                a[4 + x] += (long long)(aij * (int)(int8_t)(r.y >> (8 * x)));
            }
        }
    }
#pragma unroll
    for (int x = 0; x < 8; x++) sAcc[threadIdx.y][threadIdx.x][x] = a[x];
    __syncthreads();
    if (threadIdx.y == 0 && j < n) {
        const uint2 e1 = *reinterpret_cast<const uint2 *>(E1 + ((size_t)t * n + j) * k + 8 * cb);
        uint32_t o[8];
#pragma unroll
        for (int x = 0; x < 8; x++) {
            long long sum = (long long)(int8_t)((x < 4 ? e1.x : e1.y) >> (8 * (x & 3)));
            for (int y = 0; y < 8; y++) sum += sAcc[y][threadIdx.x][x];
            long long r = sum % (long long)mq.q;
            o[x] = (uint32_t)(r < 0 ? r + mq.q : r);
        }
        *reinterpret_cast<uint4 *>(U + ((size_t)t * n + j) * k + 8 * cb) =
            make_uint4(o[0] | (o[1] << 16), o[2] | (o[3] << 16), o[4] | (o[5] << 16), o[6] | (o[7] << 16));
    }
}

cudaError_t launch_encaps_pv_simt(Ctx *c, const uint16_t *d_A, const int8_t *d_R, const int8_t *d_E1, uint16_t *d_U,
                                  uint32_t batch, cudaStream_t st)
{
    const uint32_t m = c->p.m, n = c->p.n, k = c->p.k;
    dim3 grid((n + 31) / 32, k / 8, batch), block(32, 8);
    ProfScope prof(c, LWE_K_ENCAPS_SIMT, st);
    encaps_pv_simt_kernel<<<grid, block, 0, st>>>(d_A, d_R, d_E1, d_U, m, n, k, c->mq);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace lwe

// wide.cu -- the paper's PKE on Table 1's q = 65537 rows (n >= 8192): residues need 17 bits and cross the
// boundary as uint32 ("32-bit integers"); s, e, R, E1, e2 are small signed integers (int8).  Readings S23-S25
// of DESIGN.md section 3.
//
// How a 17-bit A reaches the 8-bit tensor pipe.  lwe_wide_load_matrix packs the public matrix once: the low 16 bits of
// every element into a uint16 matrix A16 -- which the tcgen05 kernels then read exactly like a narrow A (two byte
// planes, consumed in place) -- and the elements >= 2^16 into exception lists.  For q = 2^16 + delta only delta of
// the q residues have bit 16 set (q = 65537: the single value 65536, i.e. about m n / 65537 elements of a uniform
// A: 1024 at n = 8192), so a third byte plane would be a dense GEMM pass over an almost empty matrix; instead the
// epilogues add  2^16 * sum_{exceptions of this row / column} (small operand)  from a per-row (KeyGen) or per-column
// (Encrypt) slot list.  The lists have a fixed capacity sized from (m, n, q) for a uniform A with a wide margin; a
// matrix that does not fit is refused at load time (LWE_ERR_UNSUPPORTED), never computed wrongly.
//
// This file: the pack kernel, the CUDA-core KeyGen / Encrypt (cross-checks of the tensor kernels and the path for
// shapes those do not take), v = t^T R + e2 + mu floor(q/2), and Decrypt on uint32 residues.
#include "lwe_internal.cuh"

namespace lwe {

namespace {

constexpr int kThreads = 256;

__device__ __forceinline__ uint32_t mod_s64(long long x, uint32_t q)
{
    long long r = x % (long long)q;                      // once per output element: not on any inner loop
    return (uint32_t)(r < 0 ? r + (long long)q : r);
}

// ------------------------------------------------------------------ pack
// rows [row0, row0 + rows) of A (the panel holds exactly those rows): A16 = low halves; elements >= 2^16 are
// appended to the slot lists of their column and of their row.  One thread per 4 elements (a 16-byte load).
__global__ void __launch_bounds__(kThreads)
wide_pack_kernel(const uint32_t *__restrict__ A, uint16_t *__restrict__ A16, uint32_t row0, uint32_t rows, uint32_t n,
                 uint32_t *__restrict__ col_cnt, uint32_t *__restrict__ col_rows, uint32_t cap_col,
                 uint32_t *__restrict__ row_cnt, uint32_t *__restrict__ row_cols, uint32_t cap_row,
                 uint32_t *__restrict__ overflow, uint32_t q)
{
    const uint64_t quads = (uint64_t)rows * (n / 4);
    for (uint64_t g = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; g < quads; g += (uint64_t)gridDim.x * blockDim.x) {
        const uint4 a = __ldg(reinterpret_cast<const uint4 *>(A) + g);
        const uint32_t i = row0 + (uint32_t)(g / (n / 4)), j0 = 4 * (uint32_t)(g % (n / 4));
        reinterpret_cast<uint2 *>(A16)[(uint64_t)i * (n / 4) + j0 / 4] =
            make_uint2((a.x & 0xffffu) | (a.y << 16), (a.z & 0xffffu) | (a.w << 16));
        if ((a.x | a.y | a.z | a.w) >> 16) {
            const uint32_t w[4] = {a.x, a.y, a.z, a.w};
#pragma unroll
            for (int x = 0; x < 4; x++) {
                if (w[x] >= q) atomicOr(overflow, 2u);       // not a residue: refused (LWE_ERR_PARAM)
                if (w[x] >> 16) {
                    const uint32_t j = j0 + x;
                    const uint32_t sc = atomicAdd(col_cnt + j, 1u), sr = atomicAdd(row_cnt + i, 1u);
                    if (sc < cap_col) col_rows[(size_t)j * cap_col + sc] = i; else atomicOr(overflow, 1u);
                    if (sr < cap_row) row_cols[(size_t)i * cap_row + sr] = j; else atomicOr(overflow, 1u);
                }
            }
        }
    }
}

// ------------------------------------------------------------------ KeyGen on CUDA cores (one warp per row)
// t[b][i] = (sum_j A[i][j] s[b][j] + e[b][i]) mod q,  A[i][j] = A16[i][j] + 2^16 [j in exceptions of row i].
// Any n; the cross-check of the tensor-core kernel (LWE_OPT_KEYGEN_PATH = 1) and the path for shapes it does not take; 16-byte loads of A16 (8 elements)
// against 8 secrets, products accumulated in 32 bits (|a s| < 2^23) and flushed into 64 bits every 128 steps.
__global__ void __launch_bounds__(kThreads)
wide_keygen_simt_kernel(const uint16_t *__restrict__ A16, const uint32_t *__restrict__ row_cnt,
                        const uint32_t *__restrict__ row_cols, uint32_t cap_row, const int8_t *__restrict__ s,
                        const int8_t *__restrict__ e, uint32_t *__restrict__ t, uint32_t m, uint32_t n, uint32_t batch,
                        uint32_t q)
{
    const uint32_t lane = threadIdx.x & 31, warps = (gridDim.x * blockDim.x) >> 5;
    const uint32_t chunks = n / 8;
    for (uint32_t i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; i < m; i += warps) {
        const uint4 *Arow = reinterpret_cast<const uint4 *>(A16 + (size_t)i * n);
        for (uint32_t b = 0; b < batch; b++) {
            const int8_t *sb = s + (size_t)b * n;
            const uint2 *sb8 = reinterpret_cast<const uint2 *>(sb);
            long long acc = 0;
            int part = 0;
            uint32_t since = 0;
            for (uint32_t c = lane; c < chunks; c += 32) {
                const uint4 a = __ldg(Arow + c);
                const uint2 sv = __ldg(sb8 + c);
                const uint32_t aw[4] = {a.x, a.y, a.z, a.w}, sw[2] = {sv.x, sv.y};
#pragma unroll
                for (int x = 0; x < 8; x++) {
                    const int av = (int)((aw[x >> 1] >> (16 * (x & 1))) & 0xffffu);
                    part += av * (int)(int8_t)(sw[x >> 2] >> (8 * (x & 3)));
                }
                if (++since == 16) { acc += part; part = 0; since = 0; }    // 128 products of < 2^23 each
            }
            acc += part;
            const uint32_t cnt = min(row_cnt[i], cap_row);
            for (uint32_t x = lane; x < cnt; x += 32) acc += 65536ll * (int)sb[row_cols[(size_t)i * cap_row + x]];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
            if (lane == 0) t[(size_t)b * m + i] = mod_s64(acc + (int)e[(size_t)b * m + i], q);
        }
    }
}

// ------------------------------------------------------------------ v = t^T R + e2 + mu floor(q/2)  (+ operand copy)
// The uint32-t counterpart of prep_R_pv_and_v_kernel (encaps_aux.cu): grid (row_splits, batch); thread = (row slot,
// 4 columns = one 32-bit word of int8 R).  write_Rexp: also copy R into the GEMM's operand layout [i][b*k + c]
// (only for k % 128 != 0; otherwise the GEMM reads R in place).
__global__ void __launch_bounds__(kThreads)
wide_v_kernel(const uint32_t *__restrict__ tvec, const int8_t *__restrict__ R, const int8_t *__restrict__ e2,
              const uint8_t *__restrict__ mubits, uint8_t *__restrict__ Rexp, uint32_t *__restrict__ v,
              unsigned long long *__restrict__ acc, unsigned int *__restrict__ tickets, uint32_t m, uint32_t k,
              uint32_t ld_exp, bool write_Rexp, uint32_t q)
{
    __shared__ uint32_t sLast;
    __shared__ unsigned long long sCol[4 * kThreads];
    pdl_trigger();
    pdl_wait();
    const uint32_t b = blockIdx.y;
    const uint32_t wpr = k / 4;
    const uint32_t rows_per_iter = kThreads / wpr ? kThreads / wpr : 1;
    const uint32_t words_per_thread = (wpr + kThreads - 1) / kThreads;
    const uint32_t rslot = threadIdx.x / wpr;
    const bool active = rslot < rows_per_iter;
    const int8_t *Rb = R + (size_t)b * m * k;
    const uint32_t *tb = tvec + (size_t)b * m;
    for (uint32_t wq = 0; wq < words_per_thread; wq++) {
        const uint32_t w = (threadIdx.x % wpr) + wq * kThreads;
        long long a[4] = {0, 0, 0, 0};                   // |t_i r| < 2^17 * 2^7, summed over <= 2^20 rows
        if (active && w < wpr) {
            for (uint32_t i = blockIdx.x * rows_per_iter + rslot; i < m; i += gridDim.x * rows_per_iter) {
                const uint32_t r = __ldg(reinterpret_cast<const uint32_t *>(Rb + (size_t)i * k) + w);
                const int ti = (int)__ldg(tb + i);
                if (write_Rexp) *reinterpret_cast<uint32_t *>(Rexp + (size_t)i * ld_exp + (size_t)b * k + 4 * w) = r;
#pragma unroll
                for (int x = 0; x < 4; x++) a[x] += (long long)(ti * (int)(int8_t)(r >> (8 * x)));
            }
        }
#pragma unroll
        for (int x = 0; x < 4; x++) sCol[x * kThreads + threadIdx.x] = (active && w < wpr) ? (unsigned long long)a[x] : 0ull;
        __syncthreads();
        if (threadIdx.x < wpr && w < wpr) {
#pragma unroll
            for (int x = 0; x < 4; x++) {
                unsigned long long sum = 0;
                for (uint32_t rs = 0; rs < rows_per_iter; rs++) sum += sCol[x * kThreads + rs * wpr + threadIdx.x];
                if (sum) atomicAdd(acc + (size_t)b * k + 4 * w + x, sum);
            }
        }
        __syncthreads();
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) sLast = (atomicAdd(tickets + b, 1u) == gridDim.x - 1) ? 1u : 0u;
    __syncthreads();
    if (!sLast) return;
    __threadfence();
    for (uint32_t c = threadIdx.x; c < k; c += kThreads) {
        const long long sum = (long long)__ldcg(acc + (size_t)b * k + c);
        acc[(size_t)b * k + c] = 0;
        const uint32_t mu = (mubits[(size_t)b * (k / 8) + c / 8] >> (c % 8)) & 1u;
        v[(size_t)b * k + c] = mod_s64(sum + (long long)e2[(size_t)b * k + c] + (long long)mu * (q / 2), q);
    }
    if (threadIdx.x == 0) tickets[b] = 0;
}

// ------------------------------------------------------------------ Encrypt on CUDA cores
// U[b][j][c] = (sum_i A[i][j] R_b[i][c] + E1_b[j][c]) mod q.  grid (ceil(n/32), k/8, batch), block 32 x 8 as
// encaps_pv_simt_kernel; the exceptions of column j add 2^16 R_b[i][c].
__global__ void __launch_bounds__(256)
wide_encaps_simt_kernel(const uint16_t *__restrict__ A16, const uint32_t *__restrict__ col_cnt,
                        const uint32_t *__restrict__ col_rows, uint32_t cap_col, const int8_t *__restrict__ R,
                        const int8_t *__restrict__ E1, uint32_t *__restrict__ U, uint32_t m, uint32_t n, uint32_t k,
                        uint32_t q)
{
    __shared__ long long sAcc[8][32][8];
    const uint32_t b = blockIdx.z, cb = blockIdx.y;
    const uint32_t j = blockIdx.x * 32 + threadIdx.x;
    const int8_t *Rb = R + (size_t)b * m * k;
    long long a[8];
#pragma unroll
    for (int x = 0; x < 8; x++) a[x] = 0;
    if (j < n) {
        for (uint32_t i = threadIdx.y; i < m; i += 8) {
            const int aij = (int)__ldg(A16 + (size_t)i * n + j);
            const uint2 r = __ldg(reinterpret_cast<const uint2 *>(Rb + (size_t)i * k + 8 * cb));
#pragma unroll
            for (int x = 0; x < 4; x++) {
                a[x] += (long long)(aij * (int)(int8_t)(r.x >> (8 * x)));
                a[4 + x] += (long long)(aij * (int)(int8_t)(r.y >> (8 * x)));
            }
        }
        const uint32_t cnt = min(col_cnt[j], cap_col);
        for (uint32_t x0 = threadIdx.y; x0 < cnt; x0 += 8) {
            const uint32_t i = col_rows[(size_t)j * cap_col + x0];
            const uint2 r = __ldg(reinterpret_cast<const uint2 *>(Rb + (size_t)i * k + 8 * cb));
#pragma unroll
            for (int x = 0; x < 4; x++) {
                a[x] += 65536ll * (int)(int8_t)(r.x >> (8 * x));
                a[4 + x] += 65536ll * (int)(int8_t)(r.y >> (8 * x));
            }
        }
    }
#pragma unroll
    for (int x = 0; x < 8; x++) sAcc[threadIdx.y][threadIdx.x][x] = a[x];
    __syncthreads();
    if (threadIdx.y == 0 && j < n) {
        const uint2 e1 = *reinterpret_cast<const uint2 *>(E1 + ((size_t)b * n + j) * k + 8 * cb);
        uint32_t o[8];
#pragma unroll
        for (int x = 0; x < 8; x++) {
            long long sum = (long long)(int8_t)((x < 4 ? e1.x : e1.y) >> (8 * (x & 3)));
            for (int y = 0; y < 8; y++) sum += sAcc[y][threadIdx.x][x];
            o[x] = mod_s64(sum, q);
        }
        uint4 *dst = reinterpret_cast<uint4 *>(U + ((size_t)b * n + j) * k + 8 * cb);
        dst[0] = make_uint4(o[0], o[1], o[2], o[3]);
        dst[1] = make_uint4(o[4], o[5], o[6], o[7]);
    }
}

// ------------------------------------------------------------------ Decrypt
// d_c = (v_c - sum_j U[j][c] s_j) mod q, rounded to a bit.  The structure of decaps_kernel (decaps.cu) on uint32
// residues: a thread owns 4 columns (16 bytes) of a row, k/4 threads per row, rows split over the CTAs of an
// instance, u64 (two's complement) global partial sums, the last CTA of the instance rounds and packs.
// HBM-bound: 4 n k bytes of U per instance.
__device__ __forceinline__ uint4 ldg_stream16(const uint4 *p)
{
    uint4 r;
    asm("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

__global__ void __launch_bounds__(kThreads)
wide_decaps_kernel(const uint32_t *__restrict__ U, const uint32_t *__restrict__ v, const int8_t *__restrict__ s,
                   uint8_t *__restrict__ out, unsigned long long *__restrict__ acc, unsigned int *__restrict__ tickets,
                   uint32_t n, uint32_t k, uint32_t q)
{
    __shared__ uint32_t sLast;
    __shared__ long long sCol[kThreads * 4];
    pdl_trigger();
    pdl_wait();
    const uint32_t b = blockIdx.y;
    const uint32_t tpr = k / 4;                          // threads per row (k <= 1024 on this path)
    const uint32_t rows_per_iter = kThreads / tpr;
    const uint32_t rslot = threadIdx.x / tpr, cg = threadIdx.x % tpr;
    const bool active = rslot < rows_per_iter;
    const uint32_t *Ub = U + (size_t)b * n * k;
    const int8_t *sb = s + (size_t)b * n;
    long long a[4] = {0, 0, 0, 0};
    if (active) {
        constexpr int kUnroll = 4;
        const uint32_t per_cta = ((n + gridDim.x - 1) / gridDim.x + rows_per_iter - 1) / rows_per_iter * rows_per_iter;
        const uint32_t jbeg = blockIdx.x * per_cta, jend = min(n, jbeg + per_cta);
        uint32_t j = jbeg + rslot;
        const uint4 *up = reinterpret_cast<const uint4 *>(Ub) + (size_t)j * tpr + cg;
        const size_t ustep = (size_t)rows_per_iter * tpr;
        // products < 2^17 * 2^7 = 2^24: a 32-bit partial holds 128 rows; flushed into 64 bits every 120 rows.
        // Register-pipelined as decaps_kernel: the loads of the next four rows are issued before the current four are
        // consumed; a row past the end of the range re-reads a valid address with s = 0 (no tail of single loads).
        int p[4] = {0, 0, 0, 0};
        uint32_t since = 0;
        uint4 u0[kUnroll], u1[kUnroll];
        int s0[kUnroll], s1[kUnroll];
        auto load = [&](uint4 (&uu)[kUnroll], int (&ss)[kUnroll]) {
#pragma unroll
            for (int r = 0; r < kUnroll; r++) {
                const bool in = j + r * rows_per_iter < jend;
                uu[r] = ldg_stream16(in ? up + r * ustep : reinterpret_cast<const uint4 *>(Ub) + cg);
                ss[r] = in ? (int)__ldg(sb + j + r * rows_per_iter) : 0;
            }
            j += kUnroll * rows_per_iter;
            up += kUnroll * ustep;
        };
        auto consume = [&](const uint4 (&uu)[kUnroll], const int (&ss)[kUnroll]) {
#pragma unroll
            for (int r = 0; r < kUnroll; r++) {
                p[0] += (int)uu[r].x * ss[r]; p[1] += (int)uu[r].y * ss[r];
                p[2] += (int)uu[r].z * ss[r]; p[3] += (int)uu[r].w * ss[r];
            }
            since += kUnroll;
            if (since >= 120) {
#pragma unroll
                for (int x = 0; x < 4; x++) { a[x] += p[x]; p[x] = 0; }
                since = 0;
            }
        };
        if (j < jend) {
            load(u0, s0);
            for (;;) {
                const bool more1 = j < jend;
                if (more1) load(u1, s1);
                consume(u0, s0);
                if (!more1) break;
                const bool more0 = j < jend;
                if (more0) load(u0, s0);
                consume(u1, s1);
                if (!more0) break;
            }
        }
#pragma unroll
        for (int x = 0; x < 4; x++) a[x] += p[x];
    }
#pragma unroll
    for (int x = 0; x < 4; x++) sCol[x * kThreads + threadIdx.x] = a[x];
    __syncthreads();
    for (uint32_t c = threadIdx.x; c < k; c += kThreads) {
        const uint32_t ccg = c >> 2, x = c & 3;
        long long sum = 0;
        for (uint32_t rs = 0; rs < rows_per_iter; rs++) sum += sCol[x * kThreads + rs * tpr + ccg];
        if (sum) atomicAdd(acc + (size_t)b * k + c, (unsigned long long)sum);
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) sLast = (atomicAdd(tickets + b, 1u) == gridDim.x - 1) ? 1u : 0u;
    __syncthreads();
    if (!sLast) return;
    __threadfence();
    for (uint32_t c0 = 0; c0 < k; c0 += kThreads) {
        const uint32_t c = c0 + threadIdx.x;
        uint32_t bit = 0;
        if (c < k) {
            const long long sum = (long long)__ldcg(acc + (size_t)b * k + c);
            acc[(size_t)b * k + c] = 0;
            const uint32_t d = mod_s64((long long)v[(size_t)b * k + c] - sum, q);
            bit = (uint32_t)(((4ull * d + q) / (2ull * q)) & 1ull);
        }
        const uint32_t word = __ballot_sync(0xffffffffu, bit);
        if ((threadIdx.x & 31) == 0) {
            const uint32_t cw = c0 + (threadIdx.x & ~31u);
            for (uint32_t by = 0; by < 4 && cw + 8 * by < k; by++)
                out[(size_t)b * (k / 8) + cw / 8 + by] = (uint8_t)(word >> (8 * by));
        }
    }
    if (threadIdx.x == 0) tickets[b] = 0;
}

}  // namespace

cudaError_t launch_wide_pack(Ctx *c, const uint32_t *d_A, uint32_t row0, uint32_t rows, cudaStream_t st)
{
    const uint64_t quads = (uint64_t)rows * (c->p.n / 4);
    uint64_t blocks = (quads + kThreads - 1) / kThreads;
    const uint64_t cap = (uint64_t)c->sm_count * 16;
    if (blocks > cap) blocks = cap;
    ProfScope prof(c, LWE_K_WIDE_PACK, st);
    wide_pack_kernel<<<(uint32_t)(blocks ? blocks : 1), kThreads, 0, st>>>(
        d_A, c->d_A16, row0, rows, c->p.n, c->d_exc_col_cnt, c->d_exc_col_rows, c->exc_cap_col, c->d_exc_row_cnt,
        c->d_exc_row_cols, c->exc_cap_row, c->d_exc_overflow, c->p.q);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_wide_keygen_simt(Ctx *c, const int8_t *d_s, const int8_t *d_e, uint32_t *d_t, uint32_t batch, cudaStream_t st)
{
    const uint32_t m = c->p.m;
    uint32_t blocks = (m + kThreads / 32 - 1) / (kThreads / 32);
    const uint32_t cap = (uint32_t)c->sm_count * 8;
    if (blocks > cap) blocks = cap;
    ProfScope prof(c, LWE_K_WIDE_KEYGEN, st);
    wide_keygen_simt_kernel<<<blocks, kThreads, 0, st>>>(c->d_A16, c->d_exc_row_cnt, c->d_exc_row_cols, c->exc_cap_row, d_s,
                                                         d_e, d_t, m, c->p.n, batch, c->p.q);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_wide_v(Ctx *c, const uint32_t *d_t, const int8_t *d_R, const int8_t *d_e2, const uint8_t *d_mubits,
                          uint32_t *d_v, uint32_t batch, bool write_Rexp, cudaStream_t st)
{
    if (!write_Rexp && pv_v_stream_supported(c)) return launch_pv_v_stream(c, d_t, true, d_R, d_e2, d_mubits, d_v, batch, st);
    const uint32_t m = c->p.m, k = c->p.k;
    const uint32_t wpr = k / 4;
    const uint32_t rows_per_iter = kThreads / wpr ? kThreads / wpr : 1;
    uint32_t splits = (uint32_t)(4 * c->sm_count) / batch;
    uint32_t max_splits = (m + 4 * rows_per_iter - 1) / (4 * rows_per_iter);
    if (splits > max_splits) splits = max_splits;
    if (splits < 1) splits = 1;
    dim3 grid(splits, batch);
    ProfScope prof(c, LWE_K_PREP_R_PV, st);
    return launch_k(c, wide_v_kernel, grid, kThreads, 0, st, d_t, d_R, d_e2, d_mubits, c->d_Rexp, d_v, c->d_vacc,
                    c->d_counters + 8 + c->p.max_batch, m, k, batch * k, write_Rexp, c->p.q);
}

cudaError_t launch_wide_encaps_simt(Ctx *c, const int8_t *d_R, const int8_t *d_E1, uint32_t *d_U, uint32_t batch, cudaStream_t st)
{
    const uint32_t m = c->p.m, n = c->p.n, k = c->p.k;
    dim3 grid((n + 31) / 32, k / 8, batch), block(32, 8);
    ProfScope prof(c, LWE_K_ENCAPS_SIMT, st);
    wide_encaps_simt_kernel<<<grid, block, 0, st>>>(c->d_A16, c->d_exc_col_cnt, c->d_exc_col_rows, c->exc_cap_col, d_R, d_E1,
                                                    d_U, m, n, k, c->p.q);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_wide_decaps(Ctx *c, const uint32_t *d_U, const uint32_t *d_v, const int8_t *d_s, uint8_t *d_out,
                               uint32_t batch, cudaStream_t st)
{
    const uint32_t n = c->p.n, k = c->p.k;
    const uint32_t rows_per_iter = kThreads / (k / 4);
    int per_sm = 1;
    cudaError_t perr = kernel_prepare(c, wide_decaps_kernel, 0, kThreads, &per_sm);
    if (perr != cudaSuccess) return perr;
    uint32_t splits = (uint32_t)(per_sm * c->sm_count) / batch;
    uint32_t max_splits = (n + 4 * rows_per_iter - 1) / (4 * rows_per_iter);
    if (splits > max_splits) splits = max_splits;
    if (splits < 1) splits = 1;
    dim3 grid(splits, batch);
    ProfScope prof(c, LWE_K_DECAPS, st);
    return launch_k(c, wide_decaps_kernel, grid, kThreads, 0, st, d_U, d_v, d_s, d_out, c->d_dacc, c->d_counters + 8, n, k,
                    c->p.q);
}

}  // namespace lwe

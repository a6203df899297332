// Block-CG linear algebra kernels:
//   Gram products  G = U^H W             ("ThinQR" 12x12x1M shape of Table 6)
//   block rotations W = beta V + U K
//   s x s algebra in complex128: Cholesky, triangular / HPD inverse, products, stop scalar.
// Reductions are deterministic: fixed partition of rows over CTAs, fixed summation order, no float atomics.
#pragma once

#include <type_traits>

#include "common.cuh"
#include "ptx_async.cuh"
#include "tcgen05_ptx.cuh"

namespace cmrhs {

constexpr int kLaThreads = 256;

// ------------------------------------------------------------------------------------------------------
// Gram product, stage 1: each CTA reduces a contiguous chunk of rows to one s x s partial (double).
// Thread layout: the s x s result is cut into TT x TT sub-blocks (one per thread "tile"); the 256 threads
// are (row group) x (tile).  Products and short runs in T, flushed to double every row tile.
// ------------------------------------------------------------------------------------------------------
template <typename T, int TT, int S = 0>
__global__ void __launch_bounds__(kLaThreads)
gram_partial_kernel(const cplx<T> *__restrict__ U, const cplx<T> *__restrict__ W, int64_t n, int s_rt, int rows_per_tile,
                    zdouble *__restrict__ partial)
{
    const int s = S ? S : s_rt;              // S > 0: compile-time block width (a multiple of TT): no column guards
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx<T> *sU = reinterpret_cast<cplx<T> *>(smem_raw);
    cplx<T> *sW = sU + (size_t)rows_per_tile * s;
    const int nt = (s + TT - 1) / TT;          // tiles per dimension
    const int ntile = nt * nt;
    const int RG = kLaThreads / ntile;         // row groups (>= 1 because nt <= 16)
    const int tile = threadIdx.x % ntile, rg = threadIdx.x / ntile;
    const bool active = rg < RG;
    const int a0 = (tile / nt) * TT, b0 = (tile % nt) * TT;

    const int64_t chunk = (n + gridDim.x - 1) / gridDim.x;
    const int64_t r_begin = blockIdx.x * chunk;
    const int64_t r_end = (r_begin + chunk < n) ? r_begin + chunk : n;

    double accr[TT][TT], acci[TT][TT];
#pragma unroll
    for (int a = 0; a < TT; ++a)
#pragma unroll
        for (int b = 0; b < TT; ++b) { accr[a][b] = 0.0; acci[a][b] = 0.0; }

    for (int64_t r0 = r_begin; r0 < r_end; r0 += rows_per_tile) {
        const int nrow = (int)((r_end - r0 < rows_per_tile) ? (r_end - r0) : rows_per_tile);
        const cplx<T> *gu = U + r0 * s, *gw = W + r0 * s;
        for (int e = threadIdx.x; e < nrow * s; e += kLaThreads) { sU[e] = gu[e]; sW[e] = gw[e]; }
        __syncthreads();
        if (active) {
            cplx<T> run[TT][TT];
#pragma unroll
            for (int a = 0; a < TT; ++a)
#pragma unroll
                for (int b = 0; b < TT; ++b) { run[a][b].re = 0; run[a][b].im = 0; }
            for (int k = rg; k < nrow; k += RG) {
                cplx<T> u[TT], w[TT];
#pragma unroll
                for (int a = 0; a < TT; ++a) {
                    const bool ok = S || a0 + a < s;
                    u[a] = ok ? sU[k * s + a0 + a] : cplx<T>{0, 0};
                }
#pragma unroll
                for (int b = 0; b < TT; ++b) {
                    const bool ok = S || b0 + b < s;
                    w[b] = ok ? sW[k * s + b0 + b] : cplx<T>{0, 0};
                }
#pragma unroll
                for (int a = 0; a < TT; ++a)
#pragma unroll
                    for (int b = 0; b < TT; ++b) cmac_conj(run[a][b], u[a], w[b]);
            }
#pragma unroll
            for (int a = 0; a < TT; ++a)
#pragma unroll
                for (int b = 0; b < TT; ++b) { accr[a][b] += (double)run[a][b].re; acci[a][b] += (double)run[a][b].im; }
        }
        __syncthreads();
    }

    // reduce the row groups in a fixed order (group 0, 1, 2, ...) through shared memory; the staging buffer is
    // reused as s*s complex doubles (it is only needed when RG > 1, i.e. for small s)
    zdouble *out = partial + (size_t)blockIdx.x * s * s;
    if (RG == 1) {
        if (active) {
#pragma unroll
            for (int a = 0; a < TT; ++a)
#pragma unroll
                for (int b = 0; b < TT; ++b)
                    if (a0 + a < s && b0 + b < s) out[(a0 + a) * s + b0 + b] = {accr[a][b], acci[a][b]};
        }
        return;
    }
    double *red = reinterpret_cast<double *>(smem_raw);
    for (int g = 0; g < RG; ++g) {
        if (active && rg == g) {
#pragma unroll
            for (int a = 0; a < TT; ++a)
#pragma unroll
                for (int b = 0; b < TT; ++b)
                    if (a0 + a < s && b0 + b < s) {
                        const int e = (a0 + a) * s + b0 + b;
                        if (g == 0) { red[2 * e] = accr[a][b]; red[2 * e + 1] = acci[a][b]; }
                        else { red[2 * e] += accr[a][b]; red[2 * e + 1] += acci[a][b]; }
                    }
        }
        __syncthreads();
    }
    for (int e = threadIdx.x; e < s * s; e += kLaThreads) { out[e].re = red[2 * e]; out[e].im = red[2 * e + 1]; }
}

// ------------------------------------------------------------------------------------------------------
// Gram product, stage 1, PIPELINED form for the widths block CG runs at in complex64 (S = 16, 32 at compile time).
// gram_partial_kernel above stages a tile with per-thread loads and then works on it: with 5 CTAs per SM that keeps ~20 KB
// per SM in flight and measured 129 us at the headline shape (1.33 M rows x 16: 340 MB, 51 us at the HBM roof).  Here a tile of
// consecutive rows -- ONE contiguous range of the [n][S] block -- arrives by a bulk copy per operand into a ring of
// kGramPipeStages stages (one elected thread issues, an mbarrier per stage counts the bytes), 2 CTAs per SM, 4 x 4 sub-blocks
// per thread (two 16-byte shared-memory loads per operand and row for 16 complex multiply-adds).  Same arithmetic contract as
// above: products and runs of <= 36 rows in T, flushed to double; fixed partition and order (deterministic).
// ------------------------------------------------------------------------------------------------------
constexpr int kGramPipeStages = 3;

template <typename T, int TT>
__device__ __forceinline__ void gram_pipe_load(cplx<T> (&v)[TT], const cplx<T> *p)
{
    if constexpr (sizeof(T) == 4 && TT % 2 == 0) {
#pragma unroll
        for (int i = 0; i < TT / 2; ++i) {
            const float4 q = reinterpret_cast<const float4 *>(p)[i];
            v[2 * i] = {q.x, q.y};
            v[2 * i + 1] = {q.z, q.w};
        }
    } else {
#pragma unroll
        for (int i = 0; i < TT; ++i) v[i] = p[i];
    }
}

template <typename T, int TT, int S>
__global__ void __launch_bounds__(kLaThreads, 2)
gram_pipe_kernel(const cplx<T> *__restrict__ U, const cplx<T> *__restrict__ W, int64_t n, int rows, int flush_tiles, zdouble *__restrict__ partial)
{
    constexpr int NT = S / TT, NTILE = NT * NT, RG = kLaThreads / NTILE;
    static_assert(S % TT == 0 && kLaThreads % NTILE == 0 && (S * sizeof(cplx<T>)) % 16 == 0, "gram_pipe tiling");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const size_t tile_bytes = (size_t)rows * S * sizeof(cplx<T>);            // one operand's tile; a stage = [U tile | W tile]
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + (size_t)kGramPipeStages * 2 * tile_bytes);
    const int tile = threadIdx.x % NTILE, rg = threadIdx.x / NTILE;
    const int a0 = (tile / NT) * TT, b0 = (tile % NT) * TT;

    const int64_t chunk = (n + gridDim.x - 1) / gridDim.x;
    const int64_t r_begin = blockIdx.x * chunk;
    const int64_t r_end = (r_begin + chunk < n) ? r_begin + chunk : n;
    const int64_t ntiles = r_end > r_begin ? (r_end - r_begin + rows - 1) / rows : 0;
    if (threadIdx.x == 0) {
        for (int st = 0; st < kGramPipeStages; ++st) mbar_init(&full[st], 1);
        mbar_fence_init();
    }
    __syncthreads();
    uint64_t pol = 0;
    if (threadIdx.x == 0) pol = l2_policy_evict_first();
    auto issue = [&](int64_t t) {                 // thread 0 only
        const int st = (int)(t % kGramPipeStages);
        const int64_t r0 = r_begin + t * rows;
        const uint32_t bytes = (uint32_t)(((r_end - r0 < rows) ? (r_end - r0) : rows) * S * sizeof(cplx<T>));
        unsigned char *dst = smem_raw + (size_t)st * 2 * tile_bytes;
        mbar_arrive_expect_tx(&full[st], 2u * bytes);
        bulk_g2s(dst, U + r0 * S, bytes, &full[st], pol);
        bulk_g2s(dst + tile_bytes, W + r0 * S, bytes, &full[st], pol);
    };
    if (threadIdx.x == 0)
        for (int64_t t = 0; t < kGramPipeStages - 1 && t < ntiles; ++t) issue(t);

    double accr[TT][TT], acci[TT][TT];
    cplx<T> run[TT][TT];
#pragma unroll
    for (int a = 0; a < TT; ++a)
#pragma unroll
        for (int b = 0; b < TT; ++b) { accr[a][b] = 0.0; acci[a][b] = 0.0; run[a][b].re = 0; run[a][b].im = 0; }

    int st = 0, since_flush = 0;
    uint32_t parity = 0;
    for (int64_t t = 0; t < ntiles; ++t) {
        // the stage tile t + STAGES - 1 goes to was read last for tile t - 1: every thread is past the __syncthreads that ended it
        if (threadIdx.x == 0 && t + kGramPipeStages - 1 < ntiles) { fence_proxy_async_smem(); issue(t + kGramPipeStages - 1); }
        const int64_t r0 = r_begin + t * rows;
        const int nrow = (int)((r_end - r0 < rows) ? (r_end - r0) : rows);
        mbar_wait(&full[st], parity);
        const cplx<T> *sU = reinterpret_cast<const cplx<T> *>(smem_raw + (size_t)st * 2 * tile_bytes);
        const cplx<T> *sW = reinterpret_cast<const cplx<T> *>(smem_raw + (size_t)st * 2 * tile_bytes + tile_bytes);
        for (int k = rg; k < nrow; k += RG) {
            cplx<T> u[TT], w[TT];
            gram_pipe_load<T, TT>(u, sU + k * S + a0);
            gram_pipe_load<T, TT>(w, sW + k * S + b0);
#pragma unroll
            for (int a = 0; a < TT; ++a)
#pragma unroll
                for (int b = 0; b < TT; ++b) cmac_conj(run[a][b], u[a], w[b]);
        }
        if (++since_flush == flush_tiles || t + 1 == ntiles) {
#pragma unroll
            for (int a = 0; a < TT; ++a)
#pragma unroll
                for (int b = 0; b < TT; ++b) {
                    accr[a][b] += (double)run[a][b].re; acci[a][b] += (double)run[a][b].im;
                    run[a][b].re = 0; run[a][b].im = 0;
                }
            since_flush = 0;
        }
        if (++st == kGramPipeStages) { st = 0; parity ^= 1u; }
        __syncthreads();
    }
    // row groups in a fixed order (0, 1, 2, ...) through shared memory: every copy has landed and been read, the ring is free
    double *red = reinterpret_cast<double *>(smem_raw);
    for (int g = 0; g < RG; ++g) {
        if (rg == g) {
#pragma unroll
            for (int a = 0; a < TT; ++a)
#pragma unroll
                for (int b = 0; b < TT; ++b) {
                    const int e = (a0 + a) * S + b0 + b;
                    if (g == 0) { red[2 * e] = accr[a][b]; red[2 * e + 1] = acci[a][b]; }
                    else { red[2 * e] += accr[a][b]; red[2 * e + 1] += acci[a][b]; }
                }
        }
        __syncthreads();
    }
    zdouble *out = partial + (size_t)blockIdx.x * S * S;
    for (int e = threadIdx.x; e < S * S; e += kLaThreads) { out[e].re = red[2 * e]; out[e].im = red[2 * e + 1]; }
}

// stage 2: G[e] = sum_b partial[b][e], b in increasing order
// One warp per entry: lane l sums blocks l, l + 32, ... in increasing order, then a fixed shuffle tree.
__global__ void gram_reduce_kernel(const zdouble *__restrict__ partial, int nblocks, int ss, zdouble *__restrict__ G)
{
    const int e = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (e >= ss) return;
    double re = 0.0, im = 0.0;
    for (int b = lane; b < nblocks; b += 32) { re += partial[(size_t)b * ss + e].re; im += partial[(size_t)b * ss + e].im; }
    for (int o = 16; o > 0; o >>= 1) { re += __shfl_down_sync(0xffffffffu, re, o); im += __shfl_down_sync(0xffffffffu, im, o); }
    if (lane == 0) { G[e].re = re; G[e].im = im; }
}

// ------------------------------------------------------------------------------------------------------
// Block rotation  out = beta * Vin + U K   (n x s times s x s).  out may alias U and/or Vin: a CTA stages
// its rows of U in shared memory before it writes them.  K is complex128 on the device, rounded to T at use
// (reading R11).
// ------------------------------------------------------------------------------------------------------
template <typename T, int TC>
__global__ void __launch_bounds__(kLaThreads)
rotate_kernel(const cplx<T> *U, const zdouble *__restrict__ K, const cplx<T> *Vin, cplx<T> *out, T beta,
              int64_t n, int s, int rows_per_tile)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx<T> *sK = reinterpret_cast<cplx<T> *>(smem_raw);          // [s][s]
    cplx<T> *sU = sK + (size_t)s * s;                              // [rows_per_tile][s + 1] (padded: row lanes hit different banks)
    const int su = s + 1;
    for (int e = threadIdx.x; e < s * s; e += kLaThreads) { sK[e].re = (T)K[e].re; sK[e].im = (T)K[e].im; }
    const int ncg = (s + TC - 1) / TC;            // column groups (<= 16)
    const int RL = kLaThreads / ncg;              // row lanes
    const int cg = threadIdx.x % ncg, rl = threadIdx.x / ncg;
    const int c0 = cg * TC;
    const int64_t ntiles = (n + rows_per_tile - 1) / rows_per_tile;
    for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const int64_t r0 = t * rows_per_tile;
        const int nrow = (int)((n - r0 < rows_per_tile) ? (n - r0) : rows_per_tile);
        __syncthreads();
        const cplx<T> *gu = U + r0 * s;
        for (int e = threadIdx.x; e < nrow * s; e += kLaThreads) sU[(e / s) * su + e % s] = gu[e];
        __syncthreads();
        if (rl < RL) {
            for (int k = rl; k < nrow; k += RL) {
                cplx<T> acc[TC];
#pragma unroll
                for (int c = 0; c < TC; ++c) { acc[c].re = 0; acc[c].im = 0; }
                for (int a = 0; a < s; ++a) {
                    const cplx<T> u = sU[k * su + a];
#pragma unroll
                    for (int c = 0; c < TC; ++c)
                        if (c0 + c < s) cmac(acc[c], u, sK[a * s + c0 + c]);
                }
#pragma unroll
                for (int c = 0; c < TC; ++c)
                    if (c0 + c < s) {
                        const int64_t e = (r0 + k) * s + c0 + c;
                        cplx<T> v = acc[c];
                        if (beta != (T)0) { const cplx<T> w = Vin[e]; v.re = fma(beta, w.re, v.re); v.im = fma(beta, w.im, v.im); }
                        out[e] = v;
                    }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------------
// The two fused passes of one BlockCGrQ iteration (Fig. 2 left, statements 10-13):
//   pass 1:  X += D K1 ;  T = Q + Z K2 ;  partial(T^H T)          reads D, Z, Q, X   writes X, T
//   pass 2:  Q = T K3 ;  D = Q + D K4                             reads T, D         writes Q, D
// (K1 = M C, K2 = -M, K3 = S^-1, K4 = S^H, complex128 on the device, rounded to T at use: DESIGN.md R11.)
// 10 block passes over HBM instead of the 15 of the unfused sequence (gram, rotate x 4, gram).
// Thread layout: the s columns are cut into groups of W; a thread owns TR rows x W columns of each product
// (row lanes interleaved so a warp touches consecutive rows); the Gram part of pass 1 uses W x W sub-blocks of
// T^H T per thread and the row groups that are left, products in T, sums flushed to double once per row tile.
// ------------------------------------------------------------------------------------------------------
template <typename T> struct LaPad { static constexpr int v = sizeof(T) == 4 ? 2 : 1; };   // keeps rows 16-byte aligned, banks spread

// rows r0 .. r0 + nrow of a row-major n x s block -> shared memory with leading dimension su (coalesced)
template <typename T>
__device__ __forceinline__ void la_stage_rows(cplx<T> *dst, const cplx<T> *__restrict__ src, int64_t r0, int nrow, int s, int su)
{
    const int rpp = kLaThreads / s, row0 = threadIdx.x / s, col = threadIdx.x - row0 * s;
    if (row0 < rpp)
        for (int r = row0; r < nrow; r += rpp) dst[r * su + col] = src[(r0 + r) * s + col];
}

// the same through cp.async (16-byte chunks; 8-byte for complex64 with odd s), no wait: the caller commits and waits.
// Rows nrow .. rows_total of the buffer are zeroed with plain stores (ragged last tile).
__device__ __forceinline__ void cp_async_16(void *dst_smem, const void *src) { asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst_smem)), "l"(src) : "memory"); }
__device__ __forceinline__ void cp_async_8(void *dst_smem, const void *src) { asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(dst_smem)), "l"(src) : "memory"); }
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <typename T>
__device__ __forceinline__ void la_stage_rows_async(cplx<T> *dst, const cplx<T> *__restrict__ src, int64_t r0, int nrow, int rows_total, int s, int su)
{
    const bool wide = sizeof(T) == 8 || (s & 1) == 0;                 // 16-byte chunks: one complex128 or two complex64
    const int epc = (sizeof(T) == 4 && wide) ? 2 : 1;                  // elements per chunk
    const int cpr = s / epc;                                           // chunks per row
    const int rpp = kLaThreads / cpr, row0 = threadIdx.x / cpr, j = (threadIdx.x - row0 * cpr) * epc;
    if (row0 < rpp) {
        for (int r = row0; r < nrow; r += rpp) {
            if (wide) cp_async_16(dst + r * su + j, src + (r0 + r) * s + j);
            else cp_async_8(dst + r * su + j, src + (r0 + r) * s + j);
        }
    }
    for (int e = threadIdx.x + nrow * su; e < rows_total * su; e += kLaThreads) dst[e] = {0, 0};
}

// acc[t][c] = sum_a sU[(rl + t RL)][a] * sK[a][c0 + c]
// S > 0: s is the compile-time constant S (a multiple of W): the a-loop unrolls and the column guard disappears
template <typename T, int TR, int W, int S = 0>
__device__ __forceinline__ void la_tile_product(cplx<T> (&acc)[TR][W], const cplx<T> *sU, const cplx<T> *sK, int rl, int RL, int c0, int s_rt, int su_rt)
{
    const int s = S ? S : s_rt, su = S ? S + LaPad<T>::v : su_rt;
#pragma unroll
    for (int t = 0; t < TR; ++t)
#pragma unroll
        for (int c = 0; c < W; ++c) { acc[t][c].re = 0; acc[t][c].im = 0; }
#pragma unroll(S ? 16 : 1)
    for (int a = 0; a < s; ++a) {
        cplx<T> u[TR], k[W];
#pragma unroll
        for (int t = 0; t < TR; ++t) u[t] = sU[(rl + t * RL) * su + a];
#pragma unroll
        for (int c = 0; c < W; ++c) k[c] = (S || c0 + c < s) ? sK[a * s + c0 + c] : cplx<T>{0, 0};
#pragma unroll
        for (int t = 0; t < TR; ++t)
#pragma unroll
            for (int c = 0; c < W; ++c) cmac(acc[t][c], u[t], k[c]);
    }
}

template <typename T, int TR, int W, int S = 0>
__global__ void __launch_bounds__(kLaThreads)
bcg_fused1_kernel(const cplx<T> *__restrict__ D, const cplx<T> *__restrict__ Z, const cplx<T> *__restrict__ Q, cplx<T> *X, cplx<T> *Tout,
                  const zdouble *__restrict__ K1, const zdouble *__restrict__ K2, int64_t n, int s_rt, zdouble *__restrict__ partial)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int s = S ? S : s_rt;
    const int su = s + LaPad<T>::v;
    const int ncg = (s + W - 1) / W, RL = kLaThreads / ncg, rows = RL * TR;
    cplx<T> *sK1 = reinterpret_cast<cplx<T> *>(smem_raw), *sK2 = sK1 + s * s;
    cplx<T> *sD0 = sK2 + s * s, *sZ0 = sD0 + (size_t)2 * rows * su;     // two stages each; a stage's D buffer is reused for its T tile
    for (int e = threadIdx.x; e < s * s; e += kLaThreads) {
        sK1[e].re = (T)K1[e].re; sK1[e].im = (T)K1[e].im;
        sK2[e].re = (T)K2[e].re; sK2[e].im = (T)K2[e].im;
    }
    const int cg = threadIdx.x % ncg, rl = threadIdx.x / ncg, c0 = cg * W;
    const bool rot_active = rl < RL;
    // Gram layout: W x W sub-blocks, RG row groups
    const int ntile = ncg * ncg, RG = kLaThreads / ntile;
    const int gt = threadIdx.x % ntile, rg = threadIdx.x / ntile;
    const bool gram_active = rg < RG;
    const int ga0 = (gt / ncg) * W, gb0 = (gt % ncg) * W;
    double accr[W][W], acci[W][W];
#pragma unroll
    for (int a = 0; a < W; ++a)
#pragma unroll
        for (int b = 0; b < W; ++b) { accr[a][b] = 0.0; acci[a][b] = 0.0; }

    const int64_t ntiles = (n + rows - 1) / rows;
    auto stage = [&](int b, int64_t t) {
        const int64_t r0 = t * rows;
        const int nrow = (int)((n - r0 < rows) ? (n - r0) : rows);
        la_stage_rows_async(sD0 + (size_t)b * rows * su, D, r0, nrow, rows, s, su);
        la_stage_rows_async(sZ0 + (size_t)b * rows * su, Z, r0, nrow, rows, s, su);
    };
    int buf = 0;
    if ((int64_t)blockIdx.x < ntiles) stage(0, blockIdx.x);
    cp_async_commit();
    for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x, buf ^= 1) {
        const int64_t r0 = t * rows;
        const int nrow = (int)((n - r0 < rows) ? (n - r0) : rows);
        if (t + gridDim.x < ntiles) stage(buf ^ 1, t + gridDim.x);     // next tile in flight while this one is worked on
        cp_async_commit();
        cp_async_wait<1>();
        __syncthreads();                                   // tile t has landed for every thread (and sK is written)
        cplx<T> *sD = sD0 + (size_t)buf * rows * su, *sZ = sZ0 + (size_t)buf * rows * su;
        cplx<T> tv[TR][W];
        if (rot_active) {
            cplx<T> acc[TR][W];
            la_tile_product<T, TR, W, S>(acc, sD, sK1, rl, RL, c0, s, su);          // D K1
#pragma unroll
            for (int tt = 0; tt < TR; ++tt) {
                const int row = rl + tt * RL;
                if (row < nrow)
#pragma unroll
                    for (int c = 0; c < W; ++c)
                        if (S || c0 + c < s) {
                            const int64_t e = (r0 + row) * s + c0 + c;
                            cplx<T> x = X[e];
                            x.re += acc[tt][c].re; x.im += acc[tt][c].im;
                            X[e] = x;
                        }
            }
            la_tile_product<T, TR, W, S>(tv, sZ, sK2, rl, RL, c0, s, su);           // Z K2
#pragma unroll
            for (int tt = 0; tt < TR; ++tt) {
                const int row = rl + tt * RL;
#pragma unroll
                for (int c = 0; c < W; ++c) {
                    if (row < nrow && (S || c0 + c < s)) {
                        const int64_t e = (r0 + row) * s + c0 + c;
                        const cplx<T> q = Q[e];
                        tv[tt][c].re += q.re; tv[tt][c].im += q.im;
                        Tout[e] = tv[tt][c];
                    } else { tv[tt][c].re = 0; tv[tt][c].im = 0; }
                }
            }
        }
        __syncthreads();                                   // all reads of sD (as D) are done
        if (rot_active) {
#pragma unroll
            for (int tt = 0; tt < TR; ++tt)
#pragma unroll
                for (int c = 0; c < W; ++c)
                    if (S || c0 + c < s) sD[(rl + tt * RL) * su + c0 + c] = tv[tt][c];
        }
        __syncthreads();
        if (gram_active) {
            cplx<T> run[W][W];
#pragma unroll
            for (int a = 0; a < W; ++a)
#pragma unroll
                for (int b = 0; b < W; ++b) { run[a][b].re = 0; run[a][b].im = 0; }
            for (int k = rg; k < nrow; k += RG) {
                cplx<T> u[W], w[W];
#pragma unroll
                for (int a = 0; a < W; ++a) u[a] = (S || ga0 + a < s) ? sD[k * su + ga0 + a] : cplx<T>{0, 0};
#pragma unroll
                for (int b = 0; b < W; ++b) w[b] = (S || gb0 + b < s) ? sD[k * su + gb0 + b] : cplx<T>{0, 0};
#pragma unroll
                for (int a = 0; a < W; ++a)
#pragma unroll
                    for (int b = 0; b < W; ++b) cmac_conj(run[a][b], u[a], w[b]);
            }
#pragma unroll
            for (int a = 0; a < W; ++a)
#pragma unroll
                for (int b = 0; b < W; ++b) { accr[a][b] += (double)run[a][b].re; acci[a][b] += (double)run[a][b].im; }
        }
        __syncthreads();                                   // this stage's buffers may be restaged by the next iteration
    }
    // reduce the row groups in a fixed order through shared memory (the tile buffers are free now)
    cp_async_wait<0>();
    __syncthreads();
    double *red = reinterpret_cast<double *>(sD0);
    for (int g = 0; g < RG; ++g) {
        if (gram_active && rg == g) {
#pragma unroll
            for (int a = 0; a < W; ++a)
#pragma unroll
                for (int b = 0; b < W; ++b)
                    if (ga0 + a < s && gb0 + b < s) {
                        const int e = (ga0 + a) * s + gb0 + b;
                        if (g == 0) { red[2 * e] = accr[a][b]; red[2 * e + 1] = acci[a][b]; }
                        else { red[2 * e] += accr[a][b]; red[2 * e + 1] += acci[a][b]; }
                    }
        }
        __syncthreads();
    }
    zdouble *out = partial + (size_t)blockIdx.x * s * s;
    for (int e = threadIdx.x; e < s * s; e += kLaThreads) { out[e].re = red[2 * e]; out[e].im = red[2 * e + 1]; }
}

template <typename T, int TR, int W, int S = 0>
__global__ void __launch_bounds__(kLaThreads)
bcg_fused2_kernel(const cplx<T> *__restrict__ Tin, cplx<T> *D, cplx<T> *Qout, const zdouble *__restrict__ K3, const zdouble *__restrict__ K4,
                  int64_t n, int s_rt, uint32_t *__restrict__ colmax)
{
    // colmax (may be NULL; zeroed by the caller): per-column max |Re|, |Im| of the new D as float bit patterns -- the first
    // pre-pass of the FP16-split stencil kernel, which reads this D next, fused into its producer (order independent: atomicMax)
    __shared__ uint32_t scm[COARSE_MAX_NRHS];
    uint32_t cm[W];
#pragma unroll
    for (int c = 0; c < W; ++c) cm[c] = 0u;
    if (threadIdx.x < COARSE_MAX_NRHS) scm[threadIdx.x] = 0u;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int s = S ? S : s_rt;
    const int su = s + LaPad<T>::v;
    const int ncg = (s + W - 1) / W, RL = kLaThreads / ncg, rows = RL * TR;
    cplx<T> *sK3 = reinterpret_cast<cplx<T> *>(smem_raw), *sK4 = sK3 + s * s;
    cplx<T> *sT0 = sK4 + s * s, *sD0 = sT0 + (size_t)2 * rows * su;     // two stages each
    for (int e = threadIdx.x; e < s * s; e += kLaThreads) {
        sK3[e].re = (T)K3[e].re; sK3[e].im = (T)K3[e].im;
        sK4[e].re = (T)K4[e].re; sK4[e].im = (T)K4[e].im;
    }
    const int cg = threadIdx.x % ncg, rl = threadIdx.x / ncg, c0 = cg * W;
    const int64_t ntiles = (n + rows - 1) / rows;
    auto stage = [&](int b, int64_t t) {
        const int64_t r0 = t * rows;
        const int nrow = (int)((n - r0 < rows) ? (n - r0) : rows);
        la_stage_rows_async(sT0 + (size_t)b * rows * su, Tin, r0, nrow, rows, s, su);
        la_stage_rows_async(sD0 + (size_t)b * rows * su, (const cplx<T> *)D, r0, nrow, rows, s, su);
    };
    int buf = 0;
    if ((int64_t)blockIdx.x < ntiles) stage(0, blockIdx.x);
    cp_async_commit();
    for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x, buf ^= 1) {
        const int64_t r0 = t * rows;
        const int nrow = (int)((n - r0 < rows) ? (n - r0) : rows);
        if (t + gridDim.x < ntiles) stage(buf ^ 1, t + gridDim.x);     // (rows of D this CTA writes below are its own: no other tile reads them)
        cp_async_commit();
        cp_async_wait<1>();
        __syncthreads();
        const cplx<T> *sT = sT0 + (size_t)buf * rows * su, *sD = sD0 + (size_t)buf * rows * su;
        if (rl < RL) {
            cplx<T> q[TR][W], d[TR][W];
            la_tile_product<T, TR, W, S>(q, sT, sK3, rl, RL, c0, s, su);            // Q = T S^-1
            la_tile_product<T, TR, W, S>(d, sD, sK4, rl, RL, c0, s, su);            // D S^H
#pragma unroll
            for (int tt = 0; tt < TR; ++tt) {
                const int row = rl + tt * RL;
                if (row < nrow)
#pragma unroll
                    for (int c = 0; c < W; ++c)
                        if (S || c0 + c < s) {
                            const int64_t e = (r0 + row) * s + c0 + c;
                            Qout[e] = q[tt][c];
                            cplx<T> v;
                            v.re = q[tt][c].re + d[tt][c].re;
                            v.im = q[tt][c].im + d[tt][c].im;
                            D[e] = v;                                            // D = Q + D S^H (this CTA staged its rows of D first)
                            if (sizeof(T) == 4) {
                                const uint32_t a = __float_as_uint((float)v.re) & 0x7FFFFFFFu, b = __float_as_uint((float)v.im) & 0x7FFFFFFFu;
                                if (a <= 0x7F800000u) cm[c] = max(cm[c], a);
                                if (b <= 0x7F800000u) cm[c] = max(cm[c], b);
                            }
                        }
            }
        }
        __syncthreads();                                   // this stage's buffers may be restaged by the next iteration
    }
    cp_async_wait<0>();
    if (sizeof(T) == 4 && colmax != nullptr) {
        if (rl < RL)
#pragma unroll
            for (int c = 0; c < W; ++c)
                if ((S || c0 + c < s) && cm[c]) atomicMax(&scm[c0 + c], cm[c]);
        __syncthreads();
        if (threadIdx.x < s && scm[threadIdx.x]) atomicMax(&colmax[threadIdx.x], scm[threadIdx.x]);
    }
}

// Chebyshev recurrence, one fused elementwise pass:
//   Tn = ca * Z + cb * Tc - cp * Tp   (Z = H Tc from the stencil kernel; Tn overwrites Tp)
//   X  = cx * X + cn * Tn             (cx = 0 on the first call: X need not be initialised)
template <typename T>
__global__ void __launch_bounds__(256)
cheby_step_kernel(const cplx<T> *__restrict__ Z, const cplx<T> *__restrict__ Tc, cplx<T> *Tp, cplx<T> *X,
                  T ca, T cb, T cp, T cx, T cn, int64_t total, int s, uint32_t *__restrict__ colmax)
{
    // colmax (complex64 only; may be NULL; zeroed by the caller): per-column max |Re|, |Im| of Tn as float bit patterns, as
    // colmax_kernel would find them -- the next apply's split-FP16 pre-pass then needs no pass of its own over Tn.
    // 32 bytes per thread and array per trip (4 complex64 / 2 complex128), all loads issued before the arithmetic
    constexpr int VEC = 32 / (int)sizeof(cplx<T>);
    const int64_t nvec = total / VEC;
    __shared__ uint32_t scm[COARSE_MAX_NRHS];
    const bool want_max = sizeof(T) == 4 && colmax != nullptr;
    // a thread meets the same VEC columns on every trip when its stride is a multiple of s: then the maxima stay in registers
    const bool fixed_cols = ((int64_t)gridDim.x * blockDim.x * VEC) % s == 0;
    uint32_t mx[VEC];
#pragma unroll
    for (int u = 0; u < VEC; ++u) mx[u] = 0u;
    if (want_max) {
        if (threadIdx.x < COARSE_MAX_NRHS) scm[threadIdx.x] = 0u;
        __syncthreads();
    }
    auto note = [&](uint32_t &m, T re, T im) {
        const uint32_t a = __float_as_uint((float)re) & 0x7FFFFFFFu, b = __float_as_uint((float)im) & 0x7FFFFFFFu;
        if (a <= 0x7F800000u) m = max(m, a);
        if (b <= 0x7F800000u) m = max(m, b);
    };
    for (int64_t v = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; v < nvec; v += (int64_t)gridDim.x * blockDim.x) {
        const int64_t e0 = v * VEC;
        cplx<T> z[VEC], tc[VEC], tp[VEC], x[VEC];
#pragma unroll
        for (int u = 0; u < VEC; u += 16 / (int)sizeof(cplx<T>)) {
            *reinterpret_cast<float4 *>(&z[u]) = *reinterpret_cast<const float4 *>(&Z[e0 + u]);
            *reinterpret_cast<float4 *>(&tc[u]) = *reinterpret_cast<const float4 *>(&Tc[e0 + u]);
            if (cp != (T)0) *reinterpret_cast<float4 *>(&tp[u]) = *reinterpret_cast<const float4 *>(&Tp[e0 + u]);
            if (cx != (T)0) *reinterpret_cast<float4 *>(&x[u]) = *reinterpret_cast<const float4 *>(&X[e0 + u]);
        }
#pragma unroll
        for (int u = 0; u < VEC; ++u) {
            cplx<T> tn;
            tn.re = ca * z[u].re + cb * tc[u].re;
            tn.im = ca * z[u].im + cb * tc[u].im;
            if (cp != (T)0) { tn.re -= cp * tp[u].re; tn.im -= cp * tp[u].im; }
            cplx<T> xo = {0, 0};
            if (cx != (T)0) { xo.re = cx * x[u].re; xo.im = cx * x[u].im; }
            xo.re += cn * tn.re;
            xo.im += cn * tn.im;
            tp[u] = tn;
            x[u] = xo;
            if (want_max) {
                if (fixed_cols) note(mx[u], tn.re, tn.im);
                else { uint32_t m = 0u; note(m, tn.re, tn.im); if (m) atomicMax(&scm[(e0 + u) % s], m); }
            }
        }
#pragma unroll
        for (int u = 0; u < VEC; u += 16 / (int)sizeof(cplx<T>)) {
            *reinterpret_cast<float4 *>(&Tp[e0 + u]) = *reinterpret_cast<const float4 *>(&tp[u]);
            *reinterpret_cast<float4 *>(&X[e0 + u]) = *reinterpret_cast<const float4 *>(&x[u]);
        }
    }
    // ragged tail (total not a multiple of VEC)
    for (int64_t e = nvec * VEC + blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        const cplx<T> z = Z[e], tc = Tc[e];
        cplx<T> tn;
        tn.re = ca * z.re + cb * tc.re;
        tn.im = ca * z.im + cb * tc.im;
        if (cp != (T)0) { const cplx<T> tp = Tp[e]; tn.re -= cp * tp.re; tn.im -= cp * tp.im; }
        Tp[e] = tn;
        if (want_max) { uint32_t m = 0u; note(m, tn.re, tn.im); if (m) atomicMax(&scm[e % s], m); }
        cplx<T> x = {0, 0};
        if (cx != (T)0) { const cplx<T> xo = X[e]; x.re = cx * xo.re; x.im = cx * xo.im; }
        x.re += cn * tn.re;
        x.im += cn * tn.im;
        X[e] = x;
    }
    if (want_max) {
        if (fixed_cols) {
            const int64_t e0 = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) * VEC;
#pragma unroll
            for (int u = 0; u < VEC; ++u)
                if (mx[u]) atomicMax(&scm[(e0 + u) % s], mx[u]);
        }
        __syncthreads();
        if (threadIdx.x < s && scm[threadIdx.x]) atomicMax(&colmax[threadIdx.x], scm[threadIdx.x]);
    }
}

// ------------------------------------------------------------------------------------------------------
// Multi-RHS deflation (Eq. 7-10, 325-329): two tall-skinny products with the n x m block of eigenvectors.
//   stage 1: C = Vev^H B (m x s) -- per-CTA partials in double, summed by gram_reduce_kernel (deterministic)
//   stage 2: Qb_par = Vev (C / lambda),  b_perp = B - Vev C        (one pass over Vev and B)
// ------------------------------------------------------------------------------------------------------
struct DeflLambda { double inv[COARSE_MAX_NRHS]; };      // 1 / lambda_i, passed by value

template <typename T>
__global__ void __launch_bounds__(kLaThreads)
rgram_partial_kernel(const cplx<T> *__restrict__ Vev, int ldv, const cplx<T> *__restrict__ B, int64_t n, int m, int s, int rows_per_tile,
                     zdouble *__restrict__ partial)      // Vev: m columns of a block whose rows are ldv apart
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx<T> *sV = reinterpret_cast<cplx<T> *>(smem_raw);
    cplx<T> *sB = sV + (size_t)rows_per_tile * m;
    constexpr int MAXE = (COARSE_MAX_NRHS * COARSE_MAX_NRHS) / kLaThreads;      // entries of C per thread
    const int ms = m * s;
    double accr[MAXE], acci[MAXE];
    int ei[MAXE], er[MAXE];
#pragma unroll
    for (int j = 0; j < MAXE; ++j) {
        const int e = threadIdx.x + j * kLaThreads;
        accr[j] = 0.0; acci[j] = 0.0;
        ei[j] = e < ms ? e / s : -1;
        er[j] = e < ms ? e % s : 0;
    }
    const int64_t chunk = (n + gridDim.x - 1) / gridDim.x;
    const int64_t r_begin = blockIdx.x * chunk;
    const int64_t r_end = (r_begin + chunk < n) ? r_begin + chunk : n;
    for (int64_t r0 = r_begin; r0 < r_end; r0 += rows_per_tile) {
        const int nrow = (int)((r_end - r0 < rows_per_tile) ? (r_end - r0) : rows_per_tile);
        __syncthreads();
        for (int e = threadIdx.x; e < nrow * m; e += kLaThreads) sV[e] = Vev[(r0 + e / m) * ldv + e % m];
        for (int e = threadIdx.x; e < nrow * s; e += kLaThreads) sB[e] = B[r0 * s + e];
        __syncthreads();
#pragma unroll
        for (int j = 0; j < MAXE; ++j) {
            if (ei[j] < 0) continue;
            double re = 0.0, im = 0.0;
            for (int k = 0; k < nrow; ++k) {
                const cplx<T> v = sV[k * m + ei[j]], b = sB[k * s + er[j]];
                re += (double)v.re * (double)b.re + (double)v.im * (double)b.im;       // conj(v) * b
                im += (double)v.re * (double)b.im - (double)v.im * (double)b.re;
            }
            accr[j] += re; acci[j] += im;
        }
    }
    zdouble *out = partial + (size_t)blockIdx.x * ms;
#pragma unroll
    for (int j = 0; j < MAXE; ++j)
        if (ei[j] >= 0) out[threadIdx.x + j * kLaThreads] = {accr[j], acci[j]};
}

template <typename T>
__global__ void __launch_bounds__(kLaThreads)
deflate_update_kernel(const cplx<T> *__restrict__ Vev, int ldv, const cplx<T> *B, const zdouble *__restrict__ Cm, const DeflLambda lam,
                      cplx<T> *__restrict__ QBpar, cplx<T> *Bperp, int64_t n, int m, int s, int rows_per_tile, int accumulate)
// Bperp may alias B.  accumulate != 0 (the second and later chunks of eigenvectors): QBpar += Vev (C / lambda)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx<T> *sC = reinterpret_cast<cplx<T> *>(smem_raw);          // [m][s]   <i|b>
    cplx<T> *sCl = sC + m * s;                                     // [m][s]   <i|b> / lambda_i
    cplx<T> *sV = sCl + m * s;                                     // [rows_per_tile][m]
    for (int e = threadIdx.x; e < m * s; e += kLaThreads) {
        const double il = lam.inv[e / s];
        sC[e].re = (T)Cm[e].re; sC[e].im = (T)Cm[e].im;
        sCl[e].re = (T)(Cm[e].re * il); sCl[e].im = (T)(Cm[e].im * il);
    }
    const int64_t ntiles = (n + rows_per_tile - 1) / rows_per_tile;
    for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const int64_t r0 = t * rows_per_tile;
        const int nrow = (int)((n - r0 < rows_per_tile) ? (n - r0) : rows_per_tile);
        __syncthreads();
        for (int e = threadIdx.x; e < nrow * m; e += kLaThreads) sV[e] = Vev[(r0 + e / m) * ldv + e % m];
        __syncthreads();
        for (int e = threadIdx.x; e < nrow * s; e += kLaThreads) {
            const int k = e / s, r = e - k * s;
            cplx<T> par = {0, 0}, q = {0, 0};
            for (int i = 0; i < m; ++i) {
                const cplx<T> v = sV[k * m + i];
                cmac(par, v, sC[i * s + r]);
                cmac(q, v, sCl[i * s + r]);
            }
            const cplx<T> b = B[r0 * s + e];
            if (accumulate) {
                const cplx<T> q0 = QBpar[r0 * s + e];
                q.re += q0.re;
                q.im += q0.im;
            }
            QBpar[r0 * s + e] = q;
            Bperp[r0 * s + e] = {b.re - par.re, b.im - par.im};
        }
    }
}

// ------------------------------------------------------------------------------------------------------
// Register-tiled forms of the two deflation kernels for m and s multiples of 4 (the kernels above do one output element per
// thread and convert every operand of every multiply-add: 6.8 TFLOP/s at nev 192, nrhs 16).  Same arithmetic contract.
// stage 1: 4 x 4 sub-blocks of C = Vev^H B per thread, the threads left over split the rows (fixed-order reduction at the end);
// complex128: products and sums in double as above; complex64: products and one tile's run per thread (<= 32 terms) in float, sums in double.
// ------------------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(kLaThreads, 2)
rgram_tiled_kernel(const cplx<T> *__restrict__ Vev, int ldv, const cplx<T> *__restrict__ B, int64_t n, int m, int s, int rows_per_tile,
                   zdouble *__restrict__ partial)
{
    constexpr int TT = 4;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx<T> *sV = reinterpret_cast<cplx<T> *>(smem_raw);
    cplx<T> *sB = sV + (size_t)rows_per_tile * m;
    const int ntb = s / TT, ntile = (m / TT) * ntb, RG = kLaThreads / ntile;
    const int tile = threadIdx.x % ntile, rg = threadIdx.x / ntile;
    const bool active = rg < RG;
    const int a0 = (tile / ntb) * TT, b0 = (tile % ntb) * TT;
    double accr[TT][TT], acci[TT][TT];
#pragma unroll
    for (int a = 0; a < TT; ++a)
#pragma unroll
        for (int b = 0; b < TT; ++b) { accr[a][b] = 0.0; acci[a][b] = 0.0; }
    const int64_t chunk = (n + gridDim.x - 1) / gridDim.x;
    const int64_t r_begin = blockIdx.x * chunk;
    const int64_t r_end = (r_begin + chunk < n) ? r_begin + chunk : n;
    const int cpr = m / TT;                       // 4-element pieces per row of the eigenvector chunk
    for (int64_t r0 = r_begin; r0 < r_end; r0 += rows_per_tile) {
        const int nrow = (int)((r_end - r0 < rows_per_tile) ? (r_end - r0) : rows_per_tile);
        __syncthreads();
        for (int e = threadIdx.x; e < nrow * cpr; e += kLaThreads) {
            const int k = e / cpr, j = (e - k * cpr) * TT;
            cplx<T> v[TT];
            gram_pipe_load<T, TT>(v, Vev + (r0 + k) * ldv + j);
#pragma unroll
            for (int u = 0; u < TT; ++u) sV[k * m + j + u] = v[u];
        }
        for (int e = threadIdx.x; e < nrow * s; e += kLaThreads) sB[e] = B[r0 * s + e];
        __syncthreads();
        if (active) {
            if constexpr (sizeof(T) == 4) {
                // complex64: products and this tile's run (rows_per_tile / RG <= 32 terms) in float, the run added to the double sums --
                // the contract of the Gram kernels (gram_partial_kernel), at the FP32 rate and without a conversion per operand
                cplx<T> run[TT][TT];
#pragma unroll
                for (int a = 0; a < TT; ++a)
#pragma unroll
                    for (int c = 0; c < TT; ++c) { run[a][c].re = 0; run[a][c].im = 0; }
                for (int k = rg; k < nrow; k += RG) {
                    cplx<T> v[TT], b[TT];
                    gram_pipe_load<T, TT>(v, sV + k * m + a0);
                    gram_pipe_load<T, TT>(b, sB + k * s + b0);
#pragma unroll
                    for (int a = 0; a < TT; ++a)
#pragma unroll
                        for (int c = 0; c < TT; ++c) cmac_conj(run[a][c], v[a], b[c]);
                }
#pragma unroll
                for (int a = 0; a < TT; ++a)
#pragma unroll
                    for (int c = 0; c < TT; ++c) { accr[a][c] += (double)run[a][c].re; acci[a][c] += (double)run[a][c].im; }
            } else {
                for (int k = rg; k < nrow; k += RG) {
                    cplx<T> v[TT], b[TT];
                    gram_pipe_load<T, TT>(v, sV + k * m + a0);
                    gram_pipe_load<T, TT>(b, sB + k * s + b0);
#pragma unroll
                    for (int a = 0; a < TT; ++a)
#pragma unroll
                        for (int c = 0; c < TT; ++c) {            // conj(v) * b
                            accr[a][c] += (double)v[a].re * (double)b[c].re + (double)v[a].im * (double)b[c].im;
                            acci[a][c] += (double)v[a].re * (double)b[c].im - (double)v[a].im * (double)b[c].re;
                        }
                }
            }
        }
    }
    zdouble *out = partial + (size_t)blockIdx.x * m * s;
    if (RG == 1) {                                // one thread per sub-block: no reduction
#pragma unroll
        for (int a = 0; a < TT; ++a)
#pragma unroll
            for (int c = 0; c < TT; ++c) out[(a0 + a) * s + b0 + c] = {accr[a][c], acci[a][c]};
        return;
    }
    // row groups in a fixed order (0, 1, 2, ...) through shared memory (the launcher sizes it for m * s complex doubles)
    __syncthreads();
    double *red = reinterpret_cast<double *>(smem_raw);
    for (int g = 0; g < RG; ++g) {
        if (active && rg == g) {
#pragma unroll
            for (int a = 0; a < TT; ++a)
#pragma unroll
                for (int c = 0; c < TT; ++c) {
                    const int e = (a0 + a) * s + b0 + c;
                    if (g == 0) { red[2 * e] = accr[a][c]; red[2 * e + 1] = acci[a][c]; }
                    else { red[2 * e] += accr[a][c]; red[2 * e + 1] += acci[a][c]; }
                }
        }
        __syncthreads();
    }
    for (int e = threadIdx.x; e < m * s; e += kLaThreads) out[e] = {red[2 * e], red[2 * e + 1]};
}

// stage 2: TR rows x 4 columns of both products per thread, lanes along the rows (rows of the chunk padded by LaPad in shared
// memory), two contraction indices per 16-byte load for complex64.
template <typename T, int TR>
__global__ void __launch_bounds__(kLaThreads)
deflate_update_tiled_kernel(const cplx<T> *__restrict__ Vev, int ldv, const cplx<T> *B, const zdouble *__restrict__ Cm, const DeflLambda lam,
                            cplx<T> *__restrict__ QBpar, cplx<T> *Bperp, int64_t n, int m, int s, int RL, int accumulate)
{
    constexpr int W = 4, AV = 16 / (int)sizeof(cplx<T>);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int ld = m + LaPad<T>::v, rows = RL * TR, ncg = s / W;
    cplx<T> *sC = reinterpret_cast<cplx<T> *>(smem_raw);          // [m][s]   <i|b>
    cplx<T> *sCl = sC + m * s;                                     // [m][s]   <i|b> / lambda_i
    cplx<T> *sV = sCl + m * s;                                     // [rows][ld]
    for (int e = threadIdx.x; e < m * s; e += kLaThreads) {
        const double il = lam.inv[e / s];
        sC[e].re = (T)Cm[e].re; sC[e].im = (T)Cm[e].im;
        sCl[e].re = (T)(Cm[e].re * il); sCl[e].im = (T)(Cm[e].im * il);
    }
    const int cg = threadIdx.x / RL, rl = threadIdx.x - cg * RL, c0 = cg * W;
    const bool active = cg < ncg;
    const int cpr = m / W;
    const int64_t ntiles = (n + rows - 1) / rows;
    for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const int64_t r0 = t * rows;
        const int nrow = (int)((n - r0 < rows) ? (n - r0) : rows);
        __syncthreads();
        for (int e = threadIdx.x; e < rows * cpr; e += kLaThreads) {
            const int k = e / cpr, j = (e - k * cpr) * W;
            cplx<T> v[W];
            if (k < nrow) gram_pipe_load<T, W>(v, Vev + (r0 + k) * ldv + j);
            else {
#pragma unroll
                for (int u = 0; u < W; ++u) v[u] = {0, 0};
            }
#pragma unroll
            for (int u = 0; u < W; ++u) sV[k * ld + j + u] = v[u];
        }
        __syncthreads();
        if (active) {
            cplx<T> par[TR][W], q[TR][W];
#pragma unroll
            for (int tt = 0; tt < TR; ++tt)
#pragma unroll
                for (int c = 0; c < W; ++c) { par[tt][c].re = 0; par[tt][c].im = 0; q[tt][c].re = 0; q[tt][c].im = 0; }
            for (int i = 0; i < m; i += AV) {
                cplx<T> v[TR][AV], kc[AV][W], kl[AV][W];
#pragma unroll
                for (int tt = 0; tt < TR; ++tt) gram_pipe_load<T, AV>(v[tt], sV + (rl + tt * RL) * ld + i);
#pragma unroll
                for (int j = 0; j < AV; ++j) { gram_pipe_load<T, W>(kc[j], sC + (i + j) * s + c0); gram_pipe_load<T, W>(kl[j], sCl + (i + j) * s + c0); }
#pragma unroll
                for (int j = 0; j < AV; ++j)
#pragma unroll
                    for (int tt = 0; tt < TR; ++tt)
#pragma unroll
                        for (int c = 0; c < W; ++c) { cmac(par[tt][c], v[tt][j], kc[j][c]); cmac(q[tt][c], v[tt][j], kl[j][c]); }
            }
#pragma unroll
            for (int tt = 0; tt < TR; ++tt) {
                const int row = rl + tt * RL;
                if (row < nrow) {
                    const int64_t e0 = (r0 + row) * s + c0;
                    cplx<T> b[W], q0[W];
                    gram_pipe_load<T, W>(b, B + e0);
                    if (accumulate) gram_pipe_load<T, W>(q0, QBpar + e0);
#pragma unroll
                    for (int c = 0; c < W; ++c) {
                        if (accumulate) { q[tt][c].re += q0[c].re; q[tt][c].im += q0[c].im; }
                        b[c].re -= par[tt][c].re; b[c].im -= par[tt][c].im;
                    }
#pragma unroll
                    for (int c = 0; c < W; c += AV) {
                        *reinterpret_cast<float4 *>(QBpar + e0 + c) = *reinterpret_cast<const float4 *>(&q[tt][c]);
                        *reinterpret_cast<float4 *>(Bperp + e0 + c) = *reinterpret_cast<const float4 *>(&b[c]);
                    }
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------------
// Stacked single-Krylov CG: one alpha / beta per iteration from Frobenius inner products over the
// whole block.  Scalars live on the device (sc: 0 rho, 1 alpha, 2 beta, 3 ||B||_F^2, 4 stop = sqrt(rho / ||B||^2)).
// Reductions: fixed partition over CTAs, fixed order inside (shuffle tree, then warp 0), partials summed by one warp.
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void la_block_sum_store(double v, double *out)
{
    __shared__ double wsum[kLaThreads / 32];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < kLaThreads / 32; ++k) t += wsum[k];
        *out = t;
    }
}

template <typename T>
__global__ void __launch_bounds__(kLaThreads) fdot_partial_kernel(const cplx<T> *__restrict__ U, const cplx<T> *__restrict__ W, int64_t total,
                                                                  double *__restrict__ partial)
{
    const int64_t chunk = (total + gridDim.x - 1) / gridDim.x;
    const int64_t e0 = blockIdx.x * chunk, e1 = (e0 + chunk < total) ? e0 + chunk : total;
    double acc = 0.0;
    for (int64_t e = e0 + threadIdx.x; e < e1; e += kLaThreads) {
        const cplx<T> u = U[e], w = W[e];
        acc += (double)u.re * (double)w.re + (double)u.im * (double)w.im;         // Re conj(u) w
    }
    la_block_sum_store(acc, partial + blockIdx.x);
}

// mode 0: ||B||^2 ; 1: rho_0 (+ stop) ; 2: alpha = rho / <P, Z> ; 3: beta = rho' / rho, rho <- rho' (+ stop)
__global__ void scg_scalar_kernel(int mode, const double *__restrict__ partial, int nblocks, double *sc)
{
    double v = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += 32) v += partial[b];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if (threadIdx.x != 0) return;
    if (mode == 0) sc[3] = v > 0.0 ? v : 1.0;
    else if (mode == 1) { sc[0] = v; sc[4] = sqrt(v / sc[3]); }
    else if (mode == 2) sc[1] = sc[0] / v;
    else { sc[2] = v / sc[0]; sc[0] = v; sc[4] = sqrt(v / sc[3]); }
}

// X += alpha P ; R -= alpha Z ; partial(<R, R>)
template <typename T>
__global__ void __launch_bounds__(kLaThreads) scg_update1_kernel(const cplx<T> *__restrict__ P, const cplx<T> *__restrict__ Z, cplx<T> *X, cplx<T> *R,
                                                                 const double *__restrict__ sc, int64_t total, double *__restrict__ partial)
{
    const T alpha = (T)sc[1];
    const int64_t chunk = (total + gridDim.x - 1) / gridDim.x;
    const int64_t e0 = blockIdx.x * chunk, e1 = (e0 + chunk < total) ? e0 + chunk : total;
    double acc = 0.0;
    for (int64_t e = e0 + threadIdx.x; e < e1; e += kLaThreads) {
        const cplx<T> p = P[e], z = Z[e];
        cplx<T> x = X[e], r = R[e];
        x.re += alpha * p.re; x.im += alpha * p.im;
        r.re -= alpha * z.re; r.im -= alpha * z.im;
        X[e] = x;
        R[e] = r;
        acc += (double)r.re * (double)r.re + (double)r.im * (double)r.im;
    }
    la_block_sum_store(acc, partial + blockIdx.x);
}

// P = R + beta P
template <typename T>
__global__ void __launch_bounds__(kLaThreads) scg_update2_kernel(const cplx<T> *__restrict__ R, cplx<T> *P, const double *__restrict__ sc, int64_t total)
{
    const T beta = (T)sc[2];
    for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        const cplx<T> r = R[e];
        cplx<T> p = P[e];
        p.re = r.re + beta * p.re;
        p.im = r.im + beta * p.im;
        P[e] = p;
    }
}

// ------------------------------------------------------------------------------------------------------
// Multi-RHS transfer between grids (Eq. 14-15): one small GEMM per coarse site, one CTA per site
// (grid-stride).  basis [Vc][vb][nb], fine [Vc][vb][s], coarse [Vc][nb][s]; products in T, sums over V_block in double (project).
// ------------------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(kLaThreads)
block_project_kernel(const cplx<T> *__restrict__ Bas, const cplx<T> *__restrict__ F, cplx<T> *__restrict__ Cc, int64_t Vc, int vb, int nb, int s,
                     int rows_per_tile)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx<T> *sB = reinterpret_cast<cplx<T> *>(smem_raw);
    cplx<T> *sF = sB + (size_t)rows_per_tile * nb;
    constexpr int MAXE = (COARSE_MAX_NBASIS * COARSE_MAX_NRHS) / kLaThreads;
    const int ms = nb * s;
    int ek[MAXE], er[MAXE];
#pragma unroll
    for (int j = 0; j < MAXE; ++j) {
        const int e = threadIdx.x + j * kLaThreads;
        ek[j] = e < ms ? e / s : -1;
        er[j] = e < ms ? e % s : 0;
    }
    for (int64_t x = blockIdx.x; x < Vc; x += gridDim.x) {
        double accr[MAXE], acci[MAXE];
#pragma unroll
        for (int j = 0; j < MAXE; ++j) { accr[j] = 0.0; acci[j] = 0.0; }
        const cplx<T> *bx = Bas + x * (int64_t)vb * nb, *fx = F + x * (int64_t)vb * s;
        for (int v0 = 0; v0 < vb; v0 += rows_per_tile) {
            const int nrow = (vb - v0 < rows_per_tile) ? (vb - v0) : rows_per_tile;
            __syncthreads();
            for (int e = threadIdx.x; e < nrow * nb; e += kLaThreads) sB[e] = bx[(int64_t)v0 * nb + e];
            for (int e = threadIdx.x; e < nrow * s; e += kLaThreads) sF[e] = fx[(int64_t)v0 * s + e];
            __syncthreads();
#pragma unroll
            for (int j = 0; j < MAXE; ++j) {
                if (ek[j] < 0) continue;
                cplx<T> run = {0, 0};
                for (int v = 0; v < nrow; ++v) cmac_conj(run, sB[v * nb + ek[j]], sF[v * s + er[j]]);
                accr[j] += (double)run.re; acci[j] += (double)run.im;
            }
        }
        cplx<T> *cx = Cc + x * (int64_t)ms;
#pragma unroll
        for (int j = 0; j < MAXE; ++j)
            if (ek[j] >= 0) cx[threadIdx.x + j * kLaThreads] = {(T)accr[j], (T)acci[j]};
    }
}

template <typename T>
__global__ void __launch_bounds__(kLaThreads)
block_promote_kernel(const cplx<T> *__restrict__ Bas, const cplx<T> *__restrict__ Cc, cplx<T> *__restrict__ F, int64_t Vc, int vb, int nb, int s,
                     int rows_per_tile)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx<T> *sC = reinterpret_cast<cplx<T> *>(smem_raw);          // [nb][s]
    cplx<T> *sB = sC + nb * s;                                     // [rows_per_tile][nb + 1]
    const int ld = nb + 1;
    for (int64_t x = blockIdx.x; x < Vc; x += gridDim.x) {
        const cplx<T> *bx = Bas + x * (int64_t)vb * nb;
        cplx<T> *fx = F + x * (int64_t)vb * s;
        __syncthreads();
        for (int e = threadIdx.x; e < nb * s; e += kLaThreads) sC[e] = Cc[x * (int64_t)nb * s + e];
        for (int v0 = 0; v0 < vb; v0 += rows_per_tile) {
            const int nrow = (vb - v0 < rows_per_tile) ? (vb - v0) : rows_per_tile;
            __syncthreads();
            for (int e = threadIdx.x; e < nrow * nb; e += kLaThreads) sB[(e / nb) * ld + e % nb] = bx[(int64_t)v0 * nb + e];
            __syncthreads();
            for (int e = threadIdx.x; e < nrow * s; e += kLaThreads) {
                const int v = e / s, r = e - v * s;
                cplx<T> acc = {0, 0};
                for (int k = 0; k < nb; ++k) cmac(acc, sB[v * ld + k], sC[k * s + r]);
                fx[(int64_t)v0 * s + e] = acc;
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------------
// Tuned forms of the two transfer kernels for nbasis and nrhs multiples of 4 (Table 6's shapes: nbasis 64 x nrhs 12 x V_block 256,
// PAPER.md:570-571).  The kernels above do one output element per thread and two shared-memory loads per multiply-add
// (measured: 1.3-1.5 TB/s = 0.2 of the HBM roof); these keep 4 x 4 (project) / TR x 4 (promote) complex results per thread.
//
// project: C[x] = Basis[x]^dagger F[x] is a rectangular Gram product per coarse site.  Thread tile 4 x 4; the (nb/4)(s/4) tiles of
// a site are one GROUP of threads, and the G groups of a CTA work on G DIFFERENT sites at once (no reduction between groups, every
// group runs all rows of its own tile).  A stage of the 3-stage ring holds `rows` rows of Basis[x] and F[x] for each of the G sites --
// 2 G bulk copies of contiguous ranges, issued by a producer warp; full / empty mbarriers per stage, no CTA-wide barrier in the loop --
// and the ring runs on across the CTA's sites.
// Sums: products and runs of <= 32 rows in T, the runs added into the site's accumulator -- in double for complex128; for
// complex64 in float (two-level summation: error <= (32 + V_block/32) eps, 1e-6 at V_block 3072 against the 1e-5 bar).
// ------------------------------------------------------------------------------------------------------
constexpr int kXferConsumers = kLaThreads - 32;   // 7 consumer warps + one producer warp = kLaThreads (two CTAs per SM keep 128 registers per thread)

template <typename T>
__global__ void __launch_bounds__(kLaThreads, 2)
block_project_pipe_kernel(const cplx<T> *__restrict__ Bas, const cplx<T> *__restrict__ F, cplx<T> *__restrict__ Cc, int64_t Vc, int vb, int nb, int s,
                          int rows, int G, int flush_tiles)
{
    constexpr int TT = 4;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int ntb = s / TT, ntile = (nb / TT) * ntb;
    const size_t bytesB = (size_t)rows * nb * sizeof(cplx<T>), bytesF = (size_t)rows * s * sizeof(cplx<T>);
    const size_t site_stage = bytesB + bytesF, stage_bytes = (size_t)G * site_stage;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + kGramPipeStages * stage_bytes), *empty = full + kGramPipeStages;
    const int tile = threadIdx.x % ntile, g = threadIdx.x / ntile;
    const int a0 = (tile / ntb) * TT, b0 = (tile % ntb) * TT;

    const int tps = (vb + rows - 1) / rows;                                   // tiles per site
    // round j of this CTA: the G consecutive sites from (j gridDim + blockIdx) G
    const int64_t nchunk = (Vc + G - 1) / G;                                  // chunks of G sites
    const int64_t my_rounds = (int64_t)blockIdx.x < nchunk ? (nchunk - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    const int64_t total = my_rounds * tps;
    if (threadIdx.x == 0) {
        for (int st = 0; st < kGramPipeStages; ++st) { mbar_init(&full[st], 1); mbar_init(&empty[st], kXferConsumers / 32); }
        mbar_fence_init();
    }
    __syncthreads();
    auto issue = [&](int64_t i, uint64_t pol) {   // one thread
        const int st = (int)(i % kGramPipeStages);
        const int64_t base = ((i / tps) * gridDim.x + blockIdx.x) * G;
        const int nv = (int)((Vc - base < G) ? (Vc - base) : G);
        const int v0 = (int)(i % tps) * rows, nrow = (vb - v0 < rows) ? (vb - v0) : rows;
        const uint32_t nB = (uint32_t)((size_t)nrow * nb * sizeof(cplx<T>)), nF = (uint32_t)((size_t)nrow * s * sizeof(cplx<T>));
        mbar_arrive_expect_tx(&full[st], (uint32_t)nv * (nB + nF));
        for (int q = 0; q < nv; ++q) {
            unsigned char *dst = smem_raw + (size_t)st * stage_bytes + (size_t)q * site_stage;
            bulk_g2s(dst, Bas + ((base + q) * vb + v0) * (int64_t)nb, nB, &full[st], pol);
            bulk_g2s(dst + bytesB, F + ((base + q) * vb + v0) * (int64_t)s, nF, &full[st], pol);
        }
    };
    if (threadIdx.x >= kXferConsumers) {
        // ---- producer warp: refills a stage as soon as the 7 consumer warps have released it ----
        if (threadIdx.x == kXferConsumers) {
            const uint64_t pol = l2_policy_evict_first();
            for (int64_t i = 0; i < total; ++i) {
                const int st = (int)(i % kGramPipeStages);
                if (i >= kGramPipeStages) mbar_wait(&empty[st], (uint32_t)((i / kGramPipeStages - 1) & 1));
                issue(i, pol);
            }
        }
        return;
    }

    using Acc = typename std::conditional<sizeof(T) == 8, double, T>::type;
    Acc accr[TT][TT], acci[TT][TT];
    cplx<T> run[TT][TT];
#pragma unroll
    for (int a = 0; a < TT; ++a)
#pragma unroll
        for (int b = 0; b < TT; ++b) { accr[a][b] = 0; acci[a][b] = 0; run[a][b].re = 0; run[a][b].im = 0; }

    int st = 0, since_flush = 0;
    uint32_t parity = 0;
    for (int64_t i = 0; i < total; ++i) {
        const int t = (int)(i % tps), v0 = t * rows, nrow = (vb - v0 < rows) ? (vb - v0) : rows;
        const int64_t x = ((i / tps) * gridDim.x + blockIdx.x) * G + g;
        const bool mine = g < G && x < Vc;
        mbar_wait(&full[st], parity);
        if (mine) {
            const cplx<T> *sB = reinterpret_cast<const cplx<T> *>(smem_raw + (size_t)st * stage_bytes + (size_t)g * site_stage);
            const cplx<T> *sF = reinterpret_cast<const cplx<T> *>(smem_raw + (size_t)st * stage_bytes + (size_t)g * site_stage + bytesB);
            for (int k = 0; k < nrow; ++k) {
                cplx<T> u[TT], w[TT];
                gram_pipe_load<T, TT>(u, sB + k * nb + a0);
                gram_pipe_load<T, TT>(w, sF + k * s + b0);
#pragma unroll
                for (int a = 0; a < TT; ++a)
#pragma unroll
                    for (int b = 0; b < TT; ++b) {
                        if constexpr (sizeof(T) == 8) {       // complex128: the sums are double already, no runs
                            accr[a][b] = fma(u[a].re, w[b].re, accr[a][b]); accr[a][b] = fma(u[a].im, w[b].im, accr[a][b]);
                            acci[a][b] = fma(u[a].re, w[b].im, acci[a][b]); acci[a][b] = fma(-u[a].im, w[b].re, acci[a][b]);
                        } else {
                            cmac_conj(run[a][b], u[a], w[b]);
                        }
                    }
            }
        }
        const bool last = t == tps - 1;
        if (sizeof(T) == 4 && (++since_flush == flush_tiles || last)) {
#pragma unroll
            for (int a = 0; a < TT; ++a)
#pragma unroll
                for (int b = 0; b < TT; ++b) {
                    accr[a][b] += (Acc)run[a][b].re; acci[a][b] += (Acc)run[a][b].im;
                    run[a][b].re = 0; run[a][b].im = 0;
                }
            since_flush = 0;
        }
        if (last) {                               // the site is complete: every thread writes its own 4 x 4 block
            if (mine) {
                cplx<T> *cx = Cc + x * (int64_t)nb * s;
#pragma unroll
                for (int a = 0; a < TT; ++a)
#pragma unroll
                    for (int b = 0; b < TT; ++b) cx[(a0 + a) * s + b0 + b] = {(T)accr[a][b], (T)acci[a][b]};
            }
#pragma unroll
            for (int a = 0; a < TT; ++a)
#pragma unroll
                for (int b = 0; b < TT; ++b) { accr[a][b] = 0; acci[a][b] = 0; }
        }
        __syncwarp();
        if ((threadIdx.x & 31) == 0) mbar_arrive(&empty[st]);          // this warp has read the stage
        if (++st == kGramPipeStages) { st = 0; parity ^= 1u; }
    }
}

// promote: F[x] = Basis[x] C[x], rows of the fine block times a small matrix.  Thread tile TR rows x 4 columns, lanes along the rows;
// row tiles of Basis[x] go through cp.async into rows padded by LaPad (a warp's 16-byte loads of consecutive rows then meet
// different banks), double buffered across the CTA's sites, C[x] rides along with a site's first tile; two contraction indices per
// shared-memory load for complex64.  Sums over nbasis <= 64 terms in T.
template <typename T, int TR>
__global__ void __launch_bounds__(kLaThreads)
block_promote_tiled_kernel(const cplx<T> *__restrict__ Bas, const cplx<T> *__restrict__ Cc, cplx<T> *__restrict__ F, int64_t Vc, int vb, int nb, int s,
                           int RL)
{
    constexpr int W = 4, AV = 16 / (int)sizeof(cplx<T>);            // contraction indices per 16-byte load: 2 (complex64) or 1
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int ld = nb + LaPad<T>::v, rows = RL * TR, ncg = s / W;
    cplx<T> *sC0 = reinterpret_cast<cplx<T> *>(smem_raw);            // [2][nb * s]
    cplx<T> *sB0 = sC0 + (size_t)2 * nb * s;                         // [2][rows * ld]
    const int cg = threadIdx.x / RL, rl = threadIdx.x - cg * RL, c0 = cg * W;
    const bool active = cg < ncg;
    const int tps = (vb + rows - 1) / rows;
    const int64_t my_sites = (int64_t)blockIdx.x < Vc ? (Vc - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    const int64_t total = my_sites * tps;
    auto stage = [&](int64_t i, int buf) {
        const int64_t n = i / tps, x = blockIdx.x + n * gridDim.x;
        const int t = (int)(i - n * tps), v0 = t * rows, nrow = (vb - v0 < rows) ? (vb - v0) : rows;
        la_stage_rows_async(sB0 + (size_t)buf * rows * ld, Bas + x * (int64_t)vb * nb, v0, nrow, rows, nb, ld);
        if (t == 0) {                             // the site's coarse block, 16-byte chunks (nb * s is a multiple of 16 elements)
            cplx<T> *dst = sC0 + (size_t)(n & 1) * nb * s;
            const cplx<T> *src = Cc + x * (int64_t)nb * s;
            for (int e = threadIdx.x * AV; e < nb * s; e += kLaThreads * AV) cp_async_16(dst + e, src + e);
        }
    };
    if (total > 0) stage(0, 0);
    cp_async_commit();
    int buf = 0;
    for (int64_t i = 0; i < total; ++i, buf ^= 1) {
        if (i + 1 < total) stage(i + 1, buf ^ 1);
        cp_async_commit();
        cp_async_wait<1>();
        __syncthreads();
        const int64_t n = i / tps, x = blockIdx.x + n * gridDim.x;
        const int t = (int)(i - n * tps), v0 = t * rows, nrow = (vb - v0 < rows) ? (vb - v0) : rows;
        if (active) {
            const cplx<T> *sB = sB0 + (size_t)buf * rows * ld, *sC = sC0 + (size_t)(n & 1) * nb * s;
            cplx<T> acc[TR][W];
#pragma unroll
            for (int tt = 0; tt < TR; ++tt)
#pragma unroll
                for (int c = 0; c < W; ++c) { acc[tt][c].re = 0; acc[tt][c].im = 0; }
#pragma unroll 2
            for (int a = 0; a < nb; a += AV) {
                cplx<T> u[TR][AV], k[AV][W];
#pragma unroll
                for (int tt = 0; tt < TR; ++tt) gram_pipe_load<T, AV>(u[tt], sB + (rl + tt * RL) * ld + a);
#pragma unroll
                for (int j = 0; j < AV; ++j) gram_pipe_load<T, W>(k[j], sC + (a + j) * s + c0);
#pragma unroll
                for (int j = 0; j < AV; ++j)
#pragma unroll
                    for (int tt = 0; tt < TR; ++tt)
#pragma unroll
                        for (int c = 0; c < W; ++c) cmac(acc[tt][c], u[tt][j], k[j][c]);
            }
            cplx<T> *fx = F + (x * vb + v0) * (int64_t)s + c0;
#pragma unroll
            for (int tt = 0; tt < TR; ++tt) {
                const int row = rl + tt * RL;
                if (row < nrow) {
#pragma unroll
                    for (int c = 0; c < W; c += AV)
                        *reinterpret_cast<float4 *>(fx + (int64_t)row * s + c) = *reinterpret_cast<const float4 *>(&acc[tt][c]);
                }
            }
        }
        __syncthreads();                          // the buffer may be restaged
    }
    cp_async_wait<0>();
}

// out = a*U + b*W elementwise (used for R = B - H X and copies)
template <typename T>
__global__ void axpby_kernel(const cplx<T> *U, const cplx<T> *W, cplx<T> *out, T a, T b, int64_t total)
{
    for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        cplx<T> v;
        v.re = a * U[e].re + b * W[e].re;
        v.im = a * U[e].im + b * W[e].im;
        out[e] = v;
    }
}

// ------------------------------------------------------------------------------------------------------
// s x s complex128 algebra, one CTA, matrices in shared memory (row-major, leading dimension s).
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ zdouble zmul(zdouble a, zdouble b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
__device__ __forceinline__ zdouble zmulc(zdouble a, zdouble b) { return {a.re * b.re + a.im * b.im, a.re * b.im - a.im * b.re}; }   // conj(a)*b

__device__ void sm_load(zdouble *dst, const zdouble *src, int ss)
{
    for (int e = threadIdx.x; e < ss; e += blockDim.x) dst[e] = src[e];
    __syncthreads();
}
__device__ void sm_store(zdouble *dst, const zdouble *src, int ss)
{
    __syncthreads();
    for (int e = threadIdx.x; e < ss; e += blockDim.x) dst[e] = src[e];
}

// In place: G (Hermitian positive definite, symmetrised from its upper triangle and the conjugate of its lower)
// -> S upper triangular, positive real diagonal, G = S^H S; strict lower part zeroed.  *flag set on a bad pivot.
__device__ void sm_cholesky_upper(zdouble *G, int s, int *flag)
{
    for (int e = threadIdx.x; e < s * s; e += blockDim.x) {
        const int a = e / s, b = e % s;
        if (a < b) {
            const zdouble u = G[a * s + b], l = G[b * s + a];
            G[a * s + b] = {0.5 * (u.re + l.re), 0.5 * (u.im - l.im)};
        }
    }
    __syncthreads();
    for (int e = threadIdx.x; e < s * s; e += blockDim.x) {
        const int a = e / s, b = e % s;
        if (a > b) G[e] = {0.0, 0.0};
        if (a == b) G[e].im = 0.0;
    }
    __syncthreads();
    for (int a = 0; a < s; ++a) {
        const double d = G[a * s + a].re;
        if (!(d > 0.0) || !isfinite(d)) {
            if (threadIdx.x == 0) *flag = 1;
            __syncthreads();
            return;
        }
        const double saa = sqrt(d);
        __syncthreads();
        for (int b = a + threadIdx.x; b < s; b += blockDim.x) {
            if (b == a) G[a * s + a] = {saa, 0.0};
            else { G[a * s + b].re /= saa; G[a * s + b].im /= saa; }
        }
        __syncthreads();
        // trailing update of the upper triangle: G[c][b] -= conj(S[a][c]) S[a][b], a < c <= b
        const int m = s - a - 1;
        for (int e = threadIdx.x; e < m * m; e += blockDim.x) {
            const int c = a + 1 + e / m, b = a + 1 + e % m;
            if (b >= c) {
                const zdouble t = zmulc(G[a * s + c], G[a * s + b]);
                G[c * s + b].re -= t.re;
                G[c * s + b].im -= t.im;
            }
        }
        __syncthreads();
    }
}

// Sinv = S^-1 for upper triangular S (thread b does column b by back substitution)
__device__ void sm_upper_inverse(const zdouble *S, zdouble *Sinv, int s)
{
    for (int e = threadIdx.x; e < s * s; e += blockDim.x) Sinv[e] = {0.0, 0.0};
    __syncthreads();
    for (int b = threadIdx.x; b < s; b += blockDim.x) {
        for (int a = b; a >= 0; --a) {
            zdouble acc = {(a == b) ? 1.0 : 0.0, 0.0};
            for (int c = a + 1; c <= b; ++c) {
                const zdouble t = zmul(S[a * s + c], Sinv[c * s + b]);
                acc.re -= t.re;
                acc.im -= t.im;
            }
            const double d = S[a * s + a].re;       // real positive diagonal
            Sinv[a * s + b] = {acc.re / d, acc.im / d};
        }
    }
    __syncthreads();
}

// R = op(P) Q with op = identity (adjP = 0) or conjugate transpose (adjP = 1); R must not alias P or Q
__device__ void sm_matmul(const zdouble *P, const zdouble *Q, zdouble *R, int s, int adjP, int adjQ)
{
    for (int e = threadIdx.x; e < s * s; e += blockDim.x) {
        const int a = e / s, b = e % s;
        double re = 0.0, im = 0.0;
        for (int c = 0; c < s; ++c) {
            zdouble p = adjP ? zdouble{P[c * s + a].re, -P[c * s + a].im} : P[a * s + c];
            zdouble q = adjQ ? zdouble{Q[b * s + c].re, -Q[b * s + c].im} : Q[c * s + b];
            re += p.re * q.re - p.im * q.im;
            im += p.re * q.im + p.im * q.re;
        }
        R[e] = {re, im};
    }
    __syncthreads();
}

// G -> S (and optionally S^-1).  info: 0 or COARSE_BREAKDOWN.
__global__ void small_cholesky_kernel(const zdouble *G, zdouble *S, zdouble *Sinv, int s, int32_t *info)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    zdouble *m0 = reinterpret_cast<zdouble *>(smem_raw), *m1 = m0 + s * s;
    __shared__ int flag;
    if (threadIdx.x == 0) flag = 0;
    sm_load(m0, G, s * s);
    sm_cholesky_upper(m0, s, &flag);
    __syncthreads();
    if (flag) { if (threadIdx.x == 0) *info = COARSE_BREAKDOWN; return; }
    sm_store(S, m0, s * s);
    if (Sinv) { sm_upper_inverse(m0, m1, s); sm_store(Sinv, m1, s * s); }
    if (threadIdx.x == 0) *info = 0;
}

// M = G^-1 = S^-1 S^-H
__global__ void small_hpd_inverse_kernel(const zdouble *G, zdouble *M, int s, int32_t *info)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    zdouble *m0 = reinterpret_cast<zdouble *>(smem_raw), *m1 = m0 + s * s;
    __shared__ int flag;
    if (threadIdx.x == 0) flag = 0;
    sm_load(m0, G, s * s);
    sm_cholesky_upper(m0, s, &flag);
    __syncthreads();
    if (flag) { if (threadIdx.x == 0) *info = COARSE_BREAKDOWN; return; }
    sm_upper_inverse(m0, m1, s);
    sm_matmul(m1, m1, m0, s, 0, 1);      // Sinv * Sinv^H
    sm_store(M, m0, s * s);
    if (threadIdx.x == 0) *info = 0;
}

// Device-resident scalars/matrices of one block-CG solve (all complex128 / double)
struct BcgSmall {
    zdouble *G;       // Gram result (input of every small kernel)
    zdouble *C;       // C_k
    zdouble *K1;      // M C    (X update coefficient)   | C_0^-1 at init
    zdouble *K2;      // -M     (T = Q - Z M)
    zdouble *K3;      // S^-1
    zdouble *K4;      // S^H
    double *bnorm;    // ||B[:,r]||  (1 where the source column is zero)
    double *relres;   // [s] recursive relative residuals
    double *stop;     // [0] = max_r relres, [1] = 0 ok, else where the FIRST breakdown happened: 1 initial QR, 2 D^H Z, 3 T^H T
};

// bnorm[r] = sqrt(G[r][r]) from G = B^H B
__global__ void bcg_bnorm_kernel(BcgSmall w, int s)
{
    for (int r = threadIdx.x; r < s; r += blockDim.x) {
        const double v = sqrt(fmax(w.G[r * s + r].re, 0.0));
        w.bnorm[r] = (v == 0.0) ? 1.0 : v;
    }
}

// init: G = R^H R.  relres[r] = sqrt(G[r][r])/bnorm[r]; stop[0] = max; if max > tol: C = chol(G), K1 = C^-1
__global__ void bcg_init_kernel(BcgSmall w, int s, double tol)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    zdouble *m0 = reinterpret_cast<zdouble *>(smem_raw), *m1 = m0 + s * s;
    __shared__ int flag;
    __shared__ double worst;
    if (threadIdx.x == 0) {
        flag = 0;
        double m = 0.0;
        for (int r = 0; r < s; ++r) {
            const double rel = sqrt(fmax(w.G[r * s + r].re, 0.0)) / w.bnorm[r];
            w.relres[r] = rel;
            m = fmax(m, rel);
        }
        worst = m;
        w.stop[0] = m;
        w.stop[1] = 0.0;
    }
    sm_load(m0, w.G, s * s);
    if (worst <= tol) return;
    sm_cholesky_upper(m0, s, &flag);
    __syncthreads();
    if (flag) { if (threadIdx.x == 0) w.stop[1] = 1.0; return; }
    sm_store(w.C, m0, s * s);
    sm_upper_inverse(m0, m1, s);
    sm_store(w.K1, m1, s * s);
}

// step 1: G = D^H Z.  M = G^-1;  K1 = M C;  K2 = -M.
__global__ void bcg_step1_kernel(BcgSmall w, int s)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    zdouble *m0 = reinterpret_cast<zdouble *>(smem_raw), *m1 = m0 + s * s, *m2 = m1 + s * s;
    __shared__ int flag;
    if (threadIdx.x == 0) flag = (w.stop[1] != 0.0) ? 1 : 0;       // an earlier breakdown freezes the iteration
    sm_load(m0, w.G, s * s);
    if (!flag) sm_cholesky_upper(m0, s, &flag);
    __syncthreads();
    if (flag) {
        // breakdown contract (coarse_mrhs.h): the block passes already enqueued behind this kernel must leave X at the last
        // valid iterate: K1 = K2 = 0  =>  X += 0,  T = Q
        for (int e = threadIdx.x; e < s * s; e += blockDim.x) { w.K1[e] = {0.0, 0.0}; w.K2[e] = {0.0, 0.0}; }
        if (threadIdx.x == 0 && w.stop[1] == 0.0) w.stop[1] = 2.0;      // 2: D^H Z not positive definite (statement 9)
        return;
    }
    sm_upper_inverse(m0, m1, s);
    sm_matmul(m1, m1, m0, s, 0, 1);          // m0 = M
    sm_load(m2, w.C, s * s);
    sm_matmul(m0, m2, m1, s, 0, 0);          // m1 = M C
    sm_store(w.K1, m1, s * s);
    for (int e = threadIdx.x; e < s * s; e += blockDim.x) w.K2[e] = {-m0[e].re, -m0[e].im};
}

// step 2: G = T^H T.  S = chol(G);  K3 = S^-1;  K4 = S^H;  C <- S C;  relres, stop
__global__ void bcg_step2_kernel(BcgSmall w, int s)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    zdouble *m0 = reinterpret_cast<zdouble *>(smem_raw), *m1 = m0 + s * s, *m2 = m1 + s * s;
    __shared__ int flag;
    if (threadIdx.x == 0) flag = (w.stop[1] != 0.0) ? 1 : 0;
    sm_load(m0, w.G, s * s);
    if (!flag) sm_cholesky_upper(m0, s, &flag);
    __syncthreads();
    if (flag) {
        // breakdown contract: K3 = I, K4 = 0  =>  Q = T, D = Q (well defined, X untouched); C and the residuals keep their last values
        for (int e = threadIdx.x; e < s * s; e += blockDim.x) {
            w.K3[e] = {(e / s == e % s) ? 1.0 : 0.0, 0.0};
            w.K4[e] = {0.0, 0.0};
        }
        if (threadIdx.x == 0 && w.stop[1] == 0.0) w.stop[1] = 3.0;      // 3: T^H T not positive definite (statement 11)
        return;
    }
    sm_upper_inverse(m0, m1, s);
    sm_store(w.K3, m1, s * s);
    for (int e = threadIdx.x; e < s * s; e += blockDim.x) {
        const int a = e / s, b = e % s;
        w.K4[e] = {m0[b * s + a].re, -m0[b * s + a].im};
    }
    sm_load(m2, w.C, s * s);
    sm_matmul(m0, m2, m1, s, 0, 0);          // m1 = S C
    sm_store(w.C, m1, s * s);
    __syncthreads();
    if (threadIdx.x == 0) {
        double m = 0.0;
        for (int r = 0; r < s; ++r) {
            double acc = 0.0;
            for (int a = 0; a < s; ++a) acc += m1[a * s + r].re * m1[a * s + r].re + m1[a * s + r].im * m1[a * s + r].im;
            const double rel = sqrt(acc) / w.bnorm[r];
            w.relres[r] = rel;
            m = fmax(m, rel);
        }
        w.stop[0] = m;
    }
}

// ---- Preconditioned BlockCGrQ (Fig. 2 right): the small kernels that differ from the plain ones ----
// relres[r] = sqrt(G[r][r]) / bnorm[r] from G = z_0^H z_0; stop[0] = max, stop[1] = 0
__global__ void pbcg_rel0_kernel(BcgSmall w, int s)
{
    if (threadIdx.x == 0) {
        double m = 0.0;
        for (int r = 0; r < s; ++r) {
            const double rel = sqrt(fmax(w.G[r * s + r].re, 0.0)) / w.bnorm[r];
            w.relres[r] = rel;
            m = fmax(m, rel);
        }
        w.stop[0] = m;
        w.stop[1] = 0.0;
    }
}
// G = Z_0^H z_0 = <Z_0|Z_0>_M:  C_0 = chol(G),  K1 = C_0^-1
__global__ void pbcg_init_kernel(BcgSmall w, int s)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    zdouble *m0 = reinterpret_cast<zdouble *>(smem_raw), *m1 = m0 + s * s;
    __shared__ int flag;
    if (threadIdx.x == 0) flag = 0;
    sm_load(m0, w.G, s * s);
    sm_cholesky_upper(m0, s, &flag);
    __syncthreads();
    if (flag) { if (threadIdx.x == 0) w.stop[1] = 1.0; return; }
    sm_store(w.C, m0, s * s);
    sm_upper_inverse(m0, m1, s);
    sm_store(w.K1, m1, s * s);
}
// Euclidean residual r_k = q_k C_k:  relres[r] = sqrt((C^H G C)_rr) / bnorm[r] with G = q^H q;  stop[0] = max
__global__ void pbcg_resid_kernel(BcgSmall w, int s)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    zdouble *m0 = reinterpret_cast<zdouble *>(smem_raw), *m1 = m0 + s * s, *m2 = m1 + s * s;
    sm_load(m0, w.G, s * s);
    sm_load(m1, w.C, s * s);
    sm_matmul(m0, m1, m2, s, 0, 0);          // m2 = G C
    __shared__ double rel[COARSE_MAX_NRHS];
    for (int r = threadIdx.x; r < s; r += blockDim.x) {
        double acc = 0.0;                     // Re (C^H G C)_rr = Re sum_a conj(C[a][r]) (G C)[a][r]
        for (int a = 0; a < s; ++a) acc += m1[a * s + r].re * m2[a * s + r].re + m1[a * s + r].im * m2[a * s + r].im;
        rel[r] = sqrt(fmax(acc, 0.0)) / w.bnorm[r];
        w.relres[r] = rel[r];
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double m = 0.0;
        for (int r = 0; r < s; ++r) m = fmax(m, rel[r]);
        w.stop[0] = m;
    }
}

// column norms of a block from the diagonal of its Gram matrix: out[r] = sqrt(G[r][r]) / bnorm[r]
__global__ void bcg_truerel_kernel(BcgSmall w, int s, double *out)
{
    for (int r = threadIdx.x; r < s; r += blockDim.x) out[r] = sqrt(fmax(w.G[r * s + r].re, 0.0)) / w.bnorm[r];
}

}  // namespace cmrhs

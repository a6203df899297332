// Block-CG linear algebra on the tensor cores (complex64, wide blocks): the block rotation  out = beta Vin + U K  and the Gram
// product  G = U^H W  (Table 6 "ThinQR"), in the split-FP16 arithmetic of the
// stencil kernels (hi + 2^-11 lo in binary16 after power-of-two scalings, three tcgen05 products, FP32 accumulators in TMEM).
// At nrhs >= 32 the SIMT kernels of blockcg_kernels.cuh are FP32-pipe bound (8 n s^2 flops per product: 31 TFLOP/s reached,
// the linear algebra of an iteration cost more than the stencil apply at nrhs 64); here they are HBM-bound passes.
//
// A complex block [n][s] is the real matrix [n][2 s] it is in memory (column (r, re/im)), and the complex s x s matrix K the real
// 2s x 2s matrix Kr[(r,c)][(r',c')] = {Re K, Im K; -Im K, Re K}: 4 real multiply-adds per complex one, no padding flops.
//
// Rotation (trot_kernel), per tile of 64 rows:   D[(r',c')][row] = sum_(r,c) Kr^T[(r',c')][(r,c)] . U[row][(r,c)]
//   M side = Kr^T, constant: written ONCE into tensor memory (tcgen05.mma with the A operand from TMEM), one power-of-two scale
//   per output column; N side = the tile of U, converted on the fly to [U_hi ; U_lo] (K-major core matrices in shared memory,
//   one power-of-two scale per tile); MMA 1: Kr_hi . [U_hi ; U_lo] -> D | C, MMA 2: Kr_lo . U_hi -> C per K = 16 slab.
//   The accumulator has the OUTPUT COLUMN on the TMEM lanes, so the epilogue's stores are coalesced rows of 2 s floats.
// Gram (tgram_kernel): see below.
#pragma once

#include "stencil_h16x.cuh"

namespace cmrhs {

constexpr int kTlaThreads = 256;
constexpr int kTlaRows = 64;                          // rows of a tile
constexpr uint32_t kTlaLbo = 2 * kTlaRows * 16 + 16;  // bytes between k chunks of the converted tile: 16 row groups of 128 B, + 16 B so that
                                                      // the converter's stores spread over the banks

inline bool tla_supported(int s) { return s >= 16 && s <= 64 && s % 8 == 0; }

// power of two that maps a maximum (bit pattern of a non-negative float) into [2^13, 2^14): one bit of head room below the
// stencil kernels' [2^14, 2^15) because hi + lo of DIFFERENT elements are never added before the multiply here either; kept equal
__device__ __forceinline__ float tla_scale_from_bits(uint32_t bits) { return h_scale_from_bits(bits); }

struct TrotParams {
    const float *U;          // [n][2 s]
    const zdouble *K;        // [s][s] complex128, row major (device)
    const float *Vin;        // [n][2 s] or NULL (beta ignored)
    float *out;              // [n][2 s]; may alias U or Vin (a tile is read completely before it is written)
    float beta;
    int64_t n;
    int32_t s;
    uint32_t idesc_wide, idesc_lo;
};

__global__ void __launch_bounds__(kTlaThreads, 2) trot_kernel(const TrotParams P)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    unsigned char *tileB = smem_raw;                                   // [2 s / 8 chunks][kTlaLbo]
    const int N2 = 2 * P.s, nch = N2 / 8;
    float *inv_m = reinterpret_cast<float *>(tileB + (size_t)nch * kTlaLbo);      // [128] 1 / scale of output column m
    uint32_t *tmax = reinterpret_cast<uint32_t *>(inv_m + 128);                    // tile maximum (bit pattern)
    uint64_t *bar = reinterpret_cast<uint64_t *>(tmax + 2);
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(bar + 1);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) { mbar_init(bar, 1); mbar_fence_init(); *tmax = 0u; }
    if (warp == 4) tmem_alloc_cols(tmem_slot, 256u);
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();
    const uint32_t tmem = *tmem_slot;
    constexpr uint32_t kAcc = 0, kA = 128;             // TMEM columns: D 64 | C 64, then Kr^T hi (s columns) | lo (s columns)

    // ---- Kr^T into tensor memory, once: lane m = (r', c') holds Kr[(r,c)][(r',c')] for k = (r,c) = 0 .. 2s-1, two per column ----
    if (warp < 4) {
        const int m = 32 * warp + lane, rp = m >> 1, cp = m & 1;
        const bool live = m < N2;
        float mx = 0.f;
        if (live)
            for (int r = 0; r < P.s; ++r) { const zdouble z = P.K[r * P.s + rp]; mx = fmaxf(mx, fmaxf(fabsf((float)z.re), fabsf((float)z.im))); }
        const float sc = tla_scale_from_bits(__float_as_uint(mx));
        inv_m[m] = 1.0f / sc;
        const uint32_t lane_base = tmem + ((uint32_t)(32 * warp) << 16) + kA;
        for (int c8 = 0; c8 < P.s; c8 += 8) {          // 8 columns = 16 k = 8 complex r
            uint32_t hw[8], lw[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {              // column c8 + j: k = 2 (c8 + j), 2 (c8 + j) + 1  =  (r, 0), (r, 1) with r = c8 + j
                float a0 = 0.f, a1 = 0.f;
                if (live) {
                    const zdouble z = P.K[(c8 + j) * P.s + rp];
                    a0 = (cp == 0 ? (float)z.re : (float)z.im) * sc;          // c = 0:  Re K -> out_re,  Im K -> out_im
                    a1 = (cp == 0 ? -(float)z.im : (float)z.re) * sc;         // c = 1: -Im K -> out_re,  Re K -> out_im
                }
                const __half2 h = __floats2half2_rn(a0, a1);
                const float2 hf = __half22float2(h);
                const __half2 l = __floats2half2_rn((a0 - hf.x) * 2048.0f, (a1 - hf.y) * 2048.0f);
                hw[j] = *reinterpret_cast<const uint32_t *>(&h);
                lw[j] = *reinterpret_cast<const uint32_t *>(&l);
            }
            tmem_st_x8(lane_base + (uint32_t)c8, hw);
            tmem_st_x8(lane_base + (uint32_t)(P.s + c8), lw);
        }
        tmem_wait_st();
    }
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();

    const int64_t ntiles = (P.n + kTlaRows - 1) / kTlaRows;
    const int items = kTlaRows * nch;                  // 16-byte chunks of the converted tile (per half)
    uint32_t phase = 0;
    for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const int64_t row0 = t * kTlaRows;
        const int nrow = (int)(P.n - row0 < kTlaRows ? P.n - row0 : kTlaRows);
        // ---- load the tile (coalesced: consecutive threads, consecutive 32 bytes), tile maximum, convert, store as [U_hi ; U_lo] ----
        float v[4][8];
        uint32_t mx = 0u;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int item = threadIdx.x + kTlaThreads * i, row = item / nch, ch = item - row * nch;
            if (item < items && row < nrow) {
                const float4 a = *reinterpret_cast<const float4 *>(P.U + (row0 + row) * N2 + 8 * ch);
                const float4 b = *reinterpret_cast<const float4 *>(P.U + (row0 + row) * N2 + 8 * ch + 4);
                v[i][0] = a.x; v[i][1] = a.y; v[i][2] = a.z; v[i][3] = a.w; v[i][4] = b.x; v[i][5] = b.y; v[i][6] = b.z; v[i][7] = b.w;
            } else {
#pragma unroll
                for (int k = 0; k < 8; ++k) v[i][k] = 0.f;
            }
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const uint32_t b = __float_as_uint(v[i][k]) & 0x7FFFFFFFu;
                if (b <= 0x7F800000u) mx = max(mx, b);
            }
        }
        for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        if (lane == 0 && mx) atomicMax(tmax, mx);
        __syncthreads();
        const float tsc = tla_scale_from_bits(*tmax);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int item = threadIdx.x + kTlaThreads * i, row = item / nch, ch = item - row * nch;
            if (item >= items) continue;
            uint32_t hw[4], lw[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const float x0 = v[i][2 * u] * tsc, x1 = v[i][2 * u + 1] * tsc;
                const __half2 h = __floats2half2_rn(x0, x1);
                const float2 hf = __half22float2(h);
                const __half2 l = __floats2half2_rn((x0 - hf.x) * 2048.0f, (x1 - hf.y) * 2048.0f);
                hw[u] = *reinterpret_cast<const uint32_t *>(&h);
                lw[u] = *reinterpret_cast<const uint32_t *>(&l);
            }
            unsigned char *dst = tileB + (size_t)ch * kTlaLbo + (row >> 3) * 128 + (row & 7) * 16;
            *reinterpret_cast<uint4 *>(dst) = make_uint4(hw[0], hw[1], hw[2], hw[3]);
            *reinterpret_cast<uint4 *>(dst + (kTlaRows / 8) * 128) = make_uint4(lw[0], lw[1], lw[2], lw[3]);      // U_lo: n rows 64 .. 127
        }
        fence_proxy_async_smem();
        __syncthreads();
        // ---- MMAs: one thread ----
        if (threadIdx.x == 0) {
            *tmax = 0u;                                // (next tile's maximum; every thread has read this tile's)
            tc_fence_after_sync();
            const uint32_t b0 = smem_u32(tileB);
            const uint64_t desc_hi = umma_desc_kmajor_noswz(0u, kTlaLbo, 128u);
            for (int ks = 0; ks < N2 / 16; ++ks) {
                const uint64_t bd = desc_hi | (uint64_t)(((b0 + (uint32_t)ks * 2u * kTlaLbo) >> 4) & 0x3FFFu);
                umma_f16_ts(tmem + kAcc, tmem + kA + 8u * ks, bd, P.idesc_wide, ks ? 1u : 0u);            // Kr_hi . [U_hi ; U_lo] -> D | C
                umma_f16_ts(tmem + kAcc + 64u, tmem + kA + (uint32_t)P.s + 8u * ks, bd, P.idesc_lo, 1u);   // Kr_lo . U_hi -> C
            }
            umma_commit(bar);
        }
        mbar_wait(bar, phase);
        phase ^= 1u;
        tc_fence_after_sync();
        // ---- epilogue: lane = output column m, TMEM column = row of the tile; 8 warps: two per lane quarter, 32 rows each ----
        {
            const int q = warp & 3, half = warp >> 2, m = 32 * q + lane;
            const float sc = inv_m[m] / tsc;
            const uint32_t lane_base = tmem + ((uint32_t)(32 * q) << 16) + kAcc + (uint32_t)(32 * half);
            const bool mlive = m < N2;
            float vin[32];                             // all loads of Vin first: out may alias Vin, so the compiler keeps loads behind earlier stores
#pragma unroll
            for (int j = 0; j < 32; ++j) {
                const int row = 32 * half + j;
                vin[j] = (P.Vin && mlive && row < nrow) ? P.Vin[(row0 + row) * N2 + m] : 0.f;
            }
#pragma unroll
            for (int j8 = 0; j8 < 32; j8 += 8) {
                uint32_t d[8], c[8];
                tmem_ld_x8(lane_base + (uint32_t)j8, d);
                tmem_ld_x8(lane_base + 64u + (uint32_t)j8, c);
                tmem_wait_ld();
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    const int row = 32 * half + j8 + k;
                    if (mlive && row < nrow)
                        P.out[(row0 + row) * N2 + m] = fmaf(P.beta, vin[j8 + k], (__uint_as_float(d[k]) + __uint_as_float(c[k]) * (1.0f / 2048.0f)) * sc);
                }
            }
        }
        tc_fence_before_sync();
        __syncthreads();                               // the tile and the accumulator are free again
        tc_fence_after_sync();
    }
    __syncthreads();
    if (warp == 4) tmem_dealloc_cols(tmem, 256u);
}

// ---- Gram product G = U^H W on the tensor cores -------------------------------------------------------------------------------
//   P[(r,c)][(r',c')] = sum_rows U[row][(r,c)] W[row][(r',c')]   (M = columns of U, N = columns of W, K = rows), then
//   G[r][r'] = P[(r,0)][(r',0)] + P[(r,1)][(r',1)] + i (P[(r,0)][(r',1)] - P[(r,1)][(r',0)]).
// Both operands are MN-major (the blocks' own memory order), converted tile by tile (64 rows) into the SWIZZLE_128B image the
// stencil kernel stencil_h16.cuh uses: MMA 1: U_hi^T . [W_hi | W_lo] -> D | C, MMA 2: U_lo^T . W_hi -> C per K = 16 rows.
// A CTA owns a contiguous range of rows (split-K) and keeps D, C in tensor memory across its tiles; it
// FLUSHES them into its float64 partial (global, read-modify-write by the owning thread: deterministic) every kTgFlushRows = 256
// rows -- the tensor core truncates when it adds into its FP32 accumulator, so a run of sums is kept short (reading R11) --
// and whenever a tile's magnitude leaves the range of the CTA's current power-of-two scales (one per operand).
constexpr int kTgFlushRows = 256;
constexpr uint32_t kTgAtom = kTlaRows * 128;          // one 64-column atom of a 64-row tile

struct TgramParams {
    const float *U, *W;      // [n][2 s]
    zdouble *partial;        // [grid][s][s]
    int64_t n;
    int32_t s, natoms;       // natoms = ceil(2 s / 64)
    uint32_t idesc_wide, idesc_lo;
};

__global__ void __launch_bounds__(kTlaThreads, 2) tgram_kernel(const TgramParams P)
{
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    unsigned char *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    unsigned char *uhi = smem, *ulo = uhi + 2 * kTgAtom;                         // U: always two atoms (M = 128)
    unsigned char *whi = ulo + 2 * kTgAtom, *wlo = whi + (size_t)P.natoms * kTgAtom;      // [W_hi | W_lo]: contiguous atoms
    uint32_t *tmax = reinterpret_cast<uint32_t *>(wlo + (size_t)P.natoms * kTgAtom);      // [2] tile maxima of U, W
    uint64_t *bar = reinterpret_cast<uint64_t *>(tmax + 2);
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(bar + 1);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int N2 = 2 * P.s, nch = N2 / 8, NP = 64 * P.natoms;

    if (threadIdx.x == 0) { mbar_init(bar, 1); mbar_fence_init(); tmax[0] = 0u; tmax[1] = 0u; }
    for (int e = threadIdx.x; e < (int)((4 + 2 * P.natoms) * kTgAtom / 16); e += kTlaThreads)      // padding columns / rows stay zero
        reinterpret_cast<uint4 *>(smem)[e] = make_uint4(0u, 0u, 0u, 0u);
    if (warp == 4) tmem_alloc_cols(tmem_slot, 256u);
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();
    const uint32_t tmem = *tmem_slot;

    const int64_t ntiles = (P.n + kTlaRows - 1) / kTlaRows;
    const int64_t per = (ntiles + gridDim.x - 1) / gridDim.x, t_begin = blockIdx.x * per, t_end = (t_begin + per < ntiles) ? t_begin + per : ntiles;
    zdouble *mine = P.partial + (size_t)blockIdx.x * P.s * P.s;
    const int items = kTlaRows * nch;
    uint32_t phase = 0;
    float su = 0.f, sw = 0.f;                          // current scales (0: none yet)
    int rows_acc = 0;                                  // rows accumulated in tensor memory since the last flush
    bool wrote = false;                                // the partial has been written at least once

    // flush: tensor memory -> float64 partial.  8 warps: two per lane quarter, half of the W columns each
    auto flush = [&]() {
        const int q = warp & 3, half = warp >> 2, m = 32 * q + lane, r = m >> 1;
        const float sc = 1.0f / (su * sw);
        const uint32_t lane_base = tmem + ((uint32_t)(32 * q) << 16);
        for (int n0 = half * (NP / 2); n0 < (half + 1) * (NP / 2); n0 += 8) {
            uint32_t d[8], c[8];
            tmem_ld_x8(lane_base + (uint32_t)n0, d);
            tmem_ld_x8(lane_base + (uint32_t)(NP + n0), c);
            tmem_wait_ld();
            float p[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) p[k] = (__uint_as_float(d[k]) + __uint_as_float(c[k]) * (1.0f / 2048.0f)) * sc;
#pragma unroll
            for (int k = 0; k < 8; k += 2) {           // columns (r', 0), (r', 1)
                const float o0 = __shfl_xor_sync(0xffffffffu, p[k], 1), o1 = __shfl_xor_sync(0xffffffffu, p[k + 1], 1);
                const int rp = (n0 + k) >> 1;
                if ((m & 1) == 0 && m < N2 && rp < P.s) {
                    zdouble g = {(double)p[k] + (double)o1, (double)p[k + 1] - (double)o0};
                    zdouble *dst = mine + (size_t)r * P.s + rp;
                    if (wrote) { const zdouble old = *dst; g.re += old.re; g.im += old.im; }
                    *dst = g;
                }
            }
        }
        tc_fence_before_sync();
        __syncthreads();
        tc_fence_after_sync();
        wrote = true;
        rows_acc = 0;
    };

    for (int64_t t = t_begin; t < t_end; ++t) {
        const int64_t row0 = t * kTlaRows;
        const int nrow = (int)(P.n - row0 < kTlaRows ? P.n - row0 : kTlaRows);
        float vu[4][8], vw[4][8];
        uint32_t mu = 0u, mw = 0u;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int item = threadIdx.x + kTlaThreads * i, row = item / nch, ch = item - row * nch;
            if (item < items && row < nrow) {
                const float4 a = *reinterpret_cast<const float4 *>(P.U + (row0 + row) * N2 + 8 * ch);
                const float4 b = *reinterpret_cast<const float4 *>(P.U + (row0 + row) * N2 + 8 * ch + 4);
                const float4 c = *reinterpret_cast<const float4 *>(P.W + (row0 + row) * N2 + 8 * ch);
                const float4 d = *reinterpret_cast<const float4 *>(P.W + (row0 + row) * N2 + 8 * ch + 4);
                vu[i][0] = a.x; vu[i][1] = a.y; vu[i][2] = a.z; vu[i][3] = a.w; vu[i][4] = b.x; vu[i][5] = b.y; vu[i][6] = b.z; vu[i][7] = b.w;
                vw[i][0] = c.x; vw[i][1] = c.y; vw[i][2] = c.z; vw[i][3] = c.w; vw[i][4] = d.x; vw[i][5] = d.y; vw[i][6] = d.z; vw[i][7] = d.w;
            } else {
#pragma unroll
                for (int k = 0; k < 8; ++k) { vu[i][k] = 0.f; vw[i][k] = 0.f; }
            }
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const uint32_t bu = __float_as_uint(vu[i][k]) & 0x7FFFFFFFu, bw = __float_as_uint(vw[i][k]) & 0x7FFFFFFFu;
                if (bu <= 0x7F800000u) mu = max(mu, bu);
                if (bw <= 0x7F800000u) mw = max(mw, bw);
            }
        }
        for (int o = 16; o > 0; o >>= 1) { mu = max(mu, __shfl_xor_sync(0xffffffffu, mu, o)); mw = max(mw, __shfl_xor_sync(0xffffffffu, mw, o)); }
        if (lane == 0) { if (mu) atomicMax(&tmax[0], mu); if (mw) atomicMax(&tmax[1], mw); }
        __syncthreads();
        const float tu = __uint_as_float(tmax[0]), tw = __uint_as_float(tmax[1]);
        // the CTA's scales map the magnitude they were set on to [2^10, 2^11): 4 bits of head room before binary16 overflows
        const bool rescale = su == 0.f || tu * su >= 32768.f || tw * sw >= 32768.f || rows_acc + kTlaRows > kTgFlushRows;
        if (rescale) {                                 // (uniform over the CTA: every thread reads the same maxima)
            if (rows_acc > 0) flush();
            const bool need = su == 0.f || tu * su >= 32768.f || tw * sw >= 32768.f;
            if (need) {
                su = h_scale_from_bits(tmax[0]) * (1.0f / 16.0f);
                sw = h_scale_from_bits(tmax[1]) * (1.0f / 16.0f);
            }
        }
        const bool first = rows_acc == 0;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int item = threadIdx.x + kTlaThreads * i, row = item / nch, ch = item - row * nch;
            if (item >= items) continue;
            uint32_t uh[4], ul[4], wh[4], wl[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const float x0 = vu[i][2 * u] * su, x1 = vu[i][2 * u + 1] * su, y0 = vw[i][2 * u] * sw, y1 = vw[i][2 * u + 1] * sw;
                const __half2 hx = __floats2half2_rn(x0, x1), hy = __floats2half2_rn(y0, y1);
                const float2 fx = __half22float2(hx), fy = __half22float2(hy);
                const __half2 lx = __floats2half2_rn((x0 - fx.x) * 2048.0f, (x1 - fx.y) * 2048.0f);
                const __half2 ly = __floats2half2_rn((y0 - fy.x) * 2048.0f, (y1 - fy.y) * 2048.0f);
                uh[u] = *reinterpret_cast<const uint32_t *>(&hx); ul[u] = *reinterpret_cast<const uint32_t *>(&lx);
                wh[u] = *reinterpret_cast<const uint32_t *>(&hy); wl[u] = *reinterpret_cast<const uint32_t *>(&ly);
            }
            // SWIZZLE_128B, MN-major: atom (64 columns) | k row (128 B) | 16-byte chunk XOR (k mod 8)
            const uint32_t off = (uint32_t)(ch >> 3) * kTgAtom + (uint32_t)row * 128u + ((((uint32_t)ch & 7u) ^ ((uint32_t)row & 7u)) << 4);
            *reinterpret_cast<uint4 *>(uhi + off) = make_uint4(uh[0], uh[1], uh[2], uh[3]);
            *reinterpret_cast<uint4 *>(ulo + off) = make_uint4(ul[0], ul[1], ul[2], ul[3]);
            *reinterpret_cast<uint4 *>(whi + off) = make_uint4(wh[0], wh[1], wh[2], wh[3]);
            *reinterpret_cast<uint4 *>(wlo + off) = make_uint4(wl[0], wl[1], wl[2], wl[3]);
        }
        fence_proxy_async_smem();
        __syncthreads();
        if (threadIdx.x == 0) {
            tmax[0] = 0u;
            tmax[1] = 0u;
            tc_fence_after_sync();
            const uint32_t a_hi = smem_u32(uhi), a_lo = smem_u32(ulo), b_w = smem_u32(whi);
            for (int ks = 0; ks < kTlaRows / 16; ++ks) {
                const uint32_t adv = (uint32_t)ks * 2048u;          // 16 k rows of 128 B
                umma_f16_ss(tmem, h_desc(a_hi + adv, kTgAtom), h_desc(b_w + adv, kTgAtom), P.idesc_wide, (first && ks == 0) ? 0u : 1u);      // U_hi^T [W_hi | W_lo] -> D | C
                umma_f16_ss(tmem + (uint32_t)NP, h_desc(a_lo + adv, kTgAtom), h_desc(b_w + adv, kTgAtom), P.idesc_lo, 1u);                  // U_lo^T W_hi -> C
            }
            umma_commit(bar);
        }
        mbar_wait(bar, phase);                         // (the tile buffers are rewritten next: the MMAs must have read them)
        phase ^= 1u;
        tc_fence_after_sync();
        rows_acc += kTlaRows;
    }
    if (rows_acc > 0) flush();
    if (!wrote) {                                      // a CTA without rows: its partial is zero
        for (int e = threadIdx.x; e < P.s * P.s; e += kTlaThreads) mine[e] = {0.0, 0.0};
    }
    __syncthreads();
    if (warp == 4) tmem_dealloc_cols(tmem, 256u);
}

inline int launch_tgram(const void *U, const void *W, zdouble *partial, int max_blocks, int64_t n, int s, int num_sms, cudaStream_t stream, int *blocks_out)
{
    TgramParams P;
    P.U = static_cast<const float *>(U);
    P.W = static_cast<const float *>(W);
    P.partial = partial;
    P.n = n;
    P.s = s;
    P.natoms = (2 * s + 63) / 64;
    P.idesc_wide = umma_idesc_f16_mn(128, 2 * 64 * P.natoms);
    P.idesc_lo = umma_idesc_f16_mn(128, 64 * P.natoms);
    const size_t smem = 1024 + (size_t)(4 + 2 * P.natoms) * kTgAtom + 8 + 8 + 16;
    CMRHS_SMEM_ATTR(tgram_kernel, smem);
    const int64_t ntiles = ceil_div(n, kTlaRows);
    int grid = (int)(ntiles < 2ll * num_sms ? ntiles : 2ll * num_sms);
    if (grid > max_blocks) grid = max_blocks;
    tgram_kernel<<<grid, kTlaThreads, smem, stream>>>(P);
    CMRHS_LAUNCH_CHECK();
    *blocks_out = grid;
    return COARSE_OK;
}

inline int launch_trot(const void *U, const zdouble *K, const void *Vin, void *out, double beta, int64_t n, int s, int num_sms, cudaStream_t stream)
{
    TrotParams P;
    P.U = static_cast<const float *>(U);
    P.K = K;
    P.Vin = static_cast<const float *>(Vin);
    P.out = static_cast<float *>(out);
    P.beta = Vin ? (float)beta : 0.0f;
    P.n = n;
    P.s = s;
    P.idesc_wide = umma_idesc_f16_kk(128, 2 * kTlaRows);
    P.idesc_lo = umma_idesc_f16_kk(128, kTlaRows);
    const size_t smem = (size_t)(2 * s / 8) * kTlaLbo + 128 * 4 + 8 + 8 + 16 + 128;
    CMRHS_SMEM_ATTR(trot_kernel, smem);
    const int64_t ntiles = ceil_div(n, kTlaRows);
    const int grid = (int)(ntiles < 2ll * num_sms ? ntiles : 2ll * num_sms);
    trot_kernel<<<grid, kTlaThreads, smem, stream>>>(P);
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}

}  // namespace cmrhs

// Tensor-core stencil-GEMM kernel for complex64 on sm_100a, split-FP16 (3 products, tcgen05.mma.kind::f16).
//   Y(x) = sum_{p=0}^{80} A^p(x) . X(x + delta_p)                       (Eq. 19)
//
// Same mapping as stencil_tc.cuh (two x-adjacent sites x (Re, Im) x 32 rows on the 128 TMEM lanes, N = the neighbour's
// X tile as the real nb x 2 nrhs matrix it is in memory, 110 MMA steps per pair of sites, centre point last), but the
// operands are pairs of binary16 numbers instead of TF32:
//   a  = sA a_true            (sA: one power of two per operator, max |a| -> [2^14, 2^15))
//   a  = hi + 2^-11 lo        hi = fp16(a), lo = fp16(2^11 (a - hi))      22-23 significant bits in the same 4 bytes
//   x  = sX_r x_true          (sX_r: one power of two per right-hand side column, from a max-abs pre-pass over X)
//   Y  = (D + 2^-11 C) / (sA sX_r),   D = A_hi X_hi,  C = A_hi X_lo + A_lo X_hi   (FP32 accumulators in TMEM)
// * The operator is stored ALREADY SPLIT in HBM (coarse_op_create, same 8 bytes per complex as complex64): a stencil
//   matrix is one 8 KB tile [hi 4 KB | lo 4 KB], each half the MN-major SWIZZLE_128B shared-memory image of the
//   64 x 32 (M x K) operand [Re A ; Im A] -- one 1-D bulk copy puts it in place, the tensor core reads it from there.
//   Nothing converts A on chip: no converter warps, no TMEM operand panels (stencil_tc.cuh needs twelve warps for it).
// * M = 128 = two sites = two swizzle atoms; the descriptor's leading-dimension byte offset is the distance between
//   the two tiles.  A step whose X tile only one site uses points the other atom at a block of zeros.
// * K = 16 per instruction: 2 k-steps x (A_hi . [X_hi | X_lo] -> D | C,  then A_lo . X_hi -> C) = 4 MMAs per step
//   (stencil_tc.cuh: 8-12).
// * X: every site's tile is scaled, split and written ONCE per apply as a ready-made operand tile [hi | lo] (MN-major,
//   SWIZZLE_128B) by two pre-pass kernels (colmax_kernel, xsplit_kernel); the stencil kernel bulk-copies it like A.
//   The epilogue undoes the scales and combines Re/Im as in stencil_tc.cuh.
// * The time of one pipeline is the serial latency of its hand-shakes, not any unit's throughput: up to three CTAs
//   (independent pipelines, 128 TMEM columns each) run per SM.
// Range: elements smaller than 2^-29 of the operator's (a column's) largest element lose relative precision
// (absolute error <= 2^-25 of the largest): norm-wise errors stay at the 1e-7 level.
#pragma once

#include <cuda_fp16.h>

#include "stencil_tc.cuh"

namespace cmrhs {

// warp roles: 4 epilogue | A producer | X producer | MMA issuer | TMEM allocator; 1-3 CTAs (independent pipelines) per SM
constexpr int kHThreads = 256;
constexpr int kHMaxStagesA = 24;
constexpr int kHMaxStagesX = 8;
constexpr int kHMaxAcc = 4;
constexpr uint32_t kHTile = 8192;       // one stencil matrix: hi 4 KB | lo 4 KB
constexpr uint32_t kHZero = 2048;       // 16 K rows x 128 B of zeros (one MMA's worth of an absent site's atom)

struct HParams {
    int32_t L[4];
    int32_t ng0, ngroups;
    int32_t s;            // nrhs (multiple of 8)
    int32_t N2;           // 2 s: real columns of an X tile
    int32_t LO;           // operand column of the lo half: 2 s if 4 s <= 64 (hi | lo share one 64-column atom), else a multiple of 64
    int32_t wideN;        // LO + 2 s: N of the A_hi MMA ([X_hi | X_lo] -> D | C); the A_lo . X_hi MMA adds into C (TMEM column LO)
    int32_t acc_stride, nacc;
    int32_t tmem_cols;    // 512 (one CTA per SM), 256 (two) or 128 (three)
    int32_t sa, sxo;      // ring depths: A tiles, X operand tiles
    int32_t xo_bytes;     // fp16 X operand tile: atoms * 4096
    uint32_t idesc_wide, idesc_lo;
    int32_t tr;           // 1: transposed form (nrhs > 32): the X tile is the M-side operand (M = 2 nrhs real columns, padded to
                          //    128), the stencil matrix the N side ([A_hi | A_lo], N = 128); one accumulator (D 64 | C 64 columns)
                          //    PER SITE, so a step only one site uses costs half a step -- no M rows are spent on zeros
    uint32_t idesc_t_wide, idesc_t_lo;
    float inv_sA;         // 1 / sA
    const uint32_t *amax; // [s] bit patterns of max |Re|, |Im| per column of X (pre-pass)
};

// kind::f16, D = F32, A = B = F16, both MN-major
__host__ __device__ constexpr uint32_t umma_idesc_f16_mn(int M, int N)
{
    return (1u << 4) | (1u << 15) | (1u << 16) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
__device__ __forceinline__ void umma_f16_ss(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// MN-major SWIZZLE_128B descriptor: atoms of 64 halves (128 B) x 8 K rows; LBO = next atom along M/N, SBO = next 8 K rows (1024 B)
__device__ __forceinline__ uint64_t h_desc(uint32_t addr, uint32_t lbo_bytes)
{
    return (uint64_t)((addr >> 4) & 0x3FFFu) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16) | ((uint64_t)(1024u >> 4) << 32) |
           (1ull << 46) | (2ull << 61);
}
// byte offset of element (k, col) inside an MN-major SWIZZLE_128B block of 64-column atoms (atom stride 4096 B, 32 K rows)
__host__ __device__ __forceinline__ uint32_t h_swz(uint32_t k, uint32_t col)
{
    const uint32_t atom = col >> 6, c = col & 63u;
    return atom * 4096u + k * 128u + ((((c >> 3) ^ (k & 7u)) << 4) | ((c & 7u) << 1));
}

// power of two that maps a maximum with bit pattern `bits` (non-negative float) into [2^14, 2^15)
__host__ __device__ __forceinline__ float h_scale_from_bits(uint32_t bits)
{
    int e = (int)(bits >> 23) & 0xFF;
    if (bits == 0u || e == 0xFF) return 1.0f;
    int k = 14 - (e - 127);
    if (k > 100) k = 100;
    if (k < -100) k = -100;
    union { uint32_t u; float f; } r;
    r.u = (uint32_t)(k + 127) << 23;
    return r.f;
}

__device__ __forceinline__ int64_t h_site(const HParams &P, int x, int y, int z, int t)
{
    return x + (int64_t)P.L[0] * (y + (int64_t)P.L[1] * (z + (int64_t)P.L[2] * t));
}
__device__ __forceinline__ TcGroup h_group(const HParams &P, int g, const uint32_t *tab2, const uint32_t *tab1)
{
    TcGroup r;
    const int gx = g % P.ng0;
    int line = g / P.ng0;
    r.x0 = gx * 2;
    r.G = min(2, P.L[0] - r.x0);
    r.y = line % P.L[1]; line /= P.L[1];
    r.z = line % P.L[2];
    r.t = line / P.L[2];
    r.nsteps = r.G == 2 ? 110 : 81;
    r.tab = r.G == 2 ? tab2 : tab1;
    return r;
}
__device__ __forceinline__ int64_t h_x_site(const HParams &P, const TcGroup &g, uint32_t e)
{
    const int off3 = (int)(e & 31u), j = (int)((e >> 5) & 7u);
    const int dy = off3 % 3 - 1, dz = (off3 / 3) % 3 - 1, dt = off3 / 9 - 1;
    return h_site(P, tc_wrap(g.x0 + j - 1, P.L[0]), tc_wrap(g.y + dy, P.L[1]), tc_wrap(g.z + dz, P.L[2]), tc_wrap(g.t + dt, P.L[3]));
}

template <int kCtasPerSm, bool kTr>
__global__ void __launch_bounds__(kHThreads, kCtasPerSm)
stencil_h16_kernel(const unsigned char *__restrict__ Ah, const unsigned char *__restrict__ Xh, float2 *__restrict__ Y, const HParams P)
{
    constexpr int NB = 32;
    constexpr int kHXconvWarps = 0;          // (role offsets: the X operand arrives ready-made, nothing converts on chip)
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    // carve: [zeros 2 KB][A ring][zeros 2 KB][X operand ring][epilogue exchange][tables][scales][barriers][tmem slot]
    unsigned char *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    unsigned char *zero0 = smem;
    unsigned char *ringA = zero0 + kHZero;
    unsigned char *zero1 = ringA + (size_t)P.sa * kHTile;
    unsigned char *ringXo = zero1 + kHZero;
    float4 *exch = reinterpret_cast<float4 *>(ringXo + (size_t)P.sxo * P.xo_bytes);         // [pair 2][buf 2][part 2][j 2][lane 32]
    uint32_t *tab2 = reinterpret_cast<uint32_t *>(exch + 2 * 2 * 2 * 2 * 32);
    uint32_t *tab1 = tab2 + kTcMaxSteps;
    float *inv = reinterpret_cast<float *>(tab1 + kTcMaxSteps);      // [128] per real column: 1 / (sA sX_r)
    uint64_t *bars = reinterpret_cast<uint64_t *>(inv + 128);
    uint64_t *a_full = bars, *a_empty = a_full + kHMaxStagesA;
    uint64_t *xo_full = a_empty + kHMaxStagesA, *xo_empty = xo_full + kHMaxStagesX;
    uint64_t *acc_full = xo_empty + kHMaxStagesX, *acc_empty = acc_full + kHMaxAcc;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(acc_empty + kHMaxAcc);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#ifdef CMRHS_TC_TRACE
    long long wt[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    const long long t_begin = clock64();
#endif

    if (threadIdx.x == 0) {
        for (int i = 0; i < P.sa; ++i) { mbar_init(&a_full[i], 1); mbar_init(&a_empty[i], 1); }
        for (int i = 0; i < P.sxo; ++i) { mbar_init(&xo_full[i], 1); mbar_init(&xo_empty[i], 1); }
        for (int i = 0; i < P.nacc; ++i) { mbar_init(&acc_full[i], 1); mbar_init(&acc_empty[i], 4); }
        mbar_fence_init();
    }
    if (threadIdx.x == 32) tc_build_schedule(2, tab2);
    if (threadIdx.x == 64) tc_build_schedule(1, tab1);
    if (threadIdx.x >= 128 && threadIdx.x < 256) {
        const int col = threadIdx.x - 128;
        const float sc = col < P.N2 ? h_scale_from_bits(P.amax[col >> 1]) : 1.0f;
        inv[col] = P.inv_sA / sc;
    }
    for (int e = threadIdx.x; e < (int)(kHZero / 16); e += kHThreads) {
        reinterpret_cast<uint4 *>(zero0)[e] = make_uint4(0u, 0u, 0u, 0u);
        reinterpret_cast<uint4 *>(zero1)[e] = make_uint4(0u, 0u, 0u, 0u);
    }
    fence_proxy_async_smem();           // the zero blocks are read by the tensor core (async proxy)
    if (warp == kHXconvWarps + 7) tmem_alloc_cols(tmem_slot, (uint32_t)P.tmem_cols);
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();
    const uint32_t tmem = *tmem_slot;

    if (warp < 4) {
        // ================= epilogue: Y = combine((D + 2^-11 C) / (sA sX)) -> global =================
        const int q = warp - kHXconvWarps;                 // = warp % 4: the TMEM lane quarter this warp may access
        const int slot = q >> 1, part = q & 1;
        const uint32_t lane_base = tmem + ((uint32_t)(32 * q) << 16);
        float4 *xb = exch + slot * (2 * 2 * 2 * 32);
        TcRing rc;
        uint32_t chunk_no = 0;
        for (int g = blockIdx.x; g < P.ngroups; g += gridDim.x) {
            const TcGroup grp = h_group(P, g, tab2, tab1);
            TW(0, mbar_wait(&acc_full[rc.stage], rc.phase));
            tc_fence_after_sync();
            TW_BEGIN();
            if constexpr (kTr) {
                // lanes = real columns n = (r, re/im) of Y^T, columns = (part, i): Y_re = P[(r,0)] - Q[(r,1)], Y_im = P[(r,1)] + Q[(r,0)]
                const int n = 32 * q + lane, r = n >> 1, c = n & 1;
                const bool live = n < P.N2;
                const float sc = live ? inv[n] * 1.0f : 0.0f;
                float *Yf = reinterpret_cast<float *>(Y);
                for (int i = 0; i < grp.G; ++i) {
                    const uint32_t ds = lane_base + (uint32_t)(rc.stage * P.acc_stride) + 128u * (uint32_t)i;
                    const int64_t site = h_site(P, grp.x0 + i, grp.y, grp.z, grp.t);
#pragma unroll
                    for (int half = 0; half < 2; ++half) {
                        uint32_t dp[16], cp[16], dq[16], cq[16];
                        tmem_ld_x16(ds + 16u * half, dp);
                        tmem_ld_x16(ds + 64u + 16u * half, cp);
                        tmem_ld_x16(ds + 32u + 16u * half, dq);
                        tmem_ld_x16(ds + 96u + 16u * half, cq);
                        tmem_wait_ld();
#pragma unroll
                        for (int k = 0; k < 16; ++k) {
                            const float pv = (__uint_as_float(dp[k]) + __uint_as_float(cp[k]) * (1.0f / 2048.0f)) * sc;
                            const float qv = (__uint_as_float(dq[k]) + __uint_as_float(cq[k]) * (1.0f / 2048.0f)) * sc;
                            const float qo = __shfl_xor_sync(0xffffffffu, qv, 1);
                            const float val = c == 0 ? pv - qo : pv + qo;
                            if (live) Yf[((site * NB + 16 * half + k) * (int64_t)P.s + r) * 2 + c] = val;
                        }
                    }
                }
            } else
            if (slot < grp.G) {
                const uint32_t d = lane_base + (uint32_t)(rc.stage * P.acc_stride);
                const uint32_t c2 = d + (uint32_t)P.LO;
                const int64_t site = h_site(P, grp.x0 + slot, grp.y, grp.z, grp.t);
                float2 *yrow = Y + (site * NB + lane) * (int64_t)P.s;
                for (int c = 0; c < (P.N2 + 15) / 16; ++c, ++chunk_no) {
                    uint32_t a[16], b[16];
                    float v[16];
                    tmem_ld_x16(d + 16u * c, a);
                    tmem_ld_x16(c2 + 16u * c, b);
                    tmem_wait_ld();
#pragma unroll
                    for (int k = 0; k < 16; ++k) v[k] = (__uint_as_float(a[k]) + __uint_as_float(b[k]) * (1.0f / 2048.0f)) * inv[16 * c + k];
                    float4 *buf = xb + (chunk_no & 1u) * (2 * 2 * 32);
                    if (part == 0) {
                        buf[0 * 32 + lane] = make_float4(v[8], v[9], v[10], v[11]);
                        buf[1 * 32 + lane] = make_float4(v[12], v[13], v[14], v[15]);
                    } else {
                        buf[2 * 32 + lane] = make_float4(v[0], v[1], v[2], v[3]);
                        buf[3 * 32 + lane] = make_float4(v[4], v[5], v[6], v[7]);
                    }
                    tc_named_barrier(1 + slot, 64);
                    const float4 o0 = buf[((part ^ 1) * 2 + 0) * 32 + lane], o1 = buf[((part ^ 1) * 2 + 1) * 32 + lane];
                    float4 r0, r1;
                    if (part == 0) {        // mine: P = ReA.X (columns 0-7), theirs: Q = ImA.X (columns 0-7)
                        r0 = make_float4(v[0] - o0.y, v[1] + o0.x, v[2] - o0.w, v[3] + o0.z);
                        r1 = make_float4(v[4] - o1.y, v[5] + o1.x, v[6] - o1.w, v[7] + o1.z);
                    } else {                // mine: Q (columns 8-15), theirs: P (columns 8-15)
                        r0 = make_float4(o0.x - v[9], o0.y + v[8], o0.z - v[11], o0.w + v[10]);
                        r1 = make_float4(o1.x - v[13], o1.y + v[12], o1.z - v[15], o1.w + v[14]);
                    }
                    if (8 * c + 4 * part < P.s) {            // (false only for the upper half of the single chunk of nrhs 4)
                        float4 *dstp = reinterpret_cast<float4 *>(yrow + 8 * c + 4 * part);
                        dstp[0] = r0;
                        dstp[1] = r1;
                    }
                }
            }
            tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) mbar_arrive(&acc_empty[rc.stage]);
            TW_END(1);
            rc.advance(P.nacc);
        }
    }
    else if (warp == kHXconvWarps + 4) {
        // ================= A producer: one pre-split stencil matrix (8 KB, contiguous) per stage =================
        // A step both sites use needs its two tiles in consecutive stages (one descriptor, LBO = one stage): if the
        // pair would wrap around the ring, the last stage is passed over with an empty hand-shake (the MMA warp
        // applies the same rule).
        const uint64_t pol = l2_policy_evict_first();
        TcRing ra;
        for (int g = blockIdx.x; g < P.ngroups; g += gridDim.x) {
            const TcGroup grp = h_group(P, g, tab2, tab1);
            const int64_t site0 = h_site(P, grp.x0, grp.y, grp.z, grp.t);
            for (int step = 0; step < grp.nsteps; ++step) {
                const uint32_t e = grp.tab[step];
                const int off3 = (int)(e & 31u);
                if (!kTr && ((e >> 8) & 3u) == 3u && ra.stage == P.sa - 1) {
                    TW(0, mbar_wait(&a_empty[ra.stage], ra.phase ^ 1u));
                    if (elect_one_sync()) mbar_arrive(&a_full[ra.stage]);
                    __syncwarp();
                    ra.advance(P.sa);
                }
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    if (!((e >> (8 + i)) & 1u)) continue;
                    const int p = (int)((e >> (10 + 2 * i)) & 3u) + 3 * off3;
                    const unsigned char *src = Ah + ((site0 + i) * kNPoint + p) * (int64_t)kHTile;
                    TW(0, mbar_wait(&a_empty[ra.stage], ra.phase ^ 1u));
                    if (elect_one_sync()) {
                        mbar_arrive_expect_tx(&a_full[ra.stage], kHTile);
                        bulk_g2s(ringA + (size_t)ra.stage * kHTile, src, kHTile, &a_full[ra.stage], pol);
                    }
                    __syncwarp();
                    ra.advance(P.sa);
                }
            }
        }
    } else if (warp == kHXconvWarps + 5) {
        // ================= X producer: the neighbour's ready-made fp16 operand tile (contiguous), once per step =================
        const uint64_t pol = l2_policy_evict_last();
        TcRing ro;
        for (int g = blockIdx.x; g < P.ngroups; g += gridDim.x) {
            const TcGroup grp = h_group(P, g, tab2, tab1);
            for (int step = 0; step < grp.nsteps; ++step) {
                const unsigned char *src = Xh + h_x_site(P, grp, grp.tab[step]) * (int64_t)P.xo_bytes;
                TW(0, mbar_wait(&xo_empty[ro.stage], ro.phase ^ 1u));
                if (elect_one_sync()) {
                    mbar_arrive_expect_tx(&xo_full[ro.stage], (uint32_t)P.xo_bytes);
                    bulk_g2s(ringXo + (size_t)ro.stage * P.xo_bytes, src, (uint32_t)P.xo_bytes, &xo_full[ro.stage], pol);
                }
                __syncwarp();
                ro.advance(P.sxo);
            }
        }
    } else if (warp == kHXconvWarps + 6) {
        // ================= MMA issuer (whole warp walks the schedule, one elected lane issues) =================
        const uint32_t z0 = smem_u32(zero0), z1 = smem_u32(zero1), ring0 = smem_u32(ringA);
        TcRing ra, ro, rc;
        for (int g = blockIdx.x; g < P.ngroups; g += gridDim.x) {
            const TcGroup grp = h_group(P, g, tab2, tab1);
            TW(0, mbar_wait(&acc_empty[rc.stage], rc.phase ^ 1u));
            tc_fence_after_sync();
            const uint32_t d = tmem + (uint32_t)(rc.stage * P.acc_stride), c2 = d + (uint32_t)P.LO;
            if constexpr (kTr) {
                // transposed form: D_site[(r,c)][(part,i)] += X^T . [A_hi | A_lo]  -- one accumulator (128 columns) per site
                uint32_t seen = 0u;
                const uint32_t lo_atoms = (uint32_t)(P.LO >> 6) * 4096u;
                for (int step = 0; step < grp.nsteps; ++step) {
                    const uint32_t um = (grp.tab[step] >> 8) & 3u;
                    TcRing r1 = ra;
                    r1.advance(P.sa);
                    TW(1, mbar_wait(&a_full[ra.stage], ra.phase));
                    if (um == 3u) TW(1, mbar_wait(&a_full[r1.stage], r1.phase));
                    TW(2, mbar_wait(&xo_full[ro.stage], ro.phase));
                    tc_fence_after_sync();
                    TW_BEGIN();
                    if (elect_one_sync()) {
                        const uint32_t xo = smem_u32(ringXo + (size_t)ro.stage * P.xo_bytes);
                        int nth = 0;
#pragma unroll
                        for (int i = 0; i < 2; ++i) {
                            if (!((um >> i) & 1u)) continue;
                            const uint32_t tile = ring0 + (uint32_t)(nth == 0 ? ra.stage : r1.stage) * kHTile;
                            const uint32_t ds = d + 128u * (uint32_t)i;
#pragma unroll
                            for (int ks = 0; ks < 2; ++ks) {
                                const uint64_t x_hi = h_desc(xo + (uint32_t)ks * 2048u, 4096u);
                                const uint64_t x_lo = h_desc(xo + lo_atoms + (uint32_t)ks * 2048u, 4096u);
                                const uint64_t a_w = h_desc(tile + (uint32_t)ks * 2048u, 4096u);       // [A_hi | A_lo]: adjacent 4 KB atoms
                                const uint32_t acc = (((seen >> i) & 1u) | (uint32_t)ks) != 0u ? 1u : 0u;
                                umma_f16_ss(ds, x_hi, a_w, P.idesc_t_wide, acc);            // X_hi^T . [A_hi | A_lo] -> D | C
                                umma_f16_ss(ds + 64u, x_lo, a_w, P.idesc_t_lo, 1u);         // X_lo^T . A_hi -> C
                            }
                            ++nth;
                        }
                        umma_commit(&xo_empty[ro.stage]);
                        umma_commit(&a_empty[ra.stage]);
                        if (um == 3u) umma_commit(&a_empty[r1.stage]);
                        if (step == grp.nsteps - 1) umma_commit(&acc_full[rc.stage]);
                    }
                    __syncwarp();
                    TW_END(3);
                    seen |= um;
                    ra.advance(P.sa);
                    if (um == 3u) ra.advance(P.sa);
                    ro.advance(P.sxo);
                }
                rc.advance(P.nacc);
                continue;
            }
            for (int step = 0; step < grp.nsteps; ++step) {
                const uint32_t um = (grp.tab[step] >> 8) & 3u;
                if (um == 3u && ra.stage == P.sa - 1) {            // the pair would wrap: pass over the last stage
                    TW(1, mbar_wait(&a_full[ra.stage], ra.phase));
                    if (elect_one_sync()) mbar_arrive(&a_empty[ra.stage]);
                    __syncwarp();
                    ra.advance(P.sa);
                }
                const int st0 = ra.stage;
                TW(1, mbar_wait(&a_full[st0], ra.phase));
                if (um == 3u) TW(1, mbar_wait(&a_full[st0 + 1], ra.phase));
                TW(2, mbar_wait(&xo_full[ro.stage], ro.phase));
                tc_fence_after_sync();
                TW_BEGIN();
                if (elect_one_sync()) {
                    const uint32_t t0 = ring0 + (uint32_t)st0 * kHTile;       // first (or only) tile of the step
                    const uint32_t xo = smem_u32(ringXo + (size_t)ro.stage * P.xo_bytes);
#pragma unroll
                    for (int ks = 0; ks < 2; ++ks) {
                        const uint64_t bd = h_desc(xo + (uint32_t)ks * 2048u, 4096u);
                        const uint32_t acc = (step | ks) != 0 ? 1u : 0u;
                        uint64_t ad_hi, ad_lo;
                        const uint32_t hi = t0 + (uint32_t)ks * 2048u, lo = hi + 4096u;
                        if (um == 3u) { ad_hi = h_desc(hi, kHTile); ad_lo = h_desc(lo, kHTile); }
                        else if (um == 1u) { ad_hi = h_desc(hi, z1 - hi); ad_lo = h_desc(lo, z1 - lo); }      // site 1's atom: zeros
                        else { ad_hi = h_desc(z0, hi - z0); ad_lo = h_desc(z0, lo - z0); }                    // site 0's atom: zeros
                        umma_f16_ss(d, ad_hi, bd, P.idesc_wide, acc);       // A hi . [X hi | X lo] -> D | C
                        umma_f16_ss(c2, ad_lo, bd, P.idesc_lo, 1u);         // A lo . X hi -> C (same columns, issued after)
                    }
                    umma_commit(&xo_empty[ro.stage]);
                    umma_commit(&a_empty[st0]);
                    if (um == 3u) umma_commit(&a_empty[st0 + 1]);
                    if (step == grp.nsteps - 1) umma_commit(&acc_full[rc.stage]);
                }
                __syncwarp();
                TW_END(3);
                ra.advance(P.sa);
                if (um == 3u) ra.advance(P.sa);
                ro.advance(P.sxo);
            }
            rc.advance(P.nacc);
        }
    }
#ifdef CMRHS_TC_TRACE
    if (lane == 0 && blockIdx.x < 160) {
        wt[7] = clock64() - t_begin;
        for (int k = 0; k < 8; ++k) g_tc_trace[blockIdx.x][warp][k] = wt[k];
    }
#endif
    // ---- teardown ----
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();
    if (warp == kHXconvWarps + 7) tmem_dealloc_cols(tmem, (uint32_t)P.tmem_cols);
}

// ---- host side ------------------------------------------------------------------------------------------------
// shapes the FP16-split kernel covers: complex64, nbasis 32, nrhs a multiple of 8, or 4 (the A_lo MMA then runs at the
// minimum N = 16 and also writes 8 unused accumulator columns)
inline bool h16_supported(int nb, int s) { return nb == 32 && ((s >= 8 && s <= 64 && s % 8 == 0) || s == 4); }

// max |v| over a float array, as the bit pattern of a non-negative float (order-independent: atomicMax on the bits)
__global__ void absmax_kernel(const float *__restrict__ v, int64_t n, uint32_t *__restrict__ out)
{
    uint32_t m = 0u;
    for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
        const uint32_t b = __float_as_uint(v[e]) & 0x7FFFFFFFu;
        if (b <= 0x7F800000u) m = max(m, b);        // NaNs are skipped
    }
    for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0 && m) atomicMax(out, m);
}

// per right-hand-side column: max over rows of |Re|, |Im| of X[n][s] (bit patterns, as above).  out must be zeroed.
__global__ void __launch_bounds__(256) colmax_kernel(const float2 *__restrict__ X, int64_t n, int s, uint32_t *__restrict__ out)
{
    __shared__ uint32_t smax[64];
    if (threadIdx.x < 64) smax[threadIdx.x] = 0u;
    __syncthreads();
    const int rpp = 256 / s;                         // rows per pass of the block
    const int col = threadIdx.x % s, r = threadIdx.x / s;
    uint32_t m = 0u;
    if (r < rpp) {
        for (int64_t row = (int64_t)blockIdx.x * rpp + r; row < n; row += (int64_t)gridDim.x * rpp) {
            const float2 v = X[row * s + col];
            const uint32_t a = __float_as_uint(v.x) & 0x7FFFFFFFu, b = __float_as_uint(v.y) & 0x7FFFFFFFu;
            if (a <= 0x7F800000u) m = max(m, a);
            if (b <= 0x7F800000u) m = max(m, b);
        }
        if (m) atomicMax(&smax[col], m);
    }
    __syncthreads();
    if (threadIdx.x < s && smax[threadIdx.x]) atomicMax(&out[threadIdx.x], smax[threadIdx.x]);
}

// create-time re-layout: canonical A[t][i][k] (complex64) -> pre-split tiles Ah[t] = [hi 4 KB | lo 4 KB]; each half is
// the MN-major SWIZZLE_128B image of the 64 x 32 operand (columns 0-31: Re A[i][k], 32-63: Im A[i][k]; K row = k).
// One CTA of 256 threads per tile: thread = (k, 8-column chunk).
__global__ void __launch_bounds__(256) relayout_h16_kernel(const cplx<float> *__restrict__ A, unsigned char *__restrict__ Ah,
                                                           int64_t ntiles, float sA)
{
    const int k = threadIdx.x >> 3, ch = threadIdx.x & 7;         // chunk ch: columns 8 ch .. 8 ch + 7
    const int part = ch >> 2, i0 = (ch & 3) * 8;                    // Re (0) or Im (1) rows i0 .. i0 + 7
    for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const cplx<float> *src = A + t * 1024;
        uint32_t hw[4], lw[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const cplx<float> v0 = src[(i0 + 2 * u) * 32 + k], v1 = src[(i0 + 2 * u + 1) * 32 + k];
            const float a0 = (part ? v0.im : v0.re) * sA, a1 = (part ? v1.im : v1.re) * sA;
            const __half2 h = __floats2half2_rn(a0, a1);
            const float2 hf = __half22float2(h);
            const __half2 l = __floats2half2_rn((a0 - hf.x) * 2048.0f, (a1 - hf.y) * 2048.0f);
            hw[u] = *reinterpret_cast<const uint32_t *>(&h);
            lw[u] = *reinterpret_cast<const uint32_t *>(&l);
        }
        unsigned char *dst = Ah + t * (int64_t)kHTile + h_swz((uint32_t)k, (uint32_t)(8 * ch));
        *reinterpret_cast<uint4 *>(dst) = make_uint4(hw[0], hw[1], hw[2], hw[3]);
        *reinterpret_cast<uint4 *>(dst + 4096) = make_uint4(lw[0], lw[1], lw[2], lw[3]);
    }
}

// per-apply pre-pass 2: X (fp32, [site][k = basis row][2 s real columns]) -> Xh, one ready-made operand tile per site:
// the MN-major SWIZZLE_128B shared-memory image of [X_hi | X_lo] (scaled by the column's power of two, split into
// hi = fp16(x), lo = fp16(2^11 (x - hi))).  Every X tile is read by ~40 groups of sites; it is converted once, here.
__global__ void __launch_bounds__(256) xsplit_kernel(const float *__restrict__ X, unsigned char *__restrict__ Xh, const uint32_t *__restrict__ amax,
                                                     int64_t nsites, int s, int LO, int xo_bytes)
{
    __shared__ float scl[128];
    const int N2 = 2 * s, gpr = N2 >> 3, nchunks = 32 * gpr;
    if (threadIdx.x < 128) scl[threadIdx.x] = threadIdx.x < N2 ? h_scale_from_bits(amax[threadIdx.x >> 1]) : 1.0f;
    __syncthreads();
    for (int64_t site = blockIdx.x; site < nsites; site += gridDim.x) {
        const float *src = X + site * (int64_t)(32 * N2);
        unsigned char *dst = Xh + site * (int64_t)xo_bytes;
        for (int c = threadIdx.x; c < nchunks; c += 256) {
            const int k = c / gpr, col0 = (c - k * gpr) << 3;
            const float4 v0 = *reinterpret_cast<const float4 *>(src + k * N2 + col0);
            const float4 v1 = *reinterpret_cast<const float4 *>(src + k * N2 + col0 + 4);
            const float4 s0 = *reinterpret_cast<const float4 *>(scl + col0);
            const float4 s1 = *reinterpret_cast<const float4 *>(scl + col0 + 4);
            const float x[8] = {v0.x * s0.x, v0.y * s0.y, v0.z * s0.z, v0.w * s0.w, v1.x * s1.x, v1.y * s1.y, v1.z * s1.z, v1.w * s1.w};
            uint32_t hw[4], lw[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const __half2 h = __floats2half2_rn(x[2 * u], x[2 * u + 1]);
                const float2 hf = __half22float2(h);
                const __half2 l = __floats2half2_rn((x[2 * u] - hf.x) * 2048.0f, (x[2 * u + 1] - hf.y) * 2048.0f);
                hw[u] = *reinterpret_cast<const uint32_t *>(&h);
                lw[u] = *reinterpret_cast<const uint32_t *>(&l);
            }
            *reinterpret_cast<uint4 *>(dst + h_swz((uint32_t)k, (uint32_t)col0)) = make_uint4(hw[0], hw[1], hw[2], hw[3]);
            *reinterpret_cast<uint4 *>(dst + h_swz((uint32_t)k, (uint32_t)(LO + col0))) = make_uint4(lw[0], lw[1], lw[2], lw[3]);
        }
    }
}

// bytes of one X operand tile for nrhs = s
inline int h16_xo_bytes(int s) { return (4 * s <= 64) ? 4096 : 2 * ((2 * s + 63) / 64) * 4096; }

inline int launch_stencil_h16(const unsigned char *Ah, float inv_sA, uint32_t *amax_dev, unsigned char *Xh, const LatticeDims &d, const void *X,
                              void *Y, int s, int num_sms, cudaStream_t stream, bool have_colmax = false)
{
    if ((reinterpret_cast<uintptr_t>(X) & 15u) || (reinterpret_cast<uintptr_t>(Y) & 15u)) {
        set_error("tensor path: X and Y must be 16-byte aligned");
        return COARSE_INVALID_ARG;
    }
    HParams P;
    for (int k = 0; k < 4; ++k) P.L[k] = d.L[k];
    P.ng0 = (d.L[0] + 1) / 2;
    P.ngroups = (int32_t)((int64_t)P.ng0 * d.L[1] * d.L[2] * d.L[3]);
    P.s = s;
    P.N2 = 2 * s;
    if (4 * s <= 64) P.LO = 2 * s;
    else P.LO = 64 * ((2 * s + 63) / 64);
    P.wideN = P.LO + 2 * s;
    P.acc_stride = P.wideN;
    if (P.N2 < 16) P.acc_stride = P.LO + 16;  // nrhs 4: the A_lo MMA has N = 16
    P.tr = s > 48 ? 1 : 0;             // measured on B200: equal to the paired form at nrhs 48 and 64, 14 % faster at 56
    if (P.tr) P.acc_stride = 256;            // two sites x (D 64 | C 64)
    // independent pipelines (CTAs) per SM: as many as tensor memory (power-of-two allocations) and shared memory allow
    int cps = P.acc_stride <= 128 ? 3 : (P.acc_stride <= 256 ? 2 : 1);
    P.tmem_cols = cps == 3 ? 128 : (cps == 2 ? 256 : 512);
    P.nacc = P.tmem_cols / P.acc_stride;
    if (P.nacc > kHMaxAcc) P.nacc = kHMaxAcc;
    P.xo_bytes = h16_xo_bytes(s);
    auto clampi = [](int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); };
    const int smem_cta = cps == 3 ? 74 * 1024 : (cps == 2 ? 113 * 1024 : 227 * 1024);
    P.sxo = clampi(smem_cta / 5 / P.xo_bytes, 3, kHMaxStagesX);
    const int64_t fixed = 1024 /* alignment */ + 2 * kHZero + 2 * 2 * 2 * 2 * 32 * 16 /* exchange */ + 2 * kTcMaxSteps * 4 + 512 /* scales */ +
                          1024 /* barriers */ + 64;
    const int64_t budget = smem_cta - fixed - (int64_t)P.sxo * P.xo_bytes;
    P.sa = (int32_t)(budget / kHTile);
    if (P.sa > kHMaxStagesA) P.sa = kHMaxStagesA;
    if (P.sa < 4 || P.nacc < 1) { set_error("tensor path: shared/tensor memory plan does not fit (nrhs %d)", s); return COARSE_UNSUPPORTED; }
    P.idesc_wide = umma_idesc_f16_mn(128, P.wideN);
    P.idesc_lo = umma_idesc_f16_mn(128, P.N2 < 16 ? 16 : P.N2);
    P.idesc_t_wide = umma_idesc_f16_mn(128, 128);
    P.idesc_t_lo = umma_idesc_f16_mn(128, 64);
    P.inv_sA = inv_sA;
    P.amax = amax_dev;
    const size_t smem = (size_t)fixed + (size_t)P.sa * kHTile + (size_t)P.sxo * P.xo_bytes;

    // pre-passes over X: per-column max |x| (-> power-of-two column scales), then the split operand tiles
    // (have_colmax: the kernel that produced X -- pass 2 of a block-CG iteration -- has already left them in amax_dev)
    if (!have_colmax) {
        CMRHS_CUDA(cudaMemsetAsync(amax_dev, 0, 64 * sizeof(uint32_t), stream));
        const int64_t n = d.V * 32;
        const int rpp = 256 / s;
        const int cgrid = (int)(ceil_div(n, rpp) < (int64_t)num_sms * 8 ? ceil_div(n, rpp) : (int64_t)num_sms * 8);
        colmax_kernel<<<cgrid, 256, 0, stream>>>(static_cast<const float2 *>(X), n, s, amax_dev);
        CMRHS_LAUNCH_CHECK();
    }
    const int xgrid = (int)(d.V < (int64_t)num_sms * 8 ? d.V : (int64_t)num_sms * 8);
    xsplit_kernel<<<xgrid, 256, 0, stream>>>(static_cast<const float *>(X), Xh, amax_dev, d.V, s, P.LO, P.xo_bytes);
    CMRHS_LAUNCH_CHECK();

    if (P.tr) CMRHS_SMEM_ATTR((stencil_h16_kernel<2, true>), 113 * 1024);
    else if (cps == 3) CMRHS_SMEM_ATTR((stencil_h16_kernel<3, false>), 74 * 1024);
    else if (cps == 2) CMRHS_SMEM_ATTR((stencil_h16_kernel<2, false>), 113 * 1024);
    else CMRHS_SMEM_ATTR((stencil_h16_kernel<1, false>), 227 * 1024);
    const int slots = cps * num_sms;
    const int grid = P.ngroups < slots ? P.ngroups : slots;
    float2 *Yp = static_cast<float2 *>(Y);
    if (P.tr) stencil_h16_kernel<2, true><<<grid, kHThreads, smem, stream>>>(Ah, Xh, Yp, P);
    else if (cps == 3) stencil_h16_kernel<3, false><<<grid, kHThreads, smem, stream>>>(Ah, Xh, Yp, P);
    else if (cps == 2) stencil_h16_kernel<2, false><<<grid, kHThreads, smem, stream>>>(Ah, Xh, Yp, P);
    else stencil_h16_kernel<1, false><<<grid, kHThreads, smem, stream>>>(Ah, Xh, Yp, P);
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}

}  // namespace cmrhs

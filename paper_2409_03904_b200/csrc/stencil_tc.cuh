// Tensor-core stencil-GEMM kernel for complex64 on sm_100a (tcgen05 + TMEM + TMA), split-TF32 (3 products).
//   Y(x) = sum_{p=0}^{80} A^p(x) . X(x + delta_p)                       (Eq. 19)
//
// Mapping of the complex block product onto tcgen05.mma.kind::tf32:
//   D1[(q,i)][(r,c)] += sum_j Re A(x_q)[i][j] * X(y)[j][(r,c)]      D2 likewise with Im A
//   Y_re = D1[.,(r,0)] - D2[.,(r,1)],   Y_im = D1[.,(r,1)] + D2[.,(r,0)]     (combined once, in the epilogue)
// * M side (128 TMEM lanes) = the nbasis rows of the stencil matrices of up to FOUR lattice sites that are adjacent
//   along x (lane quarter q = site x0+q): an X tile X(y) is needed by three x-neighbours, so one tcgen05.mma
//   serves up to three (site, stencil point) tiles and each X tile is fetched 27(G+2)+G times per group of G sites
//   instead of 81 G times.
// * The stencil matrices (the HBM stream: 81 nb^2 complex per site) arrive by 2-D TMA in the caller's canonical
//   layout, 128B/64B-swizzled so that "one thread = one matrix row" reads are bank-conflict free; the converter
//   warps split every element into TF32 hi + lo (both exactly representable, round-to-nearest), de-interleave
//   re/im and write the four operand panels (Re hi, Im hi, Re lo, Im lo) into TMEM with tcgen05.st.  A is never
//   re-written to shared memory.
// * N side = the neighbour's X tile exactly as it lies in memory ([j][r][re,im] = K x N, N contiguous: an
//   MN-major UMMA operand, layout SWIZZLE_128B_BASE32B), loaded by TMA with the matching swizzle (128B_ATOM_32B); four warps round it to TF32 in place and
//   write the lo tile beside it.  Products: Ahi.Xhi + Alo.Xhi + Ahi.Xlo, FP32 accumulation in TMEM.
// * Accumulation order: the 80 off-centre points first, the centre point (which carries c*I) last.
// * Warp roles (512 threads, one persistent CTA per SM): 0-3 A converters, 4-7 X converters, 8-11 epilogue,
//   12 A producer (TMA), 13 X producer (TMA), 14 MMA issuer, 15 TMEM allocator.  All hand-offs are mbarriers.
#pragma once

#include "setup_kernels.cuh"
#include "tcgen05_ptx.cuh"

namespace cmrhs {

constexpr int kTcThreads = 512;
constexpr int kTcMaxStagesA = 16;
constexpr int kTcMaxStagesX = 4;
constexpr int kTcMaxSets = 3;

struct TcParams {
    int32_t L[4];
    int32_t ng0;          // groups per x-line = ceil(L0 / 4)
    int32_t ngroups;      // ng0 * L1 * L2 * L3
    int32_t s;            // nrhs (multiple of 8)
    int32_t N;            // 2 s: MMA N
    int32_t nxb;          // ceil(N / 32): 128-byte wide blocks per X tile (MN-major TF32 operands exist only in the
                          // SWIZZLE_128B_BASE32B layout: 32 floats along N per row, 32-byte chunks swizzled over 4 K rows)
    int32_t xt_bytes;     // bytes of one X tile, rounded up to 1024
    int32_t x_tile_tx;    // bytes TMA delivers per X tile
    int32_t sa, sx;       // ring depths
    int32_t nacc, nset;   // accumulator buffers, operand panel sets
    int32_t split;        // 1: hi.hi products and the lo correction products accumulate separately (4 N columns per buffer)
    int32_t acc_stride;   // TMEM columns per accumulator buffer (2 N or 4 N)
    uint32_t idesc;
    uint64_t xdesc_base;  // shared-memory descriptor of an X tile without the address
    uint32_t x_kadv;      // bytes between consecutive K = 8 steps of an X tile
};

template <int NB> struct TcCfg {
    static_assert(NB % 8 == 0 && NB >= 8 && NB <= 32, "tensor path: nbasis in {8,16,24,32}");
    static constexpr int KW = (2 * NB % 32 == 0) ? 32 : 16;         // floats per swizzle row of an A piece
    static constexpr int PIECES = 2 * NB / KW;
    static constexpr uint32_t SWZ_MASK = KW == 32 ? 7u : 3u;         // Swizzle<3,4,3> / Swizzle<2,4,3>
    static constexpr int JP = KW / 2;                                // complex columns per piece
    static constexpr int CH = KW / 4;                                // 16-byte chunks per piece row
    static constexpr uint32_t PIECE_BYTES = NB * KW * 4;
    static constexpr uint32_t TILE_BYTES = NB * 2 * NB * 4;
    static constexpr uint32_t STAGE_BYTES = (TILE_BYTES + 1023u) / 1024u * 1024u;
    static constexpr int KSTEPS = NB / 8;
};

// ---- schedule: (group, step) -> stencil offsets, users, neighbour ----------------------------------------------
struct TcGroup { int x0, G, y, z, t, nsteps; };
struct TcStep { int off3;      // (dy+1) + 3(dz+1) + 9(dt+1)
                int j;         // X tile at x' = x0 + j - 1
                int mode; };   // 0: all dx, 1: dx != 0 only, 2: dx == 0 only  (centre offset is swept twice: centre point last)

__device__ __forceinline__ TcGroup tc_group(const TcParams &P, int g)
{
    TcGroup r;
    const int gx = g % P.ng0;
    int line = g / P.ng0;
    r.x0 = gx * 4;
    r.G = min(4, P.L[0] - r.x0);
    r.y = line % P.L[1]; line /= P.L[1];
    r.z = line % P.L[2];
    r.t = line / P.L[2];
    r.nsteps = 27 * (r.G + 2) + r.G;
    return r;
}
__device__ __forceinline__ TcStep tc_step(const TcGroup &g, int step)
{
    TcStep s;
    const int W = g.G + 2;
    if (step < 26 * W) {
        const int o = step / W;
        s.off3 = o < 13 ? o : o + 1;
        s.j = step - o * W;
        s.mode = 0;
    } else {
        const int r = step - 26 * W;
        s.off3 = 13;
        if (r < W) { s.j = r; s.mode = 1; }
        else { s.j = r - W + 1; s.mode = 2; }
    }
    return s;
}
// bit i set <=> site x0+i of the group uses the X tile of this step (dx = j-1-i)
__device__ __forceinline__ uint32_t tc_users(const TcGroup &g, const TcStep &s)
{
    uint32_t m = 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int dx = s.j - 1 - i;
        const bool ok = i < g.G && dx >= -1 && dx <= 1 && (s.mode == 0 || (s.mode == 1 && dx != 0) || (s.mode == 2 && dx == 0));
        m |= ok ? (1u << i) : 0u;
    }
    return m;
}
__device__ __forceinline__ int tc_wrap(int c, int L) { return c < 0 ? c + L : (c >= L ? c - L : c); }
__device__ __forceinline__ int64_t tc_site(const TcParams &P, int x, int y, int z, int t)
{
    return x + (int64_t)P.L[0] * (y + (int64_t)P.L[1] * (z + (int64_t)P.L[2] * t));
}
__device__ __forceinline__ int64_t tc_x_site(const TcParams &P, const TcGroup &g, const TcStep &s)
{
    const int dy = s.off3 % 3 - 1, dz = (s.off3 / 3) % 3 - 1, dt = s.off3 / 9 - 1;
    return tc_site(P, tc_wrap(g.x0 + s.j - 1, P.L[0]), tc_wrap(g.y + dy, P.L[1]), tc_wrap(g.z + dz, P.L[2]), tc_wrap(g.t + dt, P.L[3]));
}

struct TcRing {     // stage / phase bookkeeping of an mbarrier ring
    int stage = 0;
    uint32_t phase = 0;
    __device__ __forceinline__ void advance(int depth) { if (++stage == depth) { stage = 0; phase ^= 1u; } }
};

template <int NB>
__global__ void __launch_bounds__(kTcThreads, 1)
stencil_tc_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmX, float2 *__restrict__ Y,
                  const TcParams P)
{
    using C = TcCfg<NB>;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    // carve: [A ring][X ring (hi|lo per stage)][barriers][tmem slot]
    unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    unsigned char *ringA = smem;
    unsigned char *ringX = ringA + (size_t)P.sa * C::STAGE_BYTES;
    uint64_t *bars = reinterpret_cast<uint64_t *>(ringX + (size_t)P.sx * 2 * P.xt_bytes);
    uint64_t *a_full = bars, *a_empty = a_full + kTcMaxStagesA;
    uint64_t *x_full = a_empty + kTcMaxStagesA, *x_empty = x_full + kTcMaxStagesX, *xlo_full = x_empty + kTcMaxStagesX;
    uint64_t *set_full = xlo_full + kTcMaxStagesX, *set_empty = set_full + kTcMaxSets;
    uint64_t *acc_full = set_empty + kTcMaxSets, *acc_empty = acc_full + 2;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(acc_empty + 2);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int i = 0; i < P.sa; ++i) { mbar_init(&a_full[i], 1); mbar_init(&a_empty[i], 1); }
        for (int i = 0; i < P.sx; ++i) { mbar_init(&x_full[i], 1); mbar_init(&x_empty[i], 1); mbar_init(&xlo_full[i], 4); }
        for (int i = 0; i < P.nset; ++i) { mbar_init(&set_full[i], 4); mbar_init(&set_empty[i], 1); }
        for (int i = 0; i < 2; ++i) { mbar_init(&acc_full[i], 1); mbar_init(&acc_empty[i], 4); }
        mbar_fence_init();
    }
    if (warp == 15) tmem_alloc_512(tmem_slot);
    if (warp == 12 && lane == 0) tma_prefetch_desc(&tmA);
    if (warp == 13 && lane == 0) tma_prefetch_desc(&tmX);
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();
    const uint32_t tmem = *tmem_slot;
    const uint32_t acc_cols = (uint32_t)(P.nacc * P.acc_stride);

    if (warp < 4) {
        // ================= A converters: smem tile row -> TF32 hi/lo, re/im panels -> TMEM =================
        const int q = warp;
        const uint32_t lane_base = tmem + ((uint32_t)(32 * q) << 16);
        const int i = lane;
        const bool row_ok = i < NB;
        TcRing ra, rs;                  // ra: position of the NEXT tile of the global tile sequence; rs: panel set
        uint32_t zero_sets = 0;         // panel sets whose lanes of this warp currently hold zeros
        for (int g = blockIdx.x; g < P.ngroups; g += gridDim.x) {
            const TcGroup grp = tc_group(P, g);
            for (int step = 0; step < grp.nsteps; ++step) {
                const TcStep st = tc_step(grp, step);
                const uint32_t um = tc_users(grp, st);
                const bool mine = (um >> q) & 1u;
                mbar_wait(&set_empty[rs.stage], rs.phase ^ 1u);
                tc_fence_after_sync();
                const uint32_t set_col = acc_cols + (uint32_t)rs.stage * 128u;
                if (mine) {
                    // my tile's slot in the A ring: sequence position + rank among this step's users
                    TcRing mt = ra;
                    const int rank = __popc(um & ((1u << q) - 1u));
                    for (int k = 0; k < rank; ++k) mt.advance(P.sa);
                    mbar_wait(&a_full[mt.stage], mt.phase);
                    const unsigned char *tile = ringA + (size_t)mt.stage * C::STAGE_BYTES;
#pragma unroll
                    for (int h = 0; h < C::PIECES; ++h) {
                        uint32_t hr[C::JP], hi[C::JP], lr[C::JP], li[C::JP];
#pragma unroll
                        for (int c = 0; c < C::CH; ++c) {
                            const uint32_t off = (uint32_t)h * C::PIECE_BYTES + (uint32_t)(row_ok ? i : 0) * (C::KW * 4) + (uint32_t)c * 16u;
                            const uint32_t phys = off ^ (((off >> 7) & C::SWZ_MASK) << 4);
                            float4 v = *reinterpret_cast<const float4 *>(tile + phys);
                            if (!row_ok) v = make_float4(0.f, 0.f, 0.f, 0.f);
                            float h0 = tf32_rn(v.x), h1 = tf32_rn(v.y), h2 = tf32_rn(v.z), h3 = tf32_rn(v.w);
                            hr[2 * c] = __float_as_uint(h0); hi[2 * c] = __float_as_uint(h1);
                            hr[2 * c + 1] = __float_as_uint(h2); hi[2 * c + 1] = __float_as_uint(h3);
                            lr[2 * c] = __float_as_uint(tf32_rn(v.x - h0)); li[2 * c] = __float_as_uint(tf32_rn(v.y - h1));
                            lr[2 * c + 1] = __float_as_uint(tf32_rn(v.z - h2)); li[2 * c + 1] = __float_as_uint(tf32_rn(v.w - h3));
                        }
                        const uint32_t col = set_col + (uint32_t)(h * C::JP);
                        tmem_st<C::JP>(lane_base + col, hr);
                        tmem_st<C::JP>(lane_base + col + 32u, hi);
                        tmem_st<C::JP>(lane_base + col + 64u, lr);
                        tmem_st<C::JP>(lane_base + col + 96u, li);
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&a_empty[mt.stage]);      // all lanes have read the tile
                    zero_sets &= ~(1u << rs.stage);
                } else if (!((zero_sets >> rs.stage) & 1u)) {
                    uint32_t zz[16];
#pragma unroll
                    for (int k = 0; k < 16; ++k) zz[k] = 0u;
#pragma unroll
                    for (int b = 0; b < 8; ++b) tmem_st_x16(lane_base + set_col + 16u * b, zz);
                    zero_sets |= 1u << rs.stage;
                }
                tmem_wait_st();
                tc_fence_before_sync();
                __syncwarp();
                if (lane == 0) mbar_arrive(&set_full[rs.stage]);
                rs.advance(P.nset);
                const int nuse = __popc(um);
                for (int k = 0; k < nuse; ++k) ra.advance(P.sa);
            }
        }
    } else if (warp < 8) {
        // ================= X converters: round the tile to TF32 in place (hi), write the lo tile =================
        const int tid = threadIdx.x - 128;
        const int nchunks = P.nxb * NB * 8;     // 16-byte chunks per X tile (whole 128-byte rows, zero padded by TMA)
        TcRing rx;
        for (int g = blockIdx.x; g < P.ngroups; g += gridDim.x) {
            const TcGroup grp = tc_group(P, g);
            for (int step = 0; step < grp.nsteps; ++step) {
                mbar_wait(&x_full[rx.stage], rx.phase);
                unsigned char *hi_t = ringX + (size_t)rx.stage * 2 * P.xt_bytes;
                unsigned char *lo_t = hi_t + P.xt_bytes;
                for (int c = tid; c < nchunks; c += 128) {
                    float4 v = *reinterpret_cast<const float4 *>(hi_t + 16 * c);
                    float4 h = make_float4(tf32_rn(v.x), tf32_rn(v.y), tf32_rn(v.z), tf32_rn(v.w));
                    float4 l = make_float4(tf32_rn(v.x - h.x), tf32_rn(v.y - h.y), tf32_rn(v.z - h.z), tf32_rn(v.w - h.w));
                    *reinterpret_cast<float4 *>(hi_t + 16 * c) = h;
                    *reinterpret_cast<float4 *>(lo_t + 16 * c) = l;
                }
                fence_proxy_async_smem();       // generic-proxy writes -> visible to the tensor core's async-proxy reads
                __syncwarp();
                if (lane == 0) mbar_arrive(&xlo_full[rx.stage]);
                rx.advance(P.sx);
            }
        }
    } else if (warp < 12) {
        // ================= epilogue: TMEM accumulators -> Y =================
        const int q = warp - 8;
        const uint32_t lane_base = tmem + ((uint32_t)(32 * q) << 16);
        TcRing rc;
        for (int g = blockIdx.x; g < P.ngroups; g += gridDim.x) {
            const TcGroup grp = tc_group(P, g);
            mbar_wait(&acc_full[rc.stage], rc.phase);
            tc_fence_after_sync();
            const uint32_t d1 = lane_base + (uint32_t)(rc.stage * P.acc_stride), d2 = d1 + (uint32_t)P.N;
            const bool ok = q < grp.G && lane < NB;
            const int64_t site = tc_site(P, grp.x0 + (q < grp.G ? q : 0), grp.y, grp.z, grp.t);
            float2 *yrow = Y + (site * NB + (lane < NB ? lane : 0)) * (int64_t)P.s;
            for (int c = 0; c < P.N / 16; ++c) {
                uint32_t a[16], b[16];
                tmem_ld_x16(d1 + 16u * c, a);
                tmem_ld_x16(d2 + 16u * c, b);
                if (P.split) {      // add the correction accumulators (round-to-nearest adds on the CUDA cores)
                    uint32_t ac[16], bc[16];
                    tmem_ld_x16(d1 + 2u * P.N + 16u * c, ac);
                    tmem_ld_x16(d2 + 2u * P.N + 16u * c, bc);
                    tmem_wait_ld();
#pragma unroll
                    for (int k = 0; k < 16; ++k) {
                        a[k] = __float_as_uint(__uint_as_float(a[k]) + __uint_as_float(ac[k]));
                        b[k] = __float_as_uint(__uint_as_float(b[k]) + __uint_as_float(bc[k]));
                    }
                }
                tmem_wait_ld();
                if (ok) {
                    float4 *dst = reinterpret_cast<float4 *>(yrow + 8 * c);
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        float4 o;
                        o.x = __uint_as_float(a[4 * k]) - __uint_as_float(b[4 * k + 1]);
                        o.y = __uint_as_float(a[4 * k + 1]) + __uint_as_float(b[4 * k]);
                        o.z = __uint_as_float(a[4 * k + 2]) - __uint_as_float(b[4 * k + 3]);
                        o.w = __uint_as_float(a[4 * k + 3]) + __uint_as_float(b[4 * k + 2]);
                        dst[k] = o;
                    }
                }
            }
            tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) mbar_arrive(&acc_empty[rc.stage]);
            rc.advance(P.nacc);
        }
    } else if (warp == 12) {
        // ================= A producer: one canonical stencil matrix per stage =================
        if (lane == 0) {
            const uint64_t pol = l2_policy_evict_first();
            TcRing ra;
            for (int g = blockIdx.x; g < P.ngroups; g += gridDim.x) {
                const TcGroup grp = tc_group(P, g);
                const int64_t site0 = tc_site(P, grp.x0, grp.y, grp.z, grp.t);
                for (int step = 0; step < grp.nsteps; ++step) {
                    const TcStep st = tc_step(grp, step);
                    const uint32_t um = tc_users(grp, st);
                    for (int i = 0; i < 4; ++i) {
                        if (!((um >> i) & 1u)) continue;
                        const int p = (st.j - 1 - i + 1) + 3 * st.off3;
                        const int64_t row0 = ((site0 + i) * kNPoint + p) * NB;
                        mbar_wait(&a_empty[ra.stage], ra.phase ^ 1u);
                        mbar_arrive_expect_tx(&a_full[ra.stage], C::TILE_BYTES);
                        unsigned char *dst = ringA + (size_t)ra.stage * C::STAGE_BYTES;
#pragma unroll
                        for (int h = 0; h < C::PIECES; ++h)
                            tma_load_2d(dst + h * C::PIECE_BYTES, &tmA, h * C::KW, (int32_t)row0, &a_full[ra.stage], pol);
                        ra.advance(P.sa);
                    }
                }
            }
        }
    } else if (warp == 13) {
        // ================= X producer: the neighbour's X tile, once per step =================
        if (lane == 0) {
            const uint64_t pol = l2_policy_evict_last();
            TcRing rx;
            for (int g = blockIdx.x; g < P.ngroups; g += gridDim.x) {
                const TcGroup grp = tc_group(P, g);
                for (int step = 0; step < grp.nsteps; ++step) {
                    const TcStep st = tc_step(grp, step);
                    const int64_t row0 = tc_x_site(P, grp, st) * NB;
                    mbar_wait(&x_empty[rx.stage], rx.phase ^ 1u);
                    mbar_arrive_expect_tx(&x_full[rx.stage], (uint32_t)P.x_tile_tx);
                    unsigned char *dst = ringX + (size_t)rx.stage * 2 * P.xt_bytes;
                    for (int b = 0; b < P.nxb; ++b)
                        tma_load_2d(dst + (size_t)b * NB * 128, &tmX, b * 32, (int32_t)row0, &x_full[rx.stage], pol);
                    rx.advance(P.sx);
                }
            }
        }
    } else if (warp == 14) {
        // ================= MMA issuer =================
        if (lane == 0) {
            TcRing rx, rs, rc;
            for (int g = blockIdx.x; g < P.ngroups; g += gridDim.x) {
                const TcGroup grp = tc_group(P, g);
                mbar_wait(&acc_empty[rc.stage], rc.phase ^ 1u);
                tc_fence_after_sync();
                const uint32_t d1 = tmem + (uint32_t)(rc.stage * P.acc_stride), d2 = d1 + (uint32_t)P.N;
                const uint32_t c1 = P.split ? d1 + 2u * P.N : d1, c2 = P.split ? d2 + 2u * P.N : d2;   // correction accumulators
                for (int step = 0; step < grp.nsteps; ++step) {
                    mbar_wait(&set_full[rs.stage], rs.phase);
                    mbar_wait(&xlo_full[rx.stage], rx.phase);
                    tc_fence_after_sync();
                    const uint32_t set_col = tmem + acc_cols + (uint32_t)rs.stage * 128u;
                    const uint32_t xhi = smem_u32(ringX + (size_t)rx.stage * 2 * P.xt_bytes), xlo = xhi + (uint32_t)P.xt_bytes;
#pragma unroll
                    for (int ks = 0; ks < C::KSTEPS; ++ks) {
                        const uint64_t bh = umma_smem_desc(P.xdesc_base, xhi + ks * P.x_kadv);
                        const uint64_t bl = umma_smem_desc(P.xdesc_base, xlo + ks * P.x_kadv);
                        const uint32_t acc = (step | ks) != 0 ? 1u : 0u;
                        const uint32_t kc = set_col + 8u * ks;
                        const uint32_t accc = P.split ? acc : 1u;
                        umma_tf32_ts(d1, kc, bh, P.idesc, acc);          // Re hi . X hi
                        umma_tf32_ts(c1, kc + 64u, bh, P.idesc, accc);   // Re lo . X hi
                        umma_tf32_ts(c1, kc, bl, P.idesc, 1u);           // Re hi . X lo
                        umma_tf32_ts(d2, kc + 32u, bh, P.idesc, acc);    // Im hi . X hi
                        umma_tf32_ts(c2, kc + 96u, bh, P.idesc, accc);   // Im lo . X hi
                        umma_tf32_ts(c2, kc + 32u, bl, P.idesc, 1u);     // Im hi . X lo
                    }
                    umma_commit(&set_empty[rs.stage]);
                    umma_commit(&x_empty[rx.stage]);
                    if (step == grp.nsteps - 1) umma_commit(&acc_full[rc.stage]);
                    rs.advance(P.nset);
                    rx.advance(P.sx);
                }
                rc.advance(P.nacc);
            }
        }
    }
    // ---- teardown ----
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();
    if (warp == 15) tmem_dealloc_512(tmem);
}

// ---- host side ------------------------------------------------------------------------------------------------
typedef CUresult (*TcEncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                    const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline TcEncodeTiledFn tc_encode_fn()
{
    static TcEncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess && qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<TcEncodeTiledFn>(p);
    }
    return fn;
}

// 2-D float32 tensor [rows][width] (width contiguous), box [box_rows][box_w]
inline int tc_make_tmap(CUtensorMap *out, const void *base, uint64_t width, uint64_t rows, uint32_t box_w, uint32_t box_rows,
                        CUtensorMapSwizzle swz)
{
    TcEncodeTiledFn fn = tc_encode_fn();
    if (!fn) { set_error("cuTensorMapEncodeTiled is not available from the driver"); return COARSE_CUDA_ERROR; }
    const cuuint64_t gdim[2] = {width, rows};
    const cuuint64_t gstride[1] = {width * 4};
    const cuuint32_t box[2] = {box_w, box_rows};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void *>(base), gdim, gstride, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, swz, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { set_error("cuTensorMapEncodeTiled failed with CUresult %d (width %llu rows %llu box %u x %u)", (int)r,
                                       (unsigned long long)width, (unsigned long long)rows, box_w, box_rows); return COARSE_CUDA_ERROR; }
    return COARSE_OK;
}

// shapes the tensor kernel covers: complex64, nbasis in {8,16,24,32}, nrhs a multiple of 8 (N = 2 nrhs a multiple of 16)
inline bool tc_supported(int nb, int s) { return (nb == 8 || nb == 16 || nb == 24 || nb == 32) && s >= 8 && s <= 64 && s % 8 == 0; }

template <int NB>
int launch_stencil_tc(const CUtensorMap &tmA, const LatticeDims &d, const void *X, void *Y, int s, int num_sms, cudaStream_t stream)
{
    using C = TcCfg<NB>;
    if ((reinterpret_cast<uintptr_t>(X) & 15u) || (reinterpret_cast<uintptr_t>(Y) & 15u)) {
        set_error("tensor path: X and Y must be 16-byte aligned");
        return COARSE_INVALID_ARG;
    }
    TcParams P;
    for (int k = 0; k < 4; ++k) P.L[k] = d.L[k];
    P.ng0 = (d.L[0] + 3) / 4;
    P.ngroups = (int32_t)((int64_t)P.ng0 * d.L[1] * d.L[2] * d.L[3]);
    P.s = s;
    P.N = 2 * s;
    P.nxb = (P.N + 31) / 32;
    P.x_tile_tx = P.nxb * NB * 128;           // TMA counts the whole box, out-of-range columns are zero filled
    P.xt_bytes = (P.x_tile_tx + 1023) / 1024 * 1024;
    // The tensor core adds into its FP32 accumulator with truncation, so every accumulation costs up to one ulp of |D|,
    // always towards zero.  Where tensor memory allows (4 N <= 256 columns) the small correction products get their own
    // accumulators: the main ones then see one third of the additions.
    P.split = (4 * P.N <= 256) ? 1 : 0;
    P.acc_stride = P.split ? 4 * P.N : 2 * P.N;
    P.nacc = (2 * P.acc_stride <= 256) ? 2 : 1;
    P.nset = (512 - P.nacc * P.acc_stride) / 128;
    if (P.nset > kTcMaxSets) P.nset = kTcMaxSets;
    P.sx = (2 * P.xt_bytes * 4 <= 96 * 1024) ? 4 : 3;
    const int64_t budget = 225 * 1024 - 1024 - 1024 - (int64_t)P.sx * 2 * P.xt_bytes;
    P.sa = (int32_t)(budget / C::STAGE_BYTES);
    if (P.sa > kTcMaxStagesA) P.sa = kTcMaxStagesA;
    if (P.sa < 3 || P.nset < 2) { set_error("tensor path: shared/tensor memory plan does not fit (nb %d, nrhs %d)", NB, s); return COARSE_UNSUPPORTED; }
    P.idesc = umma_idesc_tf32(128, P.N, true);
    P.xdesc_base = umma_smem_desc_base((uint32_t)(NB * 128), 512u, 1u);     // LBO: next 32 columns, SBO: next 4 K rows
    P.x_kadv = 1024u;                                                         // 8 K rows
    const size_t smem = 1024 + (size_t)P.sa * C::STAGE_BYTES + (size_t)P.sx * 2 * P.xt_bytes + 1024;

    CUtensorMap tmX;
    int st = tc_make_tmap(&tmX, X, (uint64_t)P.N, (uint64_t)d.V * NB, 32u, NB, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B);
    if (st != COARSE_OK) return st;

    auto kern = stencil_tc_kernel<NB>;
    static size_t attr_smem = 0;
    if (attr_smem < smem) {
        CMRHS_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(227 * 1024)));
        attr_smem = 227 * 1024;
    }
    const int grid = P.ngroups < num_sms ? P.ngroups : num_sms;
    kern<<<grid, kTcThreads, smem, stream>>>(tmA, tmX, static_cast<float2 *>(Y), P);
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}

template <int NB> int tc_make_tmap_A(CUtensorMap *out, const void *A, int64_t V)
{
    using C = TcCfg<NB>;
    return tc_make_tmap(out, A, (uint64_t)2 * NB, (uint64_t)V * kNPoint * NB, (uint32_t)C::KW, NB,
                        C::KW == 32 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B);
}

}  // namespace cmrhs

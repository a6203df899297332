// Tensor-core stencil-GEMM kernel for complex64 on sm_100a, split-FP16, X OPERAND IN TENSOR MEMORY, any nbasis in {8,16,24,32}.
//   Y(x) = sum_{p=0}^{80} A^p(x) . X(x + delta_p)                       (Eq. 19)
//
// Same numbers as stencil_h16.cuh (a = hi + 2^-11 lo in binary16 after a power-of-two scaling, three tensor products,
// FP32 accumulators D and C in tensor memory, Y = (D + 2^-11 C) / (sA sX_r)), in the TRANSPOSED form
//   D_x[(r,c)][(h,part,i)] += sum_k X(y)[k][(r,c)] . A^p(x)_{h,part}[i][k]          y = x + delta_p
// * M side (the 128 TMEM lanes) = the 2 nrhs real columns (r, re/im) of the neighbour's X tile, held IN TENSOR MEMORY
//   (tcgen05.mma with the A operand from TMEM): lane m, 16-bit pairs along k, [X_hi | X_lo] in nb columns.  The pre-split
//   tile arrives in a shared-memory ring by one bulk copy; loader warps (4 per lane quarter, taking turns) carry it on with
//   one 16-byte shared-memory load per lane and k chunk and tcgen05.st.  (tcgen05.cp does the same without threads and is
//   kept as a compile-time alternative, -DCMRHS_XLOAD=0: it runs in the tensor pipe's own queue at 64 B/clk, 192 clk per
//   tile during which no MMA runs -- at configs[4] 3.6 of 16.1 ms, measured by leaving the copies out.)  Every MMA then
//   reads only the stencil matrix through the shared-memory pipe.  (stencil_h16.cuh reads both operands of every MMA from
//   shared memory and is bound by that pipe from nrhs 32 up.)
// * N side = the stencil matrix, K-major without swizzle: 8 x 8 core matrices of binary16 (128 contiguous bytes), the
//   tile stored in HBM as [k chunk of 8][n group of 8] with n = (hi/lo, Re/Im, row i): 8 nb^2 bytes for ANY nb that is a
//   multiple of 8 (no padding bytes in HBM: same size as complex64); one 1-D bulk copy per stencil matrix.
//   MMA 1: X_hi^T . [A_hi | A_lo] -> D | C (N = 4 nb), MMA 2: X_lo^T . A_hi -> C (N = 2 nb), per K = 16 slab of two k chunks.
//   nb = 8, 24 (an odd number of k chunks): the last chunk c pairs its own halves instead of a zero chunk,
//     (X_lo c, X_hi c)^T . (A_hi c ; A_lo c) -> C   and   (X_hi c, 0)^T . (A_hi c ; A_lo c) -> D      (N = 2 nb each)
//   -- A_lo c follows A_hi c in the tile, so a descriptor with half the chunk stride reads them as the two k chunks of a slab; the
//   zero is ONE block of 32 nb bytes in shared memory, which the D slab's descriptor names as its second k chunk (the X side of
//   that half reads the 4 columns after the tile: finite numbers).  nb 24: 240 N x K units per stencil point instead of 288 with
//   a zero chunk in every ring stage, stages of 4608 instead of 6144 bytes, and an X tile of 24 columns: 5 X buffers.
// * A GROUP of up to GMAX x-adjacent sites (4; 3 at nbasis 32, where tensor memory holds no more accumulators) shares
//   every X tile it needs: (G + 2) x 27 tile loads per group instead of 81 G -- the gather of X through L2 is the
//   largest single cost of this kernel (measured: 21-25 % of the time at nrhs 64 with pairs of sites).
// * EVERYTHING THAT SERIALISES IS PER SITE: one accumulator (4 nb TMEM columns), one ring of stencil matrices with its own
//   producer lane, and one MMA-issuing warp per site of the group.  A single warp's dependent instruction stream
//   (barrier tests, descriptor arithmetic, 4 MMAs + 2 commits per stencil point: 600-1000 clk) is what bounds an issuer,
//   not the tensor pipe (144-192 clk per point): the sites' accumulators are independent, so their streams need no order.
//   Barriers are per site too: a parity wait cannot tell phases two apart, so every barrier has exactly one waiter
//   that sees each of its phases (X buffers: full / empty barriers per site; the loader warps of a buffer keep who used it last).
// * One persistent CTA per SM: 16 loader warps, 4 epilogue warps, one producer warp for the stencil matrices (lane i feeds
//   site i), one producer warp for the X tiles (32 source addresses computed at once), GMAX MMA issuers.
// Measured (B200, 1000 W cap): BASELINE configs[4] (16^3 x 32, nbasis 24) 15.3-15.9 ms per apply at nrhs 64 = 0.50-0.52 of the
// HBM roof (the TF32 kernel: 31.5 ms), 12.6 ms at nrhs 32 (0.61), 11.5 ms at nrhs 16 (0.66).  The board sits at its power cap
// at every width (SM clock 1.1 GHz at nrhs 64, 1.45 at 16): with the MMAs, the loaders' moves, the stencil-matrix bytes or the
// X-tile bytes left out (-DCMRHS_ABL=1..4: wrong results, timing only) the kernel takes 10.5 / 12.7 / 10.9 / 13.2 ms at nrhs 64
// but the SAME 17-18 M cycles per CTA -- less work buys clock, not cycles: energy per apply is the bound.
#pragma once
#ifndef CMRHS_ABL
#define CMRHS_ABL 0        // 1 no MMAs, 2 loaders move nothing, 3 / 4 the bulk copies of stencil matrices / X tiles carry 16 bytes: TIMING ONLY
#endif

#include "stencil_h16.cuh"

namespace cmrhs {

constexpr int kXMaxStagesA = 32;              // per site
constexpr int kXMaxBuf = 8;
constexpr int kXMaxSX = 24;                   // stages of the shared-memory ring of X tiles
constexpr int kXMaxG = 4;
constexpr int kXMaxSteps = 168;               // (G + 2) x 27 + G at G = 4: 166
constexpr int kXViews = kXMaxG * (kXMaxG + 1) / 2;      // per-site views of the schedules of G = 1..4

template <int NB> struct XCfg {
    static_assert(NB % 8 == 0 && NB >= 8 && NB <= 32, "h16x: nbasis in {8,16,24,32}");
    static constexpr int KSTEPS = (NB + 15) / 16;               // K = 16 slabs per stencil matrix
    static constexpr int NCH = NB / 8;                           // 8-wide k chunks that carry data
    static constexpr uint32_t LBO = 64u * NB;                    // bytes between k chunks: 4 nb / 8 core matrices of 128 B
    static constexpr uint32_t SBO = 128u;                        // bytes between n groups
    static constexpr uint32_t TILE_BYTES = 8u * NB * NB;         // one stencil matrix, [A_hi | A_lo]
    static constexpr uint32_t STAGE_BYTES = TILE_BYTES;          // ring stage
    static constexpr int ACC_COLS = 4 * NB;                      // D (2 nb) | C (2 nb) per site
    // TMEM columns of one X tile, 4 per k chunk ("slot").  Even NCH: [X_hi 0 .. NCH-1 | X_lo 0 .. NCH-1].  Odd NCH (nb = 8, 24), whose
    // last chunk c has no partner for a K = 16 slab: [X_hi 0 .. c-1 | X_lo 0 .. c-1 | X_lo c | X_hi c] -- the slab (X_lo c, X_hi c)
    // meets (A_hi c ; A_lo c) and gives both C products of the chunk at once; the slab (X_hi c, whatever follows: the next buffer's
    // first slot, always finite binary16 numbers) meets (A_hi c ; a block of zeros in shared memory) for D.
    static constexpr int ODD = NCH % 2;
    static constexpr int KFULL = NCH / 2;                        // K = 16 slabs made of two data chunks
    static constexpr int XLO = 4 * (NCH - ODD);                  // X_lo of the full slabs
    static constexpr int XC = 8 * (NCH - ODD);                   // odd NCH: (X_lo c, X_hi c)
    static constexpr int XD = XC + 4;                            //          (X_hi c, the 4 columns after the tile)
    static constexpr int XCOLS = 8 * NCH;
    static constexpr uint32_t ZERO_BYTES = 32u * NB;             // one k chunk of 2 nb n rows
    // tensor-memory plan (512 columns): sites per group, accumulator slots (one per site of a group; one spare at nbasis 32),
    // X buffers of XCOLS = nb columns
    static constexpr int GMAX = NB == 32 ? 3 : 4;                // (nb 24 with 3, nb 32 with 2 sites and twice the X buffers: 15 % / 7 % slower -- the issuers bound it)
    static constexpr int NACC = GMAX;                            // accumulator slot i belongs to site i of every group (its MMA warp is the one waiter)
#ifndef CMRHS_XLOAD
#define CMRHS_XLOAD 1       // 1: loader warps carry the X tile from the shared-memory ring to tensor memory (tcgen05.st); 0: tcgen05.cp movers
#endif
#ifndef CMRHS_XTURNS
#define CMRHS_XTURNS 4
#endif
#ifndef CMRHS_XTURNS24
#define CMRHS_XTURNS24 5    // nbasis 24: tensor memory has room for 5 X buffers beside 4 accumulators, and a buffer keeps its loader turn
#endif
    static constexpr bool LOAD = CMRHS_XLOAD != 0;
    static constexpr int TURNS = NB == 24 ? CMRHS_XTURNS24 : CMRHS_XTURNS;                   // loader warps per TMEM lane quarter, taking turns tile by tile
    static constexpr int NXB_FIT = (512 - NACC * ACC_COLS) / XCOLS > kXMaxBuf ? kXMaxBuf : (512 - NACC * ACC_COLS) / XCOLS;
    static constexpr int NXB = LOAD ? NXB_FIT / TURNS * TURNS : NXB_FIT;      // (a buffer always meets the same loader turn / mover)
    static constexpr int MOVERS = LOAD ? TURNS : NXB;            // owners of X buffers and ring stages: tile t belongs to owner t mod MOVERS
    static constexpr int XBASE = NACC * ACC_COLS;
    static constexpr int MWARPS = LOAD ? 4 * TURNS : (MOVERS + 3) / 4 * 4;      // (the epilogue warps must start at a multiple of 4)
    static constexpr int WARPS = MWARPS + 4 + 2 + GMAX;
    static constexpr int THREADS = 32 * WARPS;
    static_assert(XBASE + NXB * XCOLS + 4 * ODD <= 512 && NXB >= 4 && NXB <= kXMaxBuf && NXB % MOVERS == 0, "tensor memory plan");
    static_assert(NACC >= GMAX, "one accumulator per site of a group");
};

struct XParams {
    int32_t L[4];
    int32_t ng0, ngroups;
    int32_t s, N2;            // nrhs, 2 nrhs = real columns of an X tile = M rows in use
    int32_t m32;              // N2 rounded up to a multiple of 32: rows of one chunk of the split X tile
    int32_t nq;               // TMEM lane quarters in use = m32 / 32
    int32_t sa;               // depth of each site's ring of stencil matrices
    int32_t sx;               // depth of the ring of X tiles (even: a stage always meets the same loader turn)
    int32_t xh_site_bytes;    // bytes of one split X tile: 2 (hi, lo) x NCH x m32 x 16
    uint32_t idesc_wide, idesc_lo;
    float inv_sA;
    const uint32_t *amax;
};

// Schedule of a group of G <= 4 x-adjacent sites x0 .. x0+G-1: one step per X tile, the sites that use it accumulate it.
// tab entry:  bits 0-3 user mask | 4-6 j (the tile sits at x' = x0 + j - 1) | 8-9 dy+1 | 10-11 dz+1 | 12-13 dt+1
// view entry (one per stencil point of site i, in the order the site accumulates them):  bits 0-7 step | 16-22 point p
// Order: the 26 non-centre (dy,dz,dt) offsets first, then the centre offset's dx = -1, +1 points, each site's own centre point
// (p = 40, which carries c*I) last: the running float32 sums stay small until the large term arrives.
__device__ inline int hx_build_schedule(int G, uint32_t *tab, uint32_t *view /* [G][84] */)
{
    int n = 0, cnt[kXMaxG] = {0, 0, 0, 0};
    auto emit = [&](int o, int j, bool centre_pass, int only) {
        uint32_t um = 0;
        for (int i = 0; i < G; ++i) {
            const int dx = j - 1 - i;
            if (dx < -1 || dx > 1) continue;
            if (only >= 0 ? i != only : (centre_pass && dx == 0)) continue;
            um |= 1u << i;
            view[i * 84 + cnt[i]++] = (uint32_t)n | ((uint32_t)((dx + 1) + 3 * o) << 16);
        }
        if (um) tab[n++] = um | ((uint32_t)j << 4) | ((uint32_t)(o % 3) << 8) | ((uint32_t)((o / 3) % 3) << 10) | ((uint32_t)(o / 9) << 12);
    };
    for (int o = 0; o < 27; ++o) {
        if (o == 13) continue;
        for (int j = 0; j < G + 2; ++j) emit(o, j, false, -1);
    }
    for (int j = 0; j < G + 2; ++j) emit(13, j, true, -1);
    for (int i = 0; i < G; ++i) emit(13, i + 1, false, i);
    return n;
}

struct XGroup { int x0, G, y, z, t, nsteps; const uint32_t *tab; const uint32_t *view; };

template <int NB>
__global__ void __launch_bounds__(XCfg<NB>::THREADS, 1)
stencil_h16x_kernel(const unsigned char *__restrict__ Ax, const unsigned char *__restrict__ Xh, float *__restrict__ Y, const XParams P)
{
    using C = XCfg<NB>;
    constexpr int GMAX = C::GMAX;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    unsigned char *smem = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
    unsigned char *ringA = smem;                 // GMAX rings of P.sa stages: site i's stencil matrices at ring i
    unsigned char *ringX = ringA + (size_t)GMAX * P.sa * C::STAGE_BYTES;        // P.sx pre-split X tiles (+ 2 KB the tail reads of a short tile may touch)
    uint32_t *tabs = reinterpret_cast<uint32_t *>(ringX + (size_t)P.sx * P.xh_site_bytes + 2048);     // [G-1][kXMaxSteps]
    uint32_t *views = tabs + kXMaxG * kXMaxSteps;                        // [G (G-1) / 2 + i][84]
    int32_t *nsteps = reinterpret_cast<int32_t *>(views + kXViews * 84); // [G-1]
    float *inv = reinterpret_cast<float *>(nsteps + 4);                  // [128] per real column: 1 / (sA sX_r)
    uint64_t *bars = reinterpret_cast<uint64_t *>(inv + 128);
    uint64_t *a_full = bars, *a_empty = a_full + kXMaxG * kXMaxStagesA;              // [site][stage]
    uint64_t *x_full = a_empty + kXMaxG * kXMaxStagesA, *x_empty = x_full + kXMaxG * kXMaxBuf;      // [site][buffer]
    uint64_t *acc_full = x_empty + kXMaxG * kXMaxBuf, *acc_empty = acc_full + kXMaxBuf;            // [slot]
    uint64_t *x_land = acc_empty + kXMaxBuf, *x_sfree = x_land + kXMaxSX;                          // [stage of the X ring]
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(x_sfree + kXMaxSX);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int kWEpi = C::MWARPS, kWProd = kWEpi + 4, kWProdX = kWProd + 1, kWMma = kWProd + 2;
#ifdef CMRHS_TC_TRACE
    long long wt[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    const long long t_begin = clock64();
#endif

    if (threadIdx.x == 0) {
        for (int j = 0; j < GMAX; ++j) {
            for (int i = 0; i < P.sa; ++i) { mbar_init(&a_full[j * kXMaxStagesA + i], 1); mbar_init(&a_empty[j * kXMaxStagesA + i], 1); }
            for (int i = 0; i < C::NXB; ++i) { mbar_init(&x_full[j * kXMaxBuf + i], C::LOAD ? (uint32_t)P.nq : 1u); mbar_init(&x_empty[j * kXMaxBuf + i], 1); }
        }
        for (int i = 0; i < C::NACC; ++i) { mbar_init(&acc_full[i], 1); mbar_init(&acc_empty[i], 4); }
        for (int i = 0; i < P.sx; ++i) { mbar_init(&x_land[i], 1); mbar_init(&x_sfree[i], C::LOAD ? (uint32_t)P.nq : 1u); }
        mbar_fence_init();
    }
    if (warp >= 1 && warp <= GMAX && lane == 0) {
        const int G = warp;
        nsteps[G - 1] = hx_build_schedule(G, tabs + (G - 1) * kXMaxSteps, views + (G * (G - 1) / 2) * 84);
    }
    if (threadIdx.x >= 256 && threadIdx.x < 384) {
        const int col = threadIdx.x - 256;
        const float sc = col < P.N2 ? h_scale_from_bits(P.amax[col >> 1]) : 1.0f;
        inv[col] = P.inv_sA / sc;
    }
    if constexpr (C::ODD) {      // the block of zeros the odd D slab reads as its second k chunk: the first bytes of the slack after the X ring
        if (threadIdx.x < C::ZERO_BYTES / 16) reinterpret_cast<uint4 *>(ringX + (size_t)P.sx * P.xh_site_bytes)[threadIdx.x] = make_uint4(0u, 0u, 0u, 0u);
        fence_proxy_async_smem();
    }
    if (warp == kWProd) tmem_alloc_cols(tmem_slot, 512u);
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();
    const uint32_t tmem = *tmem_slot;
    if (warp >= kWEpi && warp < kWEpi + 4) {
        // the X buffers (and the 4 columns after the last one, which the odd slab of that buffer reads) start as zeros; so do the lanes
        // of quarters no loader writes (the MMAs read all 128 lanes: finite numbers, rows nobody reads)
        uint32_t zz[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) zz[k] = 0u;
        for (int cc = 0; cc < (C::NXB * C::XCOLS + 4 * C::ODD + 15) / 16 * 16 && C::XBASE + cc + 16 <= 512; cc += 16) tmem_st_x16(tmem + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)(C::XBASE + cc), zz);
        tmem_wait_st();
    }
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();

    auto group_of = [&](int g) {
        XGroup r;
        const int gx = g % P.ng0;
        int line = g / P.ng0;
        r.x0 = gx * GMAX;
        r.G = min(GMAX, P.L[0] - r.x0);
        r.y = line % P.L[1]; line /= P.L[1];
        r.z = line % P.L[2];
        r.t = line / P.L[2];
        r.nsteps = nsteps[r.G - 1];
        r.tab = tabs + (r.G - 1) * kXMaxSteps;
        r.view = views + (r.G * (r.G - 1) / 2) * 84;
        return r;
    };
    auto site_of = [&](int x, int y, int z, int t) { return x + (int64_t)P.L[0] * (y + (int64_t)P.L[1] * (z + (int64_t)P.L[2] * t)); };

    if (C::LOAD && warp < kWEpi) {
        // ================= X loaders: pre-split tile (shared-memory ring, filled by bulk copies) -> registers -> tensor memory (tcgen05.st).
        // tcgen05.cp would do this without threads, but it runs in the tensor pipe's own queue at 64 B/clk: 12 KB per tile = 192 clk during
        // which no MMA runs (measured at configs[4]: 3.6 of 16.1 ms); tcgen05.st writes 256 B/clk beside the MMAs. =================
        const int q = warp & 3, turn = warp >> 2;
        if (q < P.nq) {
            const uint32_t lane_base = tmem + ((uint32_t)(32 * q) << 16) + (uint32_t)C::XBASE;
            const uint32_t row_off = (uint32_t)(32 * q + lane) * 16u, chunk_stride = (uint32_t)P.m32 * 16u;
            int cg = blockIdx.x, cstep = 0;       // cursor in the sequence of X tiles this CTA walks
            bool more = cg < P.ngroups;
            XGroup grp;
            if (more) grp = group_of(cg);
            TcRing rs;                            // stage of the X ring that holds the cursor's tile
            auto skip = [&](int n) {
                for (int k = 0; k < n && more; ++k) {
                    rs.advance(P.sx);
                    if (++cstep == grp.nsteps) {
                        cstep = 0;
                        cg += gridDim.x;
                        more = cg < P.ngroups;
                        if (more) grp = group_of(cg);
                    }
                }
            };
            skip(turn);
            uint32_t t = (uint32_t)turn, pend = 0u, par = 0u;      // per buffer and site: who used the last tile stored there, parity of that site's next release
            while (more) {
                const uint32_t um = grp.tab[cstep] & 15u;
                const uint32_t b = t % (uint32_t)C::NXB;
                TW(2, mbar_wait(&x_land[rs.stage], rs.phase));
                const unsigned char *src = ringX + (size_t)rs.stage * P.xh_site_bytes + row_off;
                uint32_t w[8 * C::NCH];
#pragma unroll
                for (int c = 0; c < (CMRHS_ABL == 2 ? 0 : 2 * C::NCH); ++c) {
                    const uint4 v = *reinterpret_cast<const uint4 *>(src + (size_t)c * chunk_stride);
                    w[4 * c + 0] = v.x; w[4 * c + 1] = v.y; w[4 * c + 2] = v.z; w[4 * c + 3] = v.w;
                }
                fence_proxy_async_smem();         // this warp's reads of the stage are done before a bulk copy may overwrite it
                __syncwarp();
                if (lane == 0) mbar_arrive(&x_sfree[rs.stage]);
#pragma unroll
                for (int i = 0; i < GMAX; ++i) {
                    const uint32_t bit = 1u << (4u * b + i);
                    if (pend & bit) {
                        TW(0, mbar_wait(&x_empty[i * kXMaxBuf + b], (par & bit) ? 1u : 0u));
                        par ^= bit;
                    }
                }
                pend = (pend & ~(15u << (4u * b))) | (um << (4u * b));
                tc_fence_after_sync();
                TW_BEGIN();
                const uint32_t dst = lane_base + b * (uint32_t)C::XCOLS;
                if constexpr (CMRHS_ABL == 2) {
                } else if constexpr (C::NCH == 1) {
                    tmem_st_x8(dst, reinterpret_cast<const uint32_t (&)[8]>(w[0]));
                } else {
                    tmem_st_x16(dst, reinterpret_cast<const uint32_t (&)[16]>(w[0]));
                    if constexpr (C::NCH == 3) tmem_st_x8(dst + 16u, reinterpret_cast<const uint32_t (&)[8]>(w[16]));
                    if constexpr (C::NCH == 4) tmem_st_x16(dst + 16u, reinterpret_cast<const uint32_t (&)[16]>(w[16]));
                }
                tmem_wait_st();
                tc_fence_before_sync();
                __syncwarp();
                if (lane < GMAX && ((um >> lane) & 1u)) mbar_arrive(&x_full[lane * kXMaxBuf + b]);
                TW_END(1);
                t += C::TURNS;
                skip(C::TURNS);
            }
        }
    } else
    if (warp < kWEpi) {
        // ================= X movers: tile (shared-memory ring, filled by bulk copies) -> tensor memory by tcgen05.cp; warp m takes the
        // tiles t = m (mod MOVERS) and with them always the same X buffers and ring stages; one elected lane issues =================
        const int mv = warp;
        if (mv < C::MOVERS) {
            int cg = blockIdx.x, cstep = 0;
            bool more = cg < P.ngroups;
            XGroup grp;
            if (more) grp = group_of(cg);
            TcRing rs;
            auto skip = [&](int n) {
                for (int k = 0; k < n && more; ++k) {
                    rs.advance(P.sx);
                    if (++cstep == grp.nsteps) {
                        cstep = 0;
                        cg += gridDim.x;
                        more = cg < P.ngroups;
                        if (more) grp = group_of(cg);
                    }
                }
            };
            skip(mv);
            const uint32_t ringx0 = smem_u32(ringX), chunk_stride = (uint32_t)P.m32 * 16u;
            const uint64_t desc_hi = umma_desc_kmajor_noswz(0u, chunk_stride, 128u);      // LBO: next k chunk, SBO: next 8 rows
            uint32_t t = (uint32_t)mv, pend = 0u, par = 0u;
            while (more) {
                const uint32_t um = grp.tab[cstep] & 15u;
                const uint32_t b = t % (uint32_t)C::NXB;
                TW(2, mbar_wait(&x_land[rs.stage], rs.phase));
#pragma unroll
                for (int i = 0; i < GMAX; ++i) {
                    const uint32_t bit = 1u << (4u * b + i);
                    if (pend & bit) {
                        TW(0, mbar_wait(&x_empty[i * kXMaxBuf + b], (par & bit) ? 1u : 0u));
                        par ^= bit;
                    }
                }
                pend = (pend & ~(15u << (4u * b))) | (um << (4u * b));
                tc_fence_after_sync();
                TW_BEGIN();
                if (elect_one_sync()) {
                    const uint32_t src = ringx0 + (uint32_t)rs.stage * (uint32_t)P.xh_site_bytes;
                    const uint32_t dst = tmem + (uint32_t)C::XBASE + b * (uint32_t)C::XCOLS;
#pragma unroll
                    for (int c = 0; c < 2 * C::NCH; c += 2)            // the tile's 2 NCH slots of 4 columns, two per copy
                        tmem_cp_128x256b(dst + (uint32_t)(4 * c), desc_hi | (uint64_t)(((src + (uint32_t)c * chunk_stride) >> 4) & 0x3FFFu));
#pragma unroll
                    for (int i = 0; i < GMAX; ++i)
                        if ((um >> i) & 1u) umma_commit(&x_full[i * kXMaxBuf + b]);
                    umma_commit(&x_sfree[rs.stage]);
                }
                __syncwarp();
                TW_END(1);
                t += C::MOVERS;
                skip(C::MOVERS);
            }
        }
    }
    else if (warp < kWEpi + 4) {
        // ================= epilogue: Y = combine((D + 2^-11 C) / (sA sX)) -> global, one site per accumulator slot =================
        // lanes = real columns n = (r, re/im), columns = (hi/lo, part, i):  Y_re = P[(r,0)] - Q[(r,1)],  Y_im = P[(r,1)] + Q[(r,0)]
        const int q = warp - kWEpi;                       // = warp % 4: the TMEM lane quarter this warp may access
        const uint32_t lane_base = tmem + ((uint32_t)(32 * q) << 16);
        const int n = 32 * q + lane, c = n & 1;
        const bool live = n < P.N2;
        const float sc = live ? inv[n] : 0.0f;
        uint32_t fpar = 0u;                               // bit i: parity of slot i's next "full" phase
        for (int g = blockIdx.x; g < P.ngroups; g += gridDim.x) {
            const XGroup grp = group_of(g);
            for (int i = 0; i < grp.G; ++i) {
                TW(0, mbar_wait_long(&acc_full[i], (fpar >> i) & 1u, 256u));
                fpar ^= 1u << i;
                tc_fence_after_sync();
                TW_BEGIN();
                if (q < P.nq) {
                    const uint32_t ds = lane_base + (uint32_t)(i * C::ACC_COLS);
                    float *yrow = Y + site_of(grp.x0 + i, grp.y, grp.z, grp.t) * (int64_t)(NB * P.N2) + n;
#pragma unroll
                    for (int ic = 0; ic < NB / 8; ++ic) {
                        uint32_t dp[8], dq[8], cp[8], cq[8];
                        tmem_ld_x8(ds + (uint32_t)(8 * ic), dp);
                        tmem_ld_x8(ds + (uint32_t)(NB + 8 * ic), dq);
                        tmem_ld_x8(ds + (uint32_t)(2 * NB + 8 * ic), cp);
                        tmem_ld_x8(ds + (uint32_t)(3 * NB + 8 * ic), cq);
                        tmem_wait_ld();
#pragma unroll
                        for (int k = 0; k < 8; ++k) {
                            const float pv = (__uint_as_float(dp[k]) + __uint_as_float(cp[k]) * (1.0f / 2048.0f)) * sc;
                            const float qv = (__uint_as_float(dq[k]) + __uint_as_float(cq[k]) * (1.0f / 2048.0f)) * sc;
                            const float qo = __shfl_xor_sync(0xffffffffu, qv, 1);
                            const float val = c == 0 ? pv - qo : pv + qo;
                            if (live) yrow[(int64_t)(8 * ic + k) * P.N2] = val;
                        }
                    }
                }
                tc_fence_before_sync();
                __syncwarp();
                if (lane == 0) mbar_arrive(&acc_empty[i]);
                TW_END(1);
            }
        }
    } else if (warp == kWProd) {
        // ================= A producer: ONE warp running one uniform polling loop, LANE i < GMAX on site i's ring, barrier and cursor:
        // the site's 81 pre-split stencil matrices, each one contiguous bulk copy, in the order the site accumulates them =================
        const int me = lane;
        const uint64_t pol = l2_policy_evict_first();
        const int ring_no = me < GMAX ? me : 0;
        unsigned char *ring = ringA + (size_t)ring_no * P.sa * C::STAGE_BYTES;
        uint64_t *full = a_full + ring_no * kXMaxStagesA, *empty = a_empty + ring_no * kXMaxStagesA;
        TcRing ra;
        int g = blockIdx.x, k = 0;
        bool active = me < GMAX && g < P.ngroups;
        const unsigned char *src0 = nullptr;
        const uint32_t *tm = nullptr;
        auto enter_group = [&]() {               // skips the groups that have no site `me`
            while (active) {
                const XGroup grp = group_of(g);
                if (me < grp.G) {
                    tm = grp.view + me * 84;
                    src0 = Ax + (site_of(grp.x0 + me, grp.y, grp.z, grp.t) * kNPoint) * (int64_t)C::TILE_BYTES;
                    return;
                }
                g += gridDim.x;
                active = g < P.ngroups;
            }
        };
        enter_group();
        while (__any_sync(0xffffffffu, active)) {
            if (active && mbar_test_wait(&empty[ra.stage], ra.phase ^ 1u)) {
                const uint32_t p = (tm[k] >> 16) & 0x7Fu;
                constexpr uint32_t kCopy = CMRHS_ABL == 3 ? 16u : C::TILE_BYTES;
                mbar_arrive_expect_tx(&full[ra.stage], kCopy);
                bulk_g2s(ring + (size_t)ra.stage * C::STAGE_BYTES, src0 + (size_t)p * C::TILE_BYTES, kCopy, &full[ra.stage], pol);
                ra.advance(P.sa);
                if (++k == kNPoint) {
                    k = 0;
                    g += gridDim.x;
                    active = g < P.ngroups;
                    enter_group();
                }
            }
        }
    } else if (warp == kWProdX) {
        // ================= X producer: the pre-split tile of every step (contiguous in the scratch block), one bulk copy each.  The source
        // addresses of 32 steps are computed at once, one per lane (the wrap arithmetic is most of this warp's work: one lane at a time
        // it was busy 78 % of the kernel); then the copies are issued step by step =================
        const uint64_t pol = l2_policy_evict_last();
        TcRing rs;
        for (int g = blockIdx.x; g < P.ngroups; g += gridDim.x) {
            const XGroup grp = group_of(g);
            for (int s0 = 0; s0 < grp.nsteps; s0 += 32) {
                const int nb_ = min(32, grp.nsteps - s0);
                unsigned long long mine_src = 0ull;
                if (lane < nb_) {
                    const uint32_t e = grp.tab[s0 + lane];
                    const int xs = tc_wrap(grp.x0 + (int)((e >> 4) & 7u) - 1, P.L[0]), ys = tc_wrap(grp.y + (int)((e >> 8) & 3u) - 1, P.L[1]);
                    const int zs = tc_wrap(grp.z + (int)((e >> 10) & 3u) - 1, P.L[2]), ts = tc_wrap(grp.t + (int)((e >> 12) & 3u) - 1, P.L[3]);
                    mine_src = (unsigned long long)(uintptr_t)(Xh + (int64_t)(xs + P.L[0] * (ys + P.L[1] * (zs + P.L[2] * ts))) * (int64_t)P.xh_site_bytes);
                }
                for (int j = 0; j < nb_; ++j) {
                    const unsigned char *src = reinterpret_cast<const unsigned char *>((uintptr_t)__shfl_sync(0xffffffffu, mine_src, j));
                    TW(0, mbar_wait(&x_sfree[rs.stage], rs.phase ^ 1u));
                    if (lane == 0) {
                        const uint32_t xcopy = CMRHS_ABL == 4 ? 16u : (uint32_t)P.xh_site_bytes;
                        mbar_arrive_expect_tx(&x_land[rs.stage], xcopy);
                        bulk_g2s(ringX + (size_t)rs.stage * P.xh_site_bytes, src, xcopy, &x_land[rs.stage], pol);
                    }
                    rs.advance(P.sx);
                }
            }
        }
    } else if (warp < kWMma + GMAX) {
        // ================= MMA issuers, one warp PER SITE of a group; one elected lane issues.  The barrier tests of the NEXT stencil
        // point are started before the MMAs of this one (non-blocking test_wait), so their latency overlaps the issue. =================
        const int me = warp - kWMma;
        const uint32_t ring0 = smem_u32(ringA + (size_t)me * P.sa * C::STAGE_BYTES);
        const uint32_t x_base = tmem + (uint32_t)C::XBASE;
        uint64_t *afull = a_full + me * kXMaxStagesA, *aempty = a_empty + me * kXMaxStagesA;
        uint64_t *xfull = x_full + me * kXMaxBuf, *xempty = x_empty + me * kXMaxBuf;
        const uint64_t desc_hi = umma_desc_kmajor_noswz(0u, C::LBO, C::SBO);      // everything but the start address
        const uint64_t desc_odd = umma_desc_kmajor_noswz(0u, C::LBO / 2, C::SBO); // k chunk 0 = A_hi, k chunk 1 = A_lo of ONE chunk (2 nb n rows each)
        const uint64_t desc_zero = umma_desc_kmajor_noswz(0u, 0u, C::SBO);        // k chunk 0 = A_hi of that chunk, k chunk 1 = the block of zeros (LBO per stage)
        const uint32_t zero_addr = smem_u32(ringX + (size_t)P.sx * P.xh_site_bytes);
        TcRing ra;
        uint32_t epar = 1u;                       // parity to wait for on this site's "accumulator empty" barrier (first wait passes)
        uint32_t xcnt = 0;                        // X tiles before this group
        uint32_t xpar = 0u;                       // bit b: parity of this site's next "full" phase of X buffer b
        for (int g = blockIdx.x; g < P.ngroups; g += gridDim.x) {
            const XGroup grp = group_of(g);
            if (me < grp.G) {
                const uint32_t *tm = grp.view + me * 84;
                const uint32_t ds = tmem + (uint32_t)(me * C::ACC_COLS);
                TW(0, mbar_wait(&acc_empty[me], epar));
                epar ^= 1u;
                uint32_t xb = (xcnt + (tm[0] & 0xFFu)) % (uint32_t)C::NXB;
                bool okx = false, oka = false;
                for (int k = 0; k < kNPoint; ++k) {
                    if (!okx) TW(2, mbar_wait(&xfull[xb], (xpar >> xb) & 1u));
                    xpar ^= 1u << xb;
                    if (!oka) TW(1, mbar_wait(&afull[ra.stage], ra.phase));
                    tc_fence_after_sync();
                    TcRing rn = ra;
                    rn.advance(P.sa);
                    uint32_t xbn = 0u;
                    if (k + 1 < kNPoint) {
                        xbn = (xcnt + (tm[k + 1] & 0xFFu)) % (uint32_t)C::NXB;
                        okx = mbar_test_wait(&xfull[xbn], (xpar >> xbn) & 1u);
                        oka = mbar_test_wait(&afull[rn.stage], rn.phase);
                    }
                    TW_BEGIN();
                    if (elect_one_sync()) {
                        const uint32_t x_hi = x_base + xb * (uint32_t)C::XCOLS, x_lo = x_hi + (uint32_t)C::XLO;
                        const uint64_t bd0 = desc_hi | (uint64_t)(((ring0 + (uint32_t)ra.stage * C::STAGE_BYTES) >> 4) & 0x3FFFu);
#if CMRHS_ABL != 1
#pragma unroll
                        for (int ks = 0; ks < C::KFULL; ++ks) {
                            const uint64_t bd = bd0 + (uint64_t)((uint32_t)ks * 2u * C::LBO >> 4);
                            umma_f16_ts(ds, x_hi + 8u * ks, bd, P.idesc_wide, (k | ks) ? 1u : 0u);      // X_hi^T . [A_hi | A_lo] -> D | C
                            umma_f16_ts(ds + 2u * NB, x_lo + 8u * ks, bd, P.idesc_lo, 1u);              // X_lo^T . A_hi -> C
                        }
                        if constexpr (C::ODD) {   // the last chunk c: two full-rate N = 2 nb slabs instead of two half-empty N = 4 nb, 2 nb ones
                            const uint32_t ac = ring0 + (uint32_t)ra.stage * C::STAGE_BYTES + (uint32_t)(C::NCH - 1) * C::LBO;
                            const uint64_t bo = desc_odd | (uint64_t)((ac >> 4) & 0x3FFFu);
                            const uint64_t bz = desc_zero | (uint64_t)((ac >> 4) & 0x3FFFu) | ((uint64_t)(((zero_addr - ac) >> 4) & 0x3FFFu) << 16);
                            umma_f16_ts(ds + 2u * NB, x_hi + (uint32_t)C::XC, bo, P.idesc_lo, (k | C::KFULL) ? 1u : 0u);      // (X_lo c, X_hi c)^T . (A_hi c ; A_lo c) -> C
                            umma_f16_ts(ds, x_hi + (uint32_t)C::XD, bz, P.idesc_lo, (k | C::KFULL) ? 1u : 0u);                // (X_hi c, any)^T . (A_hi c ; 0) -> D
                        }
#endif
                        umma_commit(&aempty[ra.stage]);
                        umma_commit(&xempty[xb]);
                        if (k == kNPoint - 1) umma_commit(&acc_full[me]);
                    }
                    __syncwarp();
                    TW_END(3);
                    ra = rn;
                    xb = xbn;
                }
            }
            xcnt += (uint32_t)grp.nsteps;
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
    if (warp == kWProd) tmem_dealloc_cols(tmem, 512u);
}

// ---- host side ------------------------------------------------------------------------------------------------
inline bool h16x_supported(int nb, int s) { return (nb == 8 || nb == 16 || nb == 24 || nb == 32) && s >= 1 && s <= 64; }
inline int h16x_m32(int s) { return (2 * s + 31) / 32 * 32; }
// bytes of one split X tile
inline int h16x_site_bytes(int nb, int s) { return 2 * (nb / 8) * h16x_m32(s) * 16; }

// create-time re-layout: canonical A[t][i][k] (complex64) -> Ax[t] = [k chunk c][n group][n % 8][k % 8] binary16, n = (h, part, i):
// the K-major, unswizzled shared-memory image of the N x K operand [A_hi | A_lo] (8 x 8 core matrices, 128 B each).
// One thread per (c, part, i): 8 consecutive complex values in, one 16-byte row of a hi core matrix and of a lo core matrix out.
__global__ void __launch_bounds__(256) relayout_h16x_kernel(const cplx<float> *__restrict__ A, unsigned char *__restrict__ Ax, int64_t ntiles, int nb,
                                                            float sA)
{
    const int nch = nb / 8, items = nch * 2 * nb;
    const int64_t tile_bytes = 8ll * nb * nb;
    for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const cplx<float> *src = A + t * nb * nb;
        unsigned char *dst = Ax + t * tile_bytes;
        for (int e = threadIdx.x; e < items; e += 256) {
            const int c = e / (2 * nb), pi = e - c * 2 * nb, part = pi / nb, i = pi - part * nb;
            uint32_t hw[4], lw[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const cplx<float> v0 = src[i * nb + 8 * c + 2 * u], v1 = src[i * nb + 8 * c + 2 * u + 1];
                const float a0 = (part ? v0.im : v0.re) * sA, a1 = (part ? v1.im : v1.re) * sA;
                const __half2 h = __floats2half2_rn(a0, a1);
                const float2 hf = __half22float2(h);
                const __half2 l = __floats2half2_rn((a0 - hf.x) * 2048.0f, (a1 - hf.y) * 2048.0f);
                hw[u] = *reinterpret_cast<const uint32_t *>(&h);
                lw[u] = *reinterpret_cast<const uint32_t *>(&l);
            }
            const int n_hi = pi, n_lo = 2 * nb + pi;
            unsigned char *base = dst + (int64_t)c * 64 * nb;
            *reinterpret_cast<uint4 *>(base + (n_hi >> 3) * 128 + (n_hi & 7) * 16) = make_uint4(hw[0], hw[1], hw[2], hw[3]);
            *reinterpret_cast<uint4 *>(base + (n_lo >> 3) * 128 + (n_lo & 7) * 16) = make_uint4(lw[0], lw[1], lw[2], lw[3]);
        }
    }
}

// per-apply pre-pass: X (fp32, [site][k][2 s real columns]) -> Xh[site][slot][m32 rows] of 16 bytes: the 8 binary16 values
// k = 8 c .. 8 c + 7 of real column n, scaled by the column's power of two and split (hi = fp16(x), lo = fp16(2^11 (x - hi)));
// slot = the group of 4 TMEM columns the chunk goes to (XCfg).
// Rows n >= 2 s of a chunk are never written (zeroed once at create).
__global__ void __launch_bounds__(256) xsplit_x_kernel(const float *__restrict__ X, unsigned char *__restrict__ Xh, const uint32_t *__restrict__ amax,
                                                       int64_t nsites, int nb, int s, int m32, int site_bytes)
{
    __shared__ float scl[128];
    const int N2 = 2 * s, nch = nb / 8, items = nch * N2;
    if (threadIdx.x < 128) scl[threadIdx.x] = threadIdx.x < N2 ? h_scale_from_bits(amax[threadIdx.x >> 1]) : 1.0f;
    __syncthreads();
    for (int64_t site = blockIdx.x; site < nsites; site += gridDim.x) {
        const float *src = X + site * (int64_t)(nb * N2);
        unsigned char *dst = Xh + site * (int64_t)site_bytes;
        for (int e = threadIdx.x; e < items; e += 256) {
            const int c = e / N2, n = e - c * N2;
            const float sc = scl[n];
            uint32_t hw[4], lw[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const float x0 = src[(8 * c + 2 * u) * N2 + n] * sc, x1 = src[(8 * c + 2 * u + 1) * N2 + n] * sc;
                const __half2 h = __floats2half2_rn(x0, x1);
                const float2 hf = __half22float2(h);
                const __half2 l = __floats2half2_rn((x0 - hf.x) * 2048.0f, (x1 - hf.y) * 2048.0f);
                hw[u] = *reinterpret_cast<const uint32_t *>(&h);
                lw[u] = *reinterpret_cast<const uint32_t *>(&l);
            }
            const bool last_odd = (nch & 1) && c == nch - 1;       // slots as the TMEM columns of XCfg: odd nch ends with (lo c, hi c)
            const int hi_slot = last_odd ? 2 * c + 1 : c, lo_slot = last_odd ? 2 * c : (nch - (nch & 1)) + c;
            *reinterpret_cast<uint4 *>(dst + ((int64_t)hi_slot * m32 + n) * 16) = make_uint4(hw[0], hw[1], hw[2], hw[3]);
            *reinterpret_cast<uint4 *>(dst + ((int64_t)lo_slot * m32 + n) * 16) = make_uint4(lw[0], lw[1], lw[2], lw[3]);
        }
    }
}

template <int NB>
int launch_stencil_h16x(const unsigned char *Ax, float inv_sA, uint32_t *amax_dev, unsigned char *Xh, const LatticeDims &d, const void *X,
                        void *Y, int s, int num_sms, cudaStream_t stream, bool have_colmax)
{
    using C = XCfg<NB>;
    XParams P;
    for (int k = 0; k < 4; ++k) P.L[k] = d.L[k];
    P.ng0 = (d.L[0] + C::GMAX - 1) / C::GMAX;
    P.ngroups = (int32_t)((int64_t)P.ng0 * d.L[1] * d.L[2] * d.L[3]);
    P.s = s;
    P.N2 = 2 * s;
    P.m32 = h16x_m32(s);
    P.nq = P.m32 / 32;
    P.xh_site_bytes = h16x_site_bytes(NB, s);
    const int64_t fixed = 128 /* alignment */ + (kXMaxG * kXMaxSteps + kXViews * 84 + 4) * 4 + 512 /* scales */ +
                          (2 * kXMaxG * kXMaxStagesA + 2 * kXMaxG * kXMaxBuf + 2 * kXMaxBuf + 2 * kXMaxSX) * 8 + 16;
    // shared memory: about a third for the ring of X tiles (an even number of stages), the rest for the sites' rings of stencil matrices
    const int64_t budget = 226 * 1024 - fixed - 2048;
    P.sx = (int32_t)(budget / 3 / P.xh_site_bytes);
    if (P.sx > kXMaxSX) P.sx = kXMaxSX;
    P.sx = P.sx / C::MOVERS * C::MOVERS;          // a stage always meets the same loader turn (or tcgen05.cp mover)
    if (P.sx < C::MOVERS) P.sx = C::MOVERS;
    P.sa = (int32_t)((budget - (int64_t)P.sx * P.xh_site_bytes) / (C::GMAX * (int64_t)C::STAGE_BYTES));
    if (P.sa > kXMaxStagesA) P.sa = kXMaxStagesA;
    if (P.sa < 2) { set_error("h16x: shared-memory plan does not fit (nbasis %d, nrhs %d)", NB, s); return COARSE_UNSUPPORTED; }
    P.idesc_wide = umma_idesc_f16_kk(128, 4 * NB);
    P.idesc_lo = umma_idesc_f16_kk(128, 2 * NB);
    P.inv_sA = inv_sA;
    P.amax = amax_dev;
    const size_t smem = (size_t)fixed + 2048 + (size_t)C::GMAX * P.sa * C::STAGE_BYTES + (size_t)P.sx * P.xh_site_bytes;

    if (!have_colmax) {
        CMRHS_CUDA(cudaMemsetAsync(amax_dev, 0, 64 * sizeof(uint32_t), stream));
        const int64_t n = d.V * NB;
        const int rpp = 256 / s;
        const int cgrid = (int)(ceil_div(n, rpp) < (int64_t)num_sms * 8 ? ceil_div(n, rpp) : (int64_t)num_sms * 8);
        colmax_kernel<<<cgrid, 256, 0, stream>>>(static_cast<const float2 *>(X), n, s, amax_dev);
        CMRHS_LAUNCH_CHECK();
    }
    const int xgrid = (int)(d.V < (int64_t)num_sms * 8 ? d.V : (int64_t)num_sms * 8);
    xsplit_x_kernel<<<xgrid, 256, 0, stream>>>(static_cast<const float *>(X), Xh, amax_dev, d.V, NB, s, P.m32, P.xh_site_bytes);
    CMRHS_LAUNCH_CHECK();

    auto kern = stencil_h16x_kernel<NB>;
    CMRHS_SMEM_ATTR(kern, smem);
    const int grid = P.ngroups < num_sms ? P.ngroups : num_sms;
    kern<<<grid, C::THREADS, smem, stream>>>(Ax, Xh, static_cast<float *>(Y), P);
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}

}  // namespace cmrhs

// Tensor-core stencil-GEMM kernel for complex64 on sm_100a (tcgen05 + TMEM + TMA), split-TF32 (3 products).
//   Y(x) = sum_{p=0}^{80} A^p(x) . X(x + delta_p)                       (Eq. 19)
//
// Mapping of the complex block product onto tcgen05.mma.kind::tf32:
//   P[(site,i)][(r,c)] += sum_j Re A(site)[i][j] * X(y)[j][(r,c)]      Q likewise with Im A
//   Y_re = P[.,(r,0)] - Q[.,(r,1)],   Y_im = P[.,(r,1)] + Q[.,(r,0)]     (combined once, in the epilogue)
// * M side (128 TMEM lanes) = TWO lattice sites adjacent along x, each with its Re panel and its Im panel stacked
//   (lane quarter q: site slot q/2, part q%2): one accumulator of N = 2 nrhs columns serves both parts, an X tile
//   X(y) is shared by the x-neighbours, so a group of two sites takes 110 MMA steps instead of 162 (26 x 4 columns
//   of neighbours + the centre offset swept so that each site's centre point comes last).
// * The stencil matrices (the HBM stream: 81 nb^2 complex per site) are kept in a planar, k-major internal layout
//   Ak[x][p][part][k][i] (part 0 = Re, 1 = Im; written once by coarse_op_create): a whole matrix is one contiguous
//   1-D bulk copy, and "one thread = one matrix row i" reads of a column k are 32 consecutive floats (conflict free,
//   no swizzle, any nbasis).  The converter warps (three per TMEM lane quarter, taking turns step by step) split
//   every element into TF32 hi (round to nearest) + lo = x - hi (exact; the tensor core keeps its leading 11 bits)
//   and write the operand panels (hi | lo) into TMEM with tcgen05.st.  A is never re-written to shared memory.
// * N side = the neighbour's X tile exactly as it lies in memory ([j][r][re,im] = K x N, N contiguous: an
//   MN-major UMMA operand, layout SWIZZLE_128B_BASE32B), loaded by TMA with the matching swizzle (128B_ATOM_32B);
//   four warps round it to TF32 in place and write the lo tile beside it.
// * Products: Ahi.Xhi -> main accumulator D; Alo.Xhi + Ahi.Xlo -> correction accumulator C (the tensor core adds
//   into its FP32 accumulator with truncation: keeping the small products apart spares D two thirds of the
//   additions); Y = D + C is formed with a round-to-nearest add in the epilogue.
// * Accumulation order: the 80 off-centre points first, the centre point (which carries c*I) last.
// * Warp roles (768 threads, one persistent CTA per SM): 0-11 A converters (three per lane quarter, taking turns),
//   12-15 X converters, 16-19 epilogue, 20 A producer (bulk copies), 21 X producer (TMA), 22 MMA issuer,
//   23 TMEM allocator.  All hand-offs are mbarriers; the step schedule is a table in shared memory.
#pragma once

#include "setup_kernels.cuh"
#include "tcgen05_ptx.cuh"

namespace cmrhs {

constexpr int kTcThreads = 768;
constexpr int kTcConvTurns = 3;        // A converter warps per TMEM lane quarter
constexpr int kTcMaxStagesA = 32;
constexpr int kTcMaxStagesX = 8;
constexpr int kTcMaxSets = 6;
constexpr int kTcSetCols = 64;          // TMEM columns of one operand panel set: hi at +0, lo at +32
constexpr int kTcMaxSteps = 112;

struct TcParams {
    int32_t L[4];
    int32_t ng0;          // groups per x-line = ceil(L0 / 2)
    int32_t ngroups;      // ng0 * L1 * L2 * L3
    int32_t s;            // nrhs (multiple of 8)
    int32_t N;            // 2 s: MMA N
    int32_t nxb;          // ceil(N / 32): 128-byte wide blocks per X tile (MN-major TF32 operands exist only in the
                          // SWIZZLE_128B_BASE32B layout: 32 floats along N per row, 32-byte chunks swizzled over 4 K rows)
    int32_t xt_bytes;     // bytes of one X tile, rounded up to 1024
    int32_t x_tile_tx;    // bytes TMA delivers per X tile
    int32_t sa, sx;       // ring depths
    int32_t nacc, nset;   // accumulator buffers, operand panel sets (even)
    int32_t acc_stride;   // TMEM columns per accumulator buffer: D at +0, C at +N (wide: D | C' | C'' at +0, +32, +64)
    int32_t wide;         // 1: N <= 32, the X hi and lo tiles form one 64-column operand and A_hi meets both in ONE MMA
    uint32_t idesc;
    uint32_t idesc_wide;  // M 128, N 64
    uint64_t xdesc_base;  // shared-memory descriptor of an X tile without the address
    uint32_t x_kadv;      // bytes between consecutive K = 8 steps of an X tile
};

template <int NB> struct TcCfg {
    static_assert(NB % 8 == 0 && NB >= 8 && NB <= 32, "tensor path: nbasis in {8,16,24,32}");
    static constexpr uint32_t PART_FLOATS = NB * NB;                 // one part (Re or Im) of a tile: [k][i]
    static constexpr uint32_t TILE_BYTES = 2 * NB * NB * 4;
    static constexpr uint32_t STAGE_BYTES = (TILE_BYTES + 127u) / 128u * 128u;
    static constexpr int KSTEPS = NB / 8;
};

// ---- schedule ---------------------------------------------------------------------------------------------------
// A group = G <= 2 sites x0, x0+1 of one x-line.  Step table entry (one MMA step = one X tile):
//   bits 0-4  off3 = (dy+1) + 3(dz+1) + 9(dt+1)        bits 5-7  j: the X tile sits at x' = x0 + j - 1
//   bits 8-9  user mask (site slot i uses the tile, dx = j - 1 - i)     bits 10-11 / 12-13  dx + 1 of slot 0 / 1
__host__ __device__ inline int tc_build_schedule(int G, uint32_t *tab)
{
    int n = 0;
    const int W = G + 2;
    for (int o = 0; o < 27; ++o) {
        if (o == 13) continue;
        for (int j = 0; j < W; ++j) {
            uint32_t um = 0, e = (uint32_t)o | ((uint32_t)j << 5);
            for (int i = 0; i < G; ++i) {
                const int dx = j - 1 - i;
                if (dx >= -1 && dx <= 1) { um |= 1u << i; e |= (uint32_t)(dx + 1) << (10 + 2 * i); }
            }
            tab[n++] = e | (um << 8);
        }
    }
    for (int j = 0; j < W; ++j) {          // centre offset in y, z, t: the dx != 0 points first ...
        uint32_t um = 0, e = 13u | ((uint32_t)j << 5);
        for (int i = 0; i < G; ++i) {
            const int dx = j - 1 - i;
            if (dx == -1 || dx == 1) { um |= 1u << i; e |= (uint32_t)(dx + 1) << (10 + 2 * i); }
        }
        if (um) tab[n++] = e | (um << 8);
    }
    for (int i = 0; i < G; ++i)            // ... and each site's own centre point (p = 40, carries c*I) last
        tab[n++] = 13u | ((uint32_t)(i + 1) << 5) | ((1u << i) << 8) | (1u << (10 + 2 * i));
    return n;                              // 110 (G = 2) or 81 (G = 1)
}

struct TcGroup { int x0, G, y, z, t, nsteps; const uint32_t *tab; };

__device__ __forceinline__ TcGroup tc_group(const TcParams &P, int g, const uint32_t *tab2, const uint32_t *tab1)
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
__device__ __forceinline__ int tc_wrap(int c, int L) { return c < 0 ? c + L : (c >= L ? c - L : c); }
__device__ __forceinline__ int64_t tc_site(const TcParams &P, int x, int y, int z, int t)
{
    return x + (int64_t)P.L[0] * (y + (int64_t)P.L[1] * (z + (int64_t)P.L[2] * t));
}
__device__ __forceinline__ int64_t tc_x_site(const TcParams &P, const TcGroup &g, uint32_t e)
{
    const int off3 = (int)(e & 31u), j = (int)((e >> 5) & 7u);
    const int dy = off3 % 3 - 1, dz = (off3 / 3) % 3 - 1, dt = off3 / 9 - 1;
    return tc_site(P, tc_wrap(g.x0 + j - 1, P.L[0]), tc_wrap(g.y + dy, P.L[1]), tc_wrap(g.z + dz, P.L[2]), tc_wrap(g.t + dt, P.L[3]));
}

struct TcRing {     // stage / phase bookkeeping of an mbarrier ring
    int stage = 0;
    uint32_t phase = 0;
    __device__ __forceinline__ void advance(int depth) { if (++stage == depth) { stage = 0; phase ^= 1u; } }
};

__device__ __forceinline__ void tc_named_barrier(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// Optional per-role cycle accounting (compile with -DCMRHS_TC_TRACE; read back with coarse_debug_trace_read):
// TW(k, wait) adds the cycles spent in `wait` to slot k of the warp's counters; slot 7 is the warp's total.
#ifdef CMRHS_TC_TRACE
__device__ long long g_tc_trace[160][32][8];
#define TW(k, ...) do { const long long _t0 = clock64(); __VA_ARGS__; wt[k] += clock64() - _t0; } while (0)
#define TW_BEGIN() const long long _tw = clock64()
#define TW_END(k) wt[k] += clock64() - _tw
#else
#define TW(k, ...) do { __VA_ARGS__; } while (0)
#define TW_BEGIN() do {} while (0)
#define TW_END(k) do {} while (0)
#endif

template <int NB>
__global__ void __launch_bounds__(kTcThreads, 1)
stencil_tc_kernel(const float *__restrict__ Ak, const __grid_constant__ CUtensorMap tmX, float2 *__restrict__ Y,
                  const TcParams P)
{
    using C = TcCfg<NB>;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    // carve: [X ring (hi|lo per stage), 1024-byte aligned for the swizzle][A ring][epilogue exchange][schedule tables][barriers][tmem slot]
    unsigned char *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);     // keeps the shared address space
    unsigned char *ringX = smem;
    unsigned char *ringA = ringX + (size_t)P.sx * 2 * P.xt_bytes;
    float4 *exch = reinterpret_cast<float4 *>(ringA + (size_t)P.sa * C::STAGE_BYTES);      // [pair 2][buf 2][part 2][j 2][lane 32]
    uint32_t *tab2 = reinterpret_cast<uint32_t *>(exch + 2 * 2 * 2 * 2 * 32);
    uint32_t *tab1 = tab2 + kTcMaxSteps;
    uint64_t *bars = reinterpret_cast<uint64_t *>(tab1 + kTcMaxSteps);
    uint64_t *a_full = bars, *a_empty = a_full + kTcMaxStagesA;
    uint64_t *x_full = a_empty + kTcMaxStagesA, *x_empty = x_full + kTcMaxStagesX, *xlo_full = x_empty + kTcMaxStagesX;
    uint64_t *set_full = xlo_full + kTcMaxStagesX, *set_empty = set_full + kTcMaxSets;
    uint64_t *acc_full = set_empty + kTcMaxSets, *acc_empty = acc_full + 2;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(acc_empty + 2);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#ifdef CMRHS_TC_TRACE
    long long wt[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    const long long t_begin = clock64();
#endif

    if (threadIdx.x == 0) {
        for (int i = 0; i < P.sa; ++i) { mbar_init(&a_full[i], 1); mbar_init(&a_empty[i], 2); }
        for (int i = 0; i < P.sx; ++i) { mbar_init(&x_full[i], 1); mbar_init(&x_empty[i], 1); mbar_init(&xlo_full[i], 4); }
        for (int i = 0; i < P.nset; ++i) { mbar_init(&set_full[i], 4); mbar_init(&set_empty[i], 1); }
        for (int i = 0; i < 2; ++i) { mbar_init(&acc_full[i], 1); mbar_init(&acc_empty[i], 4); }
        mbar_fence_init();
    }
    if (threadIdx.x == 32) tc_build_schedule(2, tab2);
    if (threadIdx.x == 64) tc_build_schedule(1, tab1);
    if (warp == 4 * kTcConvTurns + 11) tmem_alloc_512(tmem_slot);
    if (warp == 4 * kTcConvTurns + 9 && lane == 0) tma_prefetch_desc(&tmX);
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();
    const uint32_t tmem = *tmem_slot;
    const uint32_t acc_cols = (uint32_t)(P.nacc * P.acc_stride);

    if (warp < 4 * kTcConvTurns) {
        // ================= A converters: smem tile column k, row = lane -> TF32 hi/lo of the Re or Im panel -> TMEM =================
        const int q = warp & 3, turn_mine = warp >> 2;
        const int slot = q >> 1, part = q & 1;
        const uint32_t lane_base = tmem + ((uint32_t)(32 * q) << 16);
        const bool row_ok = lane < NB;
        const uint32_t row_off = (uint32_t)part * C::PART_FLOATS + (uint32_t)(row_ok ? lane : 0);
        TcRing ra, rs;                  // ra: position of the NEXT tile of the tile sequence; rs: panel set of this step
        uint32_t zero_sets = 0;         // panel sets whose lanes of this quarter hold zeros (every warp of the quarter tracks all sets)
        int turn = 0;                   // running step counter mod kTcConvTurns: the warp whose turn it is fills this step's set
        for (int g = blockIdx.x; g < P.ngroups; g += gridDim.x) {
            const TcGroup grp = tc_group(P, g, tab2, tab1);
            for (int step = 0; step < grp.nsteps; ++step) {
                const uint32_t e = grp.tab[step];
                const uint32_t um = (e >> 8) & 3u;
                const bool mine = (um >> slot) & 1u;
                if (turn == turn_mine) {
                    TW(0, mbar_wait(&set_empty[rs.stage], rs.phase ^ 1u));
                    tc_fence_after_sync();
                    TW_BEGIN();
                    const uint32_t set_col = acc_cols + (uint32_t)rs.stage * kTcSetCols;
                    if (mine) {
                        TcRing mt = ra;                                   // my tile: sequence position + rank among the users
                        if (slot == 1 && (um & 1u)) mt.advance(P.sa);
                        TW(1, mbar_wait(&a_full[mt.stage], mt.phase));
                        const float *col = reinterpret_cast<const float *>(ringA + (size_t)mt.stage * C::STAGE_BYTES) + row_off;
#pragma unroll
                        for (int kc = 0; kc < NB / 8; ++kc) {
                            float x[8];
#pragma unroll
                            for (int u = 0; u < 8; ++u) x[u] = col[(kc * 8 + u) * NB];
                            uint32_t hi[8], lo[8];
#pragma unroll
                            for (int u = 0; u < 8; ++u) {
                                const float v = row_ok ? x[u] : 0.f;
                                const float h = tf32_rn(v);
                                hi[u] = __float_as_uint(h);
                                lo[u] = __float_as_uint(v - h);
                            }
                            tmem_st_x8(lane_base + set_col + (uint32_t)(kc * 8), hi);
                            tmem_st_x8(lane_base + set_col + 32u + (uint32_t)(kc * 8), lo);
                        }
                        __syncwarp();
                        if (lane == 0) mbar_arrive(&a_empty[mt.stage]);      // all lanes have read the tile
                    } else if (!((zero_sets >> rs.stage) & 1u)) {
                        uint32_t zz[16];
#pragma unroll
                        for (int k = 0; k < 16; ++k) zz[k] = 0u;
#pragma unroll
                        for (int b = 0; b < kTcSetCols / 16; ++b) tmem_st_x16(lane_base + set_col + 16u * b, zz);
                    }
                    tmem_wait_st();
                    tc_fence_before_sync();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&set_full[rs.stage]);
                    TW_END(2);
                }
                zero_sets = mine ? (zero_sets & ~(1u << rs.stage)) : (zero_sets | (1u << rs.stage));
                rs.advance(P.nset);
                ra.advance(P.sa);
                if (um == 3u) ra.advance(P.sa);
                turn = (turn + 1 == kTcConvTurns) ? 0 : turn + 1;
            }
        }
    } else if (warp < 4 * kTcConvTurns + 4) {
        // ================= X converters: round the tile to TF32 in place (hi), write the lo tile =================
        const int tid = threadIdx.x - 32 * 4 * kTcConvTurns;
        const int nchunks = P.nxb * NB * 8;     // 16-byte chunks per X tile (whole 128-byte rows, zero padded by TMA)
        TcRing rx;
        for (int g = blockIdx.x; g < P.ngroups; g += gridDim.x) {
            const int nsteps = (min(2, P.L[0] - (g % P.ng0) * 2) == 2) ? 110 : 81;
            for (int step = 0; step < nsteps; ++step) {
                TW(0, mbar_wait(&x_full[rx.stage], rx.phase));
                TW_BEGIN();
                unsigned char *hi_t = ringX + (size_t)rx.stage * 2 * P.xt_bytes;
                unsigned char *lo_t = hi_t + P.xt_bytes;
                int c = tid;
                for (; c + 128 < nchunks; c += 256) {          // two chunks per trip: both loads in flight
                    const float4 v0 = *reinterpret_cast<const float4 *>(hi_t + 16 * c);
                    const float4 v1 = *reinterpret_cast<const float4 *>(hi_t + 16 * (c + 128));
                    const float4 h0 = make_float4(tf32_rn(v0.x), tf32_rn(v0.y), tf32_rn(v0.z), tf32_rn(v0.w));
                    const float4 h1 = make_float4(tf32_rn(v1.x), tf32_rn(v1.y), tf32_rn(v1.z), tf32_rn(v1.w));
                    *reinterpret_cast<float4 *>(hi_t + 16 * c) = h0;
                    *reinterpret_cast<float4 *>(lo_t + 16 * c) = make_float4(v0.x - h0.x, v0.y - h0.y, v0.z - h0.z, v0.w - h0.w);
                    *reinterpret_cast<float4 *>(hi_t + 16 * (c + 128)) = h1;
                    *reinterpret_cast<float4 *>(lo_t + 16 * (c + 128)) = make_float4(v1.x - h1.x, v1.y - h1.y, v1.z - h1.z, v1.w - h1.w);
                }
                if (c < nchunks) {
                    const float4 v = *reinterpret_cast<const float4 *>(hi_t + 16 * c);
                    const float4 h = make_float4(tf32_rn(v.x), tf32_rn(v.y), tf32_rn(v.z), tf32_rn(v.w));
                    *reinterpret_cast<float4 *>(hi_t + 16 * c) = h;
                    *reinterpret_cast<float4 *>(lo_t + 16 * c) = make_float4(v.x - h.x, v.y - h.y, v.z - h.z, v.w - h.w);
                }
                fence_proxy_async_smem();       // generic-proxy writes -> visible to the tensor core's async-proxy reads
                __syncwarp();
                if (lane == 0) mbar_arrive(&xlo_full[rx.stage]);
                TW_END(1);
                rx.advance(P.sx);
            }
        }
    } else if (warp < 4 * kTcConvTurns + 8) {
        // ================= epilogue: Y = combine(D + C) -> global =================
        const int q = warp - (4 * kTcConvTurns + 4);      // = warp % 4: the TMEM lane quarter this warp may access
        const int slot = q >> 1, part = q & 1;
        const uint32_t lane_base = tmem + ((uint32_t)(32 * q) << 16);
        float4 *xb = exch + slot * (2 * 2 * 2 * 32);
        TcRing rc;
        uint32_t chunk_no = 0;          // running chunk counter: selects the exchange buffer
        for (int g = blockIdx.x; g < P.ngroups; g += gridDim.x) {
            const TcGroup grp = tc_group(P, g, tab2, tab1);
            TW(0, mbar_wait(&acc_full[rc.stage], rc.phase));
            tc_fence_after_sync();
            TW_BEGIN();
            if (slot < grp.G) {
                const uint32_t d = lane_base + (uint32_t)(rc.stage * P.acc_stride), cacc = d + (uint32_t)(P.wide ? 32 : P.N);
                const int64_t site = tc_site(P, grp.x0 + slot, grp.y, grp.z, grp.t);
                float2 *yrow = Y + (site * NB + (lane < NB ? lane : 0)) * (int64_t)P.s;
                for (int c = 0; c < P.N / 16; ++c, ++chunk_no) {
                    uint32_t a[16], b[16];
                    tmem_ld_x16(d + 16u * c, a);
                    tmem_ld_x16(cacc + 16u * c, b);
                    float v[16];
                    if (P.wide) {
                        uint32_t b2[16];
                        tmem_ld_x16(d + 64u + 16u * c, b2);
                        tmem_wait_ld();
#pragma unroll
                        for (int k = 0; k < 16; ++k) v[k] = __uint_as_float(a[k]) + (__uint_as_float(b[k]) + __uint_as_float(b2[k]));
                    } else {
                        tmem_wait_ld();
#pragma unroll
                        for (int k = 0; k < 16; ++k) v[k] = __uint_as_float(a[k]) + __uint_as_float(b[k]);
                    }
                    // the Re-panel warp finishes right-hand sides 8c..8c+3 and needs the partner's columns 0-7;
                    // the Im-panel warp finishes 8c+4..8c+7 and needs the partner's columns 8-15
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
                    if (lane < NB) {
                        float4 *dst = reinterpret_cast<float4 *>(yrow + 8 * c + 4 * part);
                        dst[0] = r0;
                        dst[1] = r1;
                    }
                }
            }
            tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) mbar_arrive(&acc_empty[rc.stage]);
            TW_END(1);
            rc.advance(P.nacc);
        }
    } else if (warp == 4 * kTcConvTurns + 8) {
        // ================= A producer: one stencil matrix (planar k-major tile, contiguous) per stage =================
        // (the whole warp walks the schedule so that every address stays warp-uniform; one elected lane issues)
        const uint64_t pol = l2_policy_evict_first();
        TcRing ra;
        for (int g = blockIdx.x; g < P.ngroups; g += gridDim.x) {
            const TcGroup grp = tc_group(P, g, tab2, tab1);
            const int64_t site0 = tc_site(P, grp.x0, grp.y, grp.z, grp.t);
            for (int step = 0; step < grp.nsteps; ++step) {
                const uint32_t e = grp.tab[step];
                const int off3 = (int)(e & 31u);
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    if (!((e >> (8 + i)) & 1u)) continue;
                    const int p = (int)((e >> (10 + 2 * i)) & 3u) + 3 * off3;
                    const float *src = Ak + ((site0 + i) * kNPoint + p) * (int64_t)(2 * C::PART_FLOATS);
                    TW(0, mbar_wait(&a_empty[ra.stage], ra.phase ^ 1u));
                    if (elect_one_sync()) {
                        mbar_arrive_expect_tx(&a_full[ra.stage], C::TILE_BYTES);
                        bulk_g2s(ringA + (size_t)ra.stage * C::STAGE_BYTES, src, C::TILE_BYTES, &a_full[ra.stage], pol);
                    }
                    __syncwarp();
                    ra.advance(P.sa);
                }
            }
        }
    } else if (warp == 4 * kTcConvTurns + 9) {
        // ================= X producer: the neighbour's X tile, once per step =================
        const uint64_t pol = l2_policy_evict_last();
        TcRing rx;
        for (int g = blockIdx.x; g < P.ngroups; g += gridDim.x) {
            const TcGroup grp = tc_group(P, g, tab2, tab1);
            for (int step = 0; step < grp.nsteps; ++step) {
                const int64_t row0 = tc_x_site(P, grp, grp.tab[step]) * NB;
                TW(0, mbar_wait(&x_empty[rx.stage], rx.phase ^ 1u));
                if (elect_one_sync()) {
                    mbar_arrive_expect_tx(&x_full[rx.stage], (uint32_t)P.x_tile_tx);
                    unsigned char *dst = ringX + (size_t)rx.stage * 2 * P.xt_bytes;
                    for (int b = 0; b < P.nxb; ++b)
                        tma_load_2d(dst + (size_t)b * NB * 128, &tmX, b * 32, (int32_t)row0, &x_full[rx.stage], pol);
                }
                __syncwarp();
                rx.advance(P.sx);
            }
        }
    } else if (warp == 4 * kTcConvTurns + 10) {
        // ================= MMA issuer =================
        // The whole warp runs the loop (all operands stay warp-uniform: no per-instruction broadcast loops in SASS);
        // one elected lane -- the same one every time -- issues the MMAs and the commits.
        TcRing rx, rs, rc;
        for (int g = blockIdx.x; g < P.ngroups; g += gridDim.x) {
            const int nsteps = (min(2, P.L[0] - (g % P.ng0) * 2) == 2) ? 110 : 81;
            TW(0, mbar_wait(&acc_empty[rc.stage], rc.phase ^ 1u));
            tc_fence_after_sync();
            const uint32_t d = tmem + (uint32_t)(rc.stage * P.acc_stride), cacc = d + (uint32_t)P.N;
            for (int step = 0; step < nsteps; ++step) {
                TW(1, mbar_wait(&set_full[rs.stage], rs.phase));
                TW(2, mbar_wait(&xlo_full[rx.stage], rx.phase));
                tc_fence_after_sync();
                TW_BEGIN();
                if (elect_one_sync()) {
                    const uint32_t a_hi = tmem + acc_cols + (uint32_t)rs.stage * kTcSetCols, a_lo = a_hi + 32u;
                    const uint32_t xhi = smem_u32(ringX + (size_t)rx.stage * 2 * P.xt_bytes), xlo = xhi + (uint32_t)P.xt_bytes;
#pragma unroll
                    for (int ks = 0; ks < C::KSTEPS; ++ks) {
                        const uint64_t bh = umma_smem_desc(P.xdesc_base, xhi + ks * P.x_kadv);
                        const uint64_t bl = umma_smem_desc(P.xdesc_base, xlo + ks * P.x_kadv);
                        const uint32_t acc = (step | ks) != 0 ? 1u : 0u;
                        if (P.wide) {
                            umma_tf32_ts(d, a_hi + 8u * ks, bh, P.idesc_wide, acc);      // A hi . [X hi | X lo] -> D | C'
                            umma_tf32_ts(d + 64u, a_lo + 8u * ks, bh, P.idesc, acc);     // A lo . X hi -> C''
                        } else {
                            umma_tf32_ts(d, a_hi + 8u * ks, bh, P.idesc, acc);       // A hi . X hi
                            umma_tf32_ts(cacc, a_lo + 8u * ks, bh, P.idesc, acc);    // A lo . X hi
                            umma_tf32_ts(cacc, a_hi + 8u * ks, bl, P.idesc, 1u);     // A hi . X lo
                        }
                    }
                    umma_commit(&set_empty[rs.stage]);
                    umma_commit(&x_empty[rx.stage]);
                    if (step == nsteps - 1) umma_commit(&acc_full[rc.stage]);
                }
                __syncwarp();
                TW_END(3);
                rs.advance(P.nset);
                rx.advance(P.sx);
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
    if (warp == 4 * kTcConvTurns + 11) tmem_dealloc_512(tmem);
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
int launch_stencil_tc(const float *Ak, const LatticeDims &d, const void *X, void *Y, int s, int num_sms, cudaStream_t stream)
{
    using C = TcCfg<NB>;
    if ((reinterpret_cast<uintptr_t>(X) & 15u) || (reinterpret_cast<uintptr_t>(Y) & 15u)) {
        set_error("tensor path: X and Y must be 16-byte aligned");
        return COARSE_INVALID_ARG;
    }
    TcParams P;
    for (int k = 0; k < 4; ++k) P.L[k] = d.L[k];
    P.ng0 = (d.L[0] + 1) / 2;
    P.ngroups = (int32_t)((int64_t)P.ng0 * d.L[1] * d.L[2] * d.L[3]);
    P.s = s;
    P.N = 2 * s;
    P.nxb = (P.N + 31) / 32;
    P.x_tile_tx = P.nxb * NB * 128;           // TMA counts the whole box, out-of-range columns are zero filled
    P.xt_bytes = (P.x_tile_tx + 1023) / 1024 * 1024;
    // tensor memory: accumulator buffers of 2 N columns (main D | correction C), the rest in panel sets of 64 columns
    P.wide = (P.nxb == 1) ? 1 : 0;
    P.acc_stride = P.wide ? 96 : 2 * P.N;
    P.nacc = (2 * P.acc_stride <= 256) ? 2 : 1;
    P.nset = (512 - P.nacc * P.acc_stride) / kTcSetCols;
    if (P.nset > kTcMaxSets) P.nset = kTcMaxSets;
    // (any converter warp may fill any set: turns go by step mod 3, sets by step mod nset)
    P.sx = 64 * 1024 / (2 * P.xt_bytes);
    if (P.sx > kTcMaxStagesX) P.sx = kTcMaxStagesX;
    if (P.sx < 3) P.sx = 3;
    const int64_t fixed = 1024 /* alignment */ + 2 * 2 * 2 * 2 * 32 * 16 /* exchange */ + 2 * kTcMaxSteps * 4 + 1024 /* barriers */ + 128 /* A ring alignment */;
    const int64_t budget = 225 * 1024 - fixed - (int64_t)P.sx * 2 * P.xt_bytes;
    P.sa = (int32_t)(budget / C::STAGE_BYTES);
    if (P.sa > kTcMaxStagesA) P.sa = kTcMaxStagesA;
    if (P.sa < 4 || P.nset < 2) { set_error("tensor path: shared/tensor memory plan does not fit (nb %d, nrhs %d)", NB, s); return COARSE_UNSUPPORTED; }
    P.idesc = umma_idesc_tf32(128, P.N, true);
    P.idesc_wide = umma_idesc_tf32(128, 64, true);
    P.xdesc_base = umma_smem_desc_base((uint32_t)(NB * 128), 512u, 1u);     // LBO: next 32 columns, SBO: next 4 K rows
    P.x_kadv = 1024u;                                                         // 8 K rows
    const size_t smem = (size_t)fixed + (size_t)P.sa * C::STAGE_BYTES + (size_t)P.sx * 2 * P.xt_bytes;

    CUtensorMap tmX;
    int st = tc_make_tmap(&tmX, X, (uint64_t)P.N, (uint64_t)d.V * NB, 32u, NB, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B);
    if (st != COARSE_OK) return st;

    auto kern = stencil_tc_kernel<NB>;
    CMRHS_SMEM_ATTR(kern, 227 * 1024);
    const int grid = P.ngroups < num_sms ? P.ngroups : num_sms;
    kern<<<grid, kTcThreads, smem, stream>>>(Ak, tmX, static_cast<float2 *>(Y), P);
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}

// create-time re-layout for the tensor kernel: canonical A[t][i][k] (complex64, interleaved) -> planar k-major
// Ak[t][part][k][i] (float32; part 0 = Re, 1 = Im).  One CTA per tile, coalesced writes.
__global__ void relayout_planar_kernel(const cplx<float> *__restrict__ A, float *__restrict__ Ak, int64_t ntiles, int nb)
{
    const int nn = nb * nb;
    for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const cplx<float> *src = A + t * nn;
        float *dst = Ak + t * 2 * nn;
        for (int e = threadIdx.x; e < nn; e += blockDim.x) {
            const int k = e / nb, i = e % nb;
            const cplx<float> v = src[i * nb + k];
            dst[e] = v.re;
            dst[nn + e] = v.im;
        }
    }
}

}  // namespace cmrhs

// Tiled SIMT stencil-GEMM kernel for sm_100a.
//   Y(x) = sum_{p=0}^{80} A^p(x) . X(x + delta_p)                       (Eq. 19)
//
// B200 design:
//  * persistent CTAs, one per SM, WARPS warps each; every WARP owns whole lattice sites: warp w of the grid
//    handles sites w, w + W_total, w + 2 W_total, ...  and keeps the full NB x S block Y(x) in registers
//    (TM x TN complex accumulators per thread) while it walks the 81 stencil points, so every A element
//    fetched from HBM is reused across all nrhs columns on chip and Y is written exactly once (the paper's
//    formulation does 81 read-modify-writes of C, one per batched-GEMM launch: PAPER.md:320, 587);
//  * every warp runs its OWN STAGES-deep shared-memory ring, filled by 1-D bulk TMA copies
//    (cp.async.bulk + mbarrier complete_tx) that its lane 0 issues: a stage carries KCH = NB/KSPLIT
//    contraction indices of one stencil matrix (k-major tile, the dominant HBM stream, L2 evict-first)
//    and the matching rows of the neighbour's X tile (L2 evict-last).  A warp is the only consumer of its
//    ring, so a stage is re-armed by the warp itself right after it has been consumed: no producer warp,
//    no empty barriers, no cross-warp synchronisation anywhere in the main loop;
//  * the chunk stream of a warp is continuous across its sites, so the ring never drains at a site boundary;
//  * neighbour indices come from the periodic neighbour table (a1): the 81 entries of a site sit in three
//    registers per lane and are broadcast with a shuffle.
#pragma once

#include "common.cuh"
#include "ptx_async.cuh"

namespace cmrhs {

// ---- compile-time configuration -------------------------------------------------------------------------
// NB     : nbasis
// TM, TN : per-thread register tile (rows x columns of Y, complex)
// GC     : thread columns per warp (thread rows GR = 32 / GC);  NB = GR*TM,  nrhs = S = GC*TN exactly
// KSPLIT : a pipeline stage carries KCH = NB/KSPLIT contraction indices of one stencil point
// STAGES : depth of each warp's ring;  WARPS : warps per CTA (one CTA per SM)
template <typename T, int NB_, int TM_, int TN_, int GC_, int KSPLIT_, int STAGES_, int WARPS_>
struct SimtConfig {
    using real = T;
    static constexpr int NB = NB_, TM = TM_, TN = TN_, GC = GC_, KSPLIT = KSPLIT_, STAGES = STAGES_, WARPS = WARPS_;
    static constexpr int GR = 32 / GC;
    static constexpr int S = GC * TN;
    static constexpr int THREADS = WARPS * 32;
    static constexpr int KCH = NB / KSPLIT;
    static constexpr int CPS = kNPoint * KSPLIT;                                // chunks (stages) per site
    static constexpr int VEC16 = 16 / (int)sizeof(cplx<T>);                    // complex elements per 16-byte vector
    static constexpr int VA = (TM % VEC16 == 0) ? VEC16 : 1;                    // vector width of the A (row) loads
    static constexpr int VX = (TN % VEC16 == 0) ? VEC16 : 1;                    // vector width of the X (column) loads
    static constexpr int A_ELEMS = KCH * NB;
    static constexpr int X_ELEMS = KCH * S;
    static constexpr uint32_t A_BYTES = A_ELEMS * sizeof(cplx<T>);
    static constexpr uint32_t X_BYTES = X_ELEMS * sizeof(cplx<T>);
    static constexpr uint32_t STAGE_BYTES = A_BYTES + X_BYTES;
    static constexpr size_t SMEM_BYTES = (size_t)WARPS * STAGES * STAGE_BYTES + (size_t)WARPS * STAGES * sizeof(uint64_t) + 16;
    static_assert(GR * GC == 32 && GR * TM == NB, "thread grid must tile NB rows");
    static_assert(NB % KSPLIT == 0, "KSPLIT must divide NB");
    static_assert(A_BYTES % 16 == 0 && X_BYTES % 16 == 0, "bulk copies need 16-byte multiples");
    static_assert(SMEM_BYTES <= 227 * 1024, "shared memory ring does not fit");
};

// row r (0..TM-1) of a thread -> matrix row; chosen so that one warp-wide vector load touches a
// contiguous, bank-conflict-free run of shared memory
template <class C> __device__ __forceinline__ int simt_row(int gr, int r)
{
    return (r / C::VA) * (C::GR * C::VA) + gr * C::VA + (r % C::VA);
}
template <class C> __device__ __forceinline__ int simt_col(int gc, int c)
{
    return (c / C::VX) * (C::GC * C::VX) + gc * C::VX + (c % C::VX);
}

template <typename T, int N, int V> struct VecLoad;
template <typename T, int N> struct VecLoad<T, N, 1> {
    __device__ static __forceinline__ void run(const cplx<T> *base, int stride_groups, cplx<T> (&out)[N])
    {
#pragma unroll
        for (int g = 0; g < N; ++g) out[g] = base[g * stride_groups];
    }
};
template <int N> struct VecLoad<float, N, 2> {
    __device__ static __forceinline__ void run(const cplx<float> *base, int stride_groups, cplx<float> (&out)[N])
    {
#pragma unroll
        for (int g = 0; g < N / 2; ++g) {
            const float4 v = *reinterpret_cast<const float4 *>(base + g * stride_groups);
            out[2 * g].re = v.x; out[2 * g].im = v.y; out[2 * g + 1].re = v.z; out[2 * g + 1].im = v.w;
        }
    }
};

template <class C>
__global__ void __launch_bounds__(C::THREADS, 1)
stencil_simt_kernel(const cplx<typename C::real> *__restrict__ At, const int32_t *__restrict__ nbr,
                    const cplx<typename C::real> *__restrict__ X, cplx<typename C::real> *__restrict__ Y, int64_t V)
{
    using T = typename C::real;
    using Z = cplx<T>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned char *ring = smem_raw + (size_t)warp * C::STAGES * C::STAGE_BYTES;
    uint64_t *full_bar = reinterpret_cast<uint64_t *>(smem_raw + (size_t)C::WARPS * C::STAGES * C::STAGE_BYTES) + warp * C::STAGES;

    constexpr int NN = C::NB * C::NB;        // elements per stencil matrix
    constexpr int NS = C::NB * C::S;         // elements per site of a vector block
    constexpr unsigned FULL = 0xffffffffu;

    // sites of this warp: first, first + stride, ...
    const int64_t stride = (int64_t)gridDim.x * C::WARPS;
    const int64_t first = (int64_t)blockIdx.x * C::WARPS + warp;
    if (first >= V) return;
    const int64_t nsites = (V - first + stride - 1) / stride;
    const int64_t nchunks = nsites * C::CPS;

    if (lane == 0) {
        for (int st = 0; st < C::STAGES; ++st) mbar_init(&full_bar[st], 1);
        mbar_fence_init();
    }
    __syncwarp();

    uint64_t pol_a = 0, pol_x = 0;
    if (lane == 0) { pol_a = l2_policy_evict_first(); pol_x = l2_policy_evict_last(); }

    // ---- issue side: chunk (site, q, h) of the continuous stream, neighbour row of the site in registers ----
    int64_t ix = first;                       // site whose chunks are being issued
    int iw = 0;                               // chunk index within that site (q * KSPLIT + h)
    int32_t n0, n1, n2;
    auto load_nbr_row = [&](int64_t x) {
        const int32_t *row = nbr + x * kNPoint;
        n0 = row[lane];
        n1 = row[lane + 32];
        n2 = (lane + 64 < kNPoint) ? row[lane + 64] : 0;
    };
    load_nbr_row(ix);
    auto issue = [&](int st) {                // all lanes call; lane 0 issues the two bulk copies of one chunk
        const int q = iw / C::KSPLIT, h = iw % C::KSPLIT;
        const int p = stencil_point_in_order(q);
        const int32_t v = p < 32 ? n0 : (p < 64 ? n1 : n2);
        const int64_t y = __shfl_sync(FULL, v, p & 31);
        if (lane == 0) {
            unsigned char *sb = ring + (size_t)st * C::STAGE_BYTES;
            fence_proxy_async_smem();
            mbar_arrive_expect_tx(&full_bar[st], C::STAGE_BYTES);
            bulk_g2s(sb, At + (ix * kNPoint + p) * (int64_t)NN + h * C::A_ELEMS, C::A_BYTES, &full_bar[st], pol_a);
            bulk_g2s(sb + C::A_BYTES, X + y * (int64_t)NS + h * C::X_ELEMS, C::X_BYTES, &full_bar[st], pol_x);
        }
        if (++iw == C::CPS) {
            iw = 0;
            ix += stride;
            if (ix < V) load_nbr_row(ix);
        }
    };

    // prologue: fill the ring
    int64_t issued = 0;
    for (; issued < C::STAGES && issued < nchunks; ++issued) issue((int)issued);

    // ---- compute side ----
    const int gr = lane / C::GC, gc = lane % C::GC;
    const int row0 = gr * C::VA;
    const int col0 = gc * C::VX;
    Z acc[C::TM][C::TN];
#pragma unroll
    for (int a = 0; a < C::TM; ++a)
#pragma unroll
        for (int b = 0; b < C::TN; ++b) { acc[a][b].re = 0; acc[a][b].im = 0; }

    int64_t cx = first;                       // site being computed
    int cw = 0;                               // chunk index within it
    int st = 0;
    uint32_t parity = 0;
    for (int64_t c = 0; c < nchunks; ++c) {
        mbar_wait(&full_bar[st], parity);
        const unsigned char *sb = ring + (size_t)st * C::STAGE_BYTES;
        const Z *sA = reinterpret_cast<const Z *>(sb) + row0;
        const Z *sX = reinterpret_cast<const Z *>(sb + C::A_BYTES) + col0;
#pragma unroll 4
        for (int k = 0; k < C::KCH; ++k) {
            Z a[C::TM], b[C::TN];
            VecLoad<T, C::TM, C::VA>::run(sA + k * C::NB, C::GR * C::VA, a);
            VecLoad<T, C::TN, C::VX>::run(sX + k * C::S, C::GC * C::VX, b);
#pragma unroll
            for (int i = 0; i < C::TM; ++i)
#pragma unroll
                for (int j = 0; j < C::TN; ++j) cmac(acc[i][j], a[i], b[j]);
        }
        __syncwarp();
        if (issued < nchunks) { issue(st); ++issued; }      // re-arm the stage just consumed
        if (++st == C::STAGES) { st = 0; parity ^= 1u; }

        if (++cw == C::CPS) {                 // site finished: write Y(x) once, start the next site
            Z *yout = Y + cx * (int64_t)NS;
#pragma unroll
            for (int i = 0; i < C::TM; ++i) {
                const int row = simt_row<C>(gr, i);
#pragma unroll
                for (int j = 0; j < C::TN; ++j) {
                    yout[row * C::S + simt_col<C>(gc, j)] = acc[i][j];
                    acc[i][j].re = 0;
                    acc[i][j].im = 0;
                }
            }
            cw = 0;
            cx += stride;
        }
    }
}

template <class C>
int launch_stencil_simt_as(const void *At, const int32_t *nbr, const void *X, void *Y, int64_t V, int num_sms, cudaStream_t stream)
{
    using Z = cplx<typename C::real>;
    auto kern = stencil_simt_kernel<C>;
    CMRHS_SMEM_ATTR(kern, C::SMEM_BYTES);
    const int64_t nctas = (V + C::WARPS - 1) / C::WARPS;
    const int grid = (int)(nctas < num_sms ? nctas : num_sms);
    kern<<<grid, C::THREADS, C::SMEM_BYTES, stream>>>(static_cast<const Z *>(At), nbr, static_cast<const Z *>(X),
                                                       static_cast<Z *>(Y), V);
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}

// Small lattices: with WARPS sites per CTA a lattice of a few hundred sites keeps only a few SMs busy (configs[0]: 256 sites = 16 CTAs of
// 16 warps) and its warps share what ONE SM can pull from L2.  When every site still gets its own warp in a single round, the same
// kernel with 2 or 4 warps per CTA spreads them over more SMs (configs[0]: 53.8 -> 32.8 us).  More rounds are never worth it: a site
// costs its 81 dependent ring turns whatever else runs (6^4 sites on 296 warps: 149 against 58 us for 81 CTAs of 16 warps).
template <class C>
int launch_stencil_simt(const void *At, const int32_t *nbr, const void *X, void *Y, int64_t V, int num_sms, cudaStream_t stream)
{
    using C4 = SimtConfig<typename C::real, C::NB, C::TM, C::TN, C::GC, C::KSPLIT, C::STAGES, 4>;
    using C2 = SimtConfig<typename C::real, C::NB, C::TM, C::TN, C::GC, C::KSPLIT, C::STAGES, 2>;
    if (C::WARPS > 2 && (V + 1) / 2 <= num_sms) return launch_stencil_simt_as<C2>(At, nbr, X, Y, V, num_sms, stream);
    if (C::WARPS > 4 && (V + 3) / 4 <= num_sms) return launch_stencil_simt_as<C4>(At, nbr, X, Y, V, num_sms, stream);
    return launch_stencil_simt_as<C>(At, nbr, X, Y, V, num_sms, stream);
}

}  // namespace cmrhs

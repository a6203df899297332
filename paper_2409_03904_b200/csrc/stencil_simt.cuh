// Tiled SIMT stencil-GEMM kernel for sm_100a.
//   Y(x) = sum_{p=0}^{80} A^p(x) . X(x + delta_p)                       (Eq. 19)
//
// B200 design:
//  * persistent CTAs, one per SM; a CTA works on groups of SITES consecutive lattice sites at a time;
//  * a producer warp streams the stencil matrices A^p(x) (k-major tiles, the dominant HBM stream) and the
//    neighbours' X tiles into a STAGES-deep shared-memory ring with 1-D bulk TMA copies
//    (cp.async.bulk + mbarrier complete_tx), A with an L2 evict-first policy, X with evict-last;
//  * SITES*CB consumer warps: warp (site, column block) owns the NB x CT block of Y(site) in registers
//    (TM x TN complex accumulators per thread) for all 81 stencil points -- every A element fetched from
//    HBM is reused across all nrhs columns on chip and Y is written exactly once (the paper's formulation
//    does 81 read-modify-writes of C);
//  * full/empty mbarriers per stage, no __syncthreads in the main loop.
#pragma once

#include "common.cuh"

namespace cmrhs {

// ---- PTX wrappers: mbarrier + bulk async copy ---------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    while (!mbar_try_wait(bar, parity)) {}
}
__device__ __forceinline__ uint64_t l2_policy_evict_first()
{
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ uint64_t l2_policy_evict_last()
{
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// 1-D bulk copy global -> shared, completion signalled on an mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar, uint64_t policy)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
            smem_u32(dst_smem)),
        "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}

// ---- compile-time configuration -------------------------------------------------------------------------
// NB     : nbasis
// TM, TN : per-thread register tile (rows x columns of Y, complex)
// GC     : thread columns per warp (thread rows GR = 32 / GC);  NB = GR*TM,  CT = GC*TN columns per warp
// SITES  : lattice sites per CTA group;  CB : column blocks per site;  nrhs = CB*CT exactly
// KSPLIT : a pipeline stage carries NB/KSPLIT contraction indices of every site of the group
template <typename T, int NB_, int TM_, int TN_, int GC_, int SITES_, int CB_, int KSPLIT_, int STAGES_>
struct SimtConfig {
    using real = T;
    static constexpr int NB = NB_, TM = TM_, TN = TN_, GC = GC_, SITES = SITES_, CB = CB_, KSPLIT = KSPLIT_, STAGES = STAGES_;
    static constexpr int GR = 32 / GC;
    static constexpr int CT = GC * TN;
    static constexpr int S = CB * CT;
    static constexpr int NWARP = SITES * CB;
    static constexpr int THREADS = (NWARP + 1) * 32;
    static constexpr int KCH = NB / KSPLIT;
    static constexpr int VEC16 = 16 / (int)sizeof(cplx<T>);                    // complex elements per 16-byte vector
    static constexpr int VA = (TM % VEC16 == 0) ? VEC16 : 1;                    // vector width of the A (row) loads
    static constexpr int VX = (TN % VEC16 == 0) ? VEC16 : 1;                    // vector width of the X (column) loads
    static constexpr int A_ELEMS = KCH * NB;                                    // per site per stage
    static constexpr int X_ELEMS = KCH * S;
    static constexpr uint32_t A_BYTES = A_ELEMS * sizeof(cplx<T>);
    static constexpr uint32_t X_BYTES = X_ELEMS * sizeof(cplx<T>);
    static constexpr uint32_t STAGE_BYTES = SITES * (A_BYTES + X_BYTES);
    static constexpr size_t SMEM_BYTES = (size_t)STAGES * STAGE_BYTES + 2 * STAGES * sizeof(uint64_t) + 16;
    static_assert(GR * GC == 32 && GR * TM == NB, "thread grid must tile NB rows");
    static_assert(NB % KSPLIT == 0, "KSPLIT must divide NB");
    static_assert(A_BYTES % 16 == 0 && X_BYTES % 16 == 0, "bulk copies need 16-byte multiples");
    static_assert(SITES <= 32, "one producer lane per site");
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
    unsigned char *stage_base = smem_raw;
    uint64_t *full_bar = reinterpret_cast<uint64_t *>(smem_raw + (size_t)C::STAGES * C::STAGE_BYTES);
    uint64_t *empty_bar = full_bar + C::STAGES;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int st = 0; st < C::STAGES; ++st) {
            mbar_init(&full_bar[st], 1);
            mbar_init(&empty_bar[st], C::NWARP);
        }
        mbar_fence_init();
    }
    __syncthreads();

    const int64_t ngroups = (V + C::SITES - 1) / C::SITES;
    constexpr int NN = C::NB * C::NB;        // elements per stencil matrix
    constexpr int NS = C::NB * C::S;         // elements per site of a vector block

    if (warp == C::NWARP) {
        // ===================== producer warp: lane l streams site l of the group =====================
        if (lane < C::SITES) {
            const uint64_t pol_a = l2_policy_evict_first();
            const uint64_t pol_x = l2_policy_evict_last();
            uint32_t it = 0;
            for (int64_t g = blockIdx.x; g < ngroups; g += gridDim.x) {
                int64_t x = g * C::SITES + lane;
                if (x >= V) x = V - 1;                       // tail group: duplicate the last site (its Y store is skipped)
                const int32_t *nrow = nbr + x * kNPoint;
                const Z *arow = At + x * (int64_t)kNPoint * NN;
                int32_t ynext = nrow[stencil_point_in_order(0)];
                for (int q = 0; q < kNPoint; ++q) {
                    const int p = stencil_point_in_order(q);
                    const int64_t y = ynext;
                    if (q + 1 < kNPoint) ynext = nrow[stencil_point_in_order(q + 1)];
#pragma unroll
                    for (int h = 0; h < C::KSPLIT; ++h, ++it) {
                        const uint32_t st = it % C::STAGES, round = it / C::STAGES;
                        mbar_wait(&empty_bar[st], (round & 1) ^ 1);
                        if (lane == 0) mbar_arrive_expect_tx(&full_bar[st], C::STAGE_BYTES);
                        __syncwarp(C::SITES >= 32 ? 0xffffffffu : ((1u << (C::SITES & 31)) - 1u));
                        unsigned char *sb = stage_base + (size_t)st * C::STAGE_BYTES;
                        Z *sA = reinterpret_cast<Z *>(sb) + lane * C::A_ELEMS;
                        Z *sX = reinterpret_cast<Z *>(sb + C::SITES * C::A_BYTES) + lane * C::X_ELEMS;
                        bulk_g2s(sA, arow + (int64_t)p * NN + h * C::A_ELEMS, C::A_BYTES, &full_bar[st], pol_a);
                        bulk_g2s(sX, X + y * (int64_t)NS + h * C::X_ELEMS, C::X_BYTES, &full_bar[st], pol_x);
                    }
                }
            }
        }
    } else {
        // ===================== consumer warps: register-tiled complex MAC =====================
        const int site_l = warp / C::CB, cb = warp % C::CB;
        const int gr = lane / C::GC, gc = lane % C::GC;
        const int row0 = gr * C::VA;                       // first row of this thread within a vector group
        const int col0 = cb * C::CT + gc * C::VX;
        uint32_t it = 0;
        for (int64_t g = blockIdx.x; g < ngroups; g += gridDim.x) {
            Z acc[C::TM][C::TN];
#pragma unroll
            for (int a = 0; a < C::TM; ++a)
#pragma unroll
                for (int b = 0; b < C::TN; ++b) { acc[a][b].re = 0; acc[a][b].im = 0; }

            for (int ph = 0; ph < kNPoint * C::KSPLIT; ++ph, ++it) {
                const uint32_t st = it % C::STAGES, round = it / C::STAGES;
                mbar_wait(&full_bar[st], round & 1);
                const unsigned char *sb = stage_base + (size_t)st * C::STAGE_BYTES;
                const Z *sA = reinterpret_cast<const Z *>(sb) + site_l * C::A_ELEMS + row0;
                const Z *sX = reinterpret_cast<const Z *>(sb + C::SITES * C::A_BYTES) + site_l * C::X_ELEMS + col0;
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
                if (lane == 0) mbar_arrive(&empty_bar[st]);
            }

            const int64_t x = g * C::SITES + site_l;
            if (x < V) {
                Z *yout = Y + x * (int64_t)NS;
#pragma unroll
                for (int i = 0; i < C::TM; ++i) {
                    const int row = simt_row<C>(gr, i);
#pragma unroll
                    for (int j = 0; j < C::TN; ++j) {
                        const int col = cb * C::CT + simt_col<C>(gc, j);
                        yout[row * C::S + col] = acc[i][j];
                    }
                }
            }
        }
    }
}

template <class C>
int launch_stencil_simt(const void *At, const int32_t *nbr, const void *X, void *Y, int64_t V, int num_sms, cudaStream_t stream)
{
    using Z = cplx<typename C::real>;
    auto kern = stencil_simt_kernel<C>;
    static bool attr_set = false;
    if (!attr_set) {
        CMRHS_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM_BYTES));
        attr_set = true;
    }
    const int64_t ngroups = (V + C::SITES - 1) / C::SITES;
    const int grid = (int)(ngroups < num_sms ? ngroups : num_sms);
    kern<<<grid, C::THREADS, C::SMEM_BYTES, stream>>>(static_cast<const Z *>(At), nbr, static_cast<const Z *>(X),
                                                       static_cast<Z *>(Y), V);
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}

}  // namespace cmrhs

// FP64 tensor-core (DMMA, mma.sync.m8n8k4.f64) variant of the tiled stencil-GEMM kernel for complex128.
//   Y(x) = sum_{p=0}^{80} A^p(x) . X(x + delta_p)                       (Eq. 19)
//
// tcgen05 has no FP64 kind; the FP64 tensor path of sm_100a is the warp-level mma.sync (SASS: DMMA), whose measured peak
// (33.0 TFLOP/s, profiles/peaks_r2.json) equals the DFMA pipe's (33.9).  What it buys is OPERAND TRAFFIC: the SIMT kernel
// loads TM + TN complex operands from shared memory per TM x TN complex multiply-adds (LSU 64 % busy at configs[1]), a DMMA
// takes an 8 x 4 and a 4 x 8 fragment (one double per lane each) for 256 multiply-adds: ~5x fewer shared-memory bytes per flop.
//
// Data movement is the SIMT kernel's (stencil_simt.cuh): every warp owns whole sites and runs its own ring of bulk copies
// (KCH contraction indices of one k-major stencil tile + the matching rows of the neighbour's X tile per stage).
// Arithmetic: X(y) as the real K x 2S matrix it is in memory; per 8-row tile of A and 8 real columns of X
//   P0 += Re A . X_re   Q0 += Im A . X_re   P1 += Re A . X_im   Q1 += Im A . X_im      (4 DMMAs per k = 4 slab)
//   Y_re = P0 - Q1,  Y_im = P1 + Q0   once per site.
// Fragments: lane l holds A[row l/4][k l%4] -- Re and Im arrive together in ONE 16-byte load -- and X[k l%4][column l/4]: the 8
// "columns" of a tile are the EVEN (re) resp. ODD (im) real columns of 8 consecutive right-hand sides, so one 16-byte load of
// (re, im) feeds both the X_re and the X_im tile.  Known cost (ncu, configs[1]: LSU wavefronts 72 % busy): the 8 lanes the LSU
// serves together hold 2 rows x 4 k, and the k rows of the bulk-copied tile are 384 / 512 bytes apart -- a 4-way bank conflict.
// Padding the rows (one bulk copy per k row) removes it but costs more than it saves (48 copies of 128-416 bytes per stage:
// configs[1] 0.61 -> 0.90 ms), so the tile keeps its one-copy layout.
//
// BALANCED mode (template flag BAL; chosen by the launcher for small lattices).  With whole sites per warp the kernel's time is
// quantised: configs[1] has 4096 sites for 148 x 8 = 1184 warps, 3.46 on average but 4 for the slowest -- measured: V = 4096 and
// V = 4736 (exactly 4 each) both take 0.614 ms (5.0 against 5.8 TB/s).  In balanced mode every warp takes one contiguous range of
// the V x 81 (site, stencil point) sequence, cut at equal counts wherever that falls; a site that two warps share is added into a
// zeroed Y with atomicAdd (double) by both -- two terms onto zero: the sum does not depend on their order, so the result stays
// bit-reproducible.  The launcher takes this mode only when every warp gets at least 81 points (no site is shared by three).
// configs[1]: 0.614 -> 0.538 ms (5.73 TB/s, 0.85 of the HBM roof).
#pragma once

#include "stencil_simt.cuh"

namespace cmrhs {

template <int NB_, int S_, int KSPLIT_, int STAGES_, int WARPS_>
struct DmmaConfig {
    static constexpr int NB = NB_, S = S_, KSPLIT = KSPLIT_, STAGES = STAGES_, WARPS = WARPS_;
    static constexpr int THREADS = WARPS * 32;
    static constexpr int KCH = NB / KSPLIT;
    static constexpr int CPS = kNPoint * KSPLIT;
    static constexpr int MT = NB / 8, NT = S / 8;          // 8-row tiles of A, groups of 8 right-hand sides
    static constexpr uint32_t A_BYTES = KCH * NB * 16, X_BYTES = KCH * S * 16, STAGE_BYTES = A_BYTES + X_BYTES;
    static constexpr int A_ELEMS = KCH * NB, X_ELEMS = KCH * S;
    static constexpr size_t SMEM_BYTES = (size_t)WARPS * STAGES * STAGE_BYTES + (size_t)WARPS * STAGES * sizeof(uint64_t) + 16;
    static_assert(NB % 8 == 0 && S % 8 == 0 && NB % KSPLIT == 0 && KCH % 4 == 0, "DMMA tiling: NB, S multiples of 8, KCH of 4");
    static_assert(SMEM_BYTES <= 227 * 1024, "shared memory ring does not fit");
};

__device__ __forceinline__ void dmma_m8n8k4(double (&c)[2], double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};" : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

template <class C, bool BAL>
__global__ void __launch_bounds__(C::THREADS, 1)
stencil_dmma_kernel(const cplx<double> *__restrict__ At, const int32_t *__restrict__ nbr, const cplx<double> *__restrict__ X,
                    cplx<double> *__restrict__ Y, int64_t V)
{
    using Z = cplx<double>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned char *ring = smem_raw + (size_t)warp * C::STAGES * C::STAGE_BYTES;
    uint64_t *full_bar = reinterpret_cast<uint64_t *>(smem_raw + (size_t)C::WARPS * C::STAGES * C::STAGE_BYTES) + warp * C::STAGES;
    constexpr int NN = C::NB * C::NB, NS = C::NB * C::S;
    constexpr unsigned FULL = 0xffffffffu;

    // whole sites, interleaved over the warps (site = first + j stride) -- or, balanced, the points [pt_begin, pt_end) of the sequence
    // g = site * 81 + q (q = position in the site's accumulation order)
    const int64_t stride = BAL ? 1 : (int64_t)gridDim.x * C::WARPS;
    const int64_t nwarps = (int64_t)gridDim.x * C::WARPS, wid = (int64_t)blockIdx.x * C::WARPS + warp;
    const int64_t pt_begin = BAL ? V * kNPoint * wid / nwarps : 0, pt_end = BAL ? V * kNPoint * (wid + 1) / nwarps : 0;
    const int64_t first = BAL ? pt_begin / kNPoint : wid;
    if (BAL ? pt_begin >= pt_end : first >= V) return;
    const int64_t nsites = BAL ? 0 : (V - first + stride - 1) / stride;
    const int64_t nchunks = BAL ? (pt_end - pt_begin) * C::KSPLIT : nsites * C::CPS;
    const int w0 = BAL ? (int)(pt_begin - first * kNPoint) * C::KSPLIT : 0;        // chunk of the first site this warp starts at
    if (lane == 0) {
        for (int st = 0; st < C::STAGES; ++st) mbar_init(&full_bar[st], 1);
        mbar_fence_init();
    }
    __syncwarp();
    uint64_t pol_a = 0, pol_x = 0;
    if (lane == 0) { pol_a = l2_policy_evict_first(); pol_x = l2_policy_evict_last(); }

    // ---- issue side (as stencil_simt.cuh) ----
    int64_t ix = first;
    int iw = w0;
    int32_t n0, n1, n2;
    auto load_nbr_row = [&](int64_t x) {
        const int32_t *row = nbr + x * kNPoint;
        n0 = row[lane];
        n1 = row[lane + 32];
        n2 = (lane + 64 < kNPoint) ? row[lane + 64] : 0;
    };
    load_nbr_row(ix);
    auto issue = [&](int st) {
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
    int64_t issued = 0;
    for (; issued < C::STAGES && issued < nchunks; ++issued) issue((int)issued);

    // ---- compute side: DMMA ----
    const int fr = lane >> 2, fk = lane & 3;           // fragment row / column index (0..7), k index (0..3)
    double p0[C::MT][C::NT][2], q0[C::MT][C::NT][2], p1[C::MT][C::NT][2], q1[C::MT][C::NT][2];
#pragma unroll
    for (int m = 0; m < C::MT; ++m)
#pragma unroll
        for (int n = 0; n < C::NT; ++n)
#pragma unroll
            for (int e = 0; e < 2; ++e) { p0[m][n][e] = 0.0; q0[m][n][e] = 0.0; p1[m][n][e] = 0.0; q1[m][n][e] = 0.0; }

    int64_t cx = first;
    int cw = w0, st = 0;
    bool whole = w0 == 0;                     // (balanced) this warp accumulates every point of site cx
    uint32_t parity = 0;
    for (int64_t c = 0; c < nchunks; ++c) {
        mbar_wait(&full_bar[st], parity);
        const unsigned char *sb = ring + (size_t)st * C::STAGE_BYTES;
        const Z *sA = reinterpret_cast<const Z *>(sb);                    // [k][NB]
        const Z *sX = reinterpret_cast<const Z *>(sb + C::A_BYTES);       // [k][S]
#pragma unroll
        for (int k4 = 0; k4 < C::KCH; k4 += 4) {
            double2 a[C::MT], x[C::NT];
#pragma unroll
            for (int m = 0; m < C::MT; ++m) a[m] = *reinterpret_cast<const double2 *>(sA + (k4 + fk) * C::NB + 8 * m + fr);
#pragma unroll
            for (int n = 0; n < C::NT; ++n) x[n] = *reinterpret_cast<const double2 *>(sX + (k4 + fk) * C::S + 8 * n + fr);
#pragma unroll
            for (int m = 0; m < C::MT; ++m)
#pragma unroll
                for (int n = 0; n < C::NT; ++n) {
                    dmma_m8n8k4(p0[m][n], a[m].x, x[n].x);
                    dmma_m8n8k4(q0[m][n], a[m].y, x[n].x);
                    dmma_m8n8k4(p1[m][n], a[m].x, x[n].y);
                    dmma_m8n8k4(q1[m][n], a[m].y, x[n].y);
                }
        }
        __syncwarp();
        if (issued < nchunks) { issue(st); ++issued; }
        if (++st == C::STAGES) { st = 0; parity ^= 1u; }

        if (++cw == C::CPS || (BAL && c + 1 == nchunks)) {       // site (or this warp's part of it) finished: C fragment of lane l = rows 8 m + l/4, right-hand sides 8 n + 2 (l%4), + 1
            Z *yout = Y + cx * (int64_t)NS;
            const bool shared_site = BAL && !(whole && cw == C::CPS);      // another warp holds the rest of this site: both add into the zeroed Y
#pragma unroll
            for (int m = 0; m < C::MT; ++m)
#pragma unroll
                for (int n = 0; n < C::NT; ++n) {
                    double4 o;
                    o.x = p0[m][n][0] - q1[m][n][0]; o.y = p1[m][n][0] + q0[m][n][0];
                    o.z = p0[m][n][1] - q1[m][n][1]; o.w = p1[m][n][1] + q0[m][n][1];
                    double2 *dst = reinterpret_cast<double2 *>(yout + (8 * m + fr) * C::S + 8 * n + 2 * fk);
                    if (shared_site) {
                        double *d = reinterpret_cast<double *>(dst);
                        atomicAdd(d, o.x); atomicAdd(d + 1, o.y); atomicAdd(d + 2, o.z); atomicAdd(d + 3, o.w);
                    } else {
                        dst[0] = make_double2(o.x, o.y);
                        dst[1] = make_double2(o.z, o.w);
                    }
#pragma unroll
                    for (int e = 0; e < 2; ++e) { p0[m][n][e] = 0.0; q0[m][n][e] = 0.0; p1[m][n][e] = 0.0; q1[m][n][e] = 0.0; }
                }
            cw = 0;
            cx += stride;
            whole = true;
        }
    }
}

template <class C>
int launch_stencil_dmma_as(const void *At, const int32_t *nbr, const void *X, void *Y, int64_t V, int num_sms, cudaStream_t stream)
{
    using Z = cplx<double>;
    const int64_t nctas = (V + C::WARPS - 1) / C::WARPS;
    const int grid = (int)(nctas < num_sms ? nctas : num_sms);
    // balanced mode: between 1 and 16 sites per warp, where the whole-site partition loses up to a site's time per warp
    const int64_t nwarps = (int64_t)grid * C::WARPS;
    if (V >= nwarps && V < 16 * nwarps && V % nwarps != 0) {
        auto kern = stencil_dmma_kernel<C, true>;
        CMRHS_SMEM_ATTR(kern, C::SMEM_BYTES);
        CMRHS_CUDA(cudaMemsetAsync(Y, 0, (size_t)V * C::NB * C::S * sizeof(Z), stream));
        kern<<<grid, C::THREADS, C::SMEM_BYTES, stream>>>(static_cast<const Z *>(At), nbr, static_cast<const Z *>(X), static_cast<Z *>(Y), V);
    } else {
        auto kern = stencil_dmma_kernel<C, false>;
        CMRHS_SMEM_ATTR(kern, C::SMEM_BYTES);
        kern<<<grid, C::THREADS, C::SMEM_BYTES, stream>>>(static_cast<const Z *>(At), nbr, static_cast<const Z *>(X), static_cast<Z *>(Y), V);
    }
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}

// small lattices: CTAs of 2 or 4 warps when every site still gets its own warp in one round (stencil_simt.cuh: launch_stencil_simt)
template <class C>
int launch_stencil_dmma(const void *At, const int32_t *nbr, const void *X, void *Y, int64_t V, int num_sms, cudaStream_t stream)
{
    using C4 = DmmaConfig<C::NB, C::S, C::KSPLIT, C::STAGES, 4>;
    using C2 = DmmaConfig<C::NB, C::S, C::KSPLIT, C::STAGES, 2>;
    if (C::WARPS > 2 && (V + 1) / 2 <= num_sms) return launch_stencil_dmma_as<C2>(At, nbr, X, Y, V, num_sms, stream);
    if (C::WARPS > 4 && (V + 3) / 4 <= num_sms) return launch_stencil_dmma_as<C4>(At, nbr, X, Y, V, num_sms, stream);
    return launch_stencil_dmma_as<C>(At, nbr, X, Y, V, num_sms, stream);
}

}  // namespace cmrhs

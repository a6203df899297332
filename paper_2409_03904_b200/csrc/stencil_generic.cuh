// Generic stencil-GEMM kernel: any 1 <= nbasis <= 64, 1 <= nrhs <= 64, both dtypes.
//   Y(x) = sum_{p=0}^{80} A^p(x) . X(x + delta_p)                       (Eq. 19)
// One CTA per site (grid-stride); per stencil point the A tile (k-major internal layout) and the
// neighbour's X tile are staged in shared memory with coalesced loads and every thread accumulates
// its outputs (i, r) in registers; Y is written once.  This is the correctness fallback for shapes
// the tiled kernels (stencil_simt.cuh) do not cover, and the reference the tiled kernels are tested against.
#pragma once

#include "common.cuh"

namespace cmrhs {

constexpr int kGenericThreads = 256;
constexpr int kGenericMaxOut = (COARSE_MAX_NBASIS * COARSE_MAX_NRHS + kGenericThreads - 1) / kGenericThreads;

template <typename T, int MAXOUT>
__global__ void __launch_bounds__(kGenericThreads)
stencil_generic_kernel(const cplx<T> *__restrict__ At, const int32_t *__restrict__ nbr, const cplx<T> *__restrict__ X,
                       cplx<T> *__restrict__ Y, int64_t V, int nb, int s)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx<T> *sA = reinterpret_cast<cplx<T> *>(smem_raw);
    cplx<T> *sX = sA + nb * nb;
    const int nn = nb * nb, ns = nb * s;

    int oi[MAXOUT], orr[MAXOUT];
#pragma unroll
    for (int o = 0; o < MAXOUT; ++o) {
        const int e = threadIdx.x + o * kGenericThreads;
        oi[o] = (e < ns) ? e / s : -1;
        orr[o] = (e < ns) ? e % s : 0;
    }

    for (int64_t x = blockIdx.x; x < V; x += gridDim.x) {
        cplx<T> acc[MAXOUT];
#pragma unroll
        for (int o = 0; o < MAXOUT; ++o) { acc[o].re = 0; acc[o].im = 0; }
        for (int q = 0; q < kNPoint; ++q) {
            const int p = stencil_point_in_order(q);
            const int64_t y = nbr[x * kNPoint + p];
            const cplx<T> *a = At + (x * kNPoint + p) * (int64_t)nn;
            const cplx<T> *xin = X + y * (int64_t)ns;
            for (int e = threadIdx.x; e < nn; e += kGenericThreads) sA[e] = a[e];
            for (int e = threadIdx.x; e < ns; e += kGenericThreads) sX[e] = xin[e];
            __syncthreads();
#pragma unroll
            for (int o = 0; o < MAXOUT; ++o) {
                if (oi[o] >= 0) {
                    const int i = oi[o], r = orr[o];
                    for (int k = 0; k < nb; ++k) cmac(acc[o], sA[k * nb + i], sX[k * s + r]);
                }
            }
            __syncthreads();
        }
        cplx<T> *yout = Y + x * (int64_t)ns;
#pragma unroll
        for (int o = 0; o < MAXOUT; ++o)
            if (oi[o] >= 0) yout[threadIdx.x + o * kGenericThreads] = acc[o];
    }
}

template <typename T>
int launch_stencil_generic(const cplx<T> *At, const int32_t *nbr, const cplx<T> *X, cplx<T> *Y, int64_t V, int nb, int s,
                           int num_sms, cudaStream_t stream)
{
    const size_t smem = (size_t)(nb * nb + nb * s) * sizeof(cplx<T>);
    const int nout = (nb * s + kGenericThreads - 1) / kGenericThreads;
    const int grid = (int)(V < (int64_t)num_sms * 8 ? V : (int64_t)num_sms * 8);
#define CMRHS_GENERIC_CASE(MO)                                                                                       \
    {                                                                                                                \
        auto kern = stencil_generic_kernel<T, MO>;                                                                   \
        CMRHS_SMEM_ATTR(kern, smem);                                                                                 \
        kern<<<grid, kGenericThreads, smem, stream>>>(At, nbr, X, Y, V, nb, s);                                      \
    }
    if (nout <= 1) CMRHS_GENERIC_CASE(1)
    else if (nout <= 2) CMRHS_GENERIC_CASE(2)
    else if (nout <= 4) CMRHS_GENERIC_CASE(4)
    else if (nout <= 8) CMRHS_GENERIC_CASE(8)
    else CMRHS_GENERIC_CASE(kGenericMaxOut)
#undef CMRHS_GENERIC_CASE
    CMRHS_LAUNCH_CHECK();
    return COARSE_OK;
}

}  // namespace cmrhs

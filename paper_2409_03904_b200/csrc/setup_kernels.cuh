// Setup-time kernels: periodic neighbour table, re-layout of the
// stencil matrices into the kernels' internal tile layout, and the device-side synthetic input
// generator (input generation only; same counter-based hash as inputs/synth.py, written independently).
#pragma once

#include "common.cuh"

namespace cmrhs {

struct LatticeDims {
    int32_t L[4];
    int64_t V;
};

__host__ __device__ __forceinline__ int64_t neighbour_site(const LatticeDims &d, int64_t x, int p)
{   // x + delta_p with periodic wrap; p = sum (d_k + 1) 3^k
    int64_t y = 0, stride = 1;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int L = d.L[k];
        int c = (int)(x % L);
        x /= L;
        c += (p % 3) - 1;
        p /= 3;
        c = (c < 0) ? c + L : (c >= L ? c - L : c);
        y += (int64_t)c * stride;
        stride *= L;
    }
    return y;
}

// nbr[x][p] = site index of x + delta_p
__global__ void neighbour_table_kernel(LatticeDims d, int32_t *__restrict__ nbr)
{
    const int64_t total = d.V * kNPoint;
    for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        const int64_t x = e / kNPoint;
        const int p = (int)(e % kNPoint);
        nbr[e] = (int32_t)neighbour_site(d, x, p);
    }
}

// Internal tile layout: At[x][p][k][i] = A[x][p][i][k]  (k-major: for a fixed contraction index k the nb
// row entries are contiguous, so a thread's register tile of rows is one vector load from shared memory).
template <typename T>
__global__ void relayout_transpose_kernel(const cplx<T> *__restrict__ A, cplx<T> *__restrict__ At, int64_t ntiles, int nb)
{
    const int nn = nb * nb;
    for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const cplx<T> *src = A + t * nn;
        cplx<T> *dst = At + t * nn;
        for (int e = threadIdx.x; e < nn; e += blockDim.x) {
            const int k = e / nb, i = e % nb;
            dst[e] = src[i * nb + k];
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// Synthetic inputs on the device.  Element idx of stream (seed, tag):
//   h = mix64(K + (idx+1)*GOLDEN), K = mix64(seed + tag*TAGMUL); u1,u2 from the two 32-bit halves;
//   z = sqrt(-ln u1) * (cos 2 pi u2 + i sin 2 pi u2)   (complex N(0,1), E|z|^2 = 1), float64 then rounded to float32.
// ---------------------------------------------------------------------------------------------------
__host__ __device__ __forceinline__ uint64_t synth_mix64(uint64_t z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

__host__ __device__ __forceinline__ uint64_t synth_key(uint64_t seed, uint64_t tag)
{
    return synth_mix64(seed + tag * 0xD1B54A32D192ED03ull);
}

__device__ __forceinline__ void synth_normal(uint64_t key, uint64_t idx, double &re, double &im)
{
    const uint64_t h = synth_mix64(key + (idx + 1) * 0x9E3779B97F4A7C15ull);
    const double u1 = __dmul_rn((double)(uint32_t)(h >> 32) + 0.5, 1.0 / 4294967296.0);
    const double u2 = __dmul_rn((double)(uint32_t)(h & 0xFFFFFFFFull) + 0.5, 1.0 / 4294967296.0);
    const double r = sqrt(-log(u1));
    const double ang = __dmul_rn(6.283185307179586476925286766559, u2);
    re = __dmul_rn(r, cos(ang));
    im = __dmul_rn(r, sin(ang));
}

enum { SYNTH_TAG_A = 1, SYNTH_TAG_G = 2 };

// raw off-diagonal entry of the independent half (p < 40): float32( z / nb )
__device__ __forceinline__ void synth_offdiag(uint64_t keyA, int64_t x, int p, int i, int j, int nb, float &re, float &im)
{
    double dr, di;
    synth_normal(keyA, (uint64_t)(((x * kNPoint + p) * nb + i) * (int64_t)nb + j), dr, di);
    re = (float)(dr / nb);
    im = (float)(di / nb);
}

template <typename T>
__global__ void synth_fill_kernel(cplx<T> *__restrict__ A, LatticeDims d, int nb, uint64_t keyA, uint64_t keyG)
{
    const int nn = nb * nb;
    const int64_t total = d.V * kNPoint * nn;
    for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        const int j = (int)(e % nb);
        const int i = (int)((e / nb) % nb);
        const int p = (int)((e / nn) % kNPoint);
        const int64_t x = e / ((int64_t)nn * kNPoint);
        float re, im;
        if (p < kCentre) {
            synth_offdiag(keyA, x, p, i, j, nb, re, im);
        } else if (p > kCentre) {   // A_p(x) = A_{80-p}(x + delta_p)^H
            const int64_t y = neighbour_site(d, x, p);
            synth_offdiag(keyA, y, kNPoint - 1 - p, j, i, nb, re, im);
            im = -im;
        } else {                    // Hrand = (G + G^H)/2 from float32-rounded G
            double ar, ai, br, bi;
            synth_normal(keyG, (uint64_t)((x * nb + i) * (int64_t)nb + j), ar, ai);
            synth_normal(keyG, (uint64_t)((x * nb + j) * (int64_t)nb + i), br, bi);
            const float gr1 = (float)(ar / nb), gi1 = (float)(ai / nb), gr2 = (float)(br / nb), gi2 = (float)(bi / nb);
            re = (float)(0.5 * ((double)gr1 + (double)gr2));
            im = (float)(0.5 * ((double)gi1 - (double)gi2));
        }
        A[e].re = (T)re;
        A[e].im = (T)im;
    }
}

// bound[x] = sum_p ||A_p(x)||_F  (one warp per site, fixed reduction order)
template <typename T>
__global__ void synth_bound_kernel(const cplx<T> *__restrict__ A, int64_t V, int nb, double *__restrict__ bound)
{
    const int nn = nb * nb;
    const int lane = threadIdx.x & 31;
    const int64_t warp = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    const int64_t nwarp = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t x = warp; x < V; x += nwarp) {
        double tot = 0.0;
        for (int p = 0; p < kNPoint; ++p) {
            const cplx<T> *a = A + (x * kNPoint + p) * nn;
            double acc = 0.0;
            for (int e = lane; e < nn; e += 32) acc += (double)a[e].re * (double)a[e].re + (double)a[e].im * (double)a[e].im;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
            tot += sqrt(acc);
        }
        if (lane == 0) bound[x] = tot;
    }
}

__global__ void max_reduce_kernel(const double *__restrict__ v, int64_t n, double *__restrict__ out)
{   // single block, deterministic
    __shared__ double sm[256];
    double m = 0.0;
    for (int64_t e = threadIdx.x; e < n; e += blockDim.x) m = fmax(m, v[e]);
    sm[threadIdx.x] = m;
    __syncthreads();
    for (int o = blockDim.x / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sm[threadIdx.x] = fmax(sm[threadIdx.x], sm[threadIdx.x + o]);
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = sm[0];
}

template <typename T>
__global__ void synth_shift_kernel(cplx<T> *__restrict__ A, int64_t V, int nb, float c)
{
    const int64_t total = V * nb;
    for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        const int64_t x = e / nb;
        const int i = (int)(e % nb);
        cplx<T> &a = A[((x * kNPoint + kCentre) * nb + i) * (int64_t)nb + i];
        a.re = (T)(float)((double)a.re + (double)c);
    }
}

template <typename T>
__global__ void synth_block_kernel(cplx<T> *__restrict__ X, int64_t total, uint64_t key)
{
    for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        double re, im;
        synth_normal(key, (uint64_t)e, re, im);
        X[e].re = (T)(float)re;
        X[e].im = (T)(float)im;
    }
}

}  // namespace cmrhs

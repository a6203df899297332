// Roofline denominators measured on the device the library runs on ("measure ... and store them
// beside MEASURED_PEAKS.json's values"): a read-only HBM stream (the access pattern of the stencil operator: it is read
// once and never written, so a copy's bandwidth is the wrong roof -- ADVICE round 1), and register-resident FFMA /
// packed FFMA2 / DFMA / DMMA (mma.sync.m8n8k4.f64) loops.  Bench helpers only: nothing on the product path calls them.
#pragma once

#include "common.cuh"

namespace cmrhs {

// every thread streams 16-byte vectors with a grid stride; the sum keeps the loads alive
__global__ void __launch_bounds__(256) peak_read_kernel(const uint4 *__restrict__ p, int64_t n16, uint32_t *__restrict__ sink)
{
    uint32_t acc = 0u;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    for (; e + 3 * stride < n16; e += 4 * stride) {
        const uint4 a = __ldcs(p + e), b = __ldcs(p + e + stride), c = __ldcs(p + e + 2 * stride), d = __ldcs(p + e + 3 * stride);
        acc ^= a.x ^ a.y ^ a.z ^ a.w ^ b.x ^ b.y ^ b.z ^ b.w ^ c.x ^ c.y ^ c.z ^ c.w ^ d.x ^ d.y ^ d.z ^ d.w;
    }
    for (; e < n16; e += stride) { const uint4 a = __ldcs(p + e); acc ^= a.x ^ a.y ^ a.z ^ a.w; }
    if (acc == 0x12345678u) atomicAdd(sink, 1u);
}

// kind 0: FFMA, 1: FFMA2 (packed fma.rn.f32x2), 2: DFMA, 3: DMMA m8n8k4.  16 independent accumulator chains per thread.
template <int KIND>
__global__ void __launch_bounds__(256) peak_alu_kernel(int iters, float seed, double *__restrict__ sink)
{
    if constexpr (KIND == 0) {
        float a[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) a[i] = seed + (float)(threadIdx.x + i);
        const float m = 1.0f + seed * 1e-9f, c = seed * 1e-7f;
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int i = 0; i < 16; ++i) a[i] = fmaf(a[i], m, c);
        }
        float s = 0.f;
#pragma unroll
        for (int i = 0; i < 16; ++i) s += a[i];
        if (s == 12345.678f) sink[0] = s;
    } else if constexpr (KIND == 1) {
        unsigned long long a[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const float2 v = make_float2(seed + (float)(threadIdx.x + i), seed + (float)i);
            a[i] = *reinterpret_cast<const unsigned long long *>(&v);
        }
        const float2 mv = make_float2(1.0f + seed * 1e-9f, 1.0f - seed * 1e-9f), cv = make_float2(seed * 1e-7f, seed * 2e-7f);
        const unsigned long long m = *reinterpret_cast<const unsigned long long *>(&mv), c = *reinterpret_cast<const unsigned long long *>(&cv);
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int i = 0; i < 16; ++i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(a[i]) : "l"(m), "l"(c));
        }
        unsigned long long s = 0;
#pragma unroll
        for (int i = 0; i < 16; ++i) s ^= a[i];
        if (s == 0x123456789abcdefull) sink[0] = 1.0;
    } else if constexpr (KIND == 2) {
        double a[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) a[i] = (double)seed + (double)(threadIdx.x + i);
        const double m = 1.0 + (double)seed * 1e-12, c = (double)seed * 1e-9;
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int i = 0; i < 16; ++i) a[i] = fma(a[i], m, c);
        }
        double s = 0.;
#pragma unroll
        for (int i = 0; i < 16; ++i) s += a[i];
        if (s == 12345.678) sink[0] = s;
    } else {
        double d[16][2];
#pragma unroll
        for (int i = 0; i < 16; ++i) { d[i][0] = (double)seed + i; d[i][1] = (double)seed - i; }
        const double a = 1.0 + (double)seed * 1e-12, b = 1.0 - (double)seed * 1e-12;
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int i = 0; i < 16; ++i)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};" : "+d"(d[i][0]), "+d"(d[i][1]) : "d"(a), "d"(b));
        }
        double s = 0.;
#pragma unroll
        for (int i = 0; i < 16; ++i) s += d[i][0] + d[i][1];
        if (s == 12345.678) sink[0] = s;
    }
}

}  // namespace cmrhs

// kern_peak.cuh -- FP32-FMA throughput microbenchmark: the denominator of "% of FP32 FMA peak".
// Independent register-resident FMA chains on every SM; no memory traffic inside the loop.
#pragma once
#include "pdm_common.cuh"

#define PDM_PEAK_CHAINS 16

template <int PACKED>
__global__ void __launch_bounds__(256) pdm_peak_kernel(float *out, int iters, float seed)
{
    float2 acc[PDM_PEAK_CHAINS];
#pragma unroll
    for (int c = 0; c < PDM_PEAK_CHAINS; ++c)
        acc[c] = make_float2(seed + c, seed - c + threadIdx.x * 1e-3f);
    const float2 a = make_float2(0.999f, 1.001f), b = make_float2(1e-3f, -1e-3f);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int c = 0; c < PDM_PEAK_CHAINS; ++c) {
            if (PACKED) {
                acc[c] = pk_fma(acc[c], a, b);
            } else {
                acc[c].x = fmaf(acc[c].x, a.x, b.x);
                acc[c].y = fmaf(acc[c].y, a.y, b.y);
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < PDM_PEAK_CHAINS; ++c) s += acc[c].x + acc[c].y;
    if (s == 123.456f) out[0] = s;     // never true: keeps the chains alive
}

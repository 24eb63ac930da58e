// kern_reduce.cuh -- A5, second half: the deterministic reduction of the per-CTA partial images.
#pragma once
#include "pdm_common.cuh"

// A5, second half: image[z][x] = sum over CTAs (fixed order) of their partial images.
static __global__ void pdm_reduce_partials(const float *__restrict__ partial, float *__restrict__ image,
                                    int nparts, int nz, int nx, int pstride)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int z = blockIdx.y;
    if (x >= nx) return;
    const size_t plane = (size_t)nz * pstride;
    const float *src = partial + (size_t)z * pstride + x;
    float s = 0.f;
    for (int c = 0; c < nparts; ++c) s += __ldcs(src + (size_t)c * plane);
    image[(size_t)z * nx + x] = s;
}

// kern_naive.cuh -- PDM_PATH_NAIVE: the paper's own mapping, kept as a cross-check scaffold.
//   K1 "next plan": one thread per pixel (w,x) of the next depth plane, Eq. (1)
//       with the looked-up filter, planes in global memory, one launch per depth level.
//   K2 "depth row": one thread per x sums the new plane over w.
// Differences from the paper: threadIdx runs along x (coalesced), not along w; the full
// 2L+1 row is applied (no folding) so this path is an independent check of the folded kernels.
#pragma once
#include "pdm_common.cuh"

__global__ void pdm_naive_step(const float2 *__restrict__ Pin, float2 *__restrict__ Pout,
                               const float *__restrict__ omega, const float *__restrict__ qrow,
                               const float2 *__restrict__ table, int nx, int nw, int ntab, int L)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int iw = blockIdx.y;
    if (x >= nx) return;
    const int j = pdm_index(omega[iw], qrow[x], ntab - 1);
    const float2 *row = table + (size_t)j * (2 * L + 1) + L;
    const float2 *p = Pin + (size_t)iw * nx;
    float ar = 0.f, ai = 0.f;
    for (int k = -L; k <= L; ++k) {
        const int xs = x - k;
        if (xs < 0 || xs >= nx) continue;
        const float2 w = row[k], v = p[xs];
        ar = fmaf(w.x, v.x, ar); ar = fmaf(-w.y, v.y, ar);
        ai = fmaf(w.x, v.y, ai); ai = fmaf(w.y, v.x, ai);
    }
    Pout[(size_t)iw * nx + x] = make_float2(ar, ai);
}

__global__ void pdm_naive_image_row(const float2 *__restrict__ P, float *__restrict__ image_row,
                                    int nx, int nw)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= nx) return;
    float s = 0.f;
    for (int iw = 0; iw < nw; ++iw) s += P[(size_t)iw * nx + x].x;   // fixed w order
    image_row[x] = s;
}

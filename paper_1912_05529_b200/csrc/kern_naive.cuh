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

// The same step with the INTERPOLATED look-up (PDM_TABLE_INTERP, reading R3c): the operator
// is the linear blend of the two rows bracketing u32 = fl32(w*q) -- j0 = floor(u32), a = u32 - j0 (exact in
// float), W_k = W_k(j0) + a (W_k(j0+1) - W_k(j0)); at or beyond the last row that row alone.
__global__ void pdm_naive_step_interp(const float2 *__restrict__ Pin, float2 *__restrict__ Pout,
                                      const float *__restrict__ omega, const float *__restrict__ qrow,
                                      const float2 *__restrict__ table, int nx, int nw, int ntab, int L)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int iw = blockIdx.y;
    if (x >= nx) return;
    const float u = fmaxf(__fmul_rn(omega[iw], qrow[x]), 0.f);
    const float f = floorf(u);
    const bool last = f >= (float)(ntab - 1);
    const int j0 = last ? ntab - 1 : (int)f, j1 = last ? j0 : j0 + 1;
    const float a = last ? 0.f : u - f;
    const float2 *row0 = table + (size_t)j0 * (2 * L + 1) + L;
    const float2 *row1 = table + (size_t)j1 * (2 * L + 1) + L;
    const float2 *p = Pin + (size_t)iw * nx;
    float ar = 0.f, ai = 0.f;
    for (int k = -L; k <= L; ++k) {
        const int xs = x - k;
        if (xs < 0 || xs >= nx) continue;
        const float2 w0 = row0[k], w1 = row1[k], v = p[xs];
        const float wx = fmaf(a, w1.x - w0.x, w0.x), wy = fmaf(a, w1.y - w0.y, w0.y);
        ar = fmaf(wx, v.x, ar); ar = fmaf(-wy, v.y, ar);
        ai = fmaf(wx, v.y, ai); ai = fmaf(wy, v.x, ai);
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

// kern_tiled.cuh -- PDM_PATH_TILED: x-tiled per-depth-step kernel with
// +-L halos for lines too long for shared memory (BASELINE.json configs[4], nx = 32768).
// Closest to what the paper itself did (planes in global memory, one grid-wide
// synchronisation per depth level), but: the tile + halo is staged once in shared memory, the
// arithmetic is the same register-tiled folded FIR as the main path (pdm_fir_group), a CTA
// walks a GROUP of frequencies for its x-tile so the q tile is read once and Re P is summed
// over the group in registers in fixed order (the paper's K2 disappears), and planes ping-pong
// in HBM: 8 B read + 8 B written per sample (+ halo 2*HG*R/tile_x).
#pragma once
#include "pdm_common.cuh"
#include "kern_march.cuh"

#define PDM_TILED_THREADS 256

struct pdm_tiled_params {
    const float2 *Pin;       // [nw][nx] plane at depth z
    float2       *Pout;      // [nw][nx] plane at depth z+1
    float        *partial;   // [wgroups][nz][pstride]
    const float  *q;         // [nz][qstride]
    const float  *omega;
    const float4 *half;
    int nx, nz, nw, ntab;
    int qstride, pstride, half16;
    int z, w_per_group;
};

template <int L, int R>
__global__ void __launch_bounds__(PDM_TILED_THREADS, 2) pdm_tiled_step(const pdm_tiled_params p)
{
    constexpr int HG = pdm_halo_groups<L, R>();
    constexpr int GS = R + 2;
    extern __shared__ __align__(16) unsigned char pdm_smem[];
    float2 *line = reinterpret_cast<float2 *>(pdm_smem);

    const int tid = threadIdx.x, T = blockDim.x;
    const int tile_x0 = blockIdx.x * T * R;
    const int x0 = tile_x0 + tid * R;
    const int ntab_m1 = p.ntab - 1;
    const int w_begin = blockIdx.y * p.w_per_group;
    const int w_end = min(p.nw, w_begin + p.w_per_group);

    float qc[R];
    {
        const int xq = min(x0, p.qstride - R);
        const float4 *qp = reinterpret_cast<const float4 *>(p.q + (size_t)p.z * p.qstride + xq);
#pragma unroll
        for (int i = 0; i < R / 4; ++i) {
            const float4 v = __ldg(qp + i);
            qc[4 * i] = v.x; qc[4 * i + 1] = v.y; qc[4 * i + 2] = v.z; qc[4 * i + 3] = v.w;
        }
    }
    float img[R];
#pragma unroll
    for (int r = 0; r < R; ++r) img[r] = 0.f;

    const int nload = (T + 2 * HG) * R;                  // samples of tile + both halos
    for (int iw = w_begin; iw < w_end; ++iw) {
        const float w = p.omega[iw];
        const float2 *src = p.Pin + (size_t)iw * p.nx;
        __syncthreads();                                  // previous frequency finished reading
        for (int s = tid; s < nload; s += T) {
            const int x = tile_x0 - HG * R + s;
            const int g = s / R;
            float2 v = make_float2(0.f, 0.f);             // R5: zero outside [0,nx)
            if (x >= 0 && x < p.nx) v = src[x];
            line[g * GS + (s - g * R)] = v;
        }
        __syncthreads();

        int j[R], toff[R];
        bool uni = true;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            j[r] = pdm_index(w, qc[r], ntab_m1);
            uni = uni && (j[r] == j[0]);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) toff[r] = j[r] * p.half16;
        const float2 *base = line + (HG + tid) * GS;
        float2 out[R];
        if (__all_sync(0xffffffffu, uni)) pdm_fir_group<L, R, true>(base, p.half, toff, out);
        else                              pdm_fir_group<L, R, false>(base, p.half, toff, out);

        float2 *dst = p.Pout + (size_t)iw * p.nx;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (x0 + r < p.nx) dst[x0 + r] = out[r];
            img[r] += out[r].x;                           // A5: fixed (increasing w) order
        }
    }
    if (x0 < p.pstride) {
        float *prow = p.partial + ((size_t)blockIdx.y * p.nz + p.z) * p.pstride + x0;
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (x0 + r < p.pstride) prow[r] = img[r];
    }
}

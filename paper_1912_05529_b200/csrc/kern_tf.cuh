// kern_tf.cuh -- time -> frequency transform of the input section.
// PAPER.md:51 / Alg. 1 (:58): each trace is Fourier transformed along time; only the nw bins of
// the migration band are needed, so this is a [nw x nt] (twiddles) times [nt x nx] (section)
// contraction:  P0[j][x] = sum_n d[n][x] * exp(-2 pi i bins[j] n / nt).
// It is a dense contraction, but FP32 accuracy is required of P0 (the 1e-4 image bar leaves no
// room for TF32/BF16 operands), so it runs on the FP32 pipe with packed FFMA2:
//   CTA = 256 x-samples x (4 bins per warp, 4..8 warps); a thread owns 8 consecutive x and 4 bins
//   (32 complex accumulators); all lanes of a warp share their 4 bins, so the twiddle (cos, -sin) of
//   (bins[j]*n) mod nt is ONE broadcast 8-byte shared-memory load per bin and time sample.  The
//   section streams through a 32-sample shared-memory chunk (coalesced rows); for every chunk the
//   CTA first gathers its bins' 32 twiddles from the nt-entry table into a small [bin][sample]
//   array (exact integer index, 4 entries per thread), so the inner loop has no index arithmetic:
//   per time sample 2 LDS.128 + 4 broadcast LDS.64 feed 32 FFMA2.
// Bound: FP32 ALU, 4 flops per (bin, time sample, x) counted = 2 executed FMAs.
#pragma once
#include "pdm_common.cuh"

#define PDM_TF_THREADS 256     // at most; the host picks 4..8 warps to fill whole waves
#define PDM_TF_XT 8            // x samples per thread
#define PDM_TF_JT 4            // bins per thread
#define PDM_TF_XB (32 * PDM_TF_XT)
#define PDM_TF_NC 32           // time samples per shared-memory chunk

struct pdm_tf_params {
    const float  *section;     // [nt][nx]
    float2       *out;         // [nw][nx]
    const int    *bins;        // [nw]
    const float2 *tw;          // [nt] (cos, -sin)(2 pi m / nt)
    int nt, nx, nw;
    int wide_out;              // 1: nx even and P0 16-byte aligned -> 16-byte stores of the result
};

template <int CW>   // floats per async copy: 4 (nx % 4 == 0 and a 16-byte aligned section) or 1
__global__ void __launch_bounds__(PDM_TF_THREADS, 2) pdm_tf_kernel(const pdm_tf_params p)
{
    extern __shared__ __align__(16) unsigned char pdm_smem[];
    float2 *tw = reinterpret_cast<float2 *>(pdm_smem);                 // [nt]
    float *chunk = reinterpret_cast<float *>(tw + ((p.nt + 1) & ~1));    // [2][NC][XB], 16-byte aligned
    float2 *twc = reinterpret_cast<float2 *>(chunk + 2 * PDM_TF_NC * PDM_TF_XB); // [2][warps*JT][NC]

    const int tid = threadIdx.x, tx = tid & 31, ty = tid >> 5;
    const int T = blockDim.x;
    const int xb0 = blockIdx.x * PDM_TF_XB;
    const int j0 = (blockIdx.y * (T >> 5) + ty) * PDM_TF_JT;
    const int jb = (T >> 5) * PDM_TF_JT;                               // bins of this CTA
    const int jcta0 = blockIdx.y * jb;

    auto issue_chunk = [&](int n0, int b) {                            // section rows n0..n0+NC-1 -> chunk[b]
        float *dst = chunk + b * PDM_TF_NC * PDM_TF_XB;
        for (int i = tid * CW; i < PDM_TF_NC * PDM_TF_XB; i += T * CW) {
            const int nl = i / PDM_TF_XB, xl = i - nl * PDM_TF_XB;
            const int n = n0 + nl, x = xb0 + xl;
            const bool valid = n < p.nt && x < p.nx;                   // CW == 4: x and nx are multiples of 4
            const float *src = p.section + (valid ? (size_t)n * p.nx + x : 0);
            const unsigned d = (unsigned)__cvta_generic_to_shared(dst + i);
            const unsigned nbytes = valid ? 4u * CW : 0u;              // 0: zero-fill (beyond nt or nx)
            if (CW == 4) asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" :: "r"(d), "l"(src), "r"(nbytes) : "memory");
            else         asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" :: "r"(d), "l"(src), "r"(nbytes) : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    issue_chunk(0, 0);
    for (int m = tid; m < p.nt; m += T) tw[m] = __ldg(p.tw + m);

    float2 acc[PDM_TF_JT][PDM_TF_XT];
#pragma unroll
    for (int jj = 0; jj < PDM_TF_JT; ++jj)
#pragma unroll
        for (int xx = 0; xx < PDM_TF_XT; ++xx) acc[jj][xx] = make_float2(0.f, 0.f);

    for (int n0 = 0, c = 0; n0 < p.nt; n0 += PDM_TF_NC, ++c) {
        const int b = c & 1;
        __syncthreads();                                               // compute of chunk c-1 done (and tw staged)
        if (n0 + PDM_TF_NC < p.nt) {
            issue_chunk(n0 + PDM_TF_NC, b ^ 1);
            asm volatile("cp.async.wait_group 1;" ::: "memory");
        } else {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
        }
        float2 *twb = twc + b * jb * PDM_TF_NC;
        for (int e = tid; e < jb * PDM_TF_NC; e += T) {                // twiddles of this chunk
            const int jl = e / PDM_TF_NC, nl = e - jl * PDM_TF_NC;
            const int bn = (jcta0 + jl < p.nw) ? __ldg(p.bins + jcta0 + jl) : 0;
            twb[e] = tw[(bn * (n0 + nl)) % p.nt];                      // bn <= nt/2, n < nt + NC: fits int32
        }
        __syncthreads();                                               // chunk c and its twiddles visible
        const float *cb = chunk + b * PDM_TF_NC * PDM_TF_XB;
        const float2 *tb = twb + ty * PDM_TF_JT * PDM_TF_NC;
#pragma unroll 8
        for (int nl = 0; nl < PDM_TF_NC; ++nl) {                       // samples beyond nt are zero
            // a thread's 8 traces are two runs of 4 (x and x + XB/2): lane stride 16 B, conflict-free
            const float4 d0 = *reinterpret_cast<const float4 *>(cb + nl * PDM_TF_XB + tx * 4);
            const float4 d1 = *reinterpret_cast<const float4 *>(cb + nl * PDM_TF_XB + PDM_TF_XB / 2 + tx * 4);
#pragma unroll
            for (int jj = 0; jj < PDM_TF_JT; ++jj) {
                const float2 t = tb[jj * PDM_TF_NC + nl];
                acc[jj][0] = pk_fma_s(d0.x, t, acc[jj][0]);
                acc[jj][1] = pk_fma_s(d0.y, t, acc[jj][1]);
                acc[jj][2] = pk_fma_s(d0.z, t, acc[jj][2]);
                acc[jj][3] = pk_fma_s(d0.w, t, acc[jj][3]);
                acc[jj][4] = pk_fma_s(d1.x, t, acc[jj][4]);
                acc[jj][5] = pk_fma_s(d1.y, t, acc[jj][5]);
                acc[jj][6] = pk_fma_s(d1.z, t, acc[jj][6]);
                acc[jj][7] = pk_fma_s(d1.w, t, acc[jj][7]);
            }
        }
    }
    const bool wide = p.wide_out != 0;                                 // 16-byte aligned rows (host-checked)
#pragma unroll
    for (int jj = 0; jj < PDM_TF_JT; ++jj) {
        if (j0 + jj >= p.nw) continue;
        float2 *row = p.out + (size_t)(j0 + jj) * p.nx;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int x = xb0 + h * (PDM_TF_XB / 2) + tx * 4;
            if (wide && x + 4 <= p.nx) {
                *reinterpret_cast<float4 *>(row + x) =
                    make_float4(acc[jj][4 * h].x, acc[jj][4 * h].y, acc[jj][4 * h + 1].x, acc[jj][4 * h + 1].y);
                *reinterpret_cast<float4 *>(row + x + 2) =
                    make_float4(acc[jj][4 * h + 2].x, acc[jj][4 * h + 2].y, acc[jj][4 * h + 3].x, acc[jj][4 * h + 3].y);
            } else {
#pragma unroll
                for (int xx = 0; xx < 4; ++xx)
                    if (x + xx < p.nx) row[x + xx] = acc[jj][4 * h + xx];
            }
        }
    }
}

// kern_fft.cuh -- time -> frequency transform of the input section as a real FFT per trace
// (SURVEY.md 8(f) N1, Alg. 1 :58: each trace is Fourier transformed along time, :25).
//   P0[j][x] = sum_n d[n][x] exp(-2 pi i bins[j] n / nt),   nt a power of two
// The contraction form (kern_tf.cuh) spends 4*nt flops per output; an FFT spends ~5*log2(nt) per
// sample of the trace and is bound by moving the section through HBM once.
//
// One CTA transforms 2*S adjacent traces (S = 4 for nt <= 4096): traces 2p and 2p+1 are packed as
// the real and imaginary part of ONE complex sequence z_p[n] = d[n][2p] + i d[n][2p+1] (so the rows
// of the time-major section are read as 8-byte pairs, 32 contiguous bytes per row and CTA), S
// complex FFTs of length nt run in shared memory -- in-place decimation in frequency, radix 4 with
// one radix-2 stage when log2(nt) is odd, per-stage twiddle tables (w_M^j, w_M^2j, w_M^3j
// interleaved, built in double at create time) -- and the two real spectra are separated on the way out,
//   A[b] = (Z[b] + conj Z[nt-b]) / 2,      B[b] = (Z[b] - conj Z[nt-b]) / (2i),
// only for the bins of the migration band, written straight into the [nw][nx] layout pdm_migrate reads.
// Shared-memory index n lives at n + (n >> 4) (one pad per 16 samples: breaks the power-of-two strides).
#pragma once
#include "pdm_common.cuh"

#define PDM_FFT_THREADS 1024

struct pdm_fft_params {
    const float  *section;     // [nt][nx]
    float2       *out;         // [nw][nx]
    const int    *bins;        // [nw]
    const float2 *tw;          // per-stage twiddle tables, stage after stage: 3 entries per butterfly column
    int nt, log2nt, nx, nw;
    int S;                     // complex sequences (= pairs of traces) per CTA
    int ntw;                   // entries of tw
    int pair_loads;            // 1: section rows can be read as aligned 8-byte pairs (nx even, aligned base)
    int wide_out;              // 1: nx even and P0 16-byte aligned -> 16-byte stores
};

__device__ __forceinline__ int pdm_fft_phys(int n) { return n + (n >> 4); }
__device__ __forceinline__ float2 pdm_cmul(float2 a, float2 w) { return make_float2(a.x * w.x - a.y * w.y, a.x * w.y + a.y * w.x); }

static __global__ void __launch_bounds__(PDM_FFT_THREADS, 1) pdm_fft_kernel(const pdm_fft_params p)
{
    extern __shared__ __align__(16) unsigned char pdm_fft_smem[];
    const int nt = p.nt, S = p.S, tid = threadIdx.x, NT = blockDim.x;
    const int NP = nt + (nt >> 4) + 1;                            // padded sequence length
    float2 *data = reinterpret_cast<float2 *>(pdm_fft_smem);     // [S][NP]
    float2 *tw = data + (size_t)S * NP;                          // [ntw]
    const int x0 = blockIdx.x * 2 * S;

    for (int i = tid; i < p.ntw; i += NT) tw[i] = __ldg(p.tw + i);
    // section rows -> S packed complex sequences; lanes run along the pairs of a row first
    const int log2S = 31 - __clz(S);
    for (int ib = tid; ib < S * nt; ib += 8 * NT) {               // 8 independent row reads in flight per thread
        float2 v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int i = ib + u * NT;
            const int pr = i & (S - 1), n = i >> log2S;
            const int x = x0 + 2 * pr;
            v[u] = make_float2(0.f, 0.f);
            if (i < S * nt) {
                const float *row = p.section + (size_t)n * p.nx;
                if (x + 1 < p.nx) {
                    if (p.pair_loads) v[u] = __ldcs(reinterpret_cast<const float2 *>(row + x));
                    else { v[u].x = __ldcs(row + x); v[u].y = __ldcs(row + x + 1); }
                } else if (x < p.nx) v[u].x = __ldcs(row + x);
            }
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int i = ib + u * NT;
            if (i < S * nt) data[(size_t)(i & (S - 1)) * NP + pdm_fft_phys(i >> log2S)] = v[u];
        }
    }
    __syncthreads();

    // radix-4 decimation-in-frequency stages: sub-transform length M -> four of length M/4
    int log2M = p.log2nt, twoff = 0;
    const int log2q_all = p.log2nt - 2;                           // butterflies per sequence and stage = nt/4
    while (log2M >= 2) {
        const int log2q = log2M - 2, q = 1 << log2q;
        for (int b = tid; b < (S << log2q_all); b += NT) {
            const int s = b >> log2q_all, r = b & ((1 << log2q_all) - 1);
            const int blk = r >> log2q, j = r & (q - 1);
            float2 *d = data + (size_t)s * NP;
            const int i0 = pdm_fft_phys((blk << log2M) + j), i1 = pdm_fft_phys((blk << log2M) + j + q);
            const int i2 = pdm_fft_phys((blk << log2M) + j + 2 * q), i3 = pdm_fft_phys((blk << log2M) + j + 3 * q);
            const float2 a0 = d[i0], a1 = d[i1], a2 = d[i2], a3 = d[i3];
            const float2 t0 = make_float2(a0.x + a2.x, a0.y + a2.y), t1 = make_float2(a0.x - a2.x, a0.y - a2.y);
            const float2 t2 = make_float2(a1.x + a3.x, a1.y + a3.y);
            const float2 t3 = make_float2(a1.y - a3.y, a3.x - a1.x);           // -i (a1 - a3)
            const float2 w1 = tw[twoff + 3 * j], w2 = tw[twoff + 3 * j + 1], w3 = tw[twoff + 3 * j + 2];
            d[i0] = make_float2(t0.x + t2.x, t0.y + t2.y);
            d[i1] = pdm_cmul(make_float2(t1.x + t3.x, t1.y + t3.y), w1);
            d[i2] = pdm_cmul(make_float2(t0.x - t2.x, t0.y - t2.y), w2);
            d[i3] = pdm_cmul(make_float2(t1.x - t3.x, t1.y - t3.y), w3);
        }
        __syncthreads();
        twoff += 3 * q;
        log2M -= 2;
    }
    if (log2M == 1) {                                             // last radix-2 stage (no twiddles)
        for (int b = tid; b < (S << (p.log2nt - 1)); b += NT) {
            const int s = b >> (p.log2nt - 1), r = b & ((1 << (p.log2nt - 1)) - 1);
            float2 *d = data + (size_t)s * NP;
            const int i0 = pdm_fft_phys(2 * r), i1 = pdm_fft_phys(2 * r + 1);
            const float2 a = d[i0], c = d[i1];
            d[i0] = make_float2(a.x + c.x, a.y + c.y);
            d[i1] = make_float2(a.x - c.x, a.y - c.y);
        }
        __syncthreads();
    }

    // in-place DIF leaves bin k at the digit-reversed position (radix-4 digits, then the radix-2 bit)
    auto pos_of = [&](int k) {
        int pos = 0, rem = p.log2nt;
        while (rem >= 2) { rem -= 2; pos += (k & 3) << rem; k >>= 2; }
        if (rem == 1) pos += k & 1;
        return pdm_fft_phys(pos);
    };
    for (int i = tid; i < S * p.nw; i += NT) {
        const int pr = i & (S - 1), jb = i >> log2S;
        const int x = x0 + 2 * pr;
        if (x >= p.nx) continue;
        const int b = __ldg(p.bins + jb);
        const float2 *d = data + (size_t)pr * NP;
        const float2 zb = d[pos_of(b)], zc = d[pos_of((nt - b) & (nt - 1))];
        const float2 A = make_float2(0.5f * (zb.x + zc.x), 0.5f * (zb.y - zc.y));
        const float2 B = make_float2(0.5f * (zb.y + zc.y), 0.5f * (zc.x - zb.x));
        float2 *o = p.out + (size_t)jb * p.nx + x;
        if (x + 1 < p.nx) {
            if (p.wide_out) __stcs(reinterpret_cast<float4 *>(o), make_float4(A.x, A.y, B.x, B.y));
            else { o[0] = A; o[1] = B; }
        } else o[0] = A;
    }
}

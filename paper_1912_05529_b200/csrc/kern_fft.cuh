// kern_fft.cuh -- time -> frequency transform of the input section as a real FFT per trace
// (SURVEY.md 8(f) N1, Alg. 1 :58: each trace is Fourier transformed along time, :25).
//   P0[j][x] = sum_n d[n][x] exp(-2 pi i bins[j] n / nt),   nt a power of two
// The contraction form (kern_tf.cuh) spends 4*nt flops per output; an FFT spends ~5*log2(nt) per
// sample of the trace and is bound by moving the section through HBM once.
//
// One CTA transforms 2*S adjacent traces (S = 4 for nt <= 4096): traces 2p and 2p+1 are packed as
// the real and imaginary part of ONE complex sequence z_p[n] = d[n][2p] + i d[n][2p+1] (so the rows
// of the time-major section are read as 8-byte pairs, 32 contiguous bytes per row and CTA), S
// complex FFTs of length nt run in shared memory -- in-place decimation in frequency, two radix-4 stages
// per pass in registers (radix 16), one radix-4 / radix-2 stage for the odd cases, per-stage twiddle tables (w_M^j, w_M^2j, w_M^3j
// interleaved, built in double at create time) -- and the two real spectra are separated on the way out,
//   A[b] = (Z[b] + conj Z[nt-b]) / 2,      B[b] = (Z[b] - conj Z[nt-b]) / (2i),
// only for the bins of the migration band, written straight into the [nw][nx] layout pdm_migrate reads.
// Shared-memory index n lives at n + (n >> 4) (one pad per 16 samples: breaks the power-of-two strides).
#pragma once
#include "pdm_common.cuh"

#define PDM_FFT_THREADS 512

struct pdm_fft_params {
    const float  *section;     // [nt][nx]
    float2       *out;         // [nw][nx]
    const int2   *binpos;      // [nw] shared-memory positions of bin b and of bin nt-b after the in-place FFT
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
    for (int i = tid; i < p.ntw; i += NT) tw[i] = __ldg(p.tw + i);      // once per (persistent) CTA
    const int ntiles = (p.nx + 2 * S - 1) / (2 * S);
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const int x0 = tile * 2 * S;
    // section rows -> S packed complex sequences; lanes run along the pairs of a row first
    const int log2S = 31 - __clz(S);
    for (int ib = tid; ib < S * nt; ib += 16 * NT) {              // 16 independent row reads in flight per thread
        float2 v[16];
#pragma unroll
        for (int u = 0; u < 16; ++u) {
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
        for (int u = 0; u < 16; ++u) {
            const int i = ib + u * NT;
            if (i < S * nt) data[(size_t)(i & (S - 1)) * NP + pdm_fft_phys(i >> log2S)] = v[u];
        }
    }
    __syncthreads();

    // Decimation-in-frequency stages.  Two radix-4 stages at a time in registers (a radix-16 pass: sub-
    // transform length M -> sixteen of length M/16) while M >= 16: level 1 is the M-stage butterfly on the
    // columns j + m1*q (q = M/16), level 2 the (M/4)-stage butterfly of the four results of one residue
    // -- 16 loads, 16 stores and 15 twiddles per 16 points instead of 32 + 32 + 24; one radix-4 stage
    // (M = 4 or 8) and one radix-2 stage (M = 2) finish odd cases.
    int log2M = p.log2nt, twoff = 0;
    while (log2M >= 4) {
        const int log2q = log2M - 4, q = 1 << log2q;
        const int tw2 = twoff + 3 * (4 * q);                      // twiddles of the (M/4)-stage follow the M-stage's
        const int per_seq = 1 << (p.log2nt - 4);                  // radix-16 butterflies per sequence
        for (int b = tid; b < S * per_seq; b += NT) {
            const int s = b >> (p.log2nt - 4), r = b & (per_seq - 1);
            const int blk = r >> log2q, j = r & (q - 1);
            float2 *d = data + (size_t)s * NP;
            const int n0 = (blk << log2M) + j;
            float2 a[16];
#pragma unroll
            for (int m = 0; m < 16; ++m) a[m] = d[pdm_fft_phys(n0 + m * q)];
            // level 1: for each m1, radix-4 over m2 (points m1 + 4 m2), twiddles w_M^{r1 (j + m1 q)}
#pragma unroll
            for (int m1 = 0; m1 < 4; ++m1) {
                const float2 a0 = a[m1], a1 = a[m1 + 4], a2 = a[m1 + 8], a3 = a[m1 + 12];
                const float2 t0 = make_float2(a0.x + a2.x, a0.y + a2.y), t1 = make_float2(a0.x - a2.x, a0.y - a2.y);
                const float2 t2 = make_float2(a1.x + a3.x, a1.y + a3.y);
                const float2 t3 = make_float2(a1.y - a3.y, a3.x - a1.x);       // -i (a1 - a3)
                const int c = twoff + 3 * (j + m1 * q);
                a[m1]      = make_float2(t0.x + t2.x, t0.y + t2.y);
                a[m1 + 4]  = pdm_cmul(make_float2(t1.x + t3.x, t1.y + t3.y), tw[c]);
                a[m1 + 8]  = pdm_cmul(make_float2(t0.x - t2.x, t0.y - t2.y), tw[c + 1]);
                a[m1 + 12] = pdm_cmul(make_float2(t1.x - t3.x, t1.y - t3.y), tw[c + 2]);
            }
            // level 2: for each residue r1 (now at a[4 r1 + m1]), radix-4 over m1, twiddles w_{M/4}^{r2 j}
            const float2 w1 = tw[tw2 + 3 * j], w2 = tw[tw2 + 3 * j + 1], w3 = tw[tw2 + 3 * j + 2];
#pragma unroll
            for (int r1 = 0; r1 < 4; ++r1) {
                const float2 a0 = a[4 * r1], a1 = a[4 * r1 + 1], a2 = a[4 * r1 + 2], a3 = a[4 * r1 + 3];
                const float2 t0 = make_float2(a0.x + a2.x, a0.y + a2.y), t1 = make_float2(a0.x - a2.x, a0.y - a2.y);
                const float2 t2 = make_float2(a1.x + a3.x, a1.y + a3.y);
                const float2 t3 = make_float2(a1.y - a3.y, a3.x - a1.x);
                // result (r1, r2) lives at n0 + (4 r1 + r2) q
                d[pdm_fft_phys(n0 + (4 * r1) * q)]     = make_float2(t0.x + t2.x, t0.y + t2.y);
                d[pdm_fft_phys(n0 + (4 * r1 + 1) * q)] = pdm_cmul(make_float2(t1.x + t3.x, t1.y + t3.y), w1);
                d[pdm_fft_phys(n0 + (4 * r1 + 2) * q)] = pdm_cmul(make_float2(t0.x - t2.x, t0.y - t2.y), w2);
                d[pdm_fft_phys(n0 + (4 * r1 + 3) * q)] = pdm_cmul(make_float2(t1.x - t3.x, t1.y - t3.y), w3);
            }
        }
        __syncthreads();
        twoff = tw2 + 3 * q;
        log2M -= 4;
    }
    const int log2q_all = p.log2nt - 2;                           // radix-4 butterflies per sequence and stage = nt/4
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

    // in-place DIF leaves bin k at the digit-reversed position (radix-4 digits, then the radix-2 bit):
    // the host tabulates it (pdm_tf_create), with the shared-memory padding applied
    for (int i = tid; i < S * p.nw; i += NT) {
        const int pr = i & (S - 1), jb = i >> log2S;
        const int x = x0 + 2 * pr;
        if (x >= p.nx) continue;
        const int2 bp = __ldg(p.binpos + jb);
        const float2 *d = data + (size_t)pr * NP;
        const float2 zb = d[bp.x], zc = d[bp.y];
        const float2 A = make_float2(0.5f * (zb.x + zc.x), 0.5f * (zb.y - zc.y));
        const float2 B = make_float2(0.5f * (zb.y + zc.y), 0.5f * (zc.x - zb.x));
        float2 *o = p.out + (size_t)jb * p.nx + x;
        if (x + 1 < p.nx) {
            if (p.wide_out) __stcs(reinterpret_cast<float4 *>(o), make_float4(A.x, A.y, B.x, B.y));
            else { o[0] = A; o[1] = B; }
        } else o[0] = A;
    }
    __syncthreads();                                              // the sequences are overwritten by the next tile
    }
}

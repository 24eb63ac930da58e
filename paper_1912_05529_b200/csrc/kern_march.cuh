// kern_march.cuh -- PDM_PATH_SMEM, the main form (BASELINE.json north_star; "block
// level synchronization" instead of kernel exit):
//   one CTA keeps one frequency's x-line in shared memory (ping-pong) and marches ALL nz depth
//   steps without the wavefield ever returning to HBM.  Per depth step:
//     A1  j = clamp(rint(w*q[z][x]))                  (R3; q rows come from L2, one pass ahead)
//     A2  taps W_0..W_L of row j                      (half table; rows this w can touch are staged
//                                                      in shared memory, else read through L1)
//     A3  P'(x) = W_0 P(x) + sum_k W_k (P(x-k)+P(x+k)) (Eq. (1) PAPER.md:45 folded with W_k == W_-k)
//     A4  __syncthreads, swap buffers
//     A5  partial[cta][z][x] (+)= Re P'(x)            (fixed order; pdm_reduce_partials sums CTAs)
//
// Register tiling: a thread owns R consecutive outputs ("group").  For tap k it needs the two
// R-wide windows P[x0-k .. x0+R-1-k] and P[x0+k .. x0+R-1+k]; going from k to k+1 each window
// slides by one sample, so with the k loop fully unrolled the windows live in 2R register pairs
// and every wavefield sample is read from shared memory once per thread (as 16-byte pairs).
// Arithmetic is packed FP32 (FFMA2/FADD2): per (k, output) one FADD2 (re,im of the folded sum)
// and two FFMA2 with the scalar-broadcast operand form (acc_a += Wr*S, acc_b += Wi*S); the
// complex result is (a.x - b.y, a.y + b.x).
//
// Shared-memory line layout: groups of R samples followed by 2 pad samples, HG all-zero halo
// groups on both sides (R5: zero outside [0,nx), so no edge branches).  Lane stride is then
// (R+2)*8 B, which makes the 16-byte window loads / stores of a quarter-warp bank-conflict free.
#pragma once
#include "pdm_common.cuh"

#define PDM_MARCH_MAX_THREADS 384

struct pdm_march_params {
    const float2 *P0;        // [nw][nx]
    float        *partial;   // [grid][nz][pstride]
    const float  *q;         // [nz][qstride]
    const float  *omega;     // [nw]
    const float4 *half;      // [ntab][half16]
    const int    *rowoff;    // [nw+1]
    const int    *rows;      // row lists
    cudaTextureObject_t tex; // the half table as a linear float4 texture
    const int4   *segs;      // work list: {line, z0, z1, hand-off slot or -1}, in execution order per CTA
    const int    *segoff;    // [grid+1] offsets into segs
    float2       *handoff;   // [nslots][nx] wavefield of a line split between two CTAs, at the split depth
    int          *flags;     // [nslots] 0 = empty, 1 = hand-off line published (reset by the consumer)
    int nx, nz, nw, ntab;
    int qstride, pstride, half16;
    int ngroups, passes, slots, map_len;
    int force_general;       // PDM_FORCE_GENERAL: never take the thread-uniform fast path (debug)
};

__host__ __device__ constexpr int pdm_floordiv(int a, int b) { return (a >= 0) ? a / b : -((-a + b - 1) / b); }
__host__ __device__ constexpr int pdm_mod(int a, int b) { return a - pdm_floordiv(a, b) * b; }
// slot offset (in float2) of sample x0+m relative to the slot of x0 (x0 = first sample of a group)
// PAD = pad samples after every group of R (2 in the one-line-per-CTA layouts, 0 in the frequency-packed one)
template <int R, int PAD = 2> __host__ __device__ constexpr int pdm_soff(int m) { return m + PAD * pdm_floordiv(m, R); }
template <int L, int R> __host__ __device__ constexpr int pdm_halo_groups() { return (L + 1 + R - 1) / R; }

__device__ __forceinline__ float2 f4lo(float4 v) { return make_float2(v.x, v.y); }
__device__ __forceinline__ float2 f4hi(float4 v) { return make_float2(v.z, v.w); }

// One group of R outputs.  `base` = &line[slot(x0)];  tbase + toff[r] = first float4 of the half
// row of output r (all equal when UNIFORM, in which case only toff[0] is read).  tbase is passed
// separately from the offsets so that after inlining the compiler still knows its address space.
// Operand form: acc_a += (W.re, W.im) * S.x, acc_b += (W.re, W.im) * S.y with the tap PAIR as the
// packed operand and the folded sample as the scalar one: the tap pair is then the same register
// pair for up to 2R consecutive FFMA2 (register-reuse cache), which keeps the register-file reads
// per instruction at <= 2 per bank; the scalar-tap form measured 0.80 of the pipe at best.
// TEXMASK: bit r set = output r fetches its tap rows through the TEXTURE unit (tex1Dfetch on the
// global half table; toff[r] is then a GLOBAL float4 index) through a 3-deep register ring, instead
// of the LSU path: the texture unit is a second gather path whose bandwidth adds to the LSU's
// (random 16-byte gathers, measured: shared memory 54 B/clk/SM, texture 23, mixed 3:1 71).
template <int L, int R, bool UNIFORM, bool DEDUP, unsigned TEXMASK = 0u, int PAD = 2>
__device__ __forceinline__ void pdm_fir_group(const float2 *__restrict__ base,
                                              const float4 *__restrict__ tbase,
                                              const int (&toff)[R], float2 (&out)[R],
                                              cudaTextureObject_t tex = 0)
{
    float2 wl[R], wr[R], acc_a[R], acc_b[R];
    float4 tw[UNIFORM ? 1 : R];
    constexpr int TMAX = L / 2;                         // last float4 of a half row that is used
    float4 tx[R][3];
#pragma unroll
    for (int r = 0; r < R; ++r)
        if ((TEXMASK >> r) & 1u) {
#pragma unroll
            for (int s = 0; s < 3; ++s)
                if (s <= TMAX) tx[r][s] = tex1Dfetch<float4>(tex, toff[r] + s);
        }
#pragma unroll
    for (int i = 0; i < R / 2; ++i) {
        const float4 v = *reinterpret_cast<const float4 *>(base + 2 * i);
        wl[2 * i] = f4lo(v); wl[2 * i + 1] = f4hi(v);
        wr[2 * i] = f4lo(v); wr[2 * i + 1] = f4hi(v);
    }
    // DEDUP (plans whose model gives nearly every sample its own row, i.e. the tap gather is the
    // bound): consecutive outputs of a thread still repeat a row often enough (smooth models) that
    // fetching a row only where it differs from the previous output's (predicated loads) pays.
    bool same[R];
#pragma unroll
    for (int r = 0; r < R; ++r)
        same[r] = ((TEXMASK >> r) & 1u) || (DEDUP && !UNIFORM && r > 0 && !((TEXMASK >> (r - 1)) & 1u) && toff[r] == toff[r - 1]);
#pragma unroll
    for (int r = 0; r < (UNIFORM ? 1 : R); ++r) {
        if (DEDUP && r > 0) tw[r] = tw[r - 1];
        if (!same[r]) tw[r] = tbase[toff[r]];
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {                       // centre tap W_0
        const float4 t = ((TEXMASK >> r) & 1u) ? tx[r][0] : tw[UNIFORM ? 0 : r];
        acc_a[r] = pk_mul_s(wl[r].x, f4lo(t));
        acc_b[r] = pk_mul_s(wl[r].y, f4lo(t));
    }
    float4 lv = make_float4(0.f, 0.f, 0.f, 0.f), rv = lv;
#pragma unroll
    for (int k = 1; k <= L; ++k) {
        if (k & 1) {                                    // two new samples per side serve k and k+1
            lv = *reinterpret_cast<const float4 *>(base + pdm_soff<R, PAD>(-k - 1));
            rv = *reinterpret_cast<const float4 *>(base + pdm_soff<R, PAD>(R + k - 1));
            wl[pdm_mod(-k, R)] = f4hi(lv);
            wr[pdm_mod(k - 1, R)] = f4lo(rv);
        } else {
            wl[pdm_mod(-k, R)] = f4lo(lv);
            wr[pdm_mod(k - 1, R)] = f4hi(rv);
#pragma unroll
            for (int r = 0; r < (UNIFORM ? 1 : R); ++r) {
                if (DEDUP && r > 0) tw[r] = tw[r - 1];
                if (!same[r]) tw[r] = tbase[toff[r] + k / 2];
            }
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float4 t = ((TEXMASK >> r) & 1u) ? tx[r][(k / 2) % 3] : tw[UNIFORM ? 0 : r];
            const float2 W = (k & 1) ? f4hi(t) : f4lo(t);
            const float2 s = pk_add(wl[pdm_mod(r - k, R)], wr[pdm_mod(r + k, R)]);
            acc_a[r] = pk_fma_s(s.x, W, acc_a[r]);
            acc_b[r] = pk_fma_s(s.y, W, acc_b[r]);
        }
        if ((k & 1) && k / 2 + 3 <= TMAX) {             // float4 k/2 is spent: refill its ring slot
#pragma unroll
            for (int r = 0; r < R; ++r)
                if ((TEXMASK >> r) & 1u) tx[r][(k / 2) % 3] = tex1Dfetch<float4>(tex, toff[r] + k / 2 + 3);
        }
    }
#pragma unroll
    for (int r = 0; r < R; ++r) out[r] = make_float2(acc_a[r].x - acc_b[r].y, acc_a[r].y + acc_b[r].x);
}

// The same group of R outputs for a table that is NOT symmetric in k (general operators, PAPER.md:39,
// :83): Eq. (1) literally, P'(x) = sum_k W_k P(x-k) with W_k and W_-k distinct.
// Table row layout: float4 unit k = (W_k, W_-k), k = 0..L (unit 0 holds W_0 twice).  Same sliding
// register windows; 4 FFMA2 per (k, output) instead of 1 FADD2 + 2 FFMA2: 8L+4 lane-ops per output.
template <int L, int R, bool UNIFORM, int PAD = 2>
__device__ __forceinline__ void pdm_fir_group_asym(const float2 *__restrict__ base,
                                                   const float4 *__restrict__ tbase,
                                                   const int (&toff)[R], float2 (&out)[R])
{
    float2 wl[R], wr[R], acc_a[R], acc_b[R];
    float4 tw[UNIFORM ? 1 : R];
#pragma unroll
    for (int i = 0; i < R / 2; ++i) {
        const float4 v = *reinterpret_cast<const float4 *>(base + 2 * i);
        wl[2 * i] = f4lo(v); wl[2 * i + 1] = f4hi(v);
        wr[2 * i] = f4lo(v); wr[2 * i + 1] = f4hi(v);
    }
#pragma unroll
    for (int r = 0; r < (UNIFORM ? 1 : R); ++r) tw[r] = tbase[toff[r]];
#pragma unroll
    for (int r = 0; r < R; ++r) {                       // centre tap W_0
        const float4 t = tw[UNIFORM ? 0 : r];
        acc_a[r] = pk_mul_s(wl[r].x, f4lo(t));
        acc_b[r] = pk_mul_s(wl[r].y, f4lo(t));
    }
    float4 lv = make_float4(0.f, 0.f, 0.f, 0.f), rv = lv;
#pragma unroll
    for (int k = 1; k <= L; ++k) {
        if (k & 1) {
            lv = *reinterpret_cast<const float4 *>(base + pdm_soff<R, PAD>(-k - 1));
            rv = *reinterpret_cast<const float4 *>(base + pdm_soff<R, PAD>(R + k - 1));
            wl[pdm_mod(-k, R)] = f4hi(lv);
            wr[pdm_mod(k - 1, R)] = f4lo(rv);
        } else {
            wl[pdm_mod(-k, R)] = f4lo(lv);
            wr[pdm_mod(k - 1, R)] = f4hi(rv);
        }
#pragma unroll
        for (int r = 0; r < (UNIFORM ? 1 : R); ++r) tw[r] = tbase[toff[r] + k];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float4 t = tw[UNIFORM ? 0 : r];
            const float2 a = wl[pdm_mod(r - k, R)];     // P(x-k): multiplied by W_k   (R11)
            const float2 b = wr[pdm_mod(r + k, R)];     // P(x+k): multiplied by W_-k
            acc_a[r] = pk_fma_s(a.x, f4lo(t), acc_a[r]);
            acc_b[r] = pk_fma_s(a.y, f4lo(t), acc_b[r]);
            acc_a[r] = pk_fma_s(b.x, f4hi(t), acc_a[r]);
            acc_b[r] = pk_fma_s(b.y, f4hi(t), acc_b[r]);
        }
    }
#pragma unroll
    for (int r = 0; r < R; ++r) out[r] = make_float2(acc_a[r].x - acc_b[r].y, acc_a[r].y + acc_b[r].x);
}

// R = 8: one CTA of up to 384 threads per SM.  R = 4 (short lines, few of them): up to 256 threads and
// at least two CTAs per SM, so that small problems put more warps on an SM.
template <int L, int R, bool TAPS_SMEM, bool DEDUP, bool SYM = true>
__global__ void __launch_bounds__(R >= 8 ? PDM_MARCH_MAX_THREADS : 256, R >= 8 ? 1 : 2) pdm_march_kernel(const pdm_march_params p)
{
    static_assert(R % 2 == 0 && R >= 2, "R must be even");
    constexpr int HG = pdm_halo_groups<L, R>();
    constexpr int GS = R + 2;
    // per-sample-row plans only: 2 of a thread's 8 tap rows through the texture unit for the shortest
    // filters, 1 of 8 for longer ones (measured best per length; more costs registers the loop needs)
    constexpr unsigned TEXMASK = (SYM && DEDUP && R == 8) ? (L <= 7 ? 0x88u : 0x80u) : 0u;
    extern __shared__ __align__(16) unsigned char pdm_smem[];
    float2 *buf_a = reinterpret_cast<float2 *>(pdm_smem);
    float2 *buf_b = buf_a + p.slots;
    unsigned short *map = reinterpret_cast<unsigned short *>(buf_b + p.slots);
    float4 *slice = reinterpret_cast<float4 *>(map + p.map_len);

    // A4 without a CTA barrier: prog[1 + w] = depth steps of the current segment that warp w has
    // completed.  A warp owns `passes` x 32 CONTIGUOUS groups, so step s+1 of warp w reads only
    // what warps w-1, w, w+1 wrote in step s (halo <= HG groups < 32): it may start as soon as
    // both neighbours have completed step s, which also covers the write-after-read on the
    // ping-pong buffer.  prog[0] and prog[nwarps + 1] are sentinels (always ahead).
    __shared__ int prog[PDM_MARCH_MAX_THREADS / 32 + 2];
    const int tid = threadIdx.x, T = blockDim.x;
    const int warp = tid >> 5, lane = tid & 31, nwarps = T >> 5;
    const int ntab_m1 = p.ntab - 1;
    for (int i = tid; i < p.slots; i += T)              // 2*slots float2 = slots float4
        reinterpret_cast<float4 *>(buf_a)[i] = make_float4(0.f, 0.f, 0.f, 0.f);

    float *const my_partial = p.partial + (size_t)blockIdx.x * p.nz * p.pstride;
    // Rows z < wz of my_partial already hold sums of earlier segments; rows >= wz are unwritten.
    int wz = 0;

    // Work list (pdm_create): whole lines, plus -- when depth-split balancing is on -- the HEAD
    // [0,z1) of one line (done first, then published through `handoff`) and the TAIL [z0,nz) of
    // another (done last, after the CTA that owns its head has published it).  Every CTA then
    // marches the same number of depth steps; lines are sequential in z but nothing
    // says a line must stay on one SM.
    const int seg_end = p.segoff[blockIdx.x + 1];
    for (int sidx = p.segoff[blockIdx.x]; sidx < seg_end; ++sidx) {
        const int4 sg = p.segs[sidx];
        const int line = sg.x, z0 = sg.y, z1 = sg.z, slot = sg.w;
        __syncthreads();                                 // previous segment (and the zero fill) done
        const float w = p.omega[line];
        if (TAPS_SMEM) {                                 // A2 staging: rows this omega can touch
            const int r0 = p.rowoff[line], nrows = p.rowoff[line + 1] - r0;
            for (int i = tid; i < nrows; i += T) map[p.rows[r0 + i]] = (unsigned short)i;
            const int n4 = nrows * p.half16;
            for (int e = tid; e < n4; e += T) {
                const int s = e / p.half16, c = e - s * p.half16;
                slice[e] = p.half[(size_t)p.rows[r0 + s] * p.half16 + c];
            }
        }
        if (z0 > 0) {                                    // TAIL: wait for the head's owner
            if (wz < p.nz) {                             // no whole line came before: define the rest
                const int n4 = (p.nz - wz) * (p.pstride / 4);
                float4 *dstz = reinterpret_cast<float4 *>(my_partial + (size_t)wz * p.pstride);
                for (int i = tid; i < n4; i += T) dstz[i] = make_float4(0.f, 0.f, 0.f, 0.f);
                wz = p.nz;
            }
            if (tid == 0) {
                unsigned v;
                do {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p.flags + slot) : "memory");
                    if (!v) __nanosleep(200);
                } while (!v);
                p.flags[slot] = 0;                       // one producer, one consumer per migrate
            }
            __syncthreads();
        }
        if (tid < nwarps + 2) {                          // sentinels and warps beyond the line: always ahead
            const bool idle = tid == 0 || tid == nwarps + 1 || (tid - 1) * p.passes * 32 >= p.ngroups;
            prog[tid] = idle ? 0x7fffffff : 0;
        }
        {                                                // P(z0): P0[line] or the hand-off
            const float2 *src = (z0 == 0) ? p.P0 + (size_t)line * p.nx : p.handoff + (size_t)slot * p.nx;
            for (int x = tid; x < p.nx; x += T) {
                const int g = x / R;
                buf_a[(HG + g) * GS + (x - g * R)] = __ldcg(src + x);
            }
        }
        __syncthreads();

        // passes in which this warp has at least one group inside the line (warp-uniform)
        const int npw = min(p.passes, max(0, (p.ngroups - warp * p.passes * 32 + 31) / 32));
        if (npw > 0) {
            float2 *cur = buf_a, *nxt = buf_b;
            const float4 *const tbase = TAPS_SMEM ? slice : p.half;
            // A1/A2 run ahead of A3 (neither depends on the wavefield): q is requested two groups
            // ahead, and the table offsets tn[] / thread-uniformity flag un of the NEXT group are
            // computed at the top of a group, before the wait on the neighbouring warps.
            float qn[R];
            int tn[R];
            bool un = false;
            auto load_q = [&](int zq, int pq) {
                const int gq = min((warp * p.passes + pq) * 32 + lane, p.ngroups - 1);
                const float4 *qp = reinterpret_cast<const float4 *>(p.q + (size_t)zq * p.qstride + (size_t)gq * R);
#pragma unroll
                for (int i = 0; i < R / 4; ++i) {
                    const float4 v = __ldg(qp + i);
                    qn[4 * i] = v.x; qn[4 * i + 1] = v.y; qn[4 * i + 2] = v.z; qn[4 * i + 3] = v.w;
                }
            };
            auto index_next = [&]() {
                int jn[R];
                bool u = true;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    jn[r] = pdm_index(w, qn[r], ntab_m1);
                    u = u && (jn[r] == jn[0]);
                }
                un = u && !p.force_general;
#pragma unroll
                for (int r = 0; r < R; ++r)
                    tn[r] = (((TEXMASK >> r) & 1u) ? jn[r] : (TAPS_SMEM ? (int)map[jn[r]] : jn[r])) * p.half16;
            };
            load_q(z0, 0);
            index_next();
            int qz = z0, qp = 1;                         // (z, pass) of the q row requested last
            if (qp == npw) { qp = 0; ++qz; }
            if (qz < z1) load_q(qz, qp);
            for (int z = z0; z < z1; ++z) {
                const bool accumulate = z < wz;
                for (int pass = 0; pass < npw; ++pass) {
                    const int g_raw = (warp * p.passes + pass) * 32 + lane;
                    const bool active = g_raw < p.ngroups;
                    const int g = active ? g_raw : p.ngroups - 1;
                    int toff[R];
#pragma unroll
                    for (int r = 0; r < R; ++r) toff[r] = tn[r];
                    const bool uni = __all_sync(0xffffffffu, un);
                    index_next();                        // next group's offsets, from the q requested a group ago
                    if (++qp == npw) { qp = 0; ++qz; }   // A1 prefetch: q two groups ahead
                    if (qz < z1) load_q(qz, qp);         // else: tn/un of groups that are never run
                    float4 *prow = reinterpret_cast<float4 *>(my_partial + (size_t)z * p.pstride + (size_t)g * R);
                    // short filters: a group is over before a DRAM load returns, and the partial image
                    // is far larger than L2 -- pull the NEXT depth step's row into L2 a step ahead
                    // (+5 % at 15 taps; long filters hide the latency anyway and lose 1.5 % to it)
                    if (L <= 15 && z + 1 < min(wz, z1))
                        asm volatile("prefetch.global.L2 [%0];" :: "l"(reinterpret_cast<const float *>(prow) + p.pstride));
                    float4 pold[R / 4];
                    if (accumulate) {                    // A5: old partial row, consumed at the end
#pragma unroll
                        for (int i = 0; i < R / 4; ++i) pold[i] = __ldcs(prow + i);
                    } else {
#pragma unroll
                        for (int i = 0; i < R / 4; ++i) pold[i] = make_float4(0.f, 0.f, 0.f, 0.f);
                    }
                    if (pass == 0 && z > z0) {           // A4: neighbours have completed step z-1
                        if (lane == 0) {
                            const int need = z - z0;
                            while (*(volatile int *)&prog[warp] < need) { }
                            while (*(volatile int *)&prog[warp + 2] < need) { }
                            __threadfence_block();
                        }
                        __syncwarp();
                    }
                    const float2 *base = cur + (HG + g) * GS;
                    float2 out[R];
                    if (SYM) {
                        if (uni) pdm_fir_group<L, R, true, false>(base, tbase, toff, out);
                        else     pdm_fir_group<L, R, false, DEDUP, TEXMASK>(base, tbase, toff, out, p.tex);
                    } else {
                        if (uni) pdm_fir_group_asym<L, R, true>(base, tbase, toff, out);
                        else     pdm_fir_group_asym<L, R, false>(base, tbase, toff, out);
                    }
                    if (active) {
                        const int x0 = g * R;
                        float2 *dst = nxt + (HG + g) * GS;
#pragma unroll
                        for (int i = 0; i < R / 2; ++i) {    // samples beyond nx stay zero (R5)
                            float2 a = out[2 * i], b = out[2 * i + 1];
                            if (x0 + 2 * i >= p.nx) a = make_float2(0.f, 0.f);
                            if (x0 + 2 * i + 1 >= p.nx) b = make_float2(0.f, 0.f);
                            *reinterpret_cast<float4 *>(dst + 2 * i) = make_float4(a.x, a.y, b.x, b.y);
                        }
#pragma unroll
                        for (int i = 0; i < R / 4; ++i) {
                            float4 v = pold[i];
                            v.x += out[4 * i].x; v.y += out[4 * i + 1].x;
                            v.z += out[4 * i + 2].x; v.w += out[4 * i + 3].x;
                            __stcs(prow + i, v);
                        }
                    }
                }
                __syncwarp();                            // A4: publish this warp's step z
                if (lane == 0) {
                    __threadfence_block();
                    *(volatile int *)&prog[warp + 1] = z - z0 + 1;
                }
                float2 *t = cur; cur = nxt; nxt = t;
            }
        }
        float2 *const cur = ((z1 - z0) & 1) ? buf_b : buf_a;   // the line at depth z1
        if (z0 == 0) wz = max(wz, z1);                   // a head or a whole line defines rows [0,z1)
        if (z1 < p.nz) {                                 // HEAD: publish the line at depth z1
            __syncthreads();                             // every warp has completed step z1-1
            float2 *dst = p.handoff + (size_t)slot * p.nx;
            for (int x = tid; x < p.nx; x += T) {
                const int g = x / R;
                __stcg(dst + x, cur[(HG + g) * GS + (x - g * R)]);
            }
            __threadfence();
            __syncthreads();
            if (tid == 0) {
                const unsigned one = 1u;
                asm volatile("st.release.gpu.global.u32 [%0], %1;" :: "l"(p.flags + slot), "r"(one) : "memory");
            }
        }
    }
}

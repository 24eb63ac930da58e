// kern_3d.cuh -- the 3-D variant of the hot path ("requires 2-D filters
// as extrapolators", :47; reading R18 of DESIGN.md):
//   P'(y,x) = sum_{ky,kx = -L..L} W[idx(x,y)][ky][kx] * P(y-ky, x-kx),   image[z][y][x] = sum_w Re P'
// One launch per depth step, planes [nw][ny][nx] ping-pong in HBM.  A CTA owns an
// (8 rows x 256 samples) output tile and walks a GROUP of frequencies for it (q tile read once, Re P
// summed over the group in registers in fixed order, as in kern_tiled.cuh).  Per frequency the tile
// plus its +-L halo rows / +-HG halo groups arrives by cp.async (zero fill outside the grid = R5) into
// one of two shared-memory buffers while the previous one is computed.  A thread owns R = 8 consecutive
// x of one row; the 2-D operator is applied as 2L+1 one-dimensional passes (one per ky) of the
// register-tiled sliding-window FIR of kern_march.cuh in its general (unfolded) form: the table row of
// (ky, .) is stored as (W[ky][kx], W[ky][-kx]) units, kx = 0..L.
#pragma once
#include "pdm_common.cuh"
#include "kern_march.cuh"
#include "kern_tiled.cuh"      // pdm_cp_async

#define PDM3_THREADS 256
#define PDM3_TY 8              // output rows per CTA (one per warp)
#define PDM3_TX 256            // output samples per row and CTA (32 lanes x 8)

struct pdm3_params {
    const float2 *Pin;       // [nw][ny][nx] plane at depth z
    float2       *Pout;      // [nw][ny][nx] plane at depth z+1
    float        *partial;   // [wgroups][nz][ny][pstride]
    const float  *q;         // [nz][ny][qstride]
    const float  *omega;     // [nw]
    const float4 *tab;       // general: [ntab][2L+1][L+1] units (W[ky][kx], W[ky][-kx]); SYM2: [ntab][L+1][(L+2)/2]
                             // units (W[ky][2t], W[ky][2t+1]), ky >= 0
    int nx, ny, nz, nw, ntab;
    int qstride, pstride;
    int z, w_per_group;
    int force_general;
    int slice_rows;          // table rows the shared-memory slice holds (0: rows are read through L1)
};

// One ky pass: acc += sum_kx W[ky][kx] * P(y-ky, x-kx) for the thread's 8 outputs -- the general
// (unfolded) register-tiled FIR of kern_march.cuh, accumulating.  tb + toff[r] = first unit of this ky's
// taps in the table row of output r (all equal when UNIFORM: one broadcast load per tap pair).
template <int L, bool UNIFORM, bool STAGED = false>
__device__ __forceinline__ void pdm3_pass(const float2 *__restrict__ base, const float4 *__restrict__ tb,
                                          const int (&toff)[8], float2 (&acc_a)[8], float2 (&acc_b)[8])
{
    constexpr int R = 8;
    float2 wl[R], wr[R];
    float4 tw[UNIFORM ? 1 : R];
#pragma unroll
    for (int i = 0; i < R / 2; ++i) {
        const float4 v = *reinterpret_cast<const float4 *>(base + 2 * i);
        wl[2 * i] = f4lo(v); wl[2 * i + 1] = f4hi(v);
        wr[2 * i] = f4lo(v); wr[2 * i + 1] = f4hi(v);
    }
#pragma unroll
    for (int r = 0; r < (UNIFORM ? 1 : R); ++r) tw[r] = STAGED ? tb[toff[r]] : __ldg(tb + toff[r]);
#pragma unroll
    for (int r = 0; r < R; ++r) {                          // kx = 0
        const float4 t = tw[UNIFORM ? 0 : r];
        acc_a[r] = pk_fma_s(wl[r].x, f4lo(t), acc_a[r]);
        acc_b[r] = pk_fma_s(wl[r].y, f4lo(t), acc_b[r]);
    }
    float4 lv = make_float4(0.f, 0.f, 0.f, 0.f), rv = lv;
#pragma unroll
    for (int k = 1; k <= L; ++k) {
        if (k & 1) {
            lv = *reinterpret_cast<const float4 *>(base + pdm_soff<R>(-k - 1));
            rv = *reinterpret_cast<const float4 *>(base + pdm_soff<R>(R + k - 1));
            wl[pdm_mod(-k, R)] = f4hi(lv);
            wr[pdm_mod(k - 1, R)] = f4lo(rv);
        } else {
            wl[pdm_mod(-k, R)] = f4lo(lv);
            wr[pdm_mod(k - 1, R)] = f4hi(rv);
        }
#pragma unroll
        for (int r = 0; r < (UNIFORM ? 1 : R); ++r) tw[r] = STAGED ? tb[toff[r] + k] : __ldg(tb + toff[r] + k);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float4 t = tw[UNIFORM ? 0 : r];
            const float2 a = wl[pdm_mod(r - k, R)];         // P(y-ky, x-kx): times W[ky][kx]
            const float2 b = wr[pdm_mod(r + k, R)];         // P(y-ky, x+kx): times W[ky][-kx]
            acc_a[r] = pk_fma_s(a.x, f4lo(t), acc_a[r]);
            acc_b[r] = pk_fma_s(a.y, f4lo(t), acc_b[r]);
            acc_a[r] = pk_fma_s(b.x, f4hi(t), acc_a[r]);
            acc_b[r] = pk_fma_s(b.y, f4hi(t), acc_b[r]);
        }
    }
}

// The same pass for operators that are bitwise symmetric in kx AND in ky (W[ky][kx] = W[-ky][kx] =
// W[ky][-kx]: circularly symmetric 2-D extrapolators): the rows y-ky and y+ky are added while their
// windows are loaded (TWO_ROWS; ky = 0 has one row) and the x-sum is folded as in the 1-D kernels,
//   acc += W[ky][0] S(x) + sum_{kx>=1} W[ky][kx] (S(x-kx) + S(x+kx)),   S = P(y-ky,.) + P(y+ky,.)
// 1 FADD2 + 2 FFMA2 per tap pair instead of 4 FFMA2, and L+1 passes instead of 2L+1.  Table units:
// (W[ky][2t], W[ky][2t+1]) pairs, t = 0..L/2, for ky = 0..L.
template <int L, bool UNIFORM, bool STAGED, bool TWO_ROWS>
__device__ __forceinline__ void pdm3_pass_sym(const float2 *__restrict__ base, const float2 *__restrict__ base2,
                                              const float4 *__restrict__ tb, const int (&toff)[8],
                                              float2 (&acc_a)[8], float2 (&acc_b)[8])
{
    constexpr int R = 8;
    float2 wl[R], wr[R];
    float4 tw[UNIFORM ? 1 : R];
    auto ld = [&](int off) {
        float4 v = *reinterpret_cast<const float4 *>(base + off);
        if (TWO_ROWS) {
            const float4 u = *reinterpret_cast<const float4 *>(base2 + off);
            const float2 a = pk_add(f4lo(v), f4lo(u)), b = pk_add(f4hi(v), f4hi(u));
            v = make_float4(a.x, a.y, b.x, b.y);
        }
        return v;
    };
#pragma unroll
    for (int i = 0; i < R / 2; ++i) {
        const float4 v = ld(2 * i);
        wl[2 * i] = f4lo(v); wl[2 * i + 1] = f4hi(v);
        wr[2 * i] = f4lo(v); wr[2 * i + 1] = f4hi(v);
    }
#pragma unroll
    for (int r = 0; r < (UNIFORM ? 1 : R); ++r) tw[r] = STAGED ? tb[toff[r]] : __ldg(tb + toff[r]);
#pragma unroll
    for (int r = 0; r < R; ++r) {                          // kx = 0
        const float4 t = tw[UNIFORM ? 0 : r];
        acc_a[r] = pk_fma_s(wl[r].x, f4lo(t), acc_a[r]);
        acc_b[r] = pk_fma_s(wl[r].y, f4lo(t), acc_b[r]);
    }
    float4 lv = make_float4(0.f, 0.f, 0.f, 0.f), rv = lv;
#pragma unroll
    for (int k = 1; k <= L; ++k) {
        if (k & 1) {
            lv = ld(pdm_soff<R>(-k - 1));
            rv = ld(pdm_soff<R>(R + k - 1));
            wl[pdm_mod(-k, R)] = f4hi(lv);
            wr[pdm_mod(k - 1, R)] = f4lo(rv);
        } else {
            wl[pdm_mod(-k, R)] = f4lo(lv);
            wr[pdm_mod(k - 1, R)] = f4hi(rv);
#pragma unroll
            for (int r = 0; r < (UNIFORM ? 1 : R); ++r) tw[r] = STAGED ? tb[toff[r] + k / 2] : __ldg(tb + toff[r] + k / 2);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float4 t = tw[UNIFORM ? 0 : r];
            const float2 W = (k & 1) ? f4hi(t) : f4lo(t);
            const float2 sm = pk_add(wl[pdm_mod(r - k, R)], wr[pdm_mod(r + k, R)]);
            acc_a[r] = pk_fma_s(sm.x, W, acc_a[r]);
            acc_b[r] = pk_fma_s(sm.y, W, acc_b[r]);
        }
    }
}

template <int L, int CH, bool SYM2 = false>
__global__ void __launch_bounds__(PDM3_THREADS, 2) pdm3_step(const pdm3_params p)
{
    constexpr int R = 8, GS = R + 2;
    constexpr int HG = pdm_halo_groups<L, R>();
    constexpr int NGX = PDM3_TX / R + 2 * HG;                    // groups per tile row incl. halo
    constexpr int NROW = PDM3_TY + 2 * L;                        // tile rows incl. halo
    constexpr int ROW_SLOTS = NGX * GS;
    constexpr int BUF_SLOTS = NROW * ROW_SLOTS;
    constexpr int KU = SYM2 ? (L + 2) / 2 : L + 1;                // float4 units per ky
    constexpr int UNITS = (SYM2 ? L + 1 : 2 * L + 1) * KU;       // float4 units per table row
    extern __shared__ __align__(16) unsigned char pdm_smem[];
    float2 *bufs = reinterpret_cast<float2 *>(pdm_smem);         // [2][NROW][NGX][GS]
    // plans whose model gives (nearly) every sample its own row: the rows this tile can touch at this
    // depth and frequency, [idx(w, q_min), idx(w, q_max)] with q over the tile, are staged per frequency
    // (odd row stride: consecutive rows in distinct bank groups); too many rows -> read through L1
    constexpr int UNITS_P = UNITS | 1;
    float4 *slice = reinterpret_cast<float4 *>(bufs + 2 * BUF_SLOTS);
    __shared__ float qred[2][PDM3_THREADS / 32];

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int tx0 = blockIdx.x * PDM3_TX, ty0 = blockIdx.y * PDM3_TY;
    const int y = ty0 + warp, x0 = tx0 + lane * R;
    const int w_begin = blockIdx.z * p.w_per_group;
    const int w_end = min(p.nw, w_begin + p.w_per_group);
    const int ntab_m1 = p.ntab - 1;
    const size_t slab = (size_t)p.ny * p.nx;

    auto issue_load = [&](int iw, int b) {
        const float2 *src = p.Pin + (size_t)iw * slab;
        float2 *dst = bufs + (size_t)b * BUF_SLOTS;
        constexpr int NCH = NGX * R / CH;                        // chunks per tile row
        for (int c = tid; c < NROW * NCH; c += PDM3_THREADS) {
            const int row = c / NCH, cc = c - row * NCH;
            const int s = cc * CH, g = s / R;
            const int yy = ty0 - L + row, xx = tx0 - HG * R + s;
            const bool valid = yy >= 0 && yy < p.ny && xx >= 0 && xx < p.nx;   // CH == 2: xx and nx are even
            pdm_cp_async<CH>(dst + row * ROW_SLOTS + g * GS + (s - g * R),
                             src + (valid ? (size_t)yy * p.nx + xx : 0), valid);
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    if (w_begin < w_end) issue_load(w_begin, 0);

    float qc[R];
    {
        const int yq = min(y, p.ny - 1), xq = min(x0, p.qstride - R);
        const float4 *qp = reinterpret_cast<const float4 *>(p.q + ((size_t)p.z * p.ny + yq) * p.qstride + xq);
        const float4 a = __ldg(qp), b = __ldg(qp + 1);
        qc[0] = a.x; qc[1] = a.y; qc[2] = a.z; qc[3] = a.w; qc[4] = b.x; qc[5] = b.y; qc[6] = b.z; qc[7] = b.w;
    }
    float img[R];
#pragma unroll
    for (int r = 0; r < R; ++r) img[r] = 0.f;
    const bool active = y < p.ny && x0 < p.nx;
    float tq_min = 0.f, tq_max = 0.f;
    if (p.slice_rows > 0) {                                // q extrema of the tile (block reduction, once)
        float lo = qc[0], hi = qc[0];
#pragma unroll
        for (int r = 1; r < R; ++r) { lo = fminf(lo, qc[r]); hi = fmaxf(hi, qc[r]); }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            lo = fminf(lo, __shfl_xor_sync(0xffffffffu, lo, o));
            hi = fmaxf(hi, __shfl_xor_sync(0xffffffffu, hi, o));
        }
        if (lane == 0) { qred[0][warp] = lo; qred[1][warp] = hi; }
        __syncthreads();
        tq_min = qred[0][0]; tq_max = qred[1][0];
#pragma unroll
        for (int i = 1; i < PDM3_THREADS / 32; ++i) { tq_min = fminf(tq_min, qred[0][i]); tq_max = fmaxf(tq_max, qred[1][i]); }
    }

    for (int iw = w_begin, it = 0; iw < w_end; ++iw, ++it) {
        const float w = p.omega[iw];
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();                                   // tile iw complete; everyone is done with tile iw-1
        if (iw + 1 < w_end) issue_load(iw + 1, (it + 1) & 1);

        int jidx[R], toff[R];
        bool un = true;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            jidx[r] = pdm_index(w, qc[r], ntab_m1);
            toff[r] = jidx[r] * UNITS;
            un = un && (jidx[r] == jidx[0]);
        }
        const bool uni = __all_sync(0xffffffffu, un && !p.force_general);
        bool staged = false;
        if (p.slice_rows > 0) {                            // CTA-uniform decisions
            const int jlo = pdm_index(w, tq_min, ntab_m1), jhi = pdm_index(w, tq_max, ntab_m1);
            staged = jhi > jlo && jhi - jlo + 1 <= p.slice_rows;
            if (staged) {
                const int nrows = jhi - jlo + 1;
                for (int e = tid; e < nrows * UNITS; e += PDM3_THREADS) {
                    const int rr = e / UNITS, u = e - rr * UNITS;
                    slice[rr * UNITS_P + u] = __ldg(p.tab + (size_t)(jlo + rr) * UNITS + u);
                }
#pragma unroll
                for (int r = 0; r < R; ++r) toff[r] = (jidx[r] - jlo) * UNITS_P;
            }
            __syncthreads();                               // slice complete (or nobody staged: still uniform)
        }
        const float2 *tile = bufs + (size_t)(it & 1) * BUF_SLOTS;
        float2 acc_a[R], acc_b[R];
#pragma unroll
        for (int r = 0; r < R; ++r) { acc_a[r] = make_float2(0.f, 0.f); acc_b[r] = make_float2(0.f, 0.f); }

        // one 1-D pass per ky (row y-ky, taps W[ky][.]); short operators: all 2L+1 passes unrolled
#define PDM3_PASSES(UNI, ST, TB)                                                                     \
        if (SYM2) {                                                                                     \
            pdm3_pass_sym<L, UNI, ST, false>(tile + (warp + L) * ROW_SLOTS + (HG + lane) * GS, nullptr, \
                                             (TB), toff, acc_a, acc_b);                                 \
            _Pragma("unroll (L <= 3 ? L : 1)")                                                          \
            for (int ky = 1; ky <= L; ++ky)                                                             \
                pdm3_pass_sym<L, UNI, ST, true>(tile + (warp + L - ky) * ROW_SLOTS + (HG + lane) * GS,  \
                                                tile + (warp + L + ky) * ROW_SLOTS + (HG + lane) * GS,  \
                                                (TB) + ky * KU, toff, acc_a, acc_b);                    \
        } else {                                                                                        \
            _Pragma("unroll (L <= 3 ? 2 * L + 1 : 1)")                                                  \
            for (int ky = -L; ky <= L; ++ky)                                                            \
                pdm3_pass<L, UNI, ST>(tile + (warp + L - ky) * ROW_SLOTS + (HG + lane) * GS,           \
                                      (TB) + (ky + L) * (L + 1), toff, acc_a, acc_b);                   \
        }
        if (staged) {
            if (uni) { PDM3_PASSES(true, true, slice) } else { PDM3_PASSES(false, true, slice) }
        } else {
            if (uni) { PDM3_PASSES(true, false, p.tab) } else { PDM3_PASSES(false, false, p.tab) }
        }
#undef PDM3_PASSES
        if (active) {
            float2 out[R];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                out[r] = make_float2(acc_a[r].x - acc_b[r].y, acc_a[r].y + acc_b[r].x);
                img[r] += out[r].x;                        // A5: fixed (increasing w) order
            }
            float2 *dst = p.Pout + (size_t)iw * slab + (size_t)y * p.nx + x0;
            if (CH == 2 && x0 + R <= p.nx) {
#pragma unroll
                for (int i = 0; i < R / 2; ++i)
                    __stcg(reinterpret_cast<float4 *>(dst) + i, make_float4(out[2 * i].x, out[2 * i].y, out[2 * i + 1].x, out[2 * i + 1].y));
            } else {
#pragma unroll
                for (int r = 0; r < R; ++r)
                    if (x0 + r < p.nx) dst[r] = out[r];
            }
        }
    }
    if (w_begin < w_end && active) {
        float *prow = p.partial + (((size_t)blockIdx.z * p.nz + p.z) * p.ny + y) * p.pstride + x0;
        *reinterpret_cast<float4 *>(prow) = make_float4(img[0], img[1], img[2], img[3]);
        *reinterpret_cast<float4 *>(prow + 4) = make_float4(img[4], img[5], img[6], img[7]);
    }
}

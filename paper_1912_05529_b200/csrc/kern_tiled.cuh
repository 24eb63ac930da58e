// kern_tiled.cuh -- PDM_PATH_TILED: x-tiled per-depth-step kernel with
// +-L halos for lines too long for shared memory (BASELINE.json configs[4], nx = 32768).
// Closest to what the paper itself did (planes in global memory, one grid-wide
// synchronisation per depth level = one launch per level), but:
//   * one resident wave of CTAs per launch; a CTA owns an x-tile and walks a GROUP of frequencies,
//     so the q tile is read once and Re P is summed over the group in registers in fixed order
//     (the paper's K2 disappears into a small fixed-order reduction over the groups);
//   * every WARP runs its own pipeline over its 32 x R samples of the tile: the sub-tile + halo of
//     the NEXT frequency is copied global -> shared memory with cp.async while the current one is
//     computed (double buffer per warp), zero-filled outside [0,nx) (R5); only __syncwarp inside
//     the frequency loop, so the 16 warps of an SM drift apart and loads, FMAs and stores overlap
//     (halo groups are fetched by both neighbouring warps: L2 hits, not HBM traffic);
//   * the arithmetic is the same register-tiled folded FIR as the main path (pdm_fir_group);
//   * results go through a shared-memory tile so that the plane is written in full 512-byte
//     warp transactions.
// HBM traffic: 8 B read + 8 B written per sample (+ halo 2*HG*R/tile_x), planes ping-pong.
#pragma once
#include "pdm_common.cuh"
#include "kern_march.cuh"

#define PDM_TILED_THREADS 256
#ifndef PDM_TILED_STAGES
#define PDM_TILED_STAGES 2      // input sub-tiles per warp (cp.async ring): STAGES-1 in flight; 3 measured 4-8 % slower
#endif

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
    int force_general;       // PDM_FORCE_GENERAL (debug)
};

// CH = samples per async-copy chunk: 2 (16-byte copies; needs nx even and 16-byte aligned planes)
// or 1 (8-byte copies, any nx).
template <int CH>
__device__ __forceinline__ void pdm_cp_async(float2 *dst_smem, const float2 *src, bool valid)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst_smem);
    const unsigned n = valid ? 8u * CH : 0u;              // src-size 0: the chunk is zero-filled
    if (CH == 2) asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" :: "r"(d), "l"(src), "r"(n) : "memory");
    else         asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" :: "r"(d), "l"(src), "r"(n) : "memory");
}

template <int L, int R, int CH, bool ALIAS, bool SYM = true>
__global__ void __launch_bounds__(PDM_TILED_THREADS, 2) pdm_tiled_step(const pdm_tiled_params p)
{
    constexpr int HG = pdm_halo_groups<L, R>();
    constexpr int GS = R + 2;
    constexpr int T = PDM_TILED_THREADS;
    constexpr int IN_SLOTS = (32 + 2 * HG) * GS;                  // per warp and buffer
    // two input buffers + an output tile; with ALIAS the consumed input buffer holds the results
    constexpr int NB = PDM_TILED_STAGES;
    constexpr int WARP_SLOTS = NB * IN_SLOTS + (ALIAS ? 0 : 32 * GS);
    extern __shared__ __align__(16) unsigned char pdm_smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    float2 *ibuf = reinterpret_cast<float2 *>(pdm_smem) + warp * WARP_SLOTS;   // [2][IN_SLOTS]

    const int tile_x0 = blockIdx.x * T * R + warp * 32 * R;       // this warp's first sample
    const int x0 = tile_x0 + lane * R;
    const int ntab_m1 = p.ntab - 1;
    const int w_begin = blockIdx.y * p.w_per_group;
    const int w_end = min(p.nw, w_begin + p.w_per_group);

    auto issue_load = [&](int iw, int b) {
        const float2 *src = p.Pin + (size_t)iw * p.nx;
        float2 *dst = ibuf + b * IN_SLOTS;
        constexpr int NCH = (32 + 2 * HG) * R / CH;
        for (int c = lane; c < NCH; c += 32) {
            const int s = c * CH, g = s / R;
            const int x = tile_x0 - HG * R + s;
            const bool valid = x >= 0 && x < p.nx;             // CH == 2: x and nx are even
            pdm_cp_async<CH>(dst + g * GS + (s - g * R), src + (valid ? x : 0), valid);
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

#pragma unroll
    for (int i = 0; i < NB - 1; ++i)
        if (w_begin + i < w_end) issue_load(w_begin + i, i);

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

    for (int iw = w_begin, it = 0; iw < w_end; ++iw, ++it) {
        const int b = it % NB;
        const float w = p.omega[iw];
        // the warp is past the compute of iteration it-1 (__syncwarp before its copy-out), so the
        // buffer it read, (it-1) % NB, may be refilled now (with the tile NB-1 frequencies ahead)
        if (iw + NB - 1 < w_end) issue_load(iw + NB - 1, (it + NB - 1) % NB);
        {                                                  // groups committed after tile iw's
            const int ahead = min(NB - 1, w_end - 1 - iw);
            if (ahead >= 2)      asm volatile("cp.async.wait_group 2;" ::: "memory");
            else if (ahead == 1) asm volatile("cp.async.wait_group 1;" ::: "memory");
            else                 asm volatile("cp.async.wait_group 0;" ::: "memory");
        }
        __syncwarp();                                      // tile of iw complete; obuf of it-1 drained

        int j[R], toff[R];
        bool uni = true;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            j[r] = pdm_index(w, qc[r], ntab_m1);
            uni = uni && (j[r] == j[0]);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) toff[r] = j[r] * p.half16;
        const float2 *base = ibuf + b * IN_SLOTS + (HG + lane) * GS;
        float2 out[R];
        const bool wuni = __all_sync(0xffffffffu, uni && !p.force_general);
        if (SYM) {
            if (wuni) pdm_fir_group<L, R, true, false>(base, p.half, toff, out);
            else      pdm_fir_group<L, R, false, false>(base, p.half, toff, out);
        } else {
            if (wuni) pdm_fir_group_asym<L, R, true>(base, p.half, toff, out);
            else      pdm_fir_group_asym<L, R, false>(base, p.half, toff, out);
        }

        // ALIAS (plans with long, per-sample table rows): the consumed input buffer doubles as the
        // output tile -- less shared memory leaves more L1 for the tap rows (+11..24 % at 51 taps on
        // random-field models, -7 % where rows are warp-uniform, hence a per-plan choice); every
        // lane must be done reading its windows before anyone overwrites them
        float2 *obuf = ALIAS ? ibuf + b * IN_SLOTS + HG * GS : ibuf + NB * IN_SLOTS;
        if (ALIAS) __syncwarp();
        float2 *od = obuf + lane * GS;
#pragma unroll
        for (int i = 0; i < R / 2; ++i)
            *reinterpret_cast<float4 *>(od + 2 * i) = make_float4(out[2 * i].x, out[2 * i].y, out[2 * i + 1].x, out[2 * i + 1].y);
#pragma unroll
        for (int r = 0; r < R; ++r) img[r] += out[r].x;   // A5: fixed (increasing w) order
        __syncwarp();                                      // obuf complete; ibuf[b] no longer read

        float2 *dst = p.Pout + (size_t)iw * p.nx;
        constexpr int NCH = 32 * R / CH;
#pragma unroll
        for (int c = lane; c < NCH; c += 32) {             // full-width warp stores
            const int s = c * CH, g = s / R;
            const int x = tile_x0 + s;
            if (x < p.nx) {
                const float2 *sp = obuf + g * GS + (s - g * R);
                if (CH == 2) *reinterpret_cast<float4 *>(dst + x) = *reinterpret_cast<const float4 *>(sp);
                else         dst[x] = *sp;
            }
        }
        // ALIAS: the output tile lives in input buffer b, which the NEXT iteration refills with
        // cp.async right away -- every lane must have copied its part out first
        if (ALIAS) __syncwarp();
    }
    if (w_begin < w_end && x0 < p.pstride) {
        float *prow = p.partial + ((size_t)blockIdx.y * p.nz + p.z) * p.pstride + x0;
#pragma unroll
        for (int i = 0; i < R / 4; ++i)
            *reinterpret_cast<float4 *>(prow + 4 * i) = make_float4(img[4 * i], img[4 * i + 1], img[4 * i + 2], img[4 * i + 3]);
    }
}

// ------------------------------------------------------------------------------------------------
// Two depth steps per launch (SURVEY.md 8(f) N2 at warp granularity): the same per-warp
// pipeline, but a warp keeps its sub-tile on chip for steps z and z+1.  Step 1 computes all 32 groups
// of the fetched sub-tile (its +-HG halo groups are real data) into a warp-private scratch tile;
// step 2 is exact on the 32 - 2*HG central groups, which are the warp's outputs.  Planes cross HBM
// once per two steps: 8 B + 8 B*(32+2HG)/(32-2HG) per sample and 2 steps instead of 32 B.  Used for
// short filters (HG <= 2) on warp-uniform models, where the one-step kernel is HBM-bound.
template <int L, int R, int CH, bool SYM = true>
__global__ void __launch_bounds__(PDM_TILED_THREADS, 2) pdm_tiled_step2(const pdm_tiled_params p)
{
    constexpr int HG = pdm_halo_groups<L, R>();
    constexpr int GS = R + 2;
    constexpr int T = PDM_TILED_THREADS;
    constexpr int KEEP = 32 - 2 * HG;                              // output groups per warp
    constexpr int IN_SLOTS = (32 + 2 * HG) * GS;                  // per warp: fetched sub-tile; scratch tile
    constexpr int NB = PDM_TILED_STAGES;
    constexpr int WARP_SLOTS = (NB + 1) * IN_SLOTS + 32 * GS;     // input ring, scratch (with zero pads), output
    extern __shared__ __align__(16) unsigned char pdm_smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    float2 *ibuf = reinterpret_cast<float2 *>(pdm_smem) + warp * WARP_SLOTS;
    float2 *sbuf = ibuf + NB * IN_SLOTS;                           // [HG pad | 32 groups | HG pad]
    float2 *obuf = sbuf + IN_SLOTS;

    // first computed group of the warp sits HG groups left of its first output
    const int tile_x0 = (blockIdx.x * (T / 32) + warp) * KEEP * R - HG * R;
    const int x0 = tile_x0 + lane * R;
    const int ntab_m1 = p.ntab - 1;
    const int w_begin = blockIdx.y * p.w_per_group;
    const int w_end = min(p.nw, w_begin + p.w_per_group);
    const bool keep = lane >= HG && lane < 32 - HG;

    for (int i = lane; i < IN_SLOTS / 2; i += 32)                  // scratch pads stay zero
        reinterpret_cast<float4 *>(sbuf)[i] = make_float4(0.f, 0.f, 0.f, 0.f);

    auto issue_load = [&](int iw, int b) {
        const float2 *src = p.Pin + (size_t)iw * p.nx;
        float2 *dst = ibuf + b * IN_SLOTS;
        constexpr int NCH = (32 + 2 * HG) * R / CH;
        for (int c = lane; c < NCH; c += 32) {
            const int s = c * CH, g = s / R;
            const int x = tile_x0 - HG * R + s;
            const bool valid = x >= 0 && x < p.nx;
            pdm_cp_async<CH>(dst + g * GS + (s - g * R), src + (valid ? x : 0), valid);
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
#pragma unroll
    for (int i = 0; i < NB - 1; ++i)
        if (w_begin + i < w_end) issue_load(w_begin + i, i);

    float qa[R], qb[R];                                            // q of steps z and z+1
    {
        const int xq = min(max(x0, 0), p.qstride - R);
        const float4 *q1 = reinterpret_cast<const float4 *>(p.q + (size_t)p.z * p.qstride + xq);
        const float4 *q2 = reinterpret_cast<const float4 *>(p.q + (size_t)(p.z + 1) * p.qstride + xq);
#pragma unroll
        for (int i = 0; i < R / 4; ++i) {
            const float4 v = __ldg(q1 + i), u = __ldg(q2 + i);
            qa[4 * i] = v.x; qa[4 * i + 1] = v.y; qa[4 * i + 2] = v.z; qa[4 * i + 3] = v.w;
            qb[4 * i] = u.x; qb[4 * i + 1] = u.y; qb[4 * i + 2] = u.z; qb[4 * i + 3] = u.w;
        }
    }
    float img1[R], img2[R];
#pragma unroll
    for (int r = 0; r < R; ++r) { img1[r] = 0.f; img2[r] = 0.f; }
    __syncwarp();

    for (int iw = w_begin, it = 0; iw < w_end; ++iw, ++it) {
        const int b = it % NB;
        const float w = p.omega[iw];
        if (iw + NB - 1 < w_end) issue_load(iw + NB - 1, (it + NB - 1) % NB);
        {
            const int ahead = min(NB - 1, w_end - 1 - iw);
            if (ahead >= 2)      asm volatile("cp.async.wait_group 2;" ::: "memory");
            else if (ahead == 1) asm volatile("cp.async.wait_group 1;" ::: "memory");
            else                 asm volatile("cp.async.wait_group 0;" ::: "memory");
        }
        __syncwarp();                                      // tile of iw complete; scratch / obuf of it-1 drained

        float2 out[R];
        int toff[R];
        bool uni;
        // ---- step z: all 32 groups of the fetched sub-tile -> scratch
        uni = true;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            toff[r] = pdm_index(w, qa[r], ntab_m1) * p.half16;
            uni = uni && (toff[r] == toff[0]);
        }
        {
            const float2 *base = ibuf + b * IN_SLOTS + (HG + lane) * GS;
            const bool wuni = __all_sync(0xffffffffu, uni && !p.force_general);
            if (SYM) {
                if (wuni) pdm_fir_group<L, R, true, false>(base, p.half, toff, out);
                else      pdm_fir_group<L, R, false, false>(base, p.half, toff, out);
            } else {
                if (wuni) pdm_fir_group_asym<L, R, true>(base, p.half, toff, out);
                else      pdm_fir_group_asym<L, R, false>(base, p.half, toff, out);
            }
        }
        if (x0 < 0 || x0 + R > p.nx) {                     // R5: zero outside [0,nx) before the next step reads it
#pragma unroll
            for (int r = 0; r < R; ++r)
                if ((unsigned)(x0 + r) >= (unsigned)p.nx) out[r] = make_float2(0.f, 0.f);
        }
        {
            float2 *sd = sbuf + (HG + lane) * GS;
#pragma unroll
            for (int i = 0; i < R / 2; ++i)
                *reinterpret_cast<float4 *>(sd + 2 * i) = make_float4(out[2 * i].x, out[2 * i].y, out[2 * i + 1].x, out[2 * i + 1].y);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) img1[r] += out[r].x;  // A5 row z (kept lanes only are stored)
        __syncwarp();                                      // scratch complete; ibuf[b] no longer read

        // ---- step z+1: exact on the central groups
        uni = true;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            toff[r] = pdm_index(w, qb[r], ntab_m1) * p.half16;
            uni = uni && (toff[r] == toff[0]);
        }
        {
            const float2 *base = sbuf + (HG + lane) * GS;
            const bool wuni = __all_sync(0xffffffffu, uni && !p.force_general);
            if (SYM) {
                if (wuni) pdm_fir_group<L, R, true, false>(base, p.half, toff, out);
                else      pdm_fir_group<L, R, false, false>(base, p.half, toff, out);
            } else {
                if (wuni) pdm_fir_group_asym<L, R, true>(base, p.half, toff, out);
                else      pdm_fir_group_asym<L, R, false>(base, p.half, toff, out);
            }
        }
        float2 *od = obuf + lane * GS;
#pragma unroll
        for (int i = 0; i < R / 2; ++i)
            *reinterpret_cast<float4 *>(od + 2 * i) = make_float4(out[2 * i].x, out[2 * i].y, out[2 * i + 1].x, out[2 * i + 1].y);
#pragma unroll
        for (int r = 0; r < R; ++r) img2[r] += out[r].x;  // A5 row z+1
        __syncwarp();                                      // obuf complete; scratch no longer read

        float2 *dst = p.Pout + (size_t)iw * p.nx;
        constexpr int NCH = KEEP * R / CH;
#pragma unroll
        for (int c = lane; c < NCH; c += 32) {             // the warp's KEEP central groups, full-width stores
            const int s = HG * R + c * CH, g = s / R;
            const int x = tile_x0 + s;
            if (x < p.nx) {                                // (x >= 0: central groups start at the tile's first output)
                const float2 *sp = obuf + g * GS + (s - g * R);
                if (CH == 2) *reinterpret_cast<float4 *>(dst + x) = *reinterpret_cast<const float4 *>(sp);
                else         dst[x] = *sp;
            }
        }
    }
    if (w_begin < w_end && keep && x0 >= 0 && x0 < p.pstride) {
        float *prow = p.partial + ((size_t)blockIdx.y * p.nz + p.z) * p.pstride + x0;
#pragma unroll
        for (int i = 0; i < R / 4; ++i) {
            *reinterpret_cast<float4 *>(prow + 4 * i) = make_float4(img1[4 * i], img1[4 * i + 1], img1[4 * i + 2], img1[4 * i + 3]);
            *reinterpret_cast<float4 *>(prow + p.pstride + 4 * i) = make_float4(img2[4 * i], img2[4 * i + 1], img2[4 * i + 2], img2[4 * i + 3]);
        }
    }
}

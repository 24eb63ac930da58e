// pdm_common.cuh -- plan layout and small device helpers shared by the kernels of libpdm.
// Product code: csrc/ shares nothing with the CPU checker (test infrastructure) of this repo.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/pdm.h"

#define PDM_HALF_ALIGN 2   // half-table rows are padded to an ODD number of 16-byte units (bank spread)

struct pdm_plan {
    int nx, nz, nw, ntab, ntaps, L;
    int Lk;               // half-length of the unrolled kernel instantiation used (>= L; taps beyond L are zero)
    float dx, dz;
    double du;
    unsigned flags;
    int path, taps_mode;
    int ntaper;           // R5b edge taper width (packed form only)
    float *d_taper;       // [ntaper]
    int prestack;         // PDM_PRESTACK: nw counts LINES = 2 x the caller's frequencies ((receiver, conj source) pairs)
    int sym;              // 1: table bitwise symmetric in k (folded kernels); 0: general kernels (8L+4 lane-ops)
    int device, sm_count, smem_optin;
    int last_cuda_error;

    // ---- data-independent device state (pdm_create) -------------------------------------------
    float  *d_omega;      // [nw]
    float  *d_q;          // [nz][qstride]  q32 = fl32(dz/(v*du)) (R3); columns >= nx repeat the last q
    int     qstride;      // row stride of d_q (multiple of 32 floats)
    float2 *d_table;      // full table [ntab][ntaps] (naive path only reads this)
    cudaTextureObject_t tex_half;   // d_half as a linear float4 texture (tap gather through the texture unit)
    float4 *d_half;       // half table rows k=0..L as (W_k, W_{k+1}) pairs, [ntab][half16] float4
    int     half16;       // float4 per row, odd
    int    *d_rowoff;     // [nw+1] offsets into d_rows
    int    *d_rows;       // per-omega list of table rows that omega can touch (compact or contiguous)
    int     max_rows;     // longest per-omega list
    int     contiguous_rows;  // 1: lists are the full ranges [jmin, jmax]; 0: compact (few distinct q)

    // ---- workspace -----------------------------------------------------------------------------
    float  *d_partial;    // march: [n_partial][nz][nx] per-CTA partial images; tiled: [wgroups][nz][nx]
    int     n_partial;
    float2 *d_plane[2];   // tiled/naive: HBM ping-pong planes [nw][nx]
    int    *d_flags;      // march: depth-split hand-off flags [nslots]
    float2 *d_handoff;    // march: [nslots][nx] wavefield of a split line at its split depth
    int4   *d_segs;       // march: work list {line, z0, z1, slot}, execution order per CTA
    int    *d_segoff;     // march: [grid+1]
    int     nslots, balanced;

    // ---- pdm_migrate_host staging --------------------------------------------------------------
    pdm_c64 *d_stage_p0;
    float   *d_stage_img;

    // ---- pdm_profile_enable: events around the dominant kernel(s) and the reduction -----------------
    int profiling, profiled;
    cudaEvent_t ev[3];

    // ---- launch configuration ------------------------------------------------------------------
    int R;                // outputs per thread of the register-tiled kernels
    int threads, grid, ctas_per_sm, smem_bytes, launches;
    int tile_x, wgroups;  // tiled path
    int tiled_T2, tile_x2, smem_bytes2;   // tiled path: two depth steps per launch (pdm_tiled_step2), its x-tile and smem
    int cluster_size, cluster_gper, cluster_passes;   // cluster path: CTAs per line, groups per CTA, passes per step
    int taps_in_smem;     // march: 1 = per-omega rows staged in shared memory, 0 = L1/L2 global rows
    // packed path (kern_pack.cuh): planes [nw][nxp] ping-pong, T depth steps per tile visit
    int nxp, pk_T, pk_TX, pk_H, pk_LS, pk_BW, pk_nbox, pk_cap, pk_passes, pk_npacks, pk_ntiles;
    int pk_gtaps;         // 1: tap rows read from the global table (a pack's row range exceeds every slice buffer)
    float2 *d_packw;      // [npacks] lowest / highest omega of a pack
    float2 *d_tileq;      // [nblocks][ntiles] min / max q over the samples a tile visit computes
    int2 *d_tile_ctas;    // [ntiles] first / last CTA that holds a piece of the tile's image
    CUtensorMap tmap_plane[2];   // TMA descriptors of d_plane[0], d_plane[1]
    double workspace_bytes;
};

// R3 index rule, device side: FLOAT product, round half to even, clamp.
__device__ __forceinline__ int pdm_index(float w, float q, int ntab_m1)
{
    int j = __float2int_rn(__fmul_rn(w, q));
    return min(max(j, 0), ntab_m1);
}

// ---- packed FP32 (sm_100a FFMA2 / FADD2): one instruction, two lanes of a 64-bit register pair ----
__device__ __forceinline__ float2 pk_fma(float2 a, float2 b, float2 c)
{
    float2 d;
    asm("{ .reg .b64 ra, rb, rc, rd;\n\t"
        "mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; mov.b64 rc, {%6,%7};\n\t"
        "fma.rn.f32x2 rd, ra, rb, rc;\n\t"
        "mov.b64 {%0,%1}, rd; }"
        : "=f"(d.x), "=f"(d.y)
        : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y), "f"(c.x), "f"(c.y));
    return d;
}
__device__ __forceinline__ float2 pk_add(float2 a, float2 b)
{
    float2 d;
    asm("{ .reg .b64 ra, rb, rd;\n\t"
        "mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5};\n\t"
        "add.rn.f32x2 rd, ra, rb;\n\t"
        "mov.b64 {%0,%1}, rd; }"
        : "=f"(d.x), "=f"(d.y)
        : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return d;
}
__device__ __forceinline__ float2 pk_mul(float2 a, float2 b)
{
    float2 d;
    asm("{ .reg .b64 ra, rb, rd;\n\t"
        "mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5};\n\t"
        "mul.rn.f32x2 rd, ra, rb;\n\t"
        "mov.b64 {%0,%1}, rd; }"
        : "=f"(d.x), "=f"(d.y)
        : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return d;
}
// scalar-broadcast forms: ptxas folds the {s,s} pair into the FFMA2 ".F32" operand (no MOV)
__device__ __forceinline__ float2 pk_fma_s(float s, float2 b, float2 c) { return pk_fma(make_float2(s, s), b, c); }
__device__ __forceinline__ float2 pk_mul_s(float s, float2 b) { return pk_mul(make_float2(s, s), b); }

// kern_pack.cuh -- PDM_PATH_PACKED: x-tiled, TEMPORALLY BLOCKED, FREQUENCY-PACKED form of the hot path
// (SURVEY.md 8(f) N2; PAPER.md:151 "block level synchronization ... some other alternative", :85).
//
// Why it exists.  Where every output sample has its own table row ("filter cutoffs may
// vary for each point": BASELINE.json configs[2], [4]) the other forms are bound by the tap gather:
// the 8 lanes of a quarter warp own x-blocks 8 samples apart, their rows fall in unrelated 16-byte
// bank groups and every LDS.128 of taps costs 2.1-2.4 shared-memory wavefronts instead of 1.  Here a
// quarter warp holds the SAME x-block of 8 ADJACENT FREQUENCIES (a "pack"): idx = rint(w*q) then moves
// by dw*q <= 1 row from lane to lane (for frequency lists at least as dense as the table), the half
// table has an odd number of 16-byte units per row, so 8 consecutive rows sit in 8 distinct bank
// groups and equal rows are a broadcast: the gather is conflict-free by construction.
//
// Work item = (x-tile, pack of 8 lines, block of T depth steps).  Per item the CTA
//   * receives the 8 line tiles (+ halo) by TMA (cp.async.bulk.tensor.2d, one 1-row box per line and
//     256-sample chunk, out-of-range samples and lines zero-filled by the copy engine = R5), line l
//     shifted by 2*l samples so that equal x of the 8 lines falls in 8 distinct bank groups; the load
//     of item i+1 is in flight while item i is computed (three line buffers: loaded / scratch / next);
//   * marches T depth steps in shared memory (ping-pong between the loaded and the scratch buffer)
//     with the same register-tiled folded FIR as the other forms (pdm_fir_group); the halo of
//     (T-1)*L + 8*HG samples per side absorbs the steps' dependence on neighbouring tiles, so planes
//     cross HBM once per T steps: 16/T bytes per sample and step instead of 16;
//   * sums Re P over the pack with a 3-stage transposing butterfly (7 SHFL) and accumulates the image
//     tile of its run of packs in shared memory; the last step's samples go from registers to the
//     output plane.
// ONE cooperative launch per migration: a CTA owns the same (tile, pack) items in every depth block;
// blocks are separated by a grid-wide barrier (the paper used kernel exit), after
// which the CTAs sum the image tiles of the block in fixed CTA order (deterministic) into the image.
// Prestack mode (xcorr, reading R17): the lines are (receiver, conjugated source) pairs of one
// frequency and the imaging condition is the zero-lag cross-correlation of the pair.
#pragma once
#include <cuda.h>
#include "pdm_common.cuh"
#include "kern_march.cuh"

#define PDM_PACK_W 8              // lines per pack = lanes of a quarter warp
#define PDM_PACK_THREADS 512      // default CTA size (also built: 384, 256)
#define PDM_PACK_NBUF 3

struct alignas(64) pdm_pack_params {
    CUtensorMap   tmap_p0;        // the caller's P0 (first depth block, when its rows are 16-byte aligned)
    CUtensorMap   tmap_plane[2];  // the plan's ping-pong planes: {x, line} of 8-byte samples, box {BW, 1}
    float2       *plane[2];       // [nw][nxp]
    float        *partial;        // [2][grid][T][nxp] image tiles per CTA, double-buffered over depth blocks
    float        *image;          // [nz][nx]
    const float  *q;              // [nz][qstride]
    const float  *omega;          // [nw]
    const float4 *half;           // [ntab][half16]
    const float2 *packw;          // [npacks] {lowest, highest} omega of the pack
    const float2 *tileq;          // [nblocks][ntiles] {min, max} q over the samples a tile visit computes
    const int2   *tile_ctas;      // [ntiles] first / last CTA holding a piece of the tile's image
    unsigned     *gbar;           // grid barrier counter (zeroed on the stream before the launch)
    int first_src;                // -1: block 0 reads P0 through tmap_p0; 1: P0 was repacked into plane[1]
    int nx, nxp, nz, nw, ntab, qstride, half16;
    int npacks, ntiles, nitems;
    int TX, H, T;                 // outputs per tile, recomputed halo per side, depth steps per block
    int LS, BW, nbox;             // line stride (samples), TMA box width, boxes per line
    int cap;                      // table rows the slice buffer holds
    int passes;                   // groups per thread and step
    int force_general;
    int xcorr;                    // prestack: lines 2i / 2i+1 are the receiver field and the conjugated source field of
                                  // frequency i; the image is sum Re(U R) over the pairs instead of sum Re P (R17)
    int accumulate;               // add to the image instead of overwriting it (several shots)
    int ntaper;                   // R5b: absorbing edge taper over this many samples per side (0: plain R5)
    const float *taper;           // [ntaper] t(d) = sin^2((pi/2)(d+1)/(ntaper+1)), d = distance to the nearer edge
};

__device__ __forceinline__ unsigned pdm_smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void pdm_mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void pdm_mbar_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void pdm_mbar_wait(unsigned bar, unsigned parity)
{
    asm volatile("{\n\t.reg .pred p;\n"
                 "PDM_WAIT_%=:\n\t"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
                 "@p bra PDM_DONE_%=;\n\t"
                 "bra PDM_WAIT_%=;\n"
                 "PDM_DONE_%=:\n\t}" :: "r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void pdm_tma_load_2d(unsigned dst, const CUtensorMap *map, int c0, int c1, unsigned bar)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 :: "r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar) : "memory");
}

// NTHREADS = CTA size the instantiation is compiled for (512: 128 registers per thread; 384: 168; 256: 255)
// GTAPS = true: tap rows are never staged; every fetch reads the global half table (L1/L2).  The plan
// takes this build (256 threads only) when one pack's row range on some tile visit is wider than any
// slice buffer -- strongly varying velocity inside a tile at the top frequencies, e.g. a salt flank or
// a model with independent samples and a 1024-row table -- so that PDM_PRESTACK / PDM_TAPER / forced
// PDM_PATH_PACKED plans exist for ANY table and model ("filter cutoffs may vary for each point").
template <int L, bool SYM, int NTHREADS, bool GTAPS = false>
__global__ void __launch_bounds__(NTHREADS, 1) pdm_pack_kernel(const __grid_constant__ pdm_pack_params p)
{
    constexpr int R = 8, W = PDM_PACK_W;
    constexpr int HG = pdm_halo_groups<L, R>();
    constexpr int MAXW = NTHREADS / 32;
    extern __shared__ __align__(128) unsigned char pdm_pack_smem[];
    __shared__ __align__(8) unsigned long long mbar[2];
    // A4 without a CTA barrier (as in kern_march.cuh): prog[1 + w] = depth steps warp w has completed
    // since the kernel started, counted THROUGH items and depth blocks.  A warp owns 4*passes contiguous
    // groups (32*passes samples >= the filter half-length), so step s+1 of warp w reads only what warps
    // w-1, w, w+1 wrote in step s and may start as soon as both neighbours have completed step s;
    // that also orders the overwrite of the ping-pong buffer.  prog[0], prog[nwarps+1]: sentinels.
    __shared__ int prog[MAXW + 2];
    __shared__ int buf_done[2];                          // per loaded buffer: warps x items that are done with it

    const int tid = threadIdx.x, NT = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarps = NT >> 5;
    const int l = lane & 7;                              // line of the pack this lane works on
    // this CTA's items of EVERY depth block (tile-major list, pack fastest): the same (tile, pack) pairs
    // each time, so staged table rows survive from block to block when they all fit
    const int i0 = (int)((long long)p.nitems * blockIdx.x / gridDim.x);
    const int i1 = (int)((long long)p.nitems * (blockIdx.x + 1) / gridDim.x);
    const int nmine = i1 - i0;

    unsigned char *sm = pdm_pack_smem + ((128u - (pdm_smem_u32(pdm_pack_smem) & 127u)) & 127u);
    const int buf_samples = W * p.LS;
    float2 *const bufs = reinterpret_cast<float2 *>(sm);
    float4 *const slice = reinterpret_cast<float4 *>(bufs + PDM_PACK_NBUF * buf_samples);
    float  *const img = reinterpret_cast<float *>(slice + (size_t)p.cap * p.half16);

    for (int i = tid; i < PDM_PACK_NBUF * buf_samples / 2; i += NT)       // pads stay finite (zero)
        reinterpret_cast<float4 *>(bufs)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (tid < nwarps + 2) prog[tid] = (tid == 0 || tid == nwarps + 1) ? 0x7fffffff : 0;
    if (tid == 0) {
        buf_done[0] = 0; buf_done[1] = 0;
        pdm_mbar_init(pdm_smem_u32(&mbar[0]), 1);
        pdm_mbar_init(pdm_smem_u32(&mbar[1]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int ntab_m1 = p.ntab - 1;
    const int gc0 = p.H / R, gc1 = gc0 + p.TX / R;       // groups whose outputs belong to this tile
    const int nblocks = (p.nz + p.T - 1) / p.T;
    int st_tile = -1, st_blk = -1, st_lo = 0, st_hi = -1, jlo = 0;   // staged: packs [st_lo, st_hi] of (st_blk, st_tile), first row
    int gs = 0;                                          // depth steps this warp has completed
    int use0 = 0, use1 = 0;                              // loads each line buffer has received in earlier blocks

    for (int blk = 0; blk < nblocks; ++blk) {
        const int z0 = blk * p.T, Tz = min(p.T, p.nz - z0);
        const bool store_plane = blk + 1 < nblocks;      // nothing reads the last block's plane
        const CUtensorMap *const tmap = blk == 0 ? (p.first_src < 0 ? &p.tmap_p0 : &p.tmap_plane[1])
                                                 : &p.tmap_plane[(blk - 1) & 1];
        float2 *const Pout = p.plane[blk & 1];
        float *const partial = p.partial + ((size_t)(blk & 1) * gridDim.x + blockIdx.x) * p.T * p.nxp;

        // Line buffers: 0 and 2 alternate as the LOADED buffer of consecutive items, 1 is the scratch half
        // of the ping-pong.  TMA: 8 lines x nbox boxes of item i0 + k into buffer 2*(k & 1); line l2 starts
        // 2*l2 samples earlier, so sample x of line l2 lands at l2*LS + (x - X0) + 2*l2.
        auto issue = [&](int k) {
            const int item = i0 + k;
            const int tl = item / p.npacks, pk = item - tl * p.npacks;
            const int X0 = tl * p.TX - p.H - R * HG;
            const unsigned bar = pdm_smem_u32(&mbar[k & 1]);
            asm volatile("fence.proxy.async;" ::: "memory");          // generic-proxy accesses (buffer, planes) are done
            pdm_mbar_expect_tx(bar, (unsigned)(W * p.nbox * p.BW * (int)sizeof(float2)));
            const unsigned dst0 = pdm_smem_u32(bufs + (size_t)(2 * (k & 1)) * buf_samples);
            for (int l2 = 0; l2 < W; ++l2)
                for (int bx = 0; bx < p.nbox; ++bx)
                    pdm_tma_load_2d(dst0 + (unsigned)((l2 * p.LS + bx * p.BW) * (int)sizeof(float2)), tmap,
                                    X0 - 2 * l2 + bx * p.BW, pk * W + l2, bar);
        };
        if (tid == 0 && nmine > 0) {
            issue(0);
            if (nmine > 1) issue(1);
        }

        int tile = i0 / p.npacks, pack = i0 - tile * p.npacks;
        int cur_tile = -1;                               // tile whose image the CTA is accumulating
        // A1 runs a step ahead of A3: the q values of the NEXT (item, step, pass) are requested before
        // the current group is computed (they come from L2)
        float qn[R];
        auto load_q = [&](int tl, int t, int pass) {
            const int g = (warp * p.passes + pass) * 4 + (lane >> 3);
            const int xg = tl * p.TX - p.H + R * g;
            const int xq = min(max(xg, 0), p.qstride - R);
            const float4 *qp = reinterpret_cast<const float4 *>(p.q + (size_t)(z0 + t) * p.qstride + xq);
            const float4 a = __ldg(qp), b = __ldg(qp + 1);
            qn[0] = a.x; qn[1] = a.y; qn[2] = a.z; qn[3] = a.w; qn[4] = b.x; qn[5] = b.y; qn[6] = b.z; qn[7] = b.w;
        };
        if (nmine > 0) load_q(tile, 0, 0);

        for (int k = 0; k < nmine; ++k) {
            const bool new_tile = tile != cur_tile;
            const bool restage = !GTAPS && (tile != st_tile || blk != st_blk || pack > st_hi || pack < st_lo);
            if (new_tile || restage) {                                    // CTA-uniform, rare
                __syncthreads();                                          // every warp is done with the old slice / tile
                if (new_tile) {
                    if (cur_tile >= 0) {                                  // the CTA leaves a tile: flush its image
                        const int x0 = cur_tile * p.TX;
                        for (int i = tid; i < Tz * p.TX; i += NT) {
                            const int t = i / p.TX, x = x0 + (i - t * p.TX);
                            if (x < p.nxp) partial[(size_t)t * p.nxp + x] = img[i];
                        }
                    }
                    for (int i = tid; i < p.T * p.TX; i += NT) img[i] = 0.f;
                    cur_tile = tile;
                }
                if (restage) {                                            // A2 staging
                    // rows this visit can touch: [idx(lowest w, q_min), idx(highest w, q_max)] with q over the
                    // samples of this (depth block, tile) only -- and as many of the CTA's next packs of the
                    // tile as the slice buffer holds (the ranges of neighbouring packs overlap almost entirely)
                    const float2 tq = p.tileq[(size_t)blk * p.ntiles + tile];
                    auto rows_of = [&](int pk) {
                        const float2 w2 = p.packw[pk];
                        return make_int2(pdm_index(w2.x, tq.x, ntab_m1), pdm_index(w2.y, tq.y, ntab_m1));
                    };
                    const int last = min(p.npacks - 1, pack + (nmine - 1 - k));
                    const int2 r0 = rows_of(pack);
                    int pe = pack, jhi = r0.y;
                    jlo = r0.x;
                    while (pe < last) {
                        const int2 n = rows_of(pe + 1);
                        const int lo2 = min(jlo, n.x), hi2 = max(jhi, n.y);
                        if (hi2 - lo2 + 1 > p.cap) break;
                        jlo = lo2; jhi = hi2; ++pe;
                    }
                    const int n4 = (jhi - jlo + 1) * p.half16;
                    const float4 *src = p.half + (size_t)jlo * p.half16;
                    for (int e = tid; e < n4; e += NT) slice[e] = src[e];
                    st_tile = tile; st_blk = blk; st_lo = pack; st_hi = pe;
                }
                __syncthreads();
            }
            const int line = pack * W + l;
            const float w = p.omega[min(line, p.nw - 1)];
            const int jloh = jlo * p.half16;
            const int bL = 2 * (k & 1);
            const int uses = ((k & 1) ? use1 : use0) + (k >> 1);          // earlier loads of this buffer
            int tile_n = tile, pack_n = pack + 1;                         // the next item
            if (pack_n == p.npacks) { pack_n = 0; ++tile_n; }

            pdm_mbar_wait(pdm_smem_u32(&mbar[k & 1]), (unsigned)uses & 1u);   // this item's tiles have landed

            for (int t = 0; t < Tz; ++t) {
                const float2 *cur = bufs + (size_t)((t & 1) ? 1 : bL) * buf_samples;
                float2 *nxt = bufs + (size_t)((t & 1) ? bL : 1) * buf_samples;
                const bool last_step = t == Tz - 1;
                for (int pass = 0; pass < p.passes; ++pass) {
                    const int g = (warp * p.passes + pass) * 4 + (lane >> 3);
                    const int xg = tile * p.TX - p.H + R * g;
                    int toff[R];
                    bool un = true;
#pragma unroll
                    for (int r = 0; r < R; ++r) {                       // A1
                        toff[r] = pdm_index(w, qn[r], ntab_m1) * p.half16 - jloh;
                        un = un && (toff[r] == toff[0]);
                    }
                    const bool uni = __all_sync(0xffffffffu, un && !p.force_general);
                    {                                                   // request the next group's q
                        int t2 = t, ps2 = pass + 1, tl2 = tile;
                        bool more = true;
                        if (ps2 == p.passes) { ps2 = 0; ++t2; }
                        if (t2 == Tz) { t2 = 0; tl2 = tile_n; more = k + 1 < nmine; }
                        if (more) load_q(tl2, t2, ps2);
                    }
                    if (pass == 0 && gs > 0) {                          // A4: neighbours have completed step gs-1
                        if (lane == 0) {
                            while (*(volatile int *)&prog[warp] < gs) { }
                            while (*(volatile int *)&prog[warp + 2] < gs) { }
                            __threadfence_block();
                        }
                        __syncwarp();
                    }
                    const int soff = l * p.LS + R * HG + R * g + 2 * l;
                    const float2 *base = cur + soff;
                    float2 out[R];
                    const float4 *const tb = GTAPS ? p.half : slice;    // jlo stays 0 with GTAPS: global row offsets
                    if (SYM) {
                        if (uni) pdm_fir_group<L, R, true, false, 0u, 0>(base, tb, toff, out);
                        else     pdm_fir_group<L, R, false, false, 0u, 0>(base, tb, toff, out);
                    } else {
                        if (uni) pdm_fir_group_asym<L, R, true, 0>(base, tb, toff, out);
                        else     pdm_fir_group_asym<L, R, false, 0>(base, tb, toff, out);
                    }
                    if (xg < 0 || xg + R > p.nx) {                      // R5: zero outside [0,nx) (edge groups only)
#pragma unroll
                        for (int r = 0; r < R; ++r)
                            if ((unsigned)(xg + r) >= (unsigned)p.nx) out[r] = make_float2(0.f, 0.f);
                    }
                    if (p.ntaper > 0 && (xg < p.ntaper || xg + R > p.nx - p.ntaper)) {   // R5b (edge groups only)
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            const int x = xg + r, d = min(x, p.nx - 1 - x);
                            if (d >= 0 && d < p.ntaper) {
                                const float t = __ldg(p.taper + d);
                                out[r].x *= t; out[r].y *= t;
                            }
                        }
                    }
                    const bool central = g >= gc0 && g < gc1;
                    if (!last_step) {
                        float2 *dst = nxt + soff;
#pragma unroll
                        for (int i = 0; i < R / 2; ++i)
                            *reinterpret_cast<float4 *>(dst + 2 * i) = make_float4(out[2 * i].x, out[2 * i].y, out[2 * i + 1].x, out[2 * i + 1].y);
                    } else if (store_plane && central && xg < p.nxp && line < p.nw) {
                        float4 *dst = reinterpret_cast<float4 *>(Pout + (size_t)line * p.nxp + xg);
#pragma unroll
                        for (int i = 0; i < R / 2; ++i)
                            __stcg(dst + i, make_float4(out[2 * i].x, out[2 * i].y, out[2 * i + 1].x, out[2 * i + 1].y));
                    }
                    // A5: sum Re P over the 8 lines of the pack (fixed tree), lane l ends with output r = l
                    float s;
                    {
                        float a4[4], a2[2];
                        const bool b2 = l & 4, b1 = l & 2, b0 = l & 1;
                        if (p.xcorr) {                                  // R17: Re(conj(S) R) = Re(U R) of the line pair,
#pragma unroll                                                          // counted once (on the even lane)
                            for (int r = 0; r < R; ++r) {
                                const float px = __shfl_xor_sync(0xffffffffu, out[r].x, 1);
                                const float py = __shfl_xor_sync(0xffffffffu, out[r].y, 1);
                                out[r].x = b0 ? 0.f : out[r].x * px - out[r].y * py;
                            }
                        }
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            const float keep = b2 ? out[i + 4].x : out[i].x, send = b2 ? out[i].x : out[i + 4].x;
                            a4[i] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
                        }
#pragma unroll
                        for (int i = 0; i < 2; ++i) {
                            const float keep = b1 ? a4[i + 2] : a4[i], send = b1 ? a4[i] : a4[i + 2];
                            a2[i] = keep + __shfl_xor_sync(0xffffffffu, send, 2);
                        }
                        const float keep = b0 ? a2[1] : a2[0], send = b0 ? a2[0] : a2[1];
                        s = keep + __shfl_xor_sync(0xffffffffu, send, 1);
                    }
                    if (central) img[t * p.TX + (g - gc0) * R + l] += s;
                }
                ++gs;
                __syncwarp();                                           // A4: publish this warp's step
                if (lane == 0) {
                    __threadfence_block();
                    *(volatile int *)&prog[warp + 1] = gs;
                }
            }
            // The warp is done with this item's loaded buffer; the LAST warp to get here refills it with
            // the tiles of item k+2 (item k+1 is already in flight in the other buffer)
            if (lane == 0) {
                __threadfence_block();
                const bool last_warp = atomicAdd(&buf_done[k & 1], 1) == (uses + 1) * nwarps - 1;
                if (last_warp && k + 2 < nmine) issue(k + 2);
            }
            tile = tile_n; pack = pack_n;
        }
        use0 += (nmine + 1) >> 1; use1 += nmine >> 1;
        __syncthreads();
        if (cur_tile >= 0) {                                              // flush the last tile's image
            const int x0 = cur_tile * p.TX;
            for (int i = tid; i < Tz * p.TX; i += NT) {
                const int t = i / p.TX, x = x0 + (i - t * p.TX);
                if (x < p.nxp) partial[(size_t)t * p.nxp + x] = img[i];
            }
        }
        // Depth blocks are ordered by a grid-wide barrier (all CTAs are co-resident: cooperative launch):
        // the planes and image tiles written above are read by other CTAs (TMA / the reduction) after it
        asm volatile("fence.proxy.async;" ::: "memory");
        __threadfence();
        __syncthreads();
        if (tid == 0) {
            const unsigned target = (unsigned)(blk + 1) * gridDim.x;
            atomicAdd(p.gbar, 1u);
            unsigned v;
            do {
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p.gbar) : "memory");
            } while (v < target);
        }
        __syncthreads();
        // A5, second half: image rows of this depth block = sum of the CTAs' tiles in CTA order
        {
            const float *part = p.partial + (size_t)(blk & 1) * gridDim.x * p.T * p.nxp;
            const int n = Tz * p.nx;
            for (int i = blockIdx.x * NT + tid; i < n; i += gridDim.x * NT) {
                const int t = i / p.nx, x = i - t * p.nx;
                const int2 c = p.tile_ctas[x / p.TX];
                float s = 0.f;
                for (int c2 = c.x; c2 <= c.y; ++c2) s += __ldcg(part + ((size_t)c2 * p.T + t) * p.nxp + x);
                float *o = p.image + (size_t)(z0 + t) * p.nx + x;
                *o = p.accumulate ? *o + s : s;
            }
        }
    }
}

// repack of a caller's P0 whose rows TMA cannot address (odd nx or an 8-byte aligned base)
static __global__ void pdm_pack_copy_in(const float2 *__restrict__ P0, float2 *__restrict__ plane, int nx, int nxp, int nw)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x, line = blockIdx.y;
    if (x < nxp) plane[(size_t)line * nxp + x] = x < nx ? P0[(size_t)line * nx + x] : make_float2(0.f, 0.f);
}

// prestack (R17): receiver lines and CONJUGATED source lines interleaved into one plane, so that the
// same operator marches both (conj(S') = sum_k W_k conj(S)(x-k)) and a line pair shares its table rows
static __global__ void pdm_pack_interleave(const float2 *__restrict__ rec, const float2 *__restrict__ src,
                                           float2 *__restrict__ plane, int nx, int nxp, int nw)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y;
    if (x >= nxp) return;
    float2 r = make_float2(0.f, 0.f), u = r;
    if (x < nx) {
        r = rec[(size_t)i * nx + x];
        const float2 s = src[(size_t)i * nx + x];
        u = make_float2(s.x, -s.y);
    }
    plane[(size_t)(2 * i) * nxp + x] = r;
    plane[(size_t)(2 * i + 1) * nxp + x] = u;
}

// pdm_api.cu -- host side of libpdm: the C ABI declared in include/pdm.h.
// Everything data-independent is validated, pre-digested and uploaded in pdm_create; pdm_migrate
// only enqueues kernels on the caller's stream.  There is no CPU fallback anywhere in this file:
// without a compute-capability-10.x device pdm_create fails with PDM_ERR_UNSUPPORTED.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "pdm_common.cuh"
#include "kern_naive.cuh"
#include "kern_peak.cuh"
#include "kern_reduce.cuh"
#include "pdm_dispatch.cuh"

#define PDM_CUDA(plan, call)                                                        \
    do {                                                                            \
        cudaError_t e_ = (call);                                                    \
        if (e_ != cudaSuccess) {                                                    \
            if (plan) (plan)->last_cuda_error = (int)e_;                            \
            return e_ == cudaErrorMemoryAllocation ? PDM_ERR_NOMEM : PDM_ERR_CUDA;  \
        }                                                                           \
    } while (0)

extern "C" const char *pdm_strerror(int code)
{
    switch (code) {
    case PDM_OK: return "ok";
    case PDM_ERR_INVALID_ARG: return "invalid argument";
    case PDM_ERR_TABLE_RANGE: return "omega*dz/(v*du) exceeds the last table row";
    case PDM_ERR_TABLE_ASYMMETRIC: return "filter table is not bitwise symmetric in k";
    case PDM_ERR_UNSUPPORTED: return "unsupported device, path or filter length";
    case PDM_ERR_NOMEM: return "out of memory";
    case PDM_ERR_CUDA: return "CUDA call failed (see pdm_info.last_cuda_error)";
    case PDM_ERR_TOO_LARGE: return "nx*nw exceeds PDM_STATIC_MAX_SAMPLES (the built-in scratch of pdm_migrate_static)";
    default: return "unknown pdm_status";
    }
}

// R3: q32 = fl32(dz / (v * du)), one rounding from double.
static inline float host_q(double dz, float v, double du) { return (float)(dz / ((double)v * du)); }
// R3: FLOAT product (no addend, so no contraction), round half to even, clamp.
static inline int host_index(float w, float q, int ntab)
{
    volatile float prod = w * q;
    long j = lrintf(prod);
    if (j < 0) j = 0;
    if (j > ntab - 1) j = ntab - 1;
    return (int)j;
}

static void free_plan(pdm_plan *p)
{
    if (!p) return;
    if (p->tex_half) cudaDestroyTextureObject(p->tex_half);
    cudaFree(p->d_omega); cudaFree(p->d_q); cudaFree(p->d_table); cudaFree(p->d_half);
    cudaFree(p->d_rowoff); cudaFree(p->d_rows); cudaFree(p->d_partial);
    cudaFree(p->d_plane[0]); cudaFree(p->d_plane[1]); cudaFree(p->d_flags);
    cudaFree(p->d_handoff); cudaFree(p->d_segs); cudaFree(p->d_segoff);
    cudaFree(p->d_stage_p0); cudaFree(p->d_stage_img);
    cudaFree(p->d_packw); cudaFree(p->d_tileq); cudaFree(p->d_tile_ctas); cudaFree(p->d_taper);
    for (int i = 0; i < 3; ++i) if (p->ev[i]) cudaEventDestroy(p->ev[i]);
    delete p;
}

template <class T>
static int dev_alloc(pdm_plan *p, T **ptr, size_t count)
{
    *ptr = nullptr;
    if (count == 0) count = 1;
    // Large requests (the per-CTA partial images of the marching form are grid*nz*nx*4 B: 5.5 GB for
    // configs[3], 39 GB for a 16384 x 4000 image) are checked against the free memory first, so that a plan
    // that cannot fit fails with PDM_ERR_NOMEM at once instead of after the driver has tried to make room.
    if (count * sizeof(T) >= ((size_t)256 << 20)) {
        size_t free_b = 0, total_b = 0;
        if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess) {
            if (count * sizeof(T) > free_b) { p->last_cuda_error = (int)cudaErrorMemoryAllocation; return PDM_ERR_NOMEM; }
        } else cudaGetLastError();
    }
    PDM_CUDA(p, cudaMalloc((void **)ptr, count * sizeof(T)));
    p->workspace_bytes += (double)(count * sizeof(T));
    return PDM_OK;
}

template <class T>
static int dev_upload(pdm_plan *p, T **ptr, const T *host, size_t count)
{
    int rc = dev_alloc(p, ptr, count);
    if (rc != PDM_OK) return rc;
    PDM_CUDA(p, cudaMemcpy(*ptr, host, count * sizeof(T), cudaMemcpyHostToDevice));
    return PDM_OK;
}

static int build_plan(pdm_plan *p, const float *omega, const float *velocity, const pdm_c64 *table);

extern "C" int pdm_create(pdm_plan **out, int nx, int nz, int nw, float dx, float dz,
                          const float *omega, const float *velocity,
                          const pdm_c64 *table, int ntab, int ntaps, double tab_du, unsigned flags)
{
    if (!out) return PDM_ERR_INVALID_ARG;
    *out = nullptr;
    if (!omega || !velocity || !table) return PDM_ERR_INVALID_ARG;
    if (nx <= 0 || nz <= 0 || nw <= 0 || ntab <= 0 || ntaps < 1 || (ntaps & 1) == 0)
        return PDM_ERR_INVALID_ARG;
    if (!(tab_du > 0.0) || !std::isfinite(tab_du) || !(dz > 0.f) || !std::isfinite(dz) ||
        !(dx > 0.f) || !std::isfinite(dx))
        return PDM_ERR_INVALID_ARG;
    if (flags & ~PDM_FLAGS_VALID) return PDM_ERR_INVALID_ARG;
    const unsigned path = flags & PDM_PATH_MASK;
    if (path > PDM_PATH_PACKED) return PDM_ERR_INVALID_ARG;
    if (ntaps > PDM_MAX_TAPS) return PDM_ERR_UNSUPPORTED;
    if ((double)nz * (double)nx > 2.0e9 || (double)nw * (double)nx > 2.0e9) return PDM_ERR_UNSUPPORTED;
    for (int i = 0; i < nw; ++i)
        if (!(omega[i] > 0.f) || !std::isfinite(omega[i])) return PDM_ERR_INVALID_ARG;
    const size_t plane = (size_t)nz * nx;
    for (size_t i = 0; i < plane; ++i)
        if (!(velocity[i] > 0.f) || !std::isfinite(velocity[i])) return PDM_ERR_INVALID_ARG;
    const int L = (ntaps - 1) / 2;
    // W_k == W_-k bit for bit in every row: the folded kernels (north_star); otherwise the general
    // kernels apply the full 2L+1 row (Eq. (1) literally, R11)
    bool symmetric = true;
    for (int j = 0; j < ntab && symmetric; ++j) {
        const pdm_c64 *row = table + (size_t)j * ntaps + L;
        for (int k = 1; k <= L; ++k)
            if (memcmp(&row[k], &row[-k], sizeof(pdm_c64)) != 0) { symmetric = false; break; }
    }
    if (!symmetric && (flags & PDM_REQUIRE_SYMMETRIC)) return PDM_ERR_TABLE_ASYMMETRIC;

    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        cudaGetLastError();
        return PDM_ERR_UNSUPPORTED;           // no usable CUDA device: fail loudly, no fallback
    }
    if (prop.major != 10) return PDM_ERR_UNSUPPORTED;

    // prestack plans carry two lines per frequency (receiver field, conjugated source field): R17
    const bool prestack = (flags & PDM_PRESTACK) != 0;
    if (prestack && path != PDM_PATH_AUTO && path != PDM_PATH_PACKED) return PDM_ERR_INVALID_ARG;
    const int ntaper = (int)((flags >> PDM_TAPER_SHIFT) & 0xFFu);       // R5b: packed form only
    if (ntaper && (prestack || (path != PDM_PATH_AUTO && path != PDM_PATH_PACKED))) return PDM_ERR_INVALID_ARG;
    // R3c: interpolated look-up -- the per-depth-step form only, plain poststack
    const bool interp = (flags & PDM_TABLE_INTERP) != 0;
    if (interp && (prestack || ntaper || (path != PDM_PATH_AUTO && path != PDM_PATH_NAIVE))) return PDM_ERR_INVALID_ARG;
    std::vector<float> omega2;
    if (prestack) {
        if ((double)2 * nw * (double)nx > 2.0e9) return PDM_ERR_UNSUPPORTED;
        omega2.resize((size_t)2 * nw);
        for (int i = 0; i < nw; ++i) omega2[2 * i] = omega2[2 * i + 1] = omega[i];
        omega = omega2.data();
        nw *= 2;
    }
    pdm_plan *p = new (std::nothrow) pdm_plan();
    if (!p) return PDM_ERR_NOMEM;
    memset(p, 0, sizeof(*p));
    p->prestack = prestack ? 1 : 0;
    p->ntaper = ntaper;
    p->nx = nx; p->nz = nz; p->nw = nw; p->ntab = ntab; p->ntaps = ntaps; p->L = L;
    p->dx = dx; p->dz = dz; p->du = tab_du; p->flags = flags;
    p->sym = symmetric ? 1 : 0;
    p->device = dev; p->sm_count = prop.multiProcessorCount;
    p->smem_optin = (int)prop.sharedMemPerBlockOptin;

    int rc = build_plan(p, omega, velocity, table);
    if (rc != PDM_OK) { free_plan(p); return rc; }
    *out = p;
    return PDM_OK;
}

// ------------------------------------------------------------------------------------------------
// kernel dispatch: filter half-lengths with a fully unrolled, register-tiled instantiation
// ------------------------------------------------------------------------------------------------
static march_fn march_kernel_for(const pdm_plan *p, bool taps_smem, bool dedup, int R)
{
    const int L = p->Lk;
    march_fn f;
    if (!p->sym) {
        f = pdm_march_kernel_asym_part0(L, taps_smem);
        if (!f) f = pdm_march_kernel_asym_part1(L, taps_smem);
        if (!f) f = pdm_march_kernel_asym_part2(L, taps_smem);
        return f;
    }
    f = pdm_march_kernel_part0(L, taps_smem, dedup, R);
    if (!f) f = pdm_march_kernel_part1(L, taps_smem, dedup, R);
    if (!f) f = pdm_march_kernel_part2(L, taps_smem, dedup, R);
    return f;
}
static cluster_fn cluster_kernel_for(const pdm_plan *p, bool taps_smem, bool dedup)
{
    const int L = p->Lk;
    if (!p->sym) {
        cluster_fn f = pdm_cluster_kernel_asym_part0(L, taps_smem);
        if (!f) f = pdm_cluster_kernel_asym_part1(L, taps_smem);
        if (!f) f = pdm_cluster_kernel_asym_part2(L, taps_smem);
        return f;
    }
    return pdm_cluster_kernel_for(L, taps_smem, dedup);
}
// output tile aliased onto the consumed input tile: only where it pays (long per-sample rows)
static bool tiled_alias(const pdm_plan *p) { return p->sym && p->contiguous_rows != 0 && p->Lk == 25; }
static tiled_fn tiled_kernel_for(const pdm_plan *p, bool wide)
{
    if (!p->sym) {
        tiled_fn f = pdm_tiled_kernel_asym_part0(p->Lk, wide);
        if (!f) f = pdm_tiled_kernel_asym_part1(p->Lk, wide);
        if (!f) f = pdm_tiled_kernel_asym_part2(p->Lk, wide);
        return f;
    }
    return pdm_tiled_kernel_for(p->Lk, wide, tiled_alias(p));
}
static pack_fn pack_kernel_for(const pdm_plan *p)
{
    pack_fn f = pdm_pack_kernel_part0(p->Lk, p->sym != 0, p->threads, p->pk_gtaps != 0);
    if (!f) f = pdm_pack_kernel_part1(p->Lk, p->sym != 0, p->threads, p->pk_gtaps != 0);
    if (!f) f = pdm_pack_kernel_part2(p->Lk, p->sym != 0, p->threads, p->pk_gtaps != 0);
    return f;
}
// TMA descriptor of a [nrows][row_samples] array of 8-byte samples (complex64 moved as opaque 64-bit
// words), one-row boxes of `box` samples, out-of-range elements read as zero (R5).  The encoder is a
// driver entry point resolved at run time: libpdm.so does not link libcuda (it must load without a GPU).
typedef CUresult (*pdm_encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);
static pdm_encode_fn tensor_map_encoder()
{
    static pdm_encode_fn enc = nullptr;
    if (!enc) {
        void *sym = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qr) != cudaSuccess ||
            qr != cudaDriverEntryPointSuccess || !sym) {
            cudaGetLastError();
            return nullptr;
        }
        enc = (pdm_encode_fn)sym;
    }
    return enc;
}
static int make_plane_map(pdm_plan *p, CUtensorMap *map, const void *base, int row_samples, int nrows, int box)
{
    const pdm_encode_fn enc = tensor_map_encoder();
    if (!enc) return PDM_ERR_UNSUPPORTED;
    const cuuint64_t dims[2] = { (cuuint64_t)row_samples, (cuuint64_t)nrows };
    const cuuint64_t strides[1] = { (cuuint64_t)row_samples * sizeof(float2) };
    const cuuint32_t boxd[2] = { (cuuint32_t)box, 1u }, estr[2] = { 1u, 1u };
    const CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_UINT64, 2, const_cast<void *>(base), dims, strides, boxd, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                           CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { p->last_cuda_error = (int)r; return PDM_ERR_CUDA; }
    return PDM_OK;
}
// Filter lengths without an instantiation of their own run on the next longer one with the extra
// taps set to zero (x + 0*s == x exactly), so every odd length up to the longest instantiation
// takes the unrolled kernels; 0 = longer than all of them (scaffold only).
static int kernel_half_length(int L)
{
#define X(LL) if (L <= LL) return LL;
    PDM_FOR_EACH_L(X)
#undef X
    return 0;
}
// Work list of the marching kernel.  Unbalanced: CTA c owns whole lines c, c+grid, ...  Balanced
// (nw >= grid): the nw*nz depth steps, laid end to end line after line, are cut into `grid` equal
// ranges; a range is [tail of a line][whole lines][head of a line].  The CTA runs its head FIRST
// (it depends on nothing) and publishes the line at the split depth, its tail LAST (by then the
// owner of that line's head has long published it), so no CTA waits on work that has not started.
static void build_segments(int nw, int nz, int grid, bool balance,
                           std::vector<int4> &segs, std::vector<int> &segoff, int &nslots)
{
    segs.clear(); segoff.assign(grid + 1, 0); nslots = 0;
    if (!balance) {
        for (int c = 0; c < grid; ++c) {
            for (int line = c; line < nw; line += grid) segs.push_back(make_int4(line, 0, nz, -1));
            segoff[c + 1] = (int)segs.size();
        }
        return;
    }
    const long long total = (long long)nw * nz;
    std::vector<int> slot_of_line(nw, -1);
    for (int c = 0; c < grid; ++c) {
        const long long a = total * c / grid, b = total * (c + 1) / grid;
        std::vector<int4> mine;
        for (long long t = a; t < b;) {
            const int line = (int)(t / nz), z0 = (int)(t - (long long)line * nz);
            const int z1 = (int)std::min<long long>(nz, z0 + (b - t));
            if ((z0 > 0 || z1 < nz) && slot_of_line[line] < 0) slot_of_line[line] = nslots++;
            mine.push_back(make_int4(line, z0, z1, (z0 > 0 || z1 < nz) ? slot_of_line[line] : -1));
            t += z1 - z0;
        }
        // execution order: head (z0 == 0, z1 < nz) first, tail (z0 > 0) last
        if (!mine.empty() && mine.back().y == 0 && mine.back().z < nz) segs.push_back(mine.back());
        for (size_t i = 0; i < mine.size(); ++i) {
            const int4 m = mine[i];
            if (m.y == 0 && m.z == nz) segs.push_back(m);
        }
        if (!mine.empty() && mine.front().y > 0) segs.push_back(mine.front());
        segoff[c + 1] = (int)segs.size();
    }
}

// Row de-duplication inside a thread (pdm_fir_group DEDUP) pays where nearly every sample has its
// own table row and the filter is short enough to leave registers: measured +4..7 % on the marching
// path for taps <= 35 on random-field models, -4 % at 51 taps, -10 % on the 128-register tiled kernel.
static bool use_dedup(const pdm_plan *p) { return p->sym && p->contiguous_rows != 0 && p->Lk <= 17; }

// the half table as a linear float4 texture: the per-sample-row kernel variants fetch part of their
// tap rows through the texture unit (a second gather path next to the LSU)
static int make_half_texture(pdm_plan *p, size_t count)
{
    cudaResourceDesc rd; memset(&rd, 0, sizeof(rd));
    rd.resType = cudaResourceTypeLinear; rd.res.linear.devPtr = p->d_half;
    rd.res.linear.desc = cudaCreateChannelDesc<float4>();
    rd.res.linear.sizeInBytes = count * sizeof(float4);
    cudaTextureDesc td; memset(&td, 0, sizeof(td));
    td.readMode = cudaReadModeElementType;
    PDM_CUDA(p, cudaCreateTextureObject(&p->tex_half, &rd, &td, nullptr));
    return PDM_OK;
}

static int halo_groups(int L, int R) { return (L + 1 + R - 1) / R; }
static int round_up(int a, int b) { return (a + b - 1) / b * b; }

// Plan of the frequency-packed, temporally blocked form (kern_pack.cuh).  Feasibility (a CTA size whose
// line tiles leave room for the table rows of one tile visit, cooperative launch) is settled BEFORE anything
// is allocated, so that AUTO can fall back to another form on PDM_ERR_UNSUPPORTED.
static int build_packed(pdm_plan *p, const float *omega, const std::vector<float> &q, const std::vector<float4> &half,
                        int Lk, int HG)
{
    const int nx = p->nx, nz = p->nz, nw = p->nw, ntab = p->ntab, R = PDM_R;
    int rc;
    // the TMA descriptor encoder is part of feasibility: without it AUTO must fall back with nothing allocated
    if (!tensor_map_encoder()) return PDM_ERR_UNSUPPORTED;
    // kern_pack.cuh: 8 adjacent frequencies per quarter warp, T depth steps per tile visit
    p->taps_mode = 2;
    p->pk_gtaps = 0;
    const int W = PDM_PACK_W;
    // the tuning bits mean something else for the other forms: read them only when this form is forced
    const bool forced = (p->flags & PDM_PATH_MASK) == PDM_PATH_PACKED;
    const unsigned nsel = forced ? (p->flags >> PDM_THREADS_SHIFT) & 0xFFu : 0u;   // CTA size / 32: 8, 12 or 16
    if (nsel && nsel != 8 && nsel != 12 && nsel != 16) return PDM_ERR_UNSUPPORTED;
    const unsigned tsel = forced ? (p->flags >> PDM_CTAS_SHIFT) & 0xFu : 0u;       // steps per tile visit
    // default: the longest T whose recomputed halo stays near 10 % of the tile
    const int T = std::min(nz, tsel ? (int)tsel : (Lk <= 7 ? 4 : (Lk <= 12 ? 3 : 2)));
    p->nxp = round_up(nx, R);
    const int npacks = (nw + W - 1) / W;
    std::vector<float2> packw(npacks);
    for (int k = 0; k < npacks; ++k) {
        float wlo = INFINITY, whi = 0.f;
        for (int i = k * W; i < std::min(nw, (k + 1) * W); ++i) { wlo = std::min(wlo, omega[i]); whi = std::max(whi, omega[i]); }
        packw[k] = make_float2(wlo, whi);
    }
    // CTA size: the largest whose line tiles leave room for the table rows one tile visit can touch
    // (512 threads = 512 samples per line and step; long filters with widely spread rows take 384 or 256)
    int NT = 0, passes = 0, TXH = 0, H = 0, TX = 0, nbox = 0, BW = 0, LS = 0, ntiles = 0, cap = 0;
    const int nblocks = (nz + T - 1) / T;
    std::vector<float2> tileq;
    size_t fixed = 0;
    // Plans that have no other form to fall back to (forced, prestack, taper) get a second round: the
    // 256-thread build that reads tap rows from the global table, for which no row range is too wide.
    const bool must_exist = forced || p->prestack || p->ntaper > 0;
    for (int round = 0; round < (must_exist ? 2 : 1) && !NT; ++round)
    for (int cand = round ? 256 : 512; cand >= 256 && !NT; cand -= 128) {
        if (nsel && cand != 32 * (int)nsel) continue;
        passes = cand == 256 ? 2 : 1;                  // groups per thread and step
        TXH = cand / W * R * passes;                   // samples a CTA computes per line and step
        H = round_up((T - 1) * Lk, R);                 // recomputed halo per side
        TX = TXH - 2 * H;
        if (TX < 8 * R) continue;
        const int w_load = TXH + 2 * R * HG + 2 * (W - 1);   // samples per line incl. fetched halo and the per-line skew
        nbox = (w_load + 255) / 256;
        BW = round_up((w_load + nbox - 1) / nbox, 16); // 128-byte aligned box starts
        LS = nbox * BW;
        const size_t lines_bytes = (size_t)PDM_PACK_NBUF * W * LS * sizeof(float2);
        const size_t img_bytes = (size_t)T * TX * sizeof(float);
        ntiles = (nx + TX - 1) / TX;
        // q extrema over the samples one tile visit computes (its T depth rows, its outputs and halo;
        // columns past nx repeat the last q, as in d_q): they bound the table rows the visit can touch
        tileq.assign((size_t)nblocks * ntiles, make_float2(0.f, 0.f));
        int maxrows = 0;
        for (int b = 0; b < nblocks; ++b)
            for (int t = 0; t < ntiles; ++t) {
                const int xa = std::max(0, t * TX - H), xb = std::min(nx - 1, t * TX - H + TXH - 1);
                float lo = INFINITY, hi = 0.f;
                for (int z = b * T; z < std::min(nz, (b + 1) * T); ++z) {
                    const float *row = q.data() + (size_t)z * p->qstride;
                    for (int x = xa; x <= xb; ++x) { lo = std::min(lo, row[x]); hi = std::max(hi, row[x]); }
                }
                tileq[(size_t)b * ntiles + t] = make_float2(lo, hi);
                for (int k = 0; k < npacks; ++k)
                    maxrows = std::max(maxrows, host_index(packw[k].y, hi, ntab) - host_index(packw[k].x, lo, ntab) + 1);
            }
        fixed = 128 + lines_bytes + img_bytes;
        const size_t budget = (size_t)p->smem_optin - 1024;   // the kernel's static shared memory counts too
        if (fixed >= budget) continue;
        if (round) {                                   // global tap rows: no slice buffer at all
            cap = 0;
            p->pk_gtaps = 1;
            p->taps_mode = 1;
        } else {
            cap = (int)((budget - fixed) / ((size_t)p->half16 * sizeof(float4)));
            if (cap < maxrows) continue;               // one pack's rows must fit next to the line tiles
            cap = std::min(cap, ntab);
        }
        NT = cand;
    }
    if (!NT) return PDM_ERR_UNSUPPORTED;
    p->pk_T = T; p->pk_TX = TX; p->pk_H = H; p->pk_LS = LS; p->pk_BW = BW; p->pk_nbox = nbox;
    p->pk_cap = cap; p->pk_passes = passes; p->pk_npacks = npacks;
    p->pk_ntiles = ntiles;
    p->threads = NT;
    p->tile_x = TX;
    p->smem_bytes = (int)(fixed + (size_t)cap * p->half16 * sizeof(float4));
    pack_fn fn = pack_kernel_for(p);
    if (!fn) return PDM_ERR_UNSUPPORTED;
    PDM_CUDA(p, cudaFuncSetAttribute((const void *)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, p->smem_bytes));
    const long long nitems = (long long)p->pk_ntiles * npacks;
    if (nitems > 0x7fffffffLL) return PDM_ERR_UNSUPPORTED;
    p->ctas_per_sm = 1;
    p->grid = (int)std::min<long long>(nitems, p->sm_count);
    p->launches = 1;
    p->n_partial = p->grid;
    {
        int coop = 0, per_sm = 0;
        PDM_CUDA(p, cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, p->device));
        PDM_CUDA(p, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void *)fn, NT, (size_t)p->smem_bytes));
        if (!coop || per_sm < 1) return PDM_ERR_UNSUPPORTED;   // the depth blocks need all CTAs co-resident
    }
    // CTA c owns items [nitems*c/grid, nitems*(c+1)/grid) of the tile-major list: the CTAs that hold
    // a piece of a tile's image are consecutive
    std::vector<int2> tile_ctas(p->pk_ntiles, make_int2(p->grid, -1));
    for (int c = 0; c < p->grid; ++c) {
        const long long a0 = nitems * c / p->grid, a1 = nitems * (c + 1) / p->grid;
        if (a0 >= a1) continue;
        for (int t = (int)(a0 / npacks); t <= (int)((a1 - 1) / npacks); ++t) {
            tile_ctas[t].x = std::min(tile_ctas[t].x, c);
            tile_ctas[t].y = std::max(tile_ctas[t].y, c);
        }
    }
    if ((rc = dev_upload(p, &p->d_half, half.data(), half.size())) != PDM_OK) return rc;
    if ((rc = dev_upload(p, &p->d_packw, packw.data(), packw.size())) != PDM_OK) return rc;
    if ((rc = dev_upload(p, &p->d_tileq, tileq.data(), tileq.size())) != PDM_OK) return rc;
    if ((rc = dev_upload(p, &p->d_tile_ctas, tile_ctas.data(), tile_ctas.size())) != PDM_OK) return rc;
    if ((rc = dev_alloc(p, &p->d_partial, (size_t)2 * p->grid * T * p->nxp)) != PDM_OK) return rc;
    if ((rc = dev_alloc(p, &p->d_flags, (size_t)1)) != PDM_OK) return rc;
    for (int i = 0; i < 2; ++i) {
        if ((rc = dev_alloc(p, &p->d_plane[i], (size_t)nw * p->nxp)) != PDM_OK) return rc;
        PDM_CUDA(p, cudaMemset(p->d_plane[i], 0, (size_t)nw * p->nxp * sizeof(float2)));
        if ((rc = make_plane_map(p, &p->tmap_plane[i], p->d_plane[i], p->nxp, nw, BW)) != PDM_OK) return rc;
    }
    if (p->ntaper) {                                       // R5b weights, formed in double
        std::vector<float> tp(p->ntaper);
        for (int d = 0; d < p->ntaper; ++d) {
            const double sn = sin(1.57079632679489661923 * (double)(d + 1) / (double)(p->ntaper + 1));
            tp[d] = (float)(sn * sn);
        }
        if ((rc = dev_upload(p, &p->d_taper, tp.data(), tp.size())) != PDM_OK) return rc;
    }
    p->path = PDM_PATH_PACKED;
    return PDM_OK;
}

static int build_plan(pdm_plan *p, const float *omega, const float *velocity, const pdm_c64 *table)
{
    const int nx = p->nx, nz = p->nz, nw = p->nw, ntab = p->ntab, ntaps = p->ntaps, L = p->L;
    const int Lk = kernel_half_length(L);                  // 0: no unrolled kernel is long enough
    p->Lk = Lk;
    // outputs per thread: PDM_R = 8 for every kernel form; the single-CTA marching form also has an
    // R = 4 build for short lines with so few of them that 8 would leave the SMs with under 8 warps
    // each (configs[0], [1]).  The form is chosen with the R = 8 layout first; R drops to 4 only once
    // the path is known to be PDM_PATH_SMEM (tiled and cluster kernels exist for R = 8 only).
    const unsigned want_path = p->flags & PDM_PATH_MASK;
    const bool small = p->sym && (want_path == PDM_PATH_AUTO || want_path == PDM_PATH_SMEM) && nx <= 1024 &&
                       (long long)nw * ((nx + 255) / 256) <= 8LL * p->sm_count &&
                       ((p->flags >> PDM_THREADS_SHIFT) & 0xFFu) == 0;   // a forced thread count means the R = 8 layout
    int R = PDM_R;
    p->R = R;

    // ---- q map (R3) and its extrema ---------------------------------------------------------
    p->qstride = round_up(nx, PDM_TILED_THREADS * PDM_R);
    std::vector<float> q((size_t)nz * p->qstride);
    float qmin = INFINITY, qmax = 0.f;
    for (int z = 0; z < nz; ++z) {
        float *row = q.data() + (size_t)z * p->qstride;
        for (int x = 0; x < nx; ++x) {
            const float v = host_q((double)p->dz, velocity[(size_t)z * nx + x], p->du);
            row[x] = v;
            qmin = std::min(qmin, v); qmax = std::max(qmax, v);
        }
        for (int x = nx; x < p->qstride; ++x) row[x] = row[nx - 1];
    }
    if (!std::isfinite(qmax) || !(qmin > 0.f)) return PDM_ERR_INVALID_ARG;
    float wmax = 0.f;
    for (int i = 0; i < nw; ++i) wmax = std::max(wmax, omega[i]);
    {
        volatile float prod = wmax * qmax;                 // fl32 product is monotone in both factors
        if (!(prod < 2.0e9f) || lrintf(prod) > ntab - 1) return PDM_ERR_TABLE_RANGE;
    }

    // ---- half table: rows k = 0..L as float4 pairs (W_2t, W_2t+1), odd number of float4 per row
    // general (asymmetric) tables: unit k = (W_k, W_-k), k = 0..L, same odd padding
    p->half16 = (p->sym ? (std::max(L, Lk) + 2) / 2 : std::max(L, Lk) + 1) | 1;   // rows padded with zero taps up to Lk
    std::vector<float4> half((size_t)ntab * p->half16, make_float4(0.f, 0.f, 0.f, 0.f));
    for (int j = 0; j < ntab; ++j)
        for (int k = 0; k <= L; ++k) {
            const pdm_c64 w = table[(size_t)j * ntaps + L + k];
            if (p->sym) {
                float4 &d = half[(size_t)j * p->half16 + k / 2];
                if (k & 1) { d.z = w.re; d.w = w.im; } else { d.x = w.re; d.y = w.im; }
            } else {
                const pdm_c64 wm = table[(size_t)j * ntaps + L - k];
                half[(size_t)j * p->half16 + k] = make_float4(w.re, w.im, wm.re, wm.im);
            }
        }

    // ---- per-omega list of rows that omega can touch ---------------------------------------------
    // few distinct q (piecewise-constant models): exact compact lists; else the full range [jmin,jmax]
    std::vector<float> uq;
    {
        const size_t cap = 2048;
        std::vector<float> seen;                           // tiny sorted set with early exit
        bool few = true;
        float last = -1.f;
        for (int z = 0; z < nz && few; ++z) {
            const float *row = q.data() + (size_t)z * p->qstride;
            for (int x = 0; x < nx; ++x) {
                const float v = row[x];
                if (v == last) continue;
                last = v;
                auto it = std::lower_bound(seen.begin(), seen.end(), v);
                if (it != seen.end() && *it == v) continue;
                seen.insert(it, v);
                if (seen.size() > cap) { few = false; break; }
            }
        }
        if (few) uq.swap(seen);
    }
    p->contiguous_rows = uq.empty() ? 1 : 0;
    std::vector<int> rowoff(nw + 1, 0), rows;
    p->max_rows = 0;
    for (int i = 0; i < nw; ++i) {
        size_t before = rows.size();
        if (p->contiguous_rows) {
            const int j0 = host_index(omega[i], qmin, ntab), j1 = host_index(omega[i], qmax, ntab);
            for (int j = j0; j <= j1; ++j) rows.push_back(j);
        } else {
            int last = -1;                                 // uq is sorted and the index is monotone in q
            for (float v : uq) {
                const int j = host_index(omega[i], v, ntab);
                if (j != last) { rows.push_back(j); last = j; }
            }
        }
        p->max_rows = std::max(p->max_rows, (int)(rows.size() - before));
        rowoff[i + 1] = (int)rows.size();
    }

    // ---- choose the kernel form ----------------------------------------------------------------------
    const unsigned want = p->flags & PDM_PATH_MASK;
    const unsigned want_taps = p->flags & PDM_TAPS_MASK;
    const bool have_L = Lk != 0;
    int HG = halo_groups(have_L ? Lk : L, R);
    int ngroups = (nx + R - 1) / R;
    int slots = (2 * HG + ngroups) * (R + 2);
    const int map_len = round_up(ntab, 8);                 // u16 row -> slot map, only with staged rows
    size_t line_bytes = (size_t)2 * slots * sizeof(float2);
    const size_t slice_bytes = (size_t)map_len * 2 + (size_t)p->max_rows * p->half16 * sizeof(float4);
    bool lines_fit = have_L && line_bytes <= (size_t)p->smem_optin;
    bool slice_fits = lines_fit && line_bytes + slice_bytes <= (size_t)p->smem_optin &&
                      p->max_rows <= 65535;

    // cluster form: C = 2, 4 or 8 CTAs per line (bits PDM_CTAS_SHIFT force it).  Among the sizes
    // whose per-CTA ping-pong segment fits shared memory, the largest that still leaves every CTA
    // >= 256 groups and keeps nw*C within one wave of SMs, else the smallest that fits.
    int cl_C = 0, cl_passes = 0, cl_nwarps = 0, cl_gper = 0;
    size_t cl_seg_bytes = 0;
    if (have_L) {
        const unsigned csel = (want == PDM_PATH_CLUSTER) ? ((p->flags >> PDM_CTAS_SHIFT) & 0xFu) : 0u;
        for (int c = 2; c <= 8; c *= 2) {
            if (csel && (int)csel != c) continue;
            const int gneed = (ngroups + c - 1) / c;
            const int ps = (gneed + PDM_MARCH_MAX_THREADS - 1) / PDM_MARCH_MAX_THREADS;
            const int nwp = (gneed + 32 * ps - 1) / (32 * ps);
            const int gp = 32 * ps * nwp;
            const size_t bytes = (size_t)2 * (2 * HG + gp) * (R + 2) * sizeof(float2);
            if (bytes > (size_t)p->smem_optin) continue;
            const bool wanted = (long long)nw * c <= p->sm_count && gneed >= 256;
            if (cl_C && !wanted) break;                    // keep the smaller size found before
            cl_C = c; cl_passes = ps; cl_nwarps = nwp; cl_gper = gp; cl_seg_bytes = bytes;
            if (!wanted) break;                            // smallest that fits
        }
    }
    const bool cl_slice_ok = cl_C && cl_seg_bytes + slice_bytes <= (size_t)p->smem_optin && p->max_rows <= 65535;
    // AUTO takes the cluster form when there are too few lines to give every SM a CTA (measured
    // 1.3-1.8x on configs[4] nw = 64 points with nx >= 4096) and the tap rows can still be staged
    const bool auto_cluster = cl_slice_ok && 2 * nw <= p->sm_count && ngroups >= 512 &&
                              (long long)nw * cl_C <= 2LL * p->sm_count;
    // ... and for lines that do not fit one CTA but do fit a PAIR (nx = 16384 with 51 taps or fewer),
    // when the tap rows can be staged and the lines fill the clusters' rounds: the wavefield then never
    // touches HBM (measured 1.05-1.2x over the x-tiled form at nw >= 1024; larger clusters lose SMs to
    // GPC fragmentation and stay with the x-tiled form)
    bool auto_pair = false;
    if (!lines_fit && cl_C == 2 && cl_slice_ok) {
        const int ncl = std::max(1, p->sm_count / 2);
        // per-sample-row models gain 1.19x from the pair at full rounds, warp-uniform ones nothing:
        // the former may waste up to 15 % of the last round and still win
        auto_pair = (double)nw / ((double)ncl * ((nw + ncl - 1) / ncl)) >= (p->contiguous_rows ? 0.85 : 0.95);
    }
    if (want == PDM_PATH_CLUSTER && !cl_C) return PDM_ERR_UNSUPPORTED;
    if (want == PDM_PATH_SMEM && !lines_fit) return PDM_ERR_UNSUPPORTED;
    if (want == PDM_PATH_TILED && !have_L) return PDM_ERR_UNSUPPORTED;  // (tiled_kernel_for has the same L list)
    if (want == PDM_PATH_PACKED && !have_L) return PDM_ERR_UNSUPPORTED;
    if (p->prestack || p->ntaper) {
        if (!have_L) return PDM_ERR_UNSUPPORTED;
        p->path = PDM_PATH_PACKED;
    } else if (p->flags & PDM_TABLE_INTERP)
        p->path = PDM_PATH_NAIVE;
    else if (want == PDM_PATH_AUTO)
        p->path = (auto_cluster || auto_pair) ? PDM_PATH_CLUSTER
                               : (lines_fit ? PDM_PATH_SMEM : (have_L ? PDM_PATH_TILED : PDM_PATH_NAIVE));
    else p->path = (int)want;
    if (p->path == PDM_PATH_SMEM && small) {               // the R = 4 build: redo the line layout
        R = PDM_R_SMALL;
        p->R = R;
        HG = halo_groups(Lk, R);
        ngroups = (nx + R - 1) / R;
        slots = (2 * HG + ngroups) * (R + 2);
        line_bytes = (size_t)2 * slots * sizeof(float2);
        lines_fit = line_bytes <= (size_t)p->smem_optin;
        slice_fits = lines_fit && line_bytes + slice_bytes <= (size_t)p->smem_optin && p->max_rows <= 65535;
        if (!lines_fit) return PDM_ERR_UNSUPPORTED;        // cannot happen for nx <= 1024; defensive
    }

    int rc;
    if ((rc = dev_upload(p, &p->d_omega, omega, (size_t)nw)) != PDM_OK) return rc;
    if ((rc = dev_upload(p, &p->d_q, q.data(), q.size())) != PDM_OK) return rc;

    // AUTO, models where (nearly) every sample has its own table row: the frequency-packed form makes the
    // tap gather bank-conflict free when the frequency list is dense against the table (adjacent lines at
    // most ~1 row apart) and replaces the x-tiled form in any case (measured on configs[4], field model:
    // 1.06-1.3x over the SMEM form at nx = 4096, 1.2-1.65x over the cluster-pair / x-tiled forms beyond)
    bool packed_done = false;
    if (want == PDM_PATH_AUTO && !p->prestack && !p->ntaper && have_L && p->sym && p->contiguous_rows) {
        float sigma = 0.f;                                  // table rows between adjacent lines of a pack
        for (int k = 0; k + 1 < nw; ++k)
            if ((k + 1) % PDM_PACK_W) sigma = std::max(sigma, fabsf(omega[k + 1] - omega[k]) * qmax);
        const bool dense = nw >= 2 * PDM_PACK_W && sigma <= 1.3f;
        const long long items = (long long)((nw + PDM_PACK_W - 1) / PDM_PACK_W) * ((nx + 447) / 448);
        // (sparse lists -- more than ~6 rows between adjacent lines -- keep the x-tiled form: 0.8-0.95x there)
        // dense lists, measured against the SMEM form (field model, nw = 1024 / 2048): 15 taps win from nx = 4096
        // (0.88x at 3072), longer filters from nx = 3072 (1.0-1.25x) and, with enough items per SM, from 2048
        const int min_nx = Lk <= 7 ? 4096 : 2048;
        const long long min_items = (long long)p->sm_count * (nx >= 3072 ? 3 : (Lk >= 25 ? 4 : 8));
        if ((p->path == PDM_PATH_TILED && sigma <= 6.f) || (dense && nx >= min_nx && items >= min_items)) {
            rc = build_packed(p, omega, q, half, Lk, HG);
            if (rc == PDM_OK) packed_done = true;
            else if (rc != PDM_ERR_UNSUPPORTED) return rc;
        }
    }
    if (packed_done) {
    } else if (p->path == PDM_PATH_SMEM) {
        if (want_taps == PDM_TAPS_SLICE || want_taps == PDM_TAPS_COMPACT) {
            if (!slice_fits) return PDM_ERR_UNSUPPORTED;
            p->taps_in_smem = 1;
        } else if (want_taps == PDM_TAPS_GLOBAL) p->taps_in_smem = 0;
        else p->taps_in_smem = slice_fits ? 1 : 0;
        p->taps_mode = p->taps_in_smem ? (p->contiguous_rows ? 2 : 3) : 1;

        const int max_threads = (R >= 8) ? PDM_MARCH_MAX_THREADS : 256;
        int passes = (ngroups + max_threads - 1) / max_threads;
        int threads = round_up((ngroups + passes - 1) / passes, 32);
        const unsigned tsel = (p->flags >> PDM_THREADS_SHIFT) & 0xFFu;
        if (tsel) {
            threads = std::min((int)tsel * 32, max_threads);
            passes = (ngroups + threads - 1) / threads;
        }
        p->threads = threads;
        p->smem_bytes = (int)(line_bytes + (p->taps_in_smem ? slice_bytes : 0));
        march_fn fn = march_kernel_for(p, p->taps_in_smem != 0, use_dedup(p), R);
        PDM_CUDA(p, cudaFuncSetAttribute((const void *)fn, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         p->smem_bytes));
        int per_sm = 0;
        PDM_CUDA(p, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void *)fn, threads,
                                                                  (size_t)p->smem_bytes));
        if (per_sm < 1) return PDM_ERR_UNSUPPORTED;
        const unsigned csel = (p->flags >> PDM_CTAS_SHIFT) & 0xFu;
        if (csel) per_sm = std::min(per_sm, (int)csel);
        p->ctas_per_sm = per_sm;
        p->grid = std::min(nw, p->sm_count * per_sm);
        p->launches = 2;
        p->n_partial = p->grid;
        {
            int coop = 0;
            PDM_CUDA(p, cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, p->device));
            // a line split needs T = nw*nz/grid >= nz (pieces are heads and tails only) and all
            // CTAs co-resident (cooperative launch); whole lines per CTA otherwise
            p->balanced = (!(p->flags & PDM_NO_BALANCE) && coop && nw > p->grid && nw % p->grid != 0) ? 1 : 0;
            std::vector<int4> segs; std::vector<int> segoff;
            build_segments(nw, nz, p->grid, p->balanced != 0, segs, segoff, p->nslots);
            if ((rc = dev_upload(p, &p->d_segs, segs.data(), segs.size())) != PDM_OK) return rc;
            if ((rc = dev_upload(p, &p->d_segoff, segoff.data(), segoff.size())) != PDM_OK) return rc;
            if ((rc = dev_alloc(p, &p->d_handoff, (size_t)std::max(1, p->nslots) * nx)) != PDM_OK) return rc;
            if ((rc = dev_alloc(p, &p->d_flags, (size_t)std::max(1, p->nslots))) != PDM_OK) return rc;
            PDM_CUDA(p, cudaMemset(p->d_flags, 0, (size_t)std::max(1, p->nslots) * sizeof(int)));
        }
        if ((rc = dev_upload(p, &p->d_half, half.data(), half.size())) != PDM_OK) return rc;
        if ((rc = dev_upload(p, &p->d_rowoff, rowoff.data(), rowoff.size())) != PDM_OK) return rc;
        if ((rc = dev_upload(p, &p->d_rows, rows.data(), rows.size())) != PDM_OK) return rc;
        if ((rc = dev_alloc(p, &p->d_partial, (size_t)p->n_partial * nz * (ngroups * R))) != PDM_OK) return rc;
        if ((rc = make_half_texture(p, half.size())) != PDM_OK) return rc;
    } else if (p->path == PDM_PATH_CLUSTER) {
        const int C = cl_C, passes = cl_passes, nwarps = cl_nwarps, gper = cl_gper;
        const size_t seg_bytes = cl_seg_bytes;
        const bool slice_ok = cl_slice_ok;
        if (want_taps == PDM_TAPS_SLICE || want_taps == PDM_TAPS_COMPACT) {
            if (!slice_ok) return PDM_ERR_UNSUPPORTED;
            p->taps_in_smem = 1;
        } else if (want_taps == PDM_TAPS_GLOBAL) p->taps_in_smem = 0;
        else p->taps_in_smem = slice_ok ? 1 : 0;
        p->taps_mode = p->taps_in_smem ? (p->contiguous_rows ? 2 : 3) : 1;
        p->threads = 32 * nwarps;
        p->cluster_size = C; p->cluster_gper = gper; p->cluster_passes = passes;
        p->smem_bytes = (int)(seg_bytes + (p->taps_in_smem ? slice_bytes : 0));
        cluster_fn fn = cluster_kernel_for(p, p->taps_in_smem != 0, use_dedup(p));
        PDM_CUDA(p, cudaFuncSetAttribute((const void *)fn, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         p->smem_bytes));
        int max_clusters = 0;
        {
            cudaLaunchConfig_t cfg = {};
            cudaLaunchAttribute at[1];
            at[0].id = cudaLaunchAttributeClusterDimension;
            at[0].val.clusterDim.x = C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
            cfg.gridDim = dim3(C * p->sm_count); cfg.blockDim = dim3(p->threads);
            cfg.dynamicSmemBytes = (size_t)p->smem_bytes; cfg.attrs = at; cfg.numAttrs = 1;
            PDM_CUDA(p, cudaOccupancyMaxActiveClusters(&max_clusters, (const void *)fn, &cfg));
        }
        if (max_clusters < 1) return PDM_ERR_UNSUPPORTED;
        p->ctas_per_sm = 1;
        p->n_partial = std::min(nw, max_clusters);
        p->grid = p->n_partial * C;
        p->launches = 2;
        if ((rc = dev_upload(p, &p->d_half, half.data(), half.size())) != PDM_OK) return rc;
        if ((rc = dev_upload(p, &p->d_rowoff, rowoff.data(), rowoff.size())) != PDM_OK) return rc;
        if ((rc = dev_upload(p, &p->d_rows, rows.data(), rows.size())) != PDM_OK) return rc;
        if ((rc = dev_alloc(p, &p->d_partial, (size_t)p->n_partial * nz * (ngroups * R))) != PDM_OK) return rc;
        if ((rc = make_half_texture(p, half.size())) != PDM_OK) return rc;
    } else if (p->path == PDM_PATH_TILED) {
        p->taps_mode = 1;
        p->threads = PDM_TILED_THREADS;
        p->tile_x = PDM_TILED_THREADS * R;
        const int xtiles = (nx + p->tile_x - 1) / p->tile_x;
        // per warp: double-buffered input sub-tile (+ halos) and an output sub-tile (unless aliased)
        p->smem_bytes = (PDM_TILED_THREADS / 32) * (PDM_TILED_STAGES * (32 + 2 * HG) + (tiled_alias(p) ? 0 : 32)) * (R + 2) * (int)sizeof(float2);
        int per_sm = 0;
        for (int wide = 0; wide < 2; ++wide) {
            tiled_fn fn = tiled_kernel_for(p, wide != 0);
            PDM_CUDA(p, cudaFuncSetAttribute((const void *)fn, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             p->smem_bytes));
            PDM_CUDA(p, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void *)fn,
                                                                      PDM_TILED_THREADS, (size_t)p->smem_bytes));
        }
        if (per_sm < 1) return PDM_ERR_UNSUPPORTED;
        p->ctas_per_sm = per_sm;
        // Two depth steps per launch (pdm_tiled_step2) where the one-step kernel is HBM-bound: short
        // filters (halo <= 2 groups) on warp-uniform models; bits 16-19 force 1 or 2 steps per launch
        int xt = xtiles;
        {
            const unsigned tsel = (want == PDM_PATH_TILED) ? (p->flags >> PDM_CTAS_SHIFT) & 0xFu : 0u;
            if (tsel > 2) return PDM_ERR_UNSUPPORTED;
            const bool can2 = Lk <= 15 && nz >= 2;
            if (tsel == 2 && !can2) return PDM_ERR_UNSUPPORTED;
            // measured (layers, nx = 16384 / 32768): 15 taps 1.04-1.2x, 25 taps 0.92-0.95x -> AUTO only up to L = 7
            if (can2 && (tsel == 2 || (tsel == 0 && !p->contiguous_rows && Lk <= 7))) {
                const int keep = 32 - 2 * HG;
                p->tile_x2 = (PDM_TILED_THREADS / 32) * keep * R;
                p->smem_bytes2 = (PDM_TILED_THREADS / 32) * ((PDM_TILED_STAGES + 1) * (32 + 2 * HG) + 32) * (R + 2) * (int)sizeof(float2);
                int per_sm2 = 0;
                for (int wide = 0; wide < 2; ++wide) {
                    tiled_fn fn2 = pdm_tiled2_kernel_for(Lk, wide != 0, p->sym != 0);
                    if (!fn2) return PDM_ERR_UNSUPPORTED;
                    PDM_CUDA(p, cudaFuncSetAttribute((const void *)fn2, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                     p->smem_bytes2));
                    PDM_CUDA(p, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm2, (const void *)fn2,
                                                                              PDM_TILED_THREADS, (size_t)p->smem_bytes2));
                }
                if (per_sm2 >= 1) {
                    p->tiled_T2 = 1;
                    per_sm = per_sm2;
                    p->ctas_per_sm = per_sm2;
                    xt = (nx + p->tile_x2 - 1) / p->tile_x2;
                }
            }
        }
        // ONE resident wave per depth step: x-tiles x frequency groups <= SMs x CTAs per SM
        int wgroups = std::max(1, std::min(nw, p->sm_count * per_sm / xt));
        const int wpg = (nw + wgroups - 1) / wgroups;
        wgroups = (nw + wpg - 1) / wpg;
        p->wgroups = wgroups;
        p->grid = xt * wgroups;
        p->launches = (p->tiled_T2 ? nz / 2 + (nz & 1) : nz) + 1;
        p->n_partial = wgroups;
        if ((rc = dev_upload(p, &p->d_half, half.data(), half.size())) != PDM_OK) return rc;
        if ((rc = dev_alloc(p, &p->d_partial, (size_t)wgroups * nz * p->qstride)) != PDM_OK) return rc;
        if ((rc = dev_alloc(p, &p->d_plane[0], (size_t)nw * nx)) != PDM_OK) return rc;
        if ((rc = dev_alloc(p, &p->d_plane[1], (size_t)nw * nx)) != PDM_OK) return rc;
    } else if (p->path == PDM_PATH_PACKED) {
        if ((rc = build_packed(p, omega, q, half, Lk, HG)) != PDM_OK) return rc;
    } else {                                                        // PDM_PATH_NAIVE
        p->taps_mode = 1;
        p->threads = 128;
        p->grid = ((nx + 127) / 128) * nw;
        p->launches = 2 * nz;
        if ((rc = dev_upload(p, &p->d_table, reinterpret_cast<const float2 *>(table),
                             (size_t)ntab * ntaps)) != PDM_OK) return rc;
        if ((rc = dev_alloc(p, &p->d_plane[0], (size_t)nw * nx)) != PDM_OK) return rc;
        if ((rc = dev_alloc(p, &p->d_plane[1], (size_t)nw * nx)) != PDM_OK) return rc;
    }
    return PDM_OK;
}

// ------------------------------------------------------------------------------------------------
// pdm_migrate: enqueue only -- no allocation, no host sync, no copies (CUDA-graph capturable)
// ------------------------------------------------------------------------------------------------
static int migrate_impl(pdm_plan *p, const pdm_c64 *P0_dev, const pdm_c64 *src_dev, float *image_dev,
                        int accumulate, void *cuda_stream);

extern "C" int pdm_migrate(pdm_plan *p, const pdm_c64 *P0_dev, float *image_dev, void *cuda_stream)
{
    if (!p || !P0_dev || !image_dev || p->prestack) return PDM_ERR_INVALID_ARG;
    return migrate_impl(p, P0_dev, nullptr, image_dev, 0, cuda_stream);
}

// P0_dev: the poststack section, or (src_dev != NULL) the receiver field of a prestack shot
static int migrate_impl(pdm_plan *p, const pdm_c64 *P0_dev, const pdm_c64 *src_dev, float *image_dev,
                        int accumulate, void *cuda_stream)
{
    int dev = -1;
    PDM_CUDA(p, cudaGetDevice(&dev));
    if (dev != p->device) { p->last_cuda_error = (int)cudaErrorInvalidDevice; return PDM_ERR_CUDA; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int nx = p->nx, nz = p->nz, nw = p->nw, L = p->L, Lk = p->Lk, R = p->R;
    const float2 *P0 = reinterpret_cast<const float2 *>(P0_dev);

    if (p->path == PDM_PATH_SMEM) {
        pdm_march_params a;
        a.P0 = P0; a.partial = p->d_partial; a.q = p->d_q; a.omega = p->d_omega;
        a.half = p->d_half; a.rowoff = p->d_rowoff; a.rows = p->d_rows; a.tex = p->tex_half;
        a.segs = p->d_segs; a.segoff = p->d_segoff; a.handoff = p->d_handoff; a.flags = p->d_flags;
        a.nx = nx; a.nz = nz; a.nw = nw; a.ntab = p->ntab;
        a.ngroups = (nx + R - 1) / R;
        a.qstride = p->qstride; a.pstride = a.ngroups * R; a.half16 = p->half16;
        a.passes = (a.ngroups + p->threads - 1) / p->threads;
        a.slots = (2 * halo_groups(Lk, R) + a.ngroups) * (R + 2);
        a.map_len = round_up(p->ntab, 8);
        a.force_general = (p->flags & PDM_FORCE_GENERAL) ? 1 : 0;
        march_fn fn = march_kernel_for(p, p->taps_in_smem != 0, use_dedup(p), R);
        if (p->profiling) PDM_CUDA(p, cudaEventRecord(p->ev[0], st));
        if (p->balanced) {                               // split lines: CTAs wait on one another
            // hand-off flags start empty even if an earlier migrate on this plan was cut short
            PDM_CUDA(p, cudaMemsetAsync(p->d_flags, 0, (size_t)std::max(1, p->nslots) * sizeof(int), st));
            void *args[] = { (void *)&a };
            PDM_CUDA(p, cudaLaunchCooperativeKernel((const void *)fn, dim3(p->grid), dim3(p->threads),
                                                    args, (size_t)p->smem_bytes, st));
        } else {
            fn<<<p->grid, p->threads, p->smem_bytes, st>>>(a);
        }
        PDM_CUDA(p, cudaGetLastError());
        if (p->profiling) PDM_CUDA(p, cudaEventRecord(p->ev[1], st));
        dim3 rg((nx + 255) / 256, nz);
        pdm_reduce_partials<<<rg, 256, 0, st>>>(p->d_partial, image_dev, p->n_partial, nz, nx, a.pstride);
        PDM_CUDA(p, cudaGetLastError());
    } else if (p->path == PDM_PATH_CLUSTER) {
        pdm_cluster_params a;
        a.P0 = P0; a.partial = p->d_partial; a.q = p->d_q; a.omega = p->d_omega;
        a.half = p->d_half; a.rowoff = p->d_rowoff; a.rows = p->d_rows;
        a.nx = nx; a.nz = nz; a.nw = nw; a.ntab = p->ntab;
        a.ngroups = (nx + R - 1) / R;
        a.qstride = p->qstride; a.pstride = a.ngroups * R; a.half16 = p->half16;
        a.passes = p->cluster_passes; a.gper = p->cluster_gper;
        a.slots = (2 * halo_groups(Lk, R) + a.gper) * (R + 2);
        a.map_len = round_up(p->ntab, 8);
        a.force_general = (p->flags & PDM_FORCE_GENERAL) ? 1 : 0;
        a.nclusters = p->n_partial;
        a.tex = p->tex_half;
        cluster_fn fn = cluster_kernel_for(p, p->taps_in_smem != 0, use_dedup(p));
        cudaLaunchConfig_t cfg = {};
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = p->cluster_size; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.gridDim = dim3(p->grid); cfg.blockDim = dim3(p->threads);
        cfg.dynamicSmemBytes = (size_t)p->smem_bytes; cfg.stream = st; cfg.attrs = at; cfg.numAttrs = 1;
        if (p->profiling) PDM_CUDA(p, cudaEventRecord(p->ev[0], st));
        PDM_CUDA(p, cudaLaunchKernelEx(&cfg, fn, a));
        if (p->profiling) PDM_CUDA(p, cudaEventRecord(p->ev[1], st));
        dim3 rg((nx + 255) / 256, nz);
        pdm_reduce_partials<<<rg, 256, 0, st>>>(p->d_partial, image_dev, p->n_partial, nz, nx, a.pstride);
        PDM_CUDA(p, cudaGetLastError());
    } else if (p->path == PDM_PATH_TILED) {
        pdm_tiled_params a;
        a.partial = p->d_partial; a.q = p->d_q; a.omega = p->d_omega; a.half = p->d_half;
        a.nx = nx; a.nz = nz; a.nw = nw; a.ntab = p->ntab;
        a.qstride = p->qstride; a.pstride = p->qstride; a.half16 = p->half16;
        a.w_per_group = (nw + p->wgroups - 1) / p->wgroups;
        a.force_general = (p->flags & PDM_FORCE_GENERAL) ? 1 : 0;
        // 16-byte async copies need every plane row 16-byte aligned: nx even and an aligned P0
        const bool wide = (nx % 2 == 0) && (((uintptr_t)P0_dev & 15u) == 0);
        tiled_fn fn = tiled_kernel_for(p, wide);
        dim3 grid((nx + p->tile_x - 1) / p->tile_x, p->wgroups);
        const float2 *src = P0;
        if (p->profiling) PDM_CUDA(p, cudaEventRecord(p->ev[0], st));
        if (p->tiled_T2) {                               // two depth steps per launch; an odd last step alone
            tiled_fn fn2 = pdm_tiled2_kernel_for(Lk, wide, p->sym != 0);
            dim3 grid2((nx + p->tile_x2 - 1) / p->tile_x2, p->wgroups);
            int k = 0;
            for (int z = 0; z + 1 < nz; z += 2, ++k) {
                a.z = z; a.Pin = src; a.Pout = p->d_plane[k & 1];
                fn2<<<grid2, PDM_TILED_THREADS, p->smem_bytes2, st>>>(a);
                src = a.Pout;
            }
            if (nz & 1) {
                a.z = nz - 1; a.Pin = src; a.Pout = p->d_plane[k & 1];
                fn<<<grid, PDM_TILED_THREADS, p->smem_bytes, st>>>(a);
            }
        } else
        for (int z = 0; z < nz; ++z) {
            a.z = z; a.Pin = src; a.Pout = p->d_plane[z & 1];
            fn<<<grid, PDM_TILED_THREADS, p->smem_bytes, st>>>(a);
            src = a.Pout;
        }
        PDM_CUDA(p, cudaGetLastError());
        if (p->profiling) PDM_CUDA(p, cudaEventRecord(p->ev[1], st));
        dim3 rg((nx + 255) / 256, nz);
        pdm_reduce_partials<<<rg, 256, 0, st>>>(p->d_partial, image_dev, p->n_partial, nz, nx, a.pstride);
        PDM_CUDA(p, cudaGetLastError());
    } else if (p->path == PDM_PATH_PACKED) {
        pdm_pack_params a;
        memset(&a, 0, sizeof(a));
        a.tmap_plane[0] = p->tmap_plane[0]; a.tmap_plane[1] = p->tmap_plane[1];
        a.plane[0] = p->d_plane[0]; a.plane[1] = p->d_plane[1];
        a.partial = p->d_partial; a.image = image_dev;
        a.q = p->d_q; a.omega = p->d_omega; a.half = p->d_half;
        a.packw = p->d_packw; a.tileq = p->d_tileq; a.tile_ctas = p->d_tile_ctas;
        a.gbar = reinterpret_cast<unsigned *>(p->d_flags);
        a.nx = nx; a.nxp = p->nxp; a.nz = nz; a.nw = nw; a.ntab = p->ntab;
        a.qstride = p->qstride; a.half16 = p->half16;
        a.npacks = p->pk_npacks; a.ntiles = p->pk_ntiles; a.nitems = p->pk_ntiles * p->pk_npacks;
        a.TX = p->pk_TX; a.H = p->pk_H; a.T = p->pk_T;
        a.LS = p->pk_LS; a.BW = p->pk_BW; a.nbox = p->pk_nbox; a.cap = p->pk_cap; a.passes = p->pk_passes;
        a.force_general = (p->flags & PDM_FORCE_GENERAL) ? 1 : 0;
        pack_fn fn = pack_kernel_for(p);
        // the first depth block reads the caller's P0 through its own TMA descriptor when its rows are
        // 16-byte aligned (nx even and an aligned base); otherwise P0 is first repacked into a plane
        a.xcorr = p->prestack; a.accumulate = accumulate;
        a.ntaper = p->ntaper; a.taper = p->d_taper;
        if (p->prestack) {                               // (receiver, conj source) line pairs into plane 1
            dim3 cg((p->nxp + 255) / 256, nw / 2);
            pdm_pack_interleave<<<cg, 256, 0, st>>>(P0, reinterpret_cast<const float2 *>(src_dev), p->d_plane[1],
                                                    nx, p->nxp, nw / 2);
            a.tmap_p0 = p->tmap_plane[1];
            a.first_src = 1;
        } else if (nx % 2 == 0 && ((uintptr_t)P0_dev & 15u) == 0) {
            int rc = make_plane_map(p, &a.tmap_p0, P0_dev, nx, nw, p->pk_BW);
            if (rc != PDM_OK) return rc;
            a.first_src = -1;
        } else {
            dim3 cg((p->nxp + 255) / 256, nw);
            pdm_pack_copy_in<<<cg, 256, 0, st>>>(P0, p->d_plane[1], nx, p->nxp, nw);
            a.tmap_p0 = p->tmap_plane[1];
            a.first_src = 1;
        }
        // one launch for all depth blocks: the CTAs synchronise between blocks on a counter in global
        // memory (cooperative launch = all co-resident), zeroed on the stream first
        PDM_CUDA(p, cudaMemsetAsync(p->d_flags, 0, sizeof(int), st));
        if (p->profiling) PDM_CUDA(p, cudaEventRecord(p->ev[0], st));
        void *args[] = { (void *)&a };
        PDM_CUDA(p, cudaLaunchCooperativeKernel((const void *)fn, dim3(p->grid), dim3(p->threads), args,
                                                (size_t)p->smem_bytes, st));
        if (p->profiling) PDM_CUDA(p, cudaEventRecord(p->ev[1], st));
    } else {
        dim3 g1((nx + 127) / 128, nw), g2((nx + 127) / 128);
        const float2 *src = P0;
        if (p->profiling) {                              // scaffold: K1+K2 interleaved, all "main"
            PDM_CUDA(p, cudaEventRecord(p->ev[0], st));
        }
        for (int z = 0; z < nz; ++z) {
            float2 *dst = p->d_plane[z & 1];
            if (p->flags & PDM_TABLE_INTERP)
                pdm_naive_step_interp<<<g1, 128, 0, st>>>(src, dst, p->d_omega, p->d_q + (size_t)z * p->qstride,
                                                           p->d_table, nx, nw, p->ntab, L);
            else
                pdm_naive_step<<<g1, 128, 0, st>>>(src, dst, p->d_omega, p->d_q + (size_t)z * p->qstride,
                                                    p->d_table, nx, nw, p->ntab, L);
            pdm_naive_image_row<<<g2, 128, 0, st>>>(dst, image_dev + (size_t)z * nx, nx, nw);
            src = dst;
        }
        PDM_CUDA(p, cudaGetLastError());
        if (p->profiling) PDM_CUDA(p, cudaEventRecord(p->ev[1], st));
    }
    if (p->profiling) { PDM_CUDA(p, cudaEventRecord(p->ev[2], st)); p->profiled = 1; }
    return PDM_OK;
}

extern "C" int pdm_migrate_shot(pdm_plan *p, const pdm_c64 *src_dev, const pdm_c64 *rec_dev, float *image_dev,
                                int accumulate, void *cuda_stream)
{
    if (!p || !src_dev || !rec_dev || !image_dev || !p->prestack) return PDM_ERR_INVALID_ARG;
    return migrate_impl(p, rec_dev, src_dev, image_dev, accumulate ? 1 : 0, cuda_stream);
}

extern "C" int pdm_profile_enable(pdm_plan *p, int enable)
{
    if (!p) return PDM_ERR_INVALID_ARG;
    if (enable && !p->ev[0])
        for (int i = 0; i < 3; ++i) PDM_CUDA(p, cudaEventCreate(&p->ev[i]));
    p->profiling = enable ? 1 : 0;
    p->profiled = 0;
    return PDM_OK;
}

extern "C" int pdm_profile_read(pdm_plan *p, float *main_ms, float *reduce_ms)
{
    if (!p || !main_ms || !reduce_ms || !p->profiling || !p->profiled) return PDM_ERR_INVALID_ARG;
    PDM_CUDA(p, cudaEventSynchronize(p->ev[2]));
    PDM_CUDA(p, cudaEventElapsedTime(main_ms, p->ev[0], p->ev[1]));
    PDM_CUDA(p, cudaEventElapsedTime(reduce_ms, p->ev[1], p->ev[2]));
    return PDM_OK;
}

extern "C" int pdm_migrate_host(pdm_plan *p, const pdm_c64 *P0_host, float *image_host, void *cuda_stream)
{
    if (!p || !P0_host || !image_host || p->prestack) return PDM_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t nP = (size_t)p->nw * p->nx, nI = (size_t)p->nz * p->nx;
    // Main form with PINNED host buffers: the kernels read P0 and write the image straight through the
    // host mapping (each byte crosses the link once either way, but inside the marching / reduction
    // kernels, overlapped with their work, instead of in two serial copies around them)
    if (p->path == PDM_PATH_SMEM) {
        cudaPointerAttributes ai, ao;
        if (cudaPointerGetAttributes(&ai, P0_host) == cudaSuccess && cudaPointerGetAttributes(&ao, image_host) == cudaSuccess &&
            ai.type == cudaMemoryTypeHost && ao.type == cudaMemoryTypeHost && ai.devicePointer && ao.devicePointer) {
            int rc = pdm_migrate(p, (const pdm_c64 *)ai.devicePointer, (float *)ao.devicePointer, cuda_stream);
            if (rc != PDM_OK) return rc;
            PDM_CUDA(p, cudaStreamSynchronize(st));
            return PDM_OK;
        }
        cudaGetLastError();
    }
    if (!p->d_stage_p0) {
        int rc;
        if ((rc = dev_alloc(p, &p->d_stage_p0, nP)) != PDM_OK) return rc;
        if ((rc = dev_alloc(p, &p->d_stage_img, nI)) != PDM_OK) return rc;
    }
    PDM_CUDA(p, cudaMemcpyAsync(p->d_stage_p0, P0_host, nP * sizeof(pdm_c64), cudaMemcpyHostToDevice, st));
    int rc = pdm_migrate(p, p->d_stage_p0, p->d_stage_img, cuda_stream);
    if (rc != PDM_OK) return rc;
    PDM_CUDA(p, cudaMemcpyAsync(image_host, p->d_stage_img, nI * sizeof(float), cudaMemcpyDeviceToHost, st));
    PDM_CUDA(p, cudaStreamSynchronize(st));
    return PDM_OK;
}

extern "C" int pdm_destroy(pdm_plan *p)
{
    free_plan(p);
    return PDM_OK;
}

extern "C" int pdm_get_info(const pdm_plan *p, pdm_info *out)
{
    if (!p || !out) return PDM_ERR_INVALID_ARG;
    memset(out, 0, sizeof(*out));
    out->path = p->path; out->taps_mode = p->taps_mode;
    out->nx = p->nx; out->nz = p->nz; out->nw = p->prestack ? p->nw / 2 : p->nw; out->ntab = p->ntab; out->ntaps = p->ntaps;
    out->grid_ctas = p->grid; out->threads_per_cta = p->threads; out->ctas_per_sm = p->ctas_per_sm;
    out->smem_bytes = p->smem_bytes; out->launches_per_migrate = p->launches;
    out->sm_count = p->sm_count; out->last_cuda_error = p->last_cuda_error;
    out->samples = (double)p->nx * (double)p->nz * (double)p->nw;
    out->counted_flops = 8.0 * p->ntaps * out->samples;
    out->executed_lane_ops = ((p->sym ? 6.0 : 8.0) * (p->Lk ? p->Lk : p->L) + 4.0) * out->samples;   // zero-padded taps are executed too
    out->table_symmetric = p->sym;
    out->workspace_bytes = p->workspace_bytes;
    return PDM_OK;
}

// ------------------------------------------------------------------------------------------------
// debug / measurement entry points
// ------------------------------------------------------------------------------------------------
__global__ void pdm_debug_index_kernel(const float *w, const float *q, int n, int ntab, int *out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = pdm_index(w[i], q[i], ntab - 1);
}

extern "C" int pdm_debug_table_index(const float *omega, const float *velocity, int n,
                                     double dz, double tab_du, int ntab, int *idx_out)
{
    if (!omega || !velocity || !idx_out || n <= 0 || ntab <= 0 || !(tab_du > 0.0)) return PDM_ERR_INVALID_ARG;
    std::vector<float> q(n);
    for (int i = 0; i < n; ++i) q[i] = host_q(dz, velocity[i], tab_du);
    float *dw = nullptr, *dq = nullptr; int *di = nullptr;
    int rc = PDM_ERR_CUDA;
    if (cudaMalloc(&dw, n * sizeof(float)) == cudaSuccess && cudaMalloc(&dq, n * sizeof(float)) == cudaSuccess &&
        cudaMalloc(&di, n * sizeof(int)) == cudaSuccess &&
        cudaMemcpy(dw, omega, n * sizeof(float), cudaMemcpyHostToDevice) == cudaSuccess &&
        cudaMemcpy(dq, q.data(), n * sizeof(float), cudaMemcpyHostToDevice) == cudaSuccess) {
        pdm_debug_index_kernel<<<(n + 255) / 256, 256>>>(dw, dq, n, ntab, di);
        if (cudaMemcpy(idx_out, di, n * sizeof(int), cudaMemcpyDeviceToHost) == cudaSuccess) rc = PDM_OK;
    }
    cudaFree(dw); cudaFree(dq); cudaFree(di);
    if (rc != PDM_OK) cudaGetLastError();
    return rc;
}

extern "C" int pdm_fp32_peak(int packed, int iters, int repeats, void *cuda_stream, double *tflops_out)
{
    if (!tflops_out || iters <= 0 || repeats <= 0) return PDM_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return PDM_ERR_UNSUPPORTED;
    }
    float *d = nullptr;
    cudaEvent_t e0, e1;
    if (cudaMalloc(&d, 256) != cudaSuccess) return PDM_ERR_NOMEM;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int grid = sms * 8, block = 256;
    double best_ms = 1e30;
    for (int r = 0; r < repeats + 1; ++r) {                 // first run is the warm-up
        cudaEventRecord(e0, st);
        if (packed) pdm_peak_kernel<1><<<grid, block, 0, st>>>(d, iters, 1.0f);
        else        pdm_peak_kernel<0><<<grid, block, 0, st>>>(d, iters, 1.0f);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaGetLastError(); cudaFree(d); return PDM_ERR_CUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms < best_ms) best_ms = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
    const double flops = (double)grid * block * (double)iters * PDM_PEAK_CHAINS * 2.0 * 2.0;
    *tflops_out = flops / (best_ms * 1e-3) / 1e12;
    return PDM_OK;
}

// ------------------------------------------------------------------------------------------------
// time -> frequency transform of the input section
// ------------------------------------------------------------------------------------------------
#include "kern_tf.cuh"
#include "kern_fft.cuh"

struct pdm_tf {
    int nt, nx, nw, device, smem_bytes, warps;
    int *d_bins;
    float2 *d_tw;
    // nt a power of two: real FFT per trace (kern_fft.cuh); else the contraction (kern_tf.cuh)
    int fft, log2nt, fft_S, fft_ntw, fft_smem, fft_grid;
    float2 *d_ftw;
    int2 *d_binpos;
};

extern "C" int pdm_tf_destroy(pdm_tf *tf)
{
    if (!tf) return PDM_OK;
    cudaFree(tf->d_bins); cudaFree(tf->d_tw); cudaFree(tf->d_ftw); cudaFree(tf->d_binpos);
    delete tf;
    return PDM_OK;
}

extern "C" int pdm_tf_create(pdm_tf **out, int nt, int nx, int nw, const int *bins)
{
    if (!out) return PDM_ERR_INVALID_ARG;
    *out = nullptr;
    if (!bins || nt <= 0 || nx <= 0 || nw <= 0) return PDM_ERR_INVALID_ARG;
    for (int j = 0; j < nw; ++j)
        if (bins[j] < 0 || bins[j] > nt / 2) return PDM_ERR_INVALID_ARG;
    if (nt > PDM_TF_MAX_NT || (double)nw * (double)nx > 2.0e9 || (double)nt * (double)nx > 8.0e9)
        return PDM_ERR_UNSUPPORTED;
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        cudaGetLastError();
        return PDM_ERR_UNSUPPORTED;                        // no usable CUDA device: no fallback
    }
    if (prop.major != 10) return PDM_ERR_UNSUPPORTED;
    pdm_tf *tf = new (std::nothrow) pdm_tf();
    if (!tf) return PDM_ERR_NOMEM;
    memset(tf, 0, sizeof(*tf));
    tf->nt = nt; tf->nx = nx; tf->nw = nw; tf->device = dev;
    tf->smem_bytes = ((nt + 1) & ~1) * (int)sizeof(float2) + 2 * PDM_TF_NC * PDM_TF_XB * (int)sizeof(float) +
                     2 * (PDM_TF_THREADS / 32) * PDM_TF_JT * PDM_TF_NC * (int)sizeof(float2);
    std::vector<float2> tw(nt);
    const double two_pi = 6.283185307179586476925286766559;
    for (int m = 0; m < nt; ++m) {                         // exact argument, one rounding to FP32
        const double a = two_pi * (double)m / (double)nt;
        tw[m] = make_float2((float)cos(a), (float)(-sin(a)));
    }
    bool ok = cudaMalloc((void **)&tf->d_bins, (size_t)nw * sizeof(int)) == cudaSuccess &&
              cudaMalloc((void **)&tf->d_tw, (size_t)nt * sizeof(float2)) == cudaSuccess &&
              cudaMemcpy(tf->d_bins, bins, (size_t)nw * sizeof(int), cudaMemcpyHostToDevice) == cudaSuccess &&
              cudaMemcpy(tf->d_tw, tw.data(), (size_t)nt * sizeof(float2), cudaMemcpyHostToDevice) == cudaSuccess &&
              cudaFuncSetAttribute((const void *)pdm_tf_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   tf->smem_bytes) == cudaSuccess &&
              cudaFuncSetAttribute((const void *)pdm_tf_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   tf->smem_bytes) == cudaSuccess;
    if (!ok) { cudaGetLastError(); pdm_tf_destroy(tf); return PDM_ERR_CUDA; }
    if (nt >= 4 && (nt & (nt - 1)) == 0) {                 // power of two: FFT form
        int lg = 0;
        while ((1 << lg) < nt) ++lg;
        std::vector<float2> ftw;                           // per radix-4 stage: (w^j, w^2j, w^3j), w = exp(-2 pi i / M)
        for (int lm = lg; lm >= 2; lm -= 2) {
            const int M = 1 << lm, q = M / 4;
            for (int j = 0; j < q; ++j)
                for (int r = 1; r <= 3; ++r) {
                    const double a = two_pi * (double)((long long)r * j % M) / (double)M;
                    ftw.push_back(make_float2((float)cos(a), (float)(-sin(a))));
                }
        }
        if (ftw.empty()) ftw.push_back(make_float2(1.f, 0.f));
        const size_t np = (size_t)nt + (nt >> 4) + 1;
        int S = 16;                                        // pairs of traces per CTA: as many as fit ~160 KB
        while (S > 1 && (S * np + ftw.size()) * sizeof(float2) > (size_t)160 * 1024) S >>= 1;
        while (S > 1 && S / 2 >= (nx + 1) / 2) S >>= 1;    // no more pairs than the section has
        const size_t smem = (S * np + ftw.size()) * sizeof(float2);
        // where the in-place DIF leaves bin k: radix-4 digits reversed, then the radix-2 bit; padded index
        auto pos_of = [&](int k) {
            int pos = 0, rem = lg;
            while (rem >= 2) { rem -= 2; pos += (k & 3) << rem; k >>= 2; }
            if (rem == 1) pos += k & 1;
            return pos + (pos >> 4);
        };
        std::vector<int2> binpos(nw);
        for (int j = 0; j < nw; ++j) binpos[j] = make_int2(pos_of(bins[j]), pos_of((nt - bins[j]) & (nt - 1)));
        if (smem <= (size_t)prop.sharedMemPerBlockOptin - 1024 &&
            cudaMalloc((void **)&tf->d_binpos, (size_t)nw * sizeof(int2)) == cudaSuccess &&
            cudaMemcpy(tf->d_binpos, binpos.data(), (size_t)nw * sizeof(int2), cudaMemcpyHostToDevice) == cudaSuccess &&
            cudaMalloc((void **)&tf->d_ftw, ftw.size() * sizeof(float2)) == cudaSuccess &&
            cudaMemcpy(tf->d_ftw, ftw.data(), ftw.size() * sizeof(float2), cudaMemcpyHostToDevice) == cudaSuccess &&
            cudaFuncSetAttribute((const void *)pdm_fft_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)smem) == cudaSuccess) {
            tf->fft = 1; tf->log2nt = lg; tf->fft_S = S; tf->fft_ntw = (int)ftw.size(); tf->fft_smem = (int)smem;
            int per_sm = 1;                                // persistent CTAs: the twiddle tables are loaded once each
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void *)pdm_fft_kernel, PDM_FFT_THREADS,
                                                              smem) != cudaSuccess || per_sm < 1) { cudaGetLastError(); per_sm = 1; }
            tf->fft_grid = prop.multiProcessorCount * per_sm;
        } else {
            cudaGetLastError();                            // fall through to the contraction form
        }
    }
    // warps per CTA (4 bins each): all tiles take the same time, so pick the CTA height that wastes
    // the least of the last wave
    double best = -1.0;
    const int xtiles = (nx + PDM_TF_XB - 1) / PDM_TF_XB;
    for (int w = 8; w >= 4; --w) {
        int per_sm = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void *)pdm_tf_kernel<4>, 32 * w,
                                                          (size_t)tf->smem_bytes) != cudaSuccess || per_sm < 1)
            continue;
        const long long tiles = (long long)xtiles * ((nw + 4 * w - 1) / (4 * w));
        const long long slots = (long long)prop.multiProcessorCount * per_sm;
        const double eff = (double)nw * xtiles / (4.0 * w) / (double)(slots * ((tiles + slots - 1) / slots))
                           * (w * per_sm >= 12 ? 1.0 : 0.8);      // fewer than 12 warps per SM: latency-bound
        if (eff > best) { best = eff; tf->warps = w; }
    }
    if (best < 0.0) { cudaGetLastError(); pdm_tf_destroy(tf); return PDM_ERR_UNSUPPORTED; }
    *out = tf;
    return PDM_OK;
}

extern "C" int pdm_tf_forward(pdm_tf *tf, const float *section_dev, pdm_c64 *P0_dev, void *cuda_stream)
{
    if (!tf || !section_dev || !P0_dev) return PDM_ERR_INVALID_ARG;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != tf->device) { cudaGetLastError(); return PDM_ERR_CUDA; }
    if (tf->fft) {
        pdm_fft_params f;
        f.section = section_dev; f.out = reinterpret_cast<float2 *>(P0_dev);
        f.binpos = tf->d_binpos; f.tw = tf->d_ftw;
        f.nt = tf->nt; f.log2nt = tf->log2nt; f.nx = tf->nx; f.nw = tf->nw;
        f.S = tf->fft_S; f.ntw = tf->fft_ntw;
        f.pair_loads = (tf->nx % 2 == 0 && ((uintptr_t)section_dev & 7u) == 0) ? 1 : 0;
        f.wide_out = (tf->nx % 2 == 0 && ((uintptr_t)P0_dev & 15u) == 0) ? 1 : 0;
        const int per_cta = 2 * tf->fft_S;
        const int ntiles = (tf->nx + per_cta - 1) / per_cta;
        pdm_fft_kernel<<<std::min(ntiles, tf->fft_grid), PDM_FFT_THREADS, tf->fft_smem, (cudaStream_t)cuda_stream>>>(f);
        if (cudaGetLastError() != cudaSuccess) return PDM_ERR_CUDA;
        return PDM_OK;
    }
    pdm_tf_params a;
    a.section = section_dev; a.out = reinterpret_cast<float2 *>(P0_dev);
    a.bins = tf->d_bins; a.tw = tf->d_tw; a.nt = tf->nt; a.nx = tf->nx; a.nw = tf->nw;
    // 16-byte stores of P0 rows need every row 16-byte aligned: nx even AND an aligned P0
    a.wide_out = (tf->nx % 2 == 0 && ((uintptr_t)P0_dev & 15u) == 0) ? 1 : 0;
    const int jb = tf->warps * PDM_TF_JT;
    dim3 grid((tf->nx + PDM_TF_XB - 1) / PDM_TF_XB, (tf->nw + jb - 1) / jb);
    if (tf->nx % 4 == 0 && ((uintptr_t)section_dev & 15u) == 0)
        pdm_tf_kernel<4><<<grid, 32 * tf->warps, tf->smem_bytes, (cudaStream_t)cuda_stream>>>(a);
    else
        pdm_tf_kernel<1><<<grid, 32 * tf->warps, tf->smem_bytes, (cudaStream_t)cuda_stream>>>(a);
    if (cudaGetLastError() != cudaSuccess) return PDM_ERR_CUDA;
    return PDM_OK;
}

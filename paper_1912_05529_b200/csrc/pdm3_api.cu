// pdm3_api.cu -- host side of the 3-D variant (include/pdm.h: pdm3_create / pdm3_migrate / pdm3_destroy /
// pdm3_get_info, reading R18).  Same contract as the 2-D calls:
// everything data-independent is validated, pre-digested and uploaded at create time, pdm3_migrate only
// enqueues kernels; no CPU fallback.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>
#include <vector>

#include "pdm_common.cuh"
#include "kern_3d.cuh"
#include "kern_reduce.cuh"

struct pdm3_plan {
    int nx, ny, nz, nw, ntab, ntaps, L, Lk;
    int device, sm_count, last_cuda_error;
    unsigned flags;
    float *d_omega, *d_q, *d_partial;
    float4 *d_tab;
    float2 *d_plane[2];
    int qstride, wgroups, smem_bytes, ctas_per_sm, grid, slice_rows, sym2;
    double workspace_bytes;
};

#define PDM3_CUDA(plan, call)                                                       \
    do {                                                                            \
        cudaError_t e_ = (call);                                                    \
        if (e_ != cudaSuccess) {                                                    \
            (plan)->last_cuda_error = (int)e_;                                      \
            return e_ == cudaErrorMemoryAllocation ? PDM_ERR_NOMEM : PDM_ERR_CUDA;  \
        }                                                                           \
    } while (0)

typedef void (*pdm3_fn)(const pdm3_params);
#define PDM3_FOR_EACH_L(X) X(1) X(2) X(3) X(5) X(7)
static int pdm3_kernel_half_length(int L)
{
#define X(LL) if (L <= LL) return LL;
    PDM3_FOR_EACH_L(X)
#undef X
    return 0;
}
static pdm3_fn pdm3_kernel_for(int Lk, bool wide, bool sym2)
{
    switch (Lk) {
#define X(LL) case LL: return sym2 ? (wide ? pdm3_step<LL, 2, true> : pdm3_step<LL, 1, true>) \
                                   : (wide ? pdm3_step<LL, 2, false> : pdm3_step<LL, 1, false>);
        PDM3_FOR_EACH_L(X)
#undef X
    default: return nullptr;
    }
}

static void pdm3_free(pdm3_plan *p)
{
    if (!p) return;
    cudaFree(p->d_omega); cudaFree(p->d_q); cudaFree(p->d_partial); cudaFree(p->d_tab);
    cudaFree(p->d_plane[0]); cudaFree(p->d_plane[1]);
    delete p;
}

template <class T>
static int pdm3_alloc(pdm3_plan *p, T **ptr, size_t count, const T *host = nullptr)
{
    *ptr = nullptr;
    PDM3_CUDA(p, cudaMalloc((void **)ptr, std::max<size_t>(count, 1) * sizeof(T)));
    p->workspace_bytes += (double)(count * sizeof(T));
    if (host) PDM3_CUDA(p, cudaMemcpy(*ptr, host, count * sizeof(T), cudaMemcpyHostToDevice));
    return PDM_OK;
}

extern "C" int pdm3_destroy(pdm3_plan *p) { pdm3_free(p); return PDM_OK; }

extern "C" int pdm3_create(pdm3_plan **out, int nx, int ny, int nz, int nw, float dz,
                           const float *omega, const float *velocity,
                           const pdm_c64 *table, int ntab, int ntaps, double tab_du, unsigned flags)
{
    if (!out) return PDM_ERR_INVALID_ARG;
    *out = nullptr;
    if (!omega || !velocity || !table) return PDM_ERR_INVALID_ARG;
    if (nx <= 0 || ny <= 0 || nz <= 0 || nw <= 0 || ntab <= 0 || ntaps < 1 || (ntaps & 1) == 0)
        return PDM_ERR_INVALID_ARG;
    if (!(tab_du > 0.0) || !std::isfinite(tab_du) || !(dz > 0.f) || !std::isfinite(dz)) return PDM_ERR_INVALID_ARG;
    if (flags & ~(PDM_FORCE_GENERAL | PDM_REQUIRE_SYMMETRIC)) return PDM_ERR_INVALID_ARG;
    const int L = (ntaps - 1) / 2, Lk = pdm3_kernel_half_length(L);
    if (!Lk) return PDM_ERR_UNSUPPORTED;                    // longer than the longest unrolled 2-D kernel (15 x 15)
    const double slab = (double)ny * (double)nx;
    if (slab * nz > 2.0e9 || slab * nw > 2.0e9) return PDM_ERR_UNSUPPORTED;
    for (int i = 0; i < nw; ++i)
        if (!(omega[i] > 0.f) || !std::isfinite(omega[i])) return PDM_ERR_INVALID_ARG;
    const size_t vol = (size_t)nz * ny * nx;
    for (size_t i = 0; i < vol; ++i)
        if (!(velocity[i] > 0.f) || !std::isfinite(velocity[i])) return PDM_ERR_INVALID_ARG;

    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        cudaGetLastError();
        return PDM_ERR_UNSUPPORTED;                        // no usable CUDA device: no fallback
    }
    if (prop.major != 10) return PDM_ERR_UNSUPPORTED;

    pdm3_plan *p = new (std::nothrow) pdm3_plan();
    if (!p) return PDM_ERR_NOMEM;
    memset(p, 0, sizeof(*p));
    p->nx = nx; p->ny = ny; p->nz = nz; p->nw = nw; p->ntab = ntab; p->ntaps = ntaps; p->L = L; p->Lk = Lk;
    p->device = dev; p->sm_count = prop.multiProcessorCount; p->flags = flags;

    // R3: q32 = fl32(dz / (v * du)); rows padded to a multiple of 8 with the last value
    p->qstride = (nx + 7) / 8 * 8;
    std::vector<float> q((size_t)nz * ny * p->qstride);
    float qmax = 0.f, wmax = 0.f;
    size_t varied = 0;                                     // rows whose q changes along x: per-sample table rows
    for (size_t r = 0; r < (size_t)nz * ny; ++r) {
        float *row = q.data() + r * p->qstride;
        for (int x = 0; x < nx; ++x) {
            row[x] = (float)((double)dz / ((double)velocity[r * nx + x] * tab_du));
            qmax = std::max(qmax, row[x]);
            if (x && row[x] != row[x - 1]) { ++varied; }
        }
        for (int x = nx; x < p->qstride; ++x) row[x] = row[nx - 1];
    }
    for (int i = 0; i < nw; ++i) wmax = std::max(wmax, omega[i]);
    {
        volatile float prod = wmax * qmax;
        if (!std::isfinite(qmax) || !(prod < 2.0e9f) || lrintf(prod) > ntab - 1) { pdm3_free(p); return PDM_ERR_TABLE_RANGE; }
    }
    // W[ky][kx] == W[-ky][kx] == W[ky][-kx] bit for bit in every row: the folded kernels (L+1 passes over
    // row sums, 1 FADD2 + 2 FFMA2 per tap pair); otherwise the general ones (Eq. (1) literally)
    bool sym2 = true;
    for (int j = 0; j < ntab && sym2; ++j)
        for (int ky = -L; ky <= L && sym2; ++ky)
            for (int kx = -L; kx <= L; ++kx) {
                const pdm_c64 *a = &table[((size_t)j * ntaps + (L + ky)) * ntaps + (L + kx)];
                const pdm_c64 *b = &table[((size_t)j * ntaps + (L - ky)) * ntaps + (L + kx)];
                const pdm_c64 *c = &table[((size_t)j * ntaps + (L + ky)) * ntaps + (L - kx)];
                if (memcmp(a, b, sizeof(pdm_c64)) != 0 || memcmp(a, c, sizeof(pdm_c64)) != 0) { sym2 = false; break; }
            }
    if (flags & PDM_REQUIRE_SYMMETRIC) { if (!sym2) { pdm3_free(p); return PDM_ERR_TABLE_ASYMMETRIC; } }
    p->sym2 = sym2 ? 1 : 0;
    const int ku = sym2 ? (Lk + 2) / 2 : Lk + 1;
    const int units = (sym2 ? Lk + 1 : 2 * Lk + 1) * ku;
    std::vector<float4> tab((size_t)ntab * units, make_float4(0.f, 0.f, 0.f, 0.f));
    for (int j = 0; j < ntab; ++j) {
        if (sym2) {                                        // units (W[ky][2t], W[ky][2t+1]), ky = 0..L
            for (int ky = 0; ky <= L; ++ky)
                for (int k = 0; k <= L; ++k) {
                    const pdm_c64 a = table[((size_t)j * ntaps + (L + ky)) * ntaps + (L + k)];
                    float4 &d = tab[(size_t)j * units + (size_t)ky * ku + k / 2];
                    if (k & 1) { d.z = a.re; d.w = a.im; } else { d.x = a.re; d.y = a.im; }
                }
        } else {                                           // units (W[ky][kx], W[ky][-kx]), kx = 0..L, ky = -L..L
            for (int ky = -L; ky <= L; ++ky)
                for (int k = 0; k <= L; ++k) {
                    const pdm_c64 a = table[((size_t)j * ntaps + (L + ky)) * ntaps + (L + k)];
                    const pdm_c64 b = table[((size_t)j * ntaps + (L + ky)) * ntaps + (L - k)];
                    tab[(size_t)j * units + (size_t)(ky + Lk) * (Lk + 1) + k] = make_float4(a.re, a.im, b.re, b.im);
                }
        }
    }

    int rc;
#define PDM3_TRY(call) do { if ((rc = (call)) != PDM_OK) { pdm3_free(p); return rc; } } while (0)
    PDM3_TRY(pdm3_alloc(p, &p->d_omega, (size_t)nw, omega));
    PDM3_TRY(pdm3_alloc(p, &p->d_q, q.size(), q.data()));
    PDM3_TRY(pdm3_alloc(p, &p->d_tab, tab.size(), tab.data()));
    const int HG = (Lk + 1 + 7) / 8;
    p->smem_bytes = 2 * (PDM3_TY + 2 * Lk) * (PDM3_TX / 8 + 2 * HG) * 10 * (int)sizeof(float2);
    // models where (nearly) every sample has its own row: a per-tile, per-frequency slice of the table in
    // shared memory (32 KB, 64 KB for the long operators) instead of gathering rows through L1
    if (varied * 4 > (size_t)nz * ny * nx) {
        const int units_p = units | 1;
        const int slice_bytes = (Lk <= 3 ? 32 : 64) * 1024;
        p->slice_rows = slice_bytes / (units_p * (int)sizeof(float4));
        p->smem_bytes += p->slice_rows * units_p * (int)sizeof(float4);
    }
    int per_sm = 0;
    for (int wide = 0; wide < 2; ++wide) {
        pdm3_fn fn = pdm3_kernel_for(Lk, wide != 0, sym2);
        cudaError_t e = cudaFuncSetAttribute((const void *)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, p->smem_bytes);
        if (e == cudaSuccess)
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void *)fn, PDM3_THREADS, (size_t)p->smem_bytes);
        if (e != cudaSuccess) { p->last_cuda_error = (int)e; pdm3_free(p); return PDM_ERR_CUDA; }
    }
    if (per_sm < 1) { pdm3_free(p); return PDM_ERR_UNSUPPORTED; }
    p->ctas_per_sm = per_sm;
    // ONE resident wave per depth step: tiles x frequency groups <= SMs x CTAs per SM
    const int tiles = ((nx + PDM3_TX - 1) / PDM3_TX) * ((ny + PDM3_TY - 1) / PDM3_TY);
    int wgroups = std::max(1, std::min(nw, p->sm_count * per_sm / tiles));
    const int wpg = (nw + wgroups - 1) / wgroups;
    p->wgroups = (nw + wpg - 1) / wpg;
    p->grid = tiles * p->wgroups;
    PDM3_TRY(pdm3_alloc(p, &p->d_partial, (size_t)p->wgroups * nz * ny * p->qstride));
    PDM3_TRY(pdm3_alloc(p, &p->d_plane[0], (size_t)nw * ny * nx));
    PDM3_TRY(pdm3_alloc(p, &p->d_plane[1], (size_t)nw * ny * nx));
#undef PDM3_TRY
    *out = p;
    return PDM_OK;
}

extern "C" int pdm3_migrate(pdm3_plan *p, const pdm_c64 *P0_dev, float *image_dev, void *cuda_stream)
{
    if (!p || !P0_dev || !image_dev) return PDM_ERR_INVALID_ARG;
    int dev = -1;
    PDM3_CUDA(p, cudaGetDevice(&dev));
    if (dev != p->device) { p->last_cuda_error = (int)cudaErrorInvalidDevice; return PDM_ERR_CUDA; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    pdm3_params a;
    a.partial = p->d_partial; a.q = p->d_q; a.omega = p->d_omega; a.tab = p->d_tab;
    a.nx = p->nx; a.ny = p->ny; a.nz = p->nz; a.nw = p->nw; a.ntab = p->ntab;
    a.qstride = p->qstride; a.pstride = p->qstride;
    a.w_per_group = (p->nw + p->wgroups - 1) / p->wgroups;
    a.force_general = (p->flags & PDM_FORCE_GENERAL) ? 1 : 0;
    a.slice_rows = p->slice_rows;
    // 16-byte copies and stores need every plane row 16-byte aligned: nx even and an aligned P0
    const bool wide = (p->nx % 2 == 0) && (((uintptr_t)P0_dev & 15u) == 0);
    pdm3_fn fn = pdm3_kernel_for(p->Lk, wide, p->sym2 != 0);
    dim3 grid((p->nx + PDM3_TX - 1) / PDM3_TX, (p->ny + PDM3_TY - 1) / PDM3_TY, p->wgroups);
    const float2 *src = reinterpret_cast<const float2 *>(P0_dev);
    for (int z = 0; z < p->nz; ++z) {
        a.z = z; a.Pin = src; a.Pout = p->d_plane[z & 1];
        fn<<<grid, PDM3_THREADS, p->smem_bytes, st>>>(a);
        src = a.Pout;
    }
    PDM3_CUDA(p, cudaGetLastError());
    dim3 rg((p->nx + 255) / 256, p->nz * p->ny);
    pdm_reduce_partials<<<rg, 256, 0, st>>>(p->d_partial, image_dev, p->wgroups, p->nz * p->ny, p->nx, a.pstride);
    PDM3_CUDA(p, cudaGetLastError());
    return PDM_OK;
}

extern "C" int pdm3_get_info(const pdm3_plan *p, pdm_info *out)
{
    if (!p || !out) return PDM_ERR_INVALID_ARG;
    memset(out, 0, sizeof(*out));
    out->path = 6;                                         // the 3-D per-step tiled kernel
    out->taps_mode = 1;
    out->nx = p->nx; out->nz = p->nz; out->nw = p->nw; out->ntab = p->ntab; out->ntaps = p->ntaps;
    out->grid_ctas = p->grid; out->threads_per_cta = PDM3_THREADS; out->ctas_per_sm = p->ctas_per_sm;
    out->smem_bytes = p->smem_bytes; out->launches_per_migrate = p->nz + 1;
    out->sm_count = p->sm_count; out->last_cuda_error = p->last_cuda_error;
    out->table_symmetric = p->sym2;
    out->samples = (double)p->nx * (double)p->ny * (double)p->nz * (double)p->nw;
    out->counted_flops = 8.0 * p->ntaps * p->ntaps * out->samples;
    out->executed_lane_ops = (p->sym2 ? (double)(p->Lk + 1) * (6.0 * p->Lk + 4.0)
                                      : 4.0 * (2 * p->Lk + 1) * (2 * p->Lk + 1)) * out->samples;
    out->workspace_bytes = p->workspace_bytes;
    return PDM_OK;
}

// pdm_static.cu -- pdm_migrate_static: the one entry point of libpdm that never allocates.
//
// Who it is for.  Some programs that would like to call this library are not allowed to create
// device memory at the moment they call it: a plug-in whose host application hands every extension a
// fixed set of device buffers and forbids the CUDA allocator, a real-time acquisition loop in which
// cudaMalloc's implicit device-wide synchronisation (and its unbounded latency) would stall the other
// streams, a process that runs close to the memory limit and must not fail half-way with an
// out-of-memory error, or a thread that may not take the allocator's locks.  Every other migration in
// this library goes through pdm_create, which allocates a plan (tables, work lists, wavefield planes).
// This file gives those callers the per-depth-step form of the migration (the mapping of
// PDM_PATH_NAIVE: one thread per (w, x) sample of the next depth plane, one launch per
// depth level, then one thread per x for the image row) with its only scratch -- the two
// ping-pong wavefield planes -- held in a fixed array that is part of the library image itself.
//
// The array.  pdm_static_planes below is 2 * PDM_STATIC_MAX_SAMPLES complex64 = 16 MiB.  The CUDA
// runtime reserves it on every GPU on which this library's code is loaded and keeps it until the
// process exits; nobody can free it.  Inside host code the identifier pdm_static_planes is only a
// handle that the runtime understands, not a device address, so the host never passes it to a
// kernel: scratch_for_current_device() asks the runtime for the real address with
// cudaGetSymbolAddress, once per device, with that device current, and the kernels receive that.
//
// Sharing.  There is one array per (process, GPU).  Every call on that GPU uses it, and a call finds
// in it whatever the previous call left.  Nothing in it has to start at zero: each depth step writes
// all nw*nx samples of one plane before the next launch on the same stream reads them, and nothing
// beyond nw*nx is ever read.  For the same reason two calls that can run on the GPU at the same time
// (different streams, or two host threads on different streams) overwrite each other's wavefield --
// the caller must order them (one stream, or an event between them).
#include <mutex>
#include "pdm_common.cuh"

static __device__ __align__(256) float2 pdm_static_planes[2 * (size_t)PDM_STATIC_MAX_SAMPLES];

// One depth step of Eq. (1) for every (w, x): t = iw*nx + x.  q32 is formed here exactly as pdm_create
// forms it on the host (R3: one rounding from double), so both entry points pick the same table rows.
static __global__ void pdm_static_step(const float2 *__restrict__ Pin, float2 *__restrict__ Pout,
                                       const float *__restrict__ omega, const float *__restrict__ vrow,
                                       const float2 *__restrict__ table, int nx, int nw, int ntab, int L,
                                       double dz, double du)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nw * nx) return;
    const int iw = t / nx, x = t - iw * nx;
    const float q = __double2float_rn(__ddiv_rn(dz, __dmul_rn((double)vrow[x], du)));
    const int j = pdm_index(omega[iw], q, ntab - 1);
    const float2 *row = table + (size_t)j * (2 * L + 1) + L;
    const float2 *p = Pin + (size_t)iw * nx;
    const int klo = max(-L, x - (nx - 1)), khi = min(L, x);       // R5: terms outside [0,nx) are zero
    float ar = 0.f, ai = 0.f;
    for (int k = klo; k <= khi; ++k) {
        const float2 w = __ldg(row + k), v = p[x - k];
        ar = fmaf(w.x, v.x, ar); ar = fmaf(-w.y, v.y, ar);
        ai = fmaf(w.x, v.y, ai); ai = fmaf(w.y, v.x, ai);
    }
    Pout[t] = make_float2(ar, ai);
}

// Imaging: image_row[x] = sum over w, in index order, of Re P(z+dz, w, x).
static __global__ void pdm_static_image_row(const float2 *__restrict__ P, float *__restrict__ image_row,
                                            int nx, int nw)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= nx) return;
    float s = 0.f;
    for (int iw = 0; iw < nw; ++iw) s += P[(size_t)iw * nx + x].x;
    image_row[x] = s;
}

// Device address of pdm_static_planes on the CURRENT device, looked up on the first call made with
// that device current and remembered.  Returns PDM_OK and *out, or the status to hand back.
#define PDM_STATIC_MAX_DEVICES 64
static int scratch_for_current_device(float2 **out)
{
    static std::mutex mu;
    static float2 *addr[PDM_STATIC_MAX_DEVICES];          // zero-initialised: "not looked up yet"
    int dev = -1, major = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= PDM_STATIC_MAX_DEVICES) {
        cudaGetLastError();
        return PDM_ERR_UNSUPPORTED;
    }
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess || major != 10) {
            cudaGetLastError();
            return PDM_ERR_UNSUPPORTED;                    // the kernels exist for sm_100a only
        }
        void *ptr = nullptr;
        if (cudaGetSymbolAddress(&ptr, pdm_static_planes) != cudaSuccess || !ptr) {
            cudaGetLastError();
            return PDM_ERR_CUDA;
        }
        addr[dev] = static_cast<float2 *>(ptr);
    }
    *out = addr[dev];
    return PDM_OK;
}

extern "C" int pdm_migrate_static(int nx, int nz, int nw, float dz,
                                  const float *omega_dev, const float *velocity_dev,
                                  const pdm_c64 *table_dev, int ntab, int ntaps, double tab_du,
                                  const pdm_c64 *P0_dev, float *image_dev, void *cuda_stream)
{
    if (nx <= 0 || nz <= 0 || nw <= 0 || ntab <= 0 || ntaps < 1 || (ntaps & 1) == 0 ||
        !(dz > 0.f) || !(tab_du > 0.0) || !omega_dev || !velocity_dev || !table_dev || !P0_dev || !image_dev)
        return PDM_ERR_INVALID_ARG;
    if (ntaps > PDM_MAX_TAPS) return PDM_ERR_UNSUPPORTED;
    if ((long long)nx * nw > (long long)PDM_STATIC_MAX_SAMPLES) return PDM_ERR_TOO_LARGE;

    float2 *planes = nullptr;
    const int rc = scratch_for_current_device(&planes);
    if (rc != PDM_OK) return rc;

    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int L = (ntaps - 1) / 2, n = nx * nw;
    const float2 *table = reinterpret_cast<const float2 *>(table_dev);
    const float2 *in = reinterpret_cast<const float2 *>(P0_dev);
    for (int iz = 0; iz < nz; ++iz) {
        float2 *out = planes + (size_t)(iz & 1) * PDM_STATIC_MAX_SAMPLES;
        pdm_static_step<<<(n + 255) / 256, 256, 0, st>>>(in, out, omega_dev, velocity_dev + (size_t)iz * nx,
                                                         table, nx, nw, ntab, L, (double)dz, tab_du);
        pdm_static_image_row<<<(nx + 127) / 128, 128, 0, st>>>(out, image_dev + (size_t)iz * nx, nx, nw);
        in = out;
    }
    if (cudaGetLastError() != cudaSuccess) return PDM_ERR_CUDA;
    return PDM_OK;
}

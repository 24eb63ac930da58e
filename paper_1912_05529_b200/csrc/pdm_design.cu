// pdm_design.cu -- extrapolator-table design on the device.
// PAPER.md:39 (the design trades filter length against propagation angle), :83 ("Designing filters
// itself is optimization problem, it takes sometime ... we design the filters in advance"), refs
// :163-165, :179-180.  The paper gives no recipe; this is the projections-onto-convex-sets style
// iteration DESIGN.md states as D1-D4, one CTA per table row, FP64 throughout:
//   D1  target on the periodic grid kappa_m = 2 pi m / N, m = 0..N/2 (responses of symmetric
//       filters are even in kappa):   D(kappa) = exp(+i sqrt(u^2 - (r kappa)^2))   |r kappa| <= u
//                                              = exp(  - sqrt((r kappa)^2 - u^2))   otherwise
//   D2  start W = truncation of IDFT(D); repeat n_iter times:
//         H_m = W_0 + 2 sum_{k>=1} W_k cos(k kappa_m)
//         passband |kappa| <= min((u/r) sin(angle), kappa_cap):  H_m <- D_m
//         elsewhere, where |H_m| > stop_cap:                      H_m <- H_m stop_cap / |H_m|
//         W_k = (1/N) [ H_0 + (-1)^k H_{N/2} + 2 sum_{m=1}^{N/2-1} H_m cos(k kappa_m) ]   (k = 0..L)
//       (the second line IS "inverse DFT, keep |k| <= L, average W_k and W_-k")
//   D3  |H| on n_check points of [0, pi]; divide the taps by max(1, max|H|) (1 + 4e-7); round to
//       complex64; mirror W_-k = W_k bit for bit.
// cos(k kappa_m) comes from an N-entry table indexed by the exact integer (k m) mod N.
#include <cmath>
#include <cstring>
#include <vector>

#include <cuda_runtime.h>
#include "../../include/pdm.h"

#define PDM_DESIGN_THREADS 256
#define PDM_DESIGN_MAX_L 64

struct pdm_design_params {
    float2 *table;            // DEVICE [ntab][ntaps]
    const double *costab;     // DEVICE [N]  cos(2 pi i / N)
    int ntab, ntaps, L, N, n_iter, n_check;
    double du, r, sin_angle, kappa_cap, stop_cap;
};

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__global__ void __launch_bounds__(PDM_DESIGN_THREADS) pdm_design_kernel(const pdm_design_params p)
{
    extern __shared__ __align__(16) unsigned char pdm_dsmem[];
    const int N = p.N, M = N / 2, L = p.L;
    double *ct = reinterpret_cast<double *>(pdm_dsmem);          // [N]     cos table
    double2 *D = reinterpret_cast<double2 *>(ct + N);            // [M+1]   target
    double2 *H = D + (M + 1);                                    // [M+1]   current response
    double2 *W = H + (M + 1);                                    // [L+1]   half taps
    __shared__ double red[PDM_DESIGN_THREADS / 32];
    __shared__ int pass_end_s;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = PDM_DESIGN_THREADS / 32;
    const int j = blockIdx.x;
    const double u = (double)j * p.du;
    const double two_pi = 6.283185307179586476925286766559;

    for (int i = tid; i < N; i += PDM_DESIGN_THREADS) ct[i] = p.costab[i];
    // D1 + passband edge: m <= pass_end  <=>  kappa_m <= min((u/r) sin(angle), kappa_cap)
    const double edge = fmin((u / p.r) * p.sin_angle, p.kappa_cap);
    for (int m = tid; m <= M; m += PDM_DESIGN_THREADS) {
        const double kap = two_pi * (double)m / (double)N;
        const double rk = p.r * kap, arg = u * u - rk * rk;
        const double root = sqrt(fabs(arg));
        double2 d;
        if (arg >= 0.0) { double s, c; sincos(root, &s, &c); d = make_double2(c, s); }
        else d = make_double2(exp(-root), 0.0);
        D[m] = d;
        H[m] = d;
    }
    if (tid == 0) {
        int e = -1;
        for (int m = 0; m <= M; ++m)
            if (two_pi * (double)m / (double)N <= edge) e = m; else break;
        pass_end_s = e;
    }
    __syncthreads();
    const int pass_end = pass_end_s;

    // inverse step: W_k from H (warp w owns k = w, w + nwarps, ...; lanes stride over m)
    auto inverse = [&]() {
        for (int k = warp; k <= L; k += nwarps) {
            double sr = 0.0, si = 0.0;
            int idx = (int)(((long long)k * lane) % N);          // (k m) mod N, advanced by (32 k) mod N
            const int step = (int)((32LL * k) % N);
            for (int m = lane; m <= M; m += 32) {
                double c = ct[idx];
                c *= (m == 0 || m == M) ? 1.0 : 2.0;
                sr += c * H[m].x; si += c * H[m].y;
                idx += step; if (idx >= N) idx -= N;
            }
            sr = warp_sum(sr); si = warp_sum(si);
            if (lane == 0) W[k] = make_double2(sr / (double)N, si / (double)N);
        }
    };
    inverse();                                                   // truncation of IDFT(D)
    __syncthreads();
    for (int it = 0; it < p.n_iter; ++it) {
        for (int m = tid; m <= M; m += PDM_DESIGN_THREADS) {     // forward + the two projections
            double hr = W[0].x, hi = W[0].y;
            int idx = 0;                                         // (k m) mod N, m < N
            for (int k = 1; k <= L; ++k) {
                idx += m; if (idx >= N) idx -= N;
                const double c = 2.0 * ct[idx];
                hr += c * W[k].x; hi += c * W[k].y;
            }
            if (m <= pass_end) { hr = D[m].x; hi = D[m].y; }
            else {
                const double mag = sqrt(hr * hr + hi * hi);
                if (mag > p.stop_cap) { const double s = p.stop_cap / fmax(mag, 1e-300); hr *= s; hi *= s; }
            }
            H[m] = make_double2(hr, hi);
        }
        __syncthreads();
        inverse();                                               // finish on the truncation step
        __syncthreads();
    }

    // D3: max |H| over n_check points of [0, pi]
    double mx = 0.0;
    for (int m = tid; m < p.n_check; m += PDM_DESIGN_THREADS) {
        const double kap = 3.14159265358979323846264338327950288 * (double)m / (double)(p.n_check - 1);
        double hr = W[0].x, hi = W[0].y;
        const double c1 = cos(kap);
        double cm = 1.0, ck = c1;                                // cos((k-1) kap), cos(k kap): Chebyshev recurrence
        for (int k = 1; k <= L; ++k) {
            hr += 2.0 * ck * W[k].x; hi += 2.0 * ck * W[k].y;
            const double cn = 2.0 * c1 * ck - cm;
            cm = ck; ck = cn;
        }
        mx = fmax(mx, sqrt(hr * hr + hi * hi));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if (lane == 0) red[warp] = mx;
    __syncthreads();
    mx = red[0];
    for (int w = 1; w < nwarps; ++w) mx = fmax(mx, red[w]);
    const double scale = 1.0 / (fmax(mx, 1.0) * (1.0 + 4e-7));
    for (int k = tid; k <= L; k += PDM_DESIGN_THREADS) {
        const float2 w = make_float2((float)(W[k].x * scale), (float)(W[k].y * scale));
        float2 *row = p.table + (size_t)j * p.ntaps + L;
        row[k] = w;
        row[-k] = w;
    }
}

extern "C" int pdm_design_table(pdm_c64 *table_host, int ntab, int ntaps, double tab_du,
                                double dz_over_dx, const pdm_design_opts *opts, void *cuda_stream)
{
    if (!table_host || ntab <= 0 || ntaps < 1 || (ntaps & 1) == 0) return PDM_ERR_INVALID_ARG;
    if (!(tab_du > 0.0) || !std::isfinite(tab_du) || !(dz_over_dx > 0.0) || !std::isfinite(dz_over_dx))
        return PDM_ERR_INVALID_ARG;
    pdm_design_opts o;
    o.n_iter = 200; o.n_grid = 2048; o.n_check = 16384;
    o.passband_angle_deg = 55.0; o.kappa_cap = 0.8 * 3.14159265358979323846; o.stop_cap = 0.9995;
    if (opts) o = *opts;
    const int L = (ntaps - 1) / 2;
    if (o.n_iter < 0 || o.n_check < 2 || o.n_grid < 4 || (o.n_grid & 1) || !(o.passband_angle_deg > 0.0) ||
        !(o.passband_angle_deg <= 90.0) || !(o.kappa_cap > 0.0) || !(o.stop_cap > 0.0))
        return PDM_ERR_INVALID_ARG;
    if (L > PDM_DESIGN_MAX_L || 2 * L + 1 > o.n_grid) return PDM_ERR_UNSUPPORTED;
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        cudaGetLastError();
        return PDM_ERR_UNSUPPORTED;                        // no usable CUDA device: no fallback
    }
    if (prop.major != 10) return PDM_ERR_UNSUPPORTED;
    const int N = o.n_grid, M = N / 2;
    const size_t smem = (size_t)N * sizeof(double) + 2 * (size_t)(M + 1) * sizeof(double2) +
                        (size_t)(L + 1) * sizeof(double2);
    if (smem > (size_t)prop.sharedMemPerBlockOptin) return PDM_ERR_UNSUPPORTED;
    cudaStream_t st = (cudaStream_t)cuda_stream;

    std::vector<double> ct(N);
    const double two_pi = 6.283185307179586476925286766559;
    for (int i = 0; i < N; ++i) ct[i] = cos(two_pi * (double)i / (double)N);
    double *d_ct = nullptr;
    float2 *d_table = nullptr;
    int rc = PDM_OK;
    const size_t nt = (size_t)ntab * ntaps;
    if (cudaMalloc((void **)&d_ct, (size_t)N * sizeof(double)) != cudaSuccess ||
        cudaMalloc((void **)&d_table, nt * sizeof(float2)) != cudaSuccess) rc = PDM_ERR_NOMEM;
    if (rc == PDM_OK &&
        (cudaMemcpyAsync(d_ct, ct.data(), (size_t)N * sizeof(double), cudaMemcpyHostToDevice, st) != cudaSuccess ||
         cudaFuncSetAttribute((const void *)pdm_design_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)smem) != cudaSuccess)) rc = PDM_ERR_CUDA;
    if (rc == PDM_OK) {
        pdm_design_params a;
        a.table = d_table; a.costab = d_ct; a.ntab = ntab; a.ntaps = ntaps; a.L = L; a.N = N;
        a.n_iter = o.n_iter; a.n_check = o.n_check; a.du = tab_du; a.r = dz_over_dx;
        a.sin_angle = sin(o.passband_angle_deg * 3.14159265358979323846 / 180.0);
        a.kappa_cap = o.kappa_cap; a.stop_cap = o.stop_cap;
        pdm_design_kernel<<<ntab, PDM_DESIGN_THREADS, smem, st>>>(a);
        if (cudaGetLastError() != cudaSuccess ||
            cudaMemcpyAsync(table_host, d_table, nt * sizeof(float2), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
            cudaStreamSynchronize(st) != cudaSuccess) rc = PDM_ERR_CUDA;
    }
    if (rc != PDM_OK) cudaGetLastError();
    cudaFree(d_ct); cudaFree(d_table);
    return rc;
}

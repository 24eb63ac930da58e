/*
 * pdm_oracle.c -- TEST INFRASTRUCTURE ONLY.  Plain, slow, FP64 CPU statement of the hot path
 * of explicit f-x poststack depth migration, written from the paper
 * (arXiv 1912.05529, /root/reference/PAPER.md) for checking the CUDA library against.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call this file.  It shares no code, header, table or helper with the
 * CUDA path (paper_1912_05529_b200/csrc) and must never be reachable from the product path.
 *
 * What it computes (citations are PAPER.md lines; R# are the readings listed in DESIGN.md):
 *
 *   Eq. (1), PAPER.md:45      u(x_i, w_r, z_{k+1}) = sum_{n=-(N-1)/2}^{(N-1)/2} h[n] u(x_{i-n}, w_r, z_k)
 *   Alg. 1,  PAPER.md:59-70   for each depth level { for each frequency { for each space {
 *                               look-up table (pre-designed 1-D FIR filters); extrapolate } }
 *                               depth row = sum over frequencies }              (nesting: R1)
 *   PAPER.md:83               the filter ("cutoff") depends on frequency and velocity and may
 *                             differ from point to point: it is looked up per OUTPUT point (R8)
 *
 *   O1  q32[z][x] = (float)( (double)dz / ((double)v32[z][x] * du) )          (R3: one rounding)
 *   O2  for each w (independent):
 *   O3      P[x] = (complex double) P0[w][x]
 *   O4      for z = 0 .. nz-1:                                               (sequential)
 *   O5        for x = 0 .. nx-1:
 *   O6          idx = clamp( lrintf( w32 * q32[z][x] ), 0, ntab-1 )          (R3: FLOAT product,
 *                                                                             round half to even)
 *   O7          acc = sum_{k=-L..L, 0 <= x-k < nx}  table[idx][L+k] * P[x-k] (Eq. 1; R5 zero edges;
 *                                                                             R11 orientation)
 *   O8          Pnew[x] = acc
 *   O9        swap(P, Pnew)
 *   O10       img_w[z][x] = Re P[x]      row z = field AFTER step z, depth (z+1) dz   (R6, R7)
 *   O11 image[z][x] = sum_w img_w[z][x]  in FP64, fixed order                 (R10)
 *
 * No symmetric folding, no tiling, no blocking: the full 2L+1 row is applied literally.
 * Parallelism: OpenMP over w only (independent lines); per-thread FP64 image accumulators
 * are summed in thread-id order, and each thread walks its w in increasing order, so the
 * result is deterministic for a fixed thread count.
 *
 * Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): P1 delta table = identity, P2 brute
 * force on tiny grids, P3 spectral identity, P4 exact phase shift in constant velocity,
 * P5 point-diffractor focusing, P7 superposition, P8 w-additivity/permutation, P9 mirror,
 * P10 energy non-growth, P11 shift invariance, P12a index rule (the function), P12b index rule
 * THROUGH the migrate loop (centre-tap-encodes-row table; a double product or a float-formed q
 * inside the loop fails it).  The edge-taper variant R5b (pdm_oracle_migrate_taper; the plain entry point
 * is that function with ntaper = 0) has its own pins in tests/test_oracle_taper_pins.py.  The file is also built with -fsanitize=address,undefined and run
 * on ragged cases (tests/test_oracle_sanitize.py).  Parity unpinned by anything external: the
 * choices R5/R6/R7 (boundary, row<->depth, velocity row) and the absolute amplitude scale R10
 * -- fixed by DESIGN.md only (P5 accepts +-1 row, so it does not pin R6 to the row either).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct { float re, im; } oracle_c64;

#define ORACLE_OK 0
#define ORACLE_ERR_ARG -1
#define ORACLE_ERR_NOMEM -2

int pdm_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* O1 (R3): q32 = fl32( dz / (v32 * du) ) -- formed in double, rounded ONCE to float. */
static float oracle_q32(double dz, float velocity, double du)
{
    return (float)(dz / ((double)velocity * du));
}

/* O6 (R3): FLOAT product (float x float -> float, no FMA involved), round half to even
 * (default rounding mode), clamp to the table.  The ONE statement of the index rule in this
 * file: pdm_oracle_migrate's inner loop and pdm_oracle_index both call it. */
static int oracle_idx(float w32, float q32, int ntab)
{
    float prod = w32 * q32;
    long j = lrintf(prod);
    if (j < 0) j = 0;
    if (j > ntab - 1) j = ntab - 1;
    return (int)j;
}

/* O1 + O6 exposed on their own (pin P12a tests the rule directly; pin P12b tests it through
 * pdm_oracle_migrate's loop). */
int pdm_oracle_index(float omega, float velocity, double dz, double du, int ntab)
{
    return oracle_idx(omega, oracle_q32(dz, velocity, du), ntab);
}

/*
 * All pointers are HOST pointers.  image_out is double [nz][nx] (O12: never rounded down).
 * If wavefield_out != NULL it receives the final field P(z = nz dz) as interleaved
 * complex double [nw][nx] (used by pins P3/P4/P10 which look at the field, not the image).
 * omega_subset: if nsub > 0, only lines omega_index[0..nsub) are migrated (bench sampling, P8).
 */
/* R5 variant (reading R5b; the paper is silent on the lateral boundary): an absorbing
 * cosine edge taper.  After every depth step the new field is multiplied by
 *     t(x) = sin^2( (pi/2) (d+1)/(ntaper+1) ),  d = min(x, nx-1-x),  for d < ntaper;  t(x) = 1 otherwise
 * BEFORE it is imaged and before the next step reads it.  ntaper = 0 is plain R5. */
static double oracle_taper(int x, int nx, int ntaper)
{
    const int d = x < nx - 1 - x ? x : nx - 1 - x;
    if (d >= ntaper) return 1.0;
    const double s = sin(1.57079632679489661923 * (double)(d + 1) / (double)(ntaper + 1));
    return s * s;
}

/* R3 variant (reading R3c; SURVEY 8(f) N3 "optional linear interpolation between rows";
 * PAPER.md:65, :83 only say the filter is looked up): instead of the nearest row, the operator is the
 * linear blend of the two rows that bracket u = w*dz/v,
 *     u32 = fl32(w32 * q32)   (the SAME float product as O6),  j0 = floor(u32),  a = u32 - j0  (exact in float),
 *     W_k = (1 - a) table[j0][k] + a table[j0 + 1][k],         j0 >= ntab-1:  W_k = table[ntab-1][k].
 * a == 0 wherever u32 is an integer, so the blend then equals the nearest-row operator.           */
static void oracle_interp_rows(float w32, float q32, int ntab, int *j0, int *j1, double *a)
{
    float u = w32 * q32;
    if (!(u > 0.0f)) u = 0.0f;
    const float f = floorf(u);
    if (f >= (float)(ntab - 1)) { *j0 = ntab - 1; *j1 = ntab - 1; *a = 0.0; return; }
    *j0 = (int)f;
    *j1 = *j0 + 1;
    *a = (double)(u - f);
}

static int oracle_migrate_core(int nx, int nz, int nw, double dz,
                               const float *omega, const float *velocity,
                               const oracle_c64 *table, int ntab, int ntaps, double du,
                               const oracle_c64 *P0,
                               const int *omega_index, int nsub, int ntaper, int interp,
                               double *image_out, double *wavefield_out);

int pdm_oracle_migrate_taper(int nx, int nz, int nw, double dz,
                             const float *omega, const float *velocity,
                             const oracle_c64 *table, int ntab, int ntaps, double du,
                             const oracle_c64 *P0,
                             const int *omega_index, int nsub, int ntaper,
                             double *image_out, double *wavefield_out)
{
    return oracle_migrate_core(nx, nz, nw, dz, omega, velocity, table, ntab, ntaps, du, P0,
                               omega_index, nsub, ntaper, 0, image_out, wavefield_out);
}

/* The interpolated-table variant R3c (plain R5 edges). */
int pdm_oracle_migrate_interp(int nx, int nz, int nw, double dz,
                              const float *omega, const float *velocity,
                              const oracle_c64 *table, int ntab, int ntaps, double du,
                              const oracle_c64 *P0,
                              const int *omega_index, int nsub,
                              double *image_out, double *wavefield_out)
{
    return oracle_migrate_core(nx, nz, nw, dz, omega, velocity, table, ntab, ntaps, du, P0,
                               omega_index, nsub, 0, 1, image_out, wavefield_out);
}

int pdm_oracle_migrate(int nx, int nz, int nw, double dz,
                       const float *omega, const float *velocity,
                       const oracle_c64 *table, int ntab, int ntaps, double du,
                       const oracle_c64 *P0,
                       const int *omega_index, int nsub,
                       double *image_out, double *wavefield_out)
{
    return pdm_oracle_migrate_taper(nx, nz, nw, dz, omega, velocity, table, ntab, ntaps, du, P0,
                                    omega_index, nsub, 0, image_out, wavefield_out);
}

static int oracle_migrate_core(int nx, int nz, int nw, double dz,
                               const float *omega, const float *velocity,
                               const oracle_c64 *table, int ntab, int ntaps, double du,
                               const oracle_c64 *P0,
                               const int *omega_index, int nsub, int ntaper, int interp,
                               double *image_out, double *wavefield_out)
{
    if (nx <= 0 || nz <= 0 || nw <= 0 || ntab <= 0 || ntaps < 1 || (ntaps & 1) == 0 || ntaper < 0 ||
        !(du > 0.0) || !omega || !velocity || !table || !P0 || !image_out)
        return ORACLE_ERR_ARG;
    const int L = (ntaps - 1) / 2;
    const int nlines = nsub > 0 ? nsub : nw;
    const size_t plane = (size_t)nz * (size_t)nx;

    /* O1 */
    float *q32 = (float *)malloc(plane * sizeof(float));
    if (!q32) return ORACLE_ERR_NOMEM;
    for (size_t i = 0; i < plane; ++i)
        q32[i] = oracle_q32(dz, velocity[i], du);

    int nthreads = pdm_oracle_num_threads();
    if (nthreads > nlines) nthreads = nlines;
    double *acc = (double *)calloc((size_t)nthreads * plane, sizeof(double));
    if (!acc) { free(q32); return ORACLE_ERR_NOMEM; }
    int failed = 0;

#pragma omp parallel num_threads(nthreads)
    {
#ifdef _OPENMP
        const int tid = omp_get_thread_num();
#else
        const int tid = 0;
#endif
        double *img = acc + (size_t)tid * plane;
        double *P = (double *)malloc(sizeof(double) * 2 * (size_t)nx);
        double *Pn = (double *)malloc(sizeof(double) * 2 * (size_t)nx);
        if (!P || !Pn) {
#pragma omp atomic write
            failed = 1;
        }
        /* every thread must reach the work-sharing loop or none: decide together after a barrier */
        int any_failed;
#pragma omp barrier
#pragma omp atomic read
        any_failed = failed;
        if (!any_failed) {
#pragma omp for schedule(static)
            for (int il = 0; il < nlines; ++il) {                       /* O2 */
                const int iw = nsub > 0 ? omega_index[il] : il;
                const float w32 = omega[iw];
                for (int x = 0; x < nx; ++x) {                          /* O3 */
                    P[2 * x] = (double)P0[(size_t)iw * nx + x].re;
                    P[2 * x + 1] = (double)P0[(size_t)iw * nx + x].im;
                }
                for (int z = 0; z < nz; ++z) {                          /* O4 */
                    const float *qrow = q32 + (size_t)z * nx;
                    for (int x = 0; x < nx; ++x) {                      /* O5 */
                        const int j = oracle_idx(w32, qrow[x], ntab);   /* O6 */
                        const oracle_c64 *row = table + (size_t)j * ntaps;
                        const oracle_c64 *row1 = row;                   /* R3c: second row and weight */
                        double a1 = 0.0;
                        if (interp) {
                            int j0, j1;
                            oracle_interp_rows(w32, qrow[x], ntab, &j0, &j1, &a1);
                            row = table + (size_t)j0 * ntaps;
                            row1 = table + (size_t)j1 * ntaps;
                        }
                        double ar = 0.0, ai = 0.0;
                        for (int k = -L; k <= L; ++k) {                 /* O7 */
                            int xs = x - k;
                            if (xs < 0 || xs >= nx) continue;
                            double wr = (double)row[L + k].re, wi = (double)row[L + k].im;
                            if (interp) {
                                wr = (1.0 - a1) * wr + a1 * (double)row1[L + k].re;
                                wi = (1.0 - a1) * wi + a1 * (double)row1[L + k].im;
                            }
                            double pr = P[2 * xs], pi = P[2 * xs + 1];
                            ar += wr * pr - wi * pi;
                            ai += wr * pi + wi * pr;
                        }
                        if (ntaper > 0) {                               /* R5b: absorbing edge taper */
                            const double t = oracle_taper(x, nx, ntaper);
                            ar *= t; ai *= t;
                        }
                        Pn[2 * x] = ar;                                 /* O8 */
                        Pn[2 * x + 1] = ai;
                    }
                    { double *t = P; P = Pn; Pn = t; }                  /* O9 */
                    double *irow = img + (size_t)z * nx;                /* O10 (+ O11 partial) */
                    for (int x = 0; x < nx; ++x) irow[x] += P[2 * x];
                }
                if (wavefield_out)
                    memcpy(wavefield_out + 2 * (size_t)il * nx, P, sizeof(double) * 2 * (size_t)nx);
            }
        }
        free(P);
        free(Pn);
    }

    if (!failed) {                                                      /* O11: fixed thread order */
        for (size_t i = 0; i < plane; ++i) {
            double s = 0.0;
            for (int t = 0; t < nthreads; ++t) s += acc[(size_t)t * plane + i];
            image_out[i] = s;
        }
    }
    free(acc);
    free(q32);
    return failed ? ORACLE_ERR_NOMEM : ORACLE_OK;
}

/*
 * Prestack (shot-profile) variant -- PAPER.md:151 ("this work can be easily extended to the
 * prestack depth migration"); the paper gives no equations for it, so this is reading R17 of
 * DESIGN.md, the textbook shot-profile scheme built from the SAME step as above:
 *
 *   S1  R(0,w,x) = recorded shot gather in f-x, S(0,w,x) = source wavefield at the surface
 *   S2  per depth step and frequency, with the SAME looked-up row W(idx(w, v(x,z))) for both:
 *         R(z+dz, x) = sum_k      W_k  R(z, x-k)      (upcoming field continued downward, Eq. (1))
 *         S(z+dz, x) = sum_k conj(W_k) S(z, x-k)      (downgoing field propagated forward:
 *                                                      the conjugate operator)
 *   S3  image[z][x] (+)= sum_w Re( conj(S(z+dz,w,x)) * R(z+dz,w,x) )      (zero-lag
 *         cross-correlation imaging condition; rows as in R6, edges as in R5, index as in R3)
 *
 * image_out is ADDED to when accumulate != 0 (several shots into one image), else overwritten.
 * Pins (tests/test_oracle_shot_pins.py): brute force on tiny grids (independent triple loop),
 * delta table closed form, spectral identity for both fields in constant velocity (asymmetric
 * table), global-phase invariance and real bilinearity, point source + point diffractor focusing.
 */
int pdm_oracle_migrate_shot(int nx, int nz, int nw, double dz,
                            const float *omega, const float *velocity,
                            const oracle_c64 *table, int ntab, int ntaps, double du,
                            const oracle_c64 *S0, const oracle_c64 *R0,
                            int accumulate, double *image_out)
{
    if (nx <= 0 || nz <= 0 || nw <= 0 || ntab <= 0 || ntaps < 1 || (ntaps & 1) == 0 ||
        !(du > 0.0) || !omega || !velocity || !table || !S0 || !R0 || !image_out)
        return ORACLE_ERR_ARG;
    const int L = (ntaps - 1) / 2;
    const size_t plane = (size_t)nz * (size_t)nx;
    float *q32 = (float *)malloc(plane * sizeof(float));
    double *buf = (double *)malloc(sizeof(double) * 8 * (size_t)nx);
    if (!q32 || !buf) { free(q32); free(buf); return ORACLE_ERR_NOMEM; }
    for (size_t i = 0; i < plane; ++i) q32[i] = oracle_q32(dz, velocity[i], du);
    if (!accumulate)
        for (size_t i = 0; i < plane; ++i) image_out[i] = 0.0;
    double *S = buf, *Sn = buf + 2 * (size_t)nx, *R = buf + 4 * (size_t)nx, *Rn = buf + 6 * (size_t)nx;
    for (int iw = 0; iw < nw; ++iw) {                                   /* fixed frequency order */
        const float w32 = omega[iw];
        for (int x = 0; x < nx; ++x) {                                  /* S1 */
            S[2 * x] = (double)S0[(size_t)iw * nx + x].re; S[2 * x + 1] = (double)S0[(size_t)iw * nx + x].im;
            R[2 * x] = (double)R0[(size_t)iw * nx + x].re; R[2 * x + 1] = (double)R0[(size_t)iw * nx + x].im;
        }
        for (int z = 0; z < nz; ++z) {
            const float *qrow = q32 + (size_t)z * nx;
            for (int x = 0; x < nx; ++x) {                              /* S2 */
                const oracle_c64 *row = table + (size_t)oracle_idx(w32, qrow[x], ntab) * ntaps;
                double rr = 0.0, ri = 0.0, sr = 0.0, si = 0.0;
                for (int k = -L; k <= L; ++k) {
                    int xs = x - k;
                    if (xs < 0 || xs >= nx) continue;
                    double wr = (double)row[L + k].re, wi = (double)row[L + k].im;
                    rr += wr * R[2 * xs] - wi * R[2 * xs + 1];          /*      W_k  * R */
                    ri += wr * R[2 * xs + 1] + wi * R[2 * xs];
                    sr += wr * S[2 * xs] + wi * S[2 * xs + 1];          /* conj(W_k) * S */
                    si += wr * S[2 * xs + 1] - wi * S[2 * xs];
                }
                Rn[2 * x] = rr; Rn[2 * x + 1] = ri;
                Sn[2 * x] = sr; Sn[2 * x + 1] = si;
            }
            { double *t = R; R = Rn; Rn = t; t = S; S = Sn; Sn = t; }
            double *irow = image_out + (size_t)z * nx;                  /* S3 */
            for (int x = 0; x < nx; ++x)
                irow[x] += S[2 * x] * R[2 * x] + S[2 * x + 1] * R[2 * x + 1];
        }
    }
    free(buf);
    free(q32);
    return ORACLE_OK;
}

/*
 * 3-D variant -- PAPER.md:41 ("can be easily extended to the 3-D depth migration, which requires
 * 2-D filters as extrapolators"), :47.  The paper gives Eq. (1) for one lateral axis only; reading
 * R18 of DESIGN.md writes it out for two:
 *
 *   T1  q32[z][y][x] = (float)(dz / (v32[z][y][x] * du))                          (R3 unchanged)
 *   T2  per frequency and depth step, per OUTPUT point (y, x):
 *         idx = clamp(lrintf(w32 * q32[z][y][x]), 0, ntab-1)
 *         P'(y,x) = sum_{ky=-L..L} sum_{kx=-L..L} table[idx][L+ky][L+kx] * P(y-ky, x-kx),
 *         terms outside the grid dropped (R5); the (ky, kx) orientation is Eq. (1)'s x_{i-n} on both axes
 *   T3  image[z][y][x] = sum_w Re P'(y,x) after the step (R6, R10)
 *
 * table is [ntab][ntaps][ntaps] (ky slow, kx fast).  OpenMP over frequencies, per-thread FP64 image
 * accumulators summed in thread order.  wavefield_out (optional): final field [nw][ny][nx] complex double.
 * Pins (tests/test_oracle_3d_pins.py): delta table, brute force, 2-D spectral identity with an
 * asymmetric table, separable table == two passes of the (pinned) 1-D oracle, x<->y transposition.
 */
int pdm_oracle_migrate3d(int nx, int ny, int nz, int nw, double dz,
                         const float *omega, const float *velocity,
                         const oracle_c64 *table, int ntab, int ntaps, double du,
                         const oracle_c64 *P0, double *image_out, double *wavefield_out)
{
    if (nx <= 0 || ny <= 0 || nz <= 0 || nw <= 0 || ntab <= 0 || ntaps < 1 || (ntaps & 1) == 0 ||
        !(du > 0.0) || !omega || !velocity || !table || !P0 || !image_out)
        return ORACLE_ERR_ARG;
    const int L = (ntaps - 1) / 2;
    const size_t slab = (size_t)ny * (size_t)nx, vol = (size_t)nz * slab;
    float *q32 = (float *)malloc(vol * sizeof(float));
    if (!q32) return ORACLE_ERR_NOMEM;
    for (size_t i = 0; i < vol; ++i) q32[i] = oracle_q32(dz, velocity[i], du);      /* T1 */
    int nthreads = pdm_oracle_num_threads();
    if (nthreads > nw) nthreads = nw;
    double *acc = (double *)calloc((size_t)nthreads * vol, sizeof(double));
    if (!acc) { free(q32); return ORACLE_ERR_NOMEM; }
    int failed = 0;
#pragma omp parallel num_threads(nthreads)
    {
#ifdef _OPENMP
        const int tid = omp_get_thread_num();
#else
        const int tid = 0;
#endif
        double *img = acc + (size_t)tid * vol;
        double *P = (double *)malloc(sizeof(double) * 2 * slab);
        double *Pn = (double *)malloc(sizeof(double) * 2 * slab);
        if (!P || !Pn) {
#pragma omp atomic write
            failed = 1;
        }
        /* every thread must reach the work-sharing loop or none: decide together after a barrier */
        int any_failed;
#pragma omp barrier
#pragma omp atomic read
        any_failed = failed;
        if (!any_failed) {
#pragma omp for schedule(static)
            for (int iw = 0; iw < nw; ++iw) {
                const float w32 = omega[iw];
                for (size_t i = 0; i < slab; ++i) {
                    P[2 * i] = (double)P0[(size_t)iw * slab + i].re;
                    P[2 * i + 1] = (double)P0[(size_t)iw * slab + i].im;
                }
                for (int z = 0; z < nz; ++z) {
                    const float *qz = q32 + (size_t)z * slab;
                    for (int y = 0; y < ny; ++y)
                        for (int x = 0; x < nx; ++x) {                               /* T2 */
                            const int j = oracle_idx(w32, qz[(size_t)y * nx + x], ntab);
                            const oracle_c64 *row = table + (size_t)j * ntaps * ntaps;
                            double ar = 0.0, ai = 0.0;
                            for (int ky = -L; ky <= L; ++ky) {
                                const int ys = y - ky;
                                if (ys < 0 || ys >= ny) continue;
                                for (int kx = -L; kx <= L; ++kx) {
                                    const int xs = x - kx;
                                    if (xs < 0 || xs >= nx) continue;
                                    const oracle_c64 wv = row[(size_t)(L + ky) * ntaps + (L + kx)];
                                    const double pr = P[2 * ((size_t)ys * nx + xs)], pi = P[2 * ((size_t)ys * nx + xs) + 1];
                                    ar += (double)wv.re * pr - (double)wv.im * pi;
                                    ai += (double)wv.re * pi + (double)wv.im * pr;
                                }
                            }
                            Pn[2 * ((size_t)y * nx + x)] = ar;
                            Pn[2 * ((size_t)y * nx + x) + 1] = ai;
                        }
                    { double *t = P; P = Pn; Pn = t; }
                    double *islab = img + (size_t)z * slab;                          /* T3 */
                    for (size_t i = 0; i < slab; ++i) islab[i] += P[2 * i];
                }
                if (wavefield_out)
                    memcpy(wavefield_out + 2 * (size_t)iw * slab, P, sizeof(double) * 2 * slab);
            }
        }
        free(P);
        free(Pn);
    }
    if (!failed)
        for (size_t i = 0; i < vol; ++i) {
            double s = 0.0;
            for (int t = 0; t < nthreads; ++t) s += acc[(size_t)t * vol + i];
            image_out[i] = s;
        }
    free(acc);
    free(q32);
    return failed ? ORACLE_ERR_NOMEM : ORACLE_OK;
}

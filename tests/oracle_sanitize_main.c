/* Driver for tests/test_oracle_sanitize.py: runs oracle/pdm_oracle.c (compiled together with this
 * file under -fsanitize=address,undefined) on small ragged problems -- filter longer than the line,
 * nx = 1, a frequency subset, the optional wavefield output -- so that an out-of-bounds read at the
 * zero edges (R5), an overflowing index or a misuse of the per-thread accumulators aborts the run.
 * TEST INFRASTRUCTURE ONLY. */
#include <stdio.h>
#include <stdlib.h>

typedef struct { float re, im; } c64;
int pdm_oracle_migrate(int nx, int nz, int nw, double dz, const float *omega, const float *velocity,
                       const c64 *table, int ntab, int ntaps, double du, const c64 *P0,
                       const int *omega_index, int nsub, double *image_out, double *wavefield_out);
int pdm_oracle_index(float omega, float velocity, double dz, double du, int ntab);

static unsigned s = 12345u;
static float rnd(void) { s = s * 1664525u + 1013904223u; return (float)(s >> 8) / 16777216.0f; }

static int run(int nx, int nz, int nw, int L, int ntab, int nsub, int want_field)
{
    const int ntaps = 2 * L + 1;
    float *omega = malloc(sizeof(float) * nw), *vel = malloc(sizeof(float) * nz * nx);
    c64 *table = malloc(sizeof(c64) * ntab * ntaps), *P0 = malloc(sizeof(c64) * nw * nx);
    int *sub = malloc(sizeof(int) * (nsub > 0 ? nsub : 1));
    double *img = malloc(sizeof(double) * nz * nx);
    double *field = want_field ? malloc(sizeof(double) * 2 * (nsub > 0 ? nsub : nw) * nx) : NULL;
    for (int i = 0; i < nw; ++i) omega[i] = 20.0f + 180.0f * rnd();
    for (int i = 0; i < nz * nx; ++i) vel[i] = 1000.0f + 2000.0f * rnd();
    for (int i = 0; i < ntab * ntaps; ++i) { table[i].re = 0.2f * (rnd() - 0.5f); table[i].im = 0.2f * (rnd() - 0.5f); }
    for (int i = 0; i < nw * nx; ++i) { P0[i].re = rnd() - 0.5f; P0[i].im = rnd() - 0.5f; }
    for (int i = 0; i < nsub; ++i) sub[i] = (i * 7) % nw;
    const double du = 200.0 * 10.0 / 1000.0 / (ntab - 1) * 0.7;   /* some products exceed the table: clamp */
    int rc = pdm_oracle_migrate(nx, nz, nw, 10.0, omega, vel, table, ntab, ntaps, du, P0,
                                nsub > 0 ? sub : NULL, nsub, img, field);
    double cs = 0.0;
    for (int i = 0; i < nz * nx; ++i) cs += img[i];
    printf("nx=%d nz=%d nw=%d L=%d ntab=%d nsub=%d rc=%d checksum=%.17g\n", nx, nz, nw, L, ntab, nsub, rc, cs);
    free(omega); free(vel); free(table); free(P0); free(sub); free(img); free(field);
    return rc;
}

int main(void)
{
    int bad = 0;
    bad |= run(37, 5, 4, 3, 9, 0, 1);
    bad |= run(5, 4, 3, 6, 5, 0, 0);      /* filter (13 taps) longer than the line */
    bad |= run(1, 3, 2, 2, 6, 0, 1);      /* nx = 1 */
    bad |= run(64, 6, 9, 12, 33, 4, 1);   /* frequency subset + wavefield output */
    bad |= run(17, 2, 1, 0, 2, 0, 0);     /* single tap, two-row table */
    bad |= pdm_oracle_index(3.5f, 1.0f, 1.0, 1.0, 1024) != 4;
    /* argument errors must be reported, not crash */
    bad |= pdm_oracle_migrate(0, 1, 1, 1.0, NULL, NULL, NULL, 1, 1, 1.0, NULL, NULL, 0, NULL, NULL) != -1;
    return bad ? 1 : 0;
}

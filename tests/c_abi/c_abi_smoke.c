/* Plain C99 client of include/celes.h: no C++, no CUDA headers, no Python.  Reads a problem written by the test
 * (tests/test_c_abi.py), runs y = W b and out = b - T W b through the HOST-buffer entry points and writes the results.
 *
 *   c_abi_smoke <in.bin> <out.bin>
 *   in.bin : int32 N, int32 lmax, double k, double pos[N][3], double radii[N], double mie_q[N][2][lmax][2],
 *            float b[N][nmax][2]
 *   out.bin: float y[N][nmax][2], float out[N][nmax][2]
 */
#include <stdio.h>
#include <stdlib.h>

#include "celes.h"

static int fail(const char* what, int code) {
    fprintf(stderr, "c_abi_smoke: %s: %s (%d)\n", what, celes_strerror(code), code);
    return 1;
}

int main(int argc, char** argv) {
    int N = 0, lmax = 0, nmax, rc;
    double k = 0.0, *pos, *rad, *q;
    float *b, *y, *out;
    size_t nvec;
    celes_ctx* ctx = NULL;
    celes_options opt = {0};
    FILE* f;
    if (argc != 3) return 2;
    f = fopen(argv[1], "rb");
    if (!f) return 2;
    if (fread(&N, sizeof(int), 1, f) != 1 || fread(&lmax, sizeof(int), 1, f) != 1 || fread(&k, sizeof(double), 1, f) != 1) return 2;
    nmax = celes_nmax(lmax);
    if (nmax < 0) return fail("celes_nmax", nmax);
    nvec = (size_t)N * (size_t)nmax * 2;
    pos = (double*)malloc(sizeof(double) * 3 * (size_t)N);
    rad = (double*)malloc(sizeof(double) * (size_t)N);
    q = (double*)malloc(sizeof(double) * 4 * (size_t)N * (size_t)lmax);
    b = (float*)malloc(sizeof(float) * nvec);
    y = (float*)malloc(sizeof(float) * nvec);
    out = (float*)malloc(sizeof(float) * nvec);
    if (!pos || !rad || !q || !b || !y || !out) return 2;
    if (fread(pos, sizeof(double), 3 * (size_t)N, f) != 3 * (size_t)N || fread(rad, sizeof(double), (size_t)N, f) != (size_t)N ||
        fread(q, sizeof(double), 4 * (size_t)N * (size_t)lmax, f) != 4 * (size_t)N * (size_t)lmax ||
        fread(b, sizeof(float), nvec, f) != nvec) return 2;
    fclose(f);
    opt.translation = CELES_TRANSLATION_ROTATED;
    rc = celes_setup(&ctx, N, lmax, pos, rad, q, k, &opt, NULL);
    if (rc != CELES_OK) return fail("celes_setup", rc);
    rc = celes_coupling_matvec_host(ctx, b, y, NULL);
    if (rc != CELES_OK) return fail("celes_coupling_matvec_host", rc);
    rc = celes_system_matvec_host(ctx, b, out, NULL);
    if (rc != CELES_OK) return fail("celes_system_matvec_host", rc);
    celes_destroy(ctx);
    f = fopen(argv[2], "wb");
    if (!f) return 2;
    if (fwrite(y, sizeof(float), nvec, f) != nvec || fwrite(out, sizeof(float), nvec, f) != nvec) return 2;
    fclose(f);
    free(pos); free(rad); free(q); free(b); free(y); free(out);
    return 0;
}

/* A C99 consumer of libkappagen: proof that include/kappagen.h is a C ABI and not a Python
 * calling convention.  Built by tests/test_c_consumer.py with gcc; links libkappagen.so and the CUDA runtime.
 *
 *   consumer errors
 *       no GPU needed: every call below must come back with the documented status and a non-empty error text.
 *   consumer sample <dtype 0|1> <n> <kappa> <theta> <seed> <offset> <i> <vx_i> <vy_i> <vz_i> <tol> [<i> ... ]
 *       kappagen_sample into cudaMalloc'ed planes, cudaMemcpy back, compare particle i with the values given
 *       (the test takes them from the oracle) to relative tolerance tol.  Prints the largest relative error. */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <cuda_runtime_api.h>

#include "kappagen.h"

#define EXPECT(call, want)                                                                          \
    do {                                                                                            \
        int rc_ = (call);                                                                           \
        if (rc_ != (want) || ((want) != KAPPAGEN_OK && strlen(kappagen_last_error()) == 0)) {       \
            fprintf(stderr, "%s: got %d, want %d (%s)\n", #call, rc_, (int)(want), kappagen_last_error()); \
            return 1;                                                                               \
        }                                                                                           \
    } while (0)

static int errors(void) {
    float dummy[4];
    double ks, a, b, c;
    EXPECT(kappagen_version() >= 100 ? 0 : 1, 0);
    EXPECT(kappagen_params(2.0, &ks, &a, &b, &c), KAPPAGEN_OK);
    if (ks != 1.5 || !(a > 0) || !(b > 0) || !(c > 0)) return 1;
    EXPECT(kappagen_params(1.5, &ks, &a, &b, &c), KAPPAGEN_EINVAL);
    EXPECT(kappagen_params(2.0, NULL, &a, &b, &c), KAPPAGEN_ENULL);
    EXPECT(kappagen_sample(0, 2.0, 1.0, 0, 0, KAPPAGEN_F32, NULL, NULL, NULL, NULL), KAPPAGEN_OK);
    EXPECT(kappagen_sample(-1, 2.0, 1.0, 0, 0, KAPPAGEN_F32, dummy, dummy, dummy, NULL), KAPPAGEN_EINVAL);
    EXPECT(kappagen_sample(4, 1.5, 1.0, 0, 0, KAPPAGEN_F32, dummy, dummy, dummy, NULL), KAPPAGEN_EINVAL);
    EXPECT(kappagen_sample(4, 2.0, -1.0, 0, 0, KAPPAGEN_F32, dummy, dummy, dummy, NULL), KAPPAGEN_EINVAL);
    EXPECT(kappagen_sample(4, 2.0, 1.0, 0, 0, 7, dummy, dummy, dummy, NULL), KAPPAGEN_EINVAL);
    EXPECT(kappagen_sample(4, 2.0, 1.0, 0, 0, KAPPAGEN_F32, NULL, dummy, dummy, NULL), KAPPAGEN_ENULL);
    EXPECT(kappagen_sample(4, 2.0, 1.0, 0, 0, KAPPAGEN_F64, (char*)dummy + 4, dummy, dummy, NULL), KAPPAGEN_EALIGN);
    EXPECT(kappagen_sample_flags(4, 2.0, 1.0, 0, 0, KAPPAGEN_F32, 6u, dummy, dummy, dummy, NULL), KAPPAGEN_EINVAL);
    EXPECT(kappagen_sample_cells(2, 4, dummy, dummy, NULL, 0, 0, 0, KAPPAGEN_F32, dummy, dummy, dummy, NULL, 0, NULL),
           KAPPAGEN_EWORKSPACE);
    EXPECT(kappagen_sample_cells_static(KAPPAGEN_STATIC_SCRATCH_BYTES / 48 + 1, 4, dummy, dummy, NULL, 0, 0, 0, KAPPAGEN_F32,
                                        dummy, dummy, dummy, NULL), KAPPAGEN_EWORKSPACE);
    if (kappagen_cells_workspace_bytes(10, KAPPAGEN_F32) != 480 || kappagen_cells_workspace_bytes(10, KAPPAGEN_F64) != 960) return 1;
    printf("errors ok\n");
    return 0;
}

static int sample(int argc, char** argv) {
    if (argc < 13 || (argc - 8) % 5 != 0) return 2;
    const int dtype = atoi(argv[2]);
    const long long n = atoll(argv[3]);
    const double kappa = atof(argv[4]), theta = atof(argv[5]);
    const unsigned long long seed = strtoull(argv[6], NULL, 10), offset = strtoull(argv[7], NULL, 10);
    const size_t es = dtype == KAPPAGEN_F32 ? 4 : 8;
    void *d[3], *h[3];
    for (int q = 0; q < 3; ++q) {
        if (cudaMalloc(&d[q], (size_t)n * es) != cudaSuccess) { fprintf(stderr, "cudaMalloc failed\n"); return 3; }
        h[q] = malloc((size_t)n * es);
    }
    EXPECT(kappagen_sample(n, kappa, theta, seed, offset, dtype, d[0], d[1], d[2], NULL), KAPPAGEN_OK);
    for (int q = 0; q < 3; ++q)
        if (cudaMemcpy(h[q], d[q], (size_t)n * es, cudaMemcpyDeviceToHost) != cudaSuccess) { fprintf(stderr, "copy failed\n"); return 3; }
    double worst = 0.0;
    for (int k = 8; k + 4 < argc; k += 5) {
        const long long i = atoll(argv[k]);
        const double tol = atof(argv[k + 4]);
        for (int q = 0; q < 3; ++q) {
            const double want = atof(argv[k + 1 + q]);
            const double got = dtype == KAPPAGEN_F32 ? (double)((float*)h[q])[i] : ((double*)h[q])[i];
            const double err = fabs(got - want) / fabs(want);
            if (err > worst) worst = err;
            if (!(err <= tol)) { fprintf(stderr, "particle %lld component %d: got %.17g want %.17g\n", i, q, got, want); return 1; }
        }
    }
    for (int q = 0; q < 3; ++q) { cudaFree(d[q]); free(h[q]); }
    printf("sample ok, max rel err %.3e\n", worst);
    return 0;
}

int main(int argc, char** argv) {
    if (argc >= 2 && strcmp(argv[1], "errors") == 0) return errors();
    if (argc >= 2 && strcmp(argv[1], "sample") == 0) return sample(argc, argv);
    fprintf(stderr, "usage: consumer errors | consumer sample ...\n");
    return 2;
}

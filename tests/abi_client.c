/*
 * abi_client.c -- a plain C99 user of include/rfoe.h (test infrastructure: compiled with gcc by tests/test_abi.py and
 * tests/test_gpu_abi_client.py, linked against librfoe.so and the CUDA runtime; no Python, no torch in the process).
 *
 *   abi_client sizeof                      print sizeof(rfoe_stats_t) and the ABI version, no device needed
 *   abi_client expand k nocc tol out.bin   build the paper's synthetic H^p (reading R12:
 *                                          H_ij = exp(-0.5 |i-j|) sin(min(i,j)+1), 0-based), Z-RFOE with stop rule A
 *                                          through rfoe_create / rfoe_bounds / rfoe_expand / rfoe_get_stats / rfoe_destroy,
 *                                          write P (k*k doubles) to out.bin and one line of key=value pairs to stdout
 */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <cuda_runtime_api.h>

#include "rfoe.h"

static int fail(const char* what, int code)
{
    fprintf(stderr, "abi_client: %s failed: %d (%s)\n", what, code, rfoe_strerror(code));
    return 1;
}

int main(int argc, char** argv)
{
    if (argc >= 2 && strcmp(argv[1], "sizeof") == 0) {
        printf("sizeof_stats=%zu version=%d max_steps=%d\n", sizeof(rfoe_stats_t), rfoe_version(), RFOE_MAX_STEPS);
        return 0;
    }
    if (argc != 6 || strcmp(argv[1], "expand") != 0) {
        fprintf(stderr, "usage: abi_client sizeof | abi_client expand k nocc tol out.bin\n");
        return 2;
    }
    const long k = atol(argv[2]), nocc = atol(argv[3]);
    const double tol = atof(argv[4]);
    const size_t bytes = (size_t)k * (size_t)k * sizeof(double);

    double* H = (double*)malloc(bytes);
    double* P = (double*)malloc(bytes);
    if (!H || !P) return 3;
    for (long i = 0; i < k; ++i)
        for (long j = 0; j < k; ++j) {
            const long lo = i < j ? i : j, d = i < j ? j - i : i - j;
            H[i * k + j] = exp(-0.5 * (double)d) * sin((double)lo + 1.0);
        }

    double *dH = NULL, *dP = NULL;
    cudaStream_t stream = NULL;
    if (cudaMalloc((void**)&dH, bytes) != cudaSuccess || cudaMalloc((void**)&dP, bytes) != cudaSuccess) return 4;
    if (cudaStreamCreate(&stream) != cudaSuccess) return 4;
    if (cudaMemcpy(dH, H, bytes, cudaMemcpyHostToDevice) != cudaSuccess) return 4;

    rfoe_handle_t h = NULL;
    int rc = rfoe_create(&h, 0, k);
    if (rc != RFOE_OK) return fail("rfoe_create", rc);
    double emin = 0.0, emax = 0.0;
    rc = rfoe_bounds(h, dH, k, &emin, &emax, (rfoe_stream_t)stream);
    if (rc != RFOE_OK) return fail("rfoe_bounds", rc);
    rc = rfoe_expand(h, dH, k, nocc, RFOE_VARIANT_SP2, tol, dP, (rfoe_stream_t)stream);
    if (rc != RFOE_OK && rc != RFOE_ERR_NOT_CONVERGED) return fail("rfoe_expand", rc);
    rfoe_stats_t st;
    if (rfoe_get_stats(h, &st) != RFOE_OK) return fail("rfoe_get_stats", 1);
    double homo = 0.0, lumo = 0.0;
    const int rc_hl = rfoe_estimate_homo_lumo(&st, &homo, &lumo);
    if (cudaMemcpy(P, dP, bytes, cudaMemcpyDeviceToHost) != cudaSuccess) return 4;

    FILE* f = fopen(argv[5], "wb");
    if (!f || fwrite(P, 1, bytes, f) != bytes) return 5;
    fclose(f);
    printf("status=%d iterations=%d converged=%d branch=%s eps_min=%.17g eps_max=%.17g bounds_min=%.17g bounds_max=%.17g "
           "tr_PH=%.17g t_last=%.17g launches=%lld resident=%d hl_status=%d homo=%.17g lumo=%.17g\n",
           rc, st.iterations, st.converged, st.branch, st.eps_min, st.eps_max, emin, emax, st.tr_PH, st.t[st.iterations],
           (long long)st.gpu_launches, st.resident, rc_hl, homo, lumo);

    rc = rfoe_destroy(h);
    if (rc != RFOE_OK) return fail("rfoe_destroy", rc);
    cudaFree(dH);
    cudaFree(dP);
    cudaStreamDestroy(stream);
    free(H);
    free(P);
    return 0;
}

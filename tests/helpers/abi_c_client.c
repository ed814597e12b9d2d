/* A plain C99 client of include/pa.h: proves that the boundary is a C ABI (no C++ or torch types) and runs the paper's
 * loop (steps 1-5) through it with HOST buffers.  Built by tests/test_abi.py with
 *   gcc -std=c99 -pedantic -Wall -Werror -I include tests/helpers/abi_c_client.c -L<pkg> -lpa_b200
 * On a CPU-only box it must report PA_ERR_CUDA from pa_create (no fallback) and exit 3; on a GPU it prints one line per
 * temperature in the paper's output format (L179-L181) and exits 0. */
#include <stdio.h>
#include <stdlib.h>
#include "pa.h"

int main(int argc, char** argv) {
    int L = argc > 1 ? atoi(argv[1]) : 16, theta = 5, i, rc;
    int64_t R = argc > 2 ? atoll(argv[2]) : 500, R_new = 0;
    size_t ws = 0;
    pa_t* h = NULL;
    pa_obs_t o;
    double beta = 0.0, lnZ[1], e[1], C[1], grid[1] = {0.25};
    int32_t* E;

    if (pa_workspace_bytes(L, R, &ws) != PA_OK || ws == 0) return 2;
    rc = pa_create(L, R, 12345u, &h);
    if (rc == PA_ERR_CUDA) { printf("no device: %s\n", pa_strerror(rc)); return 3; }
    if (rc != PA_OK) return 4;
    E = (int32_t*)malloc(sizeof(int32_t) * (size_t)pa_capacity_of(h));
    if (!E) return 5;
    if (pa_observables(h, beta, &o) != PA_OK || pa_hist_accumulate(h, beta) != PA_OK) return 6;
    for (i = 1; i <= 10; ++i) {
        double dbeta = 0.0, next;
        if (pa_adapt_dbeta(h, 0.8, beta, 0.5, &dbeta) != PA_OK) return 7;
        next = beta + dbeta >= 0.5 ? 0.5 : beta + dbeta;
        if (pa_resample(h, beta, next, &R_new) != PA_OK) return 8;
        if (pa_sweep(h, next, theta) != PA_OK) return 9;
        if (pa_energies(h, E, NULL) != PA_OK) return 10;
        if (pa_observables(h, next, &o) != PA_OK || pa_hist_accumulate(h, next) != PA_OK) return 11;
        if (o.R != R_new || pa_population(h) != R_new) return 12;
        printf("%.6f %.8f %.8f %.8f %.8f %.8f %.8f %.8f %lld %.8f  E0=%d\n", o.beta, o.e, o.C, o.absm, o.m2, o.m4,
               o.betaF_per_N, o.S_per_N, (long long)o.R, o.lnQ, (int)E[0]);
        beta = next;
        if (beta >= 0.5) break;
    }
    if (pa_reweight(h, 1, grid, lnZ, e, C, NULL, NULL) != PA_OK) return 13;
    printf("reweighted to beta=%.2f: lnZ=%.6f e=%.6f C=%.6f\n", grid[0], lnZ[0], e[0], C[0]);
    if (pa_resample(h, 0.5, 0.4, &R_new) != PA_ERR_INVALID_ARG) return 14;     /* beta' < beta */
    {   /* one more step with the population in (pageable) host memory between the calls: pa_get_words, then pa_step_host */
        size_t nw = (size_t)((pa_capacity_of(h) + 31) / 32) * (size_t)L * (size_t)L;
        uint32_t* words = (uint32_t*)malloc(sizeof(uint32_t) * nw);
        int64_t R_host = pa_population(h);
        if (!words) return 15;
        if (pa_get_words(h, words) != PA_OK) return 16;
        if (pa_step_host(h, R_host, words, 0.5, 0.55, theta, words, E, NULL, &o, &R_new) != PA_OK) return 17;
        if (o.R != R_new || pa_population(h) != R_new || o.beta != 0.55) return 18;
        printf("host step to beta=%.2f: e=%.8f R=%lld E0=%d\n", o.beta, o.e, (long long)o.R, (int)E[0]);
        free(words);
    }
    free(E);
    pa_destroy(h);
    return 0;
}

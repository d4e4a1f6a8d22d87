/* Plain-C caller of libtt (include/tt.h): proves that the boundary is a C ABI - no C++ types, no torch.
 * Built and run by tests/test_c_abi.py:  gcc c_abi_smoke.c -I include -L <pkg> -ltt -lcudart
 * Device memory comes from the CUDA runtime API; the check is the impulse response (one block
 * column defines the operator): m = e_(j0,p0)  =>  d_i = F_{i-j0}[:, p0] for i >= j0, 0 before. */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <cuda_runtime_api.h>
#include "tt.h"

int main(void) {
    const long N_d = 3, N_m = 37, N_t = 20, j0 = 4, p0 = 11;
    const size_t nF = (size_t)N_t * N_d * N_m, nm = (size_t)N_t * N_m, nd = (size_t)N_t * N_d;
    double *F = malloc(nF * 8), *m = calloc(nm, 8), *d = malloc(nd * 8);
    for (size_t i = 0; i < nF; ++i) F[i] = sin(0.37 * (double)i) * exp(-(double)(i / (N_d * N_m)) / 6.0);
    m[j0 * N_m + p0] = 1.0;
    if (tt_version() < 100) return 2;
    tt_plan* plan = NULL;
    int st = tt_plan_create(&plan, N_d, N_m, N_t, TT_F64, TT_TIME_MAJOR, 1, F, NULL);   /* host block column */
    if (st != TT_OK) { printf("tt_plan_create: %s\n", tt_status_string(st)); return st == TT_ERR_NO_DEVICE ? 77 : 3; }
    st = tt_matvec_host(plan, m, d, NULL);
    if (st != TT_OK) { printf("tt_matvec_host: %s\n", tt_status_string(st)); return 4; }
    if (cudaDeviceSynchronize() != cudaSuccess) return 5;
    double worst = 0.0;
    for (long i = 0; i < N_t; ++i)
        for (long s = 0; s < N_d; ++s) {
            const double ref = i >= j0 ? F[((i - j0) * N_d + s) * N_m + p0] : 0.0;
            const double e = fabs(d[i * N_d + s] - ref);
            if (e > worst) worst = e;
        }
    /* error paths of the ABI */
    tt_plan* bad = NULL;
    if (tt_plan_create(&bad, 0, N_m, N_t, TT_F64, TT_TIME_MAJOR, 1, F, NULL) != TT_ERR_SHAPE) return 6;
    if (tt_plan_create(&bad, N_d, N_m, 11, TT_F64, TT_TIME_MAJOR, 1, F, NULL) != TT_ERR_UNSUPPORTED_NT) return 7;
    if (tt_matvec(plan, NULL, d, NULL) != TT_ERR_NULL) return 8;
    tt_plan_destroy(plan);
    tt_plan_destroy(NULL);
    printf("c_abi_smoke: impulse response max abs error %.3e\n", worst);
    return worst <= 1e-13 ? 0 : 1;
}

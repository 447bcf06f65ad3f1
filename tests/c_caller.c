/* A plain C caller of libet.so (include/et.h): the boundary is a C ABI, no Python in between.
 * Exit codes: 0 ok, 3 no CUDA device (et_create -> ET_ERR_CUDA), anything else a failure.
 * Built and run by tests/test_abi.py. */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>

#include "et.h"

int main(void)
{
    et_ctx *ctx = NULL;
    et_status st = et_create(&ctx, 0, NULL);
    if (st != ET_OK) {
        printf("et_create failed: %d\n", (int)st);
        return st == ET_ERR_CUDA ? 3 : 4;
    }
    /* pin P2 of DESIGN.md: the 2 + 2 square with a = sigma sqrt(2 ln 2): psi in {1/2, 1/4}, T = 0.125 (Eq. 2) */
    const double sigma = 0.3, a = sigma * sqrt(2.0 * log(2.0));
    double x[4] = {0, 0, a, 0}, xbar[4] = {0, a, a, a};
    et_result r;
    st = et_T(ctx, x, 2, xbar, 2, 2, ET_F64, ET_HOST, sigma, &r);
    if (st != ET_OK) { printf("et_T failed: %d %s\n", (int)st, et_last_error(ctx)); return 5; }
    if (fabs(r.T - 0.125) > 1e-6) { printf("T = %.9g, expected 0.125\n", r.T); return 6; }
    printf("T = %.3f\n", r.T);

    /* a small permutation test: 1500 + 1500 points of a linear congruential sequence in the unit square */
    enum { N = 1500, NPERM = 40 };
    double *p = malloc(sizeof(double) * 4 * N), *q = p + 2 * N, T_perm[NPERM];
    unsigned long long s = 88172645463325252ull;
    for (int i = 0; i < 4 * N; ++i) {
        s = s * 6364136223846793005ull + 1442695040888963407ull;
        p[i] = (double)(s >> 11) / 9007199254740992.0;
    }
    for (int i = 0; i < 2 * N; ++i) q[i] = q[i] * q[i]; /* a different density for the second sample */
    et_perm_result pr;
    st = et_permutation_test(ctx, p, NULL, N, q, NULL, N, 2, ET_F64, ET_HOST, 0.2, NPERM, 12345u, T_perm, &pr);
    if (st != ET_OK) { printf("et_permutation_test failed: %d %s\n", (int)st, et_last_error(ctx)); return 7; }
    int cnt = 0;
    for (int k = 0; k < NPERM; ++k) cnt += T_perm[k] > pr.observed.T;
    if (cnt != pr.count_gt || pr.nperm != NPERM || !(pr.observed.T > 1e-3) || pr.count_gt != 0) {
        printf("inconsistent permutation result: T = %g count = %lld (recount %d)\n", pr.observed.T, (long long)pr.count_gt, cnt);
        return 8;
    }
    /* error behaviour: sigma <= 0 leaves the output untouched */
    const double before = r.T;
    if (et_T(ctx, x, 2, xbar, 2, 2, ET_F64, ET_HOST, -1.0, &r) != ET_ERR_SIGMA || r.T != before) return 9;
    printf("permutation test ok: T = %.4e, p = %.3f\n", pr.observed.T, pr.p_value);
    free(p);
    et_destroy(ctx);
    return 0;
}

/* tests/c_abi_smoke.c -- include/bltc.h used from plain C (C11), linked against libbltc.so, no Python, no torch.
 *   ./c_abi_smoke        host-only calls (no GPU needed): version, host plan, stats, error paths
 *   ./c_abi_smoke gpu    + bltc_create / bltc_convolve / direct_convolve with HOST buffers; checks the invariant
 *                        f == c with subtraction on  =>  out == -2 c / k^2 (Eq. (20)-(21))
 * Returns 0 on success, prints the first failure otherwise.  Built and run by tests/test_c_abi_from_c.py. */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "bltc.h"

#define CHECK(cond, msg) do { if (!(cond)) { fprintf(stderr, "FAIL %s (%s)\n", msg, bltc_last_error()); return 1; } } while (0)

int main(int argc, char** argv)
{
    const int64_t N = 3000;
    double* X = (double*)malloc(3 * (size_t)N * sizeof(double));
    double* w = (double*)malloc((size_t)N * sizeof(double));
    double* f = (double*)malloc(2 * (size_t)N * sizeof(double));
    double* out = (double*)malloc(2 * (size_t)N * sizeof(double));
    unsigned long long s = 88172645463325252ULL;             /* xorshift: seeded, synthetic */
    for (int64_t i = 0; i < 3 * N; ++i) { s ^= s << 13; s ^= s >> 7; s ^= s << 17; X[i] = (double)(s >> 11) / 9007199254740992.0; }
    for (int64_t i = 0; i < N; ++i) { w[i] = 1.0 / (double)N; f[i] = 0.37; f[N + i] = -1.25; }

    CHECK(strstr(bltc_version(), "sm_100a") != NULL, "version string");
    bltc_handle h = NULL;
    CHECK(bltc_create_host_plan(&h, NULL, X, NULL, N, 1.5, 4, 100, 100) == BLTC_EINVAL, "theta >= 1 rejected");
    CHECK(strlen(bltc_last_error()) > 0, "error message set");
    CHECK(bltc_create_host_plan(&h, NULL, X, NULL, N, 0.7, 4, 100, 100) == BLTC_OK, "host plan");
    bltc_stats st;
    CHECK(bltc_get_stats(h, &st) == BLTC_OK && st.n_points == N && st.n_batches > 1 && st.n_far > 0, "stats");
    CHECK(st.shard_world == 1 && st.shard_targets == N, "unsharded plan covers all targets");
    double k[2] = {1.3, 0.6};
    CHECK(bltc_convolve(h, k, f, 2, out, 1, NULL) == BLTC_ENODEVICE, "host plan cannot convolve");
    CHECK(bltc_destroy(h) == BLTC_OK, "destroy");

    if (argc > 1 && strcmp(argv[1], "gpu") == 0) {
        CHECK(bltc_create(&h, NULL, X, w, N, 0.7, 4, 100, 100) == BLTC_OK, "bltc_create");
        CHECK(bltc_convolve(h, k, f, 2, out, 1, NULL) == BLTC_OK, "bltc_convolve (host buffers)");
        for (int64_t i = 0; i < N; ++i) {
            CHECK(fabs(out[i] - (-2.0 * 0.37 / (k[0] * k[0]))) < 1e-14, "constant f, orbital 0");
            CHECK(fabs(out[N + i] - (-2.0 * -1.25 / (k[1] * k[1]))) < 1e-13, "constant f, orbital 1");
        }
        CHECK(direct_convolve(X, f, N, X, w, f, N, k, 2, out, 1, NULL) == BLTC_OK, "direct_convolve (host buffers)");
        for (int64_t i = 0; i < N; ++i)
            CHECK(fabs(out[i] - (-2.0 * 0.37 / (k[0] * k[0]))) < 1e-14, "direct, constant f");
        double res[4];
        double* psi_new = (double*)malloc((size_t)N * sizeof(double));
        for (int64_t i = 0; i < N; ++i) psi_new[i] = 2.0;    /* psi_old == 1 (normalised: sum w = 1), psi_new == 2 */
        for (int64_t i = 0; i < N; ++i) out[i] = 1.0;
        CHECK(bltc_gi_update(w, out, f, psi_new, NULL, 0, N, -0.5, res, NULL) == BLTC_OK, "bltc_gi_update");
        /* Eq. (27): delta = <f, 1 - 2> / <2, 2> = -0.37 / 4 */
        CHECK(fabs(res[0] - (-0.5 + 0.37 / 4.0)) < 1e-14 && fabs(res[2] - 2.0) < 1e-14 && fabs(psi_new[7] - 1.0) < 1e-14,
              "gi_update closed form");
        free(psi_new);
        CHECK(bltc_destroy(h) == BLTC_OK, "destroy");
    }
    free(X); free(w); free(f); free(out);
    printf("c_abi_smoke ok\n");
    return 0;
}

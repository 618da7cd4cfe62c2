/* The C ABI of include/dies.h driven from plain C: no Python, no torch.  A homogeneous sphere of grey dust in an
 * isotropic external field (PAPER.md L49-55 sources, L87 immediate re-emission), 1e6 packages, full IRE.
 *
 * Build (from the repository root, after `python __graft_entry__.py` has built libdies.so):
 *   gcc -O2 -Iinclude -I/usr/local/cuda/include tests/c_abi/c_abi_sphere.c -o /tmp/c_abi_sphere \
 *       -Lpaper_2408_13807_b200 -ldies -L/usr/local/cuda/lib64 -lcudart -lm \
 *       -Wl,-rpath,$PWD/paper_2408_13807_b200 -Wl,-rpath,/usr/local/cuda/lib64
 * Exit code 0: the run conserved energy (escaping luminosity = injected luminosity, exact integer bookkeeping) and
 * the temperatures are finite and inside the grid.  tests/test_gpu_c_example.py builds and runs it on the GPU box. */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <cuda_runtime_api.h>
#include "dies.h"

#define CHECK(call) do { int rc_ = (call); if (rc_ != DIES_OK) { \
    fprintf(stderr, "%s -> %d: %s\n", #call, rc_, dies_last_error()); return 2; } } while (0)

enum { N = 40, K = 16, NT = 200 };

int main(void)
{
    static double r[N + 1], rho[N], freq[K], ka[K], ks[K], g[K], Tg[NT], em[NT * K], J[K];
    const double PI = 3.14159265358979323846, R = 3.0e17, tau = 5.0;
    for (int i = 0; i <= N; i++) r[i] = R * i / N;
    for (int k = 0; k < K; k++) {
        freq[k] = 1e11 * pow(10.0, 4.0 * k / (K - 1));
        ka[k] = 100.0 * (0.2 + (double)k / K);                 /* cm^2 per g of dust, rising with frequency */
        ks[k] = 50.0 * (double)k / K;
        g[k] = 0.6 * (double)k / K;
        J[k] = (k >= K / 2) ? 1e-4 * exp(-0.3 * (k - K / 2)) : 0.0;   /* external field in the upper bins */
    }
    for (int i = 0; i < N; i++) rho[i] = tau / (ka[K - 1] * R);       /* optical depth tau at the last bin */
    for (int t = 0; t < NT; t++) {
        Tg[t] = 3.0 * pow(1000.0 / 3.0, (double)t / (NT - 1));
        for (int k = 0; k < K; k++)                                    /* grows with T in every bin, colour shifts up */
            em[t * K + k] = ka[k] * pow(Tg[t] / 100.0, 4.0 + 0.25 * k);
    }

    size_t bytes = 0;
    CHECK(dies_workspace_bytes(N, K, NT, 1, &bytes));
    void* ws = NULL;
    if (cudaMalloc(&ws, bytes) != cudaSuccess) { fprintf(stderr, "cudaMalloc failed\n"); return 2; }
    dies_model* m = NULL;
    CHECK(dies_create_model(N, r, rho, K, freq, ka, ks, g, NT, Tg, em, ws, bytes, &m));
    CHECK(dies_set_sources(m, J, 0.0, NULL));
    const uint64_t n = 1000000;
    CHECK(dies_run(m, n, 7, NULL, NULL));

    double T[N], Lesc[K];
    uint64_t c[DIES_N_COUNTERS];
    CHECK(dies_get_temperature(m, T, N));
    CHECK(dies_get_escape_spectrum(m, Lesc, K));
    CHECK(dies_get_counters(m, c, DIES_N_COUNTERS));

    double L_in = 0.0, L_out = 0.0;
    for (int k = 0; k < K; k++) { L_in += J[k]; L_out += Lesc[k]; }
    L_in *= 4.0 * PI * R * R * PI;
    int bad = 0;
    for (int i = 0; i < N; i++) bad += !(T[i] > Tg[0] && T[i] < Tg[NT - 1]);
    printf("packages %llu  crossings %llu  scatterings %llu  absorptions %llu\n", (unsigned long long)c[DIES_C_PACKAGES],
           (unsigned long long)c[DIES_C_CROSSINGS], (unsigned long long)c[DIES_C_SCATTERINGS],
           (unsigned long long)c[DIES_C_ABSORPTIONS]);
    printf("T(centre) %.3f K  T(surface) %.3f K  L_out / L_in - 1 = %.3e\n", T[0], T[N - 1], L_out / L_in - 1.0);
    int ok = c[DIES_C_PACKAGES] == n && c[DIES_C_ESCAPED] + c[DIES_C_TERMINATED] == n &&
             c[DIES_C_INJECTED_RAW] == c[DIES_C_ESCAPED_RAW] + c[DIES_C_TERMINATED_RAW] &&
             fabs(L_out / L_in - 1.0) < 1e-6 && bad == 0 && T[0] < T[N - 1];
    CHECK(dies_destroy(m));
    cudaFree(ws);
    puts(ok ? "OK" : "FAILED");
    return ok ? 0 : 1;
}

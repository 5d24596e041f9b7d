/* Runs the C oracle (oracle/mesh_ft_oracle.c, included as source) under AddressSanitizer + UndefinedBehaviorSanitizer:
 * one forward and one backward in both modes on a small closed mesh, over frequencies that reach every branch (k = 0,
 * generic k, k orthogonal to an edge so that two arguments of g coincide, all three equal, a tiny |k| for the series,
 * a zero-area face).  Compiled and run by tests/test_oracle_sanitizers.py; any finding aborts with a non-zero status.
 * Prints one checksum line so that the caller can see the run did real work. */
#include "../../oracle/mesh_ft_oracle.c"

#include <stdio.h>

int main(void)
{
    /* unit-ish box [0,a]x[0,b]x[0,c], 8 vertices, 12 outward triangles, plus one degenerate (zero-area) face */
    const double a = 0.7, b = 0.45, c = 0.3;
    double v[8 * 3];
    for (int i = 0; i < 8; ++i) {
        v[3 * i + 0] = (i & 1) ? a : 0.0;
        v[3 * i + 1] = (i & 2) ? b : 0.0;
        v[3 * i + 2] = (i & 4) ? c : 0.0;
    }
    const int32_t f[13 * 3] = {0, 2, 1, 1, 2, 3, 4, 5, 6, 5, 7, 6, 0, 1, 4, 1, 5, 4, 2, 6, 3,
                               3, 6, 7, 0, 4, 2, 2, 4, 6, 1, 3, 5, 3, 7, 5, 0, 0, 3};
    const double pi = 3.14159265358979323846;
    const double k[][3] = {{0, 0, 0},       {2 * pi, -4 * pi, 6 * pi}, {2 * pi, 0, 0}, {0, 0, 2 * pi / 0.3},
                           {1e-9, 2e-9, 0}, {1e-4, -1e-4, 2e-4},       {40 * pi, 38 * pi, -36 * pi}};
    const int64_t n_k = (int64_t)(sizeof(k) / sizeof(k[0]));
    double F[2 * 7], G[2 * 7], dv[8 * 3], checksum = 0.0;
    for (int q = 0; q < n_k; ++q) {
        G[2 * q] = 1.0 - 0.1 * q;
        G[2 * q + 1] = 0.25 * q;
    }
    for (int mode = 0; mode < 2; ++mode) {
        if (oracle_mesh_ft_forward(v, 8, f, 13, &k[0][0], n_k, mode, F)) return 3;
        if (oracle_mesh_ft_backward(v, 8, f, 13, &k[0][0], n_k, mode, G, dv, NULL)) return 4;
        for (int i = 0; i < 2 * n_k; ++i) checksum += F[i];
        for (int i = 0; i < 24; ++i) checksum += dv[i];
        printf("mode %d F(0) = %.15g\n", mode, F[0]);
    }
    /* the error paths: a face index out of range is refused, not read */
    const int32_t bad[3] = {0, 1, 8};
    if (oracle_mesh_ft_forward(v, 8, bad, 1, &k[0][0], 1, 0, F) != -1) return 5;
    double g2[2], g6[6];
    oracle_g(0.3, 0.3, 0.3, g2);
    oracle_g_grad(0.3, 0.3 + 1e-12, -0.2, g6);
    printf("checksum %.15g\n", checksum + g2[0] + g6[5]);
    return 0;
}

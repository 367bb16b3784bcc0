/* ASan/UBSan driver for the CPU oracle (oracle/scarf_oracle.c, oracle/angular_oracle.c) — compiled and run by
 * tests/test_sanitizers.py with -fsanitize=address,undefined.  A two-centre s..i basis (every array of the oracle at its
 * ORACLE_MAX_L extent), both paths, a few q, two states; the angular oracle on a small grid. */
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

int oracle_nbf(int n_shells, const int32_t *shell_l);
int oracle_form_factors(int n_atoms, const double *xyz, int n_shells, const int32_t *shell_atom, const int32_t *shell_l,
                        const int32_t *shell_nprim, const double *exponents, const double *coeffs, int n_states, const double *T,
                        int64_t n_q, const double *q, double prefactor, int path, int n_threads, double *out);
int oracle_angular_moments(int n_states, int n_r, int n_theta, const double *cos_theta, const double *w_theta, int n_phi, int l_max,
                           const double *f, double *R, double *f2);

int main(void)
{
    const double xyz[6] = {0.1, 0.2, -0.8, 0.3, -0.4, 0.9};
    int32_t at[14], l[14], np[14];
    double e[16], d[16];
    int ne = 0;
    for (int a = 0; a < 2; ++a)
        for (int ll = 0; ll <= 6; ++ll) {
            const int s = a * 7 + ll, n = ll == 0 ? 2 : 1;
            at[s] = a; l[s] = ll; np[s] = n;
            for (int k = 0; k < n; ++k) { e[ne] = 0.6 + 0.3 * k + 0.05 * ll; d[ne] = 0.5 + 0.25 * k; ++ne; }
        }
    const int nbf = oracle_nbf(14, l);
    double *T = calloc((size_t)2 * nbf * nbf, sizeof(double));
    for (int i = 0; i < 2 * nbf * nbf; ++i) T[i] = ((i * 2654435761u) % 1000) / 1000.0 - 0.5;
    const double q[9] = {0, 0, 0, 0.5, -1.0, 0.25, -1.6, 0.3, 1.2};
    double out0[2 * 3 * 2], out1[2 * 3 * 2];
    int bad = oracle_form_factors(2, xyz, 14, at, l, np, e, d, 2, T, 3, q, 2.0, 0, 2, out0);
    bad += oracle_form_factors(2, xyz, 14, at, l, np, e, d, 2, T, 3, q, 2.0, 1, 2, out1);
    double worst = 0, scale = 0;
    for (int i = 0; i < 12; ++i) {
        const double dlt = out0[i] - out1[i];
        if ((dlt < 0 ? -dlt : dlt) > worst) worst = dlt < 0 ? -dlt : dlt;
        if ((out0[i] < 0 ? -out0[i] : out0[i]) > scale) scale = out0[i] < 0 ? -out0[i] : out0[i];
    }
    printf("nbf %d, path 0 vs path 1: %.2e of %.2e\n", nbf, worst, scale);
    bad += !(worst <= 1e-10 * scale);
    {   /* angular oracle: 1 state, 2 radii, 3 theta, 8 phi, l_max 2 */
        const double ct[3] = {-0.7745966692414834, 0.0, 0.7745966692414834}, wt[3] = {5.0 / 9, 8.0 / 9, 5.0 / 9};
        double f[1 * 2 * 3 * 8 * 2], R[1 * 2 * 9 * 2], f2[2];
        for (int i = 0; i < 96; ++i) f[i] = 0.01 * i - 0.3;
        bad += oracle_angular_moments(1, 2, 3, ct, wt, 8, 2, f, R, f2);
    }
    free(T);
    printf(bad ? "FAILED\n" : "OK\n");
    return bad;
}

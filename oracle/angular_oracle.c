/*
 * angular_oracle.c — CPU ORACLE for the angular moments of a form factor.  TEST INFRASTRUCTURE ONLY.
 *
 * The paper expands f_s(q) = sum_{l,m} Y_l^m(qhat) R_lm(q)                       (Eq. 57)
 * and uses the isotropic average <f_s^2>_Omega = Int dOmega/4pi |f_s(q)|^2        (Eq. 59)
 *                                              = 1/4pi sum_lm |R_lm(q)|^2          (Eq. 60).
 * By orthonormality of the Y_l^m the coefficient of Eq. (57) is the projection
 *
 *     R_lm(q) = Int dOmega conj(Y_l^m(qhat)) f_s(q qhat),
 *
 * and on the product grid of config 5 (|q| x Gauss-Legendre cos(theta) x uniform phi) that
 * integral is the plain quadrature written out below, term by term, nothing separated, tabulated or reordered:
 *
 *     R_lm(s, r)  = sum_j sum_k  w_j (2 pi / n_phi)  conj(Y_l^m(theta_j, phi_k))  f(s, r, j, k)
 *     <f^2>(s, r) = 1/(4 pi) sum_j sum_k  w_j (2 pi / n_phi)  |f(s, r, j, k)|^2,       phi_k = 2 pi k / n_phi.
 *
 * Reading (the paper does not print its Y_l^m convention): orthonormal complex spherical harmonics with the
 * Condon-Shortley phase — the convention of the Wigner-3j form of the Gaunt coefficients, Eq. (56) PAPER.md:372 —
 *     Y_l^m = sqrt((2l+1)/(4 pi) (l-m)!/(l+m)!) P_l^m(cos theta) e^{i m phi},  Y_l^{-m} = (-1)^m conj(Y_l^m),
 * P_l^m from the textbook three-term recurrence of the UNNORMALISED associated Legendre functions.
 *
 * Pins (tests/test_oracle_angular.py): Y_l^m against scipy; exact recovery of the coefficients of a band-limited
 * sum of harmonics; the Rayleigh plane-wave expansion R_lm = 4 pi i^l j_l(qa) conj(Y_l^m(ahat)); Eq. (60); <1> = 1.
 * Shares no code, table or constant with paper_2512_18010_b200/csrc/.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

/* unnormalised associated Legendre P_l^m(x), 0 <= m <= l, Condon-Shortley phase included */
static double legendre_plm(int l, int m, double x)
{
    double pmm = 1.0;
    if (m > 0) {
        const double s = sqrt((1.0 - x) * (1.0 + x));
        double f = 1.0;
        for (int i = 1; i <= m; ++i) {
            pmm *= -f * s;
            f += 2.0;
        }
    }
    if (l == m) return pmm;
    double pm1 = x * (2 * m + 1) * pmm;
    if (l == m + 1) return pm1;
    double pl = 0.0;
    for (int ll = m + 2; ll <= l; ++ll) {
        pl = (x * (2 * ll - 1) * pm1 - (ll + m - 1) * pmm) / (ll - m);
        pmm = pm1;
        pm1 = pl;
    }
    return pl;
}

static double complex sph_harm(int l, int m, double cos_theta, double phi)
{
    const int ma = m < 0 ? -m : m;
    double ratio = 1.0; /* (l-ma)!/(l+ma)! */
    for (int i = l - ma + 1; i <= l + ma; ++i) ratio /= (double)i;
    const double N = sqrt((2 * l + 1) / (4.0 * M_PI) * ratio);
    const double complex y = N * legendre_plm(l, ma, cos_theta) * cexp(I * (double)ma * phi);
    if (m >= 0) return y;
    return ((ma & 1) ? -1.0 : 1.0) * conj(y);
}

/* out[(l_max+1)^2][2], index l(l+1)+m */
void oracle_sph_harm(int l_max, double cos_theta, double phi, double *out)
{
    for (int l = 0; l <= l_max; ++l)
        for (int m = -l; m <= l; ++m) {
            const double complex y = sph_harm(l, m, cos_theta, phi);
            out[2 * (l * (l + 1) + m)] = creal(y);
            out[2 * (l * (l + 1) + m) + 1] = cimag(y);
        }
}

/* f [n_states][n_r][n_theta][n_phi][2];  R [n_states][n_r][(l_max+1)^2][2];  f2 [n_states][n_r] */
int oracle_angular_moments(int n_states, int n_r, int n_theta, const double *cos_theta, const double *w_theta, int n_phi,
                           int l_max, const double *f, double *R, double *f2)
{
    if (n_states < 0 || n_r < 0 || n_theta < 1 || n_phi < 1 || l_max < 0) return -1;
    const int nlm = (l_max + 1) * (l_max + 1);
    const double dphi = 2.0 * M_PI / n_phi;
#pragma omp parallel for collapse(2) schedule(dynamic)
    for (int s = 0; s < n_states; ++s)
        for (int r = 0; r < n_r; ++r) {
            const double *fs = f + 2 * ((size_t)(s * (size_t)n_r + r) * n_theta * n_phi);
            double acc2 = 0.0;
            for (int j = 0; j < n_theta; ++j)
                for (int k = 0; k < n_phi; ++k) {
                    const double a = fs[2 * ((size_t)j * n_phi + k)], b = fs[2 * ((size_t)j * n_phi + k) + 1];
                    acc2 += w_theta[j] * dphi * (a * a + b * b);
                }
            f2[(size_t)s * n_r + r] = acc2 / (4.0 * M_PI);
            for (int l = 0; l <= l_max; ++l)
                for (int m = -l; m <= l; ++m) {
                    double complex acc = 0.0;
                    for (int j = 0; j < n_theta; ++j)
                        for (int k = 0; k < n_phi; ++k) {
                            const double complex v = fs[2 * ((size_t)j * n_phi + k)] + I * fs[2 * ((size_t)j * n_phi + k) + 1];
                            acc += w_theta[j] * dphi * conj(sph_harm(l, m, cos_theta[j], dphi * k)) * v;
                        }
                    double *o = R + 2 * (((size_t)s * n_r + r) * nlm + l * (l + 1) + m);
                    o[0] = creal(acc);
                    o[1] = cimag(acc);
                }
        }
    return 0;
}

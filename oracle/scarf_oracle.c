/*
 * scarf_oracle.c — CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, FP64 implementation of the paper's analytic Cartesian form factor
 *
 *     f_s(q) = g * sum_{mu nu} T^s_{mu nu} * Int d^3r phi_mu(r) phi_nu(r) exp(i q.r),   g = 2
 *
 * (Eq. 35) written step by step in the paper's own sigma-parameterisation and order:
 * Appendix A normalisation (Eq. A1-A5), Gaussian product (Eq. 37-39,
 * PAPER.md:263-279), binomial shift coefficients (Eq. 40-41), pair prefactor M_ij
 * (Eq. 43), probabilist's-Hermite derivative identity (Eq. 44) and
 *   path 0: the separable V-tensor form, Eq. (45)-(46), PAPER.md:309-316;
 *   path 1: the monomial D-tensor form,  Eq. (48)-(50).
 * There is no blocking, screening, fusion or reordering beyond what those equations state; the only
 * parallelism is OpenMP over q-points.  No thresholding (SURVEY.md §8(c) reading #12).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this.  It shares no code, header, table or constant with paper_2512_18010_b200/csrc/.
 *
 * Pins (tests/test_oracle_pins.py): Eq. (A7)/(A8) worked examples, s-s and p-s closed forms, 1-D and
 * 3-D brute-force quadrature, S_mumu = 1, f(0) = g Tr(T S) = 0, f(-q) = conj f(q), translation
 * covariance, dipole small-q limit (Eq. 76-80), inversion symmetry, path 0 == path 1.
 * Parity with the PAPER'S OWN numeric outputs is unpinned: the paper prints no form-factor value.
 *
 * Readings of the paper taken here: Eq. (36) exponent is
 * i q_x x - (x-x_i)^2/2sigma_i^2 - (x-x_j)^2/2sigma_j^2; r_ij^2 is the 3-D distance between the two
 * centres; every Cartesian component is its own single-term orbital with k = 1 and is individually
 * normalised; component order a descending then b descending; Fourier sign e^{+i q.r}.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_MAX_L 6
#define ORACLE_MAX_A (2 * ORACLE_MAX_L)

typedef struct {
    int nbf;
    int *atom;          /* [nbf] centre index                                   */
    int *pw;            /* [nbf][3] Cartesian powers (a, b, c)                  */
    int *nprim;         /* [nbf]                                                */
    int *off;           /* [nbf] offset of the orbital's primitives            */
    double *sigma;      /* [sum nprim] Gaussian width, sigma = (2 alpha)^-1/2   */
    double *d;          /* [sum nprim] scale factor d_mu                        */
    double *xi;         /* [sum nprim] primitive normalisation, Eq. (A4)        */
    double *N;          /* [nbf] contracted normalisation, Eq. (A5)             */
    double *dprime;     /* [sum nprim] d' = d xi N               */
    const double *xyz;  /* borrowed [n_atoms][3]                                */
} obasis;

static void obasis_free(obasis *b)
{
    free(b->atom); free(b->pw); free(b->nprim); free(b->off);
    free(b->sigma); free(b->d); free(b->xi); free(b->N); free(b->dprime);
    memset(b, 0, sizeof *b);
}

/* Eq. (38): sigma_ij = sigma_i sigma_j / sigmabar_ij,  sigmabar_ij = sqrt(sigma_i^2 + sigma_j^2) */
static double sigma_pair(double si, double sj) { return si * sj / sqrt(si * si + sj * sj); }

/* Steps 1-3 of SURVEY.md §8(c): enumerate orbitals, Eq. (A4), Eq. (A5). */
static int obasis_build(obasis *B, int n_atoms, const double *xyz, int n_shells, const int32_t *shell_atom,
                        const int32_t *shell_l, const int32_t *shell_nprim, const double *exponents,
                        const double *coeffs)
{
    memset(B, 0, sizeof *B);
    int nbf = 0, ntot = 0;
    for (int s = 0; s < n_shells; ++s) {
        int l = shell_l[s];
        if (l < 0 || l > ORACLE_MAX_L || shell_nprim[s] < 1) return -1;
        if (shell_atom[s] < 0 || shell_atom[s] >= n_atoms) return -1;
        int nc = (l + 1) * (l + 2) / 2;
        nbf += nc;
        ntot += nc * shell_nprim[s];
    }
    B->nbf = nbf; B->xyz = xyz;
    B->atom = malloc(sizeof(int) * (nbf + 1)); B->pw = malloc(sizeof(int) * 3 * (nbf + 1));
    B->nprim = malloc(sizeof(int) * (nbf + 1)); B->off = malloc(sizeof(int) * (nbf + 1));
    B->sigma = malloc(sizeof(double) * (ntot + 1)); B->d = malloc(sizeof(double) * (ntot + 1));
    B->xi = malloc(sizeof(double) * (ntot + 1)); B->dprime = malloc(sizeof(double) * (ntot + 1));
    B->N = malloc(sizeof(double) * (nbf + 1));
    int mu = 0, o = 0, p0 = 0;
    for (int s = 0; s < n_shells; ++s) {
        int l = shell_l[s], np = shell_nprim[s];
        for (int a = l; a >= 0; --a)
            for (int b = l - a; b >= 0; --b) {
                int c = l - a - b;
                B->atom[mu] = shell_atom[s];
                B->pw[3 * mu] = a; B->pw[3 * mu + 1] = b; B->pw[3 * mu + 2] = c;
                B->nprim[mu] = np; B->off[mu] = o;
                for (int k = 0; k < np; ++k) {
                    double alpha = exponents[p0 + k];
                    if (!(alpha > 0.0)) return -1;
                    double sg = 1.0 / sqrt(2.0 * alpha);
                    B->sigma[o + k] = sg;
                    B->d[o + k] = coeffs[p0 + k];
                    /* Eq. (A4), one Cartesian term with k = 1: K = 2a, 2b, 2c */
                    double prod = pow(sg, 1 + 2 * a) * tgamma(a + 0.5) * pow(sg, 1 + 2 * b) * tgamma(b + 0.5) *
                                  pow(sg, 1 + 2 * c) * tgamma(c + 0.5);
                    B->xi[o + k] = 1.0 / sqrt(prod);
                }
                /* Eq. (A5) */
                double sum = 0.0;
                for (int k = 0; k < np; ++k)
                    for (int kp = 0; kp < np; ++kp) {
                        double smn = sigma_pair(B->sigma[o + k], B->sigma[o + kp]);
                        double r2s = sqrt(2.0) * smn;
                        double prod = pow(r2s, 1 + 2 * a) * tgamma((2 * a + 1) / 2.0) * pow(r2s, 1 + 2 * b) *
                                      tgamma((2 * b + 1) / 2.0) * pow(r2s, 1 + 2 * c) * tgamma((2 * c + 1) / 2.0);
                        sum += B->d[o + k] * B->d[o + kp] * B->xi[o + k] * B->xi[o + kp] * prod;
                    }
                B->N[mu] = 1.0 / sqrt(sum);
                for (int k = 0; k < np; ++k) B->dprime[o + k] = B->d[o + k] * B->xi[o + k] * B->N[mu];
                o += np;
                ++mu;
            }
        p0 += np;
    }
    return 0;
}

static double binom(int n, int k)
{
    if (k < 0 || k > n) return 0.0;
    double r = 1.0;
    for (int i = 1; i <= k; ++i) r = r * (n - k + i) / i;
    return r;
}

static double ipow(double x, int n)
{
    double r = 1.0;
    for (int i = 0; i < n; ++i) r *= x;
    return r;
}

static double factorial(int n)
{
    double r = 1.0;
    for (int i = 2; i <= n; ++i) r *= i;
    return r;
}

/* Eq. (41): b^A_ij, A = 0..a_i+a_j, with u = X_ij - x_i, v = X_ij - x_j */
static void shift_coeffs(int ai, int aj, double u, double v, double *b)
{
    int al = ai + aj;
    for (int A = 0; A <= al; ++A) {
        int klo = ai - A > 0 ? ai - A : 0;
        int khi = ai < al - A ? ai : al - A;
        double s = 0.0;
        for (int k = klo; k <= khi; ++k) s += binom(ai, k) * binom(aj, al - k - A) * ipow(u, k) * ipow(v, al - k - A);
        b[A] = s;
    }
}

/* probabilist's Hermite polynomials by the textbook recurrence He_{n+1} = x He_n - n He_{n-1}
 * ("generated using recurrence relations") */
static void hermite_He(int nmax, double x, double *He)
{
    He[0] = 1.0;
    if (nmax >= 1) He[1] = x;
    for (int n = 1; n < nmax; ++n) He[n + 1] = x * He[n] - n * He[n - 1];
}

static double complex ipow_i(int n) /* i^n */
{
    switch (n & 3) {
    case 0: return 1.0;
    case 1: return I;
    case 2: return -1.0;
    default: return -I;
    }
}

/* Eq. (46): V_ij(q) = exp(i q X_ij - q^2 sigma_ij^2 / 2) sum_A b^A (i sigma_ij)^A He_A(q sigma_ij) */
static double complex V_tensor_1d(int ai, int aj, double xi_, double xj_, double si, double sj, double q)
{
    double sij = sigma_pair(si, sj);
    double X = sij * sij * (xi_ / (si * si) + xj_ / (sj * sj)); /* Eq. (39) */
    double b[ORACLE_MAX_A + 1], He[ORACLE_MAX_A + 1];
    int al = ai + aj;
    shift_coeffs(ai, aj, X - xi_, X - xj_, b);
    hermite_He(al, q * sij, He);
    double complex s = 0.0;
    for (int A = 0; A <= al; ++A) s += b[A] * ipow_i(A) * ipow(sij, A) * He[A];
    return cexp(I * q * X - 0.5 * q * q * sij * sij) * s;
}

/* Eq. (50): C^u_ij = i^u sum_m b^{u+2m} sigma_ij^{2(u+m)} (u+2m)! / (m! u! 2^m),  u = 0..alpha_ij */
static void C_coeffs_1d(int ai, int aj, double xi_, double xj_, double si, double sj, double complex *C)
{
    double sij = sigma_pair(si, sj);
    double X = sij * sij * (xi_ / (si * si) + xj_ / (sj * sj));
    double b[ORACLE_MAX_A + 1];
    int al = ai + aj;
    shift_coeffs(ai, aj, X - xi_, X - xj_, b);
    for (int u = 0; u <= al; ++u) {
        double s = 0.0;
        for (int m = 0; m <= (al - u) / 2; ++m)
            s += b[u + 2 * m] * ipow(sij, 2 * (u + m)) * factorial(u + 2 * m) / (factorial(m) * factorial(u) * ipow(2.0, m));
        C[u] = ipow_i(u) * s;
    }
}

/* Eq. (43) with k_i = k_j = 1:  M_ij = d'_i d'_j sigma_ij^3 exp(-r_ij^2 / (2 sigmabar_ij^2)) */
static double M_prefactor(double dpi, double dpj, double si, double sj, const double *ri, const double *rj)
{
    double sij = sigma_pair(si, sj);
    double sbar2 = si * si + sj * sj;
    double r2 = 0.0;
    for (int k = 0; k < 3; ++k) r2 += (ri[k] - rj[k]) * (ri[k] - rj[k]);
    return dpi * dpj * sij * sij * sij * exp(-r2 / (2.0 * sbar2));
}

/* (2 pi)^{3/2} sum_{k k'} M V^x V^y V^z for one ordered orbital pair at one q  (inner sums of Eq. 45) */
static double complex pair_integral_V(const obasis *B, int mu, int nu, const double *q)
{
    const double *ri = B->xyz + 3 * B->atom[mu], *rj = B->xyz + 3 * B->atom[nu];
    const int *pi_ = B->pw + 3 * mu, *pj = B->pw + 3 * nu;
    double complex s = 0.0;
    for (int k = 0; k < B->nprim[mu]; ++k)
        for (int kp = 0; kp < B->nprim[nu]; ++kp) {
            double si = B->sigma[B->off[mu] + k], sj = B->sigma[B->off[nu] + kp];
            double M = M_prefactor(B->dprime[B->off[mu] + k], B->dprime[B->off[nu] + kp], si, sj, ri, rj);
            double complex V = 1.0;
            for (int ax = 0; ax < 3; ++ax) V *= V_tensor_1d(pi_[ax], pj[ax], ri[ax], rj[ax], si, sj, q[ax]);
            s += M * V;
        }
    return pow(2.0 * M_PI, 1.5) * s;
}

/* Same quantity by Eq. (48)-(50): exp(-q^2 sigma^2/2) e^{i q.R} sum_{uvw} D^{uvw} q_x^u q_y^v q_z^w */
static double complex pair_integral_D(const obasis *B, int mu, int nu, const double *q)
{
    const double *ri = B->xyz + 3 * B->atom[mu], *rj = B->xyz + 3 * B->atom[nu];
    const int *pi_ = B->pw + 3 * mu, *pj = B->pw + 3 * nu;
    double complex s = 0.0;
    double q2 = q[0] * q[0] + q[1] * q[1] + q[2] * q[2];
    for (int k = 0; k < B->nprim[mu]; ++k)
        for (int kp = 0; kp < B->nprim[nu]; ++kp) {
            double si = B->sigma[B->off[mu] + k], sj = B->sigma[B->off[nu] + kp];
            double sij = sigma_pair(si, sj);
            double M = M_prefactor(B->dprime[B->off[mu] + k], B->dprime[B->off[nu] + kp], si, sj, ri, rj);
            double complex C[3][ORACLE_MAX_A + 1];
            double qR = 0.0;
            for (int ax = 0; ax < 3; ++ax) {
                C_coeffs_1d(pi_[ax], pj[ax], ri[ax], rj[ax], si, sj, C[ax]);
                qR += q[ax] * sij * sij * (ri[ax] / (si * si) + rj[ax] / (sj * sj)); /* q . R_ij, Eq. (39) */
            }
            double complex poly = 0.0;
            for (int u = 0; u <= pi_[0] + pj[0]; ++u)
                for (int v = 0; v <= pi_[1] + pj[1]; ++v)
                    for (int w = 0; w <= pi_[2] + pj[2]; ++w) {
                        double complex D = M * C[0][u] * C[1][v] * C[2][w]; /* Eq. (49) */
                        poly += D * ipow(q[0], u) * ipow(q[1], v) * ipow(q[2], w);
                    }
            s += exp(-0.5 * q2 * sij * sij) * cexp(I * qR) * poly;
        }
    return pow(2.0 * M_PI, 1.5) * s;
}

/* ------------------------------------------------------------------------------------------ */
/* exported API                                                                               */
/* ------------------------------------------------------------------------------------------ */

int oracle_nbf(int n_shells, const int32_t *shell_l)
{
    int nbf = 0;
    for (int s = 0; s < n_shells; ++s) nbf += (shell_l[s] + 1) * (shell_l[s] + 2) / 2;
    return nbf;
}

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* xi_out: per (orbital, primitive) in orbital order; N_out: per orbital.  n_tot_out: length of xi_out. */
int oracle_norms(int n_atoms, const double *xyz, int n_shells, const int32_t *shell_atom, const int32_t *shell_l,
                 const int32_t *shell_nprim, const double *exponents, const double *coeffs, double *xi_out,
                 double *N_out)
{
    obasis B;
    if (obasis_build(&B, n_atoms, xyz, n_shells, shell_atom, shell_l, shell_nprim, exponents, coeffs)) {
        obasis_free(&B);
        return -1;
    }
    int ntot = B.nbf ? B.off[B.nbf - 1] + B.nprim[B.nbf - 1] : 0;
    memcpy(xi_out, B.xi, sizeof(double) * ntot);
    memcpy(N_out, B.N, sizeof(double) * B.nbf);
    obasis_free(&B);
    return 0;
}

/* out[n_states][n_q][2] (re, im).  path 0: Eq. (45)/(46); path 1: Eq. (48)-(50).  T[n_states][nbf][nbf]. */
int oracle_form_factors(int n_atoms, const double *xyz, int n_shells, const int32_t *shell_atom,
                        const int32_t *shell_l, const int32_t *shell_nprim, const double *exponents,
                        const double *coeffs, int n_states, const double *T, int64_t n_q, const double *q,
                        double prefactor, int path, int n_threads, double *out)
{
    obasis B;
    if (obasis_build(&B, n_atoms, xyz, n_shells, shell_atom, shell_l, shell_nprim, exponents, coeffs)) {
        obasis_free(&B);
        return -1;
    }
    const int nbf = B.nbf;
#ifdef _OPENMP
    if (n_threads <= 0) n_threads = omp_get_max_threads();
#else
    n_threads = 1;
#endif
#pragma omp parallel for schedule(dynamic, 1) num_threads(n_threads)
    for (int64_t iq = 0; iq < n_q; ++iq) {
        double complex *acc = calloc((size_t)n_states, sizeof(double complex));
        const double *qq = q + 3 * iq;
        for (int mu = 0; mu < nbf; ++mu)
            for (int nu = 0; nu < nbf; ++nu) {
                double complex Iq = path == 0 ? pair_integral_V(&B, mu, nu, qq) : pair_integral_D(&B, mu, nu, qq);
                for (int s = 0; s < n_states; ++s) acc[s] += T[((size_t)s * nbf + mu) * nbf + nu] * Iq;
            }
        for (int s = 0; s < n_states; ++s) {
            out[((size_t)s * n_q + iq) * 2] = prefactor * creal(acc[s]);
            out[((size_t)s * n_q + iq) * 2 + 1] = prefactor * cimag(acc[s]);
        }
        free(acc);
    }
    obasis_free(&B);
    return 0;
}

/* I[nbf][nbf][2] = Int phi_mu phi_nu e^{i q.r} at ONE q (path 0).  At q = 0 its real part is the overlap S. */
int oracle_pair_matrix(int n_atoms, const double *xyz, int n_shells, const int32_t *shell_atom,
                       const int32_t *shell_l, const int32_t *shell_nprim, const double *exponents,
                       const double *coeffs, const double *q, int path, double *I_out)
{
    obasis B;
    if (obasis_build(&B, n_atoms, xyz, n_shells, shell_atom, shell_l, shell_nprim, exponents, coeffs)) {
        obasis_free(&B);
        return -1;
    }
    const int nbf = B.nbf;
#pragma omp parallel for schedule(dynamic, 1)
    for (int mu = 0; mu < nbf; ++mu)
        for (int nu = 0; nu < nbf; ++nu) {
            double complex v = path == 0 ? pair_integral_V(&B, mu, nu, q) : pair_integral_D(&B, mu, nu, q);
            I_out[((size_t)mu * nbf + nu) * 2] = creal(v);
            I_out[((size_t)mu * nbf + nu) * 2 + 1] = cimag(v);
        }
    obasis_free(&B);
    return 0;
}

/* 1-D building blocks exposed so tests can pin them against quadrature / scipy. */
void oracle_V1d(int ai, int aj, double xi_, double xj_, double sigma_i, double sigma_j, double q, double *out2)
{
    double complex v = V_tensor_1d(ai, aj, xi_, xj_, sigma_i, sigma_j, q);
    out2[0] = creal(v);
    out2[1] = cimag(v);
}

void oracle_C1d(int ai, int aj, double xi_, double xj_, double sigma_i, double sigma_j, double *out /* [ai+aj+1][2] */)
{
    double complex C[ORACLE_MAX_A + 1];
    C_coeffs_1d(ai, aj, xi_, xj_, sigma_i, sigma_j, C);
    for (int u = 0; u <= ai + aj; ++u) {
        out[2 * u] = creal(C[u]);
        out[2 * u + 1] = cimag(C[u]);
    }
}

void oracle_hermite_He(int nmax, double x, double *He) { hermite_He(nmax, x, He); }

void oracle_shift_coeffs(int ai, int aj, double u, double v, double *b) { shift_coeffs(ai, aj, u, v, b); }

// pure.cu — pure (real solid-harmonic) d, f, g, h and i shells (the paper builds such orbitals as
// several Cartesian terms with prefactors, Eq. (A2), e.g. 3d_{x^2-y^2}).
//
// The kernels work in the Cartesian basis.  A pure shell of angular momentum l has 2l+1 functions
//     phi_{lm}(r) = N_m S_lm(x, y, z) R(r),   m = -l..l,   S_lm = real solid harmonic (homogeneous polynomial of degree l),
// each a fixed linear combination of the shell's (l+1)(l+2)/2 Cartesian components, so the user's transition matrices
// are mapped once per set_transitions:   T_cart = C T_user C^T,   C = blockdiag(C_l), C_l [n_cart(l)][2l+1]
// (`transform_T_kernel`), and the overlap back:   S_user = C^T S_cart C   (host).
//
// C_l does not depend on the exponents or the contraction: every component of a shell carries the same radial part, and
// with individually normalised components (reading #9) the same-shell overlap is
//     <chi_c | chi_c'> = prod_axis (a+a'-1)!! / sqrt((2a-1)!!(2a'-1)!!)   (0 if any a+a' is odd),
// so   C_l[c][m] = N_m w_cm sqrt((2a-1)!!(2b-1)!!(2c-1)!!),  w_cm = coefficient of x^a y^b z^c in S_lm,  N_m from
// C_m^T S C_m = 1.  Order m = -l..l; sign convention S_{l,m>0} ~ Re (x+iy)^m ..., S_{l,m<0} ~ Im (x+iy)^|m| ...:
// d: xy, yz, 2z^2-x^2-y^2, xz, x^2-y^2;  f: 3x^2y-y^3, xyz, y(4z^2-x^2-y^2), z(2z^2-3x^2-3y^2), x(4z^2-x^2-y^2), z(x^2-y^2), x^3-3xy^2.
#include <cmath>
#include <cstring>

#include "kernels.cuh"

namespace scarf {

namespace {

// Coefficients w[c] of the Cartesian monomials x^a y^b z^c (component order of the library) in the real solid harmonic
// S_lm, any overall scale (the column is normalised afterwards), from the closed form
//   S_{l, m>=0} = Pi_l^m(z, r^2) A_m(x, y),   S_{l, m<0} = Pi_l^{|m|}(z, r^2) B_{|m|}(x, y),
//   A_m + i B_m = (x + i y)^m,
//   Pi_l^m = sum_{k=0}^{floor((l-m)/2)} (-1)^k C(l,k) C(2l-2k, l) (l-2k)!/(l-2k-m)! r^{2k} z^{l-2k-m},   r^2 = x^2 + y^2 + z^2,
// which reproduces the tabulated d and f functions of the header comment (signs included) and extends them to g, h, i.
// l = 1 keeps the Cartesian order x, y, z (index m + 1 = 0, 1, 2).
double binom(int n, int k)
{
    double r = 1.0;
    for (int i = 1; i <= k; ++i) r = r * (double)(n - k + i) / (double)i;
    return r;
}

void solid_harmonic_coeffs(int l, int m, double* w)   // w[ncart(l)]
{
    const int nc = ncart(l);
    for (int c = 0; c < nc; ++c) w[c] = 0.0;
    if (l == 0) { w[0] = 1.0; return; }
    if (l == 1) { w[m + 1] = 1.0; return; }
    auto comp_index = [&](int a, int b) {              // a descending, then b descending
        int idx = 0;
        for (int aa = l; aa > a; --aa) idx += l - aa + 1;
        return idx + (l - a - b);
    };
    const int ma = m < 0 ? -m : m;
    for (int k = 0; 2 * k <= l - ma; ++k) {
        double ck = ((k & 1) ? -1.0 : 1.0) * binom(l, k) * binom(2 * l - 2 * k, l);
        for (int i = 0; i < ma; ++i) ck *= (double)(l - 2 * k - i);      // (l-2k)!/(l-2k-m)!
        // (x + i y)^ma: term x^p y^(ma-p) carries i^(ma-p); A takes the real part, B the imaginary part
        for (int p = 0; p <= ma; ++p) {
            const int e = ma - p;
            double cp = 0.0;
            if (m >= 0 && (e & 1) == 0) cp = ((e / 2) & 1) ? -1.0 : 1.0;
            if (m < 0 && (e & 1) == 1) cp = (((e - 1) / 2) & 1) ? -1.0 : 1.0;
            if (cp == 0.0) continue;
            cp *= binom(ma, p);
            // r^{2k} = sum_{i+j+n=k} k!/(i! j! n!) x^{2i} y^{2j} z^{2n}
            for (int i = 0; i <= k; ++i)
                for (int j = 0; i + j <= k; ++j)       // the z power follows: l - a - b
                    w[comp_index(p + 2 * i, e + 2 * j)] += ck * cp * binom(k, i) * binom(k - i, j);
        }
    }
}

double dfact_odd(int n)   // n!! for odd n >= -1
{
    double r = 1.0;
    for (int k = n; k > 1; k -= 2) r *= k;
    return r;
}

__global__ void __launch_bounds__(256) transform_T_kernel(const double* __restrict__ Tu, double* __restrict__ Tc, int n_states,
                                                          int nbf_u, int nbf_c, const int* __restrict__ nnz,
                                                          const int* __restrict__ uidx, const double* __restrict__ ucoef)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long per = (long long)nbf_c * nbf_c;
    if (i >= per * n_states) return;
    const int s = (int)(i / per), mu = (int)((i % per) / nbf_c), nu = (int)(i % nbf_c);
    const double* T = Tu + (size_t)s * nbf_u * nbf_u;
    double acc = 0.0;
    for (int k = 0; k < nnz[mu]; ++k) {
        const double* row = T + (size_t)uidx[mu * kPureMaxNnz + k] * nbf_u;
        double r = 0.0;
        for (int k2 = 0; k2 < nnz[nu]; ++k2) r = fma(ucoef[nu * kPureMaxNnz + k2], row[uidx[nu * kPureMaxNnz + k2]], r);
        acc = fma(ucoef[mu * kPureMaxNnz + k], r, acc);
    }
    Tc[i] = acc;
}

}  // namespace

// C_l [ncart(l)][2l+1] (row-major) for a pure shell; Cartesian component order of the library.
void pure_matrix(int l, double* C)
{
    const int nc = ncart(l), np = 2 * l + 1;
    std::memset(C, 0, sizeof(double) * (size_t)nc * np);
    int pw[kMaxCart][3];
    double cf[kMaxCart];
    for (int c = 0; c < nc; ++c) {
        component_powers(l, c, pw[c]);
        cf[c] = component_factor(l, c);
    }
    for (int m = -l; m <= l; ++m) {
        double w[kMaxCart], v[kMaxCart] = {};
        solid_harmonic_coeffs(l, m, w);
        for (int c = 0; c < nc; ++c) v[c] = w[c] / cf[c];
        double nrm = 0.0;
        for (int c = 0; c < nc; ++c)
            for (int d = 0; d < nc; ++d) {
                if (v[c] == 0.0 || v[d] == 0.0) continue;
                double s = cf[c] * cf[d];
                bool zero = false;
                for (int ax = 0; ax < 3; ++ax) {
                    const int e = pw[c][ax] + pw[d][ax];
                    if (e & 1) { zero = true; break; }
                    s *= dfact_odd(e - 1);
                }
                if (!zero) nrm += v[c] * s * v[d];
            }
        const double N = 1.0 / std::sqrt(nrm);
        for (int c = 0; c < nc; ++c) C[c * np + (m + l)] = N * v[c];
    }
}

// Per Cartesian basis function: the user functions it draws from and the coefficients (row of C).  Returns nbf_user.
int build_pure_map(int n_shells, const int32_t* shell_l, const int32_t* shell_pure, std::vector<int>& nnz, std::vector<int>& uidx,
                   std::vector<double>& ucoef)
{
    int nbf_c = 0, nbf_u = 0;
    for (int i = 0; i < n_shells; ++i) nbf_c += ncart(shell_l[i]);
    nnz.assign((size_t)nbf_c, 0);
    uidx.assign((size_t)nbf_c * kPureMaxNnz, 0);
    ucoef.assign((size_t)nbf_c * kPureMaxNnz, 0.0);
    int c0 = 0;
    for (int i = 0; i < n_shells; ++i) {
        const int l = shell_l[i], nc = ncart(l);
        const bool pure = shell_pure && shell_pure[i] != 0 && l >= 2;
        if (!pure) {
            for (int c = 0; c < nc; ++c) {
                nnz[c0 + c] = 1;
                uidx[(size_t)(c0 + c) * kPureMaxNnz] = nbf_u + c;
                ucoef[(size_t)(c0 + c) * kPureMaxNnz] = 1.0;
            }
            nbf_u += nc;
        } else {
            const int np = 2 * l + 1;
            double C[kMaxCart * (2 * kMaxL + 1)];
            pure_matrix(l, C);
            for (int c = 0; c < nc; ++c) {
                int k = 0;
                for (int m = 0; m < np; ++m)
                    if (C[c * np + m] != 0.0) {
                        uidx[(size_t)(c0 + c) * kPureMaxNnz + k] = nbf_u + m;
                        ucoef[(size_t)(c0 + c) * kPureMaxNnz + k] = C[c * np + m];
                        ++k;
                    }
                nnz[c0 + c] = k;
            }
            nbf_u += np;
        }
        c0 += nc;
    }
    return nbf_u;
}

cudaError_t launch_transform_T(const double* Tu, double* Tc, int n_states, int nbf_u, int nbf_c, const int* nnz, const int* uidx,
                               const double* ucoef, cudaStream_t st)
{
    const long long n = (long long)n_states * nbf_c * nbf_c;
    if (n <= 0) return cudaSuccess;
    transform_T_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(Tu, Tc, n_states, nbf_u, nbf_c, nnz, uidx, ucoef);
    return cudaGetLastError();
}

}  // namespace scarf

// angular.cu — angular moments of S4's output on a spherical product grid.
//
//   f_s(q) = sum_lm Y_l^m(qhat) R_lm(q)                         Eq. (57)
//   R_lm(q) = Int dOmega conj(Y_l^m) f_s                        (orthonormality; quadrature on the grid of config 5)
//   <f_s^2>_Omega = Int dOmega/4pi |f_s|^2                      Eq. (59)
//
// Grid: f[state][r][theta_j][phi_k], theta nodes/weights given (Gauss-Legendre), phi_k = 2 pi k / n_phi.  The
// quadrature separates: conj(Y_l^m) = Ybar_lm(theta) e^{-i m phi} with Ybar real, so
//   step 1 (phi_dft_kernel):   F_m(row) = (2 pi/n_phi) sum_k e^{-i m phi_k} f(row, k),  m = -l_max..l_max,
//                              and rowsum2(row) = (2 pi/n_phi) sum_k |f(row, k)|^2          (row = state, r, theta)
//   step 2 (legendre_kernel):  R_lm(state, r) = sum_j w_j Ybar_lm(theta_j) F_m(state, r, j),
//                              <f^2>(state, r) = 1/(4 pi) sum_j w_j rowsum2(state, r, j).
// Step 1 reads f once (the only large array: 201 MB on config 5) and is a small dense contraction
// [2 l_max + 1] x [n_phi] per row, done in FP64 FMAs from shared memory; step 2 is tiny.  Ybar (host, fully
// normalised three-term recurrence) and the twiddles are tabulated once per call.
#include <cmath>
#include <vector>

#include "kernels.cuh"

namespace scarf {

namespace {

constexpr int kThreads = 128;

// rows_per_cta rows of n_phi complex values + n_phi twiddles in dynamic shared memory
__global__ void __launch_bounds__(kThreads) phi_dft_kernel(const double2* __restrict__ f, const double2* __restrict__ tw,
                                                           long long n_rows, int n_phi, int l_max, int rows_per_cta,
                                                           double2* __restrict__ F, double* __restrict__ rowsum2)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* s_tw = reinterpret_cast<double2*>(smem_raw);
    double2* s_f = s_tw + n_phi;
    const long long row0 = (long long)blockIdx.x * rows_per_cta;
    const int nrow = (int)min((long long)rows_per_cta, n_rows - row0);
    const int n_m = 2 * l_max + 1;
    for (int k = threadIdx.x; k < n_phi; k += kThreads) s_tw[k] = tw[k];
    const double2* src = f + (size_t)row0 * n_phi;
    for (int i = threadIdx.x; i < nrow * n_phi; i += kThreads) s_f[i] = src[i];
    __syncthreads();
    const double scale = 6.283185307179586476925286766559 / (double)n_phi;
    // one work item = (pair of rows, |m|): the twiddle e^{-i m phi_k} serves +m and -m (conjugate) and both rows,
    // 16 FMAs per 3 shared-memory loads
    const int n_rp = (nrow + 1) / 2, n_ma = l_max + 1;
    for (int o = threadIdx.x; o < n_rp * n_ma; o += kThreads) {
        const int rp = o / n_ma, ma = o % n_ma;
        const int r0 = 2 * rp, r1 = min(2 * rp + 1, nrow - 1);
        const double2* f0 = s_f + r0 * n_phi;
        const double2* f1 = s_f + r1 * n_phi;
        double pr0 = 0.0, pi0 = 0.0, nr0 = 0.0, ni0 = 0.0, pr1 = 0.0, pi1 = 0.0, nr1 = 0.0, ni1 = 0.0;
        int idx = 0;
        for (int k = 0; k < n_phi; ++k) {
            const double2 t = s_tw[idx];                    // (cos, -sin)(2 pi idx / n_phi) = e^{-i ma phi_k}
            const double2 u = f0[k], v = f1[k];
            // +ma: f * t ;  -ma: f * conj(t)
            pr0 = fma(u.x, t.x, pr0); pr0 = fma(-u.y, t.y, pr0);
            pi0 = fma(u.x, t.y, pi0); pi0 = fma(u.y, t.x, pi0);
            nr0 = fma(u.x, t.x, nr0); nr0 = fma(u.y, t.y, nr0);
            ni0 = fma(-u.x, t.y, ni0); ni0 = fma(u.y, t.x, ni0);
            pr1 = fma(v.x, t.x, pr1); pr1 = fma(-v.y, t.y, pr1);
            pi1 = fma(v.x, t.y, pi1); pi1 = fma(v.y, t.x, pi1);
            nr1 = fma(v.x, t.x, nr1); nr1 = fma(v.y, t.y, nr1);
            ni1 = fma(-v.x, t.y, ni1); ni1 = fma(v.y, t.x, ni1);
            idx += ma;
            if (idx >= n_phi) idx -= n_phi;
        }
        double2* F0 = F + (size_t)(row0 + r0) * n_m + l_max;
        F0[ma] = make_double2(pr0 * scale, pi0 * scale);
        F0[-ma] = make_double2(nr0 * scale, ni0 * scale);
        if (r1 != r0) {
            double2* F1 = F + (size_t)(row0 + r1) * n_m + l_max;
            F1[ma] = make_double2(pr1 * scale, pi1 * scale);
            F1[-ma] = make_double2(nr1 * scale, ni1 * scale);
        }
    }
    // |f|^2 row sums: one warp per row, lanes stride over k, fixed-order shuffle tree (deterministic)
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int row = warp; row < nrow; row += kThreads / 32) {
        const double2* fr = s_f + row * n_phi;
        double acc = 0.0;
        for (int k = lane; k < n_phi; k += 32) acc = fma(fr[k].x, fr[k].x, fma(fr[k].y, fr[k].y, acc));
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
        if (lane == 0) rowsum2[row0 + row] = acc * scale;
    }
}

// one CTA per (state, r): R[l(l+1)+m] = sum_j Yw[j][l(l+1)/2+|m|] * (-1)^{m<0 ? m : 0} * F[j][m + l_max]
__global__ void __launch_bounds__(kThreads) legendre_kernel(const double2* __restrict__ F, const double* __restrict__ rowsum2,
                                                            const double* __restrict__ Yw, const double* __restrict__ w_theta,
                                                            int n_theta, int l_max, double2* __restrict__ R, double* __restrict__ f2)
{
    const long long sr = blockIdx.x;
    const int n_m = 2 * l_max + 1, nlm = (l_max + 1) * (l_max + 1), nhalf = (l_max + 1) * (l_max + 2) / 2;
    const double2* Fr = F + (size_t)sr * n_theta * n_m;
    for (int o = threadIdx.x; o < nlm; o += kThreads) {
        int l = (int)sqrt((double)o);
        while (l * l > o) --l;
        while ((l + 1) * (l + 1) <= o) ++l;
        const int m = o - l * (l + 1), ma = m < 0 ? -m : m;
        const double sgn = (m < 0 && (ma & 1)) ? -1.0 : 1.0;
        double ar = 0.0, ai = 0.0;
        for (int j = 0; j < n_theta; ++j) {
            const double y = Yw[(size_t)j * nhalf + l * (l + 1) / 2 + ma];
            const double2 v = Fr[(size_t)j * n_m + (m + l_max)];
            ar = fma(y, v.x, ar);
            ai = fma(y, v.y, ai);
        }
        R[(size_t)sr * nlm + o] = make_double2(sgn * ar, sgn * ai);
    }
    if (f2 != nullptr && threadIdx.x == 0) {
        double acc = 0.0;
        for (int j = 0; j < n_theta; ++j) acc = fma(w_theta[j], rowsum2[(size_t)sr * n_theta + j], acc);
        f2[sr] = acc / 12.566370614359172953850573533118;
    }
}

}  // namespace

// Yw[j][l(l+1)/2 + m] = w_j * N_lm P_l^m(x_j), 0 <= m <= l <= l_max: fully normalised recurrence (orthonormal Y_l^m,
// Condon-Shortley phase).  HOST.
void angular_host_tables(int l_max, int n_theta, const double* cos_theta, const double* w_theta, int n_phi,
                         std::vector<double>& Yw, std::vector<double>& tw)
{
    const int nhalf = (l_max + 1) * (l_max + 2) / 2;
    Yw.assign((size_t)n_theta * nhalf, 0.0);
    const double pi = 3.14159265358979323846264338327950288;
    for (int j = 0; j < n_theta; ++j) {
        const double x = cos_theta[j], s = std::sqrt(std::max(0.0, (1.0 - x) * (1.0 + x)));
        double* y = Yw.data() + (size_t)j * nhalf;
        auto at = [&](int l, int m) -> double& { return y[l * (l + 1) / 2 + m]; };
        double pmm = std::sqrt(1.0 / (4.0 * pi));
        for (int m = 0; m <= l_max; ++m) {
            if (m > 0) pmm *= -std::sqrt((2.0 * m + 1.0) / (2.0 * m)) * s;
            at(m, m) = pmm;
            if (m + 1 <= l_max) at(m + 1, m) = std::sqrt(2.0 * m + 3.0) * x * pmm;
            for (int l = m + 2; l <= l_max; ++l) {
                const double a = std::sqrt((4.0 * l * l - 1.0) / ((double)l * l - (double)m * m));
                const double b = std::sqrt((((double)l - 1.0) * (l - 1.0) - (double)m * m) / (4.0 * (l - 1.0) * (l - 1.0) - 1.0));
                at(l, m) = a * (x * at(l - 1, m) - b * at(l - 2, m));
            }
        }
        for (int p = 0; p < nhalf; ++p) y[p] *= w_theta[j];
    }
    tw.assign((size_t)n_phi * 2, 0.0);
    for (int k = 0; k < n_phi; ++k) {
        const double a = 2.0 * pi * (double)k / (double)n_phi;
        tw[2 * k] = std::cos(a);
        tw[2 * k + 1] = -std::sin(a);
    }
}

cudaError_t angular_init_device()
{
    return cudaFuncSetAttribute(phi_dft_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024);
}

int angular_rows_per_cta(int n_phi) { return std::max(1, std::min(8, 2048 / std::max(1, n_phi))); }

cudaError_t launch_phi_dft(const double* f, const double* tw, long long n_rows, int n_phi, int l_max, double* F, double* rowsum2,
                           cudaStream_t st)
{
    if (n_rows <= 0) return cudaSuccess;
    const int rpc = angular_rows_per_cta(n_phi);
    const size_t smem = ((size_t)rpc * n_phi + n_phi) * sizeof(double2);
    const unsigned blocks = (unsigned)((n_rows + rpc - 1) / rpc);
    phi_dft_kernel<<<blocks, kThreads, smem, st>>>(reinterpret_cast<const double2*>(f), reinterpret_cast<const double2*>(tw), n_rows,
                                                   n_phi, l_max, rpc, reinterpret_cast<double2*>(F), rowsum2);
    return cudaGetLastError();
}

cudaError_t launch_legendre(const double* F, const double* rowsum2, const double* Yw, const double* w_theta, long long n_sr,
                            int n_theta, int l_max, double* R, double* f2, cudaStream_t st)
{
    if (n_sr <= 0) return cudaSuccess;
    legendre_kernel<<<(unsigned)n_sr, kThreads, 0, st>>>(reinterpret_cast<const double2*>(F), rowsum2, Yw, w_theta, n_theta, l_max,
                                                        reinterpret_cast<double2*>(R), f2);
    return cudaGetLastError();
}

}  // namespace scarf

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
// Step 1 is a dense contraction and runs on the FP64 tensor cores (angular_fused_kernel, mma.sync.m8n8k4.f64): with
//   C_m = sum_k f_k cos(m phi_k),  S_m = sum_k f_k sin(m phi_k)   (m = 0..l_max; real tables, complex f)
// F_{+m} = C_m - i S_m and F_{-m} = C_m + i S_m, so the real GEMM [rows x n_phi] . [n_phi x 2(l_max+1)] is done once for
// the real parts and once for the imaginary parts of the SAME loaded f (half the flops of the 2 l_max + 1 complex DFT
// columns).  One CTA owns one (state, r): its n_theta rows of F stay in shared memory and step 2 (the Legendre
// contraction) and the |f|^2 sums finish in the same kernel, so f is read once (201 MB on config 5) and nothing but
// R and <f^2> is written.  Tables (Ybar: host, fully normalised three-term recurrence; cos/sin in B-fragment order) are
// cached in the context.  phi_dft_kernel + legendre_kernel (SIMT) remain as the route for shapes whose F does not fit
// in shared memory.
#include <cmath>
#include <vector>

#include "ff_common.cuh"   // mbarrier / cp.async.bulk wrappers
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

// ---- fused tensor-core kernel -------------------------------------------------------------------------------------------
// DMMA m8n8k4 fragments: A[row = gid][k = tig] (one double per lane), B[k = tig][col = gid], D[row = gid][col = 2 tig + i].
// Rows = theta nodes of this (state, r); k = phi index; columns 2m (cos) and 2m+1 (sin), m = 4 nt + tig for n-tile nt.
constexpr int kFusedWarps = 4;
constexpr int kFusedMT = 2;            // 8-row tiles per warp and sweep (they share every B fragment)
constexpr int kYJ = 8;                 // theta nodes per staged chunk of the weight table (Legendre step)
constexpr int kFusedKG = 4;            // k-steps per software-pipeline group (loads of the next group overlap this group's DMMAs)
constexpr int kFusedNT = 7;            // n-tiles per pass: m = 0..27 in one pass (l_max <= 27); more passes beyond

__device__ __forceinline__ void dmma884(double (&d)[2], double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d[0]), "+d"(d[1]) : "d"(a), "d"(b));
}

// Bf: [n_nt][n_ks][32] doubles (fragment order), scale 2 pi / n_phi folded in.  F_glob != nullptr: write F and rowsum2 to
// global memory and stop (unfused route for large shapes); else finish R and f2 here.
__global__ void __launch_bounds__(kFusedWarps * 32) angular_fused_kernel(const double2* __restrict__ f, const double* __restrict__ Bf,
                                                                        const double* __restrict__ YwT, const double* __restrict__ w_theta,
                                                                        int n_theta, int n_phi, int l_max, int n_nt, int n_ks,
                                                                        double2* __restrict__ R, double* __restrict__ f2,
                                                                        double2* __restrict__ F_glob, double* __restrict__ row2_glob,
                                                                        const double* __restrict__ YwC, int ycb)
{
    __shared__ __align__(8) uint64_t ybar[2];
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const long long sr = blockIdx.x;
    const int n_m = 2 * l_max + 1;
    double* s_B = reinterpret_cast<double*>(smem_raw);                               // n_nt * n_ks * 32
    double2* s_F = reinterpret_cast<double2*>(s_B + (size_t)n_nt * n_ks * 32);       // n_theta * n_m      (fused route only)
    double* s_row2 = reinterpret_cast<double*>(s_F + (F_glob ? 0 : (size_t)n_theta * n_m));   // n_theta
    {   // cos/sin fragments -> shared memory: 16-byte loads, 8 in flight per thread (the table is a multiple of 32 doubles)
        const double2* src = reinterpret_cast<const double2*>(Bf);
        double2* dstB = reinterpret_cast<double2*>(s_B);
        const int n2 = n_nt * n_ks * 16;
#pragma unroll 8
        for (int i = threadIdx.x; i < n2; i += kFusedWarps * 32) dstB[i] = __ldg(src + i);
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, gid = lane >> 2, tig = lane & 3;
    const double2* fr = f + (size_t)sr * n_theta * n_phi;
    const double scale = 6.283185307179586476925286766559 / (double)n_phi;
    for (int row0 = warp * 8 * kFusedMT; row0 < n_theta; row0 += kFusedWarps * 8 * kFusedMT) {
        int row[kFusedMT];
        bool ok[kFusedMT];
#pragma unroll
        for (int t = 0; t < kFusedMT; ++t) { row[t] = row0 + 8 * t + gid; ok[t] = row[t] < n_theta; }
        double sq[kFusedMT];
#pragma unroll
        for (int t = 0; t < kFusedMT; ++t) sq[t] = 0.0;
        for (int nt0 = 0; nt0 < n_nt; nt0 += kFusedNT) {
            double aR[kFusedMT][kFusedNT][2], aI[kFusedMT][kFusedNT][2];
#pragma unroll
            for (int t = 0; t < kFusedMT; ++t)
#pragma unroll
                for (int n = 0; n < kFusedNT; ++n) aR[t][n][0] = aR[t][n][1] = aI[t][n][0] = aI[t][n][1] = 0.0;
            // k loop in groups of kFusedKG steps, software-pipelined: the global loads of group g + 1 are in flight while the
            // 4 kFusedNT kFusedKG DMMAs of group g run (f comes straight from HBM: ~1 us of latency to cover per load)
            auto load_group = [&](int ks0, double2 (&a)[kFusedKG][kFusedMT]) {
#pragma unroll
                for (int u = 0; u < kFusedKG; ++u) {
                    const int k = 4 * (ks0 + u) + tig;
#pragma unroll
                    for (int t = 0; t < kFusedMT; ++t)
                        a[u][t] = (ok[t] && k < n_phi) ? __ldg(fr + (size_t)row[t] * n_phi + k) : make_double2(0.0, 0.0);
                }
            };
            double2 cur[kFusedKG][kFusedMT], nxt[kFusedKG][kFusedMT];
            load_group(0, cur);
#pragma unroll 1
            for (int ks0 = 0; ks0 < n_ks; ks0 += kFusedKG) {
                if (ks0 + kFusedKG < n_ks) load_group(ks0 + kFusedKG, nxt);
#pragma unroll
                for (int u = 0; u < kFusedKG; ++u) {
                    const int ks = ks0 + u;
                    if (ks < n_ks) {
#pragma unroll
                        for (int t = 0; t < kFusedMT; ++t)
                            if (nt0 == 0) sq[t] = fma(cur[u][t].x, cur[u][t].x, fma(cur[u][t].y, cur[u][t].y, sq[t]));
#pragma unroll
                        for (int n = 0; n < kFusedNT; ++n)
                            if (nt0 + n < n_nt) {
                                const double b = s_B[((size_t)(nt0 + n) * n_ks + ks) * 32 + lane];
#pragma unroll
                                for (int t = 0; t < kFusedMT; ++t) {
                                    dmma884(aR[t][n], cur[u][t].x, b);
                                    dmma884(aI[t][n], cur[u][t].y, b);
                                }
                            }
                    }
                }
#pragma unroll
                for (int u = 0; u < kFusedKG; ++u)
#pragma unroll
                    for (int t = 0; t < kFusedMT; ++t) cur[u][t] = nxt[u][t];
            }
            // lane (gid, tig) holds, for row gid and m = 4 (nt0 + n) + tig:  C_re, S_re (aR), C_im, S_im (aI)
#pragma unroll
            for (int t = 0; t < kFusedMT; ++t)
#pragma unroll
                for (int n = 0; n < kFusedNT; ++n) {
                    const int m = 4 * (nt0 + n) + tig;
                    if (ok[t] && nt0 + n < n_nt && m <= l_max) {
                        const double2 Fp = make_double2(aR[t][n][0] + aI[t][n][1], aI[t][n][0] - aR[t][n][1]);   // C - i S
                        const double2 Fn = make_double2(aR[t][n][0] - aI[t][n][1], aI[t][n][0] + aR[t][n][1]);   // C + i S
                        double2* dstF = F_glob ? F_glob + ((size_t)sr * n_theta + row[t]) * n_m : s_F + (size_t)row[t] * n_m;
                        dstF[l_max + m] = Fp;
                        dstF[l_max - m] = Fn;
                    }
                }
        }
#pragma unroll
        for (int t = 0; t < kFusedMT; ++t) {
            double x = sq[t];
            x += __shfl_xor_sync(0xffffffffu, x, 1);
            x += __shfl_xor_sync(0xffffffffu, x, 2);
            if (tig == 0 && ok[t]) {
                if (F_glob) row2_glob[(size_t)sr * n_theta + row[t]] = x * scale;
                else s_row2[row[t]] = x * scale;
            }
        }
    }
    if (F_glob) return;
    __syncthreads();
    // step 2: R[l(l+1) +- m] = (-1)^{m for -m} sum_j Yw[j][l(l+1)/2 + m] F[j][+-m + l_max].  One work item = (m >= 0, group g):
    // the thread reads F[j][+-m] ONCE per j from shared memory and uses it for its up to kLG degrees l = m + g + k G (the
    // per-(l, m) mapping read it once per l: the shared-memory wavefronts of step 2 cost as much as the tensor-core step);
    // YwT is the transposed weight table [l(l+1)/2 + m][n_theta_pad], streamed with 16-byte loads (kLG independent loads in flight).
    constexpr int kLG = 8;
    const int nlm = (l_max + 1) * (l_max + 1), ntp = (n_theta + 1) & ~1, G = (l_max + kLG) / kLG;
    if (ycb > 0) {
        // Staged route: the weight table arrives in chunks of kYJ theta nodes, YwC[chunk][(l,m)][kYJ + 1] (one pad double per
        // row: the rows of a warp's lanes then fall on distinct banks), by cp.async.bulk into the two halves of the fragment
        // area, which step 1 no longer needs — the loads of chunk c + 1 run while chunk c is being used, instead of every
        // thread waiting on L2 for the weights of each theta pair.  One item per thread ((l_max + 1) G <= blockDim).
        unsigned char* ybuf = smem_raw;
        const int n_chunks = (n_theta + kYJ - 1) / kYJ;
        if (threadIdx.x == 0) {
            mbar_init(&ybar[0], 1);
            mbar_init(&ybar[1], 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            for (int c = 0; c < min(2, n_chunks); ++c) {
                mbar_expect_tx(&ybar[c], (uint32_t)ycb);
                bulk_g2s(ybuf + (size_t)c * ycb, reinterpret_cast<const unsigned char*>(YwC) + (size_t)c * ycb, (uint32_t)ycb, &ybar[c]);
            }
        }
        __syncthreads();
        const int item = threadIdx.x;
        const bool active = item < (l_max + 1) * G;
        const int m = active ? item / G : 0, g = active ? item % G : 0;
        int row[kLG], nk = 0;
#pragma unroll
        for (int k = 0; k < kLG; ++k) {
            const int l = m + g + k * G;
            row[k] = (l <= l_max ? l * (l + 1) / 2 + m : 0) * (kYJ + 1);
            if (active && l <= l_max) nk = k + 1;
        }
        double pr[kLG], pi[kLG], nr[kLG], ni[kLG];
#pragma unroll
        for (int k = 0; k < kLG; ++k) pr[k] = pi[k] = nr[k] = ni[k] = 0.0;
        for (int c = 0; c < n_chunks; ++c) {
            mbar_wait(&ybar[c & 1], (uint32_t)((c >> 1) & 1));
            const double* yb = reinterpret_cast<const double*>(ybuf + (size_t)(c & 1) * ycb);
#pragma unroll
            for (int jj = 0; jj < kYJ; ++jj) {
                const int j = c * kYJ + jj;
                if (j < n_theta) {
                    const double2 p0 = s_F[(size_t)j * n_m + (l_max + m)], q0 = s_F[(size_t)j * n_m + (l_max - m)];
#pragma unroll
                    for (int k = 0; k < kLG; ++k)
                        if (k < nk) {
                            const double y = yb[row[k] + jj];
                            pr[k] = fma(y, p0.x, pr[k]); pi[k] = fma(y, p0.y, pi[k]);
                            nr[k] = fma(y, q0.x, nr[k]); ni[k] = fma(y, q0.y, ni[k]);
                        }
                }
            }
            __syncthreads();                              // everybody has left this half: refill it with chunk c + 2
            if (threadIdx.x == 0 && c + 2 < n_chunks) {
                mbar_expect_tx(&ybar[c & 1], (uint32_t)ycb);
                bulk_g2s(ybuf + (size_t)(c & 1) * ycb, reinterpret_cast<const unsigned char*>(YwC) + (size_t)(c + 2) * ycb, (uint32_t)ycb,
                         &ybar[c & 1]);
            }
        }
        const double sgn = (m & 1) ? -1.0 : 1.0;
#pragma unroll
        for (int k = 0; k < kLG; ++k) {
            const int l = m + g + k * G;
            if (k < nk) {
                R[(size_t)sr * nlm + l * (l + 1) + m] = make_double2(pr[k], pi[k]);
                if (m > 0) R[(size_t)sr * nlm + l * (l + 1) - m] = make_double2(sgn * nr[k], sgn * ni[k]);
            }
        }
    } else
    for (int item = threadIdx.x; item < (l_max + 1) * G; item += blockDim.x) {
        const int m = item / G, g = item % G;
        const double2* yrow[kLG];
        int nk = 0;
#pragma unroll
        for (int k = 0; k < kLG; ++k) {
            const int l = m + g + k * G;
            yrow[k] = reinterpret_cast<const double2*>(YwT + (size_t)(l <= l_max ? l * (l + 1) / 2 + m : 0) * ntp);
            if (l <= l_max) nk = k + 1;
        }
        double pr[kLG], pi[kLG], nr[kLG], ni[kLG];
#pragma unroll
        for (int k = 0; k < kLG; ++k) pr[k] = pi[k] = nr[k] = ni[k] = 0.0;
        for (int j2 = 0; j2 < ntp / 2; ++j2) {
            const int j = 2 * j2;
            double2 y[kLG];
#pragma unroll
            for (int k = 0; k < kLG; ++k) y[k] = k < nk ? __ldg(yrow[k] + j2) : make_double2(0.0, 0.0);
            const double2 p0 = s_F[(size_t)j * n_m + (l_max + m)], q0 = s_F[(size_t)j * n_m + (l_max - m)];
            const bool two = j + 1 < n_theta;
            const double2 p1 = two ? s_F[(size_t)(j + 1) * n_m + (l_max + m)] : make_double2(0.0, 0.0);
            const double2 q1 = two ? s_F[(size_t)(j + 1) * n_m + (l_max - m)] : make_double2(0.0, 0.0);
#pragma unroll
            for (int k = 0; k < kLG; ++k) {
                pr[k] = fma(y[k].x, p0.x, pr[k]); pi[k] = fma(y[k].x, p0.y, pi[k]);
                nr[k] = fma(y[k].x, q0.x, nr[k]); ni[k] = fma(y[k].x, q0.y, ni[k]);
                pr[k] = fma(y[k].y, p1.x, pr[k]); pi[k] = fma(y[k].y, p1.y, pi[k]);
                nr[k] = fma(y[k].y, q1.x, nr[k]); ni[k] = fma(y[k].y, q1.y, ni[k]);
            }
        }
        const double sgn = (m & 1) ? -1.0 : 1.0;
#pragma unroll
        for (int k = 0; k < kLG; ++k) {
            const int l = m + g + k * G;
            if (k < nk) {
                R[(size_t)sr * nlm + l * (l + 1) + m] = make_double2(pr[k], pi[k]);
                if (m > 0) R[(size_t)sr * nlm + l * (l + 1) - m] = make_double2(sgn * nr[k], sgn * ni[k]);
            }
        }
    }
    if (f2 != nullptr && threadIdx.x == 0) {
        double acc = 0.0;
        for (int j = 0; j < n_theta; ++j) acc = fma(w_theta[j], s_row2[j], acc);
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
    cudaError_t e = cudaFuncSetAttribute(phi_dft_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(angular_fused_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kAngularMaxSmem);
    return e;
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

// B-fragment table of the fused kernel: Bf[nt][ks][lane], lane = (gid, tig) <-> B[k = 4 ks + tig][col = 8 nt + gid],
// col = 2 m + {0: cos, 1: sin}(m phi_k) * 2 pi / n_phi, phi_k = 2 pi k / n_phi; zero beyond n_phi or l_max.  The angle is
// reduced exactly on integers (m k mod n_phi) before the call to cos/sin.  HOST.
void angular_fragment_table(int l_max, int n_phi, std::vector<double>& Bf, int& n_nt, int& n_ks)
{
    n_nt = (2 * (l_max + 1) + 7) / 8;
    n_ks = (n_phi + 3) / 4;
    Bf.assign((size_t)n_nt * n_ks * 32, 0.0);
    const double pi = 3.14159265358979323846264338327950288;
    const double scale = 2.0 * pi / (double)n_phi;
    for (int nt = 0; nt < n_nt; ++nt)
        for (int ks = 0; ks < n_ks; ++ks)
            for (int lane = 0; lane < 32; ++lane) {
                const int gid = lane >> 2, tig = lane & 3, k = 4 * ks + tig, col = 8 * nt + gid, m = col / 2;
                if (k >= n_phi || m > l_max) continue;
                const long long idx = ((long long)m * k) % n_phi;
                const double a = 2.0 * pi * (double)idx / (double)n_phi;
                Bf[((size_t)nt * n_ks + ks) * 32 + lane] = scale * ((col & 1) ? std::sin(a) : std::cos(a));
            }
}

// YwT[l(l+1)/2 + m][n_theta_pad]: the transpose of Yw, rows padded with zeros to an even length (16-byte row loads).  HOST.
void angular_transpose_table(int l_max, int n_theta, const std::vector<double>& Yw, std::vector<double>& YwT)
{
    const int nhalf = (l_max + 1) * (l_max + 2) / 2, ntp = (n_theta + 1) & ~1;
    YwT.assign((size_t)nhalf * ntp, 0.0);
    for (int j = 0; j < n_theta; ++j)
        for (int p = 0; p < nhalf; ++p) YwT[(size_t)p * ntp + j] = Yw[(size_t)j * nhalf + p];
}

// Chunked weight table of the staged Legendre step: YwC[c][l(l+1)/2 + m][kYJ + 1], theta nodes c kYJ .. c kYJ + kYJ - 1 (zeros past
// n_theta and in the pad column), every chunk padded to a multiple of 16 bytes.  Returns the chunk size in bytes.  HOST.
int angular_chunk_table(int l_max, int n_theta, const std::vector<double>& Yw, std::vector<double>& YwC)
{
    const int nhalf = (l_max + 1) * (l_max + 2) / 2, nc = (n_theta + kYJ - 1) / kYJ;
    const int chunk_doubles = (nhalf * (kYJ + 1) + 1) & ~1;
    YwC.assign((size_t)nc * chunk_doubles, 0.0);
    for (int j = 0; j < n_theta; ++j)
        for (int p = 0; p < nhalf; ++p) YwC[(size_t)(j / kYJ) * chunk_doubles + (size_t)p * (kYJ + 1) + (j % kYJ)] = Yw[(size_t)j * nhalf + p];
    return chunk_doubles * 8;
}

size_t angular_fused_smem(int n_theta, int l_max, int n_nt, int n_ks, bool fused)
{
    return (size_t)n_nt * n_ks * 32 * 8 + (fused ? (size_t)n_theta * (2 * l_max + 1) * 16 : 0) + (size_t)n_theta * 8;
}

cudaError_t launch_angular_fused(const double* f, const double* Bf, const double* YwT, const double* w_theta, long long n_sr, int n_theta,
                                 int n_phi, int l_max, int n_nt, int n_ks, double* R, double* f2, double* F_glob, double* row2_glob,
                                 const double* YwC, int chunk_bytes, cudaStream_t st)
{
    if (n_sr <= 0) return cudaSuccess;
    const size_t smem = angular_fused_smem(n_theta, l_max, n_nt, n_ks, F_glob == nullptr);
    // the staged Legendre step needs two chunks inside the fragment area and one work item per thread
    const bool staged = F_glob == nullptr && YwC != nullptr && 2 * (size_t)chunk_bytes <= (size_t)n_nt * n_ks * 32 * 8 &&
                        (l_max + 1) * ((l_max + 8) / 8) <= kFusedWarps * 32;
    angular_fused_kernel<<<(unsigned)n_sr, kFusedWarps * 32, smem, st>>>(reinterpret_cast<const double2*>(f), Bf, YwT, w_theta, n_theta, n_phi,
                                                                        l_max, n_nt, n_ks, reinterpret_cast<double2*>(R), f2,
                                                                        reinterpret_cast<double2*>(F_glob), row2_glob, YwC, staged ? chunk_bytes : 0);
    return cudaGetLastError();
}

// S5 (optional output of SURVEY.md §8(a)): |f|^2 of a complex array, what Fig. 6 of the paper plots.
__global__ void __launch_bounds__(256) abs2_kernel(const double2* __restrict__ f, long long n, double* __restrict__ out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double2 v = f[i];
    out[i] = fma(v.x, v.x, v.y * v.y);
}

cudaError_t launch_abs2(const double* f_complex, long long n, double* out, cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    abs2_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(reinterpret_cast<const double2*>(f_complex), n, out);
    return cudaGetLastError();
}

}  // namespace scarf

// ff_highl.cu — S4 for the pair classes L = 7..12, i.e. pairs that involve g, h or i shells ("up to i orbitals",
// PAPER.md:134).  Same formula as the unrolled kernels (Eq. (48)),
//
//   f_s(q) += sum_{pairs of class >= 7} e^{-q^2/4p} (cos q.P + i sin q.P) (A_s(q) + i B_s(q)),
//
// for records of 120..455 Hermite coefficients per state (up to 43 KB per record at 12 states: they neither fit a shared-
// memory stage of the unrolled kernels nor a thread's registers as monomials).  One thread owns one q-point; per state and
// record it walks the degree shells n = 0..L with the powers q_x^t, q_y^u, q_z^v held in registers (compile-time indices:
// one straight-line body for all 455 monomials, left at the shell boundary n > L), reading each coefficient with a
// warp-uniform load straight from the L2-resident stream.  2 DMUL + 1 DFMA per term: a third of the FP64 pipe at best,
// on classes that the paper's own workloads (cc-pVDZ, l <= 2) and BASELINE.json's configs never populate.
//
// The kernel runs AFTER the unrolled kernel of the same tile and ADDS to `out` (same stream: ordered).  Point sets: an
// arbitrary list, or the (half of the) product grid of scarf_form_factors_grid — there it also adds the conjugate to the
// mirror point when the grid is inversion-symmetric.
#include "ff_common.cuh"

namespace scarf {

namespace {

constexpr int kThreads = 128;
constexpr int kPowMax = kMaxClass;     // 12

// one degree shell n of one record for one state: A += sum_{h in shell, n even} D_h m_h,  B likewise for odd n
template <int N>
__device__ __forceinline__ void shell_accum(const double* __restrict__ D, const double (&px)[kPowMax + 1], const double (&py)[kPowMax + 1],
                                            const double (&pz)[kPowMax + 1], double& A, double& B)
{
    double acc[4] = {0.0, 0.0, 0.0, 0.0};                          // four independent chains (DFMA latency)
    static_for<N + 1>([&](auto tc) {
        constexpr int t = N - decltype(tc)::value;                 // t descending
        static_for<N - t + 1>([&](auto uc) {
            constexpr int u = (N - t) - decltype(uc)::value;       // u descending
            constexpr int v = N - t - u, h = hindex(t, u, v);      // Hermite index of (t, u, v): kernels.cuh enumeration
            const double m = (px[t] * py[u]) * pz[v];
            acc[h & 3] = fma(D[h], m, acc[h & 3]);
        });
    });
    const double sum = (acc[0] + acc[1]) + (acc[2] + acc[3]);
    if constexpr (N & 1) B += sum;
    else A += sum;
}

__global__ void __launch_bounds__(kThreads) ff_highl_kernel(const HighLArgs a)
{
    const StreamDesc& d = *a.desc;
    long long n_high = 0;
    for (int c = kFastMaxClass + 1; c < kNClasses; ++c) n_high += d.cls_n[c];
    if (n_high == 0) return;                                        // nothing survived the screening in these classes
    const long long p = (long long)blockIdx.x * kThreads + threadIdx.x;
    if (p >= a.n_points) return;
    double q[3];
    long long i_out, i_mirror = -1;
    if (a.q != nullptr) {
        q[0] = a.q[3 * p]; q[1] = a.q[3 * p + 1]; q[2] = a.q[3 * p + 2];
        i_out = p;
    } else {
        const int iz = (int)(p % a.nz), iy = (int)((p / a.nz) % a.ny), ix = (int)(p / ((long long)a.nz * a.ny));   // ix < nx_eval
        q[0] = a.qx[ix]; q[1] = a.qy[iy]; q[2] = a.qz[iz];
        i_out = ((long long)ix * a.ny + iy) * a.nz + iz;
        if (a.sym && 2 * ix < a.nx - 1) i_mirror = a.n_q - 1 - i_out;
    }
    double px[kPowMax + 1], py[kPowMax + 1], pz[kPowMax + 1];
    px[0] = py[0] = pz[0] = 1.0;
#pragma unroll
    for (int k = 1; k <= kPowMax; ++k) { px[k] = px[k - 1] * q[0]; py[k] = py[k - 1] * q[1]; pz[k] = pz[k - 1] * q[2]; }
    const double q2 = q[0] * q[0] + q[1] * q[1] + q[2] * q[2];
    double2* out = reinterpret_cast<double2*>(a.dst);
#pragma unroll 1
    for (int s = 0; s < a.ns_real; ++s) {
        double re = 0.0, im = 0.0;
#pragma unroll 1
        for (int c = kFastMaxClass + 1; c < kNClasses; ++c) {
            const long long n_rec = d.cls_n[c];
            const int nh = nherm(c);
            const char* seg = a.base + d.cls_off[c];
#pragma unroll 1
            for (long long r = 0; r < n_rec; ++r) {
                const double* rec = reinterpret_cast<const double*>(seg + (size_t)r * d.rec_bytes[c]);
                const double ph = fma(q[0], rec[0], fma(q[1], rec[1], q[2] * rec[2]));
                const double e = exp_neg(q2 * rec[3]);
                double sn, cs;
                sincos_fast(ph, sn, cs);
                const double* D = rec + 4 + (size_t)s * nh;
                double A = 0.0, B = 0.0;
                // classes are prefixes of each other: shells 0..7 always, the rest up to this record's class
                shell_accum<0>(D, px, py, pz, A, B); shell_accum<1>(D, px, py, pz, A, B); shell_accum<2>(D, px, py, pz, A, B);
                shell_accum<3>(D, px, py, pz, A, B); shell_accum<4>(D, px, py, pz, A, B); shell_accum<5>(D, px, py, pz, A, B);
                shell_accum<6>(D, px, py, pz, A, B); shell_accum<7>(D, px, py, pz, A, B);
                if (c >= 8) shell_accum<8>(D, px, py, pz, A, B);
                if (c >= 9) shell_accum<9>(D, px, py, pz, A, B);
                if (c >= 10) shell_accum<10>(D, px, py, pz, A, B);
                if (c >= 11) shell_accum<11>(D, px, py, pz, A, B);
                if (c >= 12) shell_accum<12>(D, px, py, pz, A, B);
                const double gc = e * cs, gs = e * sn;
                re = fma(gc, A, fma(-gs, B, re));
                im = fma(gs, A, fma(gc, B, im));
            }
        }
        double2* o = out + (size_t)s * a.n_q;
        double2 v = o[i_out];
        v.x += re; v.y += im;
        o[i_out] = v;
        if (i_mirror >= 0) {
            double2 w = o[i_mirror];
            w.x += re; w.y -= im;
            o[i_mirror] = w;
        }
    }
}

}  // namespace

cudaError_t launch_ff_highl(const HighLArgs& a, cudaStream_t st)
{
    if (a.n_points <= 0 || a.ns_real <= 0) return cudaSuccess;
    ff_highl_kernel<<<(unsigned)((a.n_points + kThreads - 1) / kThreads), kThreads, 0, st>>>(a);
    return cudaGetLastError();
}

}  // namespace scarf

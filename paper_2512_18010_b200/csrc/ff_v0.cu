// ff_v0.cu — S4, baseline form: one thread per q-point, records read from global memory (warp-uniform
// addresses, served by L1/L2 broadcast), libdevice exp/sincos.  Kept as the simple, obviously-correct device
// path that the tuned kernel (ff_v1.cu) is compared with on the GPU, and as the fallback for state-tile
// sizes / classes the tuned kernel is not instantiated for.
//
//   f_s(q) += e^{-q^2/4p} (cos q.P + i sin q.P) (A_s + i B_s),   A_s = sum_{n even} D^s_h q^h,  B_s = sum_{n odd} D^s_h q^h
// (Eq. (48) PAPER.md:326 with i^n folded into D, see kernels.cuh).
#include "kernels.cuh"

namespace scarf {

template <int L, int NS>
__global__ void __launch_bounds__(128) ff_v0_kernel(const char* __restrict__ recs, long long n_pairs,
                                                    const double* __restrict__ q, long long n_q,
                                                    double* __restrict__ out, int s0, int ns_real, int accumulate)
{
    constexpr int NH = nherm(L);
    constexpr int REC = rec_doubles(L, NS);
    const long long iq = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (iq >= n_q) return;
    const double qx = q[3 * iq], qy = q[3 * iq + 1], qz = q[3 * iq + 2];
    const double q2 = qx * qx + qy * qy + qz * qz;
    double px[L + 1], py[L + 1], pz[L + 1];
    px[0] = py[0] = pz[0] = 1.0;
#pragma unroll
    for (int k = 1; k <= L; ++k) { px[k] = px[k - 1] * qx; py[k] = py[k - 1] * qy; pz[k] = pz[k - 1] * qz; }
    double mono[NH];
    {
        int h = 0;
#pragma unroll
        for (int n = 0; n <= L; ++n)
#pragma unroll
            for (int t = n; t >= 0; --t)
#pragma unroll
                for (int u = n - t; u >= 0; --u) { mono[h] = px[t] * py[u] * pz[n - t - u]; ++h; }
    }
    double re[NS], im[NS];
#pragma unroll
    for (int s = 0; s < NS; ++s) re[s] = im[s] = 0.0;

    const double* rec = reinterpret_cast<const double*>(recs);
    for (long long ip = 0; ip < n_pairs; ++ip, rec += REC) {
        const double Px = __ldg(rec), Py = __ldg(rec + 1), Pz = __ldg(rec + 2), inv4p = __ldg(rec + 3);
        const double ph = qx * Px + qy * Py + qz * Pz;
        const double e = exp(-q2 * inv4p);
        double sn, cs;
        sincos(ph, &sn, &cs);
        const double gc = e * cs, gs = e * sn;
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            const double* D = rec + 4 + s * NH;
            double A = __ldg(D), B = 0.0;
            int h = 1;
#pragma unroll
            for (int n = 1; n <= L; ++n)
#pragma unroll
                for (int t = n; t >= 0; --t)
#pragma unroll
                    for (int u = n - t; u >= 0; --u) {
                        if (n & 1) B = fma(__ldg(D + h), mono[h], B);
                        else A = fma(__ldg(D + h), mono[h], A);
                        ++h;
                    }
            re[s] = fma(gc, A, re[s]);
            im[s] = fma(gs, A, im[s]);
            if (L > 0) {
                re[s] = fma(-gs, B, re[s]);
                im[s] = fma(gc, B, im[s]);
            }
        }
    }
#pragma unroll
    for (int s = 0; s < NS; ++s)
        if (s < ns_real) {
            double2* o = reinterpret_cast<double2*>(out) + (size_t)(s0 + s) * n_q + iq;
            double2 v = make_double2(re[s], im[s]);
            if (accumulate) { const double2 old = *o; v.x += old.x; v.y += old.y; }
            *o = v;
        }
}

template <int L>
static cudaError_t launch_L(const TileStream& ts, const double* q, long long n_q, double* out, int accumulate, cudaStream_t st)
{
    const ClassStream& c = ts.cls[L];
    if (c.n <= 0 || n_q <= 0) return cudaSuccess;
    const int threads = 128;
    const unsigned blocks = (unsigned)((n_q + threads - 1) / threads);
    const char* recs = ts.base + c.off;
#define SCARF_V0_CASE(NSV)                                                                                   \
    case NSV:                                                                                                \
        ff_v0_kernel<L, NSV><<<blocks, threads, 0, st>>>(recs, c.n, q, n_q, out, ts.s0, ts.ns_real, accumulate); \
        break;
    switch (ts.NS) {
        SCARF_V0_CASE(1)
        SCARF_V0_CASE(2)
        SCARF_V0_CASE(4)
        SCARF_V0_CASE(6)
        SCARF_V0_CASE(8)
        SCARF_V0_CASE(12)
    default:
        return cudaErrorInvalidValue;
    }
#undef SCARF_V0_CASE
    return cudaGetLastError();
}

cudaError_t launch_ff_v0(int L, const TileStream& ts, const double* q, long long n_q, double* out, int accumulate, cudaStream_t st)
{
    switch (L) {
    case 0: return launch_L<0>(ts, q, n_q, out, accumulate, st);
    case 1: return launch_L<1>(ts, q, n_q, out, accumulate, st);
    case 2: return launch_L<2>(ts, q, n_q, out, accumulate, st);
    case 3: return launch_L<3>(ts, q, n_q, out, accumulate, st);
    case 4: return launch_L<4>(ts, q, n_q, out, accumulate, st);
    case 5: return launch_L<5>(ts, q, n_q, out, accumulate, st);
    case 6: return launch_L<6>(ts, q, n_q, out, accumulate, st);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace scarf

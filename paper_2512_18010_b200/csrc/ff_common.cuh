// ff_common.cuh — device building blocks shared by the form-factor kernels (ff_v1.cu: arbitrary q list; ff_grid.cu:
// Cartesian product grid): compile-time Hermite index tables, mbarrier / 1-D TMA bulk-copy wrappers, the
// per-record transcendental part and the per-record (state, Hermite index) accumulate loop of Eq. (48)
// PAPER.md:326-330.
#pragma once
#include <utility>

#include "ff_math.cuh"
#include "kernels.cuh"

namespace scarf {

constexpr int kNQ = 2;                       // q-points per thread

template <int I> using IC = std::integral_constant<int, I>;
template <class F, int... Is>
__device__ __forceinline__ void static_for_impl(F&& f, std::integer_sequence<int, Is...>) { (f(IC<Is>{}), ...); }
template <int N, class F>
__device__ __forceinline__ void static_for(F&& f) { static_for_impl(f, std::make_integer_sequence<int, N>{}); }

// total degree n = t+u+v of Hermite index h (enumeration: n ascending; see kernels.cuh)
__host__ __device__ constexpr int hdeg(int h)
{
    int n = 0;
    while (nherm(n) <= h) ++n;
    return n;
}
// exponents (t,u,v) of Hermite index h
__host__ __device__ constexpr int hexp(int h, int axis)
{
    const int n = hdeg(h);
    int idx = n == 0 ? 0 : nherm(n - 1);
    for (int t = n; t >= 0; --t)
        for (int u = n - t; u >= 0; --u) {
            if (idx == h) return axis == 0 ? t : (axis == 1 ? u : n - t - u);
            ++idx;
        }
    return 0;
}
// index of the monomial with one power of `axis` less (parent in the recurrence mono[h] = mono[parent] * q_axis)
__host__ __device__ constexpr int hindex(int t, int u, int v)
{
    const int n = t + u + v;
    int idx = n == 0 ? 0 : nherm(n - 1);
    for (int tt = n; tt >= 0; --tt)
        for (int uu = n - tt; uu >= 0; --uu) {
            if (tt == t && uu == u) return idx;
            ++idx;
        }
    return 0;
}

// ---- mbarrier / bulk-copy wrappers (PTX ISA: mbarrier, cp.async.bulk) -------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// ---- one record = transcendental part (record_trans) + the (state, h) loop (record_accum) -------------------
// The two are separate so that run_class can software-pipeline them: the exp/sincos chains of record k+1 (low
// ILP: two dependent Horner chains per q-point) are issued in the same basic block as the 4 NS n_herm independent
// accumulate FMAs of record k, which fill the FP64 pipe while the chains wait on their own results.
template <int NQA, int jq0>
__device__ __forceinline__ void record_trans(const double2* __restrict__ r2, const double (&qv)[kNQ][4],
                                             double (&gc)[NQA], double (&gs)[NQA])
{
    const double2 h0 = r2[0], h1 = r2[1];   // Px, Py | Pz, 1/(4p)
#pragma unroll
    for (int j = 0; j < NQA; ++j) {
        const double* qj = qv[jq0 + j];
        const double ph = fma(qj[0], h0.x, fma(qj[1], h0.y, qj[2] * h1.x));
        const double e = exp_neg(qj[3] * h1.y);
        double sn, cs;
        sincos_fast(ph, sn, cs);
        gc[j] = e * cs;
        gs[j] = e * sn;
    }
}

template <int L, int NS, int NQA, int jq0>
__device__ __forceinline__ void record_accum(const double2* __restrict__ r2, const double (&mono)[NQA][nherm(L)],
                                             const double (&gc)[NQA], const double (&gs)[NQA],
                                             double (&re)[kNQ][NS], double (&im)[kNQ][NS])
{
    constexpr int NH = nherm(L), N = NS * NH;
    const double2* __restrict__ D2 = r2 + 2;
    double A[NQA], B[NQA];
    static_for<(N + 1) / 2>([&](auto i2c) {
        constexpr int i2 = decltype(i2c)::value;
        const double2 c = D2[i2];
        static_for<2>([&](auto halfc) {
            constexpr int half = decltype(halfc)::value;
            constexpr int i = 2 * i2 + half;
            if constexpr (i < N) {
                constexpr int s = i / NH, h = i % NH, n = hdeg(h);
                const double cv = half ? c.y : c.x;
#pragma unroll
                for (int j = 0; j < NQA; ++j) {
                    if constexpr (h == 0) A[j] = cv;
                    else if constexpr (h == 1) B[j] = cv * mono[j][1];
                    else if constexpr (n & 1) B[j] = fma(cv, mono[j][h], B[j]);
                    else A[j] = fma(cv, mono[j][h], A[j]);
                }
                if constexpr (h == NH - 1) {
#pragma unroll
                    for (int j = 0; j < NQA; ++j) {
                        re[jq0 + j][s] = fma(gc[j], A[j], re[jq0 + j][s]);
                        im[jq0 + j][s] = fma(gs[j], A[j], im[jq0 + j][s]);
                        if constexpr (L > 0) {
                            re[jq0 + j][s] = fma(-gs[j], B[j], re[jq0 + j][s]);
                            im[jq0 + j][s] = fma(gc[j], B[j], im[jq0 + j][s]);
                        }
                    }
                }
            }
        });
    });
}

template <int L, int NQA, int jq0>
__device__ __forceinline__ void make_monomials(const double (&qv)[kNQ][4], double (&mono)[NQA][nherm(L)])
{
    constexpr int NH = nherm(L);
#pragma unroll
    for (int j = 0; j < NQA; ++j) {
        mono[j][0] = 1.0;
        static_for<NH - 1>([&](auto hc) {
            constexpr int h = decltype(hc)::value + 1;
            constexpr int t = hexp(h, 0), u = hexp(h, 1), v = hexp(h, 2);
            // peel one power off the first non-zero axis
            constexpr int ax = t > 0 ? 0 : (u > 0 ? 1 : 2);
            constexpr int parent = hindex(t - (ax == 0), u - (ax == 1), v - (ax == 2));
            mono[j][h] = parent == 0 ? qv[jq0 + j][ax] : mono[j][parent] * qv[jq0 + j][ax];
        });
    }
}

}  // namespace scarf

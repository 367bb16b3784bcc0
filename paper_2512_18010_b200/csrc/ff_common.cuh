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

// ---- optional device-side invariant checks (build with -DSCARF_DEBUG_CHECKS: python -m paper_2512_18010_b200.build --debug-checks).
// compute-sanitizer is not available on the measurement pool, so the hand-rolled pipelines carry their own bounds / protocol
// assertions; a violated one traps (the launch fails with cudaErrorLaunchFailure and every later call reports it).
#ifdef SCARF_DEBUG_CHECKS
#define SCARF_CHECK(cond)        \
    do {                         \
        if (!(cond)) __trap();   \
    } while (0)
#else
#define SCARF_CHECK(cond) ((void)0)
#endif

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

// ---- ordered fix-up tickets: the chunks of one q tile add into `out` in chunk order --------------------------------------
// ticket[tile] holds the chunk whose turn it is (0 at launch; the last chunk puts 0 back).  Whole-CTA calls.
__device__ __forceinline__ void ticket_wait(int* ticket, int turn)
{
    if (threadIdx.x == 0) {
        int v;
        do {
            asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(ticket) : "memory");
            SCARF_CHECK(v >= 0 && v <= turn);             // tickets only move forward, one chunk at a time
        } while (v != turn);
    }
    __syncthreads();
}
__device__ __forceinline__ void ticket_pass(int* ticket, int next)
{
    __threadfence();                                      // this thread's stores to `out` are visible device-wide ...
    __syncthreads();                                      // ... for every thread of the CTA, before the ticket moves on
    if (threadIdx.x == 0) asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(ticket), "r"(next) : "memory");
}

// ---- which (tile, chunk) a CTA of the (n_tiles, n_chunks) grid works on (V1Args::tile_group; CTAs are dispatched x fastest) ----
__device__ __forceinline__ void cta_tile_chunk(const V1Args& v, int& tile, int& chunk)
{
    if (v.tile_group <= 0) {
        tile = (int)blockIdx.x;
        chunk = (int)blockIdx.y;
        return;
    }
    const long long lin = (long long)blockIdx.x + (long long)gridDim.x * (long long)blockIdx.y;
    const long long per = (long long)v.tile_group * v.n_chunks;
    const int g = (int)(lin / per), rem = (int)(lin - (long long)g * per);
    const int gs = min(v.tile_group, v.n_tiles - g * v.tile_group);       // the last group may be short
    chunk = rem / gs;
    tile = g * v.tile_group + rem % gs;
    SCARF_CHECK(tile >= 0 && tile < v.n_tiles && chunk >= 0 && chunk < v.n_chunks);
}

// ---- q-adaptive cut-off helpers (fold.cu: qcut_kernel) -------------------------------------------------------------------
// smallest value of x over the CTA's threads (whole-CTA call; `sh` holds one double per warp)
__device__ __forceinline__ double block_min(double x, double* sh)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x = fmin(x, __shfl_xor_sync(0xffffffffu, x, o));
    __syncthreads();
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = x;
    __syncthreads();
    double m = sh[0];
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) m = fmin(m, sh[w]);
    return m;
}
// number of leading entries of the DESCENDING array qc[0..n) that exceed q: the records a tile with smallest |q| = q keeps
__device__ __forceinline__ int active_prefix(const double* __restrict__ qc, long long n, double q)
{
    long long lo = 0, hi = n;                             // invariant: qc[i] > q for i < lo, qc[i] <= q for i >= hi
    while (lo < hi) {
        const long long mid = (lo + hi) >> 1;
        if (qc[mid] > q) lo = mid + 1; else hi = mid;
    }
    return (int)lo;
}

// ---- what a CTA of an S4 kernel has to do (all S4 kernels: grid = q tiles x stream chunks) -------------------------------------
// Per class: the records of the CTA's chunk that its tile keeps, where they start in the stream and which table row they have —
// worked out once by threads 0..6 and parked in shared memory, so that nothing of it stays live in registers across the class loops
// (the kernels sit at the 255-register limit).  q-adaptive cut-off (option): of every class the tile keeps the records whose q_cut
// exceeds its smallest |q|.  Ticket protocol over the chunks of the tile that have work (chunk 0 always takes part: it stores, zeros
// if need be): a chunk without work leaves at once instead of holding an SM slot until its turn comes — with the cut-off the far-out
// tiles keep only a prefix of every class, i.e. only their first chunks.
struct CtaPlan {                                          // one per CTA, in shared memory
    int nrec[kFastMaxClass + 1], nact[kFastMaxClass + 1];
    unsigned long long off[kFastMaxClass + 1];            // byte offset of the first record from the stream base
    long long row[kFastMaxClass + 1];                     // its stream-order index (row of the factor tables)
    int turn, next;                                       // my turn at the tile's ticket (-1: no work), and the value I pass on
    double sh_min[8];
};
// Whole-CTA call.  q2_min: the smallest |q|^2 over this thread's valid points (1e300 if it has none); read only with the cut-off on.
template <int NS>
__device__ __forceinline__ void plan_cta(const V1Args& v, int chunk, double q2_min, CtaPlan& p)
{
    double q_min = 0.0;
    if (v.qcut != nullptr) q_min = sqrt(block_min(q2_min, p.sh_min));
    if (threadIdx.x <= kFastMaxClass) {
        const int L = threadIdx.x;
        const StreamDesc& d = *v.desc;
        const V1Chunk& ck = d.chunks[chunk];
        int n = ck.n[L];
        SCARF_CHECK(n >= 0 && ck.begin[L] >= 0 && (long long)ck.begin[L] + n <= d.cls_n[L]);
        // records of the class this TILE keeps (all of them unless the q-adaptive cut-off is on)
        const int n_act = v.qcut != nullptr ? active_prefix(v.qcut + d.cls_first[L], d.cls_n[L], q_min) : (int)d.cls_n[L];
        p.nact[L] = n_act;
        n = max(0, min(n, n_act - ck.begin[L]));
        if (v.work != nullptr && n > 0) atomicAdd(v.work + L, (unsigned long long)n);
        p.nrec[L] = n;
        p.off[L] = d.cls_off[L] + (unsigned long long)ck.begin[L] * (unsigned long long)(rec_doubles(L, NS) * 8);
        p.row[L] = d.cls_first[L] + ck.begin[L];
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const StreamDesc& d = *v.desc;
        auto has_work = [&](int k) {
            if (k == 0) return true;
            for (int L = 0; L <= kFastMaxClass; ++L)
                if (d.chunks[k].n[L] > 0 && p.nact[L] > d.chunks[k].begin[L]) return true;
            return false;
        };
        int before = 0;
        for (int k = 0; k < chunk; ++k) before += has_work(k) ? 1 : 0;
        bool later = false;
        for (int k = chunk + 1; k < v.n_chunks; ++k) later = later || has_work(k);
        p.turn = has_work(chunk) ? before : -1;             // -1: nothing to do, nothing to add
        p.next = later ? before + 1 : 0;                    // the last working chunk puts the ticket back to 0
    }
    __syncthreads();
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

// ---- product grid: two points that differ in q_x only (ff_grid.cu; the thread's points (ixl, iy, iz), (ixl + 2, iy, iz)) ----
// Eq. (48)'s polynomial, sorted by the power of q_x:  A + iB = sum_t q_x^t (Ce_t + i Co_t),
//   Ce_t = sum_{(u,v): t+u+v even} D_tuv q_y^u q_z^v,   Co_t likewise for t+u+v odd
// (i^n is folded into D).  The (q_y, q_z) sums are the same for both points: evaluated ONCE per (record, state), then
// each point needs only the short polynomial in its own q_x.  FP64 slots per (q, pair, state), accumulate included:
// L = 1: 5 + 2/2 = 6 (monomial form: 7), L = 2: 7 + 7/2 = 10.5 (13), L = 3: 9 + 16/2 = 17 (23).
__host__ __device__ constexpr int yz_index(int u, int v) { return (u + v) * (u + v + 1) / 2 - 1 + v; }   // u + v >= 1
__host__ __device__ constexpr int yz_count(int L) { return (L + 1) * (L + 2) / 2 - 1; }
// is h the first Hermite index (in stream order) of its (parity of n, t) group?
__host__ __device__ constexpr bool xgroup_first(int h)
{
    for (int g = 0; g < h; ++g)
        if (((hdeg(g) ^ hdeg(h)) & 1) == 0 && hexp(g, 0) == hexp(h, 0)) return false;
    return true;
}
__host__ __device__ constexpr bool xgroup_exists(int L, int par, int t)
{
    for (int h = 0; h < nherm(L); ++h)
        if ((hdeg(h) & 1) == par && hexp(h, 0) == t) return true;
    return false;
}

// yzm[yz_index(u, v)] = q_y^u q_z^v (1 <= u + v <= L); xp[j][t] = q_x(point j)^t
template <int L>
__device__ __forceinline__ void make_xpair_monomials(const double (&qv)[kNQ][4], double (&yzm)[yz_count(L) > 0 ? yz_count(L) : 1],
                                                     double (&xp)[kNQ][L + 1])
{
    static_for<yz_count(L)>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        constexpr int d = i < 2 ? 1 : (i < 5 ? 2 : 3);
        constexpr int v = i - (d * (d + 1) / 2 - 1), u = d - v;
        if constexpr (d == 1) yzm[i] = v ? qv[0][2] : qv[0][1];
        else if constexpr (u > 0) yzm[i] = yzm[yz_index(u - 1, v)] * qv[0][1];
        else yzm[i] = yzm[yz_index(u, v - 1)] * qv[0][2];
    });
#pragma unroll
    for (int j = 0; j < kNQ; ++j) {
        xp[j][0] = 1.0;
#pragma unroll
        for (int t = 1; t <= L; ++t) xp[j][t] = t == 1 ? qv[j][0] : xp[j][t - 1] * qv[j][0];
    }
}

template <int L, int NS>
__device__ __forceinline__ void record_accum_xpair(const double2* __restrict__ r2, const double (&yzm)[yz_count(L) > 0 ? yz_count(L) : 1],
                                                   const double (&xp)[kNQ][L + 1], const double (&gc)[kNQ], const double (&gs)[kNQ],
                                                   double (&re)[kNQ][NS], double (&im)[kNQ][NS])
{
    static_assert(L <= 3, "degree blocks take over beyond L = 3");
    constexpr int NH = nherm(L), N = NS * NH;
    const double2* __restrict__ D2 = r2 + 2;
    double G[2][L + 1];                                   // [parity of n][t]: the (q_y, q_z) sums of the current state
    static_for<(N + 1) / 2>([&](auto i2c) {
        constexpr int i2 = decltype(i2c)::value;
        const double2 c = D2[i2];
        static_for<2>([&](auto halfc) {
            constexpr int half = decltype(halfc)::value;
            constexpr int i = 2 * i2 + half;
            if constexpr (i < N) {
                constexpr int s = i / NH, h = i % NH;
                constexpr int t = hexp(h, 0), u = hexp(h, 1), v = hexp(h, 2), par = hdeg(h) & 1;
                const double cv = half ? c.y : c.x;
                if constexpr (u + v == 0) G[par][t] = cv;            // lowest degree of its group: always its first term
                else if constexpr (xgroup_first(h)) G[par][t] = cv * yzm[yz_index(u, v)];
                else G[par][t] = fma(cv, yzm[yz_index(u, v)], G[par][t]);
                if constexpr (h == NH - 1) {
#pragma unroll
                    for (int j = 0; j < kNQ; ++j) {
                        double A = G[0][0], B = 0.0;
                        static_for<L>([&](auto tc) {
                            constexpr int tt = decltype(tc)::value + 1;
                            if constexpr (xgroup_exists(L, 0, tt)) A = fma(G[0][tt], xp[j][tt], A);
                        });
                        if constexpr (L > 0) {
                            if constexpr (xgroup_exists(L, 1, 0)) B = G[1][0];
                            static_for<L>([&](auto tc) {
                                constexpr int tt = decltype(tc)::value + 1;
                                if constexpr (xgroup_exists(L, 1, tt)) {
                                    if constexpr (tt == 1 && !xgroup_exists(L, 1, 0)) B = G[1][1] * xp[j][1];
                                    else B = fma(G[1][tt], xp[j][tt], B);
                                }
                            });
                        }
                        re[j][s] = fma(gc[j], A, re[j][s]);
                        im[j][s] = fma(gs[j], A, im[j][s]);
                        if constexpr (L > 0) {
                            re[j][s] = fma(-gs[j], B, re[j][s]);
                            im[j][s] = fma(gc[j], B, im[j][s]);
                        }
                    }
                }
            }
        });
    });
}


// ---- high classes (L >= 4): degree-block evaluation ---------------------------------------------------------
// Holding all n_herm(L) monomials of two q-points in registers is impossible beyond L = 3 (35..84 doubles per
// point).  The polynomial is therefore evaluated block by block: block 0 = Hermite indices [0, 20) (degrees <= 3),
// then each degree shell n = 4..L in pieces of at most kBlkMax monomials.  A block's monomials are built once
// per batch of kBlkRec records (degree-n monomials as products of two or three held degree <= 2 monomials) and
// every block ends with its own accumulate acc += (gc + i gs)(A_blk + i B_blk) — 2 extra issue slots per state
// and block on top of the W(L) = n_herm + 3 of the work model (a shell has one parity, so only A or only B).
constexpr int kBlkMax = 16;
constexpr int kBlkRec = 2;
__host__ __device__ constexpr int blk_pieces(int n) { return (nherm(n) - nherm(n - 1) + kBlkMax - 1) / kBlkMax; }
__host__ __device__ constexpr int blk_count(int L)
{
    int c = 1;
    for (int n = 4; n <= L; ++n) c += blk_pieces(n);
    return c;
}
__host__ __device__ constexpr int blk_begin(int L, int b)   // first Hermite index of block b (b == blk_count: n_herm)
{
    if (b == 0) return 0;
    int c = 1;
    for (int n = 4; n <= L; ++n) {
        const int sz = nherm(n) - nherm(n - 1), np = blk_pieces(n), per = (sz + np - 1) / np;
        for (int p = 0; p < np; ++p, ++c)
            if (c == b) return nherm(n - 1) + p * per;
    }
    return nherm(L);
}
__host__ __device__ constexpr int var_at(int t, int u, int pos) { return pos < t ? 0 : (pos < t + u ? 1 : 2); }
// k-th factor (index of a degree <= 2 monomial; 0 = the constant 1) of monomial h written as a product of pairs
__host__ __device__ constexpr int factor_index(int h, int k)
{
    const int t = hexp(h, 0), u = hexp(h, 1), n = hdeg(h);
    if (2 * k >= n) return 0;
    int e[3] = {0, 0, 0};
    e[var_at(t, u, 2 * k)]++;
    if (2 * k + 1 < n) e[var_at(t, u, 2 * k + 1)]++;
    return hindex(e[0], e[1], e[2]);
}
__host__ __device__ constexpr int first_of_parity(int H0, int BS, int par)
{
    for (int h = H0; h < H0 + BS; ++h)
        if ((hdeg(h) & 1) == par) return h;
    return -1;
}

template <int H0, int BS, int NQA>
__device__ __forceinline__ void block_monomials(const double (&lo)[NQA][10], double (&mb)[NQA][BS])
{
#pragma unroll
    for (int j = 0; j < NQA; ++j)
        static_for<BS>([&](auto ic) {
            constexpr int h = H0 + decltype(ic)::value;
            constexpr int f0 = factor_index(h, 0), f1 = factor_index(h, 1), f2 = factor_index(h, 2);
            double m = lo[j][f0] * lo[j][f1];
            if constexpr (f2 != 0) m *= lo[j][f2];
            mb[j][decltype(ic)::value] = m;
        });
}

// acc += (gc + i gs) * sum_{h in [H0, H0+BS)} D[s][h] mono[h]      (parity of deg h routes a term to A or B)
template <int L, int NS, int NQA, int jq0, int H0, int BS>
__device__ __forceinline__ void record_accum_block(const double2* __restrict__ r2, const double (&mb)[NQA][BS],
                                                   const double (&gc)[NQA], const double (&gs)[NQA],
                                                   double (&re)[kNQ][NS], double (&im)[kNQ][NS])
{
    constexpr int NH = nherm(L);
    constexpr int hA = first_of_parity(H0, BS, 0), hB = first_of_parity(H0, BS, 1);
    const double2* __restrict__ D2 = r2 + 2;
    static_for<NS>([&](auto sc) {
        constexpr int s = decltype(sc)::value;
        double A[NQA], B[NQA];
        static_for<BS>([&](auto ic) {
            constexpr int i = decltype(ic)::value, h = H0 + i, idx = s * NH + h;
            const double2 c2 = D2[idx / 2];
            const double cv = (idx & 1) ? c2.y : c2.x;
#pragma unroll
            for (int j = 0; j < NQA; ++j) {
                if constexpr (h == 0) A[j] = cv;
                else if constexpr (h == hA) A[j] = cv * mb[j][i];
                else if constexpr (h == hB) B[j] = cv * mb[j][i];
                else if constexpr (hdeg(h) & 1) B[j] = fma(cv, mb[j][i], B[j]);
                else A[j] = fma(cv, mb[j][i], A[j]);
            }
        });
#pragma unroll
        for (int j = 0; j < NQA; ++j) {
            if constexpr (hA >= 0) {
                re[jq0 + j][s] = fma(gc[j], A[j], re[jq0 + j][s]);
                im[jq0 + j][s] = fma(gs[j], A[j], im[jq0 + j][s]);
            }
            if constexpr (hB >= 0) {
                re[jq0 + j][s] = fma(-gs[j], B[j], re[jq0 + j][s]);
                im[jq0 + j][s] = fma(gc[j], B[j], im[jq0 + j][s]);
            }
        }
    });
}

// all blocks of class L for a batch of nb <= kBlkRec records (rec0, rec0 + REC, ...) whose factors are gc/gs
template <int L, int NS>
__device__ __forceinline__ void accum_blocks(const unsigned char* rec0, int nb, const double (&qv)[kNQ][4],
                                             const double (&gc)[kBlkRec][kNQ], const double (&gs)[kBlkRec][kNQ],
                                             double (&re)[kNQ][NS], double (&im)[kNQ][NS])
{
    constexpr int REC = rec_doubles(L, NS) * 8;
    static_for<blk_count(L)>([&](auto bc) {
        constexpr int b = decltype(bc)::value;
        constexpr int H0 = blk_begin(L, b), BS = blk_begin(L, b + 1) - H0;
        double mb[kNQ][BS];
        if constexpr (b == 0) {
            static_assert(BS == nherm(3), "block 0 is the L = 3 monomial set");
            make_monomials<3, kNQ, 0>(qv, mb);
        } else {
            double lo[kNQ][10];
            make_monomials<2, kNQ, 0>(qv, lo);
            block_monomials<H0, BS, kNQ>(lo, mb);
        }
        static_for<kBlkRec>([&](auto rc) {
            constexpr int r = decltype(rc)::value;
            if (r < nb)
                record_accum_block<L, NS, kNQ, 0, H0, BS>(reinterpret_cast<const double2*>(rec0 + r * REC), mb, gc[r], gs[r], re, im);
        });
    });
}

}  // namespace scarf

// ff_row.cu — S4 on a Cartesian product grid, row decomposition (Eq. (45)-(46), (48) PAPER.md:309-330).
//
// Same sum as ff_grid.cu,
//   f_s(q) = sum_pairs X_P(ix) Y_P(iy) Z_P(iz) (A_s(q) + i B_s(q)),      A + iB = sum_tuv D_tuv q_x^t q_y^u q_z^v  (i^n folded into D),
// with the polynomial sorted by the power of q_z:
//   A + iB = sum_v q_z^v (Ge_v + i Go_v),     Ge_v = sum_{(t,u): t+u+v even} D_tuv q_x^t q_y^u,   Go_v likewise for t+u+v odd.
// A WARP owns one (ix, iy) row of 64 z-points (lane l: iz = l and l + 32), so q_x, q_y and therefore every G are the same for
// the whole warp.  Per stage of records the warp first evaluates G for all (record, state) pairs of the stage, one pair per lane
// ("pre-pass", into a warp-private shared-memory area), then every lane runs the short polynomial in its own q_z with the G as
// broadcast coefficients.  FP64 slots per (q, pair, state), accumulate included: 2, 5, 7, 9 for L = 0..3 (ff_grid.cu: 2, 6, 10.5,
// 17; monomial form: 2, 7, 13, 23) plus S(L)/64 for the pre-pass (S = 2, 7, 16).  Classes L >= 4 use the degree blocks of
// ff_common.cuh as the other kernels do.  The factor: X Y is the row's too (pre-pass, one lane per record), so a point needs
// g = (X Y) Z only: 4 slots per (q, pair) instead of 6.
//
// A CTA = 4 warps = 4 consecutive iy at one ix: a 1 x 4 x 64 box.  Everything else — the pair stream through a ring of 1-D TMA
// bulk copies on one mbarrier per stage (two stages of up to 24 records here: a stage carries 1 KB of Z factors per record), per-axis
// factor tables [box][record][point in box], cost-balanced stream chunks that add into `out` in chunk order through the box's
// ticket, the conjugate mirror store on inversion-symmetric grids, the q-adaptive prefix — is the scheme of ff_grid.cu.
// Measured on config 3 (64^3, symmetric half, B200): 6.41 ms against 7.52 ms for ff_grid.cu.  Not kept: three stages of 16 records
// (6.51 ms), a last-arriver refill instead of the __syncthreads per stage (6.68 ms).
#include "ff_common.cuh"

namespace scarf {

namespace {

constexpr int kThreads = 128;
constexpr int kWarps = kThreads / 32;
constexpr int kStages = 2;
constexpr int kStageBytes = 12288;            // records of one stage (>= the largest record, L = 6, NS = 12)
constexpr int kMaxRec = 24;                   // records per stage at most (bounds the table slices)
constexpr int kXB = kRowBX * 16, kYB = kRowBY * 16, kZB = kRowBZ * 16;   // table bytes per record and box
constexpr int kSlotBytes = kStageBytes + kMaxRec * (kXB + kYB + kZB);
static_assert(kMaxRec <= 32 && kRowBX == 1 && kRowBY == kWarps && kRowBZ == 32 * kNQ, "warp = one (ix, iy) row, two z-points per lane");

// (parity of n, power of q_z) groups of class L, par 0 first, v ascending
__host__ __device__ constexpr bool zgroup_exists(int L, int par, int v) { return ((v & 1) == par ? v : v + 1) <= L; }
__host__ __device__ constexpr int zgroup_index(int L, int par, int v)
{
    int idx = 0;
    for (int p = 0; p < 2; ++p)
        for (int vv = 0; vv <= L; ++vv) {
            if (p == par && vv == v) return idx;
            if (zgroup_exists(L, p, vv)) ++idx;
        }
    return idx;
}
__host__ __device__ constexpr int zgroup_count(int L) { return zgroup_index(L, 2, 0); }
// is h the first Hermite index (stream order) of its group?
__host__ __device__ constexpr bool zgroup_first(int h)
{
    for (int g = 0; g < h; ++g)
        if (((hdeg(g) ^ hdeg(h)) & 1) == 0 && hexp(g, 2) == hexp(h, 2)) return false;
    return true;
}
__host__ __device__ constexpr int g_stride(int L, int NS) { return (NS * zgroup_count(L) + 1) & ~1; }       // doubles per record
__host__ __device__ constexpr int stage_records(int L, int NS)
{
    const int n = kStageBytes / (rec_doubles(L, NS) * 8);
    return n < kMaxRec ? n : kMaxRec;
}
// warp-private area: XY[kMaxRec] (the row's X_P(ix) Y_P(iy) of the stage's records, complex) followed by the G of the stage
__host__ __device__ constexpr int g_warp_bytes(int NS)
{
    int m = 16;
    for (int L = 1; L <= 3; ++L) {
        const int b = stage_records(L, NS) * g_stride(L, NS) * 8;
        if (b > m) m = b;
    }
    return m + kMaxRec * 16;
}
template <int NS> constexpr int smem_bytes() { return kStages * kSlotBytes + kWarps * g_warp_bytes(NS) + 64; }

struct RPipe {
    unsigned char* buf;     // kStages slots of kSlotBytes: records | X slice | Y slice | Z slice
    uint64_t* full;
    uint32_t it;
};

__device__ __forceinline__ double2 cmul(const double2 a, const double2 b)
{
    return make_double2(fma(a.x, b.x, -(a.y * b.y)), fma(a.x, b.y, a.y * b.x));
}

// ---- pre-pass: G[record][state][group] of one stage for this warp's row ------------------------------------------------------
// xym[yz_index(t, u)] = q_x^t q_y^u (1 <= t + u <= L).  One (record, state) pair per lane and trip.
template <int L, int NS>
__device__ __forceinline__ void row_prepass(const unsigned char* sp, int cnt, const double (&xym)[yz_count(L)], double* Gw, int lane)
{
    constexpr int REC = rec_doubles(L, NS) * 8, NH = nherm(L), NG = zgroup_count(L), GS = g_stride(L, NS);
    // Unrolled over the at most TRIPS items of a lane (a rolled loop cost 1 % of the kernel more).  Measured alternatives: two or
    // three items per branch-free group, so that their loads are in flight together, shorten the pre-pass (3.8 % -> 2.2 % of the
    // samples for L = 1) but the kernel as a whole got 1.4 % slower (the main loops lost what the pre-pass gained).
    constexpr int TRIPS = (stage_records(L, NS) * NS + 31) / 32;
    const int n = cnt * NS;
#pragma unroll 5
    for (int tr = 0; tr < TRIPS; ++tr) {
        const int i = lane + 32 * tr;
        if (i >= n) break;
        const int k = i / NS, s = i - k * NS;
        const double* D = reinterpret_cast<const double*>(sp + k * REC) + 4 + s * NH;
        double G[NG];
        static_for<NH>([&](auto hc) {
            constexpr int h = decltype(hc)::value;
            constexpr int t = hexp(h, 0), u = hexp(h, 1), v = hexp(h, 2), g = zgroup_index(L, hdeg(h) & 1, v);
            const double cv = D[h];
            if constexpr (t + u == 0) G[g] = cv;
            else if constexpr (zgroup_first(h)) G[g] = cv * xym[yz_index(t, u)];
            else G[g] = fma(cv, xym[yz_index(t, u)], G[g]);
        });
        double* o = Gw + k * GS + s * NG;
#pragma unroll
        for (int g = 0; g < NG; ++g) o[g] = G[g];
    }
}

// ---- one record, L = 1..3: acc += (gc + i gs) sum_v z^v (Ge_v + i Go_v), G from the warp's area ------------------------------
template <int L, int NS>
__device__ __forceinline__ void record_accum_row(const double2* __restrict__ G2, const double (&zp)[kNQ][L + 1], const double (&gc)[kNQ],
                                                 const double (&gs)[kNQ], double (&re)[kNQ][NS], double (&im)[kNQ][NS])
{
    constexpr int NG = zgroup_count(L), N = NS * NG;
    double G[NG];
    static_for<(N + 1) / 2>([&](auto i2c) {
        constexpr int i2 = decltype(i2c)::value;
        const double2 c = G2[i2];
        static_for<2>([&](auto halfc) {
            constexpr int half = decltype(halfc)::value;
            constexpr int i = 2 * i2 + half;
            if constexpr (i < N) {
                constexpr int s = i / NG, g = i % NG;
                G[g] = half ? c.y : c.x;
                if constexpr (g == NG - 1) {
#pragma unroll
                    for (int j = 0; j < kNQ; ++j) {
                        double A = G[zgroup_index(L, 0, 0)], B = G[zgroup_index(L, 1, 0)];
                        static_for<L>([&](auto vc) {
                            constexpr int v = decltype(vc)::value + 1;
                            if constexpr (zgroup_exists(L, 0, v)) A = fma(G[zgroup_index(L, 0, v)], zp[j][v], A);
                            if constexpr (zgroup_exists(L, 1, v)) B = fma(G[zgroup_index(L, 1, v)], zp[j][v], B);
                        });
                        re[j][s] = fma(gc[j], A, re[j][s]);
                        im[j][s] = fma(gs[j], A, im[j][s]);
                        re[j][s] = fma(-gs[j], B, re[j][s]);
                        im[j][s] = fma(gc[j], B, im[j][s]);
                    }
                }
            }
        });
    });
}

// ---- one class segment of the chunk ----------------------------------------------------------------------------------------
// r0 = stream-order index of the segment's first record (row of the tables).  qv[j] = (q_x, q_y, q_z of point j, 0).
template <int L, int NS>
__device__ __forceinline__ void run_class_row(RPipe& pp, const GridArgs& a, const char* __restrict__ seg, long long r0, int n_rec,
                                              int bx, int by, int bz, int warp, int lane, double* Ww,
                                              const double (&qv)[kNQ][4], double (&re)[kNQ][NS], double (&im)[kNQ][NS])
{
    constexpr int REC = rec_doubles(L, NS) * 8;
    constexpr int SREC = stage_records(L, NS);
    static_assert(SREC >= 1, "record larger than a stage");
    const int n_st = (n_rec + SREC - 1) / SREC;
    const bool producer = threadIdx.x == 0;
    auto issue = [&](int j) {
        const int slot = (int)((pp.it + (uint32_t)j) % kStages);
        const int first = j * SREC, cnt = min(SREC, n_rec - first);
        unsigned char* sb = pp.buf + slot * kSlotBytes;
        const long long r = r0 + first;
        SCARF_CHECK(cnt >= 1 && cnt <= kMaxRec && cnt * REC <= kStageBytes && r >= 0 && r + cnt <= a.n_rows && slot >= 0 && slot < kStages);
        mbar_expect_tx(&pp.full[slot], (uint32_t)cnt * (REC + kXB + kYB + kZB));
        bulk_g2s(sb, seg + (size_t)first * REC, (uint32_t)cnt * REC, &pp.full[slot]);
        bulk_g2s(sb + kStageBytes, a.tx + ((size_t)bx * a.n_rows + r) * kRowBX, (uint32_t)cnt * kXB, &pp.full[slot]);
        bulk_g2s(sb + kStageBytes + kMaxRec * kXB, a.ty + ((size_t)by * a.n_rows + r) * kRowBY, (uint32_t)cnt * kYB, &pp.full[slot]);
        bulk_g2s(sb + kStageBytes + kMaxRec * (kXB + kYB), a.tz + ((size_t)bz * a.n_rows + r) * kRowBZ, (uint32_t)cnt * kZB,
                 &pp.full[slot]);
    };
    // per-class monomials: powers of this lane's q_z; the row's q_x^t q_y^u for the pre-pass
    double zp[kNQ][(L >= 1 && L <= 3) ? L + 1 : 1];
    double xym[(L >= 1 && L <= 3) ? yz_count(L) : 1];
    if constexpr (L >= 1 && L <= 3) {
        double pv[kNQ][4];
#pragma unroll
        for (int j = 0; j < kNQ; ++j) { pv[j][0] = qv[j][2]; pv[j][1] = qv[0][0]; pv[j][2] = qv[0][1]; pv[j][3] = 0.0; }
        make_xpair_monomials<L>(pv, xym, zp);      // roles permuted: (x, y, z) of that routine = (q_z, q_x, q_y) here
    }
    __syncthreads();                                     // all threads have left the previous segment's stages
    if (producer)
        for (int j = 0; j < min(kStages, n_st); ++j) issue(j);
    for (int j = 0; j < n_st; ++j) {
        const uint32_t g = pp.it + (uint32_t)j;
        const int slot = (int)(g % kStages);
        mbar_wait(&pp.full[slot], (g / kStages) & 1u);
        const int cnt = min(SREC, n_rec - j * SREC);
        const unsigned char* sp = pp.buf + slot * kSlotBytes;
        const double2* Xs = reinterpret_cast<const double2*>(sp + kStageBytes);
        const double2* Ys = reinterpret_cast<const double2*>(sp + kStageBytes + kMaxRec * kXB) + warp;
        const double2* Zs = reinterpret_cast<const double2*>(sp + kStageBytes + kMaxRec * (kXB + kYB)) + lane;
        // pre-pass, part 1: X Y of the row, once per record (lane k: record k) instead of once per lane and record
        double2* XYw = reinterpret_cast<double2*>(Ww);
        double* Gw = Ww + 2 * kMaxRec;
        if (lane < cnt) XYw[lane] = cmul(Xs[lane * kRowBX], Ys[lane * kRowBY]);
        if constexpr (L == 0 || L >= 4) __syncwarp();
        auto factors = [&](int k, double (&gc)[kNQ], double (&gs)[kNQ]) {      // g = X Y Z for this lane's points
            const double2 xy = XYw[k];
#pragma unroll
            for (int jj = 0; jj < kNQ; ++jj) {
                const double2 gq = cmul(Zs[k * kRowBZ + 32 * jj], xy);
                gc[jj] = gq.x;
                gs[jj] = gq.y;
            }
        };
        if constexpr (L >= 4) {                         // degree blocks, both q-points together (ff_common.cuh)
#pragma unroll 1
            for (int k0 = 0; k0 < cnt; k0 += kBlkRec) {
                const int nb = min(kBlkRec, cnt - k0);
                double gcb[kBlkRec][kNQ], gsb[kBlkRec][kNQ];
                static_for<kBlkRec>([&](auto rc) {
                    constexpr int r = decltype(rc)::value;
                    if (r < nb) factors(k0 + r, gcb[r], gsb[r]);
                });
                accum_blocks<L, NS>(sp + k0 * REC, nb, qv, gcb, gsb, re, im);
            }
        } else {
            if constexpr (L >= 1) {
                row_prepass<L, NS>(sp, cnt, xym, Gw, lane);
                __syncwarp();
            }
            auto accum = [&](int k, const double (&gc)[kNQ], const double (&gs)[kNQ]) {
                if constexpr (L == 0) {
                    double mono[kNQ][1];
#pragma unroll
                    for (int jj = 0; jj < kNQ; ++jj) mono[jj][0] = 1.0;
                    record_accum<0, NS, kNQ, 0>(reinterpret_cast<const double2*>(sp + k * REC), mono, gc, gs, re, im);
                } else {
                    record_accum_row<L, NS>(reinterpret_cast<const double2*>(Gw + k * g_stride(L, NS)), zp, gc, gs, re, im);
                }
            };
            // software-pipelined by groups of U records: the table loads and complex products of group k+1 are issued alongside
            // the accumulate of group k
            constexpr int U = L <= 1 ? 2 : 1;
            const int n_full = cnt / U * U;
            double gc[U][kNQ], gs[U][kNQ];
            if (n_full > 0) {
#pragma unroll
                for (int u = 0; u < U; ++u) factors(u, gc[u], gs[u]);
#pragma unroll 1
                for (int k = 0; k + U < n_full; k += U) {
                    double gcn[U][kNQ], gsn[U][kNQ];
#pragma unroll
                    for (int u = 0; u < U; ++u) factors(k + U + u, gcn[u], gsn[u]);
#pragma unroll
                    for (int u = 0; u < U; ++u) accum(k + u, gc[u], gs[u]);
#pragma unroll
                    for (int u = 0; u < U; ++u)
#pragma unroll
                        for (int jj = 0; jj < kNQ; ++jj) { gc[u][jj] = gcn[u][jj]; gs[u][jj] = gsn[u][jj]; }
                }
#pragma unroll
                for (int u = 0; u < U; ++u) accum(n_full - U + u, gc[u], gs[u]);
            }
#pragma unroll 1
            for (int k = n_full; k < cnt; ++k) {
                factors(k, gc[0], gs[0]);
                accum(k, gc[0], gs[0]);
            }
        }
        __syncthreads();                                 // the slot and the G areas are free again
        if (producer && j + kStages < n_st) issue(j + kStages);
    }
    pp.it += (uint32_t)n_st;
}

template <int NS>
__global__ void __launch_bounds__(kThreads, 2) ff_row_kernel(const GridArgs a)
{
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem + kStages * kSlotBytes);
    int tile, chunk;
    cta_tile_chunk(a.v, tile, chunk);
    if (threadIdx.x == 0) {
        for (int s = 0; s < kStages; ++s) mbar_init(&full_bar[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    RPipe pp = {smem, full_bar, 0u};
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double* Ww = reinterpret_cast<double*>(smem + kStages * kSlotBytes + 64 + warp * g_warp_bytes(NS));   // the warp's private area

    const int bz = tile % a.nbz, by = (tile / a.nbz) % a.nby, bx = a.bx0 + tile / (a.nbz * a.nby);
    const int ix = bx, iy = by * kRowBY + warp;
    const bool row_ok = ix < a.nx_eval && iy < a.ny;
    double qv[kNQ][4];
#pragma unroll
    for (int j = 0; j < kNQ; ++j) {
        const int iz = bz * kRowBZ + lane + 32 * j;
        const bool ok = row_ok && iz < a.nz;
        qv[j][0] = row_ok ? a.qx[ix] : 0.0;            // the row's q_x, q_y are warp-uniform whatever iz is
        qv[j][1] = row_ok ? a.qy[iy] : 0.0;
        qv[j][2] = ok ? a.qz[iz] : 0.0;
        qv[j][3] = 0.0;
    }
    double re[kNQ][NS], im[kNQ][NS];
#pragma unroll
    for (int j = 0; j < kNQ; ++j)
#pragma unroll
        for (int s = 0; s < NS; ++s) re[j][s] = im[j][s] = 0.0;

    __shared__ CtaPlan plan;                                // per class: the records this CTA evaluates; its ticket turn (ff_common.cuh)
    {
        double m2 = 1e300;
#pragma unroll
        for (int j = 0; j < kNQ; ++j)
            if (row_ok && bz * kRowBZ + lane + 32 * j < a.nz)
                m2 = fmin(m2, qv[j][0] * qv[j][0] + qv[j][1] * qv[j][1] + qv[j][2] * qv[j][2]);
        plan_cta<NS>(a.v, chunk, m2, plan);
    }
#define SCARF_ROW_CLASS(LV)                                                                                          \
    if (plan.nrec[LV] > 0)                                                                                           \
        run_class_row<LV, NS>(pp, a, a.v.base + plan.off[LV], plan.row[LV], plan.nrec[LV], bx, by, bz, warp, lane, Ww, qv, re, im);
    SCARF_ROW_CLASS(0)
    SCARF_ROW_CLASS(1)
    SCARF_ROW_CLASS(2)
    SCARF_ROW_CLASS(3)
    SCARF_ROW_CLASS(4)
    SCARF_ROW_CLASS(5)
    SCARF_ROW_CLASS(6)
#undef SCARF_ROW_CLASS

    // ---- epilogue: store (one chunk) or add into `out` in chunk order (several); the LAST chunk holds the final value and
    // also stores its conjugate at the mirror point when the grid is inversion-symmetric
    double2* dst = reinterpret_cast<double2*>(a.v.dst);
    double2* fin = a.v.dst_final != nullptr ? reinterpret_cast<double2*>(a.v.dst_final) : dst;    // finished values (last chunk)
    const int turn = plan.turn;
    if (turn < 0) return;                                   // a chunk without work (uniform over the CTA)
    const bool first = turn == 0, last = plan.next == 0;
    if (a.v.n_chunks > 1) ticket_wait(a.v.tickets + tile, turn);
#pragma unroll
    for (int j = 0; j < kNQ; ++j) {
        const int iz = bz * kRowBZ + lane + 32 * j;
        if (row_ok && iz < a.nz) {
            const long long i = ((long long)ix * a.ny + iy) * a.nz + iz;
            const bool mirror = last && a.sym && 2 * ix < a.nx - 1;
            SCARF_CHECK(i >= 0 && i < a.v.n_q);
#pragma unroll
            for (int s = 0; s < NS; ++s)
                if (s < a.v.ns_real) {
                    double2* o = dst + (size_t)s * a.v.n_q;
                    double2 v = make_double2(re[j][s], im[j][s]);
                    if (!first) {
                        const double2 p = __ldcg(o + i);
                        v.x += p.x;
                        v.y += p.y;
                    }
                    double2* w = (last ? fin : dst) + (size_t)s * a.v.n_q;
                    w[i] = v;
                    if (mirror) w[a.v.n_q - 1 - i] = make_double2(v.x, -v.y);   // f(-q) = conj f(q)
                }
        }
    }
    if (a.v.n_chunks > 1) ticket_pass(a.v.tickets + tile, plan.next);
}

template <int NS>
cudaError_t launch_row_ns(const GridArgs& a, cudaStream_t st)
{
    const dim3 grid((unsigned)a.v.n_tiles, (unsigned)a.v.n_chunks, 1);   // dispatched x fastest: chunk-major
    ff_row_kernel<NS><<<grid, kThreads, smem_bytes<NS>(), st>>>(a);
    return cudaGetLastError();
}

}  // namespace

// The kernels need more than 48 KB of dynamic shared memory: an attribute of the function on the CURRENT device.  Called by
// scarf_create for the context's device (idempotent, no process-wide flag).
cudaError_t ff_row_init_device()
{
    cudaError_t e = cudaSuccess;
#define SCARF_ROW_ATTR(NSV) \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(ff_row_kernel<NSV>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes<NSV>());
    SCARF_ROW_ATTR(1) SCARF_ROW_ATTR(2) SCARF_ROW_ATTR(4) SCARF_ROW_ATTR(6) SCARF_ROW_ATTR(8) SCARF_ROW_ATTR(12)
#undef SCARF_ROW_ATTR
    return e;
}

cudaError_t launch_ff_row(int NS, const GridArgs& a, cudaStream_t st)
{
    if (a.v.n_q <= 0 || a.v.n_chunks <= 0 || a.v.n_tiles <= 0) return cudaSuccess;
    if (a.bxs != kRowBX || a.bys != kRowBY || a.bzs != kRowBZ) return cudaErrorInvalidValue;   // tables laid out for another kernel
    switch (NS) {
    case 1: return launch_row_ns<1>(a, st);
    case 2: return launch_row_ns<2>(a, st);
    case 4: return launch_row_ns<4>(a, st);
    case 6: return launch_row_ns<6>(a, st);
    case 8: return launch_row_ns<8>(a, st);
    case 12: return launch_row_ns<12>(a, st);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace scarf

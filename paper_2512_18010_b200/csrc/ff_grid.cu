// ff_grid.cu — S4 on a Cartesian product grid (the V-tensor idea of Eq. (45)-(46)
// on a product grid the pair factor separates per axis).
//
//   q = (qx[ix], qy[iy], qz[iz]);   e^{-q^2/4p} e^{iq.P} = X_P(ix) Y_P(iy) Z_P(iz),
//   X_P(i) = exp(-qx[i]^2/4p + i qx[i] P_x)   (same for Y, Z)
//
//   f_s(q) = sum_pairs X_P(ix) Y_P(iy) Z_P(iz) (A_s(q) + i B_s(q))        Eq. (48)
//
// grid_table_kernel evaluates the (nx + ny + nz) complex factors of every kept pair once (the exp/sincos of
// ff_math.cuh, the same functions the general kernel uses); ff_grid_kernel then needs 12 FP64 issue slots per
// (2 q-points, pair) for the factor — YZ = Y Z, g0 = X0 YZ, g1 = X1 YZ — instead of 2 x 40, and shares the
// (state, Hermite index) accumulate loop with the general kernel (ff_common.cuh).
//
// Inversion symmetry.  f_s(-q) = conj f_s(q) for real T and real orbitals (Fourier sign e^{+iq.r}, Eq. (19)).
// When every axis is antisymmetric bit for bit (ax[i] == -ax[n-1-i]; the host checks) the grid maps onto itself under
// q -> -q: only the half ix < ceil(nx/2) is evaluated and the mirror point (nx-1-ix, ny-1-iy, nz-1-iz) receives the
// conjugate in the same epilogue — half the work, no approximation (tables, monomials and sums are exactly odd/even, so the
// stored value is what a direct evaluation at -q would give).
//
// Work decomposition: a CTA owns a 4 x 8 x 8 box of the grid and one cost-balanced chunk of the pair stream; the chunks of
// one box add into `out` in chunk order through the box's ticket (as in ff_v1.cu); the last chunk also stores the mirror.
// Thread t holds the points (ixl, iyl, izl) and (ixl + 2, iyl, izl), izl = t % 8, iyl = (t / 8) % 8, ixl = t / 64,
// so a warp has one ixl (X0, X1 are broadcast loads) and writes 128-byte runs along z.  Tables are laid out
// [box][record][point-in-box], so that the slice a CTA needs for a run of records is contiguous: per stage one
// TMA bulk copy for the records and one for each of the three table slices, all on one mbarrier.
#include "ff_common.cuh"

namespace scarf {

namespace {

constexpr int kThreads = 128;
constexpr int kStages = 3;
constexpr int kStageBytes = 8192;             // records of one stage (>= the largest record, L = 6, NS = 12)
constexpr int kGridSwpMaxL = 1;                // classes whose record loop is software-pipelined (L = 2 as well: 8.69 ms instead of 8.63 ms on config 3)
__host__ __device__ constexpr int grid_swp_records(int L) { return L <= 1 ? 2 : 1; }
constexpr int kMaxRec = 32;                   // records per stage at most (bounds the table slices)
constexpr int kXB = kGridBX * 16, kYB = kGridBY * 16, kZB = kGridBZ * 16;   // table bytes per record and box
constexpr int kSlotBytes = kStageBytes + kMaxRec * (kXB + kYB + kZB);
constexpr int kSmemBytes = kStages * kSlotBytes + 64;
static_assert(kGridBX * kGridBY * kGridBZ == kThreads * kNQ, "box = 2 points per thread");

struct GPipe {
    unsigned char* buf;     // kStages slots of kSlotBytes: records | X slice | Y slice | Z slice
    uint64_t* full;
    uint32_t it;
};

// ---- tables -------------------------------------------------------------------------------------------------
// one thread per (record, padded axis point); columns [0, NXp) -> X, [NXp, NXp+NYp) -> Y, rest -> Z.  The launch is sized for
// a.n_rows records (all prescreened pairs); rows beyond the kept count exit.
__global__ void __launch_bounds__(256) grid_table_kernel(const GridArgs a, double2* __restrict__ tx, double2* __restrict__ ty,
                                                         double2* __restrict__ tz)
{
    const StreamDesc& d = *a.v.desc;
    const int NXp = a.nbx * a.bxs, NYp = a.nby * a.bys, NZp = a.nbz * a.bzs, ncol = NXp + NYp + NZp;
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= d.n_kept * ncol) return;
    const long long r = idx / ncol;
    int col = (int)(idx - r * ncol);
    int c = 0;
#pragma unroll
    for (int k = 1; k < kNClasses; ++k)
        if (r >= d.cls_first[k]) c = k;
    const double* hdr = reinterpret_cast<const double*>(a.v.base + d.cls_off[c] + (size_t)(r - d.cls_first[c]) * d.rec_bytes[c]);
    const double inv4p = hdr[3];
    int axis = 0, n = a.nx_eval, B = a.bxs;
    const double* ax = a.qx;
    double2* tab = tx;
    if (col >= NXp + NYp) { axis = 2; col -= NXp + NYp; n = a.nz; B = a.bzs; ax = a.qz; tab = tz; }
    else if (col >= NXp) { axis = 1; col -= NXp; n = a.ny; B = a.bys; ax = a.qy; tab = ty; }
    double2 v = make_double2(0.0, 0.0);
    if (col < n) {
        const double q = ax[col];
        const double e = exp_neg(q * q * inv4p);
        double sn, cs;
        sincos_fast(q * hdr[axis], sn, cs);
        v = make_double2(e * cs, e * sn);
    }
    tab[((size_t)(col / B) * a.n_rows + r) * B + (col % B)] = v;
}

__device__ __forceinline__ double2 cmul(const double2 a, const double2 b)
{
    return make_double2(fma(a.x, b.x, -(a.y * b.y)), fma(a.x, b.y, a.y * b.x));
}

// ---- one class segment of the chunk ----------------------------------------------------------------------------
// r0 = stream-order index of the segment's first record (row of the tables).
template <int L, int NS>
__device__ __forceinline__ void run_class_grid(GPipe& pp, const GridArgs& a, const char* __restrict__ seg, long long r0, int n_rec,
                                               int bx, int by, int bz, int ixl, int iyl, int izl,
                                               const double (&qv)[kNQ][4], double (&re)[kNQ][NS], double (&im)[kNQ][NS])
{
    constexpr int REC = rec_doubles(L, NS) * 8;
    constexpr int SREC = (kStageBytes / REC) < kMaxRec ? (kStageBytes / REC) : kMaxRec;
    static_assert(SREC >= 1, "record larger than a stage");
    constexpr int NQA = L <= 3 ? kNQ : 1;                // q-points evaluated together (register budget)
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
        bulk_g2s(sb + kStageBytes, a.tx + ((size_t)bx * a.n_rows + r) * kGridBX, (uint32_t)cnt * kXB, &pp.full[slot]);
        bulk_g2s(sb + kStageBytes + kMaxRec * kXB, a.ty + ((size_t)by * a.n_rows + r) * kGridBY, (uint32_t)cnt * kYB, &pp.full[slot]);
        bulk_g2s(sb + kStageBytes + kMaxRec * (kXB + kYB), a.tz + ((size_t)bz * a.n_rows + r) * kGridBZ, (uint32_t)cnt * kZB,
                 &pp.full[slot]);
    };
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
        const double2* Ys = reinterpret_cast<const double2*>(sp + kStageBytes + kMaxRec * kXB);
        const double2* Zs = reinterpret_cast<const double2*>(sp + kStageBytes + kMaxRec * (kXB + kYB));
        if constexpr (L >= 4) {                         // degree blocks, both q-points together (ff_common.cuh)
#pragma unroll 1
            for (int k0 = 0; k0 < cnt; k0 += kBlkRec) {
                const int nb = min(kBlkRec, cnt - k0);
                double gcb[kBlkRec][kNQ], gsb[kBlkRec][kNQ];
                static_for<kBlkRec>([&](auto rc) {
                    constexpr int r = decltype(rc)::value;
                    if (r < nb) {
                        const int k = k0 + r;
                        const double2 yz = cmul(Ys[k * kGridBY + iyl], Zs[k * kGridBZ + izl]);
#pragma unroll
                        for (int jj = 0; jj < kNQ; ++jj) {
                            const double2 gq = cmul(Xs[k * kGridBX + ixl + 2 * jj], yz);
                            gcb[r][jj] = gq.x;
                            gsb[r][jj] = gq.y;
                        }
                    }
                });
                accum_blocks<L, NS>(sp + k0 * REC, nb, qv, gcb, gsb, re, im);
            }
        } else
        {
            // L <= 3: the thread's two points share (q_y, q_z): the (y, z) part of every polynomial is evaluated once for both
            // (ff_common.cuh: record_accum_xpair)
            constexpr int jq0 = 0;
            static_assert(NQA == kNQ, "both points together");
            double yzm[yz_count(L) > 0 ? yz_count(L) : 1], xp[kNQ][L + 1];
            make_xpair_monomials<L>(qv, yzm, xp);
            auto rec = [&](int k) { return reinterpret_cast<const double2*>(sp + k * REC); };
            auto factors = [&](int k, double (&gc)[NQA], double (&gs)[NQA]) {      // g = X Y Z for this thread's points
                const double2 yz = cmul(Ys[k * kGridBY + iyl], Zs[k * kGridBZ + izl]);
#pragma unroll
                for (int jj = 0; jj < NQA; ++jj) {
                    const double2 gq = cmul(Xs[k * kGridBX + ixl + 2 * (jq0 + jj)], yz);
                    gc[jj] = gq.x;
                    gs[jj] = gq.y;
                }
            };
            if constexpr (L <= kGridSwpMaxL) {          // software-pipelined by groups of U records: the per-lane table loads and
                constexpr int U = grid_swp_records(L);  // complex products of group k+1 are issued alongside the accumulate of group k
                const int n_full = cnt / U * U;
                double gc[U][NQA], gs[U][NQA];
                if (n_full > 0) {
#pragma unroll
                    for (int u = 0; u < U; ++u) factors(u, gc[u], gs[u]);
#pragma unroll 1
                    for (int k = 0; k + U < n_full; k += U) {
                        double gcn[U][NQA], gsn[U][NQA];
#pragma unroll
                        for (int u = 0; u < U; ++u) factors(k + U + u, gcn[u], gsn[u]);
#pragma unroll
                        for (int u = 0; u < U; ++u) record_accum_xpair<L, NS>(rec(k + u), yzm, xp, gc[u], gs[u], re, im);
#pragma unroll
                        for (int u = 0; u < U; ++u)
#pragma unroll
                            for (int jj = 0; jj < NQA; ++jj) { gc[u][jj] = gcn[u][jj]; gs[u][jj] = gsn[u][jj]; }
                    }
#pragma unroll
                    for (int u = 0; u < U; ++u) record_accum_xpair<L, NS>(rec(n_full - U + u), yzm, xp, gc[u], gs[u], re, im);
                }
#pragma unroll 1
                for (int k = n_full; k < cnt; ++k) {
                    factors(k, gc[0], gs[0]);
                    record_accum_xpair<L, NS>(rec(k), yzm, xp, gc[0], gs[0], re, im);
                }
            } else {
#pragma unroll 1
                for (int k = 0; k < cnt; ++k) {
                    double gc[NQA], gs[NQA];
                    factors(k, gc, gs);
                    record_accum_xpair<L, NS>(rec(k), yzm, xp, gc, gs, re, im);
                }
            }
        }
        __syncthreads();                                 // the slot is free again
        if (producer && j + kStages < n_st) issue(j + kStages);
    }
    pp.it += (uint32_t)n_st;
}

template <int NS>
__global__ void __launch_bounds__(kThreads, 2) ff_grid_kernel(const GridArgs a)
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
    GPipe pp = {smem, full_bar, 0u};

    const int bz = tile % a.nbz, by = (tile / a.nbz) % a.nby, bx = a.bx0 + tile / (a.nbz * a.nby);
    const int izl = threadIdx.x % kGridBZ, iyl = (threadIdx.x / kGridBZ) % kGridBY, ixl = threadIdx.x / (kGridBZ * kGridBY);
    const int iy = by * kGridBY + iyl, iz = bz * kGridBZ + izl;
    double qv[kNQ][4];
#pragma unroll
    for (int j = 0; j < kNQ; ++j) {
        const int ix = bx * kGridBX + ixl + 2 * j;
        const bool ok = ix < a.nx_eval && iy < a.ny && iz < a.nz;
        qv[j][0] = ok ? a.qx[ix] : 0.0;
        qv[j][1] = ok ? a.qy[iy] : 0.0;
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
            if (bx * kGridBX + ixl + 2 * j < a.nx_eval && iy < a.ny && iz < a.nz)
                m2 = fmin(m2, qv[j][0] * qv[j][0] + qv[j][1] * qv[j][1] + qv[j][2] * qv[j][2]);
        plan_cta<NS>(a.v, chunk, m2, plan);
    }
#define SCARF_GRID_CLASS(LV)                                                                                        \
    if (plan.nrec[LV] > 0)                                                                                          \
        run_class_grid<LV, NS>(pp, a, a.v.base + plan.off[LV], plan.row[LV], plan.nrec[LV], bx, by, bz, ixl, iyl, izl, qv, re, im);
    SCARF_GRID_CLASS(0)
    SCARF_GRID_CLASS(1)
    SCARF_GRID_CLASS(2)
    SCARF_GRID_CLASS(3)
    SCARF_GRID_CLASS(4)
    SCARF_GRID_CLASS(5)
    SCARF_GRID_CLASS(6)
#undef SCARF_GRID_CLASS

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
        const int ix = bx * kGridBX + ixl + 2 * j;
        if (ix < a.nx_eval && iy < a.ny && iz < a.nz) {
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

}  // namespace

cudaError_t launch_grid_tables(const GridArgs& a, double2* tx, double2* ty, double2* tz, cudaStream_t st)
{
    const long long ncol = (long long)a.nbx * a.bxs + (long long)a.nby * a.bys + (long long)a.nbz * a.bzs;
    const long long n = a.n_rows * ncol;
    if (n <= 0) return cudaSuccess;
    grid_table_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(a, tx, ty, tz);
    return cudaGetLastError();
}

template <int NS>
static cudaError_t launch_grid_ns(const GridArgs& a, cudaStream_t st)
{
    const dim3 grid((unsigned)a.v.n_tiles, (unsigned)a.v.n_chunks, 1);   // dispatched x fastest: chunk-major
    ff_grid_kernel<NS><<<grid, kThreads, kSmemBytes, st>>>(a);
    return cudaGetLastError();
}

// The kernels need more than 48 KB of dynamic shared memory: an attribute of the function on the CURRENT device.  Called by scarf_create for the context's device (idempotent, no process-wide flag).
cudaError_t ff_grid_init_device()
{
    cudaError_t e = cudaSuccess;
#define SCARF_GRID_ATTR(NSV) \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(ff_grid_kernel<NSV>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
    SCARF_GRID_ATTR(1) SCARF_GRID_ATTR(2) SCARF_GRID_ATTR(4) SCARF_GRID_ATTR(6) SCARF_GRID_ATTR(8) SCARF_GRID_ATTR(12)
#undef SCARF_GRID_ATTR
    return e;
}

cudaError_t launch_ff_grid(int NS, const GridArgs& a, cudaStream_t st)
{
    if (a.v.n_q <= 0 || a.v.n_chunks <= 0 || a.v.n_tiles <= 0) return cudaSuccess;
    switch (NS) {
    case 1: return launch_grid_ns<1>(a, st);
    case 2: return launch_grid_ns<2>(a, st);
    case 4: return launch_grid_ns<4>(a, st);
    case 6: return launch_grid_ns<6>(a, st);
    case 8: return launch_grid_ns<8>(a, st);
    case 12: return launch_grid_ns<12>(a, st);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace scarf

// ---- separable integrals (Eq. (64)-(65) PAPER.md:481-487) --------------------------------------------------------------
//   I_s = sum_{ix,iy,iz} fx[ix] gy[iy] hz[iz] f_s(qx[ix], qy[iy], qz[iz])
//       = sum_pairs sum_h D^s_h i^{n_h} Mx_P[t_h] My_P[u_h] Mz_P[v_h],    Mx_P[t] = sum_i fx[i] qx[i]^t X_P(i)
// — linear in the axis lengths instead of their product (the paper's point about the V-tensors).  (-1)^{n/2} resp.
// (-1)^{(n-1)/2} of i^n are already folded into D; odd n contribute through i.
namespace scarf {

namespace {

// one thread per (record, axis): 7 complex moments  Mom[record][axis][t], t = 0..kMaxClass
__global__ void __launch_bounds__(128) sep_moments_kernel(const GridArgs a, const double* __restrict__ wx, const double* __restrict__ wy,
                                                          const double* __restrict__ wz, double2* __restrict__ mom)
{
    const StreamDesc& d = *a.v.desc;
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= d.n_kept * 3) return;
    const long long r = idx / 3;
    const int axis = (int)(idx % 3);
    int c = 0;
#pragma unroll
    for (int k = 1; k < kNClasses; ++k)
        if (r >= d.cls_first[k]) c = k;
    const double* hdr = reinterpret_cast<const double*>(a.v.base + d.cls_off[c] + (size_t)(r - d.cls_first[c]) * d.rec_bytes[c]);
    const double inv4p = hdr[3], Pa = hdr[axis];
    const int n = axis == 0 ? a.nx : (axis == 1 ? a.ny : a.nz);
    const double* q = axis == 0 ? a.qx : (axis == 1 ? a.qy : a.qz);
    const double* w = axis == 0 ? wx : (axis == 1 ? wy : wz);
    double mr[kNClasses], mi[kNClasses];
#pragma unroll
    for (int t = 0; t < kNClasses; ++t) mr[t] = mi[t] = 0.0;
    for (int i = 0; i < n; ++i) {
        const double qi = q[i];
        const double e = exp_neg(qi * qi * inv4p) * w[i];
        double sn, cs;
        sincos_fast(qi * Pa, sn, cs);
        double pr = e * cs, pi = e * sn;
#pragma unroll
        for (int t = 0; t < kNClasses; ++t) {
            mr[t] += pr;
            mi[t] += pi;
            pr *= qi;
            pi *= qi;
        }
    }
#pragma unroll
    for (int t = 0; t < kNClasses; ++t) mom[(r * 3 + axis) * kNClasses + t] = make_double2(mr[t], mi[t]);
}

// block b sums records [b * per_block, ...) for every state of the tile: part[b][s]; fixed order, no atomics
__global__ void __launch_bounds__(128) sep_contract_kernel(const GridArgs a, const double2* __restrict__ mom, int per_block,
                                                           double2* __restrict__ part)
{
    __shared__ double2 red[128];
    const int s = threadIdx.x % 16, lane_r = threadIdx.x / 16;      // 16 state slots x 8 record lanes
    const StreamDesc& d = *a.v.desc;
    const long long r0 = (long long)blockIdx.x * per_block, r1 = min(d.n_kept, r0 + per_block);   // blocks past the kept count write zeros
    double accr = 0.0, acci = 0.0;
    if (s < a.v.ns_real)
        for (long long r = r0 + lane_r; r < r1; r += 8) {
            int c = 0;
#pragma unroll
            for (int k = 1; k < kNClasses; ++k)
                if (r >= d.cls_first[k]) c = k;
            const double* rec = reinterpret_cast<const double*>(a.v.base + d.cls_off[c] + (size_t)(r - d.cls_first[c]) * d.rec_bytes[c]);
            const int NH = nherm(c);
            const double* D = rec + 4 + (size_t)s * NH;
            const double2* M = mom + (size_t)r * 3 * kNClasses;
            int h = 0;
            for (int n = 0; n <= c; ++n)
                for (int t = n; t >= 0; --t)
                    for (int u = n - t; u >= 0; --u, ++h) {
                        const double2 xy = cmul(M[t], M[kNClasses + u]);
                        const double2 m = cmul(xy, M[2 * kNClasses + (n - t - u)]);
                        const double d = D[h];
                        if (n & 1) { accr -= d * m.y; acci += d * m.x; }       // i * d * m
                        else { accr += d * m.x; acci += d * m.y; }
                    }
        }
    red[threadIdx.x] = make_double2(accr, acci);
    __syncthreads();
    if (lane_r == 0) {
        double2 t = red[s];
        for (int k = 1; k < 8; ++k) { t.x += red[k * 16 + s].x; t.y += red[k * 16 + s].y; }
        part[(size_t)blockIdx.x * 16 + s] = t;
    }
}

}  // namespace

// mom: [n_rows][3][kNClasses] complex scratch; part: [ceil(n_rows / per_block)][16] complex scratch.  The launches are sized
// for a.n_rows records (all prescreened pairs); the kernels stop at the kept count they read from the descriptor.
cudaError_t launch_separable(const GridArgs& a, const double* wx, const double* wy, const double* wz, double* mom, double* part,
                             int per_block, cudaStream_t st)
{
    if (a.n_rows <= 0) return cudaSuccess;
    const long long n = a.n_rows * 3;
    sep_moments_kernel<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(a, wx, wy, wz, reinterpret_cast<double2*>(mom));
    const unsigned blocks = (unsigned)((a.n_rows + per_block - 1) / per_block);
    sep_contract_kernel<<<blocks, 128, 0, st>>>(a, reinterpret_cast<const double2*>(mom), per_block, reinterpret_cast<double2*>(part));
    return cudaGetLastError();
}

}  // namespace scarf

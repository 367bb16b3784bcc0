// ff_sph.cu — S4 on a spherical product grid (the grid of the angular moments, Eq. (57)-(60)
// PAPER.md:380-398; BASELINE.json config 5):  q = r_i (sin t_j cos phi_k, sin t_j sin phi_k, cos t_j) = r_i n_d,  d = j n_phi + k.
//
// Eq. (48) PAPER.md:326-330 along one direction n (monomials of q = r n, i^n folded into D):
//   A + iB = sum_h D_h q^h = sum_n r^n G_n,      G_n = sum_{deg h = n} D_h n_x^t n_y^u n_z^v      (even n -> A, odd n -> B),
//   e^{-q^2/4p} e^{iq.P} = E_P(r) (cos(r d_P) + i sin(r d_P)),    E_P(r) = e^{-r^2/4p},  d_P = n.P.
// A WARP owns one direction and 64 radii (lane l: i = l and l + 32): d_P and every G_n are the same for the whole warp.  Per
// stage of records the warp evaluates them once ("pre-pass": lane k takes d of record k; lane (k, s) the G of record k and
// state s; results in a warp-private shared-memory area), then every lane needs, per record, one sincos of r d_P, E_P(r) from
// a table, and per state the short polynomial in r (B = r (G_1 + G_3 r^2): the factor r is multiplied into the phase factor once
// per record): FP64 slots per (q, pair, state) 2, 4, 5, 6 for L = 0..3 (list kernel: 2, 7, 13, 23) and 24 per (q, pair) instead
// of 40.  Classes L >= 4: the degree blocks of ff_common.cuh on q = r n.
//
// Inversion symmetry.  f_s(-q) = conj f_s(q) (Eq. (19); real T, real orbitals).  When the theta nodes are
// antisymmetric bit for bit (cos_theta[j] == -cos_theta[n_theta-1-j], e.g. Gauss-Legendre nodes) and n_phi is even, -q of grid
// point (i, j, k) is grid point (i, n_theta-1-j, k + n_phi/2): the host builds the direction table with n_{mirror} = -n_d exactly,
// the kernel evaluates the first half of the directions and stores the conjugate for the mirror point.
//
// A CTA = 4 warps = 4 consecutive directions x 64 radii.  Pair stream through a 2-stage ring of 1-D TMA bulk copies (records +
// the E slice of the radius box), stream chunks with ordered fix-up tickets, q-adaptive prefix: the scheme of ff_grid.cu / ff_row.cu.
#include "ff_common.cuh"

namespace scarf {

namespace {

constexpr int kThreads = 128;
constexpr int kWarps = kThreads / 32;
constexpr int kStages = 2;
constexpr int kStageBytes = 12288;            // records of one stage (>= the largest record, L = 6, NS = 12)
constexpr int kMaxRec = 24;                   // records per stage at most (bounds the E slice and the warp areas)
constexpr int kEB = kSphBR * 8;               // E bytes per record and radius box
constexpr int kSlotBytes = kStageBytes + kMaxRec * kEB;
static_assert(kMaxRec <= 32 && kSphBD == kWarps && kSphBR == 32 * kNQ, "warp = one direction, two radii per lane");

__host__ __device__ constexpr int g_stride(int L, int NS) { return (NS * (L + 1) + 1) & ~1; }       // doubles per record
__host__ __device__ constexpr int stage_records(int L, int NS)
{
    const int n = kStageBytes / (rec_doubles(L, NS) * 8);
    return n < kMaxRec ? n : kMaxRec;
}
// warp-private area: d_P[kMaxRec] followed by the G of the stage
__host__ __device__ constexpr int warp_bytes(int NS)
{
    int m = 16;
    for (int L = 1; L <= 3; ++L) {
        const int b = stage_records(L, NS) * g_stride(L, NS) * 8;
        if (b > m) m = b;
    }
    return m + kMaxRec * 8;
}
template <int NS> constexpr int smem_bytes() { return kStages * kSlotBytes + kWarps * warp_bytes(NS) + 64; }
// is h the first Hermite index (stream order) of its degree?
__host__ __device__ constexpr bool degree_first(int h) { return h == 0 || hdeg(h - 1) != hdeg(h); }

struct SPipe {
    unsigned char* buf;     // kStages slots of kSlotBytes: records | E slice
    uint64_t* full;
    uint32_t it;
};

// ---- table: E[rbox][record][64] = exp(-r^2/4p), zero beyond the last radius ------------------------------------------------
__global__ void __launch_bounds__(256) sph_table_kernel(const SphArgs a, double* __restrict__ te)
{
    const StreamDesc& d = *a.v.desc;
    const int ncol = a.n_rbox * kSphBR;
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= d.n_kept * ncol) return;
    const long long r = idx / ncol;
    const int col = (int)(idx - r * ncol);
    int c = 0;
#pragma unroll
    for (int k = 1; k < kNClasses; ++k)
        if (r >= d.cls_first[k]) c = k;
    const double* hdr = reinterpret_cast<const double*>(a.v.base + d.cls_off[c] + (size_t)(r - d.cls_first[c]) * d.rec_bytes[c]);
    double v = 0.0;
    if (col < a.n_r) {
        const double q = a.r[col];
        v = exp_neg(q * q * hdr[3]);
    }
    te[((size_t)(col / kSphBR) * a.n_rows + r) * kSphBR + (col % kSphBR)] = v;
}

// ---- pre-pass: G[record][state][n] of one stage for this warp's direction ------------------------------------------------------
// dm[h] = n_x^t n_y^u n_z^v.  One (record, state) pair per lane and trip (unrolled; see ff_row.cu for the measured alternatives).
template <int L, int NS>
__device__ __forceinline__ void sph_prepass(const unsigned char* sp, int cnt, const double (&dm)[1][nherm(L)], double* Gw, int lane)
{
    constexpr int REC = rec_doubles(L, NS) * 8, NH = nherm(L), NG = L + 1, GS = g_stride(L, NS);
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
            constexpr int h = decltype(hc)::value, g = hdeg(h);
            const double cv = D[h];
            if constexpr (h == 0) G[0] = cv;
            else if constexpr (degree_first(h)) G[g] = cv * dm[0][h];
            else G[g] = fma(cv, dm[0][h], G[g]);
        });
        double* o = Gw + k * GS + s * NG;
#pragma unroll
        for (int g = 0; g < NG; ++g) o[g] = G[g];
    }
}

// ---- one record, L = 1..3: acc += (gc + i gs) (sum_{n even} r^n G_n + i sum_{n odd} r^n G_n), G from the warp's area -----------
// B has odd powers of r only: B = r B', B' = G_1 + G_3 r^2; the factor r goes into g once per (point, record) — gcr = gc r,
// gsr = gs r — instead of once per (point, record, state).
template <int L, int NS>
__device__ __forceinline__ void record_accum_sph(const double2* __restrict__ G2, const double (&rp)[kNQ][L + 1], const double (&gc)[kNQ],
                                                 const double (&gs)[kNQ], const double (&gcr)[kNQ], const double (&gsr)[kNQ],
                                                 double (&re)[kNQ][NS], double (&im)[kNQ][NS])
{
    constexpr int NG = L + 1, N = NS * NG;
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
                        double A = G[0], B = G[1];
                        if constexpr (L >= 2) A = fma(G[2], rp[j][2], A);
                        if constexpr (L >= 3) B = fma(G[3], rp[j][2], B);
                        re[j][s] = fma(gc[j], A, re[j][s]);
                        im[j][s] = fma(gs[j], A, im[j][s]);
                        re[j][s] = fma(-gsr[j], B, re[j][s]);
                        im[j][s] = fma(gcr[j], B, im[j][s]);
                    }
                }
            }
        });
    });
}

// ---- one class segment of the chunk ----------------------------------------------------------------------------------------
// r0 = stream-order index of the segment's first record (row of the table).  nv = the warp's direction, rv[j] = radius of point j.
template <int L, int NS>
__device__ __forceinline__ void run_class_sph(SPipe& pp, const SphArgs& a, const char* __restrict__ seg, long long r0, int n_rec,
                                              int rbox, int lane, double* Ww, const double (&nv)[3], const double (&rv)[kNQ],
                                              double (&re)[kNQ][NS], double (&im)[kNQ][NS])
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
        mbar_expect_tx(&pp.full[slot], (uint32_t)cnt * (REC + kEB));
        bulk_g2s(sb, seg + (size_t)first * REC, (uint32_t)cnt * REC, &pp.full[slot]);
        bulk_g2s(sb + kStageBytes, a.te + ((size_t)rbox * a.n_rows + r) * kSphBR, (uint32_t)cnt * kEB, &pp.full[slot]);
    };
    // per-class monomials: powers of this lane's radii; the direction's monomials for the pre-pass; q = r n for the degree blocks
    double rp[kNQ][(L >= 1 && L <= 3) ? L + 1 : 1];
    double dm[1][(L >= 1 && L <= 3) ? nherm(L) : 1];
    double qv[kNQ][4];
#pragma unroll
    for (int j = 0; j < kNQ; ++j) {
        qv[j][0] = rv[j] * nv[0]; qv[j][1] = rv[j] * nv[1]; qv[j][2] = rv[j] * nv[2]; qv[j][3] = 0.0;
    }
    if constexpr (L >= 1 && L <= 3) {
        double dv[kNQ][4];
#pragma unroll
        for (int j = 0; j < kNQ; ++j) { dv[j][0] = nv[0]; dv[j][1] = nv[1]; dv[j][2] = nv[2]; dv[j][3] = 0.0; }
        make_monomials<L, 1, 0>(dv, dm);
#pragma unroll
        for (int j = 0; j < kNQ; ++j) {
            rp[j][0] = 1.0;
#pragma unroll
            for (int n = 1; n <= L; ++n) rp[j][n] = n == 1 ? rv[j] : rp[j][n - 1] * rv[j];
        }
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
        const double* Es = reinterpret_cast<const double*>(sp + kStageBytes) + lane;
        // pre-pass, part 1: d_P = n . P, once per record (lane k: record k)
        double* Dw = Ww;
        double* Gw = Ww + kMaxRec;
        if (lane < cnt) {
            const double* hdr = reinterpret_cast<const double*>(sp + lane * REC);
            Dw[lane] = fma(nv[0], hdr[0], fma(nv[1], hdr[1], nv[2] * hdr[2]));
        }
        if constexpr (L == 0 || L >= 4) __syncwarp();
        // g = E(r) (cos(r d) + i sin(r d)) for this lane's points: gq = {gc, gs, gc r, gs r}
        auto factors = [&](int k, double (&gq)[4][kNQ]) {
            const double dP = Dw[k];
#pragma unroll
            for (int jj = 0; jj < kNQ; ++jj) {
                double sn, cs;
                sincos_fast(rv[jj] * dP, sn, cs);
                const double e = Es[k * kSphBR + 32 * jj];
                gq[0][jj] = e * cs;
                gq[1][jj] = e * sn;
                if constexpr (L >= 1 && L <= 3) {
                    gq[2][jj] = gq[0][jj] * rv[jj];
                    gq[3][jj] = gq[1][jj] * rv[jj];
                }
            }
        };
        if constexpr (L >= 4) {                         // degree blocks, both q-points together (ff_common.cuh)
#pragma unroll 1
            for (int k0 = 0; k0 < cnt; k0 += kBlkRec) {
                const int nb = min(kBlkRec, cnt - k0);
                double gcb[kBlkRec][kNQ], gsb[kBlkRec][kNQ];
                static_for<kBlkRec>([&](auto rc) {
                    constexpr int r = decltype(rc)::value;
                    if (r < nb) {
                        double gq[4][kNQ];
                        factors(k0 + r, gq);
#pragma unroll
                        for (int jj = 0; jj < kNQ; ++jj) { gcb[r][jj] = gq[0][jj]; gsb[r][jj] = gq[1][jj]; }
                    }
                });
                accum_blocks<L, NS>(sp + k0 * REC, nb, qv, gcb, gsb, re, im);
            }
        } else {
            if constexpr (L >= 1) {
                sph_prepass<L, NS>(sp, cnt, dm, Gw, lane);
                __syncwarp();
            }
            auto accum = [&](int k, const double (&gq)[4][kNQ]) {
                if constexpr (L == 0) {
                    double mono[kNQ][1];
#pragma unroll
                    for (int jj = 0; jj < kNQ; ++jj) mono[jj][0] = 1.0;
                    record_accum<0, NS, kNQ, 0>(reinterpret_cast<const double2*>(sp + k * REC), mono, gq[0], gq[1], re, im);
                } else {
                    record_accum_sph<L, NS>(reinterpret_cast<const double2*>(Gw + k * g_stride(L, NS)), rp, gq[0], gq[1], gq[2], gq[3], re, im);
                }
            };
            // software-pipelined by groups of U records: the sincos chains of group k+1 are issued alongside the accumulate of group k
            constexpr int U = L <= 1 ? 2 : 1;
            const int n_full = cnt / U * U;
            constexpr int NGQ = (L >= 1 && L <= 3) ? 4 : 2;       // components of gq that are live
            double gq[U][4][kNQ];
            if (n_full > 0) {
#pragma unroll
                for (int u = 0; u < U; ++u) factors(u, gq[u]);
#pragma unroll 1
                for (int k = 0; k + U < n_full; k += U) {
                    double gn[U][4][kNQ];
#pragma unroll
                    for (int u = 0; u < U; ++u) factors(k + U + u, gn[u]);
#pragma unroll
                    for (int u = 0; u < U; ++u) accum(k + u, gq[u]);
#pragma unroll
                    for (int u = 0; u < U; ++u)
#pragma unroll
                        for (int c = 0; c < NGQ; ++c)
#pragma unroll
                            for (int jj = 0; jj < kNQ; ++jj) gq[u][c][jj] = gn[u][c][jj];
                }
#pragma unroll
                for (int u = 0; u < U; ++u) accum(n_full - U + u, gq[u]);
            }
#pragma unroll 1
            for (int k = n_full; k < cnt; ++k) {
                factors(k, gq[0]);
                accum(k, gq[0]);
            }
        }
        __syncthreads();                                 // the slot and the warp areas are free again
        if (producer && j + kStages < n_st) issue(j + kStages);
    }
    pp.it += (uint32_t)n_st;
}

template <int NS>
__global__ void __launch_bounds__(kThreads, 2) ff_sph_kernel(const SphArgs a)
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
    SPipe pp = {smem, full_bar, 0u};
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double* Ww = reinterpret_cast<double*>(smem + kStages * kSlotBytes + 64 + warp * warp_bytes(NS));   // the warp's private area

    const int rbox = tile % a.n_rbox, dbox = tile / a.n_rbox;
    const int d = dbox * kSphBD + warp;                   // direction index j * n_phi + k
    const bool dir_ok = d < a.n_dir_eval;
    double nv[3], rv[kNQ];
#pragma unroll
    for (int c = 0; c < 3; ++c) nv[c] = dir_ok ? a.dirs[(size_t)d * 3 + c] : 0.0;
#pragma unroll
    for (int j = 0; j < kNQ; ++j) {
        const int i = rbox * kSphBR + lane + 32 * j;
        rv[j] = (dir_ok && i < a.n_r) ? a.r[i] : 0.0;
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
            if (dir_ok && rbox * kSphBR + lane + 32 * j < a.n_r) m2 = fmin(m2, rv[j] * rv[j]);     // |q| = |r| (n is a unit vector)
        plan_cta<NS>(a.v, chunk, m2, plan);
    }
#define SCARF_SPH_CLASS(LV)                                                                                          \
    if (plan.nrec[LV] > 0)                                                                                           \
        run_class_sph<LV, NS>(pp, a, a.v.base + plan.off[LV], plan.row[LV], plan.nrec[LV], rbox, lane, Ww, nv, rv, re, im);
    SCARF_SPH_CLASS(0)
    SCARF_SPH_CLASS(1)
    SCARF_SPH_CLASS(2)
    SCARF_SPH_CLASS(3)
    SCARF_SPH_CLASS(4)
    SCARF_SPH_CLASS(5)
    SCARF_SPH_CLASS(6)
#undef SCARF_SPH_CLASS

    // ---- epilogue: store (one chunk) or add into `out` in chunk order (several); the LAST chunk holds the final value and
    // also stores its conjugate at the mirror point when the grid is inversion-symmetric
    double2* dst = reinterpret_cast<double2*>(a.v.dst);
    double2* fin = a.v.dst_final != nullptr ? reinterpret_cast<double2*>(a.v.dst_final) : dst;    // finished values (last chunk)
    const int turn = plan.turn;
    if (turn < 0) return;                                   // a chunk without work (uniform over the CTA)
    const bool first = turn == 0, last = plan.next == 0;
    if (a.v.n_chunks > 1) ticket_wait(a.v.tickets + tile, turn);
    const long long n_dir = (long long)a.n_theta * a.n_phi;
    long long d_mirror = -1;
    if (a.sym && dir_ok) {
        const int jt = d / a.n_phi, kp = d - jt * a.n_phi;
        d_mirror = (long long)(a.n_theta - 1 - jt) * a.n_phi + (kp + a.n_phi / 2) % a.n_phi;
    }
#pragma unroll
    for (int j = 0; j < kNQ; ++j) {
        const int ir = rbox * kSphBR + lane + 32 * j;
        if (dir_ok && ir < a.n_r) {
            const long long i = (long long)ir * n_dir + d;
            const bool mirror = last && d_mirror >= 0;
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
                    if (mirror) w[(long long)ir * n_dir + d_mirror] = make_double2(v.x, -v.y);   // f(-q) = conj f(q)
                }
        }
    }
    if (a.v.n_chunks > 1) ticket_pass(a.v.tickets + tile, plan.next);
}

template <int NS>
cudaError_t launch_sph_ns(const SphArgs& a, cudaStream_t st)
{
    const dim3 grid((unsigned)a.v.n_tiles, (unsigned)a.v.n_chunks, 1);   // dispatched x fastest: chunk-major
    ff_sph_kernel<NS><<<grid, kThreads, smem_bytes<NS>(), st>>>(a);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_sph_table(const SphArgs& a, double* te, cudaStream_t st)
{
    const long long n = a.n_rows * (long long)a.n_rbox * kSphBR;
    if (n <= 0) return cudaSuccess;
    sph_table_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(a, te);
    return cudaGetLastError();
}

// The kernels need more than 48 KB of dynamic shared memory: an attribute of the function on the CURRENT device.  Called by
// scarf_create for the context's device (idempotent, no process-wide flag).
cudaError_t ff_sph_init_device()
{
    cudaError_t e = cudaSuccess;
#define SCARF_SPH_ATTR(NSV) \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(ff_sph_kernel<NSV>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes<NSV>());
    SCARF_SPH_ATTR(1) SCARF_SPH_ATTR(2) SCARF_SPH_ATTR(4) SCARF_SPH_ATTR(6) SCARF_SPH_ATTR(8) SCARF_SPH_ATTR(12)
#undef SCARF_SPH_ATTR
    return e;
}

cudaError_t launch_ff_sph(int NS, const SphArgs& a, cudaStream_t st)
{
    if (a.v.n_q <= 0 || a.v.n_chunks <= 0 || a.v.n_tiles <= 0) return cudaSuccess;
    switch (NS) {
    case 1: return launch_sph_ns<1>(a, st);
    case 2: return launch_sph_ns<2>(a, st);
    case 4: return launch_sph_ns<4>(a, st);
    case 6: return launch_sph_ns<6>(a, st);
    case 8: return launch_sph_ns<8>(a, st);
    case 12: return launch_sph_ns<12>(a, st);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace scarf

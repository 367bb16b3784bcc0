// ff_v1.cu — S4, the general-q hot kernel (Eq. (48)).
//
//   f_s(q) = sum_pairs e^{-q^2/4p} (cos q.P + i sin q.P) (A_s(q) + i B_s(q)),
//   A_s = sum_{n even} D^s_h q^h,  B_s = sum_{n odd} D^s_h q^h         (i^n folded into D by the fold kernel)
//
// Work decomposition.  The grid is n_tiles x n_chunks CTAs.  A tile is kTile = 2 x kThreads q-points (every
// thread keeps TWO q-points and all NS <= 12 states of both in registers: 4 NS FP64 accumulators), a chunk is a
// cost-balanced contiguous slice of the class-sorted pair stream (it may span classes; planned on the device,
// fold.cu: plan_chunks_kernel).  Chunks exist only to give the block scheduler enough equal-cost CTAs for an even
// last wave.  The n_chunks CTAs of one tile add their partial sums INTO `out` in chunk order (ff_common.cuh:
// ordered_fixup): chunk 0 stores, chunk k waits for the tile's ticket to reach k, adds and passes the ticket on —
// deterministic, no partial buffer in HBM and no second kernel (in round 1 the partials were 5 x the algorithmic
// bytes); the read-modify-write of a 48 KB tile goes through L2.  CTAs are dispatched in blockIdx order (chunk-major
// grid), so the CTA a ticket waits for is always already running.  (Measured alternative, not kept: the chunks of a
// tile as a thread-block cluster reducing through distributed shared memory — gang scheduling of 7-CTA clusters cost
// 30 % of the kernel time on config 3.)
//
// Operand delivery.  Every polynomial FMA needs its own warp-uniform coefficient.  The records of the chunk
// are staged through shared memory by 1-D TMA bulk copies (cp.async.bulk + mbarrier complete_tx), kStages
// deep, issued by one thread; all threads then read them with broadcast LDS.128 (two coefficients per load,
// each used for both q-points of the thread => 4 DFMA per LDS.128).  All loops over (state, Hermite index) are
// unrolled at compile time from the class L, so monomials and accumulators are plain registers.
//
// FP64 budget per (q, pair): 4 (arguments) + 15 (e^{-x}) + 19 (sincos) + 2 = 40 issue slots, and per
// (q, pair, state) n_herm + 3 (2 for L = 0) — the work model of DESIGN.md.
#include "ff_common.cuh"

#include <mutex>

// Scratch of the allocation-free entry point (scarf_form_factors_noalloc, include/scarf.h): the per-tile tickets of the
// ordered fix-up, one int per q tile.  256 KB on every device that loads the library, until the process exits.  In HOST code
// this name is only a stand-in for the symbol: the device address comes from cudaGetSymbolAddress (static_tickets() below).
constexpr int kStaticTickets = 65536;        // == SCARF_NOALLOC_MAX_TILES (checked in scarf_api.cu)
static __device__ __align__(256) int scarf_static_tickets[kStaticTickets];

namespace scarf {

namespace {

constexpr int kThreads = 128;
constexpr int kTile = kThreads * kNQ;        // q-points per CTA
constexpr int kStages = 3;
constexpr int kStageBytes = 8192;            // >= the largest record (L = 6, NS = 12: 8096 B)
constexpr int kSwpMaxL = 2;                  // classes whose record loop is software-pipelined
// records whose transcendentals are in flight together in the pipelined loop: two for the short bodies of L <= 1
// (measured on the B200: L = 0 74.4 -> 78.1 %, L = 1 76.8 -> 78.1 % of the DFMA peak; L = 2 loses registers to it)
__host__ __device__ constexpr int swp_records(int L) { return L <= 1 ? 2 : 1; }


struct Pipe {               // stage ring shared by all class segments of the CTA
    unsigned char* buf;     // kStages x kStageBytes
    uint64_t* full;         // kStages mbarriers
    uint32_t it;            // stages consumed so far (all threads keep the same count)
};

// ---- one class segment of the chunk: stream its records through the stage ring ---------------------------
template <int L, int NS>
__device__ __forceinline__ void run_class(Pipe& pp, const char* __restrict__ seg, int n_rec, const double (&qv)[kNQ][4],
                                          double (&re)[kNQ][NS], double (&im)[kNQ][NS])
{
    constexpr int REC = rec_doubles(L, NS) * 8;
    constexpr int SREC = kStageBytes / REC;              // records per stage (>= 1)
    static_assert(SREC >= 1, "record larger than a stage");
    constexpr int NQA = L <= 3 ? kNQ : 1;                // q-points evaluated together (register budget)
    const int n_st = (n_rec + SREC - 1) / SREC;
    const bool producer = threadIdx.x == 0;
    auto issue = [&](int j) {                            // stage j of this segment into ring slot (it0 + j) % kStages
        const int slot = (int)((pp.it + (uint32_t)j) % kStages);
        const int first = j * SREC, cnt = min(SREC, n_rec - first);
        const uint32_t bytes = (uint32_t)cnt * REC;
        SCARF_CHECK(cnt >= 1 && bytes <= (uint32_t)kStageBytes && (bytes & 15u) == 0 && slot >= 0 && slot < kStages);
        mbar_expect_tx(&pp.full[slot], bytes);
        bulk_g2s(pp.buf + slot * kStageBytes, seg + (size_t)first * REC, bytes, &pp.full[slot]);
    };
    // all threads have left the previous segment's stages
    __syncthreads();
    if (producer)
        for (int j = 0; j < min(kStages, n_st); ++j) issue(j);
    // `pp.it` is only advanced after the loop so that issue() sees the segment's base
    for (int j = 0; j < n_st; ++j) {
        const uint32_t g = pp.it + (uint32_t)j;
        const int slot = (int)(g % kStages);
        mbar_wait(&pp.full[slot], (g / kStages) & 1u);
        const int cnt = min(SREC, n_rec - j * SREC);
        const unsigned char* sp = pp.buf + slot * kStageBytes;
        if constexpr (L >= 4) {                         // degree blocks, both q-points together (ff_common.cuh)
#pragma unroll 1
            for (int k0 = 0; k0 < cnt; k0 += kBlkRec) {
                const int nb = min(kBlkRec, cnt - k0);
                double gcb[kBlkRec][kNQ], gsb[kBlkRec][kNQ];
                static_for<kBlkRec>([&](auto rc) {
                    constexpr int r = decltype(rc)::value;
                    if (r < nb) record_trans<kNQ, 0>(reinterpret_cast<const double2*>(sp + (k0 + r) * REC), qv, gcb[r], gsb[r]);
                });
                accum_blocks<L, NS>(sp + k0 * REC, nb, qv, gcb, gsb, re, im);
            }
        } else
        static_for<kNQ / NQA>([&](auto jc) {
            constexpr int jq0 = decltype(jc)::value * NQA;
            double mono[NQA][nherm(L)];
            make_monomials<L, NQA, jq0>(qv, mono);
            auto rec = [&](int k) { return reinterpret_cast<const double2*>(sp + k * REC); };
            if constexpr (L <= kSwpMaxL) {               // software-pipelined: trans(group k+1) alongside accum(group k)
                constexpr int U = swp_records(L);
                const int n_full = cnt / U * U;
                double gc[U][NQA], gs[U][NQA];
                if (n_full > 0) {
#pragma unroll
                    for (int u = 0; u < U; ++u) record_trans<NQA, jq0>(rec(u), qv, gc[u], gs[u]);
#pragma unroll 1
                    for (int k = 0; k + U < n_full; k += U) {
                        double gcn[U][NQA], gsn[U][NQA];
#pragma unroll
                        for (int u = 0; u < U; ++u) record_trans<NQA, jq0>(rec(k + U + u), qv, gcn[u], gsn[u]);
#pragma unroll
                        for (int u = 0; u < U; ++u) record_accum<L, NS, NQA, jq0>(rec(k + u), mono, gc[u], gs[u], re, im);
#pragma unroll
                        for (int u = 0; u < U; ++u)
#pragma unroll
                            for (int jj = 0; jj < NQA; ++jj) { gc[u][jj] = gcn[u][jj]; gs[u][jj] = gsn[u][jj]; }
                    }
#pragma unroll
                    for (int u = 0; u < U; ++u) record_accum<L, NS, NQA, jq0>(rec(n_full - U + u), mono, gc[u], gs[u], re, im);
                }
#pragma unroll 1
                for (int k = n_full; k < cnt; ++k) {     // fewer than U records left over
                    record_trans<NQA, jq0>(rec(k), qv, gc[0], gs[0]);
                    record_accum<L, NS, NQA, jq0>(rec(k), mono, gc[0], gs[0], re, im);
                }
            } else {
                double gc[NQA], gs[NQA];
#pragma unroll 1
                for (int k = 0; k < cnt; ++k) {
                    record_trans<NQA, jq0>(rec(k), qv, gc, gs);
                    record_accum<L, NS, NQA, jq0>(rec(k), mono, gc, gs, re, im);
                }
            }
        });
        __syncthreads();                                 // the slot is free again
        if (producer && j + kStages < n_st) issue(j + kStages);
    }
    pp.it += (uint32_t)n_st;
}

template <int NS>
__global__ void __launch_bounds__(kThreads, 2) ff_v1_kernel(const V1Args a)
{
    __shared__ __align__(128) unsigned char smem[kStages * kStageBytes];
    __shared__ __align__(8) uint64_t full_bar[kStages];
    const int tile = (int)blockIdx.x, chunk = (int)blockIdx.y;
    if (threadIdx.x == 0) {
        for (int s = 0; s < kStages; ++s) mbar_init(&full_bar[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    Pipe pp = {smem, full_bar, 0u};

    double qv[kNQ][4];
    long long iq[kNQ];
#pragma unroll
    for (int j = 0; j < kNQ; ++j) {
        iq[j] = (long long)tile * kTile + j * kThreads + threadIdx.x;
        const bool ok = iq[j] < a.n_q;
        qv[j][0] = ok ? a.q[3 * iq[j]] : 0.0;
        qv[j][1] = ok ? a.q[3 * iq[j] + 1] : 0.0;
        qv[j][2] = ok ? a.q[3 * iq[j] + 2] : 0.0;
        qv[j][3] = qv[j][0] * qv[j][0] + qv[j][1] * qv[j][1] + qv[j][2] * qv[j][2];
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
            if (iq[j] < a.n_q) m2 = fmin(m2, qv[j][3]);
        plan_cta<NS>(a, chunk, m2, plan);
    }
#define SCARF_V1_CLASS(LV) \
    if (plan.nrec[LV] > 0) run_class<LV, NS>(pp, a.base + plan.off[LV], plan.nrec[LV], qv, re, im);
    SCARF_V1_CLASS(0)
    SCARF_V1_CLASS(1)
    SCARF_V1_CLASS(2)
    SCARF_V1_CLASS(3)
    SCARF_V1_CLASS(4)
    SCARF_V1_CLASS(5)
    SCARF_V1_CLASS(6)
#undef SCARF_V1_CLASS

    // ---- epilogue: store (one chunk) or add into `out` in chunk order (several) ------------------------------------------
    double2* dst = reinterpret_cast<double2*>(a.dst);
    const int turn = plan.turn;
    if (turn < 0) return;                                   // a chunk without work (uniform over the CTA)
    const bool first = turn == 0;
    if (a.n_chunks > 1) ticket_wait(a.tickets + tile, turn);
#pragma unroll
    for (int j = 0; j < kNQ; ++j)
        if (iq[j] < a.n_q)
#pragma unroll
            for (int s = 0; s < NS; ++s)
                if (s < a.ns_real) {
                    double2* o = dst + (size_t)s * a.n_q + iq[j];
                    double2 v = make_double2(re[j][s], im[j][s]);
                    if (!first) {
                        const double2 p = __ldcg(o);      // written by another SM: read through L2
                        v.x += p.x;
                        v.y += p.y;
                    }
                    *o = v;
                }
    if (a.n_chunks > 1) ticket_pass(a.tickets + tile, plan.next);
}

}  // namespace

int v1_tile_q() { return kTile; }

cudaError_t launch_ff_v1(int NS, const V1Args& a, cudaStream_t st)
{
    if (a.n_q <= 0 || a.n_chunks <= 0) return cudaSuccess;
    const dim3 grid((unsigned)a.n_tiles, (unsigned)a.n_chunks, 1);    // dispatched x fastest: chunk-major
    switch (NS) {
    case 1: ff_v1_kernel<1><<<grid, kThreads, 0, st>>>(a); break;
    case 2: ff_v1_kernel<2><<<grid, kThreads, 0, st>>>(a); break;
    case 4: ff_v1_kernel<4><<<grid, kThreads, 0, st>>>(a); break;
    case 6: ff_v1_kernel<6><<<grid, kThreads, 0, st>>>(a); break;
    case 8: ff_v1_kernel<8><<<grid, kThreads, 0, st>>>(a); break;
    case 12: ff_v1_kernel<12><<<grid, kThreads, 0, st>>>(a); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

// ---- allocation-free variant: tickets in the static device array ---------------------------------------------------------
int v1_static_tiles() { return kStaticTickets; }

// Device address of scarf_static_tickets on the CURRENT device; resolved once per device (the address of a __device__ symbol
// differs from device to device, and the host-side name is not a device pointer).
static cudaError_t static_tickets(int** out)
{
    constexpr int kMaxDevices = 64;
    static std::mutex mu;
    static int* addr[kMaxDevices] = {};
    *out = nullptr;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (addr[dev] == nullptr) {
        int* p = nullptr;
        e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), scarf_static_tickets);
        if (e != cudaSuccess) return e;
        if (p == nullptr) return cudaErrorInvalidSymbol;
        addr[dev] = p;
    }
    *out = addr[dev];
    return cudaSuccess;
}

cudaError_t ff_v1_static_setup() { int* p; return static_tickets(&p); }

// Same kernel, same launch geometry as launch_ff_v1; a.tickets is ignored and replaced by the static array, whose first
// n_tiles entries are cleared on `st` first.  No allocation.  n_tiles beyond the array: cudaErrorInvalidValue (the C-ABI
// entry point checks the size before it gets here and reports the limit).
cudaError_t launch_ff_v1_static(int NS, V1Args a, cudaStream_t st)
{
    if (a.n_q <= 0 || a.n_chunks <= 0) return cudaSuccess;
    if (a.n_tiles > kStaticTickets) return cudaErrorInvalidValue;
    a.tickets = nullptr;
    if (a.n_chunks > 1) {
        int* t = nullptr;
        cudaError_t e = static_tickets(&t);
        if (e != cudaSuccess) return e;
        e = cudaMemsetAsync(t, 0, (size_t)a.n_tiles * sizeof(int), st);
        if (e != cudaSuccess) return e;
        a.tickets = t;
    }
    return launch_ff_v1(NS, a, st);
}

}  // namespace scarf

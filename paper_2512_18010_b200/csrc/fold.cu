// fold.cu — S3 of SURVEY.md §8(a): fold the transition matrices T^s into per-primitive-pair Hermite
// coefficients (the paper's T M D product, Eq. (48)-(49) PAPER.md:326-334), compute the screening bound,
// and pack the kept records.  Also the FP64 peak micro-benchmark.
#include <algorithm>

#include "kernels.cuh"

#ifdef SCARF_DEBUG_CHECKS
#define SCARF_CHECK(cond) do { if (!(cond)) __trap(); } while (0)
#else
#define SCARF_CHECK(cond) ((void)0)
#endif

namespace scarf {

// Index tables in the constant bank, initialised at compile time (no per-process upload step, no mutable global state):
//   herm[h] = (t,u,v,n) of Hermite index h;  comp[l][c] = (a,b,c, (2a-1)!!(2b-1)!!(2c-1)!! ) of component c of shell l.
struct IndexTables {
    unsigned char herm[kMaxHerm][4];
    unsigned short comp[kMaxL + 1][kMaxCart][4];
};
constexpr IndexTables make_index_tables()
{
    IndexTables t{};
    int h = 0;
    for (int n = 0; n <= kMaxClass; ++n)
        for (int a = n; a >= 0; --a)
            for (int b = n - a; b >= 0; --b) {
                t.herm[h][0] = (unsigned char)a; t.herm[h][1] = (unsigned char)b;
                t.herm[h][2] = (unsigned char)(n - a - b); t.herm[h][3] = (unsigned char)n;
                ++h;
            }
    for (int l = 0; l <= kMaxL; ++l) {
        int c = 0;
        for (int a = l; a >= 0; --a)
            for (int b = l - a; b >= 0; --b) {
                const int e[3] = {a, b, l - a - b};
                int df = 1;                                  // (2a-1)!!(2b-1)!!(2c-1)!! <= 11!! = 10395 for l <= 6
                for (int k = 0; k < 3; ++k)
                    for (int j = 2 * e[k] - 1; j > 1; j -= 2) df *= j;
                t.comp[l][c][0] = (unsigned short)a; t.comp[l][c][1] = (unsigned short)b;
                t.comp[l][c][2] = (unsigned short)(l - a - b); t.comp[l][c][3] = (unsigned short)df;
                ++c;
            }
    }
    return t;
}
__constant__ IndexTables c_tab = make_index_tables();

// One warp per primitive shell pair; lanes stride over the Hermite index h.
//   D^s_h = g * scale * sign(n) * sum_{ca,cb} f_ca f_cb (T^s[mu][nu] + T^s[nu][mu]) Ex[a][a'][t] Ey[b][b'][u] Ez[c][c'][v]
// and the bound B_P = max_s sum_h |D^s_h| (2 p n / e)^{n/2}  (sup over q of |q|^n e^{-q^2/4p}; 1 for n = 0).
__global__ void __launch_bounds__(128) fold_kernel(const FoldArgs a)
{
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (warp >= a.n_pairs) return;
    const PairMeta m = a.pairs[warp];
    const int la = m.la, lb = m.lb, L = m.L, nt = L + 1, nh = nherm(L);
    const int blk = (la + 1) * (lb + 1) * nt;
    const double* __restrict__ Ex = a.E + m.e_off;
    const double* __restrict__ Ey = Ex + blk;
    const double* __restrict__ Ez = Ey + blk;
    double* rec = reinterpret_cast<double*>(a.staging + a.cls_off[L] + (unsigned long long)(warp - a.class_first[L]) * a.rec_bytes[L]);
    if (lane == 0) {
        rec[0] = m.Px; rec[1] = m.Py; rec[2] = m.Pz; rec[3] = m.inv4p;
        if ((a.NS * nh) & 1) rec[4 + a.NS * nh] = 0.0;
    }
    const size_t nbf = (size_t)a.nbf;
    const double* __restrict__ T = a.T + (size_t)a.s0 * nbf * nbf;
    double bsum[kMaxStateTile];
#pragma unroll
    for (int s = 0; s < kMaxStateTile; ++s) bsum[s] = 0.0;
    const int nca = ncart(la), ncb = ncart(lb);
    for (int h = lane; h < nh; h += 32) {
        const int t = c_tab.herm[h][0], u = c_tab.herm[h][1], v = c_tab.herm[h][2], n = c_tab.herm[h][3];
        double acc[kMaxStateTile];
#pragma unroll
        for (int s = 0; s < kMaxStateTile; ++s) acc[s] = 0.0;
        for (int ca = 0; ca < nca; ++ca) {
            const int a1 = c_tab.comp[la][ca][0], b1 = c_tab.comp[la][ca][1], c1 = c_tab.comp[la][ca][2];
            const double fa = 1.0 / sqrt((double)c_tab.comp[la][ca][3]);   // = component_factor(la, ca) of the host code, bit for bit
            for (int cb = 0; cb < ncb; ++cb) {
                const int a2 = c_tab.comp[lb][cb][0], b2 = c_tab.comp[lb][cb][1], c2 = c_tab.comp[lb][cb][2];
                if (t > a1 + a2 || u > b1 + b2 || v > c1 + c2) continue;
                const double G = fa * (1.0 / sqrt((double)c_tab.comp[lb][cb][3])) * Ex[(a1 * (lb + 1) + a2) * nt + t] *
                                 Ey[(b1 * (lb + 1) + b2) * nt + u] * Ez[(c1 * (lb + 1) + c2) * nt + v];
                const size_t mu = (size_t)(m.bf0a + ca), nu = (size_t)(m.bf0b + cb);
                const double* t1 = T + mu * nbf + nu;
                const double* t2 = T + nu * nbf + mu;
#pragma unroll
                for (int s = 0; s < kMaxStateTile; ++s)
                    if (s < a.ns_real) acc[s] += G * (t1[(size_t)s * nbf * nbf] + t2[(size_t)s * nbf * nbf]);
            }
        }
        const double sign = ((n >> 1) & 1) ? -1.0 : 1.0;
        const double mn = n == 0 ? 1.0 : pow(2.0 * m.p * n * 0.36787944117144233, 0.5 * n);
        const double f = a.g * m.scale * sign;
#pragma unroll
        for (int s = 0; s < kMaxStateTile; ++s)
            if (s < a.NS) {
                const double D = s < a.ns_real ? f * acc[s] : 0.0;
                rec[4 + s * nh + h] = D;
                bsum[s] += fabs(D) * mn;
            }
    }
    double b = 0.0;
    bool bad = false;                                     // fmax drops NaN: keep a non-finite bound (non-finite T) sticky
#pragma unroll
    for (int s = 0; s < kMaxStateTile; ++s) {
        double x = bsum[s];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        bad = bad || !(x <= 1.7976931348623157e308);
        b = fmax(b, x);
    }
    if (lane == 0) {
        const double prev = a.first_tile ? 0.0 : a.bound[warp];
        a.bound[warp] = (bad || !(prev <= 1.7976931348623157e308)) ? __longlong_as_double(0x7ff8000000000000LL) : fmax(prev, b);
    }
}

cudaError_t launch_fold(const FoldArgs& a, cudaStream_t st)
{
    if (a.n_pairs <= 0) return cudaSuccess;
    const int threads = 128;
    const long long blocks = (a.n_pairs * 32 + threads - 1) / threads;
    fold_kernel<<<(unsigned)blocks, threads, 0, st>>>(a);
    return cudaGetLastError();
}

// ---- screening on the device -----------------------------------------------------------------------------------------
// One CTA.  Pass 1: sum, max and finiteness of the bounds (fixed-order tree: deterministic).  Threshold (DESIGN.md
// reading #12):  thr = max(screen_tol * mean(B), threshold_eps * max(B));  a pair is kept iff B > 0 and B >= thr.
// Pass 2: stable compaction of the kept indices (block scan over consecutive 1024-element windows, so the stream keeps
// the host's class-sorted (i, j) order), kept counts per class, sum of the dropped bounds.
constexpr int kScreenThreads = 1024;

__device__ __forceinline__ double block_reduce(double v, double* sh, bool take_max)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double w = __shfl_xor_sync(0xffffffffu, v, o);
        v = take_max ? fmax(v, w) : v + w;
    }
    __syncthreads();
    if (lane == 0) sh[warp] = v;
    __syncthreads();
    if (warp == 0) {
        v = lane < kScreenThreads / 32 ? sh[lane] : (take_max ? 0.0 : 0.0);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double w = __shfl_xor_sync(0xffffffffu, v, o);
            v = take_max ? fmax(v, w) : v + w;
        }
        if (lane == 0) sh[0] = v;
    }
    __syncthreads();
    return sh[0];
}

__global__ void __launch_bounds__(kScreenThreads) screen_kernel(const ScreenArgs a)
{
    __shared__ double sh[kScreenThreads / 32];
    __shared__ int sh_scan[kScreenThreads / 32];
    __shared__ int sh_bad;
    __shared__ int sh_cls[kNClasses];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) sh_bad = 0;
    if (tid < kNClasses) sh_cls[tid] = 0;
    double sum = 0.0, mx = 0.0;
    bool bad = false;
    for (long long i = tid; i < a.n_pairs; i += kScreenThreads) {
        const double b = a.bound[i];
        bad = bad || !isfinite(b);
        sum += b;
        mx = fmax(mx, b);
    }
    __syncthreads();
    if (bad) sh_bad = 1;
    const double sumB = block_reduce(sum, sh, false);
    const double maxB = block_reduce(mx, sh, true);
    const bool any_bad = sh_bad != 0;
    // a non-finite bound means a non-finite T: keep everything so that the NaN reaches the output instead of silent zeros
    const double thr = any_bad ? 0.0 : fmax(a.n_pairs > 0 ? a.screen_tol * sumB / (double)a.n_pairs : 0.0, a.threshold_eps * maxB);
    double dropped = 0.0;
    long long base = 0;
    for (long long w0 = 0; w0 < a.n_pairs; w0 += kScreenThreads) {
        const long long i = w0 + tid;
        bool keep = false;
        if (i < a.n_pairs) {
            const double b = a.bound[i];
            keep = any_bad || (b > 0.0 && b >= thr);
            if (!keep) dropped += b;
        }
        const unsigned m = __ballot_sync(0xffffffffu, keep);
        const int in_warp = __popc(m & ((1u << lane) - 1u));
        if (lane == 0) sh_scan[warp] = __popc(m);
        __syncthreads();
        int before = 0, total = 0;
#pragma unroll 1
        for (int k = 0; k < kScreenThreads / 32; ++k) {
            const int c = sh_scan[k];
            if (k < warp) before += c;
            total += c;
        }
        int c = -1;
        if (keep) {
            a.keep_idx[base + before + in_warp] = (int)i;
            c = 0;
#pragma unroll
            for (int k = 1; k < kNClasses; ++k)
                if (i >= a.class_first[k]) c = k;
        }
        // kept counts per class: warp-aggregated (a window usually lies in ONE class: per-thread atomics on one shared
        // word serialise 1024 ways — 0.33 ms measured); integer counts, so the order of the adds does not matter
#pragma unroll
        for (int k = 0; k < kNClasses; ++k) {
            const int n = __popc(__ballot_sync(0xffffffffu, c == k));
            if (lane == 0 && n > 0) atomicAdd(&sh_cls[k], n);
        }
        base += total;
        __syncthreads();
    }
    const double droppedB = block_reduce(dropped, sh, false);
    if (tid == 0) {
        ScreenResult r = {};
        r.n_kept = base;
        for (int c = 0; c < kNClasses; ++c) r.kept_per_class[c] = sh_cls[c];
        r.sum_bound = sumB; r.max_bound = maxB; r.dropped_bound = any_bad ? 0.0 : droppedB;
        r.bad = any_bad ? 1 : 0;
        *a.result = r;
    }
}

cudaError_t launch_screen(const ScreenArgs& a, cudaStream_t st)
{
    screen_kernel<<<1, kScreenThreads, 0, st>>>(a);
    return cudaGetLastError();
}

// One warp per kept record: copy it from the staging layout to its packed position (16-byte pieces).  Every warp derives
// the packed layout from the screening result (13-term prefix sums); block 0 also writes the tile's StreamDesc.
__global__ void __launch_bounds__(128) pack_kernel(const PackArgs a)
{
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    const ScreenResult& r = *a.result;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        StreamDesc& d = *a.desc;
        long long first = 0;
        unsigned long long off = 0;
        for (int c = 0; c < kNClasses; ++c) {
            d.cls_n[c] = r.kept_per_class[c];
            d.cls_first[c] = first;
            d.cls_off[c] = off;
            d.rec_bytes[c] = a.rec_bytes[c];
            first += r.kept_per_class[c];
            off += (unsigned long long)r.kept_per_class[c] * a.rec_bytes[c];
        }
        d.cls_first[kNClasses] = first;
        d.n_kept = r.n_kept;
        d.n_chunks = 0;
    }
    if (warp >= r.n_kept) return;
    const long long i = a.keep_idx[warp];
    int c = 0;
#pragma unroll
    for (int k = 1; k < kNClasses; ++k)
        if (i >= a.class_first[k]) c = k;
    long long kfirst = 0;
    unsigned long long doff = 0;
    for (int k = 0; k < c; ++k) {
        kfirst += r.kept_per_class[k];
        doff += (unsigned long long)r.kept_per_class[k] * a.rec_bytes[k];
    }
    SCARF_CHECK(i >= a.class_first[c] && i < a.class_first[c + 1] && warp >= kfirst && warp < kfirst + r.kept_per_class[c]);
    const uint4* s = reinterpret_cast<const uint4*>(a.staging + a.cls_off[c] + (unsigned long long)(i - a.class_first[c]) * a.rec_bytes[c]);
    uint4* d = reinterpret_cast<uint4*>(a.packed + doff + (unsigned long long)(warp - kfirst) * a.rec_bytes[c]);
    const int pieces = a.rec_bytes[c] >> 4;
    for (int k = lane; k < pieces; k += 32) d[k] = s[k];
}

cudaError_t launch_pack(const PackArgs& a, cudaStream_t st)
{
    const int threads = 128;
    const long long blocks = std::max<long long>(1, (a.n_pairs * 32 + threads - 1) / threads);   // sized for "everything kept"
    pack_kernel<<<(unsigned)blocks, threads, 0, st>>>(a);
    return cudaGetLastError();
}

// ---- q-adaptive cut-off (NEXT-2, second half; PAPER.md:499 thresholding made q-dependent) ----------------------------------
// A kept pair contributes  |term_P(q)| <= e^{-q^2/4p} sum_n c_n |q|^n,  c_n = sum_{deg h = n} max_s |D^s_h|.  The envelope
//   U_P(q) = sum_n c_n sup_{q' >= q} q'^n e^{-q'^2/4p}      (each term: its value at q beyond its peak sqrt(2 p n), else the peak)
// is non-increasing, so q_cut(P) = inf{q : U_P(q) < tau} is well defined and the pair can be skipped for every q-point with
// |q| >= q_cut at a cost of < tau each.  Records are then sorted by q_cut (descending, stable) inside their class, so that a
// q tile whose smallest |q| is q_min evaluates a PREFIX of every class: records with q_cut > q_min.  Error per (q, state):
// < (number of skipped records) * tau <= n_kept * tau, reported as scarf_stats.adaptive_bound.
__device__ double envelope(const double* c, int L, double p, double q)
{
    double u = c[0] * exp(-q * q / (4.0 * p));
    for (int n = 1; n <= L; ++n) {
        const double qs = sqrt(2.0 * p * n), qq = q > qs ? q : qs;       // beyond the peak: the value; before it: the peak
        u += c[n] * pow(qq, (double)n) * exp(-qq * qq / (4.0 * p));
    }
    return u;
}

// one thread per kept record
__global__ void __launch_bounds__(128) qcut_kernel(const AdaptArgs a)
{
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const ScreenResult& r = *a.result;
    if (k >= r.n_kept) return;
    const long long i = a.keep_idx[k];
    int c = 0;
#pragma unroll
    for (int j = 1; j < kNClasses; ++j)
        if (i >= a.class_first[j]) c = j;
    if (c > kFastMaxClass || r.bad) { a.key[k] = 1e300; return; }        // high classes are never cut
    double cn[kFastMaxClass + 1];
#pragma unroll
    for (int n = 0; n <= kFastMaxClass; ++n) cn[n] = 0.0;
    const int nh = nherm(c);
    double p = 1.0;
    for (int h = 0; h < nh; ++h) {
        double m = 0.0;
        for (int t = 0; t < a.n_tiles; ++t) {
            const double* rec = reinterpret_cast<const double*>(a.staging[t] + a.cls_off[t][c] + (unsigned long long)(i - a.class_first[c]) * a.rec_bytes[t][c]);
            if (h == 0 && t == 0) p = 0.25 / rec[3];
            for (int s = 0; s < a.NS[t]; ++s) m = fmax(m, fabs(rec[4 + s * nh + h]));
        }
        const int n = c_tab.herm[h][3];
#pragma unroll
        for (int j = 0; j <= kFastMaxClass; ++j)
            if (j == n) cn[j] += m;
    }
    const double tau = a.adaptive_tol * r.sum_bound / (double)(a.n_pairs > 0 ? a.n_pairs : 1);
    double lo = 0.0, hi = 1e4;
    if (!(envelope(cn, c, p, lo) >= tau)) { a.key[k] = 0.0; return; }    // below tau everywhere
    if (envelope(cn, c, p, hi) >= tau) { a.key[k] = 1e300; return; }     // never below tau in any sane range
    for (int it = 0; it < 64; ++it) {
        const double mid = 0.5 * (lo + hi);
        if (envelope(cn, c, p, mid) >= tau) lo = mid; else hi = mid;
    }
    a.key[k] = hi;                                                       // U(q) < tau for every q >= hi
}

// stable rank sort inside each class: position = first kept index of the class + #{j : key_j > key_k or (== and j < k)}
__global__ void __launch_bounds__(128) qcut_rank_kernel(const AdaptArgs a)
{
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const ScreenResult& r = *a.result;
    if (k >= r.n_kept) return;
    long long first = 0;
    int c = 0;
    for (; c < kNClasses; ++c) {
        if (k < first + r.kept_per_class[c]) break;
        first += r.kept_per_class[c];
    }
    const long long last = first + r.kept_per_class[c];
    const double key = a.key[k];
    long long rank = 0;
    for (long long j = first; j < last; ++j) {
        const double kj = a.key[j];
        rank += (kj > key || (kj == key && j < k)) ? 1 : 0;
    }
    a.keep_sorted[first + rank] = a.keep_idx[k];
    a.qcut_sorted[first + rank] = key;
}

cudaError_t launch_adaptive_sort(const AdaptArgs& a, cudaStream_t st)
{
    if (a.n_pairs <= 0) return cudaSuccess;
    const unsigned blocks = (unsigned)((a.n_pairs + 127) / 128);
    qcut_kernel<<<blocks, 128, 0, st>>>(a);
    qcut_rank_kernel<<<blocks, 128, 0, st>>>(a);
    return cudaGetLastError();
}

// ---- chunk planning on the device ------------------------------------------------------------------------------------
// Split the fast classes of the class-sorted stream into exactly K chunks of (nearly) equal modelled cost
// (w(c) = ns_real W(c) + ctr FP64 issue slots per record and q-point); a chunk may span classes; trailing chunks may be
// empty when there are fewer records than chunks.  One thread: <= K + 7 loop trips.
__global__ void plan_chunks_kernel(StreamDesc* d, int K, int ns_real, double ctr, int model)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    // slots per (q, pair, state): n_herm + 3; the product-grid kernel shares the (q_y, q_z) part between its two points
    // and the row kernel the (q_x, q_y) part between the 64 points of a warp
    const double kWl[kFastMaxClass + 1] = {2, 7, 13, 23, 38, 59, 87}, kWg[kFastMaxClass + 1] = {2, 6, 10.5, 17, 38, 59, 87},
                 kWr[kFastMaxClass + 1] = {2, 5.03, 7.11, 9.25, 38, 59, 87}, kWs[kFastMaxClass + 1] = {2, 4.05, 5.14, 6.3, 38, 59, 87};
    const double kWz[kFastMaxClass + 1] = {2, 4.22, 5.36, 6.56, 38, 59, 87};
    const double* kW = model == 4 ? kWz : (model == 3 ? kWs : (model == 2 ? kWr : (model == 1 ? kWg : kWl)));
    double w[kFastMaxClass + 1], total = 0.0;
    for (int c = 0; c <= kFastMaxClass; ++c) {
        w[c] = (double)ns_real * kW[c] + ctr;
        total += (double)d->cls_n[c] * w[c];
    }
    for (int k = 0; k < kMaxChunks; ++k)
        for (int c = 0; c < kNClasses; ++c) d->chunks[k].begin[c] = d->chunks[k].n[c] = 0;
    d->n_chunks = K;
    int k = 0;
    double acc = 0.0;
    bool cur_empty = true;
    for (int c = 0; c <= kFastMaxClass; ++c) {
        long long rem = d->cls_n[c], pos = 0;
        SCARF_CHECK(rem >= 0 && rem < 0x7fffffffLL);
        while (rem > 0) {
            long long take = rem;
            if (k < K - 1) {
                const double need = total * (double)(k + 1) / (double)K - acc;
                take = min(rem, (long long)llrint(need / w[c]));
                if (take <= 0) {
                    if (cur_empty) take = 1;
                    else { ++k; cur_empty = true; continue; }
                }
            }
            d->chunks[k].begin[c] = (int)pos;
            d->chunks[k].n[c] = (int)take;
            cur_empty = false;
            acc += (double)take * w[c];
            pos += take; rem -= take;
            if (k < K - 1 && acc >= total * (double)(k + 1) / (double)K - 0.5 * w[c]) { ++k; cur_empty = true; }
        }
    }
#ifdef SCARF_DEBUG_CHECKS
    for (int c = 0; c <= kFastMaxClass; ++c) {            // the chunks tile every class exactly once, in order
        long long pos = 0;
        for (int kk = 0; kk < K; ++kk)
            if (d->chunks[kk].n[c] > 0) { SCARF_CHECK(d->chunks[kk].begin[c] == pos); pos += d->chunks[kk].n[c]; }
        SCARF_CHECK(pos == d->cls_n[c]);
    }
#endif
}

cudaError_t launch_plan_chunks(StreamDesc* desc, int K, int ns_real, double ctr, cudaStream_t st, int model)
{
    plan_chunks_kernel<<<1, 32, 0, st>>>(desc, K, ns_real, ctr, model);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------
// FP64 issue-rate micro-benchmark: 8 independent DFMA chains per thread, registers only.
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dfma_peak_kernel(double* sink, int iters, long long* cycles)
{
    double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double m = 1.0000000001, c = 1e-12;
    unsigned long long g0, g1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
    const long long t0 = clock64();
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
            a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
        }
    }
    const long long t1 = clock64();
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
    const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (s == 123.456) sink[0] = s;
    // SM clock = this block's cycle count over the wall time (ns) it spans, whatever share of the kernel that is
    if (threadIdx.x == 0 && blockIdx.x == 0) { cycles[0] = t1 - t0; cycles[1] = (long long)(g1 - g0); }
}

cudaError_t run_fp64_peak(double* dfma_per_s, double* sm_clock_mhz)
{
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    double* sink = nullptr;
    long long* cyc = nullptr;
    if ((e = cudaMalloc(&sink, 8)) != cudaSuccess) return e;
    if ((e = cudaMalloc(&cyc, 16)) != cudaSuccess) { cudaFree(sink); return e; }
    cudaEvent_t ev0, ev1;
    cudaEventCreate(&ev0);
    cudaEventCreate(&ev1);
    const int blocks = sms * 4, threads = 256, iters = 20000;
    dfma_peak_kernel<<<blocks, threads>>>(sink, 2000, cyc);  // warm-up
    double best = 0.0, best_mhz = 0.0;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(ev0);
        dfma_peak_kernel<<<blocks, threads>>>(sink, iters, cyc);
        cudaEventRecord(ev1);
        e = cudaEventSynchronize(ev1);
        if (e != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, ev0, ev1);
        long long c[2] = {0, 1};
        cudaMemcpy(c, cyc, 16, cudaMemcpyDeviceToHost);
        const double rate = (double)blocks * threads * (double)iters * 64.0 / (ms * 1e-3);
        if (rate > best) {
            best = rate;
            best_mhz = c[1] > 0 ? (double)c[0] / (double)c[1] * 1e3 : 0.0;  // cycles per ns -> MHz
        }
    }
    cudaEventDestroy(ev0);
    cudaEventDestroy(ev1);
    cudaFree(sink);
    cudaFree(cyc);
    if (e != cudaSuccess) return e;
    *dfma_per_s = best;
    *sm_clock_mhz = best_mhz;
    return cudaGetLastError();
}

}  // namespace scarf

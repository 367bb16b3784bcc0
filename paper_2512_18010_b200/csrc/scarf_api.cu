// scarf_api.cu — the C ABI of include/scarf.h: context, argument checking, host<->device staging, launch order.
#include <chrono>
#include <cmath>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/scarf.h"
#include "kernels.cuh"

using namespace scarf;

namespace {

struct DevBuf {
    void* p = nullptr;
    size_t cap = 0;
    cudaError_t ensure(size_t bytes)
    {
        if (bytes <= cap) return cudaSuccess;
        if (p) cudaFree(p);
        p = nullptr; cap = 0;
        cudaError_t e = cudaMalloc(&p, bytes);
        if (e == cudaSuccess) cap = bytes;
        return e;
    }
    void release()
    {
        if (p) cudaFree(p);
        p = nullptr; cap = 0;
    }
};

// FP64 issue-slot model: per (q, pair, state) W(L), per (q, pair) C_tr.
const double kW[kNClasses] = {2, 7, 13, 23, 38, 59, 87, 123, 168, 223, 289, 367, 458};   // n_herm(L) + 3 (2 for L = 0)
const double kCtr = 40.0;
// product-grid kernel: YZ = Y Z, g0 = X0 YZ, g1 = X1 YZ: 12 slots per 2 q-points; tables: 39 per (pair, axis point)
const double kCtrGrid = 6.0, kCtrTable = 39.0;
// ... and its polynomial: the two points of a thread share (q_y, q_z), whose part is evaluated once (ff_common.cuh:
// record_accum_xpair): 6, 10.5, 17 slots for L = 1, 2, 3 instead of 7, 13, 23; the other classes as in the list kernel
const double kWGrid[kNClasses] = {2, 6, 10.5, 17, 38, 59, 87, 123, 168, 223, 289, 367, 458};
// row kernel (ff_row.cu): a warp's 64 points share (q_x, q_y): 5, 7, 9 slots per point for L = 1, 2, 3 plus the pre-pass
// (2, 7, 16 slots per (record, state)) spread over the 64 points of the row
// ... and 4 slots per point for g = (X Y) Z, X Y once per (row, pair): 4 more, spread over the row's 64 points
const double kCtrRow = 4.0 + 4.0 / 64.0;
// mirror-pair row kernel (ff_zrow.cu): E and O' are shared by the pair (+z, -z): 4, 5, 6 slots per point for L = 1, 2, 3 plus the
// pre-pass (X Y, the sums, H = X Y G: 14, 23, 36 slots per (row, pair, state)); per (q, pair): c z, s z or the four products of L = 0
const double kCtrZrow = 2.0;
const double kWZrow[kNClasses] = {2, 4 + 14 / 64.0, 5 + 23 / 64.0, 6 + 36 / 64.0, 38, 59, 87, 123, 168, 223, 289, 367, 458};
// spherical-grid kernel (ff_sph.cu): a warp's 64 radii share the direction: per point r d_P, sincos, E cos, E sin, and those two times r
// = 24 slots, d_P = n.P once per (direction, pair); the polynomial in r: 4, 5, 6 slots per point for L = 1, 2, 3 plus the
// per-direction sums G_n (3, 9, 19 slots per (direction, pair, state)); the E table: one exp (16 slots) per (pair, radius)
const double kCtrSph = 24.0 + 3.0 / 64.0, kCtrSphTable = 16.0;
const double kWSph[kNClasses] = {2, 4 + 3 / 64.0, 5 + 9 / 64.0, 6 + 19 / 64.0, 38, 59, 87, 123, 168, 223, 289, 367, 458};
const double kWRow[kNClasses] = {2, 5 + 2 / 64.0, 7 + 7 / 64.0, 9 + 16 / 64.0, 38, 59, 87, 123, 168, 223, 289, 367, 458};

}  // namespace

struct AngularCache {             // host tables of scarf_angular_moments and the arguments they were built for
    bool valid = false;
    int n_phi = 0, l_max = 0, n_nt = 0, n_ks = 0;
    std::vector<double> ct, wt, Yw, YwT, YwC, tw, Bf;
    int chunk_bytes = 0;
};

struct scarf_ctx {
    int device = -1;
    bool host_only = true;
    cudaStream_t stream = nullptr;
    double prefactor = 2.0, screen_tol = 1e-16, threshold_eps = 0.0;
    bool timing = false;
    int n_chunks_opt = 0;     // 0 auto, else the number of stream chunks of the S4 kernels
    double adaptive_tol = 0.0;  // > 0: q-adaptive cut-off (tau = adaptive_tol * mean bound); takes effect at set_transitions
    const double* qcut_dev = nullptr;   // q_cut per record of the current stream (sorted order), or nullptr
    double last_q_tiles = 0.0;          // q tiles of the last S4 call (for the skipped-work statistics)
    double last_ctr = 40.0;
    int grid_symmetry = 1;    // 1: use f(-q) = conj f(q) on inversion-symmetric product grids; 0: never
    int host_tile_group = 0;  // tiles per dispatch group when the kernel writes a pinned host `out` (0: automatic)
    int grid_tile_group = -1; // tiles per dispatch group of the product-grid kernels with a device `out` (-1: automatic, 0: none)
    int host_zero_copy = 1;   // 1: a pinned host `out` of the product-grid calls is written by the kernel itself (no device->host copies)
    int grid_variant = -1;    // product-grid kernel: 0 box kernel (ff_grid.cu), 1 row kernel (ff_row.cu), -1 by the grid's shape
    const double* last_grid_w = nullptr;   // work model of the last product-grid call (kWGrid or kWRow)
    double last_grid_ctr = 6.0;            // ... and its per-(q, pair) slots (kCtrGrid or kCtrRow)
    double last_table_ctr = 39.0;          // ... and the slots per table entry (kCtrTable or kCtrSphTable)
    // direction table of scarf_form_factors_sph and the arguments it was built for
    std::vector<double> sph_ct;
    int sph_n_phi = 0, sph_sym = -1;
    DevBuf d_sph_dirs;
    bool last_was_grid = false;            // the last S4 call was scarf_form_factors_grid
    int fft_density_variant = 1;  // 1: DMMA kernel, 0: SIMT kernel (fft_method.cu)
    int check_parseval = 0;       // 1: scarf_fft_form_factors also evaluates both sides of Eq. (75)
    int parseval_states = 0;      // states whose sums the last scarf_fft_form_factors call left in d_parseval
    DevBuf d_parseval;
    int angular_variant = 1;      // 1: fused DMMA kernel, 0: SIMT phi kernel + Legendre kernel (angular.cu)
    AngularCache ang;
    std::string err;
    HostSetup hs;
    bool have_basis = false, have_T = false;
    bool any_pure = false;                 // some shell is pure: T and S are mapped through pure_*
    int nbf_user = 0;                      // basis functions as the caller counts them
    std::vector<int> pure_nnz, pure_uidx;
    std::vector<double> pure_ucoef;
    int n_states = 0;
    int sm_count = 148;
    DevBuf d_pairs, d_E, d_bound, d_T, d_q, d_out, d_keep, d_desc, d_screen, d_tickets, d_key, d_keep2, d_qcut, d_work, d_axes, d_tab, d_ang_in, d_ang_F, d_ang_tab, d_ang_out, d_pure_map, d_Tcart, d_prim, d_V, d_fft, d_Csym;
    const double* Tc_dev = nullptr;        // context-owned Cartesian T of the last set_transitions (FFT method)
    std::vector<DevBuf> staging, packed;
    std::vector<TileStream> tiles;
    scarf_stats st = {};
    // screening result of the last set_transitions: written on the device, copied to pinned host memory asynchronously and
    // harvested when somebody needs it (scarf_get_stats) or when it is already there (cudaEventQuery)
    ScreenResult* h_screen = nullptr;      // pinned
    cudaEvent_t ev_screen = nullptr;
    bool screen_pending = false, T_bad = false, work_pending = false;
    double grid_eval_points = 0.0, grid_table_cols = 0.0;   // geometry of the last product-grid call (for its work model)
    cudaEvent_t ev0 = nullptr, ev1 = nullptr, ev_m0 = nullptr, ev_m1 = nullptr, ev_slice = nullptr;
    cudaStream_t copy_stream = nullptr;    // device->host copies of form_factors' output slices
    CufftPlan fft_plan;                    // cuFFT plan of the last scarf_fft_form_factors grid (this context's device)
};

namespace {

int fail(scarf_ctx* c, int code, const std::string& msg)
{
    if (c) c->err = msg;
    return code;
}

int cuda_fail(scarf_ctx* c, cudaError_t e, const char* where)
{
    cudaGetLastError();
    if (e == cudaErrorMemoryAllocation) return fail(c, SCARF_ENOMEM, std::string(where) + ": out of device memory");
    return fail(c, SCARF_ECUDA, std::string(where) + ": " + cudaGetErrorString(e));
}

#define CU(call, where)                                        \
    do {                                                       \
        cudaError_t e__ = (call);                              \
        if (e__ != cudaSuccess) return cuda_fail(ctx, e__, where); \
    } while (0)

bool is_device_ptr(const void* p)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

// Device alias of a pinned (page-locked, mapped) host buffer, or nullptr for pageable host memory.
double* mapped_host_alias(const void* p)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return nullptr;
    }
    return a.type == cudaMemoryTypeHost ? static_cast<double*>(a.devicePointer) : nullptr;
}

bool all_finite(const double* x, size_t n)
{
    // exponent field all ones <=> NaN or Inf; integer test so that the loop vectorises (a serial FP sum cost 1.6 ms per call on
    // config 3's q and T, inside the end-to-end step)
    uint64_t bad = 0;
    const long long nn = (long long)n;
    // large arrays (config 4's T: 34 MB) on up to 8 host threads: 3 ms -> 0.5 ms
#pragma omp parallel for reduction(| : bad) schedule(static) num_threads(8) if (nn >= (1LL << 20))
    for (long long i = 0; i < nn; ++i) {
        uint64_t b;
        std::memcpy(&b, x + i, sizeof(b));
        bad |= (uint64_t)((~b & 0x7ff0000000000000ULL) == 0);
    }
    return bad == 0;
}

int tile_size_for(int ns)  // smallest instantiated state tile >= ns (ns <= 12)
{
    static const int sizes[] = {1, 2, 4, 6, 8, 12};
    for (int s : sizes)
        if (s >= ns) return s;
    return kMaxStateTile;
}

// Number of stream chunks for a launch over n_tiles q tiles: enough equal-cost CTAs for ~24 waves (2 resident CTAs per SM),
// so that the ragged last wave costs a few per cent; 1 when the tiles alone give that many.  The chunks of a tile add into
// `out` one after the other (ordered tickets, ~2 us per step), so K is also kept below sqrt(T1 / 2 us), T1 = the modelled time
// of one tile's whole stream on one CTA slot (from the prescreened pair counts, which the host knows): tiny jobs (config 1:
// T1 ~ 30 us) would otherwise spend longer passing tickets than computing.
int choose_chunks(const scarf_ctx* ctx, long long n_tiles, double ctr, int ns_real, int forced)
{
    if (forced > 0) return std::min(forced, kMaxChunks);
    long long K = (24LL * 2 * ctx->sm_count + n_tiles / 2) / std::max<long long>(1, n_tiles);
    double slots = 0.0;
    for (int c = 0; c <= kFastMaxClass; ++c) slots += (double)ctx->hs.class_count[c] * ((double)ns_real * kW[c] + ctr);
    const double t1_us = slots * 256.0 / (64.0 * 1.9e9 / 2.0) * 1e6;
    K = std::min<long long>(K, (long long)std::llround(std::sqrt(t1_us / 2.0)));
    return (int)std::max<long long>(1, std::min<long long>(K, kMaxChunks));
}

bool has_high_classes(const HostSetup& hs)   // any prescreened pair of class > kFastMaxClass (needs ff_highl.cu)
{
    for (int c = kFastMaxClass + 1; c < kNClasses; ++c)
        if (hs.class_count[c] > 0) return true;
    return false;
}

// per-tile tickets of the ordered fix-up (ff_common.cuh): zeroed before every multi-chunk launch
int prepare_tickets(scarf_ctx* ctx, long long n_tiles, int n_chunks, cudaStream_t st, int** out)
{
    *out = nullptr;
    if (n_chunks <= 1) return SCARF_OK;
    CU(ctx->d_tickets.ensure((size_t)n_tiles * sizeof(int)), "alloc tickets");
    CU(cudaMemsetAsync(ctx->d_tickets.p, 0, (size_t)n_tiles * sizeof(int), st), "clear tickets");
    *out = static_cast<int*>(ctx->d_tickets.p);
    return SCARF_OK;
}

// Screening result of the last set_transitions -> stats.  wait: block until it has arrived; else only take it if it is there.
int harvest_screen(scarf_ctx* c, bool wait)
{
    if (!c->screen_pending) return SCARF_OK;
    cudaError_t e = wait ? cudaEventSynchronize(c->ev_screen) : cudaEventQuery(c->ev_screen);
    if (e == cudaErrorNotReady) { cudaGetLastError(); return SCARF_OK; }
    if (e != cudaSuccess) return cuda_fail(c, e, "screening result");
    c->screen_pending = false;
    const ScreenResult& r = *c->h_screen;
    scarf_stats& s = c->st;
    s.n_pairs_kept = r.n_kept;
    s.dropped_bound = r.dropped_bound;
    s.n_herm_kept = 0; s.slots_per_q = 0.0; s.stream_bytes = 0.0;
    for (int k = 0; k < kNClasses; ++k) {
        s.pairs_kept_per_class[k] = r.kept_per_class[k];
        s.n_herm_kept += r.kept_per_class[k] * nherm(k);
        s.slots_per_q += (double)r.kept_per_class[k] * ((double)c->n_states * kW[k] + kCtr * (double)c->tiles.size());
        for (const auto& t : c->tiles) s.stream_bytes += (double)r.kept_per_class[k] * (double)(rec_doubles(k, t.NS) * 8);
    }
    s.evals_per_q = (double)r.n_kept * (double)c->n_states;
    c->T_bad = r.bad != 0;
    return SCARF_OK;
}

const char* kBadT = "the transition matrices passed to set_transitions contain NaN/Inf (detected on the device); results are NaN";


void free_device(scarf_ctx* c)
{
    c->d_pairs.release(); c->d_E.release(); c->d_bound.release(); c->d_T.release(); c->d_q.release();
    c->d_out.release(); c->d_keep.release(); c->d_desc.release(); c->d_screen.release(); c->d_tickets.release(); c->d_key.release(); c->d_keep2.release(); c->d_qcut.release(); c->d_work.release(); c->qcut_dev = nullptr; c->d_parseval.release(); c->parseval_states = 0;
    c->d_axes.release(); c->d_tab.release(); c->d_sph_dirs.release();
    c->d_ang_in.release(); c->d_ang_F.release(); c->d_ang_tab.release(); c->d_ang_out.release();
    c->d_pure_map.release(); c->d_Tcart.release();
    c->d_prim.release(); c->d_V.release(); c->d_fft.release(); c->d_Csym.release();
    c->Tc_dev = nullptr;
    for (auto& b : c->staging) b.release();
    for (auto& b : c->packed) b.release();
    c->staging.clear(); c->packed.clear(); c->tiles.clear();
}

}  // namespace

extern "C" {

const char* scarf_version(void) { return "scarf 0.2 (sm_100a)"; }

int scarf_create(scarf_ctx** out, int device)
{
    if (!out) return SCARF_EINVAL;
    *out = nullptr;
    scarf_ctx* ctx = new (std::nothrow) scarf_ctx();
    if (!ctx) return SCARF_ENOMEM;
    if (device >= 0) {
        int n = 0;
        cudaError_t e = cudaGetDeviceCount(&n);
        if (e != cudaSuccess || device >= n) {
            cudaGetLastError();
            delete ctx;
            return SCARF_ENODEVICE;
        }
        e = cudaSetDevice(device);
        // per-device function attributes (idempotent; set for every context so that no process-wide flag is needed)
        if (e == cudaSuccess) e = ff_grid_init_device();
        if (e == cudaSuccess) e = ff_row_init_device();
        if (e == cudaSuccess) e = ff_zrow_init_device();
        if (e == cudaSuccess) e = ff_sph_init_device();
        if (e == cudaSuccess) e = angular_init_device();
        if (e == cudaSuccess) e = density_fused_init_device();
        if (e == cudaSuccess) e = cudaMallocHost(reinterpret_cast<void**>(&ctx->h_screen), sizeof(ScreenResult));
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_screen, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, device);
        if (e == cudaSuccess) e = cudaEventCreate(&ctx->ev0);
        if (e == cudaSuccess) e = cudaEventCreate(&ctx->ev1);
        if (e == cudaSuccess) e = cudaEventCreate(&ctx->ev_m0);
        if (e == cudaSuccess) e = cudaEventCreate(&ctx->ev_m1);
        if (e != cudaSuccess) {
            cudaGetLastError();
            delete ctx;
            return SCARF_ECUDA;
        }
        ctx->device = device;
        ctx->host_only = false;
    }
    *out = ctx;
    return SCARF_OK;
}

void scarf_destroy(scarf_ctx* ctx)
{
    if (!ctx) return;
    if (!ctx->host_only) {
        cudaSetDevice(ctx->device);
        cudaStreamSynchronize(ctx->stream);
        free_device(ctx);
        cufft_plan_release(ctx->fft_plan);
        if (ctx->ev0) cudaEventDestroy(ctx->ev0);
        if (ctx->ev1) cudaEventDestroy(ctx->ev1);
        if (ctx->ev_m0) cudaEventDestroy(ctx->ev_m0);
        if (ctx->ev_m1) cudaEventDestroy(ctx->ev_m1);
        if (ctx->ev_slice) cudaEventDestroy(ctx->ev_slice);
        if (ctx->ev_screen) cudaEventDestroy(ctx->ev_screen);
        if (ctx->h_screen) cudaFreeHost(ctx->h_screen);
        if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    }
    delete ctx;
}

int scarf_set_stream(scarf_ctx* ctx, void* cuda_stream)
{
    if (!ctx) return SCARF_EINVAL;
    ctx->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    return SCARF_OK;
}

int scarf_set_option(scarf_ctx* ctx, const char* key, double value)
{
    if (!ctx || !key) return SCARF_EINVAL;
    if (!std::isfinite(value)) return fail(ctx, SCARF_EINVAL, "set_option: non-finite value");
    const std::string k(key);
    if (k == "prefactor") ctx->prefactor = value;
    else if (k == "screen_tol") {
        if (value < 0) return fail(ctx, SCARF_EINVAL, "set_option: screen_tol must be >= 0");
        ctx->screen_tol = value;
    } else if (k == "timing") ctx->timing = value != 0.0;
    else if (k == "threshold_eps") { if (!(value >= 0.0)) return fail(ctx, SCARF_EINVAL, "set_option: threshold_eps < 0"); ctx->threshold_eps = value; }
    else if (k == "adaptive_tol") {
        if (value < 0) return fail(ctx, SCARF_EINVAL, "set_option: adaptive_tol must be >= 0");
        ctx->adaptive_tol = value;
    } else if (k == "grid_symmetry") {
        if (value != 0.0 && value != 1.0) return fail(ctx, SCARF_EINVAL, "set_option: grid_symmetry must be 0 or 1");
        ctx->grid_symmetry = (int)value;
    } else if (k == "grid_tile_group") {
        if (value < -1 || value > 1e6) return fail(ctx, SCARF_EINVAL, "set_option: grid_tile_group outside -1..1e6");
        ctx->grid_tile_group = (int)value;
    } else if (k == "host_tile_group") {
        if (value < 0 || value > 1e6) return fail(ctx, SCARF_EINVAL, "set_option: host_tile_group outside 0..1e6");
        ctx->host_tile_group = (int)value;
    } else if (k == "host_zero_copy") {
        if (value != 0.0 && value != 1.0) return fail(ctx, SCARF_EINVAL, "set_option: host_zero_copy must be 0 or 1");
        ctx->host_zero_copy = (int)value;
    } else if (k == "grid_variant") {
        if (value != 0.0 && value != 1.0 && value != 2.0 && value != -1.0) return fail(ctx, SCARF_EINVAL, "set_option: grid_variant must be -1, 0, 1 or 2");
        ctx->grid_variant = (int)value;
    } else if (k == "n_chunks") {
        if (value < 0 || value > kMaxChunks) return fail(ctx, SCARF_EINVAL, "set_option: n_chunks outside 0..32");
        ctx->n_chunks_opt = (int)value;
    } else if (k == "check_parseval") {
        ctx->check_parseval = value != 0.0;
    } else if (k == "angular_variant") {
        if (value != 0.0 && value != 1.0) return fail(ctx, SCARF_EINVAL, "set_option: angular_variant must be 0 or 1");
        ctx->angular_variant = (int)value;
    } else if (k == "fft_density_variant") {
        if (value != 0.0 && value != 1.0 && value != 2.0) return fail(ctx, SCARF_EINVAL, "set_option: fft_density_variant must be 0, 1 or 2");
        ctx->fft_density_variant = (int)value;
    }
    else return fail(ctx, SCARF_EINVAL, "set_option: unknown key '" + k + "'");
    return SCARF_OK;
}

int scarf_set_basis(scarf_ctx* ctx, int n_atoms, const double* atom_xyz, int n_shells, const int32_t* shell_atom,
                    const int32_t* shell_l, const int32_t* shell_nprim, const double* exponents, const double* coeffs)
{
    return scarf_set_basis_pure(ctx, n_atoms, atom_xyz, n_shells, shell_atom, shell_l, shell_nprim, exponents, coeffs, nullptr);
}

int scarf_set_basis_pure(scarf_ctx* ctx, int n_atoms, const double* atom_xyz, int n_shells, const int32_t* shell_atom,
                         const int32_t* shell_l, const int32_t* shell_nprim, const double* exponents, const double* coeffs,
                         const int32_t* shell_pure)
{
    if (!ctx) return SCARF_EINVAL;
    try {
        const auto t0 = std::chrono::steady_clock::now();
        ctx->have_basis = ctx->have_T = false;
        std::string err;
        int rc = build_setup(n_atoms, atom_xyz, n_shells, shell_atom, shell_l, shell_nprim, exponents, coeffs, ctx->hs, err);
        if (rc != SCARF_OK) return fail(ctx, rc, err);
        const HostSetup& hs = ctx->hs;
        ctx->any_pure = false;
        if (shell_pure)
            for (int i = 0; i < n_shells; ++i) ctx->any_pure = ctx->any_pure || (shell_pure[i] != 0 && shell_l[i] >= 2);
        ctx->nbf_user = build_pure_map(n_shells, shell_l, ctx->any_pure ? shell_pure : nullptr, ctx->pure_nnz, ctx->pure_uidx, ctx->pure_ucoef);
        if (!ctx->host_only && ctx->any_pure) {
            CU(cudaSetDevice(ctx->device), "set_basis");
            const size_t nb = (size_t)hs.nbf, bytes = nb * 4 + nb * kPureMaxNnz * 4 + nb * kPureMaxNnz * 8 + 64;
            CU(ctx->d_pure_map.ensure(bytes), "set_basis: alloc pure map");
            char* base = static_cast<char*>(ctx->d_pure_map.p);   // [ucoef (8-byte aligned) | uidx | nnz]
            CU(cudaMemcpyAsync(base, ctx->pure_ucoef.data(), nb * kPureMaxNnz * 8, cudaMemcpyHostToDevice, ctx->stream), "set_basis: upload");
            CU(cudaMemcpyAsync(base + nb * kPureMaxNnz * 8, ctx->pure_uidx.data(), nb * kPureMaxNnz * 4, cudaMemcpyHostToDevice, ctx->stream), "set_basis: upload");
            CU(cudaMemcpyAsync(base + nb * kPureMaxNnz * 12, ctx->pure_nnz.data(), nb * 4, cudaMemcpyHostToDevice, ctx->stream), "set_basis: upload");
        }
        if (!ctx->host_only) {
            CU(cudaSetDevice(ctx->device), "set_basis");
            CU(ctx->d_pairs.ensure(std::max<size_t>(64, hs.pairs.size() * sizeof(PairMeta))), "set_basis: alloc pairs");
            CU(ctx->d_E.ensure(std::max<size_t>(64, hs.E.size() * sizeof(double))), "set_basis: alloc E");
            CU(cudaMemcpyAsync(ctx->d_pairs.p, hs.pairs.data(), hs.pairs.size() * sizeof(PairMeta), cudaMemcpyHostToDevice, ctx->stream), "set_basis: upload pairs");
            CU(cudaMemcpyAsync(ctx->d_E.p, hs.E.data(), hs.E.size() * sizeof(double), cudaMemcpyHostToDevice, ctx->stream), "set_basis: upload E");
            CU(cudaStreamSynchronize(ctx->stream), "set_basis: sync");  // the host vectors may be rebuilt by the next call
        }
        scarf_stats& st = ctx->st;
        st = scarf_stats();
        st.n_atoms = hs.n_atoms; st.n_shells = hs.n_shells; st.n_prim_shells = (int32_t)hs.prim.size();
        st.nbf = ctx->nbf_user; st.l_max = hs.l_max;
        st.n_pairs_all = hs.n_pairs_all;
        st.n_pairs_prescreened = (int64_t)hs.pairs.size();
        st.cart_term_pairs = hs.cart_term_pairs;
        st.last_setup_host_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
        ctx->have_basis = true;
        return SCARF_OK;
    } catch (const std::bad_alloc&) {
        return fail(ctx, SCARF_ENOMEM, "set_basis: out of host memory");
    } catch (...) {
        return fail(ctx, SCARF_EINVAL, "set_basis: unexpected exception");
    }
}

int scarf_nbf(const scarf_ctx* ctx)
{
    if (!ctx) return SCARF_EINVAL;
    if (!ctx->have_basis) return SCARF_ESTATE;
    return ctx->nbf_user;
}

int scarf_overlap(scarf_ctx* ctx, double* S_host)
{
    if (!ctx || !S_host) return SCARF_EINVAL;
    if (!ctx->have_basis) return fail(ctx, SCARF_ESTATE, "overlap: set_basis first");
    if (!ctx->any_pure) {
        overlap_from_setup(ctx->hs, S_host);
        return SCARF_OK;
    }
    try {   // S_user = C^T S_cart C
        const int nc = ctx->hs.nbf, nu = ctx->nbf_user;
        std::vector<double> Sc((size_t)nc * nc), half((size_t)nc * nu, 0.0);
        overlap_from_setup(ctx->hs, Sc.data());
        for (int mu = 0; mu < nc; ++mu)
            for (int nv = 0; nv < nc; ++nv)
                for (int k = 0; k < ctx->pure_nnz[nv]; ++k)
                    half[(size_t)mu * nu + ctx->pure_uidx[(size_t)nv * kPureMaxNnz + k]] +=
                        Sc[(size_t)mu * nc + nv] * ctx->pure_ucoef[(size_t)nv * kPureMaxNnz + k];
        std::memset(S_host, 0, sizeof(double) * (size_t)nu * nu);
        for (int mu = 0; mu < nc; ++mu)
            for (int k = 0; k < ctx->pure_nnz[mu]; ++k) {
                const int a = ctx->pure_uidx[(size_t)mu * kPureMaxNnz + k];
                const double c = ctx->pure_ucoef[(size_t)mu * kPureMaxNnz + k];
                for (int b = 0; b < nu; ++b) S_host[(size_t)a * nu + b] += c * half[(size_t)mu * nu + b];
            }
    } catch (const std::bad_alloc&) {
        return fail(ctx, SCARF_ENOMEM, "overlap: out of host memory");
    }
    return SCARF_OK;
}

int scarf_set_transitions(scarf_ctx* ctx, int n_states, const double* T)
{
    if (!ctx) return SCARF_EINVAL;
    if (ctx->host_only) return fail(ctx, SCARF_ENODEVICE, "set_transitions: host-only context; there is no CPU fallback");
    if (!ctx->have_basis) return fail(ctx, SCARF_ESTATE, "set_transitions: set_basis first");
    if (n_states < 1 || !T) return fail(ctx, SCARF_EINVAL, "set_transitions: n_states < 1 or null T");
    try {
        ctx->have_T = false;
        const HostSetup& hs = ctx->hs;
        const size_t nbf = (size_t)ctx->nbf_user, tsz = (size_t)n_states * nbf * nbf;
        const long long np = (long long)hs.pairs.size();
        CU(cudaSetDevice(ctx->device), "set_transitions");
        cudaStream_t st = ctx->stream;
        const double* dT = T;
        const bool T_host = !is_device_ptr(T);
        if (T_host) {       // validated below, on the host, while the device already folds it
            CU(ctx->d_T.ensure(tsz * sizeof(double)), "set_transitions: alloc T");
            CU(cudaMemcpyAsync(ctx->d_T.p, T, tsz * sizeof(double), cudaMemcpyHostToDevice, st), "set_transitions: upload T");
            dT = static_cast<const double*>(ctx->d_T.p);
        }
        if (ctx->any_pure) {   // T_cart = C T_user C^T (pure.cu); the fold works on Cartesian components
            const size_t nc = (size_t)hs.nbf;
            CU(ctx->d_Tcart.ensure((size_t)n_states * nc * nc * sizeof(double)), "set_transitions: alloc T_cart");
            const char* base = static_cast<const char*>(ctx->d_pure_map.p);
            CU(launch_transform_T(dT, static_cast<double*>(ctx->d_Tcart.p), n_states, ctx->nbf_user, hs.nbf,
                                  reinterpret_cast<const int*>(base + nc * kPureMaxNnz * 12), reinterpret_cast<const int*>(base + nc * kPureMaxNnz * 8),
                                  reinterpret_cast<const double*>(base), st), "set_transitions: pure transform kernel");
            dT = static_cast<const double*>(ctx->d_Tcart.p);
        } else if (dT == T) {   // caller-owned device T: keep a copy (inputs are copied; the FFT method reads T later)
            CU(ctx->d_T.ensure(tsz * sizeof(double)), "set_transitions: alloc T");
            CU(cudaMemcpyAsync(ctx->d_T.p, T, tsz * sizeof(double), cudaMemcpyDeviceToDevice, st), "set_transitions: copy T");
            dT = static_cast<const double*>(ctx->d_T.p);
        }
        ctx->Tc_dev = dT;
        // state tiles
        std::vector<TileStream> tiles;
        for (int s0 = 0; s0 < n_states; s0 += kMaxStateTile) {
            TileStream t = {};
            t.s0 = s0;
            t.ns_real = std::min(kMaxStateTile, n_states - s0);
            t.NS = tile_size_for(t.ns_real);
            tiles.push_back(t);
        }
        if (ctx->staging.size() < tiles.size()) ctx->staging.resize(tiles.size());
        if (ctx->packed.size() < tiles.size()) ctx->packed.resize(tiles.size());
        CU(ctx->d_bound.ensure(std::max<size_t>(64, (size_t)np * sizeof(double))), "set_transitions: alloc bound");
        CU(ctx->d_keep.ensure(std::max<size_t>(64, (size_t)np * sizeof(int))), "set_transitions: alloc index");
        CU(ctx->d_desc.ensure(tiles.size() * sizeof(StreamDesc)), "set_transitions: alloc descriptors");
        CU(ctx->d_screen.ensure(sizeof(ScreenResult)), "set_transitions: alloc screening result");
        if (ctx->timing) CU(cudaEventRecord(ctx->ev0, st), "set_transitions: event");
        // S3: fold every tile into a staging stream that holds ALL prescreened pairs (class-sorted) and the bounds B_P
        for (size_t it = 0; it < tiles.size(); ++it) {
            TileStream& t = tiles[it];
            FoldArgs a = {};
            a.pairs = static_cast<const PairMeta*>(ctx->d_pairs.p);
            a.n_pairs = np;
            a.E = static_cast<const double*>(ctx->d_E.p);
            a.T = dT;
            a.nbf = hs.nbf; a.s0 = t.s0; a.ns_real = t.ns_real; a.NS = t.NS;
            a.first_tile = it == 0;
            a.g = ctx->prefactor;
            a.bound = static_cast<double*>(ctx->d_bound.p);
            unsigned long long off = 0;
            for (int c = 0; c < kNClasses; ++c) {
                a.class_first[c] = hs.class_first[c];
                a.cls_off[c] = off;
                a.rec_bytes[c] = rec_doubles(c, t.NS) * 8;
                off += (unsigned long long)hs.class_count[c] * a.rec_bytes[c];
            }
            a.class_first[kNClasses] = hs.class_first[kNClasses];
            CU(ctx->staging[it].ensure(std::max<unsigned long long>(64, off)), "set_transitions: alloc staging");
            CU(ctx->packed[it].ensure(std::max<unsigned long long>(64, off)), "set_transitions: alloc packed");
            a.staging = static_cast<char*>(ctx->staging[it].p);
            CU(launch_fold(a, st), "set_transitions: fold kernel");
            t.staging = a.staging;
            t.staging_bytes = off;
            t.base = static_cast<char*>(ctx->packed[it].p);
            t.desc = static_cast<StreamDesc*>(ctx->d_desc.p) + it;
        }
        // screening on the device (reading #12): B_P < max(screen_tol * mean(B), threshold_eps * max(B)) is dropped; stable
        // compaction; then every tile's kept records are packed and its descriptor written.  No device->host round trip.
        ScreenArgs sa = {};
        sa.bound = static_cast<const double*>(ctx->d_bound.p);
        sa.n_pairs = np;
        for (int c = 0; c <= kNClasses; ++c) sa.class_first[c] = hs.class_first[c];
        sa.screen_tol = ctx->screen_tol;
        sa.threshold_eps = ctx->threshold_eps;
        sa.keep_idx = static_cast<int*>(ctx->d_keep.p);
        sa.result = static_cast<ScreenResult*>(ctx->d_screen.p);
        CU(launch_screen(sa, st), "set_transitions: screen kernel");
        // q-adaptive cut-off (option adaptive_tol): q_cut per kept record, records re-ordered by it inside each class
        const int* keep_for_pack = sa.keep_idx;
        ctx->qcut_dev = nullptr;
        if (ctx->adaptive_tol > 0.0) {
            if ((int)tiles.size() > kMaxAdaptTiles) return fail(ctx, SCARF_EINVAL, "set_transitions: adaptive_tol supports at most 96 states");
            CU(ctx->d_key.ensure(std::max<size_t>(64, (size_t)np * sizeof(double))), "set_transitions: alloc keys");
            CU(ctx->d_qcut.ensure(std::max<size_t>(64, (size_t)np * sizeof(double))), "set_transitions: alloc q_cut");
            CU(ctx->d_keep2.ensure(std::max<size_t>(64, (size_t)np * sizeof(int))), "set_transitions: alloc index");
            CU(ctx->d_work.ensure(kNClasses * sizeof(unsigned long long)), "set_transitions: alloc counters");
            AdaptArgs aa = {};
            aa.keep_idx = sa.keep_idx;
            aa.result = sa.result;
            for (int c = 0; c <= kNClasses; ++c) aa.class_first[c] = hs.class_first[c];
            aa.n_tiles = (int)tiles.size();
            for (size_t it = 0; it < tiles.size(); ++it) {
                aa.staging[it] = tiles[it].staging;
                aa.NS[it] = tiles[it].NS;
                unsigned long long off = 0;
                for (int c = 0; c < kNClasses; ++c) {
                    aa.cls_off[it][c] = off;
                    aa.rec_bytes[it][c] = rec_doubles(c, tiles[it].NS) * 8;
                    off += (unsigned long long)hs.class_count[c] * aa.rec_bytes[it][c];
                }
            }
            aa.adaptive_tol = ctx->adaptive_tol;
            aa.n_pairs = np;
            aa.key = static_cast<double*>(ctx->d_key.p);
            aa.keep_sorted = static_cast<int*>(ctx->d_keep2.p);
            aa.qcut_sorted = static_cast<double*>(ctx->d_qcut.p);
            CU(launch_adaptive_sort(aa, st), "set_transitions: q-adaptive kernels");
            keep_for_pack = aa.keep_sorted;
            ctx->qcut_dev = aa.qcut_sorted;
        }
        for (size_t it = 0; it < tiles.size(); ++it) {
            const TileStream& t = tiles[it];
            PackArgs pa = {};
            pa.staging = t.staging;
            pa.packed = t.base;
            pa.keep_idx = keep_for_pack;
            pa.result = sa.result;
            pa.desc = t.desc;
            pa.n_pairs = np;
            unsigned long long off = 0;
            for (int c = 0; c < kNClasses; ++c) {
                pa.class_first[c] = hs.class_first[c];
                pa.cls_off[c] = off;
                pa.rec_bytes[c] = rec_doubles(c, t.NS) * 8;
                off += (unsigned long long)hs.class_count[c] * pa.rec_bytes[c];
            }
            pa.class_first[kNClasses] = hs.class_first[kNClasses];
            CU(launch_pack(pa, st), "set_transitions: pack kernel");
        }
        CU(cudaMemcpyAsync(ctx->h_screen, ctx->d_screen.p, sizeof(ScreenResult), cudaMemcpyDeviceToHost, st), "set_transitions: result copy");
        CU(cudaEventRecord(ctx->ev_screen, st), "set_transitions: event");
        ctx->screen_pending = true;
        ctx->T_bad = false;
        ctx->tiles = tiles;
        ctx->n_states = n_states;
        scarf_stats& s = ctx->st;
        s.n_states = n_states;
        s.n_pairs_kept = -1;      // unknown until harvested (scarf_get_stats waits for it)
        s.last_fold_launches = (int32_t)(2 * tiles.size() + 1 + (ctx->any_pure ? 1 : 0) + (ctx->qcut_dev ? 2 : 0));
        s.adaptive_bound = 0.0; s.last_adaptive_work_fraction = 1.0;
        if (ctx->timing) {
            CU(cudaEventRecord(ctx->ev1, st), "set_transitions: event");
            CU(cudaEventSynchronize(ctx->ev1), "set_transitions: event sync");
            float ms = 0.f;
            cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1);
            ctx->st.last_fold_ms = ms;
        }
        // Host T: NaN/Inf check (a pass over n_states nbf^2 doubles, 0.3 ms on config 3) AFTER the upload and the kernels have been
        // queued, so that it overlaps them; a bad T still fails this very call, and nothing of it stays behind.
        if (T_host && !all_finite(T, tsz)) {
            cudaStreamSynchronize(st);
            ctx->screen_pending = false;
            return fail(ctx, SCARF_EINVAL, "set_transitions: NaN/Inf in T");
        }
        ctx->have_T = true;
        return SCARF_OK;
    } catch (const std::bad_alloc&) {
        return fail(ctx, SCARF_ENOMEM, "set_transitions: out of host memory");
    } catch (...) {
        return fail(ctx, SCARF_EINVAL, "set_transitions: unexpected exception");
    }
}

int scarf_form_factors(scarf_ctx* ctx, int64_t n_q, const double* q, double* out)
{
    if (!ctx) return SCARF_EINVAL;
    if (ctx->host_only) return fail(ctx, SCARF_ENODEVICE, "form_factors: host-only context; there is no CPU fallback");
    if (!ctx->have_T) return fail(ctx, SCARF_ESTATE, "form_factors: set_basis and set_transitions first");
    if (n_q < 0) return fail(ctx, SCARF_EINVAL, "form_factors: n_q < 0");
    if (n_q == 0) return SCARF_OK;
    if (!q || !out) return fail(ctx, SCARF_EINVAL, "form_factors: null q or out");
    try {
        CU(cudaSetDevice(ctx->device), "form_factors");
        cudaStream_t st = ctx->stream;
        if (harvest_screen(ctx, false) != SCARF_OK) return SCARF_ECUDA;
        if (ctx->T_bad) return fail(ctx, SCARF_EINVAL, std::string("form_factors: ") + kBadT);
        const size_t qbytes = (size_t)n_q * 3 * sizeof(double);
        const size_t obytes = (size_t)ctx->n_states * (size_t)n_q * 2 * sizeof(double);
        const double* dq = q;
        double* dout = out;
        const bool q_host = !is_device_ptr(q), out_host = !is_device_ptr(out);
        if (q_host) {
            if (!all_finite(q, (size_t)n_q * 3)) return fail(ctx, SCARF_EINVAL, "form_factors: NaN/Inf in q");
            CU(ctx->d_q.ensure(qbytes), "form_factors: alloc q");
            CU(cudaMemcpyAsync(ctx->d_q.p, q, qbytes, cudaMemcpyHostToDevice, st), "form_factors: upload q");
            dq = static_cast<const double*>(ctx->d_q.p);
        }
        if (out_host) {
            CU(ctx->d_out.ensure(obytes), "form_factors: alloc out");
            dout = static_cast<double*>(ctx->d_out.p);
        }
        if (ctx->timing) CU(cudaEventRecord(ctx->ev0, st), "form_factors: event");
        int launches = 0;
        double main_ms = 0.0;
        if (ctx->qcut_dev) {
            CU(cudaMemsetAsync(ctx->d_work.p, 0, kNClasses * sizeof(unsigned long long), st), "form_factors: clear counters");
            ctx->last_q_tiles = 0.0; ctx->last_ctr = kCtr; ctx->last_was_grid = false; ctx->work_pending = true;
        }
        // all state tiles for the q range [dq, dq + 3 n_q) into dout [n_states][n_q]
        auto run_range = [&](const double* dq, long long n_q, double* dout) -> int {
        for (const TileStream& t : ctx->tiles) {
            V1Args a = {};
            a.base = t.base;
            a.desc = t.desc;
            a.q = dq;
            a.n_q = n_q;
            const long long n_tiles = (n_q + v1_tile_q() - 1) / v1_tile_q();
            if (n_tiles > 0x7fffffffLL) return fail(ctx, SCARF_EINVAL, "form_factors: n_q too large for one call");
            a.n_tiles = (int)n_tiles;
            a.n_chunks = choose_chunks(ctx, n_tiles, kCtr, t.ns_real, ctx->n_chunks_opt);
            a.ns_real = t.ns_real;
            a.dst = dout + (size_t)t.s0 * n_q * 2;
            if (int rc = prepare_tickets(ctx, n_tiles, a.n_chunks, st, &a.tickets)) return rc;
            a.qcut = ctx->qcut_dev;
            a.work = ctx->qcut_dev ? static_cast<unsigned long long*>(ctx->d_work.p) : nullptr;
            if (&t == &ctx->tiles.front()) ctx->last_q_tiles += (double)n_tiles;
            CU(launch_plan_chunks(t.desc, a.n_chunks, t.ns_real, kCtr, st), "form_factors: chunk planning kernel");
            if (ctx->timing) CU(cudaEventRecord(ctx->ev_m0, st), "form_factors: event");
            CU(launch_ff_v1(t.NS, a, st), "form_factors: kernel");
            if (ctx->timing) {
                CU(cudaEventRecord(ctx->ev_m1, st), "form_factors: event");
                CU(cudaEventSynchronize(ctx->ev_m1), "form_factors: event sync");
                float ms = 0.f;
                cudaEventElapsedTime(&ms, ctx->ev_m0, ctx->ev_m1);
                main_ms += ms;
            }
            ctx->st.last_n_chunks = a.n_chunks;
            launches += 2;
            if (has_high_classes(ctx->hs)) {            // pairs with g, h, i shells: separate kernel, adds to out
                HighLArgs h = {};
                h.base = t.base; h.desc = t.desc; h.q = dq;
                h.ns_real = t.ns_real; h.n_points = n_q; h.n_q = n_q; h.dst = a.dst;
                CU(launch_ff_highl(h, st), "form_factors: high-class kernel");
                ++launches;
            }
        }
        return SCARF_OK;
        };
        // Host output: the q range is cut into slices whose device->host copies (second stream) overlap the kernels of
        // the next slice; each slice is computed into its own contiguous [n_states][slice] scratch and copied with a 2-D copy.
        const int n_slices = (out_host && n_q >= 4 * 16384) ? 4 : 1;
        if (n_slices == 1) {
            const int rc = run_range(dq, n_q, dout);
            if (rc != SCARF_OK) return rc;
        } else {
            if (!ctx->copy_stream) CU(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking), "form_factors: copy stream");
            if (!ctx->ev_slice) CU(cudaEventCreateWithFlags(&ctx->ev_slice, cudaEventDisableTiming), "form_factors: event");
            const long long per = ((n_q + n_slices - 1) / n_slices + 255) & ~255LL;
            // On any failure the copies already queued into the caller's `out` must have landed before we return
            // (the caller may free `out` as soon as it sees the error code).
            auto drain = [&](int rc) { cudaStreamSynchronize(ctx->copy_stream); cudaStreamSynchronize(st); return rc; };
            for (long long q0 = 0; q0 < n_q; q0 += per) {
                const long long nq_s = std::min(per, n_q - q0);
                double* d_s = dout + (size_t)ctx->n_states * (size_t)q0 * 2;      // slice k occupies [n_states][nq_s] at this offset
                const int rc = run_range(dq + 3 * q0, nq_s, d_s);
                if (rc != SCARF_OK) return drain(rc);
                cudaError_t e = cudaEventRecord(ctx->ev_slice, st);
                if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_slice, 0);
                // one contiguous copy per state (a 2-D copy would need a pitch of n_q*16 bytes, beyond memPitch for n_q >= 2^27)
                for (int s = 0; s < ctx->n_states && e == cudaSuccess; ++s)
                    e = cudaMemcpyAsync(out + ((size_t)s * (size_t)n_q + (size_t)q0) * 2, d_s + (size_t)s * (size_t)nq_s * 2,
                                        (size_t)nq_s * 16, cudaMemcpyDeviceToHost, ctx->copy_stream);
                if (e != cudaSuccess) return drain(cuda_fail(ctx, e, "form_factors: download slice"));
            }
        }
        ctx->st.last_kernel_launches = launches;
        if (ctx->timing) {
            CU(cudaEventRecord(ctx->ev1, st), "form_factors: event");
            CU(cudaEventSynchronize(ctx->ev1), "form_factors: event sync");
            float ms = 0.f;
            cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1);
            ctx->st.last_kernel_ms = ms;
            ctx->st.last_main_kernel_ms = main_ms;
        }
        if (out_host && n_slices > 1) {
            CU(cudaStreamSynchronize(ctx->copy_stream), "form_factors: sync copies");
            CU(cudaStreamSynchronize(st), "form_factors: sync");
        } else if (out_host) {
            CU(cudaMemcpyAsync(out, dout, obytes, cudaMemcpyDeviceToHost, st), "form_factors: download out");
            CU(cudaStreamSynchronize(st), "form_factors: sync");
        } else if (q_host) {
            CU(cudaStreamSynchronize(st), "form_factors: sync");  // pageable q must not be reused before the copy ends
        }
        if (out_host || q_host) {                                   // the stream has drained: the screening result is there
            if (harvest_screen(ctx, true) != SCARF_OK) return SCARF_ECUDA;
            if (ctx->T_bad) return fail(ctx, SCARF_EINVAL, std::string("form_factors: ") + kBadT);
        }
        return SCARF_OK;
    } catch (const std::bad_alloc&) {
        return fail(ctx, SCARF_ENOMEM, "form_factors: out of host memory");
    } catch (...) {
        return fail(ctx, SCARF_EINVAL, "form_factors: unexpected exception");
    }
}

// Allocation-free S4 (include/scarf.h): the launches of scarf_form_factors for device q / device out, with the tickets of the
// ordered fix-up in ff_v1.cu's static device array.  Nothing here allocates device memory or synchronises.
int scarf_form_factors_noalloc(scarf_ctx* ctx, int64_t n_q, const double* q_dev, double* out_dev)
{
    static_assert(SCARF_NOALLOC_MAX_TILES == 65536, "keep in step with kStaticTickets (ff_v1.cu)");
    if (!ctx) return SCARF_EINVAL;
    if (ctx->host_only) return fail(ctx, SCARF_ENODEVICE, "form_factors_noalloc: host-only context; there is no CPU fallback");
    if (!ctx->have_T) return fail(ctx, SCARF_ESTATE, "form_factors_noalloc: set_basis and set_transitions first");
    if (n_q < 0) return fail(ctx, SCARF_EINVAL, "form_factors_noalloc: n_q < 0");
    if (n_q == 0) return SCARF_OK;
    const long long n_tiles = (n_q + v1_tile_q() - 1) / v1_tile_q();
    if (v1_static_tiles() != SCARF_NOALLOC_MAX_TILES) return fail(ctx, SCARF_EINVAL, "form_factors_noalloc: library built inconsistently");
    if (n_tiles > SCARF_NOALLOC_MAX_TILES)
        return fail(ctx, SCARF_EINVAL, "form_factors_noalloc: n_q = " + std::to_string((long long)n_q) + " exceeds the static scratch (" +
                                           std::to_string(SCARF_NOALLOC_MAX_TILES) + " tiles of " + std::to_string(v1_tile_q()) + " q-points = " +
                                           std::to_string((long long)SCARF_NOALLOC_MAX_TILES * v1_tile_q()) +
                                           " q-points per call); split the point set or use scarf_form_factors");
    if (!q_dev || !out_dev) return fail(ctx, SCARF_EINVAL, "form_factors_noalloc: null q or out");
    try {
        CU(cudaSetDevice(ctx->device), "form_factors_noalloc");
        if (!is_device_ptr(q_dev) || !is_device_ptr(out_dev))
            return fail(ctx, SCARF_EINVAL, "form_factors_noalloc: q and out must be device pointers (staging host data would allocate)");
        cudaStream_t st = ctx->stream;
        if (harvest_screen(ctx, false) != SCARF_OK) return SCARF_ECUDA;          // non-blocking
        if (ctx->T_bad) return fail(ctx, SCARF_EINVAL, std::string("form_factors_noalloc: ") + kBadT);
        CU(ff_v1_static_setup(), "form_factors_noalloc: static scratch address");
        int launches = 0;
        if (ctx->qcut_dev) {                       // q-adaptive cut-off: counters were allocated by set_transitions
            CU(cudaMemsetAsync(ctx->d_work.p, 0, kNClasses * sizeof(unsigned long long), st), "form_factors_noalloc: clear counters");
            ctx->last_q_tiles = 0.0; ctx->last_ctr = kCtr; ctx->last_was_grid = false; ctx->work_pending = true;
        }
        for (const TileStream& t : ctx->tiles) {
            V1Args a = {};
            a.base = t.base;
            a.desc = t.desc;
            a.q = q_dev;
            a.n_q = n_q;
            a.n_tiles = (int)n_tiles;
            a.n_chunks = choose_chunks(ctx, n_tiles, kCtr, t.ns_real, ctx->n_chunks_opt);
            a.ns_real = t.ns_real;
            a.dst = out_dev + (size_t)t.s0 * n_q * 2;
            a.qcut = ctx->qcut_dev;
            a.work = ctx->qcut_dev ? static_cast<unsigned long long*>(ctx->d_work.p) : nullptr;
            if (&t == &ctx->tiles.front()) ctx->last_q_tiles += (double)n_tiles;
            CU(launch_plan_chunks(t.desc, a.n_chunks, t.ns_real, kCtr, st), "form_factors_noalloc: chunk planning kernel");
            CU(launch_ff_v1_static(t.NS, a, st), "form_factors_noalloc: kernel");
            ctx->st.last_n_chunks = a.n_chunks;
            launches += 2;
            if (has_high_classes(ctx->hs)) {            // pairs with g, h, i shells: separate kernel, adds to out
                HighLArgs h = {};
                h.base = t.base; h.desc = t.desc; h.q = q_dev;
                h.ns_real = t.ns_real; h.n_points = n_q; h.n_q = n_q; h.dst = a.dst;
                CU(launch_ff_highl(h, st), "form_factors_noalloc: high-class kernel");
                ++launches;
            }
        }
        ctx->st.last_kernel_launches = launches;
        return SCARF_OK;
    } catch (const std::bad_alloc&) {
        return fail(ctx, SCARF_ENOMEM, "form_factors_noalloc: out of host memory");
    } catch (...) {
        return fail(ctx, SCARF_EINVAL, "form_factors_noalloc: unexpected exception");
    }
}

int scarf_form_factors_grid(scarf_ctx* ctx, int32_t nx, const double* qx, int32_t ny, const double* qy, int32_t nz,
                            const double* qz, double* out)
{
    if (!ctx) return SCARF_EINVAL;
    if (ctx->host_only) return fail(ctx, SCARF_ENODEVICE, "form_factors_grid: host-only context; there is no CPU fallback");
    if (!ctx->have_T) return fail(ctx, SCARF_ESTATE, "form_factors_grid: set_basis and set_transitions first");
    if (nx < 0 || ny < 0 || nz < 0) return fail(ctx, SCARF_EINVAL, "form_factors_grid: negative axis length");
    const long long n_q = (long long)nx * ny * nz;
    if (n_q == 0) return SCARF_OK;
    if (!qx || !qy || !qz || !out) return fail(ctx, SCARF_EINVAL, "form_factors_grid: null axis or out");
    try {
        CU(cudaSetDevice(ctx->device), "form_factors_grid");
        cudaStream_t st = ctx->stream;
        if (harvest_screen(ctx, false) != SCARF_OK) return SCARF_ECUDA;
        if (ctx->T_bad) return fail(ctx, SCARF_EINVAL, std::string("form_factors_grid: ") + kBadT);
        // axes -> one device buffer [nx | ny | nz]; a host copy of every axis decides whether the grid is inversion-symmetric
        const double* ax_in[3] = {qx, qy, qz};
        const int ax_n[3] = {nx, ny, nz};
        CU(ctx->d_axes.ensure(((size_t)nx + ny + nz) * sizeof(double)), "form_factors_grid: alloc axes");
        double* dax[3];
        std::vector<double> hax[3];
        size_t off = 0;
        bool need_sync = false, all_host = true;
        for (int k = 0; k < 3; ++k) {
            dax[k] = static_cast<double*>(ctx->d_axes.p) + off;
            off += (size_t)ax_n[k];
            const bool host = !is_device_ptr(ax_in[k]);
            all_host = all_host && host;
            if (host && !all_finite(ax_in[k], (size_t)ax_n[k])) return fail(ctx, SCARF_EINVAL, "form_factors_grid: NaN/Inf in an axis");
        }
        if (all_host) {      // one staged upload instead of three (pageable host -> device copies of this size are staged by
                             // the runtime before the call returns: no sync needed, the vector may die at once)
            std::vector<double> cat;
            cat.reserve(off);
            for (int k = 0; k < 3; ++k) cat.insert(cat.end(), ax_in[k], ax_in[k] + ax_n[k]);
            CU(cudaMemcpyAsync(ctx->d_axes.p, cat.data(), off * sizeof(double), cudaMemcpyHostToDevice, st), "form_factors_grid: copy axes");
        }
        for (int k = 0; k < 3; ++k) {
            const bool host = !is_device_ptr(ax_in[k]);
            if (!all_host)
                CU(cudaMemcpyAsync(dax[k], ax_in[k], (size_t)ax_n[k] * sizeof(double), host ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, st),
                   "form_factors_grid: copy axis");
            {   // a host copy of every axis: the symmetry decisions below
                hax[k].resize((size_t)ax_n[k]);
                if (host) std::memcpy(hax[k].data(), ax_in[k], (size_t)ax_n[k] * sizeof(double));
                else {
                    CU(cudaMemcpyAsync(hax[k].data(), ax_in[k], (size_t)ax_n[k] * sizeof(double), cudaMemcpyDeviceToHost, st),
                       "form_factors_grid: read axis");
                    need_sync = true;
                }
            }
        }
        if (need_sync) CU(cudaStreamSynchronize(st), "form_factors_grid: sync");   // device axes: documented in scarf.h
        // inversion symmetry: every axis antisymmetric, bit for bit (then q -> -q maps grid point i to n_q - 1 - i)
        bool sym = ctx->grid_symmetry != 0 && nx >= 2;
        for (int k = 0; k < 3 && sym; ++k)
            for (int i = 0; i < ax_n[k] && sym; ++i) sym = hax[k][(size_t)i] == -hax[k][(size_t)(ax_n[k] - 1 - i)];
        const int nx_eval = sym ? (nx + 1) / 2 : nx;
        // Kernel: the row kernel (a warp = 64 z-points of one (ix, iy) row, 4 rows per CTA) needs fewer FP64 slots per point but
        // wastes the lanes beyond the end of a row; it is taken when the 4 x 64 boxes are at least 80 % full.
        const double row_fill = ((double)ny * nz) / ((double)((ny + kRowBY - 1) / kRowBY * kRowBY) * (double)((nz + kRowBZ - 1) / kRowBZ * kRowBZ));
        // Mirror-pair row kernel: needs a z axis that is antisymmetric bit for bit (a lane's two points are +z and -z of its row; this is
        // independent of the inversion symmetry of the whole grid); its boxes are 4 (y) x 32 mirror pairs.
        bool z_antisym = nz >= 2;
        for (int i = 0; i < nz && z_antisym; ++i) z_antisym = hax[2][(size_t)i] == -hax[2][(size_t)(nz - 1 - i)];
        const int nz_half = (nz + 1) / 2;
        const double zrow_fill = ((double)ny * nz_half) / ((double)((ny + kZrowBY - 1) / kZrowBY * kZrowBY) * (double)((nz_half + kZrowBZ - 1) / kZrowBZ * kZrowBZ));
        // Taken from 75 % full boxes on (a 24-pair row is three whole M tiles of its tensor-core classes): measured on config 2's 48-point
        // rows, job 1.94 ms against 2.17 ms for the box kernel.
        const bool zrow = z_antisym && (ctx->grid_variant == 2 || (ctx->grid_variant < 0 && zrow_fill >= 0.75));
        const bool row = !zrow && (ctx->grid_variant == 1 || (ctx->grid_variant != 0 && row_fill >= 0.8));
        const int BXs = zrow ? kZrowBX : (row ? kRowBX : kGridBX), BYs = zrow ? kZrowBY : (row ? kRowBY : kGridBY),
                  BZs = zrow ? kZrowBZ : (row ? kRowBZ : kGridBZ);
        const double* kWg = zrow ? kWZrow : (row ? kWRow : kWGrid);
        const double ctr_g = zrow ? kCtrZrow : (row ? kCtrRow : kCtrGrid);
        const int nbx = (nx_eval + BXs - 1) / BXs, nby = (ny + BYs - 1) / BYs, nbz = ((zrow ? nz_half : nz) + BZs - 1) / BZs;
        const long long n_tiles = (long long)nbx * nby * nbz;
        if (n_tiles > 0x7fffffffLL) return fail(ctx, SCARF_EINVAL, "form_factors_grid: grid too large for one call");
        const size_t obytes = (size_t)ctx->n_states * (size_t)n_q * 2 * sizeof(double);
        double* dout = out;
        const bool out_host = !is_device_ptr(out);
        if (out_host) {
            CU(ctx->d_out.ensure(obytes), "form_factors_grid: alloc out");
            dout = static_cast<double*>(ctx->d_out.p);
        }
        if (ctx->timing) CU(cudaEventRecord(ctx->ev0, st), "form_factors_grid: event");
        int launches = 0;
        double main_ms = 0.0;
        if (ctx->qcut_dev) {
            CU(cudaMemsetAsync(ctx->d_work.p, 0, kNClasses * sizeof(unsigned long long), st), "form_factors_grid: clear counters");
            ctx->last_q_tiles = (double)n_tiles; ctx->last_ctr = ctr_g; ctx->last_was_grid = true; ctx->last_grid_w = kWg; ctx->work_pending = true;
        }
        const long long ncol = (long long)nbx * BXs + (long long)nby * BYs + (long long)nbz * BZs;
        const long long n_rows = (long long)ctx->hs.pairs.size();    // prescreened pairs: an upper bound of the kept count
        // Pinned host `out`: the last chunk of every box stores the finished values straight into it (a mapped alias), so the output
        // crosses PCIe while the kernel runs and no copy follows it; partial sums of the chunks stay in the device scratch.
        double* out_alias = (out_host && ctx->host_zero_copy && !has_high_classes(ctx->hs)) ? mapped_host_alias(out) : nullptr;
        const int n_slabs = (out_host && !out_alias && nbx >= 4 && n_q >= 4 * 16384 && !has_high_classes(ctx->hs)) ? 4 : 1;
        if (n_slabs > 1) {
            if (!ctx->copy_stream) CU(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking), "form_factors_grid: copy stream");
            if (!ctx->ev_slice) CU(cudaEventCreateWithFlags(&ctx->ev_slice, cudaEventDisableTiming), "form_factors_grid: event");
        }
        // on any failure the copies already queued into the caller's `out` must have landed before we return
        auto drain = [&](int rc) { cudaStreamSynchronize(ctx->copy_stream); cudaStreamSynchronize(st); return rc; };
        for (const TileStream& t : ctx->tiles) {
            GridArgs a = {};
            const size_t tab_elems = (size_t)std::max<long long>(1, n_rows) * (size_t)ncol;
            if (tab_elems * 16 > (size_t)32e9) return fail(ctx, SCARF_ENOMEM, "form_factors_grid: factor tables would exceed 32 GB");
            CU(ctx->d_tab.ensure(tab_elems * 16), "form_factors_grid: alloc tables");
            double2* tx = static_cast<double2*>(ctx->d_tab.p);
            double2* ty = tx + (size_t)n_rows * nbx * BXs;
            double2* tz = ty + (size_t)n_rows * nby * BYs;
            a.bxs = BXs; a.bys = BYs; a.bzs = BZs;
            a.v.base = t.base;
            a.v.desc = t.desc;
            a.v.n_q = n_q;
            a.v.n_tiles = (int)n_tiles;
            a.v.ns_real = t.ns_real;
            a.v.dst = dout + (size_t)t.s0 * n_q * 2;
            a.v.dst_final = out_alias ? out_alias + (size_t)t.s0 * n_q * 2 : nullptr;
            a.qx = dax[0]; a.qy = dax[1]; a.qz = dax[2];
            a.nx = nx; a.ny = ny; a.nz = nz;
            a.nbx = nbx; a.nby = nby; a.nbz = nbz;
            a.sym = sym ? 1 : 0;
            a.nx_eval = nx_eval;
            a.tx = tx; a.ty = ty; a.tz = tz;
            a.n_rows = n_rows;
            a.v.qcut = ctx->qcut_dev;
            a.v.work = ctx->qcut_dev ? static_cast<unsigned long long*>(ctx->d_work.p) : nullptr;
            {
                GridArgs at = a;
                if (zrow) at.nz = nz_half;              // the Z table of the mirror-pair kernel covers the first half of the axis
                CU(launch_grid_tables(at, tx, ty, tz, st), "form_factors_grid: table kernel");
            }
            ++launches;
            // Host output: the x boxes are cut into slabs; the device->host copies of a finished slab (and of its mirror slab on
            // a symmetric grid) run on a second stream while the next slab is being computed.
            for (int sl = 0; sl < n_slabs; ++sl) {
                const int b0 = (int)((long long)nbx * sl / n_slabs), b1 = (int)((long long)nbx * (sl + 1) / n_slabs);
                if (b1 <= b0) continue;
                const long long tiles_s = (long long)(b1 - b0) * nby * nbz;
                a.bx0 = b0;
                a.v.n_tiles = (int)tiles_s;
                a.v.n_chunks = choose_chunks(ctx, tiles_s, ctr_g, t.ns_real, ctx->n_chunks_opt);
                // the mirror-pair kernel pays per chunk for its layout exchanges and short last k-tiles: measured flat from 6 to 14 chunks
                // on configs 3 and 4, 1.90-1.94 ms for 3..12 chunks against 2.05 ms for 25 on config 2
                if (zrow && ctx->n_chunks_opt <= 0) a.v.n_chunks = std::min(a.v.n_chunks, 12);
                // Pinned host `out`: the CTAs are dispatched chunk-major inside groups of tiles, group after group, so that finished
                // tiles leave for the host all along the kernel's run (chunk-major over all tiles would send everything in the last
                // 1/n_chunks of it).  Measured on config 3 (ms per call, host `out`): groups of 128 tiles (3/7 of the CTA slots) and
                // about 8 waves of CTAs (5 chunks) 6.60; 14 chunks 6.76; groups of 16 / 32 / 64 / 256 / 296 tiles (14 chunks) 7.27 /
                // 6.96 / 6.89 / 7.01 / 7.15 (small groups: the chunks of a tile run side by side and queue at its ticket; large
                // groups: a long tail); no groups 7.04; device `out` 6.46.
                if (out_alias) {
                    const long long slots = 2LL * ctx->sm_count;
                    if (ctx->n_chunks_opt <= 0) a.v.n_chunks = (int)std::max<long long>(1, std::min<long long>(a.v.n_chunks, (8 * slots + tiles_s - 1) / tiles_s));
                    a.v.tile_group = a.v.n_chunks > 1 ? (int)std::max<long long>(1, 3 * slots / 7) : 0;
                    if (a.v.tile_group > 0 && ctx->host_tile_group > 0) a.v.tile_group = ctx->host_tile_group;
                } else {
                    a.v.tile_group = a.v.n_chunks > 1 && ctx->grid_tile_group > 0 ? ctx->grid_tile_group : 0;
                }
                if (int rc = prepare_tickets(ctx, tiles_s, a.v.n_chunks, st, &a.v.tickets)) return n_slabs > 1 ? drain(rc) : rc;
                CU(launch_plan_chunks(t.desc, a.v.n_chunks, t.ns_real, ctr_g, st, /*model=*/zrow ? 4 : (row ? 2 : 1)), "form_factors_grid: chunk planning kernel");
                if (ctx->timing) CU(cudaEventRecord(ctx->ev_m0, st), "form_factors_grid: event");
                CU(zrow ? launch_ff_zrow(t.NS, a, st) : (row ? launch_ff_row(t.NS, a, st) : launch_ff_grid(t.NS, a, st)), "form_factors_grid: kernel");
                if (ctx->timing) {
                    CU(cudaEventRecord(ctx->ev_m1, st), "form_factors_grid: event");
                    CU(cudaEventSynchronize(ctx->ev_m1), "form_factors_grid: event sync");
                    float ms = 0.f;
                    cudaEventElapsedTime(&ms, ctx->ev_m0, ctx->ev_m1);
                    main_ms += ms;
                }
                ctx->st.last_n_chunks = a.v.n_chunks;
                launches += 2;
                if (n_slabs > 1) {
                    const long long plane = (long long)ny * nz;
                    const long long ix0 = (long long)b0 * BXs, ix1 = std::min<long long>((long long)b1 * BXs, nx_eval);
                    cudaError_t e = cudaEventRecord(ctx->ev_slice, st);
                    if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_slice, 0);
                    for (int s = 0; s < t.ns_real && e == cudaSuccess; ++s) {
                        const size_t so = (size_t)(t.s0 + s) * (size_t)n_q;
                        e = cudaMemcpyAsync(out + (so + (size_t)(ix0 * plane)) * 2, dout + (so + (size_t)(ix0 * plane)) * 2,
                                            (size_t)((ix1 - ix0) * plane) * 16, cudaMemcpyDeviceToHost, ctx->copy_stream);
                        if (e == cudaSuccess && sym)       // the mirror slab: ix in [nx - ix1, nx - ix0)
                            e = cudaMemcpyAsync(out + (so + (size_t)((nx - ix1) * plane)) * 2, dout + (so + (size_t)((nx - ix1) * plane)) * 2,
                                                (size_t)((ix1 - ix0) * plane) * 16, cudaMemcpyDeviceToHost, ctx->copy_stream);
                    }
                    if (e != cudaSuccess) return drain(cuda_fail(ctx, e, "form_factors_grid: download slab"));
                }
            }
            if (has_high_classes(ctx->hs)) {
                HighLArgs h = {};
                h.base = t.base; h.desc = t.desc; h.q = nullptr;
                h.qx = dax[0]; h.qy = dax[1]; h.qz = dax[2];
                h.nx = nx; h.ny = ny; h.nz = nz; h.nx_eval = nx_eval; h.sym = sym ? 1 : 0;
                h.ns_real = t.ns_real; h.n_points = (long long)nx_eval * ny * nz; h.n_q = n_q; h.dst = a.v.dst;
                CU(launch_ff_highl(h, st), "form_factors_grid: high-class kernel");
                ++launches;
            }
        }
        ctx->st.last_kernel_launches = launches;
        ctx->grid_eval_points = (double)nx_eval * ny * nz;
        ctx->grid_table_cols = (double)(nx_eval + ny + nz);
        ctx->st.last_grid_symmetric = sym ? 1 : 0;
        ctx->last_grid_w = kWg;
        ctx->last_grid_ctr = ctr_g;
        ctx->last_table_ctr = kCtrTable;
        ctx->st.last_grid_variant = zrow ? 2 : (row ? 1 : 0);
        ctx->st.last_grid_slots = -1.0;            // filled by scarf_get_stats from the kept counts
        if (ctx->timing) {
            CU(cudaEventRecord(ctx->ev1, st), "form_factors_grid: event");
            CU(cudaEventSynchronize(ctx->ev1), "form_factors_grid: event sync");
            float ms = 0.f;
            cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1);
            ctx->st.last_kernel_ms = ms;
            ctx->st.last_main_kernel_ms = main_ms;
        }
        if (out_host) {
            if (n_slabs > 1) CU(cudaStreamSynchronize(ctx->copy_stream), "form_factors_grid: sync copies");
            else if (!out_alias) CU(cudaMemcpyAsync(out, dout, obytes, cudaMemcpyDeviceToHost, st), "form_factors_grid: download out");
            CU(cudaStreamSynchronize(st), "form_factors_grid: sync");
            if (harvest_screen(ctx, true) != SCARF_OK) return SCARF_ECUDA;
            if (ctx->T_bad) return fail(ctx, SCARF_EINVAL, std::string("form_factors_grid: ") + kBadT);
        }
        return SCARF_OK;
    } catch (const std::bad_alloc&) {
        return fail(ctx, SCARF_ENOMEM, "form_factors_grid: out of host memory");
    } catch (...) {
        return fail(ctx, SCARF_EINVAL, "form_factors_grid: unexpected exception");
    }
}

int scarf_form_factors_sph(scarf_ctx* ctx, int32_t n_r, const double* r, int32_t n_theta, const double* cos_theta, int32_t n_phi,
                           double* out)
{
    if (!ctx) return SCARF_EINVAL;
    if (ctx->host_only) return fail(ctx, SCARF_ENODEVICE, "form_factors_sph: host-only context; there is no CPU fallback");
    if (!ctx->have_T) return fail(ctx, SCARF_ESTATE, "form_factors_sph: set_basis and set_transitions first");
    if (n_r < 0 || n_theta < 0 || n_phi < 0) return fail(ctx, SCARF_EINVAL, "form_factors_sph: negative grid size");
    const long long n_dir = (long long)n_theta * n_phi, n_q = n_dir * n_r;
    if (n_q == 0) return SCARF_OK;
    if (!r || !cos_theta || !out) return fail(ctx, SCARF_EINVAL, "form_factors_sph: null r, cos_theta or out");
    if (is_device_ptr(r) || is_device_ptr(cos_theta)) return fail(ctx, SCARF_EINVAL, "form_factors_sph: r and cos_theta must be HOST pointers");
    if (n_dir > 0x7fffffffLL / 4) return fail(ctx, SCARF_EINVAL, "form_factors_sph: too many directions for one call");
    try {
        if (!all_finite(r, (size_t)n_r) || !all_finite(cos_theta, (size_t)n_theta)) return fail(ctx, SCARF_EINVAL, "form_factors_sph: NaN/Inf in r or cos_theta");
        for (int j = 0; j < n_theta; ++j)
            if (std::fabs(cos_theta[j]) > 1.0) return fail(ctx, SCARF_EINVAL, "form_factors_sph: |cos_theta| > 1");
        CU(cudaSetDevice(ctx->device), "form_factors_sph");
        cudaStream_t st = ctx->stream;
        if (harvest_screen(ctx, false) != SCARF_OK) return SCARF_ECUDA;
        if (ctx->T_bad) return fail(ctx, SCARF_EINVAL, std::string("form_factors_sph: ") + kBadT);
        // inversion symmetry: -q of (i, j, k) is the grid point (i, n_theta-1-j, k + n_phi/2) when the theta nodes are antisymmetric
        // bit for bit and n_phi is even
        bool sym = ctx->grid_symmetry != 0 && (n_phi % 2) == 0;
        for (int j = 0; j < n_theta && sym; ++j) sym = cos_theta[j] == -cos_theta[n_theta - 1 - j];
        const int mid = (n_theta % 2) ? n_theta / 2 : -1;
        const int n_dir_eval = sym ? (n_theta / 2) * n_phi + (mid >= 0 ? n_phi / 2 : 0) : (int)n_dir;
        // direction table (cached: rebuilt when the nodes, n_phi or the symmetry decision change); mirror directions are the exact
        // negatives of the evaluated ones, so that the stored conjugate is what the kernel would compute at -q
        const bool cached = ctx->sph_n_phi == n_phi && ctx->sph_sym == (sym ? 1 : 0) && ctx->sph_ct.size() == (size_t)n_theta &&
                            std::memcmp(ctx->sph_ct.data(), cos_theta, (size_t)n_theta * sizeof(double)) == 0;
        std::vector<double> dirs;
        auto build_dirs = [&]() {
            dirs.assign((size_t)n_dir * 3, 0.0);
            const double two_pi = 6.283185307179586476925286766559;
            auto direct = [&](int j, int k) {
                const double c = cos_theta[j], s = std::sqrt(std::max(0.0, 1.0 - c * c)), ph = two_pi * (double)k / (double)n_phi;
                double* o = &dirs[((size_t)j * n_phi + k) * 3];
                o[0] = s * std::cos(ph); o[1] = s * std::sin(ph); o[2] = c;
            };
            for (int j = 0; j < n_theta; ++j)
                for (int k = 0; k < n_phi; ++k) {
                    const bool evaluated = !sym || j < n_theta / 2 || (j == mid && k < n_phi / 2);
                    if (evaluated) direct(j, k);
                }
            if (sym)
                for (int j = 0; j < n_theta; ++j)
                    for (int k = 0; k < n_phi; ++k) {
                        const bool evaluated = j < n_theta / 2 || (j == mid && k < n_phi / 2);
                        if (evaluated) continue;
                        const double* src = &dirs[((size_t)(n_theta - 1 - j) * n_phi + (k + n_phi / 2) % n_phi) * 3];
                        double* o = &dirs[((size_t)j * n_phi + k) * 3];
                        o[0] = -src[0]; o[1] = -src[1]; o[2] = -src[2];
                    }
        };
        if (has_high_classes(ctx->hs)) {
            // pairs with g, h, i shells: the same points as a list through scarf_form_factors (its high-class kernel)
            build_dirs();
            std::vector<double> q((size_t)n_q * 3);
            for (int i = 0; i < n_r; ++i)
                for (long long d = 0; d < n_dir; ++d)
                    for (int c = 0; c < 3; ++c) q[((size_t)i * n_dir + d) * 3 + c] = r[i] * dirs[(size_t)d * 3 + c];
            const int rc = scarf_form_factors(ctx, n_q, q.data(), out);
            if (rc == SCARF_OK) CU(cudaStreamSynchronize(st), "form_factors_sph: sync");      // q dies with this frame
            ctx->st.last_grid_symmetric = 0;
            ctx->st.last_grid_variant = -1;
            return rc;
        }
        CU(ctx->d_axes.ensure((size_t)n_r * sizeof(double)), "form_factors_sph: alloc radii");
        CU(cudaMemcpyAsync(ctx->d_axes.p, r, (size_t)n_r * sizeof(double), cudaMemcpyHostToDevice, st), "form_factors_sph: copy radii");
        if (!cached) {
            build_dirs();
            CU(ctx->d_sph_dirs.ensure(dirs.size() * sizeof(double)), "form_factors_sph: alloc directions");
            CU(cudaMemcpyAsync(ctx->d_sph_dirs.p, dirs.data(), dirs.size() * sizeof(double), cudaMemcpyHostToDevice, st), "form_factors_sph: copy directions");
            ctx->sph_ct.assign(cos_theta, cos_theta + n_theta);
            ctx->sph_n_phi = n_phi;
            ctx->sph_sym = sym ? 1 : 0;
        }
        const int n_rbox = (n_r + kSphBR - 1) / kSphBR, n_dbox = (n_dir_eval + kSphBD - 1) / kSphBD;
        const long long n_tiles = (long long)n_rbox * n_dbox;
        const size_t obytes = (size_t)ctx->n_states * (size_t)n_q * 2 * sizeof(double);
        double* dout = out;
        const bool out_host = !is_device_ptr(out);
        if (out_host) {
            CU(ctx->d_out.ensure(obytes), "form_factors_sph: alloc out");
            dout = static_cast<double*>(ctx->d_out.p);
        }
        // (No direct stores into a pinned host `out` here, unlike scarf_form_factors_grid: a lane owns a radius, so the kernel writes
        // 16-byte pieces at a stride of n_theta n_phi 16 B; over PCIe that took 54 ms on config 5 against 34.8 ms with the copy.)
        if (ctx->timing) CU(cudaEventRecord(ctx->ev0, st), "form_factors_sph: event");
        int launches = 0;
        double main_ms = 0.0;
        if (ctx->qcut_dev) {
            CU(cudaMemsetAsync(ctx->d_work.p, 0, kNClasses * sizeof(unsigned long long), st), "form_factors_sph: clear counters");
            ctx->last_q_tiles = (double)n_tiles; ctx->last_ctr = kCtrSph; ctx->last_was_grid = true; ctx->last_grid_w = kWSph; ctx->work_pending = true;
        }
        const long long n_rows = (long long)ctx->hs.pairs.size();    // prescreened pairs: an upper bound of the kept count
        for (const TileStream& t : ctx->tiles) {
            SphArgs a = {};
            const size_t tab_elems = (size_t)std::max<long long>(1, n_rows) * (size_t)n_rbox * kSphBR;
            CU(ctx->d_tab.ensure(tab_elems * sizeof(double)), "form_factors_sph: alloc table");
            double* te = static_cast<double*>(ctx->d_tab.p);
            a.v.base = t.base;
            a.v.desc = t.desc;
            a.v.n_q = n_q;
            a.v.n_tiles = (int)n_tiles;
            a.v.ns_real = t.ns_real;
            a.v.dst = dout + (size_t)t.s0 * n_q * 2;
            a.v.qcut = ctx->qcut_dev;
            a.v.work = ctx->qcut_dev ? static_cast<unsigned long long*>(ctx->d_work.p) : nullptr;
            a.r = static_cast<const double*>(ctx->d_axes.p);
            a.dirs = static_cast<const double*>(ctx->d_sph_dirs.p);
            a.n_r = n_r; a.n_theta = n_theta; a.n_phi = n_phi;
            a.n_dir_eval = n_dir_eval;
            a.n_rbox = n_rbox; a.n_dbox = n_dbox;
            a.sym = sym ? 1 : 0;
            a.te = te;
            a.n_rows = n_rows;
            CU(launch_sph_table(a, te, st), "form_factors_sph: table kernel");
            a.v.n_chunks = choose_chunks(ctx, n_tiles, kCtrSph, t.ns_real, ctx->n_chunks_opt);
            if (int rc = prepare_tickets(ctx, n_tiles, a.v.n_chunks, st, &a.v.tickets)) return rc;
            CU(launch_plan_chunks(t.desc, a.v.n_chunks, t.ns_real, kCtrSph, st, /*model=*/3), "form_factors_sph: chunk planning kernel");
            if (ctx->timing) CU(cudaEventRecord(ctx->ev_m0, st), "form_factors_sph: event");
            CU(launch_ff_sph(t.NS, a, st), "form_factors_sph: kernel");
            if (ctx->timing) {
                CU(cudaEventRecord(ctx->ev_m1, st), "form_factors_sph: event");
                CU(cudaEventSynchronize(ctx->ev_m1), "form_factors_sph: event sync");
                float ms = 0.f;
                cudaEventElapsedTime(&ms, ctx->ev_m0, ctx->ev_m1);
                main_ms += ms;
            }
            ctx->st.last_n_chunks = a.v.n_chunks;
            launches += 3;
        }
        ctx->st.last_kernel_launches = launches;
        ctx->grid_eval_points = (double)n_dir_eval * n_r;
        ctx->grid_table_cols = (double)n_r;
        ctx->st.last_grid_symmetric = sym ? 1 : 0;
        ctx->st.last_grid_variant = 3;
        ctx->last_grid_w = kWSph;
        ctx->last_grid_ctr = kCtrSph;
        ctx->last_table_ctr = kCtrSphTable;
        ctx->st.last_grid_slots = -1.0;            // filled by scarf_get_stats from the kept counts
        if (ctx->timing) {
            CU(cudaEventRecord(ctx->ev1, st), "form_factors_sph: event");
            CU(cudaEventSynchronize(ctx->ev1), "form_factors_sph: event sync");
            float ms = 0.f;
            cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1);
            ctx->st.last_kernel_ms = ms;
            ctx->st.last_main_kernel_ms = main_ms;
        }
        if (out_host) {
            CU(cudaMemcpyAsync(out, dout, obytes, cudaMemcpyDeviceToHost, st), "form_factors_sph: download out");
            CU(cudaStreamSynchronize(st), "form_factors_sph: sync");
            if (harvest_screen(ctx, true) != SCARF_OK) return SCARF_ECUDA;
            if (ctx->T_bad) return fail(ctx, SCARF_EINVAL, std::string("form_factors_sph: ") + kBadT);
        }
        return SCARF_OK;
    } catch (const std::bad_alloc&) {
        return fail(ctx, SCARF_ENOMEM, "form_factors_sph: out of host memory");
    } catch (...) {
        return fail(ctx, SCARF_EINVAL, "form_factors_sph: unexpected exception");
    }
}

int scarf_separable_integral(scarf_ctx* ctx, int32_t nx, const double* qx, const double* fx, int32_t ny, const double* qy,
                             const double* gy, int32_t nz, const double* qz, const double* hz, double* out)
{
    if (!ctx) return SCARF_EINVAL;
    if (ctx->host_only) return fail(ctx, SCARF_ENODEVICE, "separable_integral: host-only context; there is no CPU fallback");
    if (!ctx->have_T) return fail(ctx, SCARF_ESTATE, "separable_integral: set_basis and set_transitions first");
    if (nx < 1 || ny < 1 || nz < 1 || !qx || !fx || !qy || !gy || !qz || !hz || !out)
        return fail(ctx, SCARF_EINVAL, "separable_integral: empty axis or null pointer");
    const double* in[6] = {qx, qy, qz, fx, gy, hz};
    const int len[6] = {nx, ny, nz, nx, ny, nz};
    for (int k = 0; k < 6; ++k)
        if (!all_finite(in[k], (size_t)len[k])) return fail(ctx, SCARF_EINVAL, "separable_integral: NaN/Inf in an axis or weight array");
    try {
        CU(cudaSetDevice(ctx->device), "separable_integral");
        cudaStream_t st = ctx->stream;
        CU(ctx->d_axes.ensure(2 * ((size_t)nx + ny + nz) * sizeof(double)), "separable_integral: alloc axes");
        double* d[6];
        size_t off = 0;
        for (int k = 0; k < 6; ++k) {
            d[k] = static_cast<double*>(ctx->d_axes.p) + off;
            off += (size_t)len[k];
            CU(cudaMemcpyAsync(d[k], in[k], (size_t)len[k] * sizeof(double), cudaMemcpyHostToDevice, st), "separable_integral: upload");
        }
        const int per_block = 64;
        int launches = 0;
        const long long n_rows = (long long)ctx->hs.pairs.size();   // upper bound of the kept count (the kernels read the real one)
        for (const TileStream& t : ctx->tiles) {
            for (int k = 0; k < t.ns_real; ++k) out[2 * (t.s0 + k)] = out[2 * (t.s0 + k) + 1] = 0.0;
            if (n_rows == 0) continue;
            GridArgs a = {};
            a.v.base = t.base;
            a.v.desc = t.desc;
            a.v.ns_real = t.ns_real;
            a.qx = d[0]; a.qy = d[1]; a.qz = d[2];
            a.nx = nx; a.ny = ny; a.nz = nz;
            a.n_rows = n_rows;
            const size_t n_blocks = (size_t)((n_rows + per_block - 1) / per_block);
            const size_t mom_bytes = (size_t)n_rows * 3 * kNClasses * 16, part_bytes = n_blocks * 16 * 16;
            CU(ctx->d_tab.ensure(mom_bytes + part_bytes), "separable_integral: alloc scratch");
            double* mom = static_cast<double*>(ctx->d_tab.p);
            double* part = mom + mom_bytes / 8;
            CU(launch_separable(a, d[3], d[4], d[5], mom, part, per_block, st), "separable_integral: kernels");
            launches += 2;
            std::vector<double> hp(n_blocks * 32);
            CU(cudaMemcpyAsync(hp.data(), part, part_bytes, cudaMemcpyDeviceToHost, st), "separable_integral: download");
            CU(cudaStreamSynchronize(st), "separable_integral: sync");
            for (size_t b = 0; b < n_blocks; ++b)           // block order: deterministic
                for (int k = 0; k < t.ns_real; ++k) {
                    out[2 * (t.s0 + k)] += hp[(b * 16 + k) * 2];
                    out[2 * (t.s0 + k) + 1] += hp[(b * 16 + k) * 2 + 1];
                }
        }
        ctx->st.last_kernel_launches = launches;
        CU(cudaStreamSynchronize(st), "separable_integral: sync");
        return SCARF_OK;
    } catch (const std::bad_alloc&) {
        return fail(ctx, SCARF_ENOMEM, "separable_integral: out of host memory");
    } catch (...) {
        return fail(ctx, SCARF_EINVAL, "separable_integral: unexpected exception");
    }
}

int scarf_angular_moments(scarf_ctx* ctx, int32_t n_states, int32_t n_r, int32_t n_theta, const double* cos_theta,
                          const double* w_theta, int32_t n_phi, int32_t l_max, const double* f, double* R_out, double* f2_out)
{
    if (!ctx) return SCARF_EINVAL;
    if (ctx->host_only) return fail(ctx, SCARF_ENODEVICE, "angular_moments: host-only context; there is no CPU fallback");
    if (n_states < 0 || n_r < 0 || n_theta < 1 || n_phi < 1 || l_max < 0)
        return fail(ctx, SCARF_EINVAL, "angular_moments: bad shape");
    if (l_max > 64) return fail(ctx, SCARF_EINVAL, "angular_moments: l_max > 64");
    if (n_phi > 2048) return fail(ctx, SCARF_EINVAL, "angular_moments: n_phi > 2048");
    if (n_phi < 2 * l_max + 1) return fail(ctx, SCARF_EINVAL, "angular_moments: n_phi must be >= 2 l_max + 1 (phi aliasing)");
    const long long n_sr = (long long)n_states * n_r;
    if (n_sr == 0) return SCARF_OK;
    if (!cos_theta || !w_theta || !f || !R_out) return fail(ctx, SCARF_EINVAL, "angular_moments: null pointer");
    if (!all_finite(cos_theta, (size_t)n_theta) || !all_finite(w_theta, (size_t)n_theta))
        return fail(ctx, SCARF_EINVAL, "angular_moments: NaN/Inf in the theta nodes or weights");
    for (int j = 0; j < n_theta; ++j)
        if (std::fabs(cos_theta[j]) > 1.0) return fail(ctx, SCARF_EINVAL, "angular_moments: |cos theta| > 1");
    try {
        CU(cudaSetDevice(ctx->device), "angular_moments");
        cudaStream_t st = ctx->stream;
        const long long n_rows = n_sr * n_theta;
        const int n_m = 2 * l_max + 1, nlm = (l_max + 1) * (l_max + 1);
        // host tables, cached in the context: rebuilt and uploaded only when the nodes, weights, n_phi or l_max change
        AngularCache& ac = ctx->ang;
        const bool same = ac.valid && ac.n_phi == n_phi && ac.l_max == l_max && (int)ac.ct.size() == n_theta &&
                          std::memcmp(ac.ct.data(), cos_theta, sizeof(double) * (size_t)n_theta) == 0 &&
                          std::memcmp(ac.wt.data(), w_theta, sizeof(double) * (size_t)n_theta) == 0;
        if (!same) {
            ac.valid = false;
            ac.ct.assign(cos_theta, cos_theta + n_theta);
            ac.wt.assign(w_theta, w_theta + n_theta);
            ac.n_phi = n_phi; ac.l_max = l_max;
            angular_host_tables(l_max, n_theta, cos_theta, w_theta, n_phi, ac.Yw, ac.tw);
            angular_fragment_table(l_max, n_phi, ac.Bf, ac.n_nt, ac.n_ks);
            angular_transpose_table(l_max, n_theta, ac.Yw, ac.YwT);
            ac.chunk_bytes = angular_chunk_table(l_max, n_theta, ac.Yw, ac.YwC);
            // device layout (tw, Bf, YwT, YwC have even lengths: every block stays 16-byte aligned): [tw | Bf | YwT | YwC | Yw | w_theta]
            const size_t tab_doubles = ac.tw.size() + ac.Bf.size() + ac.YwT.size() + ac.YwC.size() + ac.Yw.size() + (size_t)n_theta;
            CU(ctx->d_ang_tab.ensure(tab_doubles * sizeof(double)), "angular_moments: alloc tables");
            double* base = static_cast<double*>(ctx->d_ang_tab.p);
            // pageable sources are staged by the runtime before each call returns; the cached vectors outlive the copies anyway
            CU(cudaMemcpyAsync(base, ac.tw.data(), ac.tw.size() * sizeof(double), cudaMemcpyHostToDevice, st), "angular_moments: upload");
            CU(cudaMemcpyAsync(base + ac.tw.size(), ac.Bf.data(), ac.Bf.size() * sizeof(double), cudaMemcpyHostToDevice, st), "angular_moments: upload");
            double* p = base + ac.tw.size() + ac.Bf.size();
            CU(cudaMemcpyAsync(p, ac.YwT.data(), ac.YwT.size() * sizeof(double), cudaMemcpyHostToDevice, st), "angular_moments: upload");
            p += ac.YwT.size();
            CU(cudaMemcpyAsync(p, ac.YwC.data(), ac.YwC.size() * sizeof(double), cudaMemcpyHostToDevice, st), "angular_moments: upload");
            p += ac.YwC.size();
            CU(cudaMemcpyAsync(p, ac.Yw.data(), ac.Yw.size() * sizeof(double), cudaMemcpyHostToDevice, st), "angular_moments: upload");
            p += ac.Yw.size();
            CU(cudaMemcpyAsync(p, w_theta, (size_t)n_theta * sizeof(double), cudaMemcpyHostToDevice, st), "angular_moments: upload");
            ac.valid = true;
        }
        double* dtw = static_cast<double*>(ctx->d_ang_tab.p);
        double* dBf = dtw + ac.tw.size();
        double* dYwT = dBf + ac.Bf.size();
        double* dYwC = dYwT + ac.YwT.size();
        double* dYw = dYwC + ac.YwC.size();
        double* dw = dYw + ac.Yw.size();
        const size_t fbytes = (size_t)n_rows * n_phi * 2 * sizeof(double);
        const double* df = f;
        const bool f_host = !is_device_ptr(f);
        if (f_host) {
            CU(ctx->d_ang_in.ensure(fbytes), "angular_moments: alloc f");
            CU(cudaMemcpyAsync(ctx->d_ang_in.p, f, fbytes, cudaMemcpyHostToDevice, st), "angular_moments: upload f");
            df = static_cast<const double*>(ctx->d_ang_in.p);
        }
        const size_t rbytes = (size_t)n_sr * nlm * 2 * sizeof(double), f2bytes = (size_t)n_sr * sizeof(double);
        const bool R_host = !is_device_ptr(R_out), f2_host = f2_out && !is_device_ptr(f2_out);
        double *dR = R_out, *df2 = f2_out;
        if (R_host || f2_host) {
            CU(ctx->d_ang_out.ensure(rbytes + f2bytes), "angular_moments: alloc out");
            if (R_host) dR = static_cast<double*>(ctx->d_ang_out.p);
            if (f2_host) df2 = static_cast<double*>(ctx->d_ang_out.p) + (size_t)n_sr * nlm * 2;
        }
        if (ctx->timing) CU(cudaEventRecord(ctx->ev0, st), "angular_moments: event");
        // route: fused tensor-core kernel (F rows of one (state, r) in shared memory); for shapes whose F does not fit, the
        // same kernel writes F to global memory and legendre_kernel finishes; if even the cos/sin fragments do not fit, SIMT
        const size_t smem_fused = angular_fused_smem(n_theta, l_max, ac.n_nt, ac.n_ks, true);
        const size_t smem_unfused = angular_fused_smem(n_theta, l_max, ac.n_nt, ac.n_ks, false);
        if (ctx->angular_variant == 1 && smem_fused <= (size_t)kAngularMaxSmem) {
            CU(launch_angular_fused(df, dBf, dYwT, dw, n_sr, n_theta, n_phi, l_max, ac.n_nt, ac.n_ks, dR, df2, nullptr, nullptr, dYwC, ac.chunk_bytes, st),
               "angular_moments: fused kernel");
            ctx->st.last_kernel_launches = 1;
        } else {
            // scratch: F [n_rows][n_m] complex, rowsum2 [n_rows]
            CU(ctx->d_ang_F.ensure(((size_t)n_rows * n_m * 2 + (size_t)n_rows) * sizeof(double)), "angular_moments: alloc scratch");
            double* dF = static_cast<double*>(ctx->d_ang_F.p);
            double* drow2 = dF + (size_t)n_rows * n_m * 2;
            if (ctx->angular_variant == 1 && smem_unfused <= (size_t)kAngularMaxSmem)
                CU(launch_angular_fused(df, dBf, dYwT, dw, n_sr, n_theta, n_phi, l_max, ac.n_nt, ac.n_ks, nullptr, nullptr, dF, drow2, nullptr, 0, st),
                   "angular_moments: phi kernel (DMMA)");
            else
                CU(launch_phi_dft(df, dtw, n_rows, n_phi, l_max, dF, drow2, st), "angular_moments: phi kernel");
            CU(launch_legendre(dF, drow2, dYw, dw, n_sr, n_theta, l_max, dR, df2, st), "angular_moments: legendre kernel");
            ctx->st.last_kernel_launches = 2;
        }
        if (ctx->timing) {
            CU(cudaEventRecord(ctx->ev1, st), "angular_moments: event");
            CU(cudaEventSynchronize(ctx->ev1), "angular_moments: event sync");
            float ms = 0.f;
            cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1);
            ctx->st.last_kernel_ms = ms;
        }
        if (R_host) CU(cudaMemcpyAsync(R_out, dR, rbytes, cudaMemcpyDeviceToHost, st), "angular_moments: download R");
        if (f2_host) CU(cudaMemcpyAsync(f2_out, df2, f2bytes, cudaMemcpyDeviceToHost, st), "angular_moments: download f2");
        // host buffers: the copies must have finished before the caller reads / reuses them; all-device calls stay asynchronous
        if (R_host || f2_host || f_host) CU(cudaStreamSynchronize(st), "angular_moments: sync");
        return SCARF_OK;
    } catch (const std::bad_alloc&) {
        return fail(ctx, SCARF_ENOMEM, "angular_moments: out of host memory");
    } catch (...) {
        return fail(ctx, SCARF_EINVAL, "angular_moments: unexpected exception");
    }
}

int scarf_abs2(scarf_ctx* ctx, int64_t n, const double* f, double* out)
{
    if (!ctx) return SCARF_EINVAL;
    if (ctx->host_only) return fail(ctx, SCARF_ENODEVICE, "abs2: host-only context; there is no CPU fallback");
    if (n < 0) return fail(ctx, SCARF_EINVAL, "abs2: n < 0");
    if (n == 0) return SCARF_OK;
    if (!f || !out) return fail(ctx, SCARF_EINVAL, "abs2: null pointer");
    CU(cudaSetDevice(ctx->device), "abs2");
    cudaStream_t st = ctx->stream;
    const bool f_host = !is_device_ptr(f), o_host = !is_device_ptr(out);
    const double* df = f;
    double* dout = out;
    if (f_host) {
        CU(ctx->d_ang_in.ensure((size_t)n * 16), "abs2: alloc");
        CU(cudaMemcpyAsync(ctx->d_ang_in.p, f, (size_t)n * 16, cudaMemcpyHostToDevice, st), "abs2: upload");
        df = static_cast<const double*>(ctx->d_ang_in.p);
    }
    if (o_host) {
        CU(ctx->d_ang_out.ensure((size_t)n * 8), "abs2: alloc");
        dout = static_cast<double*>(ctx->d_ang_out.p);
    }
    CU(launch_abs2(df, n, dout, st), "abs2: kernel");
    if (o_host) CU(cudaMemcpyAsync(out, dout, (size_t)n * 8, cudaMemcpyDeviceToHost, st), "abs2: download");
    if (o_host || f_host) CU(cudaStreamSynchronize(st), "abs2: sync");
    return SCARF_OK;
}

/* Eq. (81)-(82) PAPER.md:591-596: least-squares fit  <|f_s|^2>_Omega(q) ~ A + B q^2 + C q^4  over the points with
 * |q| <= q_max (all points if q_max <= 0).  HOST arrays.  Normal equations in the scaled variable x = (q / q_ref)^2,
 * q_ref = the largest |q| used, solved by Gaussian elimination with partial pivoting. */
int scarf_oscillator_fit(int32_t n_states, int32_t n_r, const double* q_abs, const double* f2, double q_max, double* coef_out)
{
    if (n_states < 0 || n_r < 1 || !q_abs || !f2 || !coef_out) return SCARF_EINVAL;
    if (!all_finite(q_abs, (size_t)n_r) || !all_finite(f2, (size_t)n_states * n_r) || !std::isfinite(q_max)) return SCARF_EINVAL;
    std::vector<int> use;
    double q_ref = 0.0;
    for (int i = 0; i < n_r; ++i)
        if (q_max <= 0.0 || std::fabs(q_abs[i]) <= q_max) {
            use.push_back(i);
            q_ref = std::max(q_ref, std::fabs(q_abs[i]));
        }
    if (use.size() < 3 || !(q_ref > 0.0)) return SCARF_EINVAL;    // three unknowns
    for (int s = 0; s < n_states; ++s) {
        double N[3][4] = {};
        for (int i : use) {
            const double x = (q_abs[i] / q_ref) * (q_abs[i] / q_ref), b[3] = {1.0, x, x * x}, y = f2[(size_t)s * n_r + i];
            for (int r = 0; r < 3; ++r) {
                for (int c = 0; c < 3; ++c) N[r][c] += b[r] * b[c];
                N[r][3] += b[r] * y;
            }
        }
        for (int c = 0; c < 3; ++c) {
            int piv = c;
            for (int r = c + 1; r < 3; ++r)
                if (std::fabs(N[r][c]) > std::fabs(N[piv][c])) piv = r;
            if (!(std::fabs(N[piv][c]) > 0.0)) return SCARF_EINVAL;    // fewer than three distinct |q|
            for (int k = 0; k < 4; ++k) std::swap(N[c][k], N[piv][k]);
            for (int r = 0; r < 3; ++r)
                if (r != c) {
                    const double m = N[r][c] / N[c][c];
                    for (int k = c; k < 4; ++k) N[r][k] -= m * N[c][k];
                }
        }
        coef_out[3 * s + 0] = N[0][3] / N[0][0];
        coef_out[3 * s + 1] = N[1][3] / N[1][1] / (q_ref * q_ref);
        coef_out[3 * s + 2] = N[2][3] / N[2][2] / (q_ref * q_ref * q_ref * q_ref);
    }
    return SCARF_OK;
}

int scarf_fft_form_factors(scarf_ctx* ctx, int32_t nx, int32_t ny, int32_t nz, const double* x_min, const double* box_len,
                           double* out)
{
    if (!ctx) return SCARF_EINVAL;
    if (ctx->host_only) return fail(ctx, SCARF_ENODEVICE, "fft_form_factors: host-only context; there is no CPU fallback");
    if (!ctx->have_T || !ctx->Tc_dev) return fail(ctx, SCARF_ESTATE, "fft_form_factors: set_basis and set_transitions first");
    if (nx < 1 || ny < 1 || nz < 1 || !x_min || !box_len || !out) return fail(ctx, SCARF_EINVAL, "fft_form_factors: bad grid or null pointer");
    for (int k = 0; k < 3; ++k)
        if (!std::isfinite(x_min[k]) || !std::isfinite(box_len[k]) || !(box_len[k] > 0))
            return fail(ctx, SCARF_EINVAL, "fft_form_factors: box lengths must be finite and > 0");
    try {
        CU(cudaSetDevice(ctx->device), "fft_form_factors");
        cudaStream_t st = ctx->stream;
        const HostSetup& hs = ctx->hs;
        FftGrid g = {};
        g.nx = nx; g.ny = ny; g.nz = nz;
        g.P = (long long)nx * ny * nz;
        for (int k = 0; k < 3; ++k) { g.xmin[k] = x_min[k]; g.len[k] = box_len[k]; }
        const int nbf_pad = (hs.nbf + 7) & ~7;
        // default route: orbital values evaluated per point tile inside the density kernel (no V buffer); the V-buffer routes
        // remain for bases whose tile does not fit in shared memory and as second implementations (variants 2 and 0)
        const bool fused = ctx->fft_density_variant == 1 && density_fused_fits(nbf_pad);
        const size_t vbytes = fused ? 0 : (size_t)hs.nbf * (size_t)((g.P + 7) / 8 * 8) * sizeof(double);
        const size_t fbytes = (size_t)ctx->n_states * (size_t)g.P * 2 * sizeof(double);
        if ((double)vbytes + 2.0 * (double)fbytes > 64e9) return fail(ctx, SCARF_ENOMEM, "fft_form_factors: grid needs more than 64 GB of scratch");
        // primitive shells and the first primitive of every contracted shell
        std::vector<int> first;
        for (size_t i = 0; i < hs.prim.size(); ++i)
            if (i == 0 || hs.prim[i].shell != hs.prim[i - 1].shell) first.push_back((int)i);
        const int n_sh = (int)first.size();
        first.push_back((int)hs.prim.size());
        const size_t pbytes = hs.prim.size() * sizeof(PrimShell);
        CU(ctx->d_prim.ensure(pbytes + first.size() * sizeof(int) + 64), "fft_form_factors: alloc basis");
        char* pb = static_cast<char*>(ctx->d_prim.p);
        CU(cudaMemcpyAsync(pb, hs.prim.data(), pbytes, cudaMemcpyHostToDevice, st), "fft_form_factors: upload basis");
        CU(cudaMemcpyAsync(pb + pbytes, first.data(), first.size() * sizeof(int), cudaMemcpyHostToDevice, st), "fft_form_factors: upload basis");
        if (!fused) CU(ctx->d_V.ensure(vbytes), "fft_form_factors: alloc orbital values");
        CU(ctx->d_fft.ensure(fbytes), "fft_form_factors: alloc transform buffer");
        const bool out_host = !is_device_ptr(out);
        double* dout = out;
        if (out_host) {
            CU(ctx->d_out.ensure(fbytes), "fft_form_factors: alloc out");
            dout = static_cast<double*>(ctx->d_out.p);
        }
        if (ctx->timing) CU(cudaEventRecord(ctx->ev0, st), "fft_form_factors: event");
        double* dV = fused ? nullptr : static_cast<double*>(ctx->d_V.p);
        double* dF = static_cast<double*>(ctx->d_fft.p);
        const PrimShell* dprim = reinterpret_cast<const PrimShell*>(pb);
        const int* dfirst = reinterpret_cast<const int*>(pb + pbytes);
        int launches = 0;
        if (!fused) {
            CU(launch_orbitals(dprim, dfirst, n_sh, hs.nbf, g, dV, st), "fft_form_factors: orbital kernel");
            ++launches;
        }
        for (int s0 = 0; s0 < ctx->n_states; s0 += kMaxStateTile) {
            const int ns_t = std::min(kMaxStateTile, ctx->n_states - s0);
            if (ctx->fft_density_variant == 0) {
                CU(launch_density(dV, ctx->Tc_dev, hs.nbf, g.P, s0, ns_t, ctx->prefactor, dF, st), "fft_form_factors: density kernel");
                ++launches;
            } else {
                CU(ctx->d_Csym.ensure((size_t)kMaxStateTile * nbf_pad * nbf_pad * sizeof(double)), "fft_form_factors: alloc C");
                double* dC = static_cast<double*>(ctx->d_Csym.p);
                if (fused) {
                    CU(launch_symmetrize(ctx->Tc_dev, dC, hs.nbf, nbf_pad, s0, ns_t, st), "fft_form_factors: symmetrize kernel");
                    CU(launch_density_fused(dprim, dfirst, n_sh, g, dC, hs.nbf, nbf_pad, s0, ns_t, ctx->prefactor, dF, st),
                       "fft_form_factors: fused density kernel (DMMA)");
                } else
                    CU(launch_density_mma(dV, ctx->Tc_dev, dC, hs.nbf, nbf_pad, g.P, s0, ns_t, ctx->prefactor, dF, st),
                       "fft_form_factors: density kernel (DMMA)");
                launches += 2;
            }
        }
        CU(cudaStreamSynchronize(st), "fft_form_factors: sync");   // `first` (pageable) goes out of scope; cuFFT plans below
        // Parseval check (Eq. 75), option "check_parseval": V_pix sum_abc |Phi|^2 now, (1 / V_box) sum_q |f|^2 after the transform
        double* dpar = nullptr;
        const double vbox = box_len[0] * box_len[1] * box_len[2];
        if (ctx->check_parseval) {
            CU(ctx->d_parseval.ensure(((size_t)ctx->n_states * 2 + (size_t)ctx->n_states * 256) * sizeof(double)), "fft_form_factors: alloc sums");
            dpar = static_cast<double*>(ctx->d_parseval.p);
            CU(launch_sumsq(dF, g.P, ctx->n_states, vbox / (double)g.P, dpar + 2 * ctx->n_states, dpar, 2, 0, st), "fft_form_factors: Parseval sum");
        }
        const int frc = cufft_inverse_batch(ctx->fft_plan, dF, nx, ny, nz, ctx->n_states, st);
        if (frc < 0) return fail(ctx, SCARF_ECUDA, "fft_form_factors: the cuFFT library (libcufft.so.11) could not be loaded");
        if (frc > 0) return fail(ctx, frc == 2 ? SCARF_ENOMEM : SCARF_ECUDA, "fft_form_factors: cuFFT error " + std::to_string(frc));
        CU(launch_fft_post(dF, g, ctx->n_states, dout, st), "fft_form_factors: post kernel");
        if (dpar) {
            CU(launch_sumsq(dout, g.P, ctx->n_states, 1.0 / vbox, dpar + 2 * ctx->n_states, dpar, 2, 1, st), "fft_form_factors: Parseval sum");
            ctx->parseval_states = ctx->n_states;
            launches += 4;
        } else
            ctx->parseval_states = 0;
        ctx->st.last_kernel_launches = launches + 1;
        if (ctx->timing) {
            CU(cudaEventRecord(ctx->ev1, st), "fft_form_factors: event");
            CU(cudaEventSynchronize(ctx->ev1), "fft_form_factors: event sync");
            float ms = 0.f;
            cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1);
            ctx->st.last_kernel_ms = ms;
        }
        if (out_host) {
            CU(cudaMemcpyAsync(out, dout, fbytes, cudaMemcpyDeviceToHost, st), "fft_form_factors: download out");
            CU(cudaStreamSynchronize(st), "fft_form_factors: sync");
        }
        return SCARF_OK;
    } catch (const std::bad_alloc&) {
        return fail(ctx, SCARF_ENOMEM, "fft_form_factors: out of host memory");
    } catch (...) {
        return fail(ctx, SCARF_EINVAL, "fft_form_factors: unexpected exception");
    }
}

int scarf_fft_parseval(scarf_ctx* ctx, double* out_host)
{
    if (!ctx || !out_host) return SCARF_EINVAL;
    if (ctx->host_only) return fail(ctx, SCARF_ENODEVICE, "fft_parseval: host-only context");
    if (ctx->parseval_states <= 0) return fail(ctx, SCARF_ESTATE, "fft_parseval: set option check_parseval = 1 and call scarf_fft_form_factors first");
    CU(cudaSetDevice(ctx->device), "fft_parseval");
    CU(cudaMemcpyAsync(out_host, ctx->d_parseval.p, (size_t)ctx->parseval_states * 2 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream),
       "fft_parseval: download");
    CU(cudaStreamSynchronize(ctx->stream), "fft_parseval: sync");
    return SCARF_OK;
}

int scarf_get_stats(scarf_ctx* ctx, scarf_stats* out)
{
    if (!ctx || !out) return SCARF_EINVAL;
    if (!ctx->host_only && ctx->screen_pending) {         // the kept counts come back lazily: wait for them here
        cudaSetDevice(ctx->device);
        const int rc = harvest_screen(ctx, true);
        if (rc != SCARF_OK) return rc;
    }
    if (ctx->st.last_grid_slots < 0.0 && !ctx->screen_pending) {
        double slots = 0.0, tab = 0.0;
        const double nt = (double)ctx->tiles.size();
        for (int c = 0; c < kNClasses; ++c) {
            slots += (double)ctx->st.pairs_kept_per_class[c] * ctx->grid_eval_points * ((double)ctx->n_states * (ctx->last_grid_w ? ctx->last_grid_w : kWGrid)[c] + nt * ctx->last_grid_ctr);
            tab += (double)ctx->st.pairs_kept_per_class[c] * nt * ctx->grid_table_cols * ctx->last_table_ctr;
        }
        ctx->st.last_grid_slots = slots + tab;
        ctx->st.last_grid_kernel_slots = slots;
    }
    if (!ctx->host_only && ctx->qcut_dev && !ctx->screen_pending) {
        const double np_all = (double)std::max<size_t>(1, ctx->hs.pairs.size());
        ctx->st.adaptive_bound = (double)ctx->st.n_pairs_kept * ctx->adaptive_tol * ctx->h_screen->sum_bound / np_all;
        if (ctx->work_pending) {                                  // records evaluated per class by the last S4 call
            unsigned long long wk[kNClasses] = {};
            cudaSetDevice(ctx->device);
            if (cudaMemcpyAsync(wk, ctx->d_work.p, sizeof wk, cudaMemcpyDeviceToHost, ctx->stream) == cudaSuccess &&
                cudaStreamSynchronize(ctx->stream) == cudaSuccess) {
                const double nt = (double)std::max<size_t>(1, ctx->tiles.size());
                double done = 0.0, full = 0.0;
                for (int c = 0; c <= kFastMaxClass; ++c) {
                    const double w = (double)ctx->n_states / nt * (ctx->last_was_grid ? (ctx->last_grid_w ? ctx->last_grid_w : kWGrid)[c] : kW[c]) + ctx->last_ctr;
                    done += (double)wk[c] * w;
                    full += (double)ctx->st.pairs_kept_per_class[c] * ctx->last_q_tiles * nt * w;
                }
                ctx->st.last_adaptive_work_fraction = full > 0.0 ? done / full : 1.0;
                ctx->work_pending = false;
            } else
                cudaGetLastError();
        }
    }
    *out = ctx->st;
    if (ctx->T_bad) return fail(ctx, SCARF_EINVAL, std::string("get_stats: ") + kBadT);
    return SCARF_OK;
}

const char* scarf_last_error(const scarf_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int scarf_fp64_peak(int device, double* dfma_per_s, double* sm_clock_mhz)
{
    if (!dfma_per_s || !sm_clock_mhz) return SCARF_EINVAL;
    int n = 0;
    if (cudaGetDeviceCount(&n) != cudaSuccess || device < 0 || device >= n) {
        cudaGetLastError();
        return SCARF_ENODEVICE;
    }
    if (cudaSetDevice(device) != cudaSuccess) return SCARF_ECUDA;
    return run_fp64_peak(dfma_per_s, sm_clock_mhz) == cudaSuccess ? SCARF_OK : SCARF_ECUDA;
}

int scarf_host_hermite_E(int la, int lb, double alpha, double beta, double Ax, double Bx, double* E_out)
{
    if (la < 0 || lb < 0 || la > kMaxL || lb > kMaxL || !(alpha > 0) || !(beta > 0) || !E_out) return SCARF_EINVAL;
    const double p = alpha + beta, P = (alpha * Ax + beta * Bx) / p;
    hermite_E_axis(la, lb, p, P - Ax, P - Bx, std::exp(-alpha * beta / p * (Ax - Bx) * (Ax - Bx)), E_out);
    return SCARF_OK;
}

int scarf_host_ylm_table(int l_max, int n_theta, const double* cos_theta, const double* w_theta, double* Yw_out)
{
    if (l_max < 0 || l_max > 64 || n_theta < 1 || !cos_theta || !w_theta || !Yw_out) return SCARF_EINVAL;
    for (int j = 0; j < n_theta; ++j)
        if (!(std::fabs(cos_theta[j]) <= 1.0)) return SCARF_EINVAL;
    std::vector<double> Yw, tw;
    angular_host_tables(l_max, n_theta, cos_theta, w_theta, 1, Yw, tw);
    std::memcpy(Yw_out, Yw.data(), Yw.size() * sizeof(double));
    return SCARF_OK;
}

int scarf_host_shell_norms(int l, int nprim, const double* exponents, const double* coeffs, double* c_out)
{
    if (!exponents || !coeffs || !c_out || l < 0 || l > kMaxL || nprim < 1) return SCARF_EINVAL;
    std::vector<double> cp((size_t)nprim);
    int rc = shell_coefficients(l, nprim, exponents, coeffs, cp.data());
    if (rc != SCARF_OK) return rc;
    for (int c = 0; c < ncart(l); ++c)
        for (int k = 0; k < nprim; ++k) c_out[c * nprim + k] = cp[(size_t)k] * component_factor(l, c);
    return SCARF_OK;
}

}  // extern "C"

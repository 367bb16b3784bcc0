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
const double kW[kNClasses] = {2, 7, 13, 23, 38, 59, 87};
const double kCtr = 40.0;
// product-grid kernel: YZ = Y Z, g0 = X0 YZ, g1 = X1 YZ: 12 slots per 2 q-points; tables: 39 per (pair, axis point)
const double kCtrGrid = 6.0, kCtrTable = 39.0;

}  // namespace

struct scarf_ctx {
    int device = -1;
    bool host_only = true;
    cudaStream_t stream = nullptr;
    double prefactor = 2.0, screen_tol = 1e-16, threshold_eps = 0.0;
    bool timing = false;
    int n_chunks_opt = 0;     // 0 auto, else the number of stream chunks of the S4 kernels
    int fft_density_variant = 1;  // 1: DMMA kernel, 0: SIMT kernel (fft_method.cu)
    std::string err;
    HostSetup hs;
    bool have_basis = false, have_T = false;
    bool any_pure = false;                 // some shell is pure: T and S are mapped through pure_*
    int nbf_user = 0;                      // basis functions as the caller counts them
    std::vector<int> pure_nnz, pure_uidx;
    std::vector<double> pure_ucoef;
    int n_states = 0;
    int sm_count = 148;
    DevBuf d_pairs, d_E, d_bound, d_T, d_q, d_out, d_src, d_dst, d_nb, d_partial, d_axes, d_tab, d_ang_in, d_ang_F, d_ang_tab, d_ang_out, d_pure_map, d_Tcart, d_prim, d_V, d_fft, d_Csym;
    const double* Tc_dev = nullptr;        // context-owned Cartesian T of the last set_transitions (FFT method)
    std::vector<DevBuf> staging, packed;
    std::vector<TileStream> tiles;
    scarf_stats st = {};
    cudaEvent_t ev0 = nullptr, ev1 = nullptr, ev_slice = nullptr;
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

bool all_finite(const double* x, size_t n)
{
    // exponent field all ones <=> NaN or Inf; integer test so that the loop vectorises (a serial FP sum cost 1.6 ms per call on
    // config 3's q and T, inside the end-to-end step)
    uint64_t bad = 0;
    for (size_t i = 0; i < n; ++i) {
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

// Split the tile's class-sorted stream into <= K chunks of (nearly) equal modelled cost; a chunk may span classes.
// Returns the number of non-empty chunks written to `out`.
int build_chunks(const TileStream& t, int K, V1Chunk* out, double ctr = kCtr)
{
    double w[kNClasses], total = 0.0;
    long long nrec = 0;
    for (int c = 0; c < kNClasses; ++c) {
        w[c] = (double)t.ns_real * kW[c] + ctr;
        total += (double)t.cls[c].n * w[c];
        nrec += t.cls[c].n;
    }
    if (nrec == 0) return 0;
    K = (int)std::max<long long>(1, std::min<long long>(K, nrec));
    int k = 0;
    double acc = 0.0;
    std::memset(out, 0, sizeof(V1Chunk) * (size_t)K);
    bool cur_empty = true;
    for (int c = 0; c < kNClasses; ++c) {
        long long rem = t.cls[c].n, pos = 0;
        while (rem > 0) {
            long long take = rem;
            if (k < K - 1) {
                const double need = total * (double)(k + 1) / (double)K - acc;
                take = std::min<long long>(rem, (long long)std::llround(need / w[c]));
                if (take <= 0) {
                    if (cur_empty) take = 1;
                    else { ++k; cur_empty = true; continue; }
                }
            }
            out[k].begin[c] = (int)pos;
            out[k].n[c] = (int)take;
            cur_empty = false;
            acc += (double)take * w[c];
            pos += take; rem -= take;
            if (k < K - 1 && acc >= total * (double)(k + 1) / (double)K - 0.5 * w[c]) { ++k; cur_empty = true; }
        }
    }
    int n = 0;                                     // compact away chunks that stayed empty
    for (int i = 0; i < K; ++i) {
        bool any = false;
        for (int c = 0; c < kNClasses; ++c) any = any || out[i].n[c] > 0;
        if (any) { if (n != i) out[n] = out[i]; ++n; }
    }
    return n;
}

void free_device(scarf_ctx* c)
{
    c->d_pairs.release(); c->d_E.release(); c->d_bound.release(); c->d_T.release(); c->d_q.release();
    c->d_out.release(); c->d_src.release(); c->d_dst.release(); c->d_nb.release(); c->d_partial.release();
    c->d_axes.release(); c->d_tab.release();
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
        if (e == cudaSuccess) e = angular_init_device();
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, device);
        if (e == cudaSuccess) e = cudaEventCreate(&ctx->ev0);
        if (e == cudaSuccess) e = cudaEventCreate(&ctx->ev1);
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
        if (ctx->ev_slice) cudaEventDestroy(ctx->ev_slice);
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
    else if (k == "n_chunks") {
        if (value < 0 || value > kMaxChunks) return fail(ctx, SCARF_EINVAL, "set_option: n_chunks outside 0..32");
        ctx->n_chunks_opt = (int)value;
    } else if (k == "fft_density_variant") {
        if (value != 0.0 && value != 1.0) return fail(ctx, SCARF_EINVAL, "set_option: fft_density_variant must be 0 or 1");
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
        if (!is_device_ptr(T)) {
            if (!all_finite(T, tsz)) return fail(ctx, SCARF_EINVAL, "set_transitions: NaN/Inf in T");
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
        if (ctx->timing) CU(cudaEventRecord(ctx->ev0, st), "set_transitions: event");
        // fold every tile into a staging stream that holds ALL prescreened pairs
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
            a.staging = static_cast<char*>(ctx->staging[it].p);
            CU(launch_fold(a, st), "set_transitions: fold kernel");
            t.base = a.staging;
            t.bytes = off;
            for (int c = 0; c < kNClasses; ++c) {
                t.cls[c].n = hs.class_count[c];
                t.cls[c].off = a.cls_off[c];
                t.cls[c].rec_bytes = a.rec_bytes[c];
            }
        }
        // screening: B_P < screen_tol * mean(B) is dropped (rigorous: total dropped <= screen_tol * sum B)
        std::vector<double> bound((size_t)np);
        CU(cudaMemcpyAsync(bound.data(), ctx->d_bound.p, (size_t)np * sizeof(double), cudaMemcpyDeviceToHost, st), "set_transitions: read bounds");
        CU(cudaStreamSynchronize(st), "set_transitions: sync");
        double sumB = 0.0;
        for (double b : bound) {
            if (!std::isfinite(b)) return fail(ctx, SCARF_EINVAL, "set_transitions: NaN/Inf produced by T (device input not finite?)");
            sumB += b;
        }
        double maxB = 0.0;
        for (double b : bound) maxB = std::max(maxB, b);
        // default: B_P < screen_tol * mean(B); NEXT-2 option (paper-style): B_P < threshold_eps * max(B)
        const double thr = std::max(np > 0 ? ctx->screen_tol * sumB / (double)np : 0.0, ctx->threshold_eps * maxB);
        double dropped_bound = 0.0;
        for (double b : bound)
            if (!(b > 0.0 && b >= thr)) dropped_bound += b;
        std::vector<unsigned long long> src, dst;
        std::vector<int> nb;
        long long kept_per_class[kNClasses] = {};
        std::vector<long long> kept_idx;
        kept_idx.reserve((size_t)np);
        for (int c = 0; c < kNClasses; ++c)
            for (long long i = hs.class_first[c]; i < hs.class_first[c + 1]; ++i)
                if (bound[(size_t)i] > 0.0 && bound[(size_t)i] >= thr) {
                    kept_idx.push_back(i);
                    ++kept_per_class[c];
                }
        const long long n_kept = (long long)kept_idx.size();
        if (n_kept < np) {
            src.resize((size_t)n_kept); dst.resize((size_t)n_kept); nb.resize((size_t)n_kept);
            CU(ctx->d_src.ensure(std::max<size_t>(64, (size_t)n_kept * 8)), "set_transitions: alloc");
            CU(ctx->d_dst.ensure(std::max<size_t>(64, (size_t)n_kept * 8)), "set_transitions: alloc");
            CU(ctx->d_nb.ensure(std::max<size_t>(64, (size_t)n_kept * 4)), "set_transitions: alloc");
            for (size_t it = 0; it < tiles.size(); ++it) {
                TileStream& t = tiles[it];
                unsigned long long off = 0, new_off[kNClasses];
                for (int c = 0; c < kNClasses; ++c) {
                    new_off[c] = off;
                    off += (unsigned long long)kept_per_class[c] * t.cls[c].rec_bytes;
                }
                size_t k = 0;
                for (int c = 0; c < kNClasses; ++c) {
                    long long j = 0;
                    for (; k < kept_idx.size() && kept_idx[k] < hs.class_first[c + 1]; ++k, ++j) {
                        src[k] = t.cls[c].off + (unsigned long long)(kept_idx[k] - hs.class_first[c]) * t.cls[c].rec_bytes;
                        dst[k] = new_off[c] + (unsigned long long)j * t.cls[c].rec_bytes;
                        nb[k] = t.cls[c].rec_bytes;
                    }
                }
                CU(ctx->packed[it].ensure(std::max<unsigned long long>(64, off)), "set_transitions: alloc packed");
                CU(cudaMemcpyAsync(ctx->d_src.p, src.data(), (size_t)n_kept * 8, cudaMemcpyHostToDevice, st), "set_transitions: upload");
                CU(cudaMemcpyAsync(ctx->d_dst.p, dst.data(), (size_t)n_kept * 8, cudaMemcpyHostToDevice, st), "set_transitions: upload");
                CU(cudaMemcpyAsync(ctx->d_nb.p, nb.data(), (size_t)n_kept * 4, cudaMemcpyHostToDevice, st), "set_transitions: upload");
                CU(launch_pack(static_cast<const char*>(ctx->staging[it].p), static_cast<char*>(ctx->packed[it].p),
                               static_cast<const unsigned long long*>(ctx->d_src.p), static_cast<const unsigned long long*>(ctx->d_dst.p),
                               static_cast<const int*>(ctx->d_nb.p), n_kept, st), "set_transitions: pack kernel");
                CU(cudaStreamSynchronize(st), "set_transitions: sync");  // src/dst/nb host vectors are reused per tile
                t.base = static_cast<char*>(ctx->packed[it].p);
                t.bytes = off;
                for (int c = 0; c < kNClasses; ++c) {
                    t.cls[c].n = kept_per_class[c];
                    t.cls[c].off = new_off[c];
                }
            }
        }
        if (ctx->timing) {
            CU(cudaEventRecord(ctx->ev1, st), "set_transitions: event");
            CU(cudaEventSynchronize(ctx->ev1), "set_transitions: event sync");
            float ms = 0.f;
            cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1);
            ctx->st.last_fold_ms = ms;
        }
        ctx->tiles = tiles;
        ctx->n_states = n_states;
        scarf_stats& s = ctx->st;
        s.n_states = n_states;
        s.n_pairs_kept = n_kept;
        s.dropped_bound = dropped_bound;
        s.n_herm_kept = 0; s.slots_per_q = 0.0; s.stream_bytes = 0.0;
        for (int c = 0; c < kNClasses; ++c) {
            s.pairs_kept_per_class[c] = kept_per_class[c];
            s.n_herm_kept += kept_per_class[c] * nherm(c);
            s.slots_per_q += (double)kept_per_class[c] * ((double)n_states * kW[c] + kCtr * (double)tiles.size());
        }
        for (const auto& t : tiles) s.stream_bytes += (double)t.bytes;
        s.evals_per_q = (double)n_kept * (double)n_states;
        s.last_fold_launches = (int32_t)(tiles.size() * (n_kept < np ? 2 : 1));
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
        // all state tiles for the q range [dq, dq + 3 n_q) into dout [n_states][n_q]
        auto run_range = [&](const double* dq, long long n_q, double* dout) -> int {
        for (const TileStream& t : ctx->tiles) {
            long long nrec = 0;
            for (int L = 0; L < kNClasses; ++L) nrec += t.cls[L].n;
            double* tile_out = dout + (size_t)t.s0 * n_q * 2;
            if (nrec == 0) {  // no pair survived (T == 0): the answer is exactly zero
                CU(cudaMemsetAsync(tile_out, 0, (size_t)t.ns_real * n_q * 2 * sizeof(double), st), "form_factors: memset");
                continue;
            }
            V1Args a = {};
            a.base = t.base;
            for (int L = 0; L < kNClasses; ++L) a.cls_off[L] = t.cls[L].off;
            a.q = dq;
            a.n_q = n_q;
            const long long n_tiles = (n_q + v1_tile_q() - 1) / v1_tile_q();
            if (n_tiles > 0x7fffffffLL / kMaxChunks) return fail(ctx, SCARF_EINVAL, "form_factors: n_q too large for one call");
            a.n_tiles = (int)n_tiles;
            // ~24 waves of CTAs (2 resident per SM) so that the ragged last wave costs a few per cent
            long long K = ctx->n_chunks_opt > 0 ? ctx->n_chunks_opt : (24LL * 2 * ctx->sm_count + n_tiles / 2) / n_tiles;
            K = std::max<long long>(1, std::min<long long>(K, kMaxChunks));
            const size_t per_chunk = (size_t)t.ns_real * (size_t)n_q * 16;
            while (K > 1 && (double)K * (double)per_chunk > 4e9) --K;  // partial buffer <= 4 GB
            a.n_chunks = build_chunks(t, (int)K, a.chunks);
            a.ns_real = t.ns_real;
            if (a.n_chunks == 1) {
                a.dst = tile_out;
                a.chunk_stride = 0;
                CU(launch_ff_v1(t.NS, a, st), "form_factors: kernel");
                ++launches;
            } else {
                CU(ctx->d_partial.ensure((size_t)a.n_chunks * per_chunk), "form_factors: alloc partials");
                a.dst = static_cast<double*>(ctx->d_partial.p);
                a.chunk_stride = (long long)t.ns_real * n_q;
                CU(launch_ff_v1(t.NS, a, st), "form_factors: kernel");
                CU(launch_reduce_partials(a.dst, tile_out, a.chunk_stride, a.chunk_stride, a.n_chunks, st), "form_factors: reduce kernel");
                launches += 2;
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
        return SCARF_OK;
    } catch (const std::bad_alloc&) {
        return fail(ctx, SCARF_ENOMEM, "form_factors: out of host memory");
    } catch (...) {
        return fail(ctx, SCARF_EINVAL, "form_factors: unexpected exception");
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
        const int nbx = (nx + kGridBX - 1) / kGridBX, nby = (ny + kGridBY - 1) / kGridBY, nbz = (nz + kGridBZ - 1) / kGridBZ;
        const long long n_tiles = (long long)nbx * nby * nbz;
        if (n_tiles > 0x7fffffffLL / kMaxChunks) return fail(ctx, SCARF_EINVAL, "form_factors_grid: grid too large for one call");
        // axes -> one device buffer [nx | ny | nz]
        const double* ax_in[3] = {qx, qy, qz};
        const int ax_n[3] = {nx, ny, nz};
        CU(ctx->d_axes.ensure(((size_t)nx + ny + nz) * sizeof(double)), "form_factors_grid: alloc axes");
        double* dax[3];
        size_t off = 0;
        bool any_host_axis = false;
        for (int k = 0; k < 3; ++k) {
            dax[k] = static_cast<double*>(ctx->d_axes.p) + off;
            off += (size_t)ax_n[k];
            const bool host = !is_device_ptr(ax_in[k]);
            if (host && !all_finite(ax_in[k], (size_t)ax_n[k])) return fail(ctx, SCARF_EINVAL, "form_factors_grid: NaN/Inf in an axis");
            any_host_axis = any_host_axis || host;
            CU(cudaMemcpyAsync(dax[k], ax_in[k], (size_t)ax_n[k] * sizeof(double), host ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, st),
               "form_factors_grid: copy axis");
        }
        const size_t obytes = (size_t)ctx->n_states * (size_t)n_q * 2 * sizeof(double);
        double* dout = out;
        const bool out_host = !is_device_ptr(out);
        if (out_host) {
            CU(ctx->d_out.ensure(obytes), "form_factors_grid: alloc out");
            dout = static_cast<double*>(ctx->d_out.p);
        }
        if (ctx->timing) CU(cudaEventRecord(ctx->ev0, st), "form_factors_grid: event");
        int launches = 0;
        double slots = 0.0;
        const long long ncol = (long long)nbx * kGridBX + (long long)nby * kGridBY + (long long)nbz * kGridBZ;
        for (const TileStream& t : ctx->tiles) {
            GridArgs a = {};
            long long nrec = 0;
            for (int L = 0; L < kNClasses; ++L) {
                a.class_first[L] = nrec;
                a.rec_bytes[L] = t.cls[L].rec_bytes;
                a.v.cls_off[L] = t.cls[L].off;
                nrec += t.cls[L].n;
                slots += (double)t.cls[L].n * ((double)n_q * ((double)t.ns_real * kW[L] + kCtrGrid) + (double)(nx + ny + nz) * kCtrTable);
            }
            double* tile_out = dout + (size_t)t.s0 * n_q * 2;
            if (nrec == 0) {
                CU(cudaMemsetAsync(tile_out, 0, (size_t)t.ns_real * n_q * 2 * sizeof(double), st), "form_factors_grid: memset");
                continue;
            }
            const size_t tab_elems = (size_t)nrec * (size_t)ncol;
            if (tab_elems * 16 > (size_t)32e9) return fail(ctx, SCARF_ENOMEM, "form_factors_grid: factor tables would exceed 32 GB");
            CU(ctx->d_tab.ensure(tab_elems * 16), "form_factors_grid: alloc tables");
            double2* tx = static_cast<double2*>(ctx->d_tab.p);
            double2* ty = tx + (size_t)nrec * nbx * kGridBX;
            double2* tz = ty + (size_t)nrec * nby * kGridBY;
            a.v.base = t.base;
            a.v.n_q = n_q;
            a.v.n_tiles = (int)n_tiles;
            a.v.ns_real = t.ns_real;
            a.qx = dax[0]; a.qy = dax[1]; a.qz = dax[2];
            a.nx = nx; a.ny = ny; a.nz = nz;
            a.nbx = nbx; a.nby = nby; a.nbz = nbz;
            a.tx = tx; a.ty = ty; a.tz = tz;
            a.n_rec = nrec;
            CU(launch_grid_tables(a, tx, ty, tz, st), "form_factors_grid: table kernel");
            ++launches;
            long long K = ctx->n_chunks_opt > 0 ? ctx->n_chunks_opt : (24LL * 2 * ctx->sm_count + n_tiles / 2) / n_tiles;
            K = std::max<long long>(1, std::min<long long>(K, kMaxChunks));
            const size_t per_chunk = (size_t)t.ns_real * (size_t)n_q * 16;
            while (K > 1 && (double)K * (double)per_chunk > 4e9) --K;
            a.v.n_chunks = build_chunks(t, (int)K, a.v.chunks, kCtrGrid);
            if (a.v.n_chunks == 1) {
                a.v.dst = tile_out;
                a.v.chunk_stride = 0;
                CU(launch_ff_grid(t.NS, a, st), "form_factors_grid: kernel");
                ++launches;
            } else {
                CU(ctx->d_partial.ensure((size_t)a.v.n_chunks * per_chunk), "form_factors_grid: alloc partials");
                a.v.dst = static_cast<double*>(ctx->d_partial.p);
                a.v.chunk_stride = (long long)t.ns_real * n_q;
                CU(launch_ff_grid(t.NS, a, st), "form_factors_grid: kernel");
                CU(launch_reduce_partials(a.v.dst, tile_out, a.v.chunk_stride, a.v.chunk_stride, a.v.n_chunks, st),
                   "form_factors_grid: reduce kernel");
                launches += 2;
            }
        }
        ctx->st.last_kernel_launches = launches;
        ctx->st.last_grid_slots = slots;
        if (ctx->timing) {
            CU(cudaEventRecord(ctx->ev1, st), "form_factors_grid: event");
            CU(cudaEventSynchronize(ctx->ev1), "form_factors_grid: event sync");
            float ms = 0.f;
            cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1);
            ctx->st.last_kernel_ms = ms;
        }
        if (out_host) {
            CU(cudaMemcpyAsync(out, dout, obytes, cudaMemcpyDeviceToHost, st), "form_factors_grid: download out");
            CU(cudaStreamSynchronize(st), "form_factors_grid: sync");
        } else if (any_host_axis) {
            CU(cudaStreamSynchronize(st), "form_factors_grid: sync");  // pageable axes must not be reused before the copy ends
        }
        return SCARF_OK;
    } catch (const std::bad_alloc&) {
        return fail(ctx, SCARF_ENOMEM, "form_factors_grid: out of host memory");
    } catch (...) {
        return fail(ctx, SCARF_EINVAL, "form_factors_grid: unexpected exception");
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
        for (const TileStream& t : ctx->tiles) {
            GridArgs a = {};
            long long nrec = 0;
            for (int L = 0; L < kNClasses; ++L) {
                a.class_first[L] = nrec;
                a.rec_bytes[L] = t.cls[L].rec_bytes;
                a.v.cls_off[L] = t.cls[L].off;
                nrec += t.cls[L].n;
            }
            for (int k = 0; k < t.ns_real; ++k) out[2 * (t.s0 + k)] = out[2 * (t.s0 + k) + 1] = 0.0;
            if (nrec == 0) continue;
            a.v.base = t.base;
            a.v.ns_real = t.ns_real;
            a.qx = d[0]; a.qy = d[1]; a.qz = d[2];
            a.nx = nx; a.ny = ny; a.nz = nz;
            a.n_rec = nrec;
            const size_t n_blocks = (size_t)((nrec + per_block - 1) / per_block);
            const size_t mom_bytes = (size_t)nrec * 3 * kNClasses * 16, part_bytes = n_blocks * 16 * 16;
            CU(ctx->d_tab.ensure(mom_bytes + part_bytes), "separable_integral: alloc scratch");
            double* mom = static_cast<double*>(ctx->d_tab.p);
            double* part = mom + mom_bytes / 8;
            CU(launch_separable(a, t.NS, d[3], d[4], d[5], mom, part, per_block, st), "separable_integral: kernels");
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
        const int n_m = 2 * l_max + 1, nlm = (l_max + 1) * (l_max + 1), nhalf = (l_max + 1) * (l_max + 2) / 2;
        std::vector<double> Yw, tw;
        angular_host_tables(l_max, n_theta, cos_theta, w_theta, n_phi, Yw, tw);
        // tables: [tw (read as double2: first, 16-byte aligned) | Yw | w_theta]
        const size_t tab_doubles = Yw.size() + tw.size() + (size_t)n_theta;
        CU(ctx->d_ang_tab.ensure(tab_doubles * sizeof(double)), "angular_moments: alloc tables");
        double* dtw = static_cast<double*>(ctx->d_ang_tab.p);
        double* dYw = dtw + tw.size();
        double* dw = dYw + Yw.size();
        CU(cudaMemcpyAsync(dYw, Yw.data(), Yw.size() * sizeof(double), cudaMemcpyHostToDevice, st), "angular_moments: upload");
        CU(cudaMemcpyAsync(dtw, tw.data(), tw.size() * sizeof(double), cudaMemcpyHostToDevice, st), "angular_moments: upload");
        CU(cudaMemcpyAsync(dw, w_theta, (size_t)n_theta * sizeof(double), cudaMemcpyHostToDevice, st), "angular_moments: upload");
        const size_t fbytes = (size_t)n_rows * n_phi * 2 * sizeof(double);
        const double* df = f;
        if (!is_device_ptr(f)) {
            CU(ctx->d_ang_in.ensure(fbytes), "angular_moments: alloc f");
            CU(cudaMemcpyAsync(ctx->d_ang_in.p, f, fbytes, cudaMemcpyHostToDevice, st), "angular_moments: upload f");
            df = static_cast<const double*>(ctx->d_ang_in.p);
        }
        // scratch: F [n_rows][n_m] complex, rowsum2 [n_rows]
        CU(ctx->d_ang_F.ensure(((size_t)n_rows * n_m * 2 + (size_t)n_rows) * sizeof(double)), "angular_moments: alloc scratch");
        double* dF = static_cast<double*>(ctx->d_ang_F.p);
        double* drow2 = dF + (size_t)n_rows * n_m * 2;
        const size_t rbytes = (size_t)n_sr * nlm * 2 * sizeof(double), f2bytes = (size_t)n_sr * sizeof(double);
        const bool R_host = !is_device_ptr(R_out), f2_host = f2_out && !is_device_ptr(f2_out);
        double *dR = R_out, *df2 = f2_out;
        if (R_host || f2_host) {
            CU(ctx->d_ang_out.ensure(rbytes + f2bytes), "angular_moments: alloc out");
            if (R_host) dR = static_cast<double*>(ctx->d_ang_out.p);
            if (f2_host) df2 = static_cast<double*>(ctx->d_ang_out.p) + (size_t)n_sr * nlm * 2;
        }
        (void)nhalf;
        if (ctx->timing) CU(cudaEventRecord(ctx->ev0, st), "angular_moments: event");
        CU(launch_phi_dft(df, dtw, n_rows, n_phi, l_max, dF, drow2, st), "angular_moments: phi kernel");
        CU(launch_legendre(dF, drow2, dYw, dw, n_sr, n_theta, l_max, dR, df2, st), "angular_moments: legendre kernel");
        ctx->st.last_kernel_launches = 2;
        if (ctx->timing) {
            CU(cudaEventRecord(ctx->ev1, st), "angular_moments: event");
            CU(cudaEventSynchronize(ctx->ev1), "angular_moments: event sync");
            float ms = 0.f;
            cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1);
            ctx->st.last_kernel_ms = ms;
        }
        if (R_host) CU(cudaMemcpyAsync(R_out, dR, rbytes, cudaMemcpyDeviceToHost, st), "angular_moments: download R");
        if (f2_host) CU(cudaMemcpyAsync(f2_out, df2, f2bytes, cudaMemcpyDeviceToHost, st), "angular_moments: download f2");
        // the host tables (Yw, tw) are pageable and go out of scope: the copies must have finished
        CU(cudaStreamSynchronize(st), "angular_moments: sync");
        return SCARF_OK;
    } catch (const std::bad_alloc&) {
        return fail(ctx, SCARF_ENOMEM, "angular_moments: out of host memory");
    } catch (...) {
        return fail(ctx, SCARF_EINVAL, "angular_moments: unexpected exception");
    }
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
        const size_t vbytes = (size_t)hs.nbf * (size_t)((g.P + 7) / 8 * 8) * sizeof(double);
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
        CU(ctx->d_V.ensure(vbytes), "fft_form_factors: alloc orbital values");
        CU(ctx->d_fft.ensure(fbytes), "fft_form_factors: alloc transform buffer");
        const bool out_host = !is_device_ptr(out);
        double* dout = out;
        if (out_host) {
            CU(ctx->d_out.ensure(fbytes), "fft_form_factors: alloc out");
            dout = static_cast<double*>(ctx->d_out.p);
        }
        if (ctx->timing) CU(cudaEventRecord(ctx->ev0, st), "fft_form_factors: event");
        double* dV = static_cast<double*>(ctx->d_V.p);
        double* dF = static_cast<double*>(ctx->d_fft.p);
        CU(launch_orbitals(reinterpret_cast<const PrimShell*>(pb), reinterpret_cast<const int*>(pb + pbytes), n_sh, hs.nbf, g, dV, st),
           "fft_form_factors: orbital kernel");
        int launches = 1;
        for (int s0 = 0; s0 < ctx->n_states; s0 += kMaxStateTile) {
            const int ns_t = std::min(kMaxStateTile, ctx->n_states - s0);
            if (ctx->fft_density_variant == 0) {
                CU(launch_density(dV, ctx->Tc_dev, hs.nbf, g.P, s0, ns_t, ctx->prefactor, dF, st), "fft_form_factors: density kernel");
                ++launches;
            } else {
                const int nbf_pad = (hs.nbf + 7) & ~7;
                CU(ctx->d_Csym.ensure((size_t)kMaxStateTile * nbf_pad * nbf_pad * sizeof(double)), "fft_form_factors: alloc C");
                CU(launch_density_mma(dV, ctx->Tc_dev, static_cast<double*>(ctx->d_Csym.p), hs.nbf, nbf_pad, g.P, s0, ns_t,
                                      ctx->prefactor, dF, st), "fft_form_factors: density kernel (DMMA)");
                launches += 2;
            }
        }
        CU(cudaStreamSynchronize(st), "fft_form_factors: sync");   // `first` (pageable) goes out of scope; cuFFT plans below
        const int frc = cufft_inverse_batch(ctx->fft_plan, dF, nx, ny, nz, ctx->n_states, st);
        if (frc < 0) return fail(ctx, SCARF_ECUDA, "fft_form_factors: the cuFFT library (libcufft.so.11) could not be loaded");
        if (frc > 0) return fail(ctx, frc == 2 ? SCARF_ENOMEM : SCARF_ECUDA, "fft_form_factors: cuFFT error " + std::to_string(frc));
        CU(launch_fft_post(dF, g, ctx->n_states, dout, st), "fft_form_factors: post kernel");
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

int scarf_get_stats(scarf_ctx* ctx, scarf_stats* out)
{
    if (!ctx || !out) return SCARF_EINVAL;
    *out = ctx->st;
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

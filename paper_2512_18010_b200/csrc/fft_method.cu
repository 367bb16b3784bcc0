// fft_method.cu — the paper's FFT method as a second route to f_s(q) (Section III, Eq. (19)-(34)
// PAPER.md:140-222): tabulate the transition density on a regular real-space grid and transform it.
//
//   x_abc = x_min + L (a/N_x, b/N_y, c/N_z)                                   Eq. (25)-(28)
//   Phi_s(x) = g sum_pq T^s_pq phi_q(x) phi_p(x),  g = 2                      Eq. (20)
//   f_s(q) ~= V_pix sum_abc Phi_abc e^{+i q.x_abc},  q = 2 pi (alpha/L_x, beta/L_y, gamma/L_z)    Eq. (27), (30)-(33)
//   output index ia <-> alpha = ia - floor(N/2)  ("most negative frequencies first")
//
// Kernels: orbital_kernel (values of every contracted Cartesian orbital at every grid point, in tiles of 8 points),
// symmetrize_kernel + density_mma_kernel (the quadratic form v^T T^s v for up to 12 states per pass on the FP64 tensor
// cores, mma.sync.m8n8k4.f64; the method of the product), density_kernel (the same form with SIMT FMAs, T blocks in
// shared memory; kept as option "fft_density_variant" = 0 and as a second implementation the tests compare with),
// cuFFT Z2Z (library step, loaded with dlopen at first use so that libscarf.so itself has no cuFFT dependency; the plan
// belongs to the context), fft_post_kernel (V_pix, the phase e^{i q.x_min}, the reordering).
// This is an approximation of f_s (box truncation, grid spacing); its CPU oracle is oracle/fft_method.py.
#include <dlfcn.h>

#include <cmath>
#include <mutex>

#include "kernels.cuh"

namespace scarf {

namespace {

constexpr int kPts = 128;     // points per CTA
constexpr int kNB = 16, kMB = 8;

// orbital values are stored in tiles of 8 points: V[(p / 8)][mu][p % 8], so that the 4 nu x 8 points of a DMMA A fragment
// are 256 contiguous bytes (the plain [mu][point] layout costs 4 cache lines per fragment load and made L1 the limiter)
__device__ __forceinline__ size_t vidx(int mu, long long p, int nbf) { return ((size_t)(p >> 3) * nbf + mu) * 8 + (size_t)(p & 7); }

__device__ __forceinline__ double dfo(int n)   // (2n-1)!!
{
    double r = 1.0;
    for (int k = 2 * n - 1; k > 1; k -= 2) r *= k;
    return r;
}

__global__ void __launch_bounds__(kPts) orbital_kernel(const PrimShell* __restrict__ prim, const int* __restrict__ shell_first,
                                                       FftGrid g, int nbf, double* __restrict__ V)
{
    const long long p = (long long)blockIdx.x * kPts + threadIdx.x;
    if (p >= g.P) return;
    const int sh = blockIdx.y;
    const int k0 = shell_first[sh], k1 = shell_first[sh + 1];
    const int ic = (int)(p % g.nz), ib = (int)((p / g.nz) % g.ny), ia = (int)(p / ((long long)g.nz * g.ny));
    const PrimShell& ps = prim[k0];
    const double dx = g.xmin[0] + g.len[0] * ((double)ia / g.nx) - ps.A[0];
    const double dy = g.xmin[1] + g.len[1] * ((double)ib / g.ny) - ps.A[1];
    const double dz = g.xmin[2] + g.len[2] * ((double)ic / g.nz) - ps.A[2];
    const double r2 = dx * dx + dy * dy + dz * dz;
    double rad = 0.0;
    for (int k = k0; k < k1; ++k) rad = fma(prim[k].cprim, exp(-prim[k].alpha * r2), rad);
    const int l = ps.l;
    double px[kMaxL + 1], py[kMaxL + 1], pz[kMaxL + 1];
    px[0] = py[0] = pz[0] = 1.0;
#pragma unroll
    for (int i = 1; i <= kMaxL; ++i) { px[i] = px[i - 1] * dx; py[i] = py[i - 1] * dy; pz[i] = pz[i - 1] * dz; }
    int c = 0;
    for (int a = l; a >= 0; --a)                        // component order: a descending, then b descending
        for (int b = l - a; b >= 0; --b) {
            const int cc = l - a - b;
            V[vidx(ps.bf0 + c, p, nbf)] = rad * px[a] * py[b] * pz[cc] * rsqrt(dfo(a) * dfo(b) * dfo(cc));
            ++c;
        }
}

// Phi_s(p) = g sum_{mu <= nu} c_{mu nu} v_mu v_nu,  c = T_mumu on the diagonal, T_munu + T_numu above it.
__global__ void __launch_bounds__(kPts) density_kernel(const double* __restrict__ V, const double* __restrict__ T, int nbf, long long P,
                                                       int s0, int ns, double g, double2* __restrict__ out)
{
    __shared__ __align__(16) double sT[kMaxStateTile][kMB][kNB];
    const long long p = (long long)blockIdx.x * kPts + threadIdx.x;
    const bool valid = p < P;
    double acc[kMaxStateTile];
#pragma unroll
    for (int s = 0; s < kMaxStateTile; ++s) acc[s] = 0.0;
    for (int nb0 = 0; nb0 < nbf; nb0 += kNB) {
        double v[kNB];
#pragma unroll
        for (int i = 0; i < kNB; ++i) v[i] = (valid && nb0 + i < nbf) ? V[vidx(nb0 + i, p, nbf)] : 0.0;
        for (int mb0 = 0; mb0 < nbf && mb0 <= nb0 + kNB - 1; mb0 += kMB) {
            __syncthreads();
            for (int idx = threadIdx.x; idx < kMaxStateTile * kMB * kNB; idx += kPts) {
                const int s = idx / (kMB * kNB), m = (idx / kNB) % kMB, n = idx % kNB;
                const int mu = mb0 + m, nu = nb0 + n;
                double val = 0.0;
                if (s < ns && mu < nbf && nu < nbf && nu >= mu) {
                    const double* Ts = T + (size_t)(s0 + s) * nbf * nbf;
                    val = Ts[(size_t)mu * nbf + nu];
                    if (nu > mu) val += Ts[(size_t)nu * nbf + mu];
                }
                sT[s][m][n] = val;
            }
            __syncthreads();
#pragma unroll
            for (int m = 0; m < kMB; ++m) {
                const double vm = (valid && mb0 + m < nbf) ? V[vidx(mb0 + m, p, nbf)] : 0.0;
#pragma unroll
                for (int s = 0; s < kMaxStateTile; ++s) {
                    double w = 0.0;
#pragma unroll
                    for (int n = 0; n < kNB; ++n) w = fma(sT[s][m][n], v[n], w);
                    acc[s] = fma(vm, w, acc[s]);
                }
            }
        }
    }
    if (valid)
#pragma unroll
        for (int s = 0; s < kMaxStateTile; ++s)
            if (s < ns) out[(size_t)(s0 + s) * P + p] = make_double2(g * acc[s], 0.0);
}

// ---- the same quadratic form on the FP64 tensor cores (DMMA m8n8k4) ---------------------------------------------------
// W[p][mu] = sum_{nu >= mu} C_s[mu][nu] v_nu(p) is a dense contraction [points x nbf] . [nbf x nbf]: A = V tile (8 points x
// 4 nu), B = C_s^T tile (4 nu x 8 mu), D = W tile (8 points x 8 mu) accumulated over nu; then Phi_s(p) = sum_mu W[p][mu] v_mu(p)
// in the epilogue of every mu-chunk.  A warp owns 16 points (two M tiles share every B fragment) and all 12 states of the
// pass; fragments are read straight from global memory / L1, both stored in fragment order (256 contiguous bytes per
// load).  C_s is the zero-padded upper-triangular matrix written by symmetrize_kernel: T_mumu on the diagonal,
// T_munu + T_numu above, 0 below.  DMMA holds the FP64 pipe
// at its full rate with 4 register reads per 8 lane-FMAs, so it is free of the read-port bound of the SIMT form.
// C in DMMA B-fragment order: Cf[s][mu-chunk][nu-chunk][lane], lane = (gid, tig) <-> C_s[8 mc + gid][4 kc + tig]
// (a fragment load is then 256 contiguous bytes instead of 8 rows)
__global__ void __launch_bounds__(256) symmetrize_kernel(const double* __restrict__ T, int nbf, int nbf_pad, int s0, int ns,
                                                         double* __restrict__ C)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long per = (long long)nbf_pad * nbf_pad;
    if (i >= per * kMaxStateTile) return;
    const int s = (int)(i / per);
    const long long r = i % per;
    const int lane = (int)(r & 31), n_kc = nbf_pad / 4;
    const int kc = (int)((r >> 5) % n_kc), mc = (int)((r >> 5) / n_kc);
    const int mu = 8 * mc + (lane >> 2), nu = 4 * kc + (lane & 3);
    double v = 0.0;
    if (s < ns && mu < nbf && nu < nbf && nu >= mu) {
        const double* Ts = T + (size_t)(s0 + s) * nbf * nbf;
        v = Ts[(size_t)mu * nbf + nu];
        if (nu > mu) v += Ts[(size_t)nu * nbf + mu];
    }
    C[i] = v;
}

__device__ __forceinline__ void dmma884(double (&d)[2], double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d[0]), "+d"(d[1]) : "d"(a), "d"(b));
}

constexpr int kMmaWarps = 4;
constexpr int kMmaMT = 2;       // 8-point M tiles per warp (they share every B fragment)
constexpr int kMmaNSP = 12;     // states per pass: 4 NSP + 2 NSP accumulator doubles per lane (occupancy vs B-fragment reuse)
static_assert(kMaxStateTile % kMmaNSP == 0, "states per pass must divide the state tile");
// s_off: first state (within the tile) of this pass
__global__ void __launch_bounds__(kMmaWarps * 32) density_mma_kernel(const double* __restrict__ V, const double* __restrict__ C, int nbf,
                                                                     int nbf_pad, long long P, int s0, int ns, int s_off, double g,
                                                                     double2* __restrict__ out)
{
    const int lane = threadIdx.x & 31, gid = lane >> 2, tig = lane & 3;
    const long long p0 = ((long long)blockIdx.x * kMmaWarps + (threadIdx.x >> 5)) * (8 * kMmaMT);
    if (p0 >= P) return;
    long long pt[kMmaMT];
    bool ok[kMmaMT];
#pragma unroll
    for (int t = 0; t < kMmaMT; ++t) { pt[t] = p0 + 8 * t + gid; ok[t] = pt[t] < P; }
    const size_t per = (size_t)nbf_pad * nbf_pad;
    double phi[kMmaMT][kMmaNSP];
#pragma unroll
    for (int t = 0; t < kMmaMT; ++t)
#pragma unroll
        for (int s = 0; s < kMmaNSP; ++s) phi[t][s] = 0.0;
    for (int mu0 = 0; mu0 < nbf_pad; mu0 += 8) {
        double D[kMmaMT][kMmaNSP][2];
#pragma unroll
        for (int t = 0; t < kMmaMT; ++t)
#pragma unroll
            for (int s = 0; s < kMmaNSP; ++s) D[t][s][0] = D[t][s][1] = 0.0;
        const double* Cb = C + (size_t)s_off * per + (size_t)(mu0 / 8) * (nbf_pad / 4) * 32 + lane;   // + 32 * k-chunk
#pragma unroll 1
        for (int nu0 = mu0; nu0 < nbf_pad; nu0 += 4) {
            const int nu = nu0 + tig;
            double av[kMmaMT];                                               // A[row = gid][k = tig] = v_nu(point)
#pragma unroll
            for (int t = 0; t < kMmaMT; ++t) av[t] = (ok[t] && nu < nbf) ? V[vidx(nu, pt[t], nbf)] : 0.0;
#pragma unroll
            for (int s = 0; s < kMmaNSP; ++s) {
                const double bf = Cb[(size_t)s * per + (size_t)(nu0 / 4) * 32];
#pragma unroll
                for (int t = 0; t < kMmaMT; ++t) dmma884(D[t][s], av[t], bf);
            }
        }
        // D[row = gid][col = 2 tig + i] = W[point][mu0 + 2 tig + i]
        const int m0 = mu0 + 2 * tig, m1 = m0 + 1;
#pragma unroll
        for (int t = 0; t < kMmaMT; ++t) {
            const double v0 = (ok[t] && m0 < nbf) ? V[vidx(m0, pt[t], nbf)] : 0.0, v1 = (ok[t] && m1 < nbf) ? V[vidx(m1, pt[t], nbf)] : 0.0;
#pragma unroll
            for (int s = 0; s < kMmaNSP; ++s) phi[t][s] = fma(D[t][s][0], v0, fma(D[t][s][1], v1, phi[t][s]));
        }
    }
#pragma unroll
    for (int s = 0; s < kMmaNSP; ++s)
#pragma unroll
        for (int t = 0; t < kMmaMT; ++t) {
            double x = phi[t][s];
            x += __shfl_xor_sync(0xffffffffu, x, 1);
            x += __shfl_xor_sync(0xffffffffu, x, 2);
            if (tig == 0 && s_off + s < ns && ok[t]) out[(size_t)(s0 + s_off + s) * P + pt[t]] = make_double2(g * x, 0.0);
        }
}

// ---- fused route: orbital values evaluated per point tile straight into shared memory ---------------------------------------
// The kernel above reads V from HBM (nbf x P x 8 B: 3.2 GB at 190 bf / 128^3, 10 GB at 600 bf) and every warp streams the whole
// fragment table of C for its 16 points.  Here a CTA owns PT = 8 MT points: phase A evaluates every contracted orbital at those
// points into a shared-memory tile Vs[nu][point] (row stride PT + 4 doubles: the 4 nu x 8 points of an A fragment then fall on 16
// distinct 8-byte banks per half-warp); phase B runs the same DMMA contraction with A fragments from that tile.  The 8 warps
// split the work as (state group of kFusedNSW states) x (parity of the mu chunk), so every B fragment of C is read ONCE per CTA
// and feeds MT point tiles (4 or 8 instead of 2): the L2 traffic of the fragments drops by MT / 2 and the V buffer disappears.
// NPAR = 2: 8 warps, one CTA per SM (large tiles); NPAR = 1: 4 warps (one per state group) and two CTAs per SM, so that one CTA's
// orbital phase overlaps the other's tensor-core phase (small bases).
constexpr int kFusedNSW = 3;                 // states per warp; 12 / 3 = 4 state groups x 2 mu parities = 8 warps
constexpr int kFusedKPF = 4;                 // k-steps whose B fragments are in flight ahead of the DMMAs
static_assert(kMaxStateTile == 4 * kFusedNSW, "state groups");

// 1 / sqrt((2a-1)!!(2b-1)!!(2c-1)!!) at compile time (Newton iterations on small integers converge to the correctly rounded
// double well within the parity tolerance; the tabulating kernel above calls rsqrt at run time)
constexpr double cx_sqrt(double x)
{
    double y = x > 1.0 ? x : 1.0;
    for (int i = 0; i < 64; ++i) y = 0.5 * (y + x / y);
    return y;
}
constexpr double cx_dfo(int n)
{
    double r = 1.0;
    for (int k = 2 * n - 1; k > 1; k -= 2) r *= k;
    return r;
}
constexpr double comp_factor(int a, int b, int c) { return 1.0 / cx_sqrt(cx_dfo(a) * cx_dfo(b) * cx_dfo(c)); }

// all components of one shell of angular momentum LL at one point: dst[c * stride] (component order a desc, b desc), everything
// compile-time indexed (no local memory)
template <int LL>
__device__ __forceinline__ void shell_components(double rad, double dx, double dy, double dz, double* __restrict__ dst, int stride)
{
    double px[LL + 1], py[LL + 1], pz[LL + 1];
    px[0] = py[0] = pz[0] = 1.0;
#pragma unroll
    for (int i = 1; i <= LL; ++i) { px[i] = px[i - 1] * dx; py[i] = py[i - 1] * dy; pz[i] = pz[i - 1] * dz; }
    int c = 0;
#pragma unroll
    for (int a = LL; a >= 0; --a)
#pragma unroll
        for (int b = LL - a; b >= 0; --b) {
            dst[(size_t)c * stride] = (rad * comp_factor(a, b, LL - a - b)) * ((px[a] * py[b]) * pz[LL - a - b]);
            ++c;
        }
}

__device__ __forceinline__ void orbital_values_at(const PrimShell* __restrict__ prim, int k0, int k1, double x, double y, double z,
                                                  double* __restrict__ dst, int stride)   // dst[c * stride], c = component
{
    const double Ax = __ldg(&prim[k0].A[0]), Ay = __ldg(&prim[k0].A[1]), Az = __ldg(&prim[k0].A[2]);
    const int l = __ldg(&prim[k0].l);
    const double dx = x - Ax, dy = y - Ay, dz = z - Az;
    const double r2 = dx * dx + dy * dy + dz * dz;
    double rad = 0.0;
    for (int k = k0; k < k1; ++k) rad = fma(__ldg(&prim[k].cprim), exp(-__ldg(&prim[k].alpha) * r2), rad);
    switch (l) {
    case 0: shell_components<0>(rad, dx, dy, dz, dst, stride); break;
    case 1: shell_components<1>(rad, dx, dy, dz, dst, stride); break;
    case 2: shell_components<2>(rad, dx, dy, dz, dst, stride); break;
    case 3: shell_components<3>(rad, dx, dy, dz, dst, stride); break;
    case 4: shell_components<4>(rad, dx, dy, dz, dst, stride); break;
    case 5: shell_components<5>(rad, dx, dy, dz, dst, stride); break;
    default: shell_components<6>(rad, dx, dy, dz, dst, stride); break;
    }
}

template <int MT, int NPAR>
__global__ void __launch_bounds__(4 * NPAR * 32) density_fused_kernel(const PrimShell* __restrict__ prim, const int* __restrict__ shell_first,
                                                                          int n_shells, FftGrid g, const double* __restrict__ C, int nbf,
                                                                          int nbf_pad, int s0, int ns, double gfac, double2* __restrict__ out)
{
    constexpr int PT = 8 * MT, S = PT + 4;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* Vs = reinterpret_cast<double*>(smem_raw);                 // [nbf_pad][S]
    double* phis = Vs + (size_t)nbf_pad * S;                          // [kMaxStateTile][PT]
    const long long p0 = (long long)blockIdx.x * PT;
    // ---- phase A: orbital values of this CTA's points
    for (int i = threadIdx.x; i < (nbf_pad - nbf) * S; i += blockDim.x) Vs[(size_t)nbf * S + i] = 0.0;   // zero padding rows
    // a work item = (shell, point); consecutive threads take consecutive points of one shell, so a warp's loads of the shell data
    // are broadcasts and its switch on l is uniform
    for (int idx = threadIdx.x; idx < n_shells * PT; idx += blockDim.x) {
        const int sh = idx / PT, pt = idx % PT;
        const long long p = p0 + pt;
        const int k0 = __ldg(shell_first + sh), k1 = __ldg(shell_first + sh + 1);
        double* dst = Vs + (size_t)__ldg(&prim[k0].bf0) * S + pt;
        // points past the end of the grid are evaluated at the grid origin (finite values, never stored)
        const long long pe = p < g.P ? p : 0;
        const int ic = (int)(pe % g.nz), ib = (int)((pe / g.nz) % g.ny), ia = (int)(pe / ((long long)g.nz * g.ny));
        orbital_values_at(prim, k0, k1, g.xmin[0] + g.len[0] * ((double)ia / g.nx), g.xmin[1] + g.len[1] * ((double)ib / g.ny),
                          g.xmin[2] + g.len[2] * ((double)ic / g.nz), dst, S);
    }
    __syncthreads();
    // ---- phase B: W[p][mu] = sum_{nu >= mu} C_s[mu][nu] v_nu(p) on the tensor cores, phi_s(p) += sum_mu W[p][mu] v_mu(p)
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, gid = lane >> 2, tig = lane & 3;
    const int sg = warp & 3, par = warp >> 2, s_off = sg * kFusedNSW;
    const size_t per = (size_t)nbf_pad * nbf_pad;
    const int n_kc = nbf_pad / 4;
    double phi[MT][kFusedNSW];
#pragma unroll
    for (int t = 0; t < MT; ++t)
#pragma unroll
        for (int s = 0; s < kFusedNSW; ++s) phi[t][s] = 0.0;
    if (s_off < ns) {
        for (int mc = par; mc < nbf_pad / 8; mc += NPAR) {
            double D[MT][kFusedNSW][2];
#pragma unroll
            for (int t = 0; t < MT; ++t)
#pragma unroll
                for (int s = 0; s < kFusedNSW; ++s) D[t][s][0] = D[t][s][1] = 0.0;
            const double* Cb = C + (size_t)s_off * per + (size_t)mc * n_kc * 32 + lane;   // + s * per + kc * 32
            const int kc0 = 2 * mc;                                    // nu0 = mu0: first k-chunk of the upper triangle
            auto load_b = [&](int kc, double (&b)[kFusedKPF][kFusedNSW]) {
#pragma unroll
                for (int u = 0; u < kFusedKPF; ++u)
#pragma unroll
                    for (int s = 0; s < kFusedNSW; ++s) b[u][s] = kc + u < n_kc ? __ldg(Cb + (size_t)s * per + (size_t)(kc + u) * 32) : 0.0;
            };
            double bc[kFusedKPF][kFusedNSW], bn[kFusedKPF][kFusedNSW];
            load_b(kc0, bc);
#pragma unroll 1
            for (int kc = kc0; kc < n_kc; kc += kFusedKPF) {
                if (kc + kFusedKPF < n_kc) load_b(kc + kFusedKPF, bn);
#pragma unroll
                for (int u = 0; u < kFusedKPF; ++u)
                    if (kc + u < n_kc) {
                        const double* vrow = Vs + (size_t)(4 * (kc + u) + tig) * S + gid;   // A[row = gid][k = tig] = v_nu(point)
#pragma unroll
                        for (int t = 0; t < MT; ++t) {
                            const double av = vrow[8 * t];
#pragma unroll
                            for (int s = 0; s < kFusedNSW; ++s) dmma884(D[t][s], av, bc[u][s]);
                        }
                    }
#pragma unroll
                for (int u = 0; u < kFusedKPF; ++u)
#pragma unroll
                    for (int s = 0; s < kFusedNSW; ++s) bc[u][s] = bn[u][s];
            }
            // D[row = gid][col = 2 tig + i] = W[point][8 mc + 2 tig + i]
            const double* v0 = Vs + (size_t)(8 * mc + 2 * tig) * S + gid;
#pragma unroll
            for (int t = 0; t < MT; ++t) {
                const double a0 = v0[8 * t], a1 = v0[S + 8 * t];
#pragma unroll
                for (int s = 0; s < kFusedNSW; ++s) phi[t][s] = fma(D[t][s][0], a0, fma(D[t][s][1], a1, phi[t][s]));
            }
        }
    }
    // ---- reduce over the 4 column lanes, then over the two mu parities (fixed order), store
#pragma unroll
    for (int t = 0; t < MT; ++t)
#pragma unroll
        for (int s = 0; s < kFusedNSW; ++s) {
            double x = phi[t][s];
            x += __shfl_xor_sync(0xffffffffu, x, 1);
            x += __shfl_xor_sync(0xffffffffu, x, 2);
            phi[t][s] = x;
        }
    if (NPAR == 2 && par == 0 && tig == 0)
#pragma unroll
        for (int t = 0; t < MT; ++t)
#pragma unroll
            for (int s = 0; s < kFusedNSW; ++s) phis[(s_off + s) * PT + 8 * t + gid] = phi[t][s];
    if (NPAR == 2) __syncthreads();
    if (par == NPAR - 1 && tig == 0)
#pragma unroll
        for (int t = 0; t < MT; ++t)
#pragma unroll
            for (int s = 0; s < kFusedNSW; ++s) {
                const long long p = p0 + 8 * t + gid;
                if (s_off + s < ns && p < g.P)
                    out[(size_t)(s0 + s_off + s) * g.P + p] = make_double2(gfac * ((NPAR == 2 ? phis[(s_off + s) * PT + 8 * t + gid] : 0.0) + phi[t][s]), 0.0);
            }
}

// out[s][(ia, ib, ic)] = V_pix e^{i q.x_min} F[s][(alpha mod N, ...)],  alpha = ia - floor(N/2)
__global__ void __launch_bounds__(256) fft_post_kernel(const double2* __restrict__ F, FftGrid g, int ns, double2* __restrict__ out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.P * ns) return;
    const long long p = i % g.P;
    const int s = (int)(i / g.P);
    const int ic = (int)(p % g.nz), ib = (int)((p / g.nz) % g.ny), ia = (int)(p / ((long long)g.nz * g.ny));
    const int al = ia - g.nx / 2, be = ib - g.ny / 2, ga = ic - g.nz / 2;
    const long long src = ((long long)((al + g.nx) % g.nx) * g.ny + (be + g.ny) % g.ny) * g.nz + (ga + g.nz) % g.nz;
    const double twopi = 6.283185307179586476925286766559;
    const double ph = twopi * (al / g.len[0] * g.xmin[0] + be / g.len[1] * g.xmin[1] + ga / g.len[2] * g.xmin[2]);
    double sn, cs;
    sincos(ph, &sn, &cs);
    const double vpix = g.len[0] * g.len[1] * g.len[2] / (double)g.P;
    const double2 f = F[(size_t)s * g.P + src];
    out[i] = make_double2(vpix * (f.x * cs - f.y * sn), vpix * (f.x * sn + f.y * cs));
}

// ---- Parseval check, Eq. (75) PAPER.md:557-562 ---------------------------------------------------------------------------
// sum_i |a_i|^2 per state of a complex array [ns][P]: kSumBlocks blocks per state over contiguous slices, fixed-order tree
// inside a block, then one thread per state adds the block sums in block order (deterministic).
constexpr int kSumBlocks = 256;
__global__ void __launch_bounds__(256) sumsq_kernel(const double2* __restrict__ a, long long P, double* __restrict__ part)
{
    __shared__ double sh[8];
    const int s = blockIdx.y;
    const long long per = (P + kSumBlocks - 1) / kSumBlocks, i0 = (long long)blockIdx.x * per, i1 = min(P, i0 + per);
    double acc = 0.0;
    for (long long i = i0 + threadIdx.x; i < i1; i += 256) {
        const double2 v = a[(size_t)s * P + i];
        acc = fma(v.x, v.x, fma(v.y, v.y, acc));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t += sh[w];
        part[(size_t)s * kSumBlocks + blockIdx.x] = t;
    }
}
__global__ void sumsq_final_kernel(const double* __restrict__ part, int ns, double scale, double* __restrict__ out, int stride, int col)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= ns) return;
    double t = 0.0;
    for (int b = 0; b < kSumBlocks; ++b) t += part[(size_t)s * kSumBlocks + b];
    out[(size_t)s * stride + col] = t * scale;
}

// ---- cuFFT through dlopen (library step; keeps libscarf.so free of a link-time cuFFT dependency) -------------------
// The function table is immutable once loaded (std::call_once); plans are owned by the calling context (CufftPlan).
typedef int (*PlanFn)(int*, int, int, int, int);
typedef int (*SetStreamFn)(int, cudaStream_t);
typedef int (*ExecFn)(int, void*, void*, int);
typedef int (*DestroyFn)(int);
struct CufftApi {
    void* h = nullptr;
    PlanFn plan3d = nullptr;
    SetStreamFn set_stream = nullptr;
    ExecFn exec_z2z = nullptr;
    DestroyFn destroy = nullptr;
};

const CufftApi* cufft_api()
{
    static CufftApi api;
    static std::once_flag once;
    std::call_once(once, [] {
        const char* names[] = {"libcufft.so.11", "/usr/local/cuda/lib64/libcufft.so.11", "libcufft.so", "/usr/local/cuda/lib64/libcufft.so"};
        void* h = nullptr;
        for (const char* n : names) {
            h = dlopen(n, RTLD_NOW | RTLD_LOCAL);
            if (h) break;
        }
        if (!h) return;
        api.plan3d = (PlanFn)dlsym(h, "cufftPlan3d");
        api.set_stream = (SetStreamFn)dlsym(h, "cufftSetStream");
        api.exec_z2z = (ExecFn)dlsym(h, "cufftExecZ2Z");
        api.destroy = (DestroyFn)dlsym(h, "cufftDestroy");
        if (!api.plan3d || !api.set_stream || !api.exec_z2z || !api.destroy) {
            dlclose(h);
            return;
        }
        api.h = h;
    });
    return api.h ? &api : nullptr;
}

}  // namespace

cudaError_t launch_orbitals(const PrimShell* prim, const int* shell_first, int n_shells, int nbf, const FftGrid& g, double* V, cudaStream_t st)
{
    if (g.P <= 0 || n_shells <= 0) return cudaSuccess;
    dim3 grid((unsigned)((g.P + kPts - 1) / kPts), (unsigned)n_shells);
    orbital_kernel<<<grid, kPts, 0, st>>>(prim, shell_first, g, nbf, V);
    return cudaGetLastError();
}

cudaError_t launch_density(const double* V, const double* T, int nbf, long long P, int s0, int ns, double g, double* out_complex,
                           cudaStream_t st)
{
    if (P <= 0 || ns <= 0) return cudaSuccess;
    density_kernel<<<(unsigned)((P + kPts - 1) / kPts), kPts, 0, st>>>(V, T, nbf, P, s0, ns, g, reinterpret_cast<double2*>(out_complex));
    return cudaGetLastError();
}

cudaError_t launch_density_mma(const double* V, const double* T, double* Csym, int nbf, int nbf_pad, long long P, int s0, int ns,
                               double g, double* out_complex, cudaStream_t st)
{
    if (P <= 0 || ns <= 0) return cudaSuccess;
    const long long nsym = (long long)kMaxStateTile * nbf_pad * nbf_pad;
    symmetrize_kernel<<<(unsigned)((nsym + 255) / 256), 256, 0, st>>>(T, nbf, nbf_pad, s0, ns, Csym);
    const long long per_cta = 8LL * kMmaMT * kMmaWarps;
    for (int s_off = 0; s_off < ns; s_off += kMmaNSP)
        density_mma_kernel<<<(unsigned)((P + per_cta - 1) / per_cta), kMmaWarps * 32, 0, st>>>(V, Csym, nbf, nbf_pad, P, s0, ns, s_off, g,
                                                                                           reinterpret_cast<double2*>(out_complex));
    return cudaGetLastError();
}

// Shared memory of the fused density kernel for MT point tiles per CTA; 0 if it does not fit.
static size_t fused_smem(int nbf_pad, int MT) { return ((size_t)nbf_pad * (8 * MT + 4) + (size_t)kMaxStateTile * 8 * MT) * sizeof(double); }

cudaError_t density_fused_init_device()
{
    cudaError_t e = cudaFuncSetAttribute(density_fused_kernel<8, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kDensityFusedMaxSmem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(density_fused_kernel<8, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, kDensityFusedMaxSmem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(density_fused_kernel<4, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, kDensityFusedMaxSmem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(density_fused_kernel<2, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, kDensityFusedMaxSmem);
    return e;
}

bool density_fused_fits(int nbf_pad) { return fused_smem(nbf_pad, 2) <= (size_t)kDensityFusedMaxSmem; }

// Csym must have been filled by launch_symmetrize for this (s0, ns).
cudaError_t launch_density_fused(const PrimShell* prim, const int* shell_first, int n_shells, const FftGrid& g, const double* Csym, int nbf,
                                 int nbf_pad, int s0, int ns, double gfac, double* out_complex, cudaStream_t st)
{
    if (g.P <= 0 || ns <= 0) return cudaSuccess;
    double2* out = reinterpret_cast<double2*>(out_complex);
    // 64 points per CTA: two 4-warp CTAs per SM while their tiles fit, else one 8-warp CTA; then 32 and 16 points
#define SCARF_FUSED(MTV, NPARV, PTS)                                                                                             \
    density_fused_kernel<MTV, NPARV><<<(unsigned)((g.P + PTS - 1) / PTS), 4 * NPARV * 32, fused_smem(nbf_pad, MTV), st>>>(          \
        prim, shell_first, n_shells, g, Csym, nbf, nbf_pad, s0, ns, gfac, out)
    if (fused_smem(nbf_pad, 8) <= (size_t)(110 * 1024)) SCARF_FUSED(8, 1, 64);
    else if (fused_smem(nbf_pad, 8) <= (size_t)kDensityFusedMaxSmem) SCARF_FUSED(8, 2, 64);
    else if (fused_smem(nbf_pad, 4) <= (size_t)kDensityFusedMaxSmem) SCARF_FUSED(4, 2, 32);
    else SCARF_FUSED(2, 2, 16);
#undef SCARF_FUSED
    return cudaGetLastError();
}

cudaError_t launch_symmetrize(const double* T, double* Csym, int nbf, int nbf_pad, int s0, int ns, cudaStream_t st)
{
    const long long nsym = (long long)kMaxStateTile * nbf_pad * nbf_pad;
    symmetrize_kernel<<<(unsigned)((nsym + 255) / 256), 256, 0, st>>>(T, nbf, nbf_pad, s0, ns, Csym);
    return cudaGetLastError();
}

cudaError_t launch_fft_post(const double* F, const FftGrid& g, int ns, double* out, cudaStream_t st)
{
    const long long n = g.P * ns;
    if (n <= 0) return cudaSuccess;
    fft_post_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(reinterpret_cast<const double2*>(F), g, ns, reinterpret_cast<double2*>(out));
    return cudaGetLastError();
}

// out[s * stride + col] = scale * sum_i |a[s][i]|^2, s < ns; scratch: ns * 256 doubles.
cudaError_t launch_sumsq(const double* a_complex, long long P, int ns, double scale, double* scratch, double* out, int stride, int col,
                         cudaStream_t st)
{
    if (ns <= 0 || P <= 0) return cudaSuccess;
    sumsq_kernel<<<dim3(kSumBlocks, (unsigned)ns), 256, 0, st>>>(reinterpret_cast<const double2*>(a_complex), P, scratch);
    sumsq_final_kernel<<<(unsigned)((ns + 63) / 64), 64, 0, st>>>(scratch, ns, scale, out, stride, col);
    return cudaGetLastError();
}

// In-place unnormalised transforms sum_abc f e^{+2 pi i (...)} of ns arrays [nx][ny][nz] of complex doubles with the
// context's plan (created on the device that is current, i.e. the context's; re-planned when the grid changes).
// Returns 0, -1 (cuFFT library not loadable) or a positive cufftResult.
int cufft_inverse_batch(CufftPlan& pl, double* data, int nx, int ny, int nz, int ns, cudaStream_t st)
{
    const CufftApi* api = cufft_api();
    if (!api) return -1;
    if (pl.handle < 0 || pl.nx != nx || pl.ny != ny || pl.nz != nz) {
        cufft_plan_release(pl);
        int h = 0;
        const int rc = api->plan3d(&h, nx, ny, nz, 0x69 /* CUFFT_Z2Z */);
        if (rc != 0) return rc;
        pl.handle = h; pl.nx = nx; pl.ny = ny; pl.nz = nz;
    }
    int rc = api->set_stream(pl.handle, st);
    if (rc != 0) return rc;
    const size_t per = (size_t)nx * ny * nz * 2;
    for (int s = 0; s < ns; ++s) {
        rc = api->exec_z2z(pl.handle, data + (size_t)s * per, data + (size_t)s * per, 1 /* CUFFT_INVERSE */);
        if (rc != 0) return rc;
    }
    return 0;
}

void cufft_plan_release(CufftPlan& pl)
{
    const CufftApi* api = cufft_api();
    if (api && pl.handle >= 0) api->destroy(pl.handle);
    pl = CufftPlan();
}

}  // namespace scarf

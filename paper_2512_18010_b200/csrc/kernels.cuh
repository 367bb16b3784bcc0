// kernels.cuh — device-side data layout and launcher prototypes shared by scarf_api.cu and the kernel files.
//
// Pair stream ("records"), one per kept primitive shell pair, grouped by class L = la + lb, per state tile:
//
//     double  Px, Py, Pz, inv4p                 32-byte header (Gaussian-product centre, 1/(4p))
//     double  D[NS][n_herm(L)]                  folded coefficients, state-major, Hermite index h fastest
//     double  0 (only if NS*n_herm is odd)      pad to a 16-byte multiple
//
// Hermite index h enumerates (t,u,v) by total degree n = t+u+v ascending, then t descending, then u descending,
// so the list for class L is a prefix of the list for class L+1.  The factor i^n of (iq)^t is folded into D:
// even n carry (-1)^{n/2} and contribute to the real polynomial A, odd n carry (-1)^{(n-1)/2} and contribute
// to the imaginary polynomial B;   term = e^{-q^2/4p} (cos qP + i sin qP) (A + iB).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>
#include <vector>

#include "host_setup.hpp"

namespace scarf {

constexpr int kMaxStateTile = 12;  // states whose accumulators one thread keeps in registers

__host__ __device__ inline constexpr int rec_doubles(int L, int NS)
{
    return 4 + ((NS * nherm(L) + 1) & ~1);
}

// ---- device-resident description of one state tile's packed pair stream ---------------------------------------------
// Written on the device by the screening / pack / chunk-planning kernels of fold.cu, read by every S4 kernel, so that
// scarf_set_transitions needs no device->host round trip (the host never learns the kept counts unless asked:
// scarf_get_stats).  A chunk is a cost-balanced contiguous slice of the class-sorted stream; per class c it covers
// records [begin[c], begin[c] + n[c]) of that class.
constexpr int kMaxChunks = 32;
struct V1Chunk {
    int begin[kNClasses];
    int n[kNClasses];
};
struct StreamDesc {
    long long n_kept;                       // records in the packed stream
    long long cls_n[kNClasses];             // kept records per class
    long long cls_first[kNClasses + 1];     // stream-order index of each class's first record
    unsigned long long cls_off[kNClasses];  // byte offset of each class's first record from the stream base
    int rec_bytes[kNClasses];
    int n_chunks;                           // chunks planned by the last plan_chunks launch (some may be empty)
    V1Chunk chunks[kMaxChunks];
};
struct ScreenResult {                       // device -> pinned host, read lazily (scarf_get_stats)
    long long n_kept;
    long long kept_per_class[kNClasses];
    double sum_bound, max_bound, dropped_bound;
    int bad, pad;                           // bad != 0: a bound was NaN/Inf (non-finite T): nothing is dropped, the output carries the NaN
};

struct TileStream {            // one state tile of the pair stream (host bookkeeping; the counts live in `desc`)
    int s0, ns_real, NS;       // first state, real states, padded/templated state count
    int pad;
    char* staging;             // device: records of ALL prescreened pairs, class-sorted (written by the fold)
    char* base;                // device: packed stream of the kept pairs
    StreamDesc* desc;          // device
    unsigned long long staging_bytes;
};

struct FoldArgs {
    const PairMeta* pairs;
    long long n_pairs;
    const double* E;
    const double* T;           // [ns_total][nbf][nbf]
    int nbf, s0, ns_real, NS;
    int first_tile, pad;
    double g;
    char* staging;             // tile stream laid out for ALL prescreened pairs
    double* bound;             // [n_pairs] screening bound B_P
    long long class_first[kNClasses + 1];
    unsigned long long cls_off[kNClasses];
    int rec_bytes[kNClasses];
};

struct ScreenArgs {
    const double* bound;       // [n_pairs]
    long long n_pairs;
    long long class_first[kNClasses + 1];   // prescreened pairs per class (host knows these)
    double screen_tol, threshold_eps;
    int* keep_idx;             // [n_pairs] out: source index of the k-th kept record (stable order)
    ScreenResult* result;      // device
};

struct PackArgs {
    const char* staging;
    char* packed;
    const int* keep_idx;
    const ScreenResult* result;
    StreamDesc* desc;          // written by block 0
    long long n_pairs;
    long long class_first[kNClasses + 1];
    unsigned long long cls_off[kNClasses];  // of the staging layout
    int rec_bytes[kNClasses];
};

constexpr int kMaxAdaptTiles = 8;           // state tiles the q-adaptive cut-off supports (96 states)
struct AdaptArgs {
    const int* keep_idx;                    // stable, class-sorted kept indices (screen_kernel)
    const ScreenResult* result;
    long long class_first[kNClasses + 1];   // of the prescreened (staging) order
    int n_tiles;
    const char* staging[kMaxAdaptTiles];    // every state tile's staging stream
    unsigned long long cls_off[kMaxAdaptTiles][kNClasses];
    int rec_bytes[kMaxAdaptTiles][kNClasses];
    int NS[kMaxAdaptTiles];
    double adaptive_tol;                    // tau = adaptive_tol * mean bound
    long long n_pairs;
    double* key;                            // [n_pairs] out: q_cut of the k-th kept record (screen order)
    int* keep_sorted;                       // [n_pairs] out: kept indices, q_cut-descending inside each class
    double* qcut_sorted;                    // [n_pairs] out: q_cut in that order (what the S4 kernels search)
};

cudaError_t launch_adaptive_sort(const AdaptArgs& a, cudaStream_t st);
cudaError_t launch_fold(const FoldArgs& a, cudaStream_t st);
cudaError_t launch_screen(const ScreenArgs& a, cudaStream_t st);
cudaError_t launch_pack(const PackArgs& a, cudaStream_t st);
// cost-balanced split of the FAST classes (0..kFastMaxClass) of the stream into exactly K chunks (K <= kMaxChunks);
// w(c) = ns_real * W(c) + ctr.  One thread; ~2 us.
// model: per-class slot counts of 0 the list kernel, 1 the box kernel (ff_grid.cu), 2 the row kernel (ff_row.cu), 3 the spherical-grid kernel (ff_sph.cu), 4 the mirror-pair row kernel (ff_zrow.cu)
cudaError_t launch_plan_chunks(StreamDesc* desc, int K, int ns_real, double ctr, cudaStream_t st, int model = 0);

// v1 (ff_v1.cu): the general-q kernel.  Grid = (n_tiles, n_chunks), dispatched chunk-major; the chunks of one q tile add
// their partial sums into `out` in chunk order through a per-tile ticket (no partial buffer in HBM, no second kernel).
constexpr int kFastMaxClass = 6;            // classes 0..6 (shells up to f with f) run in the unrolled kernels
struct V1Args {
    const char* base;                       // tile stream base
    const StreamDesc* desc;                 // device: class offsets, chunk table
    const double* q;                        // [n_q][3]
    long long n_q;
    int n_tiles, n_chunks;                  // grid = (n_tiles, n_chunks)
    int ns_real;
    int tile_group;                         // product-grid kernels: 0 = CTAs dispatched chunk-major over ALL tiles; G > 0 = chunk-major inside
                                            // groups of G consecutive tiles, group after group (finished tiles leave the kernel all along
                                            // its run instead of in its last 1/n_chunks: what a pinned host `out` needs, see dst_final)
    double* dst;                            // out + s0*n_q*2
    double* dst_final;                      // product-grid kernels: where the LAST chunk of a tile stores the finished values (and the
                                            // mirror points): nullptr = dst; else a device alias of the caller's pinned host `out`, so that
                                            // the results cross PCIe as the kernel produces them (partial sums stay in dst, on the device)
    int* tickets;                           // [n_tiles], all zero at launch and again at exit (n_chunks > 1 only)
    const double* qcut;                     // q-adaptive cut-off: q_cut per record in stream order (descending inside a class); nullptr: off
    unsigned long long* work;               // [kNClasses] += records evaluated per CTA and class (q-adaptive statistics); nullptr: off
};
int v1_tile_q();                            // q-points per CTA
cudaError_t launch_ff_v1(int NS, const V1Args& a, cudaStream_t st);
// allocation-free variant (scarf_form_factors_noalloc): tickets in a static device array of v1_static_tiles() entries
int v1_static_tiles();
cudaError_t ff_v1_static_setup();            // resolves the array's address on the current device (once per device)
cudaError_t launch_ff_v1_static(int NS, V1Args a, cudaStream_t st);

// high classes (ff_highl.cu): pairs with g, h, i shells (L = 7..12); runs after the unrolled kernel and ADDS to out.
struct HighLArgs {
    const char* base;                       // tile stream base
    const StreamDesc* desc;
    const double* q;                        // list mode: [n_points][3]; nullptr: product-grid mode
    const double *qx, *qy, *qz;             // grid mode: axes; points = (ix < nx_eval, iy, iz)
    int nx, ny, nz, nx_eval, sym, ns_real;
    long long n_points;                     // points evaluated (n_q, or nx_eval*ny*nz)
    long long n_q;                          // points per state in out
    double* dst;                            // out + s0*n_q*2
};
cudaError_t launch_ff_highl(const HighLArgs& a, cudaStream_t st);

// grid (ff_grid.cu): Cartesian product grid q = (qx[ix], qy[iy], qz[iz]), index (ix*ny + iy)*nz + iz.  The
// Gaussian/phase factor separates, e^{-q^2/4p} e^{iq.P} = X_P(ix) Y_P(iy) Z_P(iz) (the V-tensor idea of Eq. (45)-(46)
// PAPER.md:309-316), so it is tabulated once per (pair, axis point) and S4 needs two complex multiplies per
// (q, pair) instead of an exp and a sincos.  A CTA owns a kGridBX x kGridBY x kGridBZ box of the grid.
constexpr int kGridBX = 4, kGridBY = 8, kGridBZ = 8;
struct GridArgs {
    V1Args v;                               // stream, desc, dst as for v1; v.q unused; v.n_q = nx*ny*nz
    const double *qx, *qy, *qz;             // axes (device)
    int nx, ny, nz;
    int nbx, nby, nbz;                      // boxes per axis.  With `sym` the boxes cover ix < nx_eval only
    int bx0, pad0;                          // this launch covers x boxes bx0 .. bx0 + v.n_tiles/(nby*nbz) - 1 (host output is computed in x slabs)
    int sym, nx_eval;                       // sym != 0: the grid is inversion-symmetric (every axis ax[i] == -ax[n-1-i] bit for bit):
                                            // only ix < nx_eval = ceil(nx/2) is evaluated and f(-q) = conj f(q) is stored for the mirror point
    const double2 *tx, *ty, *tz;            // tables [box][row][box edge] of (re, im); zero beyond the axis end
    long long n_rows;                       // row stride of the tables (>= kept records; the prescreened count, known to the host)
    int bxs, bys, bzs, pad1;                // box edges the tables are laid out for: kGridB* (ff_grid.cu) or kRowB* (ff_row.cu)
};
cudaError_t launch_grid_tables(const GridArgs& a, double2* tx, double2* ty, double2* tz, cudaStream_t st);
cudaError_t launch_ff_grid(int NS, const GridArgs& a, cudaStream_t st);
cudaError_t ff_grid_init_device();           // per-device function attributes (dynamic shared memory); idempotent
// row decomposition (ff_row.cu): a warp owns one (ix, iy) row of 64 z-points, so the (q_x, q_y) part of every polynomial is
// warp-uniform: it is evaluated once per (record, state, row) by the warp's lanes in parallel, and a point only needs the short
// polynomial in its own q_z.  Same GridArgs, tables laid out for 1 x 4 x 64 boxes.
constexpr int kRowBX = 1, kRowBY = 4, kRowBZ = 64;
cudaError_t launch_ff_row(int NS, const GridArgs& a, cudaStream_t st);
cudaError_t ff_row_init_device();
// mirror-pair row kernel (ff_zrow.cu): the row kernel on a grid whose z axis is antisymmetric bit for bit; a lane's two points are
// (+z, -z).  GridArgs as for the row kernel except: nbz counts boxes of 32 mirror PAIRS and the Z table (box edge 32) covers the
// first ceil(nz/2) points of the axis.
constexpr int kZrowBX = 1, kZrowBY = 4, kZrowBZ = 32;
cudaError_t launch_ff_zrow(int NS, const GridArgs& a, cudaStream_t st);
cudaError_t ff_zrow_init_device();
// spherical product grid (ff_sph.cu): q = r_i n_d, n_d = (sin t_j cos phi_k, sin t_j sin phi_k, cos t_j), d = j n_phi + k; point index
// i * n_theta * n_phi + d (the layout of scarf_angular_moments' input).  A warp owns one direction and 64 radii.
constexpr int kSphBD = 4, kSphBR = 64;
struct SphArgs {
    V1Args v;                               // stream, desc, dst, tickets, qcut as for v1; v.q unused; v.n_q = n_r * n_theta * n_phi
    const double* r;                        // [n_r] radii (device)
    const double* dirs;                     // [n_theta * n_phi][3] unit vectors (device); with `sym` dirs[mirror(d)] == -dirs[d] exactly
    int n_r, n_theta, n_phi;
    int n_dir_eval;                         // directions evaluated: all, or the first half (in d order) of an inversion-symmetric grid
    int n_rbox, n_dbox;                     // tiles = n_dbox * n_rbox (radius box fastest)
    int sym, pad0;
    const double* te;                       // table E[rbox][row][kSphBR] = exp(-r^2/4p); zero beyond the last radius
    long long n_rows;                       // row stride of the table (the prescreened pair count)
};
cudaError_t launch_sph_table(const SphArgs& a, double* te, cudaStream_t st);
cudaError_t launch_ff_sph(int NS, const SphArgs& a, cudaStream_t st);
cudaError_t ff_sph_init_device();
cudaError_t launch_separable(const GridArgs& a, const double* wx, const double* wy, const double* wz, double* mom, double* part,
                             int per_block, cudaStream_t st);   // grids sized for a.n_rows records; part[block][16] complex

// angular moments (angular.cu, NEXT-3)
void angular_host_tables(int l_max, int n_theta, const double* cos_theta, const double* w_theta, int n_phi,
                         std::vector<double>& Yw, std::vector<double>& tw);
cudaError_t angular_init_device();           // per-device function attributes; idempotent
constexpr int kAngularMaxSmem = 200 * 1024;  // dynamic shared memory the fused kernel may use (B fragments + F rows)
void angular_fragment_table(int l_max, int n_phi, std::vector<double>& Bf, int& n_nt, int& n_ks);
void angular_transpose_table(int l_max, int n_theta, const std::vector<double>& Yw, std::vector<double>& YwT);
int angular_chunk_table(int l_max, int n_theta, const std::vector<double>& Yw, std::vector<double>& YwC);   // returns the chunk size in bytes
size_t angular_fused_smem(int n_theta, int l_max, int n_nt, int n_ks, bool fused);
// F_glob == nullptr: fused (R, f2 written); else F [n_sr][n_theta][2 l_max + 1] complex and row2 [n_sr][n_theta] are written instead
cudaError_t launch_angular_fused(const double* f, const double* Bf, const double* YwT, const double* w_theta, long long n_sr, int n_theta,
                                 int n_phi, int l_max, int n_nt, int n_ks, double* R, double* f2, double* F_glob, double* row2_glob,
                                 const double* YwC, int chunk_bytes, cudaStream_t st);   // YwC: chunked weight table (staged Legendre step) or nullptr
cudaError_t launch_phi_dft(const double* f, const double* tw, long long n_rows, int n_phi, int l_max, double* F, double* rowsum2,
                           cudaStream_t st);
cudaError_t launch_legendre(const double* F, const double* rowsum2, const double* Yw, const double* w_theta, long long n_sr,
                            int n_theta, int l_max, double* R, double* f2, cudaStream_t st);

cudaError_t launch_abs2(const double* f_complex, long long n, double* out, cudaStream_t st);   // S5: |f|^2

// pure (solid-harmonic) shells (pure.cu, NEXT-5): T_cart = C T_user C^T
constexpr int kPureMaxNnz = 4;              // user functions one Cartesian component contributes to, at most
void pure_matrix(int l, double* C);         // [ncart(l)][2l+1]
int build_pure_map(int n_shells, const int32_t* shell_l, const int32_t* shell_pure, std::vector<int>& nnz, std::vector<int>& uidx,
                   std::vector<double>& ucoef);
cudaError_t launch_transform_T(const double* Tu, double* Tc, int n_states, int nbf_u, int nbf_c, const int* nnz, const int* uidx,
                               const double* ucoef, cudaStream_t st);

// FFT method (fft_method.cu, NEXT-4)
struct FftGrid {
    int nx, ny, nz, pad;
    long long P;                            // nx*ny*nz
    double xmin[3], len[3];
};
cudaError_t launch_orbitals(const PrimShell* prim, const int* shell_first, int n_shells, int nbf, const FftGrid& g, double* V,
                            cudaStream_t st);   // V in tiles of 8 points: [(P+7)/8][nbf][8]
cudaError_t launch_density(const double* V, const double* T, int nbf, long long P, int s0, int ns, double g, double* out_complex,
                           cudaStream_t st);
cudaError_t launch_density_mma(const double* V, const double* T, double* Csym, int nbf, int nbf_pad, long long P, int s0, int ns,
                               double g, double* out_complex, cudaStream_t st);
constexpr int kDensityFusedMaxSmem = 225 * 1024;
cudaError_t density_fused_init_device();
bool density_fused_fits(int nbf_pad);        // the orbital tile of 16 points fits in shared memory
cudaError_t launch_symmetrize(const double* T, double* Csym, int nbf, int nbf_pad, int s0, int ns, cudaStream_t st);
cudaError_t launch_density_fused(const PrimShell* prim, const int* shell_first, int n_shells, const FftGrid& g, const double* Csym, int nbf,
                                 int nbf_pad, int s0, int ns, double gfac, double* out_complex, cudaStream_t st);
// Parseval sums (Eq. 75): out[s * stride + col] = scale * sum_i |a[s][i]|^2; scratch holds ns * 256 doubles
cudaError_t launch_sumsq(const double* a_complex, long long P, int ns, double scale, double* scratch, double* out, int stride, int col,
                         cudaStream_t st);
cudaError_t launch_fft_post(const double* F, const FftGrid& g, int ns, double* out, cudaStream_t st);
struct CufftPlan { int handle = -1, nx = 0, ny = 0, nz = 0; };   // owned by a context, tied to its device
int cufft_inverse_batch(CufftPlan& pl, double* data, int nx, int ny, int nz, int ns, cudaStream_t st);
void cufft_plan_release(CufftPlan& pl);

cudaError_t run_fp64_peak(double* dfma_per_s, double* sm_clock_mhz);

}  // namespace scarf

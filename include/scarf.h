/*
 * scarf.h — C ABI of libscarf: analytic 3-D molecular scattering form factors on one B200 (sm_100a).
 *
 *     f_s(q) = g * sum_{mu nu} T^s_{mu nu} * Int d^3r  phi_mu(r) phi_nu(r) exp(i q.r)          (g = 2)
 *
 * This is the "Cartesian grid method" of arxiv 2512.18010 (SCarFFF): Eq. (35) /root/reference/PAPER.md:244,
 * evaluated in closed form as Eq. (48)-(50) PAPER.md:326-338 (the monomial D-tensor form) for a stack of
 * transition density matrices T^s over an arbitrary list of momentum-transfer vectors q, all in FP64.
 * The paper defines no API (it is a script-driven Julia package); the calls below follow its
 * statement that the method "depends only on the availability of a transition density matrix and a
 * selection of any Gaussian basis set" plus geometry.
 *
 * Pipeline:
 *   scarf_set_basis        S0 orbital normalisation, Eq. (A1)-(A5) PAPER.md:619-641;
 *                          S1 primitive-shell-pair setup = Gaussian product, Eq. (37)-(39), (43) PAPER.md:263-300;
 *                          S2 per-axis Hermite expansion coefficients (McMurchie-Davidson recurrences; they equal
 *                             K_AB * C^u / i^u of Eq. (50)).            Host work + one upload.
 *   scarf_set_transitions  S3 fold T^s into per-pair coefficients D^s (Eq. (48)-(49)), screen,
 *                             pack the pair stream.                                  Device kernels.
 *   scarf_form_factors     S4 the hot kernel: for every q, sum over pairs of
 *                             exp(-q^2/4p) e^{i q.P} sum_t D^s_t (i q)^t  (Eq. (48)). Device kernel(s).
 * Around it: scarf_form_factors_grid / scarf_separable_integral (product grids: per-axis factor
 * tables, Eq. (45)-(46), (64)-(65)), scarf_angular_moments (R_lm and <f^2>_Omega, Eq. (57)-(60)),
 * scarf_fft_form_factors (the paper's FFT method, Eq. (19)-(34); approximate), scarf_set_basis_pure (solid-harmonic
 * d/f shells, Eq. (A2)), option "threshold_eps" (paper-style thresholding).
 *
 * Conventions
 *   - Atomic units: positions in bohr, exponents in bohr^-2, q in bohr^-1.  No unit conversion happens here.
 *   - Fourier sign e^{+i q.r} (Eq. 19), so f(-q) = conj f(q) for real T.
 *   - Cartesian components of a shell of angular momentum l: (a,b,c), a+b+c = l, a descending then b
 *     descending: p = x,y,z; d = xx,xy,xz,yy,yz,zz; f = xxx,xxy,xxz,xyy,xyz,xzz,yyy,yyz,yzz,zzz.
 *     Every component is individually normalised to 1.  Basis functions are numbered shell by
 *     shell in this component order.
 *   - Contraction coefficients multiply unit-normalised primitives (Eq. A3); the contracted orbital
 *     is then renormalised (Eq. A5).
 *   - Every call returns SCARF_OK (0) or a negative SCARF_E* code; scarf_last_error() holds the text.  No C++
 *     exception crosses this boundary.  There is no mutable process-wide state: device constant tables are
 *     compile-time initialised, kernel attributes are set per context at scarf_create, the cuFFT plan belongs to
 *     the context (the only process-wide object is the immutable cuFFT function table, loaded once under
 *     std::call_once).  A context is not thread-safe; distinct contexts are independent and may be driven from
 *     different threads and on different devices.  ONE exception, by design: scarf_form_factors_noalloc keeps its scratch
 *     in a static device array shared by all contexts on a device (see there); no other call touches it.
 *   - Argument range: |q . P| <= 2^30 for every Gaussian-product centre P (i.e. |q| * molecular extent < 1e9);
 *     full accuracy of the phase needs |q . P| <~ 1e5.  e^{-q^2/4p} underflows to (effectively) 0 for large |q|, any
 *     finite q is safe there.  Host q arrays are checked for NaN/Inf; device arrays are not.
 *   - Inputs are COPIED during set_* (the caller keeps ownership and may free at once).  Outputs are caller-owned.
 *   - "host or device" pointers are classified with cudaPointerGetAttributes: device and managed memory are used
 *     in place; pinned or pageable host memory is staged through context-owned device buffers and the call
 *     returns after the copy back has completed.  With device pointers the work is asynchronous on the context
 *     stream.
 *   - There is NO CPU fallback: without a usable CUDA device scarf_set_transitions / scarf_form_factors fail with
 *     SCARF_ENODEVICE.
 */
#ifndef SCARF_H
#define SCARF_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SCARF_OK 0
#define SCARF_EINVAL (-1)    /* bad argument, shape, l > SCARF_MAX_L, non-positive exponent, NaN/Inf in host input */
#define SCARF_ESTATE (-2)    /* calls out of order (e.g. form_factors before set_transitions)                      */
#define SCARF_ENOMEM (-3)    /* host or device allocation failed                                                   */
#define SCARF_ECUDA (-4)     /* CUDA runtime error; text in scarf_last_error                                       */
#define SCARF_ENODEVICE (-5) /* the context was created host-only (device < 0) or no device is usable              */

#define SCARF_MAX_L 6        /* highest shell angular momentum (i); pair classes L = l_a + l_b <= 12  */
#define SCARF_N_CLASSES (2 * SCARF_MAX_L + 1)

typedef struct scarf_ctx scarf_ctx; /* opaque; owns every device buffer it allocates */

/* Counters filled by scarf_get_stats.  "pair" = primitive shell pair (A,k) <= (B,k'). */
typedef struct scarf_stats {
    int32_t n_atoms, n_shells, n_prim_shells, nbf, n_states, l_max;
    int64_t n_pairs_all;                       /* all primitive shell pairs, A <= B                                 */
    int64_t n_pairs_prescreened;               /* after the T-independent host screen (K_AB underflow)              */
    int64_t n_pairs_kept;                      /* after the T-dependent bound screen (set_transitions); the screening
                                                * runs on the device and scarf_get_stats WAITS for its result        */
    int64_t pairs_kept_per_class[SCARF_N_CLASSES];
    int64_t n_herm_kept;                       /* sum over kept pairs of n_herm(L) = (L+1)(L+2)(L+3)/6              */
    int64_t cart_term_pairs;                   /* ordered Cartesian-term pairs, the paper's N_c^2 (Eq. 68)          */
    double stream_bytes;                       /* packed pair stream read by the hot kernel                         */
    double slots_per_q;                        /* FP64 issue-slot model per q-point        */
    double evals_per_q;                        /* kept pairs x states                                               */
    double last_setup_host_ms;                 /* scarf_set_basis host time                                         */
    double last_fold_ms, last_kernel_ms;       /* device time of the last S3 / S4 (CUDA events; 0 until queried)    */
    int32_t last_kernel_launches;              /* kernels launched by the last scarf_form_factors                   */
    int32_t last_fold_launches;                /* kernels launched by the last scarf_set_transitions               */
    double last_grid_slots;                    /* FP64 issue-slot model of the last scarf_form_factors_grid call    */
    double dropped_bound;                      /* sum of the bounds B_P of all dropped pairs: |f_s(q) - exact| <= this, any q, s */
    int32_t last_grid_symmetric;               /* 1 if the last scarf_form_factors_grid call used f(-q) = conj f(q)  */
    int32_t last_n_chunks;                     /* stream chunks (= cluster size) of the last S4 launch                */
    double last_main_kernel_ms;                /* "timing": device time of the S4 kernel(s) alone (no tables/planning)*/
    double last_grid_kernel_slots;             /* FP64 issue-slot model of the product-grid S4 kernel alone (no tables)*/
    double adaptive_bound;                     /* option adaptive_tol: |f_s(q) - exact| <= this for every q, s (0 when off) */
    double last_adaptive_work_fraction;        /* modelled work of the last S4 call / work without the cut-off (1 when off) */
    int32_t last_grid_variant;                 /* kernel of the last product-grid call: 0 box, 1 row, 2 mirror-pair row (option grid_variant), 3 scarf_form_factors_sph */
    int32_t reserved0;
} scarf_stats;

/* device >= 0: CUDA ordinal.  device < 0: host-only context (set_basis, overlap, stats work; the rest ENODEVICE). */
int scarf_create(scarf_ctx** out, int device);
void scarf_destroy(scarf_ctx* ctx);

/* cuda_stream: a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = the legacy default stream. */
int scarf_set_stream(scarf_ctx* ctx, void* cuda_stream);

/* Options.  "prefactor": g, default 2.0 (Eq. 18, spin sum); takes effect at the next set_transitions.
 *           "screen_tol": default 1e-16; a pair is dropped when its rigorous bound
 *                         B_P = max_s sum_t |D^s_t| sup_q |q|^n e^{-q^2/4p} is below screen_tol * mean(B);
 *                         0 keeps everything.  The paper's own epsilon = 1e-6 thresholding is an
 *                         approximation and is NOT applied.
 *           "threshold_eps": default 0 (off).  Paper-style thresholding ("discarding all Cartesian pair
 *                         index combinations for which |M T / (M T)_max| < epsilon"), restated on this library's unit:
 *                         a primitive shell pair is also dropped when B_P < threshold_eps * max_P B_P (B_P already is
 *                         the max over the states, so a pair survives if any transition needs it).  An APPROXIMATION
 *                         whose error is bounded: scarf_stats.dropped_bound.  Takes effect at set_transitions.
 *           "adaptive_tol": default 0 (off).  q-adaptive evaluation: with tau = adaptive_tol *
 *                         mean(B), a kept pair P is skipped for the q tiles that lie entirely beyond q_cut(P), the radius
 *                         past which its rigorous envelope sum_n c_n sup_{q' >= q} q'^n e^{-q'^2/4p} stays below tau
 *                         (e^{-q^2/4p} kills diffuse pairs at large |q|).  An APPROXIMATION with a reported bound:
 *                         |f_s(q) - exact| <= scarf_stats.adaptive_bound = n_kept * tau <= adaptive_tol * sum(B) for every
 *                         q and s; scarf_stats.last_adaptive_work_fraction says how much work was left.  Records are
 *                         re-ordered by q_cut inside their class (results differ from the default path by round-off
 *                         even where nothing is skipped).  Takes effect at set_transitions; at most 96 states.
 *           "timing": 1 records CUDA-event times of S3/S4 into the stats (adds a stream sync per call).
 *           "n_chunks": default 0 (automatic).  1..32 forces the number of cost-balanced slices the pair stream is cut
 *                         into (the S4 grid is q-tiles x chunks; the chunks of one q tile add their partial sums into
 *                         `out` in chunk order, so results agree to FP64 round-off for any value).  A tuning/testing knob.
 *           "grid_symmetry": default 1.  scarf_form_factors_grid evaluates only one half of a product grid whose three
 *                         axes are antisymmetric bit for bit (ax[i] == -ax[n-1-i]) and stores conj f for the mirror
 *                         points (f(-q) = conj f(q), exact for real T); 0 always evaluates every point.
 *           "host_zero_copy": default 1.  When `out` of scarf_form_factors_grid is PINNED host memory
 *                         (cudaHostAlloc / cudaHostRegister; torch's pin_memory), the kernel stores the finished values straight
 *                         into it through its mapped device alias — the output crosses PCIe while the kernel runs and no
 *                         device->host copy follows; partial sums stay on the device.  0: always compute on the device and copy.
 *                         Pageable host memory always takes the copy.  The call returns when `out` is complete either way.
 *           "host_tile_group": default 0 (automatic).  Tiles per dispatch group of the product-grid kernels when they write a
 *                         pinned host `out` (see host_zero_copy).  A tuning/testing knob; results do not depend on it.
 *           "grid_tile_group": default -1 (automatic).  Tiles per dispatch group of the product-grid kernels when `out` is device
 *                         memory: the CTAs run chunk-major inside groups of this many tiles, group after group, so that CTAs
 *                         working on different pair classes (FP64-pipe loops, tensor-core loops) share an SM.  0 = chunk-major
 *                         over all tiles.  A tuning/testing knob; results do not depend on it.
 *           "grid_variant": default -1 (automatic).  Kernel of scarf_form_factors_grid: 0 = box kernel (a CTA owns a 4 x 8 x 8
 *                         box of the grid; the two points of a thread share (q_y, q_z)), 1 = row kernel (a warp owns 64
 *                         consecutive z-points of one (ix, iy) row, so the (q_x, q_y) part of every polynomial is evaluated
 *                         once per warp: fewer FP64 operations per point, but lanes beyond the end of a row idle), 2 = mirror-pair
 *                         row kernel (needs a z axis with qz[i] == -qz[nz-1-i] bit for bit, else the choice is automatic: a lane
 *                         owns the points +z and -z of its row and accumulates their half sum and half difference, whose
 *                         polynomials in z^2 are shared by the pair), -1 = the mirror-pair kernel when the z axis allows it and
 *                         its 4 (y) x 32 (pairs) boxes are at least 75 % full, else the row kernel when its 4 x 64 boxes are at least 80 % full,
 *                         else the box kernel.  Same results to round-off.
 *           "fft_density_variant": default 1 = FP64 tensor-core (DMMA) density kernel of scarf_fft_form_factors with the
 *                         orbital values evaluated per point tile in shared memory (falls back to 2 when the tile of a
 *                         very large basis does not fit), 2 = DMMA kernel reading orbital values tabulated in device
 *                         memory (nbf * nx*ny*nz doubles of scratch), 0 = SIMT kernel on the same table (same results to
 *                         round-off; slower).
 *           "check_parseval": default 0.  1: scarf_fft_form_factors also evaluates both sides of Parseval's relation
 *                         (Eq. 75, the paper's check_parseval flag); read them with scarf_fft_parseval.
 *           "angular_variant": default 1 = fused FP64 tensor-core kernel of scarf_angular_moments, 0 = SIMT kernels
 *                         (same result to round-off; slower).
 *           Unknown keys and out-of-range values: SCARF_EINVAL.                                                      */
int scarf_set_option(scarf_ctx* ctx, const char* key, double value);

/* HOST pointers.  atom_xyz [n_atoms][3].  Shell i sits on atom shell_atom[i], has angular momentum shell_l[i]
 * (0..SCARF_MAX_L) and shell_nprim[i] >= 1 primitives taken consecutively from exponents[] / coeffs[].
 * Invalidates any transitions set before. */
int scarf_set_basis(scarf_ctx* ctx, int n_atoms, const double* atom_xyz, int n_shells, const int32_t* shell_atom,
                    const int32_t* shell_l, const int32_t* shell_nprim, const double* exponents,
                    const double* coeffs);

/* As scarf_set_basis, with shell_pure[i] != 0 marking shell i as PURE (real solid harmonics, 2l+1 functions, order
 * m = -l..l: d = xy, yz, 2z^2-x^2-y^2, xz, x^2-y^2; f = y(3x^2-y^2), xyz, y(4z^2-x^2-y^2), z(2z^2-3x^2-3y^2),
 * x(4z^2-x^2-y^2), z(x^2-y^2), x(x^2-3y^2); each normalised to 1) — the multi-term Cartesian orbitals of Eq. (A2)
 * PAPER.md:625-627.  The flag is ignored for l < 2.  shell_pure == NULL: all Cartesian.  scarf_nbf, scarf_overlap
 * and the T of scarf_set_transitions are then in that mixed basis; internally T_cart = C T C^T. */
int scarf_set_basis_pure(scarf_ctx* ctx, int n_atoms, const double* atom_xyz, int n_shells, const int32_t* shell_atom,
                         const int32_t* shell_l, const int32_t* shell_nprim, const double* exponents,
                         const double* coeffs, const int32_t* shell_pure);

int scarf_nbf(const scarf_ctx* ctx); /* number of contracted Cartesian basis functions, or a negative code */

/* AO overlap S[nbf][nbf] (= Int phi_mu phi_nu, the q = 0 pair integral) into HOST memory, from the S1/S2 tables. */
int scarf_overlap(scarf_ctx* ctx, double* S_host);

/* T [n_states][nbf][nbf], row-major FP64, real, need not be symmetric.  Host or device pointer.
 * May be called repeatedly on one basis.  Everything runs on the context stream without a device->host round trip:
 * fold, screening (threshold, stable compaction), packing and the stream descriptor stay on the device; the kept-pair
 * counts reach the host only through scarf_get_stats.  Host T is checked for NaN/Inf here (SCARF_EINVAL); device T is
 * checked on the device: a non-finite T keeps every pair (the NaN reaches the output) and SCARF_EINVAL is returned by
 * scarf_get_stats and by the next S4 call that finds the screening result already on the host. */
int scarf_set_transitions(scarf_ctx* ctx, int n_states, const double* T);

/* q [n_q][3] FP64; out [n_states][n_q][2] FP64 (re, im interleaved).  Host or device pointers, independently.
 * Any point set (no grid structure is assumed).  May be called repeatedly. */
int scarf_form_factors(scarf_ctx* ctx, int64_t n_q, const double* q, double* out);

/* The same call for callers that must not allocate (CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): Eq. (48) PAPER.md:326-330 with the same kernels and the same chunking as scarf_form_factors, so the result is
 * bit-identical to it.  This entry point calls no cudaMalloc/cudaFree and no allocating library routine, and never
 * synchronises: it only enqueues work on the context stream.
 *   q [n_q][3], out [n_states][n_q][2]: DEVICE pointers, both owned by the caller (host pointers: SCARF_EINVAL — staging
 *   them would need an allocation).
 *   Scratch: the per-tile tickets of the ordered chunk fix-up (one int per tile of 256 q-points) live in a static device
 *   array of SCARF_NOALLOC_MAX_TILES entries (256 KB, held by every GPU that loads the library until the process exits)
 *   instead of a context buffer.  n_q > 256 * SCARF_NOALLOC_MAX_TILES = 16 777 216 is rejected with SCARF_EINVAL and a
 *   message naming the limit; cut larger point sets into several calls.
 *   The array is shared by ALL contexts of the process on that device and keeps the last call's contents; every call clears
 *   the entries it uses (on the context stream) before its kernel.  Calls that overlap on the GPU — two contexts on
 *   different streams — race on it: serialise such calls (one stream, or events).  Calls on one stream are ordered.
 *   Needs a context that has seen set_basis and set_transitions (those allocate; call them before the capture / the loop).
 *   The option "timing" is ignored here (its event synchronisation would block); stats carry launches and chunk count. */
#define SCARF_NOALLOC_MAX_TILES 65536
int scarf_form_factors_noalloc(scarf_ctx* ctx, int64_t n_q, const double* q_dev, double* out_dev);

/* The same f_s(q) on a Cartesian PRODUCT grid q = (qx[ix], qy[iy], qz[iz]), out index (ix*ny + iy)*nz + iz:
 * out [n_states][nx*ny*nz][2].  On such a grid the pair factor separates per axis (the V-tensor idea of Eq. (45)-(46)
 * PAPER.md:309-316): e^{-q^2/4p} e^{iq.P} = X_P(ix) Y_P(iy) Z_P(iz).  The three factors of every kept pair are
 * tabulated once per call (nx+ny+nz complex numbers per pair, device memory owned by the context) and the kernel
 * spends 2 complex multiplies per (q, pair) instead of an exp and a sincos.  Axes need not be uniform or sorted.
 * qx, qy, qz and out: host or device pointers, independently.  Results equal scarf_form_factors on the expanded
 * point list up to FP64 round-off.  SCARF_ENOMEM if the tables would exceed 32 GB.
 * Inversion symmetry (option "grid_symmetry", default on): the axes are inspected on the host; HOST axes cost nothing,
 * DEVICE axes are read back first (a few hundred bytes and one stream synchronisation per call) — pass the axes from
 * host memory when the call must stay asynchronous.  scarf_stats.last_grid_symmetric says which path ran. */
int scarf_form_factors_grid(scarf_ctx* ctx, int32_t nx, const double* qx, int32_t ny, const double* qy, int32_t nz,
                            const double* qz, double* out);

/* The same f_s(q) on a SPHERICAL product grid — the grid of scarf_angular_moments (Eq. (57)-(60) PAPER.md:380-398):
 *     q = r[i] (sin t_j cos phi_k, sin t_j sin phi_k, cos t_j),  cos t_j = cos_theta[j],  phi_k = 2 pi k / n_phi,
 * out [n_states][n_r][n_theta][n_phi][2], point index (i*n_theta + j)*n_phi + k — exactly the input layout of
 * scarf_angular_moments.  Along one direction n the polynomial of Eq. (48) PAPER.md:326-330 is a polynomial in r whose
 * coefficients (the sums of D over each total degree, weighted with the monomials of n) and the phase slope n.P are the same for
 * every radius: they are evaluated once per (direction, pair, state), the Gaussian e^{-r^2/4p} comes from a table per (pair, radius).
 * Inversion symmetry (option "grid_symmetry", default on): when cos_theta[j] == -cos_theta[n_theta-1-j] bit for bit (Gauss-Legendre
 * nodes) and n_phi is even, -q of a grid point is a grid point; half of the directions are evaluated and the mirror points get
 * conj f (f(-q) = conj f(q), exact for real T).  The library builds the direction table itself (mirror directions are the exact
 * negatives): its points agree with a caller's own list of the same grid to FP64 round-off of the trigonometric functions.
 * r, cos_theta: HOST pointers (r finite, |cos_theta| <= 1).  out: host or device; with a device `out` the call is asynchronous
 * on the context stream.  Results equal scarf_form_factors on the expanded point list up to FP64 round-off.  Bases with
 * g, h, i shells run that list path internally.  scarf_stats: last_grid_symmetric, last_grid_variant = 3, last_grid_kernel_slots. */
int scarf_form_factors_sph(scarf_ctx* ctx, int32_t n_r, const double* r, int32_t n_theta, const double* cos_theta, int32_t n_phi,
                           double* out);

/* Separable integrals (Eq. (64)-(65) PAPER.md:481-487): the weighted sum of f_s over a Cartesian product grid,
 *     out[s] = sum_{ix,iy,iz} fx[ix] gy[iy] hz[iz] f_s(qx[ix], qy[iy], qz[iz])        (fx = quadrature weight x f(qx), ...),
 * i.e. a quadrature of I_sep = Int d^3q f(q_x) g(q_y) h(q_z) f_s(q), evaluated WITHOUT forming f_s on the grid: per pair
 * the three 1-D moments sum_i fx[i] qx[i]^t X_P(i) are contracted with the folded coefficients, so the cost is linear in
 * nx + ny + nz (the paper's use of the V-tensors).  All pointers HOST; out [n_states][2]. */
int scarf_separable_integral(scarf_ctx* ctx, int32_t nx, const double* qx, const double* fx, int32_t ny, const double* qy,
                             const double* gy, int32_t nz, const double* qz, const double* hz, double* out);

/* Angular moments of form factors given on a spherical product grid:
 *     f_s(q) = sum_lm Y_l^m(qhat) R_lm(q)   (Eq. 57)   =>   R_lm(q) = Int dOmega conj(Y_l^m(qhat)) f_s(q),
 *     <f_s^2>_Omega = Int dOmega/4pi |f_s(q)|^2                       (Eq. 59),
 * both by the grid's own quadrature: theta nodes cos_theta[j] with weights w_theta[j] (e.g. Gauss-Legendre),
 * phi_k = 2 pi k / n_phi uniform.  Y_l^m: orthonormal, Condon-Shortley phase.
 *   f      [n_states][n_r][n_theta][n_phi][2]  (re, im) — the layout scarf_form_factors writes for the point list
 *          q = r_i (sin t_j cos phi_k, sin t_j sin phi_k, cos t_j), index (i*n_theta + j)*n_phi + k.  Host or device.
 *   R_out  [n_states][n_r][(l_max+1)^2][2], index l(l+1)+m.  Host or device.
 *   f2_out [n_states][n_r] or NULL.  Host or device.
 *   cos_theta, w_theta: HOST.  Needs n_phi >= 2 l_max + 1 (no phi aliasing), n_phi <= 2048, l_max <= 64; exact for
 *   band limit l + l' <= 2 n_theta - 1 with Gauss-Legendre nodes.  Independent of the basis and transitions set.
 *   The quadrature tables are cached in the context (rebuilt only when nodes, weights, n_phi or l_max change); with
 *   device pointers for f, R_out and f2_out the call is asynchronous on the context stream. */
int scarf_angular_moments(scarf_ctx* ctx, int32_t n_states, int32_t n_r, int32_t n_theta, const double* cos_theta,
                          const double* w_theta, int32_t n_phi, int32_t l_max, const double* f, double* R_out,
                          double* f2_out);

/* S5, the optional output of the hot path: out[i] = |f[i]|^2 for n complex values (what Fig. 6 plots), e.g.
 * n = n_states * n_q of a form-factor array.  f [n][2], out [n]: host or device pointers, independently; asynchronous on
 * the context stream when both are device pointers. */
int scarf_abs2(scarf_ctx* ctx, int64_t n, const double* f, double* out);

/* Oscillator-strength fit, Eq. (81)-(82) PAPER.md:591-596: least squares of  <|f_s|^2>_Omega(q) ~ A + B q^2 + C q^4  over the
 * radial points with |q_abs[i]| <= q_max (q_max <= 0: all of them; at least three distinct |q| are needed).  f2 is the
 * [n_states][n_r] array scarf_angular_moments returns, q_abs [n_r] the radii; coef_out [n_states][3] = (A, B, C).
 * B = |g mu|^2 / 3 with mu the transition dipole of Eq. (77) and g the prefactor the form factors were computed with
 * (f_s -> i g q.mu, Eq. 76); A absorbs a non-zero f(0), C the finite-q curvature.  HOST pointers; no device work. */
int scarf_oscillator_fit(int32_t n_states, int32_t n_r, const double* q_abs, const double* f2, double q_max, double* coef_out);

/* The paper's FFT method (Section III, Eq. (19)-(34) PAPER.md:140-222) as a second, APPROXIMATE
 * route to f_s: the transition density Phi_s(x) = g sum_pq T_pq phi_q(x) phi_p(x) (Eq. 20) is tabulated at
 * x_abc = x_min + box_len * (a/nx, b/ny, c/nz) (Eq. 25-28) and transformed (cuFFT, loaded at first use),
 *     out[s][(ia*ny + ib)*nz + ic] = V_pix sum_abc Phi_abc exp(+i q.x_abc),  q = 2 pi ((ia - nx/2)/box_len[0], ...)
 * (Eq. 27, 30-33; integer division; "most negative frequencies first").  Accuracy is set by the box (truncation) and
 * the spacing (aliasing beyond pi/h), not by this library.  x_min, box_len: HOST double[3].  out [n_states][nx*ny*nz][2],
 * host or device.  Scratch: 2 complex arrays of the output size (+ nbf*nx*ny*nz doubles with fft_density_variant 0 or 2;
 * SCARF_ENOMEM above 64 GB). */
int scarf_fft_form_factors(scarf_ctx* ctx, int32_t nx, int32_t ny, int32_t nz, const double* x_min, const double* box_len,
                           double* out);

/* Parseval check of the FFT method, Eq. (75):  Int d^3r |Phi_s(r)|^2 = Int d^3q/(2 pi)^3 |f_s(q)|^2, on the grids
 * of the last scarf_fft_form_factors call made with option "check_parseval" = 1:
 *     out[s][0] = V_pix sum_abc |Phi_abc|^2,      out[s][1] = (1 / (Lx Ly Lz)) sum_q |f_s(q)|^2      (d^3q/(2 pi)^3 = 1/V_box per point).
 * The two agree to round-off for ANY box (discrete Parseval), so a mismatch flags a broken transform/normalisation, while
 * comparing out[s][0] across boxes/spacings shows truncation and aliasing ("grids with insufficient extent or resolution").
 * out: HOST [n_states][2].  Synchronises the context stream.  SCARF_ESTATE if no checked call was made. */
int scarf_fft_parseval(scarf_ctx* ctx, double* out_host);

int scarf_get_stats(scarf_ctx* ctx, scarf_stats* out);
const char* scarf_last_error(const scarf_ctx* ctx);
const char* scarf_version(void);

/* Measured FP64 issue peak of the device: runs a register-only chain of dependent-free DFMAs on every SM and
 * returns lane-level DFMA per second (1 "slot" = 2 flop) and the SM clock (MHz) observed during the run.
 * This is the denominator of the roofline fraction bench.py reports. */
int scarf_fp64_peak(int device, double* dfma_per_s, double* sm_clock_mhz);

/* Host-side building blocks, exported so the CPU test-suite can pin them without a GPU.
 * scarf_host_hermite_E: E[(la+1)][(lb+1)][(la+lb+1)] for one axis, McMurchie-Davidson:
 *     (x-Ax)^i (x-Bx)^j e^{-alpha (x-Ax)^2 - beta (x-Bx)^2} = sum_t E_t^{ij} (d/dPx)^t e^{-p (x-Px)^2}.
 * scarf_host_shell_norms: c[(component, primitive)] effective coefficients of one shell, component-major. */
int scarf_host_hermite_E(int la, int lb, double alpha, double beta, double Ax, double Bx, double* E_out);
int scarf_host_shell_norms(int l, int nprim, const double* exponents, const double* coeffs, double* c_out);
/* scarf_host_ylm_table: the theta part of scarf_angular_moments' quadrature, Yw[j][l(l+1)/2 + m] =
 * w_theta[j] * N_lm P_l^m(cos_theta[j]) for 0 <= m <= l <= l_max (orthonormal Y_l^m = N_lm P_l^m e^{i m phi},
 * Condon-Shortley phase); Yw_out [n_theta][(l_max+1)(l_max+2)/2]. */
int scarf_host_ylm_table(int l_max, int n_theta, const double* cos_theta, const double* w_theta, double* Yw_out);

#ifdef __cplusplus
}
#endif
#endif /* SCARF_H */

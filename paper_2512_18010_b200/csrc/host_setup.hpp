// host_setup.hpp — S0 (normalisation), S1 (primitive-shell-pair setup) and S2 (Hermite expansion coefficients)
// of SURVEY.md §8(a), on the host, in the standard alpha-parameterisation of quantum chemistry
// (alpha = 1/(2 sigma^2); PAPER.md:625 Eq. A2).  Derivation route: Gaussian product theorem +
// McMurchie-Davidson recurrences; this is deliberately NOT the paper's binomial/Hermite-polynomial route
// (Eq. 40-50), which the oracle follows.  The two are bridged by E_u = K_AB C^u / i^u.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace scarf {

constexpr int kMaxL = 6;                    // highest shell angular momentum (i; "up to i orbitals")
constexpr int kMaxClass = 2 * kMaxL;        // highest pair class L = la + lb
constexpr int kNClasses = kMaxClass + 1;

inline constexpr int ncart(int l) { return (l + 1) * (l + 2) / 2; }
inline constexpr int nherm(int L) { return (L + 1) * (L + 2) * (L + 3) / 6; }
constexpr int kMaxCart = ncart(kMaxL);      // 28
constexpr int kMaxHerm = nherm(kMaxClass);  // 455

struct PrimShell {
    int32_t shell, atom, l, bf0;  // contracted shell it belongs to, centre, angular momentum, first basis function
    double alpha;                 // exponent
    double cprim;                 // N_shell * d_k * (2 alpha/pi)^{3/4} (4 alpha)^{l/2}   (component factor applied separately)
    double A[3];
};

// One primitive shell pair (i <= j in primitive-shell order), POD, uploaded as is for the fold kernel.
struct PairMeta {
    double Px, Py, Pz, inv4p;  // Gaussian-product centre P = (alpha A + beta B)/p and 1/(4p): the record header
    double scale;              // w (pi/p)^{3/2} cprim_i cprim_j,  w = 1/2 if i == j else 1
    double p;                  // alpha + beta
    int32_t bf0a, bf0b;        // first basis function of shell(i), shell(j)
    uint32_t e_off;            // offset (doubles) of this pair's E tables: 3 axes x (la+1)(lb+1)(L+1)
    uint8_t la, lb, L, pad;
};
static_assert(sizeof(PairMeta) == 64, "PairMeta must be 64 bytes");

struct HostSetup {
    int n_atoms = 0, n_shells = 0, nbf = 0, l_max = 0;
    std::vector<PrimShell> prim;
    std::vector<PairMeta> pairs;          // sorted by class L (stable in (i,j) order)
    std::vector<double> E;                // Hermite expansion coefficients
    int64_t n_pairs_all = 0;              // before the K_AB-underflow prescreen
    int64_t class_count[kNClasses] = {};  // prescreened pairs per class
    int64_t class_first[kNClasses + 1] = {};
    int64_t cart_term_pairs = 0;          // ordered Cartesian-term pairs (paper's N_c^2)
};

// E[(la+1)][(lb+1)][(la+lb+1)] for one axis; e000 is the value of E_0^{00} (K_AB^{(x)} or 1).
void hermite_E_axis(int la, int lb, double p, double XPA, double XPB, double e000, double* E);

// component factor 1/sqrt((2a-1)!!(2b-1)!!(2c-1)!!) of component `comp` of a shell with angular momentum l
double component_factor(int l, int comp);
void component_powers(int l, int comp, int abc[3]);

// cprim for the primitives of one shell (same for every component).
int shell_coefficients(int l, int nprim, const double* exps, const double* coefs, double* cprim_out);

// Returns 0 or a negative SCARF_E* code with `err` set.
int build_setup(int n_atoms, const double* xyz, int n_shells, const int32_t* shell_atom, const int32_t* shell_l,
                const int32_t* shell_nprim, const double* exps, const double* coefs, HostSetup& out,
                std::string& err);

// S[nbf][nbf] from the pair tables (E_0 E_0 E_0 (pi/p)^{3/2}).
void overlap_from_setup(const HostSetup& hs, double* S);

}  // namespace scarf

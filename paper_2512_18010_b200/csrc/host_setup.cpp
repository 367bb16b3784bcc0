// host_setup.cpp — see host_setup.hpp.  Plain C++17, no CUDA.
#include "host_setup.hpp"

#include <algorithm>
#include <cmath>
#include <cstring>

#include "../../include/scarf.h"

namespace scarf {

static const double kPi = 3.14159265358979323846;

static double double_factorial_odd(int n)  // (2n-1)!!, n >= 0
{
    double r = 1.0;
    for (int k = 1; k <= n; ++k) r *= (2 * k - 1);
    return r;
}

void component_powers(int l, int comp, int abc[3])
{
    int idx = 0;
    for (int a = l; a >= 0; --a)
        for (int b = l - a; b >= 0; --b) {
            if (idx == comp) {
                abc[0] = a; abc[1] = b; abc[2] = l - a - b;
                return;
            }
            ++idx;
        }
    abc[0] = abc[1] = abc[2] = 0;
}

double component_factor(int l, int comp)
{
    int abc[3];
    component_powers(l, comp, abc);
    return 1.0 / std::sqrt(double_factorial_odd(abc[0]) * double_factorial_odd(abc[1]) * double_factorial_odd(abc[2]));
}

// S0.  A primitive x^a y^b z^c e^{-alpha r^2} normalised to 1 has the constant
//   (2 alpha/pi)^{3/4} (4 alpha)^{l/2} / sqrt((2a-1)!!(2b-1)!!(2c-1)!!)            (equals xi of Eq. A4).
// The self-overlap of the contracted orbital (Eq. A5) is then, for every component of the shell alike,
//   sum_{kk'} d_k d_k' (2 sqrt(alpha_k alpha_k') / (alpha_k + alpha_k'))^{l + 3/2},
// because the double factorials of the primitive constants cancel those of the Gaussian moment.
int shell_coefficients(int l, int nprim, const double* exps, const double* coefs, double* cprim_out)
{
    if (l < 0 || l > kMaxL || nprim < 1) return SCARF_EINVAL;
    double self = 0.0;
    for (int k = 0; k < nprim; ++k) {
        if (!(exps[k] > 0.0) || !std::isfinite(exps[k]) || !std::isfinite(coefs[k])) return SCARF_EINVAL;
        for (int kp = 0; kp < nprim; ++kp)
            self += coefs[k] * coefs[kp] * std::pow(2.0 * std::sqrt(exps[k] * exps[kp]) / (exps[k] + exps[kp]), l + 1.5);
    }
    if (!(self > 0.0) || !std::isfinite(self)) return SCARF_EINVAL;
    const double N = 1.0 / std::sqrt(self);
    for (int k = 0; k < nprim; ++k)
        cprim_out[k] = N * coefs[k] * std::pow(2.0 * exps[k] / kPi, 0.75) * std::pow(4.0 * exps[k], 0.5 * l);
    return SCARF_OK;
}

// S2, one axis.  McMurchie-Davidson:
//   E_t^{i+1,j} = E_{t-1}^{ij}/(2p) + X_PA E_t^{ij} + (t+1) E_{t+1}^{ij},  same with X_PB for j+1;  E_t^{ij} = 0 outside 0..i+j.
void hermite_E_axis(int la, int lb, double p, double XPA, double XPB, double e000, double* E)
{
    const int L = la + lb, nt = L + 1;
    auto at = [&](int i, int j, int t) -> double& { return E[(i * (lb + 1) + j) * nt + t]; };
    std::fill(E, E + (la + 1) * (lb + 1) * nt, 0.0);
    const double h = 0.5 / p;
    at(0, 0, 0) = e000;
    for (int i = 0; i < la; ++i)
        for (int t = 0; t <= i + 1; ++t) {
            double v = XPA * at(i, 0, t);
            if (t > 0) v += h * at(i, 0, t - 1);
            if (t + 1 <= i) v += (t + 1) * at(i, 0, t + 1);
            at(i + 1, 0, t) = v;
        }
    for (int j = 0; j < lb; ++j)
        for (int i = 0; i <= la; ++i)
            for (int t = 0; t <= i + j + 1; ++t) {
                double v = XPB * at(i, j, t);
                if (t > 0) v += h * at(i, j, t - 1);
                if (t + 1 <= i + j) v += (t + 1) * at(i, j, t + 1);
                at(i, j + 1, t) = v;
            }
}

int build_setup(int n_atoms, const double* xyz, int n_shells, const int32_t* shell_atom, const int32_t* shell_l,
                const int32_t* shell_nprim, const double* exps, const double* coefs, HostSetup& hs, std::string& err)
{
    hs = HostSetup();
    if (n_atoms < 1 || n_shells < 1 || !xyz || !shell_atom || !shell_l || !shell_nprim || !exps || !coefs) {
        err = "set_basis: null pointer or empty basis";
        return SCARF_EINVAL;
    }
    for (int i = 0; i < 3 * n_atoms; ++i)
        if (!std::isfinite(xyz[i])) {
            err = "set_basis: non-finite atom coordinate";
            return SCARF_EINVAL;
        }
    hs.n_atoms = n_atoms;
    hs.n_shells = n_shells;
    // ---- S0: primitive shells with their effective coefficients
    int bf = 0, p0 = 0;
    std::vector<double> tmp;
    for (int s = 0; s < n_shells; ++s) {
        const int l = shell_l[s], np = shell_nprim[s], at = shell_atom[s];
        if (l < 0 || l > kMaxL) {
            err = "set_basis: shell angular momentum outside 0.." + std::to_string(kMaxL);
            return SCARF_EINVAL;
        }
        if (np < 1 || at < 0 || at >= n_atoms) {
            err = "set_basis: bad shell_nprim or shell_atom";
            return SCARF_EINVAL;
        }
        tmp.resize(np);
        if (shell_coefficients(l, np, exps + p0, coefs + p0, tmp.data()) != SCARF_OK) {
            err = "set_basis: non-positive / non-finite exponent or coefficient, or a shell that normalises to zero";
            return SCARF_EINVAL;
        }
        for (int k = 0; k < np; ++k) {
            PrimShell ps;
            ps.shell = s; ps.atom = at; ps.l = l; ps.bf0 = bf;
            ps.alpha = exps[p0 + k];
            ps.cprim = tmp[k];
            for (int d = 0; d < 3; ++d) ps.A[d] = xyz[3 * at + d];
            hs.prim.push_back(ps);
        }
        hs.l_max = std::max(hs.l_max, l);
        bf += ncart(l);
        p0 += np;
    }
    hs.nbf = bf;
    // ---- S1: pairs i <= j, Gaussian product theorem, K_AB-underflow prescreen, class counting
    const int64_t np_all = (int64_t)hs.prim.size();
    hs.n_pairs_all = np_all * (np_all + 1) / 2;
    {
        int64_t nc = 0;
        for (const auto& ps : hs.prim) nc += ncart(ps.l);
        hs.cart_term_pairs = nc * nc;
    }
    struct Tmp { int32_t i, j; double mu_r2; };
    std::vector<Tmp> keep[kNClasses];
    const double kDropExp = 120.0;  // K_AB = e^{-mu R^2} < 8e-53: below anything FP64 can resolve against O(1) terms
    for (int32_t i = 0; i < np_all; ++i) {
        const PrimShell& a = hs.prim[i];
        for (int32_t j = i; j < np_all; ++j) {
            const PrimShell& b = hs.prim[j];
            double r2 = 0.0;
            for (int d = 0; d < 3; ++d) r2 += (a.A[d] - b.A[d]) * (a.A[d] - b.A[d]);
            const double mur2 = a.alpha * b.alpha / (a.alpha + b.alpha) * r2;
            if (mur2 > kDropExp) continue;
            keep[a.l + b.l].push_back({i, j, mur2});
        }
    }
    int64_t total = 0;
    size_t e_total = 0;
    for (int c = 0; c < kNClasses; ++c) {
        hs.class_first[c] = total;
        hs.class_count[c] = (int64_t)keep[c].size();
        total += hs.class_count[c];
        for (const auto& t : keep[c]) {
            const int la = hs.prim[t.i].l, lb = hs.prim[t.j].l;
            e_total += 3 * (size_t)(la + 1) * (lb + 1) * (la + lb + 1);
        }
    }
    hs.class_first[kNClasses] = total;
    if (e_total >= (size_t)0xFFFFFFFFu) {
        err = "set_basis: basis too large (E table offset overflow)";
        return SCARF_EINVAL;
    }
    hs.pairs.resize((size_t)total);
    hs.E.resize(e_total);
    // ---- S2: fill
    size_t e_off = 0, idx = 0;
    for (int c = 0; c < kNClasses; ++c)
        for (const auto& t : keep[c]) {
            const PrimShell& a = hs.prim[t.i];
            const PrimShell& b = hs.prim[t.j];
            PairMeta& m = hs.pairs[idx++];
            const double p = a.alpha + b.alpha;
            const double P[3] = {(a.alpha * a.A[0] + b.alpha * b.A[0]) / p, (a.alpha * a.A[1] + b.alpha * b.A[1]) / p,
                                 (a.alpha * a.A[2] + b.alpha * b.A[2]) / p};
            m.Px = P[0]; m.Py = P[1]; m.Pz = P[2];
            m.inv4p = 0.25 / p;
            m.p = p;
            const double w = (t.i == t.j) ? 0.5 : 1.0;
            m.scale = w * std::pow(kPi / p, 1.5) * a.cprim * b.cprim;
            m.bf0a = a.bf0; m.bf0b = b.bf0;
            m.la = (uint8_t)a.l; m.lb = (uint8_t)b.l; m.L = (uint8_t)(a.l + b.l); m.pad = 0;
            m.e_off = (uint32_t)e_off;
            const size_t blk = (size_t)(a.l + 1) * (b.l + 1) * (a.l + b.l + 1);
            const double K = std::exp(-t.mu_r2);
            for (int d = 0; d < 3; ++d)
                hermite_E_axis(a.l, b.l, p, P[d] - a.A[d], P[d] - b.A[d], d == 0 ? K : 1.0, hs.E.data() + e_off + d * blk);
            e_off += 3 * blk;
        }
    return SCARF_OK;
}

void overlap_from_setup(const HostSetup& hs, double* S)
{
    const int n = hs.nbf;
    std::fill(S, S + (size_t)n * n, 0.0);
    for (const PairMeta& m : hs.pairs) {
        const int la = m.la, lb = m.lb, nt = m.L + 1;
        const size_t blk = (size_t)(la + 1) * (lb + 1) * nt;
        const double* Ex = hs.E.data() + m.e_off;
        const double *Ey = Ex + blk, *Ez = Ey + blk;
        for (int ca = 0; ca < ncart(la); ++ca) {
            int A[3];
            component_powers(la, ca, A);
            const double fa = component_factor(la, ca);
            for (int cb = 0; cb < ncart(lb); ++cb) {
                int B[3];
                component_powers(lb, cb, B);
                const double fb = component_factor(lb, cb);
                const double v = m.scale * fa * fb * Ex[(A[0] * (lb + 1) + B[0]) * nt] * Ey[(A[1] * (lb + 1) + B[1]) * nt] *
                                 Ez[(A[2] * (lb + 1) + B[2]) * nt];
                // scale carries w = 1/2 on the diagonal primitive pair, where the ordered (ca, cb) loop already
                // visits both orders; adding v to both [mu][nu] and [nu][mu] is therefore right in both cases.
                S[(size_t)(m.bf0a + ca) * n + (m.bf0b + cb)] += v;
                S[(size_t)(m.bf0b + cb) * n + (m.bf0a + ca)] += v;
            }
        }
    }
}

}  // namespace scarf

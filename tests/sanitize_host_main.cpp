// ASan/UBSan driver for the library's host code (csrc/host_setup.cpp: S0-S2) — compiled and run by
// tests/test_sanitizers.py with -fsanitize=address,undefined.  Bases: every shell type s..i on three centres with
// contractions, far-apart centres (K_AB prescreen), a single s primitive; overlap from the pair tables.
#include <cmath>
#include <cstdio>
#include <string>
#include <vector>

#include "../paper_2512_18010_b200/csrc/host_setup.hpp"

using namespace scarf;

static int run(int n_atoms, const std::vector<double>& xyz, const std::vector<int32_t>& at, const std::vector<int32_t>& l,
               const std::vector<int32_t>& np, const std::vector<double>& e, const std::vector<double>& d)
{
    HostSetup hs;
    std::string err;
    const int rc = build_setup(n_atoms, xyz.data(), (int)l.size(), at.data(), l.data(), np.data(), e.data(), d.data(), hs, err);
    if (rc != 0) { std::printf("build_setup failed: %s\n", err.c_str()); return 1; }
    std::vector<double> S((size_t)hs.nbf * hs.nbf);
    overlap_from_setup(hs, S.data());
    double worst = 0.0;
    for (int i = 0; i < hs.nbf; ++i) worst = std::fmax(worst, std::fabs(S[(size_t)i * hs.nbf + i] - 1.0));
    std::printf("nbf %d pairs %zu of %lld, max |S_ii - 1| = %.2e\n", hs.nbf, hs.pairs.size(), (long long)hs.n_pairs_all, worst);
    return worst < 1e-12 ? 0 : 1;
}

int main()
{
    int bad = 0;
    {   // s..i on three centres, contracted s and g
        std::vector<double> xyz = {0, 0, -0.7, 0.3, -0.4, 0.9, 40.0, 0, 0};
        std::vector<int32_t> at, l, np;
        std::vector<double> e, d;
        for (int a = 0; a < 3; ++a)
            for (int ll = 0; ll <= kMaxL; ++ll) {
                const int n = (ll == 0 || ll == 4) ? 3 : 1;
                at.push_back(a); l.push_back(ll); np.push_back(n);
                for (int k = 0; k < n; ++k) { e.push_back(0.4 * (k + 1) * (1.0 + 0.1 * ll)); d.push_back(0.3 + 0.2 * k); }
            }
        bad += run(3, xyz, at, l, np, e, d);
    }
    {   // one s primitive
        bad += run(1, {0, 0, 0}, {0}, {0}, {1}, {1.3}, {1.0});
    }
    {   // rejected inputs must not touch memory out of bounds
        HostSetup hs;
        std::string err;
        const double xyz[3] = {0, 0, 0}, e[1] = {-1.0}, d[1] = {1.0};
        const int32_t at[1] = {0}, l7[1] = {kMaxL + 1}, l0[1] = {0}, np1[1] = {1};
        bad += build_setup(1, xyz, 1, at, l7, np1, d, d, hs, err) == 0;
        bad += build_setup(1, xyz, 1, at, l0, np1, e, d, hs, err) == 0;
    }
    std::printf(bad ? "FAILED\n" : "OK\n");
    return bad;
}

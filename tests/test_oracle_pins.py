"""Pins of the CPU oracle against things OTHER than itself (no GPU needed).

Each test names what it would catch.  Sources: the paper's printed worked examples (Eq. A7/A8), textbook
closed forms, scipy's Hermite polynomials, brute-force quadrature of the definition (tests/bruteforce.py),
and invariants of the definition (SURVEY.md §8(c) "What pins each part").
"""
import math
import os

import numpy as np
import pytest
from scipy.special import eval_hermitenorm

import workloads as W
from tests import bruteforce as bf

HERE = os.path.dirname(os.path.abspath(__file__))


def mk_basis(xyz, shells):
    """shells: list of (atom, l, [exponents], [coeffs])."""
    return W.Basis(np.array(xyz, float).reshape(-1, 3),
                   np.array([s[0] for s in shells], np.int32), np.array([s[1] for s in shells], np.int32),
                   np.array([len(s[2]) for s in shells], np.int32),
                   np.array([e for s in shells for e in s[2]], float),
                   np.array([d for s in shells for d in s[3]], float))


def unit_T(n, i, j):
    T = np.zeros((1, n, n))
    T[0, i, j] = 1.0
    return T


# --------------------------------------------------------------------------------------------------
# S0: normalisation — the paper's own worked examples (golden fixture, Eq. A7 / A8)
# --------------------------------------------------------------------------------------------------
def _golden_rows():
    rows = []
    with open(os.path.join(HERE, "golden", "appendixA_worked_examples.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            p = line.split()
            rows.append((p[0], [float(x) for x in p[1:]]))
    return rows


def test_norm_worked_examples_A7_A8(oracle_mod):
    """Catches: wrong Gamma argument / sigma power in (A4); wrong sigma_mu_nu or sqrt(2) factor in (A5)."""
    n7 = n8 = 0
    for kind, v in _golden_rows():
        if kind == "A7":
            sigma, xi_ref = v
            b = mk_basis([[0, 0, 0]], [(0, 1, [1.0 / (2 * sigma ** 2)], [1.0])])
            xi, N = oracle_mod.norms(b)
            assert xi[2] == pytest.approx(xi_ref, rel=1e-14)      # p_z is the third component (x, y, z)
            n7 += 1
        else:
            d0, d1, s0, s1, N_ref = v
            b = mk_basis([[0.3, -0.2, 0.9]], [(0, 1, [1 / (2 * s0 ** 2), 1 / (2 * s1 ** 2)], [d0, d1])])
            xi, N = oracle_mod.norms(b)
            assert N[2] == pytest.approx(N_ref, rel=1e-13)
            n8 += 1
    assert n7 >= 3 and n8 >= 3


@pytest.mark.parametrize("l", [0, 1, 2, 3])
def test_primitive_norm_textbook(oracle_mod, l):
    """xi d=1 single primitive == textbook (2a/pi)^{3/4} (4a)^{l/2} / sqrt((2a-1)!!(2b-1)!!(2c-1)!!)."""
    alpha = 0.77
    b = mk_basis([[0, 0, 0]], [(0, l, [alpha], [1.0])])
    xi, N = oracle_mod.norms(b)

    def df(n):
        return 1.0 if n <= 0 else float(np.prod(np.arange(n, 0, -2)))

    for i, (a, bb, c) in enumerate(W.cartesian_components(l)):
        ref = (2 * alpha / math.pi) ** 0.75 * (4 * alpha) ** (l / 2) / math.sqrt(df(2 * a - 1) * df(2 * bb - 1) * df(2 * c - 1))
        assert xi[i] * N[i] == pytest.approx(ref, rel=1e-13)
        assert N[i] == pytest.approx(1.0, rel=1e-13)      # one unit-normalised primitive with d = 1


# --------------------------------------------------------------------------------------------------
# 1-D building blocks
# --------------------------------------------------------------------------------------------------
def test_hermite_vs_scipy(oracle_mod):
    for x in (-2.3, -0.4, 0.0, 0.9, 3.1):
        He = oracle_mod.hermite_He(12, x)
        ref = np.array([eval_hermitenorm(n, x) for n in range(13)])
        np.testing.assert_allclose(He, ref, rtol=1e-12, atol=1e-12)


def test_shift_coeffs_vs_polynomial_product(oracle_mod):
    """Eq. (40)-(41): (x+u)^ai (x+v)^aj == sum_A b^A x^A, checked with numpy polynomial multiplication."""
    P = np.polynomial.polynomial
    for ai in range(4):
        for aj in range(4):
            u, v = 0.37, -1.21
            ref = P.polymul(P.polypow([u, 1.0], ai), P.polypow([v, 1.0], aj))
            np.testing.assert_allclose(oracle_mod.shift_coeffs(ai, aj, u, v), ref, rtol=1e-13, atol=1e-14)


def _quad1d(a, xi, si, b, xj, sj, q, h=0.01, half=25.0):
    x = np.arange(min(xi, xj) - half, max(xi, xj) + half, h)
    f = (x - xi) ** a * (x - xj) ** b * np.exp(1j * q * x - (x - xi) ** 2 / (2 * si * si) - (x - xj) ** 2 / (2 * sj * sj))
    return h * np.sum(f)


@pytest.mark.parametrize("ai,aj", [(0, 0), (1, 0), (0, 1), (1, 1), (2, 1), (2, 2), (3, 2), (3, 3)])
def test_V1d_vs_quadrature(oracle_mod, ai, aj):
    """Eq. (36)->(46): Int (x-xi)^a (x-xj)^b e^{iqx - ...} dx = sqrt(2pi) sigma_ij e^{-x_ij^2/2 sigmabar^2} V(q).
    Catches: sign of i, He argument, b^A index, X_ij weights, sigma_ij vs sigmabar_ij."""
    xi, xj, si, sj = 0.4, -1.1, 0.8, 1.3
    sij = si * sj / math.hypot(si, sj)
    pref = math.sqrt(2 * math.pi) * sij * math.exp(-(xi - xj) ** 2 / (2 * (si * si + sj * sj)))
    for q in (-3.0, -0.7, 0.0, 0.31, 2.2):
        ref = _quad1d(ai, xi, si, aj, xj, sj, q)
        got = pref * oracle_mod.V1d(ai, aj, xi, xj, si, sj, q)
        assert abs(got - ref) <= 2e-12 * max(1.0, abs(ref))


def test_hermite_derivative_identity_eq44(oracle_mod):
    """Eq. (44) via its integral form: Int x^A e^{iqx - x^2/2s^2} dx = sqrt(2pi) s (i s)^A He_A(q s) e^{-q^2 s^2/2}."""
    s = 0.9
    x = np.arange(-20, 20, 0.01)
    for A in range(7):
        for q in (-1.7, 0.0, 0.6, 2.9):
            ref = 0.01 * np.sum(x ** A * np.exp(1j * q * x - x * x / (2 * s * s)))
            got = math.sqrt(2 * math.pi) * s * (1j * s) ** A * oracle_mod.hermite_He(max(A, 1), q * s)[A] * math.exp(-q * q * s * s / 2)
            assert abs(got - ref) <= 1e-11 * max(1.0, abs(ref))


def test_C1d_monomial_equals_V1d(oracle_mod):
    """Eq. (50): exp(iqX - q^2 s^2/2) sum_u C^u q^u == V(q)  (1-D statement of Eq. 45 == Eq. 48)."""
    xi, xj, si, sj = -0.3, 0.9, 0.6, 1.1
    sij = si * sj / math.hypot(si, sj)
    X = sij ** 2 * (xi / si ** 2 + xj / sj ** 2)
    for ai, aj in [(0, 0), (1, 2), (3, 1), (3, 3)]:
        C = oracle_mod.C1d(ai, aj, xi, xj, si, sj)
        for q in (-2.0, 0.4, 1.9):
            got = np.exp(1j * q * X - q * q * sij * sij / 2) * sum(C[u] * q ** u for u in range(ai + aj + 1))
            ref = oracle_mod.V1d(ai, aj, xi, xj, si, sj, q)
            assert abs(got - ref) <= 1e-13 * max(1.0, abs(ref))


# --------------------------------------------------------------------------------------------------
# one primitive pair in 3-D: closed forms
# --------------------------------------------------------------------------------------------------
QS = np.array([[0, 0, 0], [0.3, -0.2, 0.5], [-1.5, 2.0, 0.7], [4.0, 0.0, -3.0], [0.0, 0.0, 6.0]], float)


def test_ss_closed_form(oracle_mod):
    """g N_a N_b (pi/p)^{3/2} e^{-mu|A-B|^2} e^{-q^2/4p} e^{i q.P}  (textbook Gaussian product theorem)."""
    A, B = np.array([0.1, -0.4, 0.3]), np.array([-0.9, 0.5, 1.2])
    al, be = 0.8, 2.3
    b = mk_basis([A, B], [(0, 0, [al], [1.0]), (1, 0, [be], [0.6])])
    p = al + be
    mu = al * be / p
    P = (al * A + be * B) / p
    Na, Nb = (2 * al / math.pi) ** 0.75, (2 * be / math.pi) ** 0.75
    for g in (2.0, 1.0):
        got = oracle_mod.form_factors(b, unit_T(2, 0, 1), QS, prefactor=g)[0]
        ref = g * Na * Nb * (math.pi / p) ** 1.5 * math.exp(-mu * np.sum((A - B) ** 2)) * \
            np.exp(-np.sum(QS * QS, axis=1) / (4 * p)) * np.exp(1j * QS @ P)
        np.testing.assert_allclose(got, ref, rtol=1e-13, atol=1e-15)
        got1 = oracle_mod.form_factors(b, unit_T(2, 0, 1), QS, prefactor=g, path=1)[0]
        np.testing.assert_allclose(got1, ref, rtol=1e-13, atol=1e-15)


def test_ps_same_centre_closed_form(oracle_mod):
    """Int (x-Ax) e^{-a|r-A|^2} e^{-b|r-A|^2} e^{iq.r} = (i q_x / 2p)(pi/p)^{3/2} e^{-q^2/4p} e^{iq.A}, p = a+b."""
    A = np.array([0.2, 0.7, -0.5])
    al, be = 1.3, 0.45
    b = mk_basis([A], [(0, 1, [al], [1.0]), (0, 0, [be], [1.0])])
    p = al + be
    Np = (2 * al / math.pi) ** 0.75 * math.sqrt(4 * al)
    Ns = (2 * be / math.pi) ** 0.75
    for comp in range(3):
        got = oracle_mod.form_factors(b, unit_T(4, comp, 3), QS, prefactor=1.0)[0]
        ref = Np * Ns * (1j * QS[:, comp] / (2 * p)) * (math.pi / p) ** 1.5 * \
            np.exp(-np.sum(QS * QS, axis=1) / (4 * p)) * np.exp(1j * QS @ A)
        np.testing.assert_allclose(got, ref, rtol=1e-13, atol=1e-15)


def test_overlap_textbook_sp(oracle_mod):
    """<s_A | p_z,B> = N N' (P_z - B_z) (pi/p)^{3/2} K_AB; <s_A|s_B> likewise.  Catches transposed centres."""
    A, B = np.array([0.0, 0.3, -0.8]), np.array([0.5, -0.2, 0.9])
    al, be = 0.9, 1.7
    b = mk_basis([A, B], [(0, 0, [al], [1.0]), (1, 1, [be], [1.0])])
    S = oracle_mod.overlap(b)
    p = al + be
    P = (al * A + be * B) / p
    K = math.exp(-al * be / p * np.sum((A - B) ** 2))
    Ns, Np = (2 * al / math.pi) ** 0.75, (2 * be / math.pi) ** 0.75 * math.sqrt(4 * be)
    for k in range(3):
        ref = Ns * Np * (P[k] - B[k]) * (math.pi / p) ** 1.5 * K
        assert S[0, 1 + k] == pytest.approx(ref, rel=1e-13)
        assert S[1 + k, 0] == pytest.approx(ref, rel=1e-13)


# --------------------------------------------------------------------------------------------------
# whole f_s on tiny inputs: brute-force quadrature of the definition
# --------------------------------------------------------------------------------------------------
def test_full_3d_quadrature_reduced_tiny(oracle_mod):
    """Eq. (35) on a box, 2 atoms, contracted s and p shells plus a d shell, exponents in [0.3, 3]."""
    rng = np.random.default_rng(5)
    b = mk_basis([[0, 0, -0.7], [0.2, -0.1, 0.7]],
                 [(0, 0, [2.7, 0.45], [0.5, 0.8]), (0, 1, [1.1], [1.0]),
                  (1, 0, [0.9], [1.0]), (1, 1, [1.9, 0.35], [0.3, 0.9]), (1, 2, [0.8], [1.0])])
    n = b.nbf
    T = rng.normal(size=(2, n, n))
    q = np.array([[0, 0, 0], [0.4, -0.3, 0.8], [-1.2, 0.9, 0.1], [2.0, 1.5, -2.5]], float)
    ref = bf.form_factor_3d(b, T, q, box=9.0, h=0.15)
    for path in (0, 1):
        got = oracle_mod.form_factors(b, T, q, path=path)
        assert np.max(np.abs(got - ref)) <= 1e-10 * np.max(np.abs(ref))


def test_separable_quadrature_config1(oracle_mod):
    """Config 1 exactly as generated (exponents up to 30), a handful of q-points of its grid."""
    w = W.make_workload(1, oracle_mod.overlap)
    idx = np.array([0, 17, 1234, 2048, 4095])
    q = w.q[idx]
    ref = bf.form_factor_separable(w.basis, w.T, q)
    got = oracle_mod.form_factors(w.basis, w.T, q)
    scale = np.max(np.abs(oracle_mod.form_factors(w.basis, w.T, w.q[::37])))
    assert np.max(np.abs(got - ref)) <= 1e-11 * scale


def test_separable_quadrature_with_d_and_f(oracle_mod):
    """d and f shells on different centres (component order and per-component normalisation)."""
    rng = np.random.default_rng(11)
    b = mk_basis([[0.0, 0.1, -0.6], [0.4, -0.3, 0.9]],
                 [(0, 2, [1.3, 0.5], [0.7, 0.4]), (1, 3, [0.9], [1.0]), (1, 1, [2.2], [1.0])])
    n = b.nbf
    T = rng.normal(size=(1, n, n))
    q = np.array([[0.5, -1.0, 0.25], [-2.0, 0.3, 1.7]])
    ref = bf.form_factor_separable(b, T, q, h=0.04)
    for path in (0, 1):
        got = oracle_mod.form_factors(b, T, q, path=path)
        assert np.max(np.abs(got - ref)) <= 1e-11 * np.max(np.abs(ref))


# --------------------------------------------------------------------------------------------------
# invariants of the definition
# --------------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def wl2(oracle_mod):
    return W.make_workload(2, oracle_mod.overlap)


def test_unit_diagonal_overlap_and_trace_zero(oracle_mod, wl2):
    """S_mumu = 1 and f_s(0) = g Tr(T^s S) = 0 for S-orthonormal MOs."""
    S = oracle_mod.overlap(wl2.basis)
    np.testing.assert_allclose(np.diag(S), 1.0, rtol=0, atol=5e-15)
    np.testing.assert_allclose(S, S.T, rtol=0, atol=1e-15)
    f0 = oracle_mod.form_factors(wl2.basis, wl2.T, np.zeros((1, 3)))
    ref = 2.0 * np.einsum("smn,mn->s", wl2.T, S)
    np.testing.assert_allclose(f0[:, 0], ref, rtol=0, atol=1e-13)
    assert np.max(np.abs(f0)) < 1e-13


def test_symmetries(oracle_mod, wl2):
    rng = np.random.default_rng(3)
    q = rng.uniform(-6, 6, size=(6, 3))
    b, T = wl2.basis, wl2.T[:3]
    f = oracle_mod.form_factors(b, T, q)
    scale = np.max(np.abs(f))
    # f(-q) = conj f(q): real T, real orbitals, e^{+iq.r}
    np.testing.assert_allclose(oracle_mod.form_factors(b, T, -q), np.conj(f), rtol=0, atol=1e-13 * scale)
    # only the symmetric part of T contributes
    np.testing.assert_allclose(oracle_mod.form_factors(b, np.transpose(T, (0, 2, 1)), q), f, rtol=0, atol=1e-13 * scale)
    # linearity in T and in the prefactor
    mix = 0.3 * T[0] - 1.7 * T[1]
    np.testing.assert_allclose(oracle_mod.form_factors(b, mix, q)[0], 0.3 * f[0] - 1.7 * f[1], rtol=0, atol=1e-13 * scale)
    np.testing.assert_allclose(oracle_mod.form_factors(b, T, q, prefactor=1.0), 0.5 * f, rtol=0, atol=1e-14 * scale)
    # translating every atom by a multiplies f by exp(i q.a)
    a = np.array([0.7, -1.3, 0.4])
    b2 = W.Basis(b.atom_xyz + a, b.shell_atom, b.shell_l, b.shell_nprim, b.exponents, b.coeffs)
    np.testing.assert_allclose(oracle_mod.form_factors(b2, T, q), f * np.exp(1j * q @ a)[None, :], rtol=0, atol=1e-12 * scale)


def test_small_q_dipole(oracle_mod):
    """Eq. (76)-(80): grad_q Im f_s |_0 = g sum T_{mu nu} <mu| r |nu>, dipole integrals by quadrature."""
    w = W.make_workload(1, oracle_mod.overlap)
    b, T = w.basis, w.T
    zero = np.zeros(3)
    eps = 1e-4
    for k in range(3):
        ex = tuple(1 if j == k else 0 for j in range(3))
        dip = bf.pair_matrix_separable(b, zero, extra=ex).real
        mu_ref = 2.0 * np.sum(T[0] * dip)
        dq = np.zeros((2, 3))
        dq[0, k], dq[1, k] = eps, -eps
        f = oracle_mod.form_factors(b, T, dq)[0]
        grad = (f[0].imag - f[1].imag) / (2 * eps)
        assert grad == pytest.approx(mu_ref, rel=1e-6, abs=1e-9)


def test_inversion_symmetry(oracle_mod):
    """centro-symmetric molecule => f purely imaginary for ungerade T, purely real for gerade T."""
    rng = np.random.default_rng(9)
    sh = lambda at: [(at, 0, [3.1, 0.4], [0.4, 0.7]), (at, 1, [1.2], [1.0]), (at, 2, [0.7], [1.0])]
    b = mk_basis([[0.3, -0.2, 0.8], [-0.3, 0.2, -0.8]], sh(0) + sh(1))
    n = b.nbf
    half = n // 2
    ls = np.concatenate([np.full((l + 1) * (l + 2) // 2, l) for l in (0, 1, 2)])
    sign = (-1.0) ** ls

    def invert(c):      # (I c): orbital on atom 0 <-> same orbital on atom 1, times (-1)^l
        out = np.empty_like(c)
        out[:half], out[half:] = sign * c[half:], sign * c[:half]
        return out

    c1, c2 = rng.normal(size=n), rng.normal(size=n)
    g1, u1, g2 = c1 + invert(c1), c2 - invert(c2), c2 + invert(c2)
    q = rng.uniform(-4, 4, size=(5, 3))
    f_u = oracle_mod.form_factors(b, np.outer(g1, u1), q)[0]
    f_g = oracle_mod.form_factors(b, np.outer(g1, g2), q)[0]
    assert np.max(np.abs(f_u.real)) <= 1e-13 * np.max(np.abs(f_u))
    assert np.max(np.abs(f_g.imag)) <= 1e-13 * np.max(np.abs(f_g))
    assert np.max(np.abs(f_u)) > 1e-3 and np.max(np.abs(f_g)) > 1e-3


def test_path0_equals_path1(oracle_mod, wl2):
    """Eq. (45) V-tensor form == Eq. (48) monomial form on a basis with s, p, d shells."""
    q = W.make_q(2)[0][::9001]
    f0 = oracle_mod.form_factors(wl2.basis, wl2.T, q, path=0)
    f1 = oracle_mod.form_factors(wl2.basis, wl2.T, q, path=1)
    assert np.max(np.abs(f0 - f1)) <= 1e-12 * np.max(np.abs(f0))

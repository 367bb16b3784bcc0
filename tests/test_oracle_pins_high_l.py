"""Pins of the CPU oracle for g, h and i shells (l = 4, 5, 6; "up to i orbitals") against things other than
itself — written BEFORE the library learned these shells.  Same sources as tests/test_oracle_pins.py: textbook closed
forms, numpy polynomial products, brute-force 1-D quadrature of Eq. (36), separable quadrature of the definition
(tests/bruteforce.py, which imports neither side).  A wrong binomial limit in Eq. (41), a Hermite recurrence that breaks
beyond He_6, or a Gamma-function slip in Eq. (A4)/(A5) at high powers would fail here."""
import math

import numpy as np
import pytest

import workloads as W
from tests import bruteforce as bf
from tests.test_oracle_pins import _quad1d, mk_basis


@pytest.mark.parametrize("l", [4, 5, 6])
def test_primitive_norm_textbook_high_l(oracle_mod, l):
    """xi N of one unit-normalised primitive == (2a/pi)^{3/4} (4a)^{l/2} / sqrt((2a-1)!!(2b-1)!!(2c-1)!!), every component."""
    alpha = 0.77
    b = mk_basis([[0, 0, 0]], [(0, l, [alpha], [1.0])])
    xi, N = oracle_mod.norms(b)

    def df(n):
        return 1.0 if n <= 0 else float(np.prod(np.arange(n, 0, -2)))

    comps = W.cartesian_components(l)
    assert len(comps) == (l + 1) * (l + 2) // 2
    for i, (a, bb, c) in enumerate(comps):
        ref = (2 * alpha / math.pi) ** 0.75 * (4 * alpha) ** (l / 2) / math.sqrt(df(2 * a - 1) * df(2 * bb - 1) * df(2 * c - 1))
        assert xi[i] * N[i] == pytest.approx(ref, rel=1e-13)
        assert N[i] == pytest.approx(1.0, rel=1e-13)


def test_shift_coeffs_up_to_6(oracle_mod):
    """Eq. (40)-(41) for every (a_i, a_j) up to (6, 6) against numpy polynomial multiplication."""
    P = np.polynomial.polynomial
    u, v = 0.37, -1.21
    for ai in range(7):
        for aj in range(7):
            ref = P.polymul(P.polypow([u, 1.0], ai), P.polypow([v, 1.0], aj))
            np.testing.assert_allclose(oracle_mod.shift_coeffs(ai, aj, u, v), ref, rtol=1e-12, atol=1e-13)


@pytest.mark.parametrize("ai,aj", [(4, 0), (0, 5), (4, 4), (5, 3), (6, 2), (6, 5), (6, 6)])
def test_V1d_vs_quadrature_high_powers(oracle_mod, ai, aj):
    """Eq. (36) -> (46) by brute-force trapezoid quadrature, powers up to (6, 6) (He_12, b^A up to A = 12)."""
    xi, xj, si, sj = 0.4, -1.1, 0.8, 1.3
    sij = si * sj / math.hypot(si, sj)
    pref = math.sqrt(2 * math.pi) * sij * math.exp(-(xi - xj) ** 2 / (2 * (si * si + sj * sj)))
    for q in (-3.0, -0.7, 0.0, 0.31, 2.2):
        ref = _quad1d(ai, xi, si, aj, xj, sj, q)
        got = pref * oracle_mod.V1d(ai, aj, xi, xj, si, sj, q)
        scale = max(abs(_quad1d(ai, xi, si, aj, xj, sj, 0.0)), 1.0)      # the integral's own size at q = 0
        assert abs(got - ref) <= 1e-11 * scale


def test_C1d_equals_V1d_high_powers(oracle_mod):
    """Eq. (50) (monomial form) == Eq. (46) (Hermite form) at powers up to (6, 6): the two oracle paths, 1-D."""
    xi, xj, si, sj = -0.3, 0.9, 0.7, 1.1
    sij = si * sj / math.hypot(si, sj)
    X = sij * sij * (xi / (si * si) + xj / (sj * sj))
    for ai, aj in ((4, 4), (6, 3), (6, 6)):
        C = oracle_mod.C1d(ai, aj, xi, xj, si, sj)
        for q in (-1.7, 0.2, 2.5):
            poly = sum(C[u] * q ** u for u in range(ai + aj + 1))
            got = np.exp(1j * q * X - 0.5 * q * q * sij * sij) * poly
            ref = oracle_mod.V1d(ai, aj, xi, xj, si, sj, q)
            assert abs(got - ref) <= 1e-11 * max(1.0, abs(ref))


def _ghi_basis():
    return mk_basis([[0.0, 0.1, -0.6], [0.4, -0.3, 0.9]],
                    [(0, 4, [1.1, 0.45], [0.7, 0.4]), (1, 5, [0.8], [1.0]), (1, 6, [0.9], [1.0]), (0, 1, [1.6], [1.0])])


def test_unit_diagonal_overlap_g_h_i(oracle_mod):
    """S_mumu = 1 for every component of contracted g and single-primitive h, i shells (Eq. A5), and the whole
    overlap matrix against separable quadrature with the normalisation re-derived by quadrature."""
    b = _ghi_basis()
    S = oracle_mod.overlap(b)
    np.testing.assert_allclose(np.diag(S), 1.0, rtol=0, atol=1e-12)
    ref = bf.pair_matrix_separable(b, np.zeros(3), h=0.04).real
    assert np.max(np.abs(S - ref)) <= 1e-10


def test_separable_quadrature_with_g_h_i(oracle_mod):
    """Form factors of a two-centre g/h/i(+p) basis (every pair class L = 2..12) against separable quadrature of the
    definition, random non-symmetric T, both oracle paths."""
    rng = np.random.default_rng(12)
    b = _ghi_basis()
    n = b.nbf
    assert n == 15 + 21 + 28 + 3
    T = rng.normal(size=(1, n, n))
    q = np.array([[0.5, -1.0, 0.25], [-1.6, 0.3, 1.2]])
    ref = bf.form_factor_separable(b, T, q, h=0.04)
    for path in (0, 1):
        got = oracle_mod.form_factors(b, T, q, path=path)
        assert np.max(np.abs(got - ref)) <= 1e-10 * np.max(np.abs(ref))

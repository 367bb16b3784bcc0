"""Pins of the FFT-method oracle (oracle/fft_method.py; Section III, Eq. (19)-(34) PAPER.md:140-222)."""
import numpy as np
import pytest

import workloads as W


@pytest.fixture(scope="module")
def offt(oracle_mod):
    from oracle import fft_method
    return fft_method


def soft_basis():
    """s, p and d shells with exponents in [0.3, 0.8] on two close atoms: the tabulated density is band limited to
    ~1e-11 at pi/h for h = 0.25 bohr and vanishes at 8 bohr, so the Riemann sum of Eq. (19) is spectrally accurate."""
    xyz = np.array([[0.2, -0.1, 0.5], [-0.3, 0.4, -0.6]])
    return W.Basis(xyz, np.array([0, 0, 0, 1, 1], np.int32), np.array([0, 1, 2, 0, 1], np.int32),
                   np.array([2, 1, 1, 1, 2], np.int32), np.array([0.8, 0.35, 0.6, 0.5, 0.45, 0.7, 0.3]),
                   np.array([0.6, 0.5, 1.0, 1.0, 1.0, 0.4, 0.7]))


def test_fft_route_converges_to_the_analytic_form_factor(oracle_mod, offt):
    b = soft_basis()
    rng = np.random.default_rng(4)
    T = rng.normal(size=(2, b.nbf, b.nbf))
    n, x_min, L = (64, 64, 64), np.array([-8.0, -8.0, -8.0]), np.array([16.0, 16.0, 16.0])
    f = offt.form_factors(b, T, n, x_min, L)
    q = offt.q_points(n, L)
    idx = W.sample_q_indices(q.shape[0], 400, seed=1)
    idx = idx[np.max(np.abs(q[idx]), axis=1) < 9.0]                   # away from the Nyquist faces (aliases)
    f_ref = oracle_mod.form_factors(b, T, q[idx])
    for s in range(2):
        assert np.max(np.abs(f[s, idx] - f_ref[s])) <= 1e-8 * np.max(np.abs(f_ref[s]))
    # q = 0 sits at index (N/2, N/2, N/2) and equals V_pix * sum(Phi) = g Tr(T S) up to the quadrature error
    i0 = (32 * 64 + 32) * 64 + 32
    assert np.allclose(q[i0], 0.0)
    S = oracle_mod.overlap(b)
    assert np.allclose(f[:, i0], 2.0 * np.einsum("spq,pq->s", T, S), rtol=1e-9)


def test_transform_equals_plain_triple_sum_odd_and_even_sizes(offt):
    rng = np.random.default_rng(5)
    n, x_min, L = (5, 4, 6), np.array([-1.0, 0.3, -2.2]), np.array([3.0, 2.5, 4.1])
    phi = rng.normal(size=(2, *n))
    f = offt.transform(phi, x_min, L)
    q = offt.q_points(n, L)
    assert np.allclose(q[0], -2 * np.pi * np.array([2, 2, 3]) / L)    # most negative frequency first
    ref = offt.direct_sum(phi, x_min, L, q)
    assert np.max(np.abs(f - ref)) <= 1e-12 * np.max(np.abs(ref))


def test_density_is_the_orbital_product(oracle_mod, offt):
    """Phi at one point against the definition written out with a single orbital pair, and its integral = g S_pq."""
    b = soft_basis()
    n, x_min, L = (48, 48, 48), np.array([-9.0, -9.0, -9.0]), np.array([18.0, 18.0, 18.0])
    p, q_ = 2, 7
    T = np.zeros((1, b.nbf, b.nbf))
    T[0, p, q_] = 1.0
    phi = offt.density_grid(b, T, n, x_min, L)
    V = offt.orbital_values(b, offt.grid_points(n, x_min, L))
    assert np.allclose(phi.ravel(), 2.0 * V[p] * V[q_], rtol=1e-14, atol=1e-300)
    vpix = np.prod(L) / np.prod(n)
    assert abs(phi.sum() * vpix - 2.0 * oracle_mod.overlap(b)[p, q_]) <= 1e-9
    # every orbital is normalised on the grid too (Appendix A)
    assert np.allclose(np.sum(V * V, axis=1) * vpix, 1.0, rtol=1e-9)


def test_parseval_eq75(oracle_mod, offt):
    """Eq. (75): Int d^3r |Phi|^2 = Int d^3q/(2 pi)^3 |f|^2.  On the method's grids the relation is exact
    (discrete Parseval): V_pix sum |Phi_abc|^2 == (1 / V_box) sum_q |f_q|^2 — a pin of the transform's normalisation (V_pix,
    unnormalised DFT, unit-modulus phase) that is independent of the triple-sum pin; and on a soft basis in a large box both
    equal the analytic continuum value Int d^3q/(2 pi)^3 |f|^2 by quadrature of the ANALYTIC oracle on the same q grid."""
    b = soft_basis()
    rng = np.random.default_rng(6)
    T = rng.normal(size=(2, b.nbf, b.nbf))
    for n, x_min, L in (((12, 9, 10), np.array([-3.0, -2.5, -3.5]), np.array([6.0, 5.5, 7.0])),
                        ((40, 40, 40), np.array([-8.0] * 3), np.array([16.0] * 3))):
        phi = offt.density_grid(b, T, n, x_min, L)
        f = offt.transform(phi, x_min, L)
        vpix, vbox = np.prod(L) / np.prod(n), np.prod(L)
        lhs = vpix * np.sum(phi ** 2, axis=(1, 2, 3))
        rhs = np.sum(np.abs(f) ** 2, axis=1) / vbox
        np.testing.assert_allclose(lhs, rhs, rtol=1e-13)
    # continuum check on the large box: the analytic form factor on the same q lattice gives the same q-space integral
    q = offt.q_points(n, L)
    f_ana = oracle_mod.form_factors(b, T, q)
    np.testing.assert_allclose(np.sum(np.abs(f_ana) ** 2, axis=1) / vbox, lhs, rtol=1e-6)

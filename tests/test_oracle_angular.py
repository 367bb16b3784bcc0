"""Pins of the angular-moment oracle (oracle/angular_oracle.c; Eq. (57), (59), (60) PAPER.md:380-398) against things
other than itself: scipy's spherical harmonics, exact coefficient recovery of a band-limited function, the Rayleigh
plane-wave expansion (spherical Bessel functions from scipy) and Parseval (Eq. 60)."""
import numpy as np
import pytest
from scipy import special as sp


def grid(n_theta, n_phi):
    ct, w = np.polynomial.legendre.leggauss(n_theta)
    phi = 2.0 * np.pi * np.arange(n_phi) / n_phi
    return ct, w, phi


def scipy_Y(l, m, ct, phi):
    return sp.sph_harm_y(l, m, np.arccos(ct), phi)


def test_sph_harm_matches_scipy(oracle_mod):
    rng = np.random.default_rng(1)
    for ct, phi in zip(rng.uniform(-1, 1, 6), rng.uniform(0, 2 * np.pi, 6)):
        y = oracle_mod.sph_harm(24, ct, phi)
        for l in (0, 1, 2, 5, 13, 24):
            for m in range(-l, l + 1):
                ref = scipy_Y(l, m, ct, phi)
                assert abs(y[l * (l + 1) + m] - ref) <= 2e-13 * max(1.0, abs(ref)), (l, m)


def test_band_limited_coefficients_recovered(oracle_mod):
    """f = sum c_lm Y_lm with l <= 6: Gauss-Legendre (10 nodes) x uniform phi (16) integrates conj(Y) f exactly."""
    rng = np.random.default_rng(2)
    L = 6
    ct, w, phi = grid(10, 16)
    c = rng.normal(size=(2, 3, (L + 1) ** 2)) + 1j * rng.normal(size=(2, 3, (L + 1) ** 2))
    CT, PH = np.meshgrid(ct, phi, indexing="ij")
    f = np.zeros((2, 3, 10, 16), complex)
    for l in range(L + 1):
        for m in range(-l, l + 1):
            f += c[:, :, l * (l + 1) + m, None, None] * scipy_Y(l, m, CT, PH)[None, None]
    R, f2 = oracle_mod.angular_moments(f, ct, w, 16, L)
    assert np.max(np.abs(R - c)) <= 1e-13 * np.max(np.abs(c))
    # Eq. (60): <|f|^2> = 1/4pi sum |R_lm|^2 (|f|^2 has degree 12 <= 2*10-1 and |m| <= 12 < 16: exact)
    assert np.allclose(f2, np.sum(np.abs(c) ** 2, axis=-1) / (4 * np.pi), rtol=1e-13)
    # asking for more harmonics than the function has gives zeros there
    R8, _ = oracle_mod.angular_moments(f, ct, w, 16, 7)
    assert np.max(np.abs(R8[..., (L + 1) ** 2:])) <= 1e-13 * np.max(np.abs(c))


def test_rayleigh_plane_wave(oracle_mod):
    """f(q) = exp(i q.a)  =>  R_lm(q) = 4 pi i^l j_l(q a) conj(Y_lm(ahat)); <|f|^2> = 1."""
    a = np.array([0.4, -0.7, 1.1])
    an = np.linalg.norm(a)
    qs = np.array([0.3, 2.0, 6.0])
    ct, w, phi = grid(40, 64)
    CT, PH = np.meshgrid(ct, phi, indexing="ij")
    ST = np.sqrt(1 - CT ** 2)
    qhat = np.stack([ST * np.cos(PH), ST * np.sin(PH), CT], axis=-1)
    f = np.exp(1j * qs[:, None, None] * (qhat @ a)[None])[None]
    L = 12
    R, f2 = oracle_mod.angular_moments(f, ct, w, 64, L)
    assert np.allclose(f2, 1.0, rtol=1e-13)
    cta, pha = a[2] / an, np.arctan2(a[1], a[0])
    for ir, q in enumerate(qs):
        for l in range(L + 1):
            for m in range(-l, l + 1):
                ref = 4 * np.pi * (1j ** l) * sp.spherical_jn(l, q * an) * np.conj(scipy_Y(l, m, cta, pha))
                assert abs(R[0, ir, l * (l + 1) + m] - ref) <= 1e-12, (q, l, m)


def test_gaussian_pair_closed_form(oracle_mod):
    """One s-type pair: f = C exp(-q^2/4p) exp(i q.P) (the s-s closed form the form-factor oracle is pinned to)
    => R_lm(q) = C exp(-q^2/4p) 4 pi i^l j_l(q|P|) conj(Y_lm(Phat)): ties the moments to the S4 output format."""
    P = np.array([0.9, 0.2, -0.5])
    p, Cn = 1.7, 0.83
    Pn = np.linalg.norm(P)
    qs = np.geomspace(0.05, 8.0, 5)
    ct, w, phi = grid(32, 48)
    CT, PH = np.meshgrid(ct, phi, indexing="ij")
    ST = np.sqrt(1 - CT ** 2)
    qhat = np.stack([ST * np.cos(PH), ST * np.sin(PH), CT], axis=-1)
    f = (Cn * np.exp(-qs ** 2 / (4 * p))[:, None, None] * np.exp(1j * qs[:, None, None] * (qhat @ P)[None]))[None]
    R, f2 = oracle_mod.angular_moments(f, ct, w, 48, 8)
    assert np.allclose(f2[0], (Cn * np.exp(-qs ** 2 / (4 * p))) ** 2, rtol=1e-12)
    ctP, phP = P[2] / Pn, np.arctan2(P[1], P[0])
    for ir, q in enumerate(qs):
        for l in range(9):
            for m in range(-l, l + 1):
                ref = Cn * np.exp(-q * q / (4 * p)) * 4 * np.pi * (1j ** l) * sp.spherical_jn(l, q * Pn) * np.conj(scipy_Y(l, m, ctP, phP))
                assert abs(R[0, ir, l * (l + 1) + m] - ref) <= 1e-12

"""Pins of the pure-shell oracle (oracle/pure.py; multi-term Cartesian orbitals of Eq. (A2)) and CPU
checks of the library's host side for pure shells (C ABI, host-only context) against it."""
import numpy as np
import pytest
from scipy import special as sp

import workloads as W


@pytest.fixture(scope="module")
def opure(oracle_mod):
    from oracle import pure
    return pure


@pytest.mark.parametrize("l", [2, 3, 4, 5, 6])
def test_pure_functions_orthonormal_also_when_contracted(oracle_mod, opure, l):
    """2l+1 functions, orthonormal within the shell, for one primitive and for a contracted shell (the matrix is
    built from one primitive: pins the claim that it does not depend on the radial part)."""
    C = opure.pure_matrix(l)
    assert C.shape == ((l + 1) * (l + 2) // 2, 2 * l + 1)
    for exps, coefs in (((1.0,), (1.0,)), ((3.1, 0.9, 0.25), (0.3, 0.8, 0.5))):
        b = W.Basis(np.zeros((1, 3)), np.array([0], np.int32), np.array([l], np.int32), np.array([len(exps)], np.int32),
                    np.array(exps), np.array(coefs))
        S = C.T @ oracle_mod.overlap(b) @ C
        assert np.max(np.abs(S - np.eye(2 * l + 1))) <= 1e-13
    # the l(l-1)/2... contaminants (s-like r^2 for d, p-like r^2 x for f) are orthogonal to every pure function
    b = W.Basis(np.zeros((1, 3)), np.array([0, 0], np.int32), np.array([l, l - 2], np.int32), np.array([1, 1], np.int32),
                np.array([1.0, 1.0]), np.array([1.0, 1.0]))
    S = oracle_mod.overlap(b)
    nc = (l + 1) * (l + 2) // 2
    assert np.max(np.abs(C.T @ S[:nc, nc:])) <= 1e-13


@pytest.mark.parametrize("l,m", [(2, -2), (2, 0), (2, 2), (3, -3), (3, -1), (3, 0), (3, 2), (4, -3), (4, 0), (4, 4), (5, -5), (5, 2),
                                 (6, -6), (6, -1), (6, 0), (6, 5)])
def test_pure_pair_integral_against_3d_quadrature(oracle_mod, opure, l, m):
    """phi_lm defined DIRECTLY (N r^l Y^real_lm(rhat) e^{-a r^2}, scipy's Y) times an s Gaussian on another centre:
    Int phi_lm phi_s e^{iq.r} d^3r by 3-D trapezoid quadrature against the oracle route (C T C^T through the pinned
    Cartesian oracle)."""
    a, bta = 0.9, 0.7
    A, B = np.array([0.1, -0.2, 0.3]), np.array([-0.6, 0.5, 0.9])
    basis = W.Basis(np.stack([A, B]), np.array([0, 1], np.int32), np.array([l, 0], np.int32), np.array([1, 1], np.int32),
                    np.array([a, bta]), np.array([1.0, 1.0]))
    pure = [1, 0]
    nu = 2 * l + 2
    T = np.zeros((1, nu, nu))
    T[0, m + l, nu - 1] = 1.0
    qs = np.array([[0.0, 0.0, 0.0], [0.7, -0.4, 1.1], [-1.5, 2.0, 0.3]])
    f = opure.form_factors(basis, pure, T, qs, prefactor=1.0)[0]
    h, half = 0.1, 8.0
    ax = np.arange(-half, half + h / 2, h)
    X, Y, Z = np.meshgrid(ax, ax, ax, indexing="ij")
    dx, dy, dz = X - A[0], Y - A[1], Z - A[2]
    r = np.sqrt(dx * dx + dy * dy + dz * dz)
    rs = np.where(r > 0, r, 1.0)
    theta, phi = np.arccos(np.clip(dz / rs, -1, 1)), np.arctan2(dy, dx)
    Nn = np.sqrt(2.0 * (2 * a) ** (l + 1.5) / sp.gamma(l + 1.5))
    phi_a = Nn * r ** l * opure.real_sph_harm(l, m, theta, phi) * np.exp(-a * r * r)
    phi_b = (2 * bta / np.pi) ** 0.75 * np.exp(-bta * ((X - B[0]) ** 2 + (Y - B[1]) ** 2 + (Z - B[2]) ** 2))
    dens = phi_a * phi_b
    for iq, q in enumerate(qs):
        ref = np.sum(dens * np.exp(1j * (q[0] * X + q[1] * Y + q[2] * Z))) * h ** 3
        assert abs(f[iq] - ref) <= 1e-10, (q, f[iq], ref)


def mixed_basis():
    xyz = np.array([[0.0, 0.1, -0.8], [0.4, -0.3, 0.9], [-1.1, 0.6, 0.2]])
    shell_atom = np.array([0, 0, 0, 0, 1, 1, 1, 2, 2], np.int32)
    shell_l = np.array([0, 1, 2, 3, 0, 2, 3, 2, 1], np.int32)
    shell_pure = np.array([0, 1, 1, 1, 1, 0, 1, 1, 0], np.int32)     # flags on s/p are ignored
    nprim = np.array([2, 1, 2, 1, 1, 1, 1, 1, 2], np.int32)
    n = int(nprim.sum())
    rng = np.random.default_rng(3)
    exps = rng.uniform(0.4, 2.5, size=n)
    coefs = rng.uniform(0.3, 1.0, size=n)
    return W.Basis(xyz, shell_atom, shell_l, nprim, exps, coefs), shell_pure


def test_library_host_side_pure_overlap(oracle_mod, opure):
    from paper_2512_18010_b200 import binding
    b, pure = mixed_basis()
    with binding.Scarf(None) as sc:
        sc.set_basis(b, shell_pure=pure)
        nbf = 1 + 3 + 5 + 7 + 1 + 6 + 7 + 5 + 3
        assert sc.nbf == nbf
        S = sc.overlap()
    S_ref = opure.overlap(b, pure)
    assert S.shape == (nbf, nbf)
    assert np.max(np.abs(S - S_ref)) <= 1e-12
    assert np.allclose(np.diag(S), 1.0, atol=1e-13)

"""CPU ORACLE for pure (real solid-harmonic) shells.  TEST INFRASTRUCTURE ONLY.

The paper builds pure orbitals (its example: 3d_{x^2-y^2}) as several Cartesian terms with prefactors inside one
orbital, Eq. (A2), normalised as a whole.  Here that is written out from the DEFINITION
of the functions instead of from a table of prefactors:

    phi_lm(r) = N S_lm(r) R(r),   S_lm(r) = |r|^l Y^real_lm(rhat),   m = -l..l,
    Y^real_{l0} = Y_l^0,  Y^real_{l,m>0} = sqrt2 (-1)^m Re Y_l^m,  Y^real_{l,m<0} = sqrt2 (-1)^m Im Y_l^{|m|}

with Y_l^m from scipy (orthonormal, Condon-Shortley).  S_lm is a homogeneous polynomial of degree l, so phi_lm is a
linear combination of the shell's Cartesian components chi_c — the functions the pinned Cartesian oracle
(scarf_oracle.c) evaluates; the coefficients are found by fitting S_lm at random points onto the components' polynomial
parts (exact: the residual is checked), then each phi_lm is normalised with the ORACLE's own overlap of that shell.
The radial part R is the same for every component of a shell (the exponent-dependent part of Eq. (A4)/(A5) depends on
l only), so one primitive suffices for the fit; tests/test_oracle_pure.py pins that claim on a contracted shell
(orthonormality) and the whole construction against 3-D quadrature of phi_lm defined directly through scipy's Y_l^m.

    f_s(q) [mixed basis] = oracle.form_factors(basis, C T C^T, q),   C = blockdiag(C_l or identity).

Shares no code, table or constant with paper_2512_18010_b200/csrc/pure.cu (which tabulates the monomial
coefficients of S_lm); only the arithmetic-free helpers of the top-level `workloads` module are used.
"""
from __future__ import annotations

import numpy as np
from scipy import special as sp

import oracle
import workloads as W


def real_sph_harm(l: int, m: int, theta, phi):
    if m == 0:
        return sp.sph_harm_y(l, 0, theta, phi).real
    y = sp.sph_harm_y(l, abs(m), theta, phi)
    s = np.sqrt(2.0) * (-1.0) ** abs(m)
    return s * (y.real if m > 0 else y.imag)


def _one_shell(l, exps, coefs):
    return W.Basis(np.zeros((1, 3)), np.array([0], np.int32), np.array([l], np.int32), np.array([len(exps)], np.int32),
                   np.asarray(exps, float), np.asarray(coefs, float))


def pure_matrix(l: int, exps=(1.0,), coefs=(1.0,)) -> np.ndarray:
    """C_l [n_cart(l)][2l+1]: phi_lm = sum_c C[c][m] chi_c, unit norm.  l = 0, 1: identity (x, y, z order kept)."""
    comps = W.cartesian_components(l)
    nc = len(comps)
    if l < 2:
        return np.eye(nc)
    b = _one_shell(l, exps, coefs)
    xi, N = oracle.norms(b)                                  # effective coefficient of primitive 0 of every component
    coef = N * xi.reshape(nc, len(exps))[:, 0]
    rng = np.random.default_rng(100 + l)
    r = rng.normal(size=(200, 3))
    rn = np.linalg.norm(r, axis=1)
    theta, phi = np.arccos(r[:, 2] / rn), np.arctan2(r[:, 1], r[:, 0])
    A = np.stack([coef[c] * r[:, 0] ** a * r[:, 1] ** bb * r[:, 2] ** cc for c, (a, bb, cc) in enumerate(comps)], axis=1)
    C = np.zeros((nc, 2 * l + 1))
    for m in range(-l, l + 1):
        t = rn ** l * real_sph_harm(l, m, theta, phi)
        x, *_ = np.linalg.lstsq(A, t, rcond=None)
        assert np.max(np.abs(A @ x - t)) <= 1e-12 * np.max(np.abs(t)), "S_lm is not in the span of the components"
        C[:, m + l] = x
    S = oracle.overlap(b)
    for k in range(2 * l + 1):
        C[:, k] /= np.sqrt(C[:, k] @ S @ C[:, k])
    C[np.abs(C) < 1e-14] = 0.0
    return C


def basis_matrix(basis, shell_pure) -> np.ndarray:
    """C [nbf_cart][nbf_user] for the mixed basis (pure where shell_pure[i] != 0 and l >= 2)."""
    blocks = []
    for i, l in enumerate(np.asarray(basis.shell_l)):
        nc = (l + 1) * (l + 2) // 2
        blocks.append(pure_matrix(int(l)) if (shell_pure[i] and l >= 2) else np.eye(nc))
    nr, ncol = sum(b.shape[0] for b in blocks), sum(b.shape[1] for b in blocks)
    C = np.zeros((nr, ncol))
    r = c = 0
    for b in blocks:
        C[r:r + b.shape[0], c:c + b.shape[1]] = b
        r += b.shape[0]
        c += b.shape[1]
    return C


def form_factors(basis, shell_pure, T, q, **kw) -> np.ndarray:
    C = basis_matrix(basis, shell_pure)
    T = np.asarray(T, float)
    if T.ndim == 2:
        T = T[None]
    Tc = np.einsum("ma,sab,nb->smn", C, T, C)
    return oracle.form_factors(basis, Tc, q, **kw)


def overlap(basis, shell_pure) -> np.ndarray:
    C = basis_matrix(basis, shell_pure)
    return C.T @ oracle.overlap(basis) @ C

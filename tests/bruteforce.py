"""Brute-force real-space quadrature of the DEFINITION of the form factor (Eq. 35):

    f_s(q) = g * sum_{mu nu} T_{mu nu} Int d^3r phi_mu(r) phi_nu(r) exp(i q.r)

Pure numpy; imports neither the oracle nor the CUDA path.  Normalisation constants are themselves
obtained by quadrature (Int chi^2 = 1 per primitive, then per contracted orbital: Eq. A3 and
PAPER.md:633), so nothing here shares a formula with either implementation.

Trapezoid quadrature of a Gaussian integrand on a uniform grid converges like exp(-pi^2 / (p h^2)),
so h = 0.15 is exact to round-off for p <= 6 and h = 0.02 for p <= 60+.
"""
from __future__ import annotations

import numpy as np


def components(l):
    return [(a, b, l - a - b) for a in range(l, -1, -1) for b in range(l - a, -1, -1)]


def orbitals(basis):
    """List of (centre[3], (a,b,c), exponents[n], coeffs[n]) per contracted Cartesian orbital."""
    out = []
    p0 = 0
    for s in range(len(basis.shell_l)):
        l, n = int(basis.shell_l[s]), int(basis.shell_nprim[s])
        ctr = np.asarray(basis.atom_xyz[int(basis.shell_atom[s])], float)
        e = np.asarray(basis.exponents[p0:p0 + n], float)
        d = np.asarray(basis.coeffs[p0:p0 + n], float)
        for abc in components(l):
            out.append((ctr, abc, e, d))
        p0 += n
    return out


# ---------------------------------------------------------------------------------------------
# (i) full 3-D trapezoid on a box
# ---------------------------------------------------------------------------------------------
def form_factor_3d(basis, T, q, box=9.0, h=0.15, prefactor=2.0):
    T = np.asarray(T, float)
    if T.ndim == 2:
        T = T[None]
    q = np.asarray(q, float).reshape(-1, 3)
    ax = np.arange(-box, box + 0.5 * h, h)
    X, Y, Z = np.meshgrid(ax, ax, ax, indexing="ij")
    w = h ** 3
    phis = []
    for ctr, (a, b, c), e, d in orbitals(basis):
        dx, dy, dz = X - ctr[0], Y - ctr[1], Z - ctr[2]
        r2 = dx * dx + dy * dy + dz * dz
        ang = dx ** a * dy ** b * dz ** c
        phi = np.zeros_like(X)
        for ek, dk in zip(e, d):
            prim = ang * np.exp(-ek * r2)
            prim /= np.sqrt(np.sum(prim * prim) * w)          # Eq. (A3) with d = 1, numerically
            phi += dk * prim
        phi /= np.sqrt(np.sum(phi * phi) * w)                 # contracted orbital normalised to 1
        phis.append(phi.ravel())
    Phi = np.array(phis)                                      # [nbf][npts]
    R = np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1)
    out = np.zeros((T.shape[0], q.shape[0]), complex)
    for s in range(T.shape[0]):
        rho = np.einsum("mp,mn,np->p", Phi, T[s], Phi, optimize=True)    # transition density, Eq. (20) / 2
        for iq in range(q.shape[0]):
            out[s, iq] = prefactor * w * np.sum(rho * np.exp(1j * (R @ q[iq])))
    return out


# ---------------------------------------------------------------------------------------------
# (ii) separable: each primitive-pair integral = product of three 1-D trapezoid integrals
# ---------------------------------------------------------------------------------------------
def _int1d(a, Ax, alpha, b, Bx, beta, qx, extra_pow=0, h=0.02, half=14.0):
    """Int (x-Ax)^a (x-Bx)^b x^extra exp(-alpha (x-Ax)^2 - beta (x-Bx)^2 + i qx x) dx."""
    lo, hi = min(Ax, Bx) - half, max(Ax, Bx) + half
    x = np.arange(lo, hi + 0.5 * h, h)
    f = (x - Ax) ** a * (x - Bx) ** b * x ** extra_pow * np.exp(-alpha * (x - Ax) ** 2 - beta * (x - Bx) ** 2)
    return h * np.sum(f * np.exp(1j * qx * x))


def _prim_pair(ctrA, abcA, alpha, ctrB, abcB, beta, q, extra=(0, 0, 0), h=0.02):
    v = 1.0 + 0j
    for k in range(3):
        v *= _int1d(abcA[k], ctrA[k], alpha, abcB[k], ctrB[k], beta, q[k], extra[k], h=h)
    return v


def _norm_coeffs(orb, h=0.02):
    """Effective primitive coefficients of a normalised contracted orbital, all by quadrature."""
    ctr, abc, e, d = orb
    zero = np.zeros(3)
    n = np.array([1.0 / np.sqrt(_prim_pair(ctr, abc, ek, ctr, abc, ek, zero, h=h).real) for ek in e])
    c = d * n
    s = 0.0
    for i in range(len(e)):
        for j in range(len(e)):
            s += c[i] * c[j] * _prim_pair(ctr, abc, e[i], ctr, abc, e[j], zero, h=h).real
    return c / np.sqrt(s)


def pair_matrix_separable(basis, q, extra=(0, 0, 0), h=0.02):
    """[nbf][nbf] complex: Int phi_mu phi_nu x^ex y^ey z^ez exp(i q.r) d^3r."""
    orbs = orbitals(basis)
    cs = [_norm_coeffs(o, h=h) for o in orbs]
    n = len(orbs)
    M = np.zeros((n, n), complex)
    for i, (cA, abcA, eA, _dA) in enumerate(orbs):
        for j, (cB, abcB, eB, _dB) in enumerate(orbs):
            v = 0j
            for ka in range(len(eA)):
                for kb in range(len(eB)):
                    v += cs[i][ka] * cs[j][kb] * _prim_pair(cA, abcA, eA[ka], cB, abcB, eB[kb], q, extra, h=h)
            M[i, j] = v
    return M


def form_factor_separable(basis, T, q, prefactor=2.0, h=0.02):
    T = np.asarray(T, float)
    if T.ndim == 2:
        T = T[None]
    q = np.asarray(q, float).reshape(-1, 3)
    out = np.zeros((T.shape[0], q.shape[0]), complex)
    for iq in range(q.shape[0]):
        M = pair_matrix_separable(basis, q[iq], h=h)
        for s in range(T.shape[0]):
            out[s, iq] = prefactor * np.sum(T[s] * M)
    return out

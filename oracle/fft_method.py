"""CPU ORACLE for the paper's FFT method (Section III, Eq. (19)-(34)).  TEST INFRASTRUCTURE ONLY.

Step by step, in the paper's order and notation:

  1. tabulate the transition density on a regular grid inside the box [x_min, x_min + L) (Eq. 25-28):
         x_abc = x_min + L * (a/N_x, b/N_y, c/N_z),   a = 0..N_x-1, ...
         Phi_abc = 2 sum_pq T_pq phi_q(x_abc) phi_p(x_abc)                                  (Eq. 20)
     with the contracted, normalised Cartesian orbitals of Appendix A (coefficients N_mu d_k xi_k from the pinned
     scarf_oracle.c: oracle.norms);
  2. discrete transform (Eq. 24, a library FFT serves as this step) and Eq. (27)/(30)-(33):
         f_s(q_{alpha beta gamma}) ~= V_pix sum_abc Phi_abc exp(+i q . x_abc),    q = 2 pi (alpha/L_x, beta/L_y, gamma/L_z),
         V_pix = L_x L_y L_z / (N_x N_y N_z)                                                (Eq. 29)
     i.e. V_pix exp(+i q . x_min) times the unnormalised inverse-sign DFT of Phi;
  3. reorder so that the most negative frequencies come first: output index ia <-> alpha = ia - floor(N/2).

Reading (#19): Eq. (32) as printed, f* ~ V_pix e^{+i q.x_min} F*_{alpha beta gamma} with F* "the forward FFT of
the complex conjugate array", has the wrong sign of the phase against its own Eq. (27)/(31) (F[Phi*](q) = Int e^{-iq.x}
Phi* carries e^{-i q.x_min}); what is computed here is the Riemann sum of Eq. (19) itself, which is what Eq. (27)-(31)
derive.  Phi is real for real T, so conjugating the array is a no-op.

Pins (tests/test_oracle_fft.py): the result converges to the ANALYTIC form factor of the pinned Cartesian oracle on a
soft basis (independent route: closed-form integrals vs tabulate-and-transform); the FFT step against the plain triple
sum on a tiny grid; the q = 0 element equals V_pix * sum(Phi).  Shares no code with paper_2512_18010_b200/csrc/.
"""
from __future__ import annotations

import numpy as np

import oracle
import workloads as W


def orbital_values(basis, pts) -> np.ndarray:
    """[nbf][n_pts]: phi_mu(x) = sum_k N_mu d_k xi_{mu k} (x-A)^a (y-A)^b (z-A)^c exp(-alpha_k |x-A|^2)  (Eq. A2)."""
    xi, N = oracle.norms(basis)
    pts = np.asarray(pts, float)
    out = []
    k0 = 0          # running offset into exponents / coeffs
    o = 0           # running offset into xi (per orbital, per primitive)
    mu = 0
    for sh in range(len(basis.shell_l)):
        l, n = int(basis.shell_l[sh]), int(basis.shell_nprim[sh])
        A = basis.atom_xyz[basis.shell_atom[sh]]
        d = pts - A
        r2 = np.sum(d * d, axis=1)
        al, dk = basis.exponents[k0:k0 + n], basis.coeffs[k0:k0 + n]
        for (a, b, c) in W.cartesian_components(l):
            rad = np.zeros(len(pts))
            for k in range(n):
                rad += N[mu] * dk[k] * xi[o + k] * np.exp(-al[k] * r2)
            out.append(d[:, 0] ** a * d[:, 1] ** b * d[:, 2] ** c * rad)
            o += n
            mu += 1
        k0 += n
    return np.array(out)


def grid_points(n, x_min, box_len) -> np.ndarray:
    ax = [x_min[i] + box_len[i] * np.arange(n[i]) / n[i] for i in range(3)]
    X, Y, Z = np.meshgrid(*ax, indexing="ij")
    return np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1)


def density_grid(basis, T, n, x_min, box_len, prefactor: float = 2.0) -> np.ndarray:
    """Phi [n_states][nx][ny][nz] (Eq. 20)."""
    T = np.asarray(T, float)
    if T.ndim == 2:
        T = T[None]
    V = orbital_values(basis, grid_points(n, x_min, box_len))
    phi = prefactor * np.einsum("spq,qx,px->sx", T, V, V)
    return phi.reshape(T.shape[0], *n)


def q_axes(n, box_len):
    return [2.0 * np.pi * (np.arange(n[i]) - n[i] // 2) / box_len[i] for i in range(3)]


def q_points(n, box_len) -> np.ndarray:
    QX, QY, QZ = np.meshgrid(*q_axes(n, box_len), indexing="ij")
    return np.stack([QX.ravel(), QY.ravel(), QZ.ravel()], axis=1)


def transform(phi, x_min, box_len) -> np.ndarray:
    """Steps 2-3 for Phi [n_states][nx][ny][nz]: complex [n_states][nx*ny*nz], index (ia*ny + ib)*nz + ic."""
    ns, nx, ny, nz = phi.shape
    n = (nx, ny, nz)
    vpix = float(np.prod(box_len)) / (nx * ny * nz)
    F = np.fft.ifftn(phi, axes=(1, 2, 3)) * (nx * ny * nz)            # sum_abc Phi exp(+2 pi i (a alpha/N + ...))
    F = np.fft.fftshift(F, axes=(1, 2, 3))                            # alpha = ia - floor(N/2)
    qx, qy, qz = q_axes(n, box_len)
    phase = np.exp(1j * (qx[:, None, None] * x_min[0] + qy[None, :, None] * x_min[1] + qz[None, None, :] * x_min[2]))
    return (vpix * phase[None] * F).reshape(ns, -1)


def form_factors(basis, T, n, x_min, box_len, prefactor: float = 2.0) -> np.ndarray:
    return transform(density_grid(basis, T, n, x_min, box_len, prefactor), np.asarray(x_min, float), np.asarray(box_len, float))


def direct_sum(phi, x_min, box_len, q) -> np.ndarray:
    """V_pix sum_abc Phi_abc exp(i q . x_abc) for a list of q, by the plain triple sum (tiny grids only)."""
    ns = phi.shape[0]
    n = phi.shape[1:]
    pts = grid_points(n, x_min, box_len)
    vpix = float(np.prod(box_len)) / np.prod(n)
    return vpix * (phi.reshape(ns, -1) @ np.exp(1j * (pts @ np.asarray(q, float).T)))

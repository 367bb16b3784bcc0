"""ctypes front end of the CPU oracle (oracle/scarf_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  It never imports paper_2512_18010_b200's CUDA binding; it accepts the plain-array `Basis`
container of the top-level `workloads` module (the shared, arithmetic-free input generator) by duck typing.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int32)
        basis_args = [C.c_int, dp, C.c_int, ip, ip, ip, dp, dp]
        L.oracle_nbf.argtypes = [C.c_int, ip]
        L.oracle_nbf.restype = C.c_int
        L.oracle_max_threads.restype = C.c_int
        L.oracle_norms.argtypes = basis_args + [dp, dp]
        L.oracle_norms.restype = C.c_int
        L.oracle_form_factors.argtypes = basis_args + [C.c_int, dp, C.c_int64, dp, C.c_double, C.c_int, C.c_int, dp]
        L.oracle_form_factors.restype = C.c_int
        L.oracle_pair_matrix.argtypes = basis_args + [dp, C.c_int, dp]
        L.oracle_pair_matrix.restype = C.c_int
        L.oracle_V1d.argtypes = [C.c_int, C.c_int] + [C.c_double] * 5 + [dp]
        L.oracle_V1d.restype = None
        L.oracle_C1d.argtypes = [C.c_int, C.c_int] + [C.c_double] * 4 + [dp]
        L.oracle_C1d.restype = None
        L.oracle_hermite_He.argtypes = [C.c_int, C.c_double, dp]
        L.oracle_hermite_He.restype = None
        L.oracle_shift_coeffs.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, dp]
        L.oracle_shift_coeffs.restype = None
        L.oracle_sph_harm.argtypes = [C.c_int, C.c_double, C.c_double, dp]
        L.oracle_sph_harm.restype = None
        L.oracle_angular_moments.argtypes = [C.c_int, C.c_int, C.c_int, dp, dp, C.c_int, C.c_int, dp, dp, dp]
        L.oracle_angular_moments.restype = C.c_int
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int32))


def _basis_args(b):
    xyz = np.ascontiguousarray(b.atom_xyz, np.float64)
    sa = np.ascontiguousarray(b.shell_atom, np.int32)
    sl = np.ascontiguousarray(b.shell_l, np.int32)
    sn = np.ascontiguousarray(b.shell_nprim, np.int32)
    e = np.ascontiguousarray(b.exponents, np.float64)
    d = np.ascontiguousarray(b.coeffs, np.float64)
    keep = (xyz, sa, sl, sn, e, d)
    return keep, [xyz.shape[0], _dp(xyz), sl.shape[0], _ip(sa), _ip(sl), _ip(sn), _dp(e), _dp(d)]


def max_threads() -> int:
    return int(lib().oracle_max_threads())


def nbf(basis) -> int:
    sl = np.ascontiguousarray(basis.shell_l, np.int32)
    return int(lib().oracle_nbf(sl.shape[0], _ip(sl)))


def norms(basis):
    """(xi per (orbital, primitive) flattened in orbital order, N per orbital): Eq. (A4), (A5)."""
    keep, args = _basis_args(basis)
    n = nbf(basis)
    l = np.asarray(basis.shell_l, np.int64)
    ntot = int(np.sum((l + 1) * (l + 2) // 2 * np.asarray(basis.shell_nprim, np.int64)))
    xi = np.zeros(ntot)
    N = np.zeros(n)
    if lib().oracle_norms(*args, _dp(xi), _dp(N)) != 0:
        raise ValueError("oracle_norms: bad basis")
    return xi, N


def form_factors(basis, T, q, prefactor: float = 2.0, path: int = 0, n_threads: int = 0) -> np.ndarray:
    """complex128 [n_states][n_q]; path 0 = Eq. (45)/(46), path 1 = Eq. (48)-(50)."""
    keep, args = _basis_args(basis)
    T = np.ascontiguousarray(T, np.float64)
    q = np.ascontiguousarray(q, np.float64).reshape(-1, 3)
    n = nbf(basis)
    if T.ndim == 2:
        T = T[None]
    if T.shape[1:] != (n, n):
        raise ValueError("T must be [n_states][nbf][nbf]")
    out = np.zeros((T.shape[0], q.shape[0], 2))
    rc = lib().oracle_form_factors(*args, T.shape[0], _dp(T), q.shape[0], _dp(q), float(prefactor), int(path),
                                   int(n_threads), _dp(out))
    if rc != 0:
        raise ValueError("oracle_form_factors: bad basis")
    return out[..., 0] + 1j * out[..., 1]


def pair_matrix(basis, q, path: int = 0) -> np.ndarray:
    """complex128 [nbf][nbf]: Int phi_mu phi_nu exp(i q.r) d^3r at one q."""
    keep, args = _basis_args(basis)
    q = np.ascontiguousarray(q, np.float64).reshape(3)
    n = nbf(basis)
    out = np.zeros((n, n, 2))
    if lib().oracle_pair_matrix(*args, _dp(q), int(path), _dp(out)) != 0:
        raise ValueError("oracle_pair_matrix: bad basis")
    return out[..., 0] + 1j * out[..., 1]


def overlap(basis) -> np.ndarray:
    """AO overlap S = pair_matrix at q = 0 (real part; the imaginary part is exactly 0 there)."""
    return np.ascontiguousarray(pair_matrix(basis, np.zeros(3)).real)


def V1d(ai, aj, xi, xj, sigma_i, sigma_j, q) -> complex:
    out = np.zeros(2)
    lib().oracle_V1d(ai, aj, xi, xj, sigma_i, sigma_j, q, _dp(out))
    return complex(out[0], out[1])


def C1d(ai, aj, xi, xj, sigma_i, sigma_j) -> np.ndarray:
    out = np.zeros((ai + aj + 1, 2))
    lib().oracle_C1d(ai, aj, xi, xj, sigma_i, sigma_j, _dp(out))
    return out[:, 0] + 1j * out[:, 1]


def hermite_He(nmax: int, x: float) -> np.ndarray:
    out = np.zeros(nmax + 1)
    lib().oracle_hermite_He(nmax, x, _dp(out))
    return out


def shift_coeffs(ai, aj, u, v) -> np.ndarray:
    out = np.zeros(ai + aj + 1)
    lib().oracle_shift_coeffs(ai, aj, u, v, _dp(out))
    return out


def sph_harm(l_max: int, cos_theta: float, phi: float) -> np.ndarray:
    """complex128 [(l_max+1)^2], index l(l+1)+m: orthonormal Y_l^m with the Condon-Shortley phase."""
    out = np.zeros(((l_max + 1) ** 2, 2))
    lib().oracle_sph_harm(int(l_max), float(cos_theta), float(phi), _dp(out))
    return out[:, 0] + 1j * out[:, 1]


def angular_moments(f, cos_theta, w_theta, n_phi: int, l_max: int):
    """f: complex [n_states][n_r][n_theta][n_phi] on the product grid (theta nodes/weights given, phi_k = 2 pi k/n_phi).
    Returns (R complex [n_states][n_r][(l_max+1)^2], <f^2>_Omega real [n_states][n_r]): Eq. (57), (59)."""
    f = np.asarray(f, np.complex128)
    ns, nr, nt, nph = f.shape
    if nph != n_phi or len(cos_theta) != nt or len(w_theta) != nt:
        raise ValueError("angular_moments: shape mismatch")
    fr = np.ascontiguousarray(np.stack([f.real, f.imag], axis=-1))
    ct = np.ascontiguousarray(cos_theta, np.float64)
    wt = np.ascontiguousarray(w_theta, np.float64)
    nlm = (l_max + 1) ** 2
    R = np.zeros((ns, nr, nlm, 2))
    f2 = np.zeros((ns, nr))
    if lib().oracle_angular_moments(ns, nr, nt, _dp(ct), _dp(wt), int(n_phi), int(l_max), _dp(fr), _dp(R), _dp(f2)) != 0:
        raise ValueError("oracle_angular_moments: bad arguments")
    return R[..., 0] + 1j * R[..., 1], f2

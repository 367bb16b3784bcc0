"""Seeded synthetic workloads shaped like the paper's (BASELINE.json `configs`).

This module (top level, outside both `paper_2512_18010_b200/` and `oracle/`) is the ONLY code shared by the CUDA
path and the CPU oracle.  It holds none of the
method's arithmetic: no Gaussian integrals, no normalisation constants, no form factors.  The one
place a workload needs the method (the AO overlap matrix S, used to Löwdin-orthonormalise the
random molecular orbitals and for the cond(S) guard) is passed in by the caller as `overlap_fn`:
tests pass the oracle's, `bench.py` passes the library's `scarf_overlap`.

The paper's own workloads are its 100-molecule test set (H, C, N, S, F; 1-20 heavy atoms; cc-pVDZ;
first 12 singlet states; 50^3-200^3 grids; PAPER.md:466, 477 = Table I caption, Fig. 4).  Neither
the molecules, the TD-DFT transition matrices nor the basis-set tables are available, so the five
configs below stand in for them with the same shape: ~10 heavy atoms, 12 transitions, l <= 2-3,
~2 primitives per shell, 1e5-1e6 q-points.

Config numbering here is 1-based as in SURVEY.md §8(a); BASELINE.json `configs[k-1]` is config k.

Conventions (SURVEY.md §8(c) readings #9, #13, #14, #16, #17):
  * atomic units: bohr, bohr^-1, bohr^-2;
  * Cartesian component order within a shell: a descending, then b descending (x,y,z; xx,xy,xz,yy,yz,zz; ...);
  * T is [n_states][nbf][nbf], real, AO basis, T^s = sum_ia X^s_ia c_i c_a^T (Eq. 17, Y = 0),
    ||X^s||_F = 1;
  * Cartesian grid: linspace(-Q, Q, N) inclusive per axis, point index (ix*N + iy)*N + iz;
  * spherical product grid: |q| log-spaced [0.05, 20] x Gauss-Legendre cos(theta) x uniform phi in [0, 2pi).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Callable, Optional

import numpy as np

N_CONFIGS = 5


@dataclass
class Basis:
    """Contracted Cartesian GTO basis in the layout the C-ABI takes (include/scarf.h)."""
    atom_xyz: np.ndarray      # [n_atoms][3] float64, bohr
    shell_atom: np.ndarray    # [n_shells] int32
    shell_l: np.ndarray       # [n_shells] int32
    shell_nprim: np.ndarray   # [n_shells] int32
    exponents: np.ndarray     # [sum nprim] float64, bohr^-2
    coeffs: np.ndarray        # [sum nprim] float64, coefficients of unit-normalised primitives

    @property
    def n_atoms(self) -> int:
        return int(self.atom_xyz.shape[0])

    @property
    def n_shells(self) -> int:
        return int(self.shell_l.shape[0])

    @property
    def nbf(self) -> int:
        l = self.shell_l.astype(np.int64)
        return int(np.sum((l + 1) * (l + 2) // 2))

    @property
    def n_prim_shells(self) -> int:
        return int(np.sum(self.shell_nprim))


@dataclass
class Workload:
    name: str
    config: int
    seed: int
    basis: Basis
    T: np.ndarray             # [n_states][nbf][nbf] float64
    q: np.ndarray             # [n_q][3] float64
    grid: dict = field(default_factory=dict)   # description of the q set
    cond_S: float = float("nan")
    n_occ: int = 0
    n_virt: int = 0

    @property
    def n_states(self) -> int:
        return int(self.T.shape[0])

    @property
    def n_q(self) -> int:
        return int(self.q.shape[0])


def cartesian_components(l: int):
    """(a, b, c) triples with a+b+c = l; a descending, then b descending."""
    return [(a, b, l - a - b) for a in range(l, -1, -1) for b in range(l - a, -1, -1)]


# --------------------------------------------------------------------------------------------
# q grids
# --------------------------------------------------------------------------------------------
def cartesian_axis(n: int, qmax: float) -> np.ndarray:
    """linspace(-qmax, qmax, n), made EXACTLY inversion-symmetric: ax[i] == -ax[n-1-i] bit for bit.  The grid of
    reading #13 is symmetric under q -> -q; numpy's linspace rounds the two halves differently (a few ulp), which
    would hide that symmetry from a bitwise test.  (ax - ax[::-1])/2 is antisymmetric by construction."""
    ax = np.linspace(-qmax, qmax, n)
    return 0.5 * (ax - ax[::-1])


def cartesian_grid(n: int, qmax: float) -> np.ndarray:
    ax = cartesian_axis(n, qmax)
    qx, qy, qz = np.meshgrid(ax, ax, ax, indexing="ij")
    return np.ascontiguousarray(np.stack([qx.ravel(), qy.ravel(), qz.ravel()], axis=1))


def spherical_grid(n_r: int = 128, n_theta: int = 64, n_phi: int = 128,
                   qmin: float = 0.05, qmax: float = 20.0) -> np.ndarray:
    r = np.geomspace(qmin, qmax, n_r)
    ct, _w = np.polynomial.legendre.leggauss(n_theta)
    st = np.sqrt(np.maximum(0.0, 1.0 - ct * ct))
    ph = 2.0 * np.pi * np.arange(n_phi) / n_phi
    R, CT, PH = np.meshgrid(r, ct, ph, indexing="ij")
    ST = np.broadcast_to(st[None, :, None], R.shape)
    q = np.stack([R * ST * np.cos(PH), R * ST * np.sin(PH), R * CT], axis=-1)
    return np.ascontiguousarray(q.reshape(-1, 3))


# --------------------------------------------------------------------------------------------
# geometry
# --------------------------------------------------------------------------------------------
def _random_walk_atoms(rng, n_heavy: int, n_h: int) -> np.ndarray:
    """New atom 2.5-3.0 bohr from a random existing heavy atom, rejected if < 2.0 bohr from any atom."""
    pts = [np.zeros(3)]

    def place(n_anchor):
        for _ in range(100000):
            anchor = pts[rng.integers(0, n_anchor)]
            d = rng.normal(size=3)
            d /= np.linalg.norm(d)
            cand = anchor + rng.uniform(2.5, 3.0) * d
            if min(np.linalg.norm(cand - p) for p in pts) >= 2.0:
                pts.append(cand)
                return
        raise RuntimeError("atom placement failed")

    while len(pts) < n_heavy:
        place(len(pts))
    for _ in range(n_h):
        place(n_heavy)
    xyz = np.array(pts)
    return xyz - xyz.mean(axis=0)


def _ring_atoms() -> np.ndarray:
    ang = 2.0 * np.pi * np.arange(6) / 6.0
    heavy = np.stack([2.6 * np.cos(ang), 2.6 * np.sin(ang), np.zeros(6)], axis=1)
    hyd = np.stack([4.7 * np.cos(ang), 4.7 * np.sin(ang), np.zeros(6)], axis=1)
    return np.concatenate([heavy, hyd], axis=0)


# --------------------------------------------------------------------------------------------
# shells
# --------------------------------------------------------------------------------------------
def _draw_exponents(rng, n: int, lo: float, hi: float, taken: list) -> np.ndarray:
    """n log-uniform exponents in [lo, hi], every ratio to the ones in `taken` (same atom, same l)
    and to each other >= 1.5 (redraw otherwise).  Falls back to a geometric ladder if the range is
    too narrow for rejection sampling to succeed."""
    out = []
    for _ in range(n):
        for _try in range(2000):
            a = float(np.exp(rng.uniform(np.log(lo), np.log(hi))))
            if all(max(a, b) / min(a, b) >= 1.5 for b in taken + out):
                out.append(a)
                break
        else:
            # narrow range: widen upward deterministically
            a = max(taken + out + [lo]) * 1.5
            out.append(a)
    return np.sort(np.array(out))[::-1]


def _build_shells(rng, atom_kinds, layouts, ranges):
    """atom_kinds[i] in layouts; layouts[kind] = list of (l, nprim or (lo,hi) for a uniform draw);
    ranges[kind][l] = (lo, hi) exponent range."""
    shell_atom, shell_l, shell_nprim, exps, cofs = [], [], [], [], []
    for ia, kind in enumerate(atom_kinds):
        taken = {}
        for (l, depth) in layouts[kind](ia):
            n = int(rng.integers(depth[0], depth[1] + 1)) if isinstance(depth, tuple) else int(depth)
            lo, hi = ranges[kind][l]
            e = _draw_exponents(rng, n, lo, hi, taken.setdefault(l, []))
            taken[l].extend(e.tolist())
            d = rng.uniform(0.2, 1.0, size=n)
            shell_atom.append(ia)
            shell_l.append(l)
            shell_nprim.append(n)
            exps.extend(e.tolist())
            cofs.extend(d.tolist())
    return (np.array(shell_atom, np.int32), np.array(shell_l, np.int32), np.array(shell_nprim, np.int32),
            np.array(exps, np.float64), np.array(cofs, np.float64))


def _basis_for_config(config: int, rng) -> Basis:
    if config == 1:
        xyz = np.array([[0.0, 0.0, -0.7], [0.0, 0.0, 0.7]])
        kinds = ["X", "X"]
        layouts = {"X": lambda ia: [(0, 3), (0, 3), (1, 3)]}
        ranges = {"X": {0: (0.1, 30.0), 1: (0.1, 30.0)}}
    elif config == 2:
        xyz = _ring_atoms()
        kinds = ["C"] * 6 + ["H"] * 6
        layouts = {"C": lambda ia: [(0, (1, 6)), (0, (1, 6)), (0, (1, 6)), (1, (1, 6)), (1, (1, 6)), (2, 1)],
                   "H": lambda ia: [(0, (1, 6)), (0, (1, 6))]}
        r = (0.08, 5000.0)
        ranges = {"C": {0: r, 1: r, 2: r}, "H": {0: r}}
    elif config in (3, 5):
        xyz = _random_walk_atoms(rng, 10, 8)
        kinds = ["C"] * 10 + ["H"] * 8
        layouts = {"C": lambda ia: [(0, 5), (0, 1), (0, 1), (1, 3), (1, 1), (2, 1)],
                   "H": lambda ia: [(0, 3), (0, 1), (1, 1)]}
        ranges = {"C": {0: (0.1, 3000.0), 1: (0.1, 40.0), 2: (0.5, 1.2)},
                  "H": {0: (0.1, 15.0), 1: (0.6, 1.0)}}
    elif config == 4:
        xyz = _random_walk_atoms(rng, 30, 20)
        kinds = ["C"] * 30 + ["H"] * 20
        layouts = {"C": lambda ia: ([(0, 6), (0, 2), (0, 1), (1, 4), (1, 1), (2, 1)]
                                    + ([(3, 1)] if ia % 6 == 0 else [])),
                   "H": lambda ia: [(0, 3), (0, 1), (1, 1)]}
        r = (0.05, 10000.0)
        ranges = {"C": {0: r, 1: r, 2: r, 3: r}, "H": {0: r, 1: r}}
    else:
        raise ValueError(f"config must be 1..{N_CONFIGS}")
    sa, sl, sn, e, d = _build_shells(rng, kinds, layouts, ranges)
    return Basis(np.ascontiguousarray(xyz, dtype=np.float64), sa, sl, sn, e, d)


_STATES = {1: (1, 1, 1), 2: (12, 5, 5), 3: (12, 8, 8), 4: (12, 10, 10), 5: (12, 8, 8)}
_GRIDS = {1: ("cartesian", 16, 4.0), 2: ("cartesian", 48, 8.0), 3: ("cartesian", 64, 10.0),
          4: ("cartesian", 64, 12.0), 5: ("spherical", (128, 64, 128), (0.05, 20.0))}
_NAMES = {1: "tiny-2atom-10bf-16^3", 2: "benzene-like-12atom-102bf-12st-48^3",
          3: "10heavy+8H-190bf-12st-64^3", 4: "30heavy+20H-600bf-12st-64^3",
          5: "10heavy+8H-190bf-12st-sph128x64x128"}


def make_q(config: int) -> tuple[np.ndarray, dict]:
    kind, n, lim = _GRIDS[config]
    if kind == "cartesian":
        return cartesian_grid(n, lim), {"kind": "cartesian", "n_per_axis": n, "qmax": lim}
    return (spherical_grid(n[0], n[1], n[2], lim[0], lim[1]),
            {"kind": "spherical", "n_r": n[0], "n_theta": n[1], "n_phi": n[2], "qmin": lim[0], "qmax": lim[1]})


def transitions_from_mos(S: np.ndarray, rng, n_states: int, n_occ: int, n_virt: int) -> np.ndarray:
    """Random S-orthonormal MOs (Löwdin: C = S^-1/2 Q) and T^s = sum_ia X^s_ia c_i c_a^T, ||X^s||_F = 1."""
    nbf = S.shape[0]
    w, U = np.linalg.eigh(0.5 * (S + S.T))
    S_inv_half = (U / np.sqrt(w)) @ U.T
    Q, _ = np.linalg.qr(rng.normal(size=(nbf, nbf)))
    C = S_inv_half @ Q
    Cocc, Cvir = C[:, :n_occ], C[:, n_occ:n_occ + n_virt]
    T = np.empty((n_states, nbf, nbf))
    for s in range(n_states):
        X = rng.normal(size=(n_occ, n_virt))
        X /= np.linalg.norm(X)
        T[s] = Cocc @ X @ Cvir.T
    return T


def make_workload(config: int, overlap_fn: Callable[[Basis], np.ndarray], seed: Optional[int] = None,
                  max_cond: float = 1e6, max_reseed: int = 20, with_q: bool = True) -> Workload:
    """Build config `config` (1..5).  `overlap_fn(basis)` must return the AO overlap matrix S
    (nbf x nbf, S_mu_mu = 1) computed by the caller's own implementation of the method."""
    if seed is None:
        seed = 1000 + config
    n_states, n_occ, n_virt = _STATES[config]
    last = None
    for bump in range(max_reseed + 1):
        rng = np.random.default_rng(seed + 7919 * bump)
        basis = _basis_for_config(config, rng)
        S = np.asarray(overlap_fn(basis), dtype=np.float64)
        if S.shape != (basis.nbf, basis.nbf):
            raise ValueError("overlap_fn returned the wrong shape")
        w = np.linalg.eigvalsh(0.5 * (S + S.T))
        cond = float(w[-1] / w[0]) if w[0] > 0 else float("inf")
        last = cond
        if cond <= max_cond:
            T = transitions_from_mos(S, rng, n_states, n_occ, n_virt)
            if with_q:
                q, grid = make_q(config)
            else:
                q, grid = np.zeros((0, 3)), {"kind": "none"}
            return Workload(_NAMES[config], config, seed + 7919 * bump, basis, np.ascontiguousarray(T), q, grid,
                            cond, n_occ, n_virt)
    raise RuntimeError(f"cond(S) guard not met after {max_reseed} reseeds (last cond {last:.3g})")


def sample_q_indices(n_q: int, n_sample: int, seed: int = 0) -> np.ndarray:
    """Seeded sample of q indices for sampled parity at full size: first, last, middle + random."""
    rng = np.random.default_rng(seed)
    fixed = np.array([0, n_q - 1, n_q // 2, n_q // 2 - 1], dtype=np.int64)
    rnd = rng.choice(n_q, size=max(0, min(n_q, n_sample) - fixed.size), replace=False)
    return np.unique(np.concatenate([fixed, rnd]))

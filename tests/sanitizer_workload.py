"""Small run through every kernel of libscarf, meant to be executed under compute-sanitizer on the GPU box:

    compute-sanitizer --tool memcheck  --error-exitcode 1 python tests/sanitizer_workload.py
    compute-sanitizer --tool racecheck --error-exitcode 1 python tests/sanitizer_workload.py
    compute-sanitizer --tool synccheck --error-exitcode 1 python tests/sanitizer_workload.py
    compute-sanitizer --tool initcheck --error-exitcode 1 python tests/sanitizer_workload.py

(results: profiles/r02_sanitizers.md).  Sizes are tiny (the tools slow kernels down 10-100 x) but span several q tiles,
several stream chunks (ticket fix-up), every pair class 0..12, two state tiles, ragged shapes.  No oracle here: parity is
the job of the pytest suite; this script only has to touch every code path and ends by printing a checksum."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import workloads as W                                   # noqa: E402
from paper_2512_18010_b200 import Scarf                 # noqa: E402


def basis(lmax):
    rng = np.random.default_rng(61)
    sa, sl, sn, ex, co = [], [], [], [], []
    for atom in (0, 1):
        for l in range(lmax + 1):
            n = 2 if l in (0, 4) else 1
            sa.append(atom); sl.append(l); sn.append(n)
            ex.extend(sorted(rng.uniform(0.5, 1.6, size=n) * (2.0 if n == 2 else 1.0), reverse=True))
            co.extend(rng.uniform(0.4, 1.0, size=n))
    return W.Basis(np.array([[0.1, 0.2, -0.8], [0.3, -0.4, 0.9]]), np.array(sa, np.int32), np.array(sl, np.int32),
                   np.array(sn, np.int32), np.array(ex), np.array(co))


def main():
    import torch
    rng = np.random.default_rng(1)
    total = 0.0
    with Scarf(0) as sc:
        for lmax, n_states, n_q in ((3, 13, 700), (6, 2, 130)):
            b = basis(lmax)
            sc.set_basis(b)
            T = rng.normal(size=(n_states, b.nbf, b.nbf))
            q = rng.uniform(-4, 4, size=(n_q, 3))
            for opts in ({"n_chunks": 0, "adaptive_tol": 0.0}, {"n_chunks": 3, "adaptive_tol": 0.0}, {"n_chunks": 5, "adaptive_tol": 1e-6}):
                for k, v in opts.items():
                    sc.set_option(k, v)
                sc.set_transitions(torch.as_tensor(T, device="cuda"))
                total += float(np.abs(sc.form_factors(torch.as_tensor(q, device="cuda")).cpu().numpy()).sum())
                total += float(np.abs(sc.form_factors(q)).sum())
                ax = [W.cartesian_axis(6, 3.0), W.cartesian_axis(9, 2.5), W.cartesian_axis(5, 3.5)]
                total += float(np.abs(sc.form_factors_grid(*ax)).sum())
                ax[1] = np.linspace(-2, 3, 9)
                total += float(np.abs(sc.form_factors_grid(*ax)).sum())
                # the three product-grid kernels by name (box, row, mirror-pair row with its tensor-core classes) on rows long
                # enough for the row kernels; 13 states = a tile of 12 (mma.sync path) and a tile of 1 (DFMA path)
                axr = [W.cartesian_axis(3, 3.0), W.cartesian_axis(5, 2.5), W.cartesian_axis(66, 3.5)]
                for variant in (0, 1, 2):
                    sc.set_option("grid_variant", variant)
                    total += float(np.abs(sc.form_factors_grid(*axr)).sum())
                    assert sc.stats()["last_grid_variant"] == variant
                sc.set_option("grid_variant", -1)
                if lmax == 3:                           # the spherical-grid kernel (two radius boxes, inversion-symmetric directions)
                    ct, _ = np.polynomial.legendre.leggauss(6)
                    total += float(np.abs(sc.form_factors_sph(np.geomspace(0.1, 3.0, 70), ct, 8).cpu().numpy()).sum())
                sc.stats()
            sc.set_option("n_chunks", 0); sc.set_option("adaptive_tol", 0.0)
            sc.set_transitions(T)
            w = [rng.uniform(0.1, 1, a.size) for a in ax]
            total += float(np.abs(sc.separable_integral(ax[0], w[0], ax[1], w[1], ax[2], w[2])).sum())
            sc.set_option("check_parseval", 1)
            for variant in (1, 2, 0):
                sc.set_option("fft_density_variant", variant)
                total += float(np.abs(sc.fft_form_factors((8, 6, 10), np.array([-6.0, -6.0, -6.5]), np.array([12.0, 12.5, 13.0]),
                                                          device_out=False)).sum())
            total += float(sc.fft_parseval().sum())
        # pure shells
        flags = np.array([0, 0, 1, 1, 1, 1, 1] * 2, np.int32)
        sc.set_basis(b, shell_pure=flags)
        T = rng.normal(size=(2, sc.nbf, sc.nbf))
        sc.set_transitions(T)
        total += float(np.abs(sc.form_factors(q[:40])).sum())
        # angular moments: fused tensor-core kernel, the unfused tensor-core route (F too large), and the SIMT kernels
        for shape, l_max in (((2, 3, 10, 18), 6), ((1, 1, 150, 64), 31), ((1, 2, 5, 2048), 3)):
            f = rng.normal(size=shape) + 1j * rng.normal(size=shape)
            ct, wt = np.polynomial.legendre.leggauss(shape[2])
            for variant in (1, 0):
                sc.set_option("angular_variant", variant)
                R, f2 = sc.angular_moments(torch.as_tensor(f, device="cuda"), ct, wt, shape[3], l_max, n_r=shape[1])
                total += float(R.abs().sum().item()) + float(f2.sum().item())
        total += float(sc.abs2(torch.as_tensor(f, device="cuda")).sum().item())
    assert np.isfinite(total)
    print("sanitizer workload done, checksum %.6e" % total)


if __name__ == "__main__":
    main()

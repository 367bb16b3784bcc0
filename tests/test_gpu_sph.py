"""GPU parity of scarf_form_factors_sph (csrc/ff_sph.cu; the spherical product grid of the angular
moments, Eq. (57)-(60) PAPER.md:380-398; S4 = Eq. (48)): a warp owns one direction and 64 radii, the
per-direction sums of the polynomial and the phase slope n.P are evaluated once per (direction, pair, state); half of the
directions on an inversion-symmetric grid (reading #6: f(-q) = conj f(q)).  Against the CPU oracle on the expanded point list
at 1e-10 * max|f_s|, and against the list kernel."""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-10


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests must run on the B200 box")
    return torch


@pytest.fixture(scope="module")
def Scarf():
    from paper_2512_18010_b200 import Scarf as S
    return S


def sph_points(r, ct, n_phi):
    """The grid as a point list, index (i*n_theta + j)*n_phi + k — written out here from the definition in scarf.h."""
    st = np.sqrt(np.maximum(0.0, 1.0 - ct * ct))
    ph = 2.0 * np.pi * np.arange(n_phi) / n_phi
    R, CT, PH = np.meshgrid(r, ct, ph, indexing="ij")
    ST = np.broadcast_to(st[None, :, None], R.shape)
    return np.ascontiguousarray(np.stack([R * ST * np.cos(PH), R * ST * np.sin(PH), R * CT], axis=-1).reshape(-1, 3))


def assert_parity(f_gpu, f_ref, tol=TOL):
    assert f_gpu.shape == f_ref.shape
    for s in range(f_ref.shape[0]):
        scale = np.max(np.abs(f_ref[s]))
        err = np.max(np.abs(f_gpu[s] - f_ref[s]))
        assert err <= tol * scale, f"state {s}: max err {err:.3e} > {tol:g} * {scale:.3e}"


def all_class_basis():
    """s, p, d, f shells on two centres (a contracted s on each): every pair class L = 0..6 is populated."""
    return W.Basis(np.array([[0.1, 0.2, -0.9], [0.3, -0.4, 1.0]]), np.array([0, 0, 0, 0, 1, 1, 1, 1], np.int32),
                   np.array([0, 1, 2, 3, 0, 1, 2, 3], np.int32), np.array([2, 1, 1, 1, 2, 1, 1, 1], np.int32),
                   np.array([2.1, 0.4, 1.3, 0.9, 0.7, 1.9, 0.5, 1.1, 0.8, 0.6]),
                   np.array([0.5, 0.6, 1.0, 1.0, 1.0, 0.7, 0.4, 1.0, 1.0, 1.0]))


def sph_ff(Scarf, torch, basis, T, r, ct, n_phi, device=True, **options):
    with Scarf(0) as sc:
        sc.set_basis(basis)
        for k, v in options.items():
            sc.set_option(k, v)
        sc.set_transitions(torch.as_tensor(T, dtype=torch.float64, device="cuda").contiguous())
        f = sc.form_factors_sph(r, ct, n_phi, device=device)
        if device:
            torch.cuda.synchronize()
            return f.cpu().numpy(), sc.stats()
        return np.array(f), sc.stats()


@pytest.mark.parametrize("shape", [(1, 1, 1), (5, 4, 8), (70, 3, 6), (64, 5, 4), (33, 2, 7), (130, 1, 2)])
@pytest.mark.parametrize("n_states", [12, 13])
def test_sph_ragged_shapes_all_classes(oracle_mod, Scarf, torch_cuda, shape, n_states):
    """Rows of 64 radii, 4 directions per CTA: shapes below, at and above one box, ragged in both; arbitrary (unsorted, also
    negative) radii and non-symmetric theta nodes; all classes L = 0..6; one and two state tiles."""
    n_r, n_t, n_p = shape
    b = all_class_basis()
    rng = np.random.default_rng(sum(shape) + n_states)
    T = rng.normal(size=(n_states, b.nbf, b.nbf))
    r = rng.uniform(-1.0, 6.0, size=n_r)
    ct = rng.uniform(-1.0, 1.0, size=n_t)
    f, st = sph_ff(Scarf, torch_cuda, b, T, r, ct, n_p)
    assert st["last_grid_variant"] == 3 and st["last_grid_symmetric"] == 0
    assert_parity(f, oracle_mod.form_factors(b, T, sph_points(r, ct, n_p)))


@pytest.mark.parametrize("n_states", [1, 2, 3, 5, 7])
def test_sph_state_tile_sizes(oracle_mod, Scarf, torch_cuda, n_states):
    b = all_class_basis()
    rng = np.random.default_rng(170 + n_states)
    T = rng.normal(size=(n_states, b.nbf, b.nbf))
    r = np.geomspace(0.05, 7.0, 40)
    ct = np.array([-0.8, 0.1, 0.6])
    f, _ = sph_ff(Scarf, torch_cuda, b, T, r, ct, 5)
    assert_parity(f, oracle_mod.form_factors(b, T, sph_points(r, ct, 5)))


@pytest.mark.parametrize("shape", [(9, 4, 8), (66, 5, 6), (3, 1, 2), (4, 7, 12), (5, 2, 2)])
@pytest.mark.parametrize("device", [True, False])
def test_sph_inversion_symmetry_both_halves(oracle_mod, Scarf, torch_cuda, shape, device):
    """Gauss-Legendre theta nodes (antisymmetric bit for bit) and even n_phi: the first half of the directions is evaluated (for odd
    n_theta also half of the equator row), the mirror point (i, n_theta-1-j, k + n_phi/2) gets the conjugate.  Every point of both
    halves against the oracle; the stored values obey the mirror relation exactly; the plain path agrees to round-off."""
    n_r, n_t, n_p = shape
    b = all_class_basis()
    rng = np.random.default_rng(sum(shape))
    T = rng.normal(size=(12, b.nbf, b.nbf))
    r = np.geomspace(0.05, 6.0, n_r)
    ct, _ = np.polynomial.legendre.leggauss(n_t)
    assert np.array_equal(ct, -ct[::-1])
    f_ref = oracle_mod.form_factors(b, T, sph_points(r, ct, n_p))
    f, st = sph_ff(Scarf, torch_cuda, b, T, r, ct, n_p, device=device)
    assert st["last_grid_symmetric"] == 1 and st["last_grid_variant"] == 3
    assert_parity(f, f_ref)
    g = f.reshape(12, n_r, n_t, n_p)
    assert np.array_equal(np.roll(g[:, :, ::-1, :], n_p // 2, axis=3), np.conj(g))
    f0, st0 = sph_ff(Scarf, torch_cuda, b, T, r, ct, n_p, device=device, grid_symmetry=0)
    assert st0["last_grid_symmetric"] == 0
    assert np.max(np.abs(f0 - f)) <= 1e-13 * np.max(np.abs(f_ref))
    assert_parity(f0, f_ref)


def test_sph_not_symmetric_falls_back(oracle_mod, Scarf, torch_cuda):
    """Odd n_phi, a node off by one ulp, a shifted node set: every direction is evaluated."""
    b = all_class_basis()
    rng = np.random.default_rng(7)
    T = rng.normal(size=(3, b.nbf, b.nbf))
    r = np.linspace(0.1, 4.0, 6)
    ct, _ = np.polynomial.legendre.leggauss(4)
    ulp = ct.copy()
    ulp[0] = np.nextafter(ulp[0], 1.0)
    for nodes, n_p in ((ct, 7), (ulp, 8), (ct * 0.9 + 0.05, 8)):
        f, st = sph_ff(Scarf, torch_cuda, b, T, r, nodes, n_p)
        assert st["last_grid_symmetric"] == 0
        assert_parity(f, oracle_mod.form_factors(b, T, sph_points(r, nodes, n_p)))


@pytest.mark.parametrize("K", [1, 2, 7, 32])
def test_sph_chunk_counts(oracle_mod, Scarf, torch_cuda, K):
    b = all_class_basis()
    rng = np.random.default_rng(190 + K)
    T = rng.normal(size=(5, b.nbf, b.nbf))
    r = np.geomspace(0.05, 5.0, 67)
    ct, _ = np.polynomial.legendre.leggauss(3)
    f, st = sph_ff(Scarf, torch_cuda, b, T, r, ct, 6, n_chunks=K)
    assert st["last_n_chunks"] == K and st["last_grid_symmetric"] == 1
    assert_parity(f, oracle_mod.form_factors(b, T, sph_points(r, ct, 6)))
    z, _ = sph_ff(Scarf, torch_cuda, b, np.zeros_like(T), r, ct, 6, n_chunks=K)
    assert not np.any(z)


def test_sph_config5_full_size_sampled_and_list_kernel(oracle_mod, Scarf, torch_cuda):
    """Config 5 (128 x 64 x 128 points, 12 states) in the launch configuration bench.py times: the oracle on a seeded sample of
    points, the list kernel (scarf_form_factors on the workload's own point list) on every point."""
    torch = torch_cuda
    w = W.make_workload(5, oracle_mod.overlap)
    g = w.grid
    r = np.geomspace(g["qmin"], g["qmax"], g["n_r"])
    ct, _ = np.polynomial.legendre.leggauss(g["n_theta"])
    idx = W.sample_q_indices(w.n_q, 160, seed=5)
    f_ref = oracle_mod.form_factors(w.basis, w.T, w.q[idx])
    with Scarf(0) as sc:
        sc.set_basis(w.basis)
        sc.set_transitions(torch.as_tensor(w.T, device="cuda"))
        fs = sc.form_factors_sph(r, ct, g["n_phi"])
        st = sc.stats()
        assert st["last_grid_symmetric"] == 1 and st["last_grid_variant"] == 3
        fl = sc.form_factors(torch.as_tensor(w.q, device="cuda"))
        torch.cuda.synchronize()
        assert_parity(fs[:, torch.as_tensor(idx, device="cuda")].cpu().numpy(), f_ref)
        scale = fl.abs().amax(dim=1)
        err = (fs - fl).abs().amax(dim=1)
        assert bool((err <= 1e-11 * scale).all()), (err / scale).max().item()


def test_sph_feeds_angular_moments(oracle_mod, Scarf, torch_cuda):
    """The output layout is scarf_angular_moments' input layout: R_lm and <f^2> from the spherical path equal those from the list path."""
    torch = torch_cuda
    b = all_class_basis()
    rng = np.random.default_rng(3)
    T = rng.normal(size=(4, b.nbf, b.nbf))
    n_r, n_t, n_p, l_max = 6, 8, 16, 4
    r = np.geomspace(0.1, 3.0, n_r)
    ct, wt = np.polynomial.legendre.leggauss(n_t)
    with Scarf(0) as sc:
        sc.set_basis(b)
        sc.set_transitions(T)
        R1, f21 = sc.angular_moments(sc.form_factors_sph(r, ct, n_p), ct, wt, n_p, l_max, n_r=n_r)
        R2, f22 = sc.angular_moments(sc.form_factors(torch.as_tensor(sph_points(r, ct, n_p), device="cuda")), ct, wt, n_p, l_max, n_r=n_r)
        torch.cuda.synchronize()
        assert float((R1 - R2).abs().max()) <= 1e-12 * float(R2.abs().max())
        assert float((f21 - f22).abs().max()) <= 1e-12 * float(f22.abs().max())


def test_sph_high_classes_list_fallback_and_errors(oracle_mod, Scarf, torch_cuda):
    """A basis with a g shell (pair classes beyond 6) runs the list path internally; argument errors."""
    b = W.Basis(np.array([[0.0, 0.1, -0.2], [0.4, -0.3, 0.9]]), np.array([0, 1, 1], np.int32), np.array([4, 0, 1], np.int32),
                np.array([1, 1, 1], np.int32), np.array([0.9, 1.2, 0.7]), np.array([1.0, 1.0, 1.0]))
    rng = np.random.default_rng(12)
    T = rng.normal(size=(2, b.nbf, b.nbf))
    r = np.linspace(0.2, 3.0, 5)
    ct, _ = np.polynomial.legendre.leggauss(4)
    f, st = sph_ff(Scarf, torch_cuda, b, T, r, ct, 6)
    assert st["last_grid_variant"] == -1
    assert_parity(f, oracle_mod.form_factors(b, T, sph_points(r, ct, 6)))
    w = W.make_workload(1, oracle_mod.overlap)
    with Scarf(0) as sc:
        sc.set_basis(w.basis)
        with pytest.raises(Exception):
            sc.form_factors_sph(r, ct, 6)                  # no transitions yet
        sc.set_transitions(w.T)
        assert sc.form_factors_sph(r, ct, 0).shape == (1, 0)
        with pytest.raises(Exception):
            sc.form_factors_sph(r, np.array([0.5, 1.5]), 4)        # |cos theta| > 1
        bad = r.copy()
        bad[2] = np.inf
        with pytest.raises(Exception):
            sc.form_factors_sph(bad, ct, 4)


@pytest.mark.parametrize("symmetric", [True, False])
def test_sph_pinned_and_pageable_host_output(oracle_mod, Scarf, torch_cuda, symmetric):
    """Host `out`, pinned or pageable (computed on the device, one copy; the kernel's strided 16-byte stores are not sent over PCIe):
    bit-identical to the device-output call; oracle on every point."""
    torch = torch_cuda
    b = all_class_basis()
    rng = np.random.default_rng(31 + symmetric)
    T = rng.normal(size=(13, b.nbf, b.nbf))
    n_r, n_t, n_p = 70, 5, 6
    r = np.geomspace(0.05, 6.0, n_r)
    ct = np.polynomial.legendre.leggauss(n_t)[0] if symmetric else rng.uniform(-1, 1, size=n_t)
    n_q = n_r * n_t * n_p
    f_ref = oracle_mod.form_factors(b, T, sph_points(r, ct, n_p))
    with Scarf(0) as sc:
        sc.set_basis(b)
        sc.set_option("n_chunks", 5)
        sc.set_transitions(torch.as_tensor(T, device="cuda"))
        f_dev = sc.form_factors_sph(r, ct, n_p)
        torch.cuda.synchronize()
        f_dev = f_dev.cpu().numpy()
        assert sc.stats()["last_grid_symmetric"] == int(symmetric)
        pinned = torch.full((13, n_q, 2), float("nan"), dtype=torch.float64).pin_memory()
        f_pin = sc.form_factors_sph(r, ct, n_p, out=pinned).numpy().copy()
        sc.set_option("host_zero_copy", 0)
        f_np = np.array(sc.form_factors_sph(r, ct, n_p, device=False))
    assert_parity(f_pin, f_ref)
    assert np.array_equal(f_pin, f_dev) and np.array_equal(f_np, f_dev)

"""GPU parity of scarf_fft_form_factors (the paper's FFT method, Eq. (19)-(34) PAPER.md:140-222)
against its CPU oracle (oracle/fft_method.py) on the same grid, and convergence to the analytic kernel's result."""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu


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


def assert_parity(f_gpu, f_ref, tol=1e-10):
    assert f_gpu.shape == f_ref.shape
    for s in range(f_ref.shape[0]):
        scale = np.max(np.abs(f_ref[s]))
        err = np.max(np.abs(f_gpu[s] - f_ref[s]))
        assert err <= tol * scale, f"state {s}: max err {err:.3e} > {tol:g} * {scale:.3e}"


@pytest.mark.parametrize("n,n_states", [((8, 8, 8), 1), ((24, 20, 28), 3), ((15, 9, 21), 13), ((1, 5, 2), 2)])
def test_fft_method_matches_oracle(oracle_mod, Scarf, torch_cuda, n, n_states):
    """Even, odd and ragged grid sizes (several CTAs and a tail), one and two state tiles, an off-centre box;
    basis with s, p, d, f shells and contractions (config-1 atoms plus a d/f centre)."""
    torch = torch_cuda
    from oracle import fft_method as offt
    b = W.Basis(np.array([[0.0, 0.0, 0.7], [0.0, 0.0, -0.7], [0.9, -0.5, 0.1]]), np.array([0, 0, 1, 1, 2, 2], np.int32),
                np.array([0, 1, 0, 2, 3, 1], np.int32), np.array([3, 2, 1, 1, 1, 2], np.int32),
                np.array([5.0, 1.2, 0.3, 2.0, 0.6, 0.9, 1.1, 0.8, 1.5, 0.4]),
                np.array([0.3, 0.6, 0.4, 0.7, 0.5, 1.0, 1.0, 1.0, 0.6, 0.8]))
    rng = np.random.default_rng(sum(n) + n_states)
    T = rng.normal(size=(n_states, b.nbf, b.nbf))
    x_min, L = np.array([-5.0, -4.5, -6.0]), np.array([10.5, 9.0, 11.0])
    f_ref = offt.form_factors(b, T, n, x_min, L)
    with Scarf(0) as sc:
        sc.set_basis(b)
        sc.set_transitions(torch.as_tensor(T, device="cuda"))
        f = sc.fft_form_factors(n, x_min, L)
        torch.cuda.synchronize()
        assert_parity(f.cpu().numpy(), f_ref)
        fh = sc.fft_form_factors(n, x_min, L, device_out=False)          # host output buffer
        assert np.array_equal(fh, f.cpu().numpy())
        sc.set_transitions(T)                                            # host T
        assert np.array_equal(sc.fft_form_factors(n, x_min, L, device_out=False), fh)
        sc.set_option("fft_density_variant", 0)                          # SIMT density kernel instead of the DMMA one
        assert_parity(sc.fft_form_factors(n, x_min, L, device_out=False), f_ref)


def test_fft_method_converges_to_the_analytic_kernel(oracle_mod, Scarf, torch_cuda):
    """Soft basis, 64^3 grid of spacing 0.25 bohr: the two GPU routes (tabulate-and-transform vs Eq. 48 in closed form)
    agree to 1e-8 away from the Nyquist faces; pure d shell included (T in the mixed basis)."""
    torch = torch_cuda
    from oracle import fft_method as offt
    from tests.test_oracle_fft import soft_basis
    b = soft_basis()
    pure = np.array([0, 0, 1, 0, 0], np.int32)
    nbf = b.nbf - 1
    rng = np.random.default_rng(8)
    T = rng.normal(size=(2, nbf, nbf))
    n, x_min, L = (64, 64, 64), np.array([-8.0] * 3), np.array([16.0] * 3)
    q = offt.q_points(n, L)
    idx = np.flatnonzero(np.max(np.abs(q), axis=1) < 9.0)[::97]
    with Scarf(0) as sc:
        sc.set_basis(b, shell_pure=pure)
        sc.set_transitions(T)
        f_fft = sc.fft_form_factors(n, x_min, L)[:, torch.as_tensor(idx, device="cuda")].cpu().numpy()
        f_ana = sc.form_factors(q[idx])
    for s in range(2):
        assert np.max(np.abs(f_fft[s] - f_ana[s])) <= 1e-8 * np.max(np.abs(f_ana[s]))


def test_fft_method_argument_checks(oracle_mod, Scarf, torch_cuda):
    w = W.make_workload(1, oracle_mod.overlap)
    with Scarf(0) as sc:
        sc.set_basis(w.basis)
        with pytest.raises(Exception):
            sc.fft_form_factors((4, 4, 4), np.zeros(3), np.ones(3))       # no transitions yet
        sc.set_transitions(w.T)
        with pytest.raises(Exception):
            sc.fft_form_factors((4, 4, 4), np.zeros(3), np.array([1.0, 0.0, 1.0]))
        with pytest.raises(Exception):
            sc.fft_form_factors((4, 0, 4), np.zeros(3), np.ones(3))


@pytest.mark.parametrize("config,n,extra_states", [(3, (20, 12, 28), 0), (3, (10, 6, 14), 1), (4, (10, 6, 14), 0), (4, (5, 6, 7), 1)])
def test_fft_density_at_config_basis_sizes(oracle_mod, Scarf, torch_cuda, config, n, extra_states):
    """The DMMA density kernel at the basis sizes bench.py times: config 3's basis (nbf = 190 -> padded
    to 192: the last mu/nu fragments are partly zero padding, 24 mu-chunks) and config 4's (nbf = 600, f shells), 12 states
    (one pass) and 13 (two state tiles), on a small ragged real-space grid (several CTAs and a partial warp) against the
    oracle's orbital-product einsum; both density kernels."""
    torch = torch_cuda
    from oracle import fft_method as offt
    w = W.make_workload(config, oracle_mod.overlap, with_q=False)
    T = w.T
    if extra_states:
        rng = np.random.default_rng(config)
        T = np.concatenate([T, 0.05 * rng.normal(size=(extra_states, w.basis.nbf, w.basis.nbf))], axis=0)
    lo = w.basis.atom_xyz.min(axis=0) - 1.5
    L = w.basis.atom_xyz.max(axis=0) + 1.5 - lo
    f_ref = offt.form_factors(w.basis, T, n, lo, L)
    with Scarf(0) as sc:
        sc.set_basis(w.basis)
        sc.set_transitions(torch.as_tensor(T, device="cuda"))
        for variant in (1, 2, 0):
            sc.set_option("fft_density_variant", variant)
            f = sc.fft_form_factors(n, lo, L)
            torch.cuda.synchronize()
            assert_parity(f.cpu().numpy(), f_ref)


@pytest.mark.parametrize("n_s", [1, 2, 3, 4, 5, 6, 7, 8])
def test_fft_density_padded_fragments(oracle_mod, Scarf, torch_cuda, n_s):
    """nbf = 24 + n_s: every residue of nbf mod 8 (and mod 4), so the zero-padded rows/columns of the last DMMA fragments are
    exercised against the oracle (not only GPU against GPU)."""
    torch = torch_cuda
    from oracle import fft_method as offt
    rng = np.random.default_rng(100 + n_s)
    atoms = np.array([[0.0, 0.0, 0.7], [0.0, 0.0, -0.7], [0.9, -0.5, 0.1]])
    sa = [0, 0, 1, 1, 2, 2] + [int(i % 3) for i in range(n_s)]
    sl = [0, 1, 0, 2, 3, 1] + [0] * n_s
    sn = [3, 2, 1, 1, 1, 2] + [1] * n_s
    ex = [5.0, 1.2, 0.3, 2.0, 0.6, 0.9, 1.1, 0.8, 1.5, 0.4] + list(0.25 * 1.7 ** np.arange(n_s))
    co = [0.3, 0.6, 0.4, 0.7, 0.5, 1.0, 1.0, 1.0, 0.6, 0.8] + [1.0] * n_s
    b = W.Basis(atoms, np.array(sa, np.int32), np.array(sl, np.int32), np.array(sn, np.int32), np.array(ex), np.array(co))
    assert b.nbf == 24 + n_s
    T = rng.normal(size=(5, b.nbf, b.nbf))
    n, x_min, L = (9, 11, 7), np.array([-5.0, -4.5, -6.0]), np.array([10.5, 9.0, 11.0])
    f_ref = offt.form_factors(b, T, n, x_min, L)
    with Scarf(0) as sc:
        sc.set_basis(b)
        sc.set_transitions(T)
        for variant in (1, 2, 0):
            sc.set_option("fft_density_variant", variant)
            assert_parity(sc.fft_form_factors(n, x_min, L, device_out=False), f_ref)


def test_parseval_check_eq75(oracle_mod, Scarf, torch_cuda):
    """Option check_parseval (the paper's check_parseval flag, Eq. (75)): both sides as the library reports
    them against the oracle's arrays, ragged grid, 13 states (two tiles); ESTATE without a checked call."""
    from oracle import fft_method as offt
    from paper_2512_18010_b200.binding import ScarfError, SCARF_ESTATE
    from tests.test_oracle_fft import soft_basis
    b = soft_basis()
    rng = np.random.default_rng(15)
    T = rng.normal(size=(13, b.nbf, b.nbf))
    n, x_min, L = (14, 9, 11), np.array([-4.0, -3.5, -4.5]), np.array([8.0, 7.5, 9.0])
    phi = offt.density_grid(b, T, n, x_min, L)
    f_ref = offt.transform(phi, x_min, L)
    vpix, vbox = np.prod(L) / np.prod(n), np.prod(L)
    with Scarf(0) as sc:
        sc.set_basis(b)
        sc.set_transitions(T)
        sc.fft_form_factors(n, x_min, L)
        with pytest.raises(ScarfError) as e:
            sc.fft_parseval()
        assert e.value.code == SCARF_ESTATE
        sc.set_option("check_parseval", 1)
        sc.fft_form_factors(n, x_min, L)
        P = sc.fft_parseval()
    np.testing.assert_allclose(P[:, 0], vpix * np.sum(phi ** 2, axis=(1, 2, 3)), rtol=1e-12)
    np.testing.assert_allclose(P[:, 1], np.sum(np.abs(f_ref) ** 2, axis=1) / vbox, rtol=1e-12)
    np.testing.assert_allclose(P[:, 0], P[:, 1], rtol=1e-12)

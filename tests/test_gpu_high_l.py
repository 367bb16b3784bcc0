"""GPU parity for shells up to i (l = 6, pair classes L = 0..12; "up to i orbitals"):
the unrolled kernels (classes 0..6) plus the high-class kernel (csrc/ff_highl.cu, classes 7..12) against the oracle, on
point lists and product grids (plain and inversion-symmetric), several state tiles, pure g/h/i shells."""
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


def spdfghi_basis():
    """Two centres, each with s, p, d, f, g, h, i shells (a contracted g): every pair class L = 0..12 is populated."""
    rng = np.random.default_rng(61)
    sa, sl, sn, ex, co = [], [], [], [], []
    for atom in (0, 1):
        for l in range(7):
            n = 2 if l in (0, 4) else 1
            sa.append(atom); sl.append(l); sn.append(n)
            ex.extend(sorted(rng.uniform(0.5, 1.6, size=n) * (2.0 if n == 2 else 1.0), reverse=True))
            co.extend(rng.uniform(0.4, 1.0, size=n))
    return W.Basis(np.array([[0.1, 0.2, -0.8], [0.3, -0.4, 0.9]]), np.array(sa, np.int32), np.array(sl, np.int32),
                   np.array(sn, np.int32), np.array(ex), np.array(co))


def assert_parity(f_gpu, f_ref, tol=TOL):
    assert f_gpu.shape == f_ref.shape
    for s in range(f_ref.shape[0]):
        scale = np.max(np.abs(f_ref[s]))
        err = np.max(np.abs(f_gpu[s] - f_ref[s]))
        assert err <= tol * scale, f"state {s}: max err {err:.3e} > {tol:g} * {scale:.3e}"


def expand(qx, qy, qz):
    X, Y, Z = np.meshgrid(qx, qy, qz, indexing="ij")
    return np.ascontiguousarray(np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1))


@pytest.mark.parametrize("n_states", [1, 12, 13])
def test_all_classes_0_to_12_point_list(oracle_mod, torch_cuda, n_states):
    from paper_2512_18010_b200 import Scarf
    torch = torch_cuda
    b = spdfghi_basis()
    rng = np.random.default_rng(n_states)
    T = rng.normal(size=(n_states, b.nbf, b.nbf))
    q = rng.uniform(-4, 4, size=(301, 3))
    q[0] = 0.0
    f_ref = oracle_mod.form_factors(b, T, q)
    with Scarf(0) as sc:
        sc.set_basis(b)
        sc.set_transitions(torch.as_tensor(T, device="cuda"))
        f = sc.form_factors(torch.as_tensor(q, device="cuda"))
        torch.cuda.synchronize()
        st = sc.stats()
        assert all(n > 0 for n in st["pairs_kept_per_class"]) and len(st["pairs_kept_per_class"]) == 13
        assert_parity(f.cpu().numpy(), f_ref)
        assert_parity(sc.form_factors(q), f_ref)                       # host buffers


def test_all_classes_product_grid_plain_and_symmetric(oracle_mod, torch_cuda):
    from paper_2512_18010_b200 import Scarf
    b = spdfghi_basis()
    rng = np.random.default_rng(77)
    T = rng.normal(size=(3, b.nbf, b.nbf))
    for axes, sym in (([W.cartesian_axis(6, 3.0), W.cartesian_axis(5, 2.5), W.cartesian_axis(9, 3.5)], 1),
                      ([np.linspace(-3, 2, 5), np.linspace(-2, 3, 9), np.linspace(-1, 4, 6)], 0)):
        f_ref = oracle_mod.form_factors(b, T, expand(*axes))
        with Scarf(0) as sc:
            sc.set_basis(b)
            sc.set_transitions(T)
            f = sc.form_factors_grid(*axes)
            assert sc.stats()["last_grid_symmetric"] == sym
        assert_parity(f, f_ref)
        if sym:
            assert np.array_equal(f[:, ::-1], np.conj(f))


def test_pure_g_h_i_shells(oracle_mod, torch_cuda):
    """Pure g, h, i shells mixed with Cartesian ones: T in the mixed basis, oracle = oracle/pure.py."""
    from oracle import pure as opure
    from paper_2512_18010_b200 import Scarf
    from tests.test_oracle_pins_high_l import _ghi_basis
    b = _ghi_basis()
    flags = np.array([1, 0, 1, 0], np.int32)
    rng = np.random.default_rng(5)
    nbf = opure.basis_matrix(b, flags).shape[1]
    T = rng.normal(size=(2, nbf, nbf))
    q = rng.uniform(-3, 3, size=(150, 3))
    f_ref = opure.form_factors(b, flags, T, q)
    with Scarf(0) as sc:
        sc.set_basis(b, shell_pure=flags)
        assert sc.nbf == nbf
        sc.set_transitions(T)
        assert_parity(sc.form_factors(q), f_ref)


def test_separable_integral_and_fft_method_with_g_h_i(oracle_mod, torch_cuda):
    """The other entry points on a basis with high shells: separable integrals (moments up to t = 12) against the oracle's
    weighted grid sum, and the FFT method's orbital tabulation against its oracle."""
    from oracle import fft_method as offt
    from paper_2512_18010_b200 import Scarf
    from tests.test_oracle_pins_high_l import _ghi_basis
    b = _ghi_basis()
    rng = np.random.default_rng(9)
    T = rng.normal(size=(2, b.nbf, b.nbf))
    qx, qy, qz = np.linspace(-2, 2, 7), np.linspace(-1.5, 2.5, 5), np.linspace(-2.5, 1.5, 6)
    wx, wy, wz = rng.uniform(0.1, 1, 7), rng.uniform(0.1, 1, 5), rng.uniform(0.1, 1, 6)
    f_ref = oracle_mod.form_factors(b, T, expand(qx, qy, qz)).reshape(2, 7, 5, 6)
    I_ref = np.einsum("sxyz,x,y,z->s", f_ref, wx, wy, wz)
    n, x_min, L = (8, 6, 10), np.array([-6.0, -6.0, -6.5]), np.array([12.0, 12.5, 13.0])
    ff_ref = offt.form_factors(b, T, n, x_min, L)
    with Scarf(0) as sc:
        sc.set_basis(b)
        sc.set_transitions(T)
        I = sc.separable_integral(qx, wx, qy, wy, qz, wz)
        scale = np.einsum("sxyz,x,y,z->s", np.abs(f_ref), wx, wy, wz)
        assert np.all(np.abs(I - I_ref) <= 1e-12 * scale)
        assert_parity(sc.fft_form_factors(n, x_min, L, device_out=False), ff_ref)

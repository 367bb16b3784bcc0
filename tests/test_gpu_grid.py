"""GPU parity of the product-grid path (scarf_form_factors_grid; Eq. (45)-(46), (48)
PAPER.md:309-330) against the CPU oracle evaluated on the expanded point list, at the north-star tolerance
1e-10 * max|f_s|, and against the general kernel (same stream, different factor route)."""
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


def expand(qx, qy, qz):
    X, Y, Z = np.meshgrid(qx, qy, qz, indexing="ij")
    return np.ascontiguousarray(np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1))


def assert_parity(f_gpu, f_ref, tol=TOL):
    assert f_gpu.shape == f_ref.shape
    for s in range(f_ref.shape[0]):
        scale = np.max(np.abs(f_ref[s]))
        err = np.max(np.abs(f_gpu[s] - f_ref[s]))
        assert err <= tol * scale, f"state {s}: max err {err:.3e} > {tol:g} * {scale:.3e}"


def grid_ff(Scarf, torch, basis, T, qx, qy, qz, device_axes=True):
    with Scarf(0) as sc:
        sc.set_basis(basis)
        sc.set_transitions(torch.as_tensor(T, dtype=torch.float64, device="cuda").contiguous())
        if device_axes:
            ax = [torch.as_tensor(a, dtype=torch.float64, device="cuda").contiguous() for a in (qx, qy, qz)]
            f = sc.form_factors_grid(*ax)
            torch.cuda.synchronize()
            return f.cpu().numpy(), sc.stats()
        f = sc.form_factors_grid(np.asarray(qx), np.asarray(qy), np.asarray(qz))
        return np.array(f), sc.stats()


def test_grid_config1_full(oracle_mod, Scarf, torch_cuda):
    w = W.make_workload(1, oracle_mod.overlap)
    ax = W.cartesian_axis(w.grid["n_per_axis"], w.grid["qmax"])
    f, st = grid_ff(Scarf, torch_cuda, w.basis, w.T, ax, ax, ax)
    assert np.array_equal(expand(ax, ax, ax), w.q)          # same point order as the config's q list
    assert_parity(f, oracle_mod.form_factors(w.basis, w.T, w.q))
    assert st["last_kernel_launches"] >= 2                  # table kernel + grid kernel


@pytest.mark.parametrize("shape", [(1, 1, 1), (1, 7, 3), (5, 1, 9), (4, 8, 8), (5, 9, 9), (13, 17, 11), (2, 3, 40)])
def test_grid_ragged_shapes_nonuniform_axes(oracle_mod, Scarf, torch_cuda, shape):
    """Boxes are 4 x 8 x 8: shapes below, at and above one box, ragged in every axis; unsorted, non-uniform axes."""
    w = W.make_workload(1, oracle_mod.overlap)
    rng = np.random.default_rng(sum(shape))
    qx, qy, qz = (rng.uniform(-5, 5, size=n) for n in shape)
    f, _ = grid_ff(Scarf, torch_cuda, w.basis, w.T, qx, qy, qz)
    assert_parity(f, oracle_mod.form_factors(w.basis, w.T, expand(qx, qy, qz)))


def test_grid_high_l_12_states_host_axes(oracle_mod, Scarf, torch_cuda):
    """All pair classes L = 0..6 (s, p, d, f shells on two centres), 12 states, host pointers for axes and out."""
    b = W.Basis(np.array([[0.1, 0.2, -0.9], [0.3, -0.4, 1.0]]), np.array([0, 0, 0, 0, 1, 1, 1, 1], np.int32),
                np.array([0, 1, 2, 3, 0, 1, 2, 3], np.int32), np.array([2, 1, 1, 1, 2, 1, 1, 1], np.int32),
                np.array([2.1, 0.4, 1.3, 0.9, 0.7, 1.9, 0.5, 1.1, 0.8, 0.6]),
                np.array([0.5, 0.6, 1.0, 1.0, 1.0, 0.7, 0.4, 1.0, 1.0, 1.0]))
    rng = np.random.default_rng(11)
    T = rng.normal(size=(12, b.nbf, b.nbf))
    qx, qy, qz = np.linspace(-6, 6, 9), np.linspace(-5, 5.5, 10), np.linspace(-4, 6, 11)
    f, st = grid_ff(Scarf, torch_cuda, b, T, qx, qy, qz, device_axes=False)
    assert sum(1 for n in st["pairs_kept_per_class"] if n > 0) == 7
    assert_parity(f, oracle_mod.form_factors(b, T, expand(qx, qy, qz)))


@pytest.mark.parametrize("n_states", [1, 3, 13])
def test_grid_state_tiles(oracle_mod, Scarf, torch_cuda, n_states):
    w = W.make_workload(1, oracle_mod.overlap)
    rng = np.random.default_rng(n_states)
    T = rng.normal(size=(n_states, w.basis.nbf, w.basis.nbf))
    ax = np.linspace(-3, 3, 10)
    f, _ = grid_ff(Scarf, torch_cuda, w.basis, T, ax, ax[:7], ax[:9])
    assert_parity(f, oracle_mod.form_factors(w.basis, T, expand(ax, ax[:7], ax[:9])))


@pytest.mark.parametrize("config,n_sample", [(2, 200), (3, 160), (4, 40)])
def test_grid_full_size_sampled(oracle_mod, Scarf, torch_cuda, config, n_sample):
    """Configs 2-4 are Cartesian product grids: full size on the GPU in the launch configuration bench.py times,
    compared with the oracle on a seeded sample of points, and with the general kernel on every point."""
    torch = torch_cuda
    w = W.make_workload(config, oracle_mod.overlap)
    ax = W.cartesian_axis(w.grid["n_per_axis"], w.grid["qmax"])
    idx = W.sample_q_indices(w.n_q, n_sample, seed=config)
    f_ref = oracle_mod.form_factors(w.basis, w.T, w.q[idx])
    with Scarf(0) as sc:
        sc.set_basis(w.basis)
        sc.set_transitions(torch.as_tensor(w.T, device="cuda"))
        axd = torch.as_tensor(ax, device="cuda")
        fg = sc.form_factors_grid(axd, axd, axd)
        fl = sc.form_factors(torch.as_tensor(w.q, device="cuda"))
        torch.cuda.synchronize()
        assert_parity(fg[:, torch.as_tensor(idx, device="cuda")].cpu().numpy(), f_ref)
        scale = fl.abs().amax(dim=1)
        err = (fg - fl).abs().amax(dim=1)
        assert bool((err <= 1e-11 * scale).all()), (err / scale).max().item()


def test_grid_empty_and_errors(oracle_mod, Scarf, torch_cuda):
    w = W.make_workload(1, oracle_mod.overlap)
    ax = np.linspace(-1, 1, 4)
    with Scarf(0) as sc:
        sc.set_basis(w.basis)
        with pytest.raises(Exception):
            sc.form_factors_grid(ax, ax, ax)                # no transitions yet
        sc.set_transitions(np.zeros_like(w.T))
        f = sc.form_factors_grid(ax, ax, ax)                # T = 0: exactly zero
        assert f.shape == (1, 64) and not np.any(f)
        sc.set_transitions(w.T)
        assert sc.form_factors_grid(ax, ax[:0], ax).shape == (1, 0)
        bad = ax.copy()
        bad[1] = np.nan
        with pytest.raises(Exception):
            sc.form_factors_grid(ax, bad, ax)


@pytest.mark.parametrize("n_states", [1, 12, 14])
def test_separable_integral_equals_weighted_grid_sum(oracle_mod, Scarf, torch_cuda, n_states):
    """Eq. (64)-(65) PAPER.md:481-487: I_sep by 1-D moments per pair (linear in nx+ny+nz) against the plain weighted sum
    of the ORACLE's f_s over the product grid; all classes L = 0..6 present."""
    b = W.Basis(np.array([[0.1, 0.2, -0.9], [0.3, -0.4, 1.0]]), np.array([0, 0, 0, 0, 1, 1, 1, 1], np.int32),
                np.array([0, 1, 2, 3, 0, 1, 2, 3], np.int32), np.array([2, 1, 1, 1, 2, 1, 1, 1], np.int32),
                np.array([2.1, 0.4, 1.3, 0.9, 0.7, 1.9, 0.5, 1.1, 0.8, 0.6]),
                np.array([0.5, 0.6, 1.0, 1.0, 1.0, 0.7, 0.4, 1.0, 1.0, 1.0]))
    rng = np.random.default_rng(40 + n_states)
    T = rng.normal(size=(n_states, b.nbf, b.nbf))
    qx, qy, qz = np.linspace(-4, 4, 9), rng.uniform(-3, 3, 7), np.linspace(-5, 2, 11)
    fx, gy, hz = rng.normal(size=9), np.exp(-qy ** 2), rng.uniform(0.1, 1, 11)
    f = oracle_mod.form_factors(b, T, expand(qx, qy, qz)).reshape(n_states, 9, 7, 11)
    ref = np.einsum("sxyz,x,y,z->s", f, fx, gy, hz)
    with Scarf(0) as sc:
        sc.set_basis(b)
        sc.set_transitions(T)
        got = sc.separable_integral(qx, fx, qy, gy, qz, hz)
        assert np.array_equal(got, sc.separable_integral(qx, fx, qy, gy, qz, hz))      # deterministic
    scale = np.einsum("sxyz,x,y,z->s", np.abs(f), np.abs(fx), np.abs(gy), np.abs(hz))
    assert np.all(np.abs(got - ref) <= 1e-12 * scale), np.max(np.abs(got - ref) / scale)


def test_separable_integral_full_size_config3(oracle_mod, Scarf, torch_cuda):
    """Config 3 at full size (64^3, 9141 pairs, 12 states): the moment route against the weighted sum of the grid path's
    own output (itself parity-checked against the oracle above) — a property that holds at any size."""
    torch = torch_cuda
    w = W.make_workload(3, oracle_mod.overlap)
    ax = W.cartesian_axis(w.grid["n_per_axis"], w.grid["qmax"])
    wt = np.full_like(ax, ax[1] - ax[0])
    fx, gy, hz = wt * np.exp(-0.05 * ax ** 2), wt * np.cos(0.3 * ax), wt / (1.0 + ax ** 2)
    with Scarf(0) as sc:
        sc.set_basis(w.basis)
        sc.set_transitions(torch.as_tensor(w.T, device="cuda"))
        axd = torch.as_tensor(ax, device="cuda")
        f = sc.form_factors_grid(axd, axd, axd).view(w.n_states, 64, 64, 64)
        W3 = torch.as_tensor(np.einsum("x,y,z->xyz", fx, gy, hz), device="cuda")
        ref = (f * W3).sum(dim=(1, 2, 3)).cpu().numpy()
        scale = (f.abs() * W3.abs()).sum(dim=(1, 2, 3)).cpu().numpy()
        got = sc.separable_integral(ax, fx, ax, gy, ax, hz)
    assert np.all(np.abs(got - ref) <= 1e-11 * scale), np.max(np.abs(got - ref) / scale)


def _all_class_basis():
    return W.Basis(np.array([[0.1, 0.2, -0.9], [0.3, -0.4, 1.0]]), np.array([0, 0, 0, 0, 1, 1, 1, 1], np.int32),
                   np.array([0, 1, 2, 3, 0, 1, 2, 3], np.int32), np.array([2, 1, 1, 1, 2, 1, 1, 1], np.int32),
                   np.array([2.1, 0.4, 1.3, 0.9, 0.7, 1.9, 0.5, 1.1, 0.8, 0.6]),
                   np.array([0.5, 0.6, 1.0, 1.0, 1.0, 0.7, 0.4, 1.0, 1.0, 1.0]))


@pytest.mark.parametrize("shape", [(8, 8, 8), (9, 7, 11), (2, 2, 2), (3, 1, 1), (10, 16, 9), (13, 5, 6)])
@pytest.mark.parametrize("device_axes", [True, False])
def test_grid_inversion_symmetry_matches_oracle_on_both_halves(oracle_mod, Scarf, torch_cuda, shape, device_axes):
    """f_s(-q) = conj f_s(q) (reading #6, Eq. (19)): on an exactly inversion-symmetric product grid only the
    half ix < ceil(nx/2) is evaluated and the mirror point gets the conjugate.  Even, odd (centre plane its own mirror) and
    ragged sizes, all classes L = 0..6, 12 states; every point of BOTH halves against the oracle."""
    torch = torch_cuda
    b = _all_class_basis()
    rng = np.random.default_rng(sum(shape))
    T = rng.normal(size=(12, b.nbf, b.nbf))
    axes = [W.cartesian_axis(n, 3.0 + k) if n > 1 else np.zeros(1) for k, n in enumerate(shape)]
    f_ref = oracle_mod.form_factors(b, T, expand(*axes))
    f, st = grid_ff(Scarf, torch, b, T, *axes, device_axes=device_axes)
    assert st["last_grid_symmetric"] == 1
    assert_parity(f, f_ref)
    assert np.array_equal(f[:, ::-1], np.conj(f))                       # exact mirror relation of the stored values
    with Scarf(0) as sc:                                                # the plain path gives the same values to round-off
        sc.set_basis(b)
        sc.set_transitions(T)
        sc.set_option("grid_symmetry", 0)
        f0 = sc.form_factors_grid(*axes)
        assert sc.stats()["last_grid_symmetric"] == 0
    assert np.max(np.abs(f0 - f)) <= 1e-13 * np.max(np.abs(f_ref))
    assert_parity(f0, f_ref)


def test_grid_not_symmetric_falls_back(oracle_mod, Scarf, torch_cuda):
    """One axis off by one ulp, one axis shifted, numpy's plain linspace (not bitwise antisymmetric): the plain path runs."""
    b = _all_class_basis()
    rng = np.random.default_rng(5)
    T = rng.normal(size=(3, b.nbf, b.nbf))
    sym = W.cartesian_axis(8, 4.0)
    ulp = sym.copy()
    ulp[1] = np.nextafter(ulp[1], 10.0)
    for axes in ((sym, sym, ulp), (sym + 0.25, sym, sym), (sym, np.linspace(-10, 10, 64)[:8], sym)):
        f, st = grid_ff(Scarf, torch_cuda, b, T, *axes)
        assert st["last_grid_symmetric"] == 0
        assert_parity(f, oracle_mod.form_factors(b, T, expand(*axes)))


@pytest.mark.parametrize("K", [1, 2, 3, 7, 32])
def test_chunk_counts_general_and_grid(oracle_mod, Scarf, torch_cuda, K):
    """Option n_chunks: the pair stream cut into K cost-balanced slices whose partial sums are added by the thread-block
    cluster in chunk order; every class, more chunks than some classes have records, both S4 kernels, against the oracle."""
    torch = torch_cuda
    b = _all_class_basis()
    rng = np.random.default_rng(40 + K)
    T = rng.normal(size=(5, b.nbf, b.nbf))
    q = rng.uniform(-5, 5, size=(700, 3))
    axes = [np.linspace(-4, 4, 9), np.linspace(-3, 5, 10), np.linspace(-5, 3, 7)]
    f_ref = oracle_mod.form_factors(b, T, q)
    g_ref = oracle_mod.form_factors(b, T, expand(*axes))
    with Scarf(0) as sc:
        sc.set_basis(b)
        sc.set_option("n_chunks", K)
        sc.set_transitions(torch.as_tensor(T, device="cuda"))
        f = sc.form_factors(torch.as_tensor(q, device="cuda"))
        g = sc.form_factors_grid(*[torch.as_tensor(a, device="cuda") for a in axes])
        torch.cuda.synchronize()
        assert_parity(f.cpu().numpy(), f_ref)
        assert_parity(g.cpu().numpy(), g_ref)
        sc.set_transitions(np.zeros_like(T))                            # no record survives: zeros through the same launches
        assert np.all(sc.form_factors(q) == 0) and np.all(sc.form_factors_grid(*axes) == 0)


@pytest.mark.parametrize("shape,symmetric", [((40, 41, 40), True), ((41, 40, 40), True), ((43, 39, 40), False)])
def test_grid_host_output_in_slabs_matches_device_output(oracle_mod, Scarf, torch_cuda, shape, symmetric):
    """Host `out` with >= 65 536 points is computed in four x slabs whose downloads (the slab and, on a symmetric grid, its
    mirror slab) overlap the next slab's kernel: bit-identical to the device-output call (same chunking per box is not
    guaranteed, so: equal to round-off), every point; oracle on a sample; even and odd nx, plain grid."""
    torch = torch_cuda
    w = W.make_workload(1, oracle_mod.overlap)
    rng = np.random.default_rng(sum(shape))
    T = rng.normal(size=(3, w.basis.nbf, w.basis.nbf))
    axes = [W.cartesian_axis(n, 3.0 + 0.5 * k) for k, n in enumerate(shape)]
    if not symmetric:
        axes[0] = axes[0] + 0.125
    with Scarf(0) as sc:
        sc.set_basis(w.basis)
        sc.set_transitions(T)
        f_host = sc.form_factors_grid(*axes)                                        # numpy in -> host out, slabs
        assert sc.stats()["last_grid_symmetric"] == int(symmetric)
        f_dev = sc.form_factors_grid(*[torch.as_tensor(a, device="cuda") for a in axes]).cpu().numpy()
    scale = np.max(np.abs(f_dev), axis=1, keepdims=True)
    assert np.max(np.abs(f_host - f_dev) / scale) <= 1e-13
    q = expand(*axes)
    idx = W.sample_q_indices(q.shape[0], 200, seed=5)
    assert_parity(f_host[:, idx], oracle_mod.form_factors(w.basis, T, q[idx]))

"""GPU parity of the row kernel of the product-grid path (csrc/ff_row.cu, option grid_variant = 1; SURVEY.md §8(f) NEXT-1;
Eq. (45)-(46), (48) PAPER.md:309-330): a warp owns 64 z-points of one (ix, iy) row and evaluates the (q_x, q_y) part of every
polynomial once per (record, state).  Against the CPU oracle on the expanded point list at 1e-10 * max|f_s|, and against the
box kernel (grid_variant = 0)."""
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


def all_class_basis():
    """s, p, d, f shells on two centres (a contracted s on each): every pair class L = 0..6 is populated."""
    return W.Basis(np.array([[0.1, 0.2, -0.9], [0.3, -0.4, 1.0]]), np.array([0, 0, 0, 0, 1, 1, 1, 1], np.int32),
                   np.array([0, 1, 2, 3, 0, 1, 2, 3], np.int32), np.array([2, 1, 1, 1, 2, 1, 1, 1], np.int32),
                   np.array([2.1, 0.4, 1.3, 0.9, 0.7, 1.9, 0.5, 1.1, 0.8, 0.6]),
                   np.array([0.5, 0.6, 1.0, 1.0, 1.0, 0.7, 0.4, 1.0, 1.0, 1.0]))


def grid_ff(Scarf, torch, basis, T, axes, variant, device=True, **options):
    with Scarf(0) as sc:
        sc.set_basis(basis)
        sc.set_option("grid_variant", variant)
        for k, v in options.items():
            sc.set_option(k, v)
        sc.set_transitions(torch.as_tensor(T, dtype=torch.float64, device="cuda").contiguous())
        if device:
            f = sc.form_factors_grid(*[torch.as_tensor(a, dtype=torch.float64, device="cuda").contiguous() for a in axes])
            torch.cuda.synchronize()
            return f.cpu().numpy(), sc.stats()
        f = sc.form_factors_grid(*[np.asarray(a) for a in axes])
        return np.array(f), sc.stats()


@pytest.mark.parametrize("shape", [(1, 1, 1), (3, 5, 64), (2, 4, 70), (5, 9, 33), (2, 3, 130), (3, 1, 7)])
@pytest.mark.parametrize("n_states", [12, 13])
def test_row_kernel_ragged_shapes_all_classes(oracle_mod, Scarf, torch_cuda, shape, n_states):
    """Rows of 64 z-points, 4 rows per CTA: shapes below, at and above one box, ragged in y and z, unsorted non-uniform axes;
    all classes L = 0..6 (pre-pass classes 1..3, degree blocks 4..6); one and two state tiles (12 + 1)."""
    b = all_class_basis()
    rng = np.random.default_rng(sum(shape) + n_states)
    T = rng.normal(size=(n_states, b.nbf, b.nbf))
    axes = [rng.uniform(-5, 5, size=n) for n in shape]
    f, st = grid_ff(Scarf, torch_cuda, b, T, axes, 1)
    assert st["last_grid_variant"] == 1 and st["last_grid_symmetric"] == 0
    assert sum(1 for n in st["pairs_kept_per_class"] if n > 0) == 7
    assert_parity(f, oracle_mod.form_factors(b, T, expand(*axes)))


@pytest.mark.parametrize("n_states", [1, 2, 3, 5, 7])
def test_row_kernel_state_tile_sizes(oracle_mod, Scarf, torch_cuda, n_states):
    """Every instantiated state-tile size (1, 2, 4, 6, 8 padded) through the pre-pass and the accumulate."""
    b = all_class_basis()
    rng = np.random.default_rng(70 + n_states)
    T = rng.normal(size=(n_states, b.nbf, b.nbf))
    axes = [np.linspace(-3, 4, 3), np.linspace(-4, 3, 6), np.linspace(-5, 5, 40)]
    f, st = grid_ff(Scarf, torch_cuda, b, T, axes, 1)
    assert st["last_grid_variant"] == 1
    assert_parity(f, oracle_mod.form_factors(b, T, expand(*axes)))


@pytest.mark.parametrize("shape", [(6, 8, 64), (7, 6, 66), (2, 2, 2), (5, 4, 33)])
@pytest.mark.parametrize("device", [True, False])
def test_row_kernel_inversion_symmetry_both_halves(oracle_mod, Scarf, torch_cuda, shape, device):
    """f_s(-q) = conj f_s(q) (reading #6, Eq. (19)) in the row kernel: half the x planes evaluated, the mirror
    point stored as the conjugate; even and odd nx; every point of both halves against the oracle; exact mirror relation."""
    b = all_class_basis()
    rng = np.random.default_rng(sum(shape))
    T = rng.normal(size=(12, b.nbf, b.nbf))
    axes = [W.cartesian_axis(n, 3.0 + k) for k, n in enumerate(shape)]
    f_ref = oracle_mod.form_factors(b, T, expand(*axes))
    f, st = grid_ff(Scarf, torch_cuda, b, T, axes, 1, device=device)
    assert st["last_grid_variant"] == 1 and st["last_grid_symmetric"] == 1
    assert_parity(f, f_ref)
    assert np.array_equal(f[:, ::-1], np.conj(f))
    f0, st0 = grid_ff(Scarf, torch_cuda, b, T, axes, 0, device=device)        # the box kernel: same values to round-off
    assert st0["last_grid_variant"] == 0
    assert np.max(np.abs(f0 - f)) <= 1e-13 * np.max(np.abs(f_ref))


@pytest.mark.parametrize("K", [1, 2, 7, 32])
def test_row_kernel_chunk_counts(oracle_mod, Scarf, torch_cuda, K):
    """Option n_chunks with the row kernel: the chunks of a box add into `out` in chunk order through the box's ticket; more
    chunks than some classes have records; T = 0 gives exact zeros through the same launches."""
    b = all_class_basis()
    rng = np.random.default_rng(90 + K)
    T = rng.normal(size=(5, b.nbf, b.nbf))
    axes = [np.linspace(-4, 4, 3), np.linspace(-3, 5, 10), np.linspace(-5, 3, 67)]
    f, st = grid_ff(Scarf, torch_cuda, b, T, axes, 1, n_chunks=K)
    assert st["last_grid_variant"] == 1 and st["last_n_chunks"] == K
    assert_parity(f, oracle_mod.form_factors(b, T, expand(*axes)))
    z, _ = grid_ff(Scarf, torch_cuda, b, np.zeros_like(T), axes, 1, n_chunks=K)
    assert not np.any(z)


def test_row_kernel_automatic_choice(oracle_mod, Scarf, torch_cuda):
    """grid_variant = -1 (default): the row kernel runs when its 4 x 64 boxes are at least 80 % full, the box kernel otherwise;
    either way the oracle's values."""
    w = W.make_workload(1, oracle_mod.overlap)
    for shape, expect in (((3, 8, 64), 1), ((3, 8, 56), 1), ((4, 8, 48), 0), ((4, 5, 64), 0), ((2, 7, 128), 1)):
        rng = np.random.default_rng(sum(shape))
        axes = [rng.uniform(-4, 4, size=n) for n in shape]
        f, st = grid_ff(Scarf, torch_cuda, w.basis, w.T, axes, -1)
        assert st["last_grid_variant"] == expect, shape
        assert_parity(f, oracle_mod.form_factors(w.basis, w.T, expand(*axes)))


@pytest.mark.parametrize("config,n_sample", [(3, 160), (4, 40)])
def test_row_kernel_full_size_sampled(oracle_mod, Scarf, torch_cuda, config, n_sample):
    """Configs 3 and 4 (64^3, inversion-symmetric) at full size with the row kernel (grid_variant = 1; the automatic choice on these
    grids is the mirror-pair kernel, tests/test_gpu_grid_zrow.py) against the oracle on a seeded sample of points from both halves,
    and against the list kernel on every point."""
    torch = torch_cuda
    w = W.make_workload(config, oracle_mod.overlap)
    ax = W.cartesian_axis(w.grid["n_per_axis"], w.grid["qmax"])
    idx = W.sample_q_indices(w.n_q, n_sample, seed=config)
    f_ref = oracle_mod.form_factors(w.basis, w.T, w.q[idx])
    with Scarf(0) as sc:
        sc.set_basis(w.basis)
        sc.set_option("grid_variant", 1)
        sc.set_transitions(torch.as_tensor(w.T, device="cuda"))
        axd = torch.as_tensor(ax, device="cuda")
        fg = sc.form_factors_grid(axd, axd, axd)
        st = sc.stats()
        assert st["last_grid_variant"] == 1 and st["last_grid_symmetric"] == 1
        fl = sc.form_factors(torch.as_tensor(w.q, device="cuda"))
        torch.cuda.synchronize()
        assert_parity(fg[:, torch.as_tensor(idx, device="cuda")].cpu().numpy(), f_ref)
        scale = fl.abs().amax(dim=1)
        err = (fg - fl).abs().amax(dim=1)
        assert bool((err <= 1e-11 * scale).all()), (err / scale).max().item()


def test_row_kernel_q_adaptive_bound(oracle_mod, Scarf, torch_cuda):
    """Option adaptive_tol with the row kernel: the box keeps a prefix of every class; error against the exact path on every
    point below the reported bound."""
    torch = torch_cuda
    w = W.make_workload(2, oracle_mod.overlap)
    ax = W.cartesian_axis(64, w.grid["qmax"])
    axes = [ax[:6], ax[:8], ax]
    exact, _ = grid_ff(Scarf, torch, w.basis, w.T, axes, 1)
    for tol in (1e-12, 1e-6):
        f, st = grid_ff(Scarf, torch, w.basis, w.T, axes, 1, adaptive_tol=tol)
        assert st["last_grid_variant"] == 1 and st["adaptive_bound"] > 0
        assert np.max(np.abs(f - exact)) <= st["adaptive_bound"] + 1e-12 * np.max(np.abs(exact))
        assert st["last_adaptive_work_fraction"] <= 1.0


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("shape,symmetric", [((6, 8, 64), True), ((5, 7, 70), False)])
def test_pinned_host_output_written_by_the_kernel(oracle_mod, Scarf, torch_cuda, variant, shape, symmetric):
    """Option host_zero_copy (default on): a PINNED host `out` receives the finished values from the last chunk of every box through
    its mapped alias (no device->host copy); several chunks so that partial sums go through the device scratch.  Bit-identical to
    the device-output call and to the copy path (host_zero_copy = 0, and a pageable numpy `out`); oracle on every point."""
    torch = torch_cuda
    b = all_class_basis()
    rng = np.random.default_rng(sum(shape) + variant)
    T = rng.normal(size=(13, b.nbf, b.nbf))
    axes = [W.cartesian_axis(n, 3.0 + k) for k, n in enumerate(shape)] if symmetric else [rng.uniform(-4, 4, size=n) for n in shape]
    n_q = int(np.prod(shape))
    f_ref = oracle_mod.form_factors(b, T, expand(*axes))
    with Scarf(0) as sc:
        sc.set_basis(b)
        sc.set_option("grid_variant", variant)
        sc.set_option("n_chunks", 5)
        sc.set_transitions(torch.as_tensor(T, device="cuda"))
        f_dev = sc.form_factors_grid(*[torch.as_tensor(a, device="cuda") for a in axes])
        torch.cuda.synchronize()
        f_dev = f_dev.cpu().numpy()
        assert sc.stats()["last_grid_symmetric"] == int(symmetric)
        pinned = torch.full((13, n_q, 2), float("nan"), dtype=torch.float64).pin_memory()
        f_pin = sc.form_factors_grid(*axes, out=pinned).numpy().copy()
        sc.set_option("host_zero_copy", 0)
        pinned2 = torch.full((13, n_q, 2), float("nan"), dtype=torch.float64).pin_memory()
        f_copy = sc.form_factors_grid(*axes, out=pinned2).numpy().copy()
        f_np = np.array(sc.form_factors_grid(*axes))
    assert_parity(f_pin, f_ref)
    assert np.array_equal(f_pin, f_dev) and np.array_equal(f_copy, f_dev) and np.array_equal(f_np, f_dev)


@pytest.mark.parametrize("tile_group", [1, 3, 1000])
def test_pinned_host_output_tile_groups(oracle_mod, Scarf, torch_cuda, tile_group):
    """Option host_tile_group: with a pinned host `out` the CTAs are dispatched chunk-major inside groups of tiles; a group of one
    tile, a ragged last group, one group for everything: same values as the device-output call, bit for bit."""
    torch = torch_cuda
    b = all_class_basis()
    rng = np.random.default_rng(tile_group)
    T = rng.normal(size=(12, b.nbf, b.nbf))
    axes = [W.cartesian_axis(n, 3.0 + k) for k, n in enumerate((4, 14, 70))]          # 2 x 4 x 2 = 16 boxes of 1 x 4 x 64 (x halved)
    n_q = 4 * 14 * 70
    with Scarf(0) as sc:
        sc.set_basis(b)
        sc.set_option("grid_variant", 1)
        sc.set_option("n_chunks", 4)
        sc.set_option("host_tile_group", tile_group)
        sc.set_transitions(torch.as_tensor(T, device="cuda"))
        f_dev = sc.form_factors_grid(*[torch.as_tensor(a, device="cuda") for a in axes])
        torch.cuda.synchronize()
        pinned = torch.full((12, n_q, 2), float("nan"), dtype=torch.float64).pin_memory()
        f_pin = sc.form_factors_grid(*axes, out=pinned).numpy().copy()
    assert np.array_equal(f_pin, f_dev.cpu().numpy())
    assert_parity(f_pin, oracle_mod.form_factors(b, T, expand(*axes)))

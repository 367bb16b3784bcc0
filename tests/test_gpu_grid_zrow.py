"""GPU parity of the mirror-pair row kernel of the product-grid path (csrc/ff_zrow.cu, option grid_variant = 2; SURVEY.md §8(f)
NEXT-1; Eq. (45)-(46), (48) PAPER.md:309-330): on a grid whose z axis is antisymmetric bit for bit a lane owns the points +z and -z
of its (ix, iy) row and accumulates their half sum and half difference.  Against the CPU oracle on the expanded point list at
1e-10 * max|f_s|, and against the row kernel (grid_variant = 1)."""
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


def antisym_axis(n, rng, qmax=5.0):
    """n points with ax[i] == -ax[n-1-i] bit for bit, non-uniform (the middle point of an odd axis is exactly 0)."""
    h = np.sort(rng.uniform(0.05, qmax, size=n // 2))
    mid = [0.0] if n % 2 else []
    return np.concatenate([-h[::-1], mid, h])


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


@pytest.mark.parametrize("shape", [(1, 1, 2), (3, 5, 64), (2, 4, 70), (5, 9, 33), (2, 3, 130), (3, 1, 7)])
@pytest.mark.parametrize("n_states", [12, 13])
def test_zrow_kernel_ragged_shapes_all_classes(oracle_mod, Scarf, torch_cuda, shape, n_states):
    """Rows of 32 mirror pairs, 4 rows per CTA: even and odd nz (the middle point is its own partner), below, at and above one box,
    ragged in y; arbitrary x and y axes (no inversion symmetry of the grid), non-uniform antisymmetric z; all classes L = 0..6
    ((S', D') accumulation for 0..3, conversion, degree blocks for 4..6); one and two state tiles."""
    b = all_class_basis()
    rng = np.random.default_rng(sum(shape) + n_states)
    T = rng.normal(size=(n_states, b.nbf, b.nbf))
    axes = [rng.uniform(-5, 5, size=shape[0]), rng.uniform(-5, 5, size=shape[1]), antisym_axis(shape[2], rng)]
    f, st = grid_ff(Scarf, torch_cuda, b, T, axes, 2)
    assert st["last_grid_variant"] == 2 and st["last_grid_symmetric"] == 0
    assert sum(1 for n in st["pairs_kept_per_class"] if n > 0) == 7
    assert_parity(f, oracle_mod.form_factors(b, T, expand(*axes)))


@pytest.mark.parametrize("n_states", [1, 2, 3, 5, 7])
def test_zrow_kernel_state_tile_sizes(oracle_mod, Scarf, torch_cuda, n_states):
    b = all_class_basis()
    rng = np.random.default_rng(270 + n_states)
    T = rng.normal(size=(n_states, b.nbf, b.nbf))
    axes = [np.linspace(-3, 4, 3), np.linspace(-4, 3, 6), antisym_axis(40, rng)]
    f, st = grid_ff(Scarf, torch_cuda, b, T, axes, 2)
    assert st["last_grid_variant"] == 2
    assert_parity(f, oracle_mod.form_factors(b, T, expand(*axes)))


@pytest.mark.parametrize("shape", [(6, 8, 64), (7, 6, 66), (2, 2, 2), (5, 4, 33)])
@pytest.mark.parametrize("device", [True, False])
def test_zrow_kernel_with_inversion_symmetry(oracle_mod, Scarf, torch_cuda, shape, device):
    """All three axes antisymmetric: half of the x planes evaluated by the mirror-pair kernel, f(-q) = conj f(q) stored for the
    other half; every point against the oracle, exact mirror relation, the row kernel agrees to round-off."""
    b = all_class_basis()
    rng = np.random.default_rng(sum(shape))
    T = rng.normal(size=(12, b.nbf, b.nbf))
    axes = [W.cartesian_axis(n, 3.0 + k) for k, n in enumerate(shape)]
    f_ref = oracle_mod.form_factors(b, T, expand(*axes))
    f, st = grid_ff(Scarf, torch_cuda, b, T, axes, 2, device=device)
    assert st["last_grid_variant"] == 2 and st["last_grid_symmetric"] == 1
    assert_parity(f, f_ref)
    assert np.array_equal(f[:, ::-1], np.conj(f))
    f1, st1 = grid_ff(Scarf, torch_cuda, b, T, axes, 1, device=device)
    assert st1["last_grid_variant"] == 1
    assert np.max(np.abs(f1 - f)) <= 1e-13 * np.max(np.abs(f_ref))


@pytest.mark.parametrize("K", [1, 2, 7, 32])
def test_zrow_kernel_chunk_counts_and_pinned_output(oracle_mod, Scarf, torch_cuda, K):
    torch = torch_cuda
    b = all_class_basis()
    rng = np.random.default_rng(290 + K)
    T = rng.normal(size=(5, b.nbf, b.nbf))
    axes = [np.linspace(-4, 4, 3), np.linspace(-3, 5, 10), antisym_axis(67, rng)]
    f, st = grid_ff(Scarf, torch_cuda, b, T, axes, 2, n_chunks=K)
    assert st["last_grid_variant"] == 2 and st["last_n_chunks"] == K
    assert_parity(f, oracle_mod.form_factors(b, T, expand(*axes)))
    z, _ = grid_ff(Scarf, torch_cuda, b, np.zeros_like(T), axes, 2, n_chunks=K)
    assert not np.any(z)
    with Scarf(0) as sc:                                                 # pinned host out: written by the last chunks, bit-identical
        sc.set_basis(b)
        sc.set_option("grid_variant", 2)
        sc.set_option("n_chunks", K)
        sc.set_option("host_tile_group", 3)
        sc.set_transitions(T)
        pinned = torch.full((5, 3 * 10 * 67, 2), float("nan"), dtype=torch.float64).pin_memory()
        assert np.array_equal(sc.form_factors_grid(*axes, out=pinned).numpy(), f)


@pytest.mark.parametrize("n_states,K", [(4, 1), (8, 3), (12, 1), (12, 5), (24, 2)])
def test_zrow_tensor_core_classes_full_stages(oracle_mod, Scarf, torch_cuda, n_states, K):
    """Classes 0, 1 and 2 on the FP64 tensor cores (state tiles of 4, 8, 12 states: whole N tiles of mma.sync.m8n8k4.f64): config 2's
    basis has thousands of records per class, so the stages are full (24 / 24 / 12 records), the last one of a segment is short (the
    zero rows of a missing record) and with K > 1 the chunks start and end inside a class.  Against the oracle on every point, and
    against the row kernel (DFMA loops, grid_variant = 1) at 1e-12."""
    w = W.make_workload(2, oracle_mod.overlap)
    rng = np.random.default_rng(40 + n_states + K)
    T = rng.normal(size=(n_states, w.basis.nbf, w.basis.nbf)) / w.basis.nbf
    axes = [rng.uniform(-6, 6, size=2), rng.uniform(-6, 6, size=5), antisym_axis(66, rng, qmax=7.0)]
    f, st = grid_ff(Scarf, torch_cuda, w.basis, T, axes, 2, n_chunks=K)
    assert st["last_grid_variant"] == 2 and st["last_n_chunks"] == K
    assert st["pairs_kept_per_class"][0] > 1000 and st["pairs_kept_per_class"][1] > 1000 and st["pairs_kept_per_class"][2] > 500
    f_row, st_row = grid_ff(Scarf, torch_cuda, w.basis, T, axes, 1, n_chunks=K)
    assert st_row["last_grid_variant"] == 1
    assert_parity(f, f_row, tol=1e-12)
    assert_parity(f, oracle_mod.form_factors(w.basis, T, expand(*axes)))


def test_zrow_kernel_choice(oracle_mod, Scarf, torch_cuda):
    """grid_variant = 2 on a z axis that is not antisymmetric falls back to the automatic choice; grid_variant = -1 picks the
    mirror-pair kernel when the z axis allows it and the boxes are at least 75 % full; either way the oracle's values."""
    w = W.make_workload(1, oracle_mod.overlap)
    rng = np.random.default_rng(17)
    az = antisym_axis(64, rng)
    off = az.copy()
    off[3] = np.nextafter(off[3], 10.0)
    az48 = antisym_axis(48, rng)                      # 24 mirror pairs = 75 % of a box: three whole M tiles of the tensor-core classes
    for axes, variant, expect in (((az[:3], az[:8], az), -1, 2), ((az[:3], az[:8], az48), -1, 2), ((az[:3], az[:8], off), -1, 1), ((az[:3], az[:8], off), 2, 1),
                                  ((az[:3], az[:8], az[16:48]), -1, 0), ((az[:3], az[:5], az), -1, 0), ((az[:3], az[:8], az), 1, 1)):
        f, st = grid_ff(Scarf, torch_cuda, w.basis, w.T, axes, variant)
        assert st["last_grid_variant"] == expect, (variant, expect)
        assert_parity(f, oracle_mod.form_factors(w.basis, w.T, expand(*axes)))


@pytest.mark.parametrize("config,n_sample", [(3, 160), (4, 40)])
def test_zrow_kernel_full_size_sampled(oracle_mod, Scarf, torch_cuda, config, n_sample):
    """Configs 3 and 4 (64^3, inversion-symmetric) in the launch configuration bench.py times — the mirror-pair kernel is the
    automatic choice there — against the oracle on a seeded sample of points, and against the list kernel on every point."""
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
        st = sc.stats()
        assert st["last_grid_variant"] == 2 and st["last_grid_symmetric"] == 1
        fl = sc.form_factors(torch.as_tensor(w.q, device="cuda"))
        torch.cuda.synchronize()
        assert_parity(fg[:, torch.as_tensor(idx, device="cuda")].cpu().numpy(), f_ref)
        scale = fl.abs().amax(dim=1)
        err = (fg - fl).abs().amax(dim=1)
        assert bool((err <= 1e-11 * scale).all()), (err / scale).max().item()


def test_zrow_kernel_q_adaptive_bound(oracle_mod, Scarf, torch_cuda):
    torch = torch_cuda
    w = W.make_workload(2, oracle_mod.overlap)
    ax = W.cartesian_axis(64, w.grid["qmax"])
    axes = [ax[:6], ax[:8], ax]
    exact, _ = grid_ff(Scarf, torch, w.basis, w.T, axes, 2)
    for tol in (1e-12, 1e-6):
        f, st = grid_ff(Scarf, torch, w.basis, w.T, axes, 2, adaptive_tol=tol)
        assert st["last_grid_variant"] == 2 and st["adaptive_bound"] > 0
        assert np.max(np.abs(f - exact)) <= st["adaptive_bound"] + 1e-12 * np.max(np.abs(exact))
        assert st["last_adaptive_work_fraction"] <= 1.0

"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same seeded
inputs.  Tolerance (BASELINE.json north_star): max_q |f_gpu - f_oracle| <= 1e-10 * max_q |f_oracle| per state.

Inputs are generated with the ORACLE's overlap (no oracle input ever comes from the CUDA path).
Small configs are compared on their full grids; configs 3-5 run on the GPU at full size, in the launch
configuration bench.py times, and are compared on a seeded sample of q-points the oracle evaluates one by one,
plus properties that hold at any size (f(-q) = conj f(q), host/device pointer agreement).
"""
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


def gpu_form_factors(Scarf, torch, basis, T, q, **opts):
    with Scarf(0) as sc:
        for k, v in opts.items():
            sc.set_option(k, v)
        sc.set_basis(basis)
        sc.set_transitions(torch.as_tensor(T, dtype=torch.float64, device="cuda").contiguous())
        qd = torch.as_tensor(q, dtype=torch.float64, device="cuda").contiguous()
        f = sc.form_factors(qd)
        torch.cuda.synchronize()
        return f.cpu().numpy(), sc.stats()


def assert_parity(f_gpu, f_ref, tol=TOL):
    assert f_gpu.shape == f_ref.shape
    for s in range(f_ref.shape[0]):
        scale = np.max(np.abs(f_ref[s]))
        err = np.max(np.abs(f_gpu[s] - f_ref[s]))
        assert err <= tol * scale, f"state {s}: max err {err:.3e} > {tol:g} * {scale:.3e}"


def test_config1_full_grid(oracle_mod, Scarf, torch_cuda):
    w = W.make_workload(1, oracle_mod.overlap)
    f_ref = oracle_mod.form_factors(w.basis, w.T, w.q)
    f_gpu, st = gpu_form_factors(Scarf, torch_cuda, w.basis, w.T, w.q)
    assert_parity(f_gpu, f_ref)
    assert st["n_pairs_all"] == 171 and st["nbf"] == 10


def test_config2_strided_grid(oracle_mod, Scarf, torch_cuda):
    w = W.make_workload(2, oracle_mod.overlap)
    f_gpu, st = gpu_form_factors(Scarf, torch_cuda, w.basis, w.T, w.q)
    idx = W.sample_q_indices(w.n_q, 300, seed=2)
    f_ref = oracle_mod.form_factors(w.basis, w.T, w.q[idx])
    assert_parity(f_gpu[:, idx], f_ref)
    # properties on the full grid: the grid is symmetric under q -> -q (index reversal)
    np.testing.assert_allclose(f_gpu[:, ::-1], np.conj(f_gpu), rtol=0, atol=1e-12 * np.max(np.abs(f_gpu)))


@pytest.mark.parametrize("config,n_sample", [(3, 160), (4, 40), (5, 160)])
def test_full_size_sampled(oracle_mod, Scarf, torch_cuda, config, n_sample):
    w = W.make_workload(config, oracle_mod.overlap)
    f_gpu, st = gpu_form_factors(Scarf, torch_cuda, w.basis, w.T, w.q)
    assert f_gpu.shape == (12, w.n_q)
    idx = W.sample_q_indices(w.n_q, n_sample, seed=config)
    f_ref = oracle_mod.form_factors(w.basis, w.T, w.q[idx])
    assert_parity(f_gpu[:, idx], f_ref)
    assert np.all(np.isfinite(f_gpu.view(np.float64)))
    if w.grid["kind"] == "cartesian":
        np.testing.assert_allclose(f_gpu[:, ::-1], np.conj(f_gpu), rtol=0, atol=1e-12 * np.max(np.abs(f_gpu)))


def test_unscreened_equals_screened(oracle_mod, Scarf, torch_cuda):
    """screen_tol = 0 keeps every pair; the default screen must change nothing at the 1e-10 level."""
    w = W.make_workload(2, oracle_mod.overlap)
    q = w.q[::211]
    f_a, st_a = gpu_form_factors(Scarf, torch_cuda, w.basis, w.T, q, screen_tol=0.0)
    f_b, st_b = gpu_form_factors(Scarf, torch_cuda, w.basis, w.T, q)
    assert st_a["n_pairs_kept"] >= st_b["n_pairs_kept"]
    assert np.max(np.abs(f_a - f_b)) <= 1e-13 * np.max(np.abs(f_a))
    f_ref = oracle_mod.form_factors(w.basis, w.T, q)
    assert_parity(f_a, f_ref)


@pytest.mark.parametrize("n_states", [1, 2, 3, 5, 7, 12, 13, 25])
def test_state_counts_and_tiles(oracle_mod, Scarf, torch_cuda, n_states):
    """State tiles: padded tile sizes and more than one tile of 12."""
    w = W.make_workload(1, oracle_mod.overlap)
    rng = np.random.default_rng(n_states)
    T = rng.normal(size=(n_states, w.basis.nbf, w.basis.nbf))
    q = w.q[::13]
    f_ref = oracle_mod.form_factors(w.basis, T, q)
    f_gpu, _ = gpu_form_factors(Scarf, torch_cuda, w.basis, T, q)
    assert_parity(f_gpu, f_ref)


@pytest.mark.parametrize("n_q", [1, 2, 31, 33, 127, 129, 257, 1000])
def test_ragged_q_counts(oracle_mod, Scarf, torch_cuda, n_q):
    w = W.make_workload(1, oracle_mod.overlap)
    rng = np.random.default_rng(n_q)
    q = rng.uniform(-5, 5, size=(n_q, 3))
    q[0] = 0.0                                  # q = 0 exactly: f = g Tr(T S) = 0
    f_ref = oracle_mod.form_factors(w.basis, w.T, q)
    f_gpu, _ = gpu_form_factors(Scarf, torch_cuda, w.basis, w.T, q)
    scale = max(np.max(np.abs(f_ref)), 1e-3)
    assert np.max(np.abs(f_gpu - f_ref)) <= TOL * scale
    assert abs(f_gpu[0, 0]) < 1e-13


def test_high_l_classes(oracle_mod, Scarf, torch_cuda):
    """d and f shells on two centres: classes L = 0..6 all populated."""
    from tests.test_oracle_pins import mk_basis
    rng = np.random.default_rng(4)
    sh = lambda at: [(at, 0, [2.1, 0.4], [0.5, 0.6]), (at, 1, [1.3, 0.3], [0.7, 0.5]), (at, 2, [0.9], [1.0]), (at, 3, [0.7], [1.0])]
    b = mk_basis([[0.1, 0.2, -0.9], [0.3, -0.4, 1.0]], sh(0) + sh(1))
    T = rng.normal(size=(3, b.nbf, b.nbf))
    q = rng.uniform(-6, 6, size=(200, 3))
    f_ref = oracle_mod.form_factors(b, T, q)
    f_gpu, st = gpu_form_factors(Scarf, torch_cuda, b, T, q)
    assert all(n > 0 for n in st["pairs_kept_per_class"][:7])
    assert_parity(f_gpu, f_ref)


def test_large_q_and_far_atoms(oracle_mod, Scarf, torch_cuda):
    """Large phases q.P (argument reduction of sincos) and strong Gaussian damping (exp underflow)."""
    from tests.test_oracle_pins import mk_basis
    rng = np.random.default_rng(8)
    b = mk_basis([[40.0, -35.0, 20.0], [41.5, -34.0, 21.0]],
                 [(0, 0, [900.0, 3.0], [0.5, 0.6]), (0, 1, [50.0], [1.0]), (1, 0, [0.2], [1.0]), (1, 2, [1.1], [1.0])])
    T = rng.normal(size=(2, b.nbf, b.nbf))
    q = rng.uniform(-60, 60, size=(300, 3))
    f_ref = oracle_mod.form_factors(b, T, q)
    f_gpu, _ = gpu_form_factors(Scarf, torch_cuda, b, T, q)
    assert_parity(f_gpu, f_ref)


def test_host_and_device_pointers_agree(oracle_mod, Scarf, torch_cuda):
    torch = torch_cuda
    w = W.make_workload(1, oracle_mod.overlap)
    q = w.q[::7].copy()
    with Scarf(0) as sc:
        sc.set_basis(w.basis)
        sc.set_transitions(w.T)                                  # host T
        f_host = sc.form_factors(q).copy()                       # host q, host out
        qd = torch.as_tensor(q, device="cuda")
        f_dev = sc.form_factors(qd).cpu().numpy()                # device q, device out
        out_pinned = torch.empty((1, q.shape[0], 2), dtype=torch.float64).pin_memory()
        f_mixed = sc.form_factors(qd, out=out_pinned).numpy().copy()   # device q, pinned host out
    assert np.array_equal(f_host, f_dev) and np.array_equal(f_host, f_mixed)
    assert_parity(f_host, oracle_mod.form_factors(w.basis, w.T, q))


def test_repeated_calls_and_prefactor(oracle_mod, Scarf, torch_cuda):
    w = W.make_workload(2, oracle_mod.overlap)
    q = w.q[::997]
    with Scarf(0) as sc:
        sc.set_basis(w.basis)
        sc.set_transitions(w.T[:4])
        f4 = sc.form_factors(q).copy()
        sc.set_transitions(w.T)                                  # new stack on the same basis
        f12 = sc.form_factors(q).copy()
        f12b = sc.form_factors(q).copy()                         # repeat
        sc.set_option("prefactor", 1.0)
        sc.set_transitions(w.T)
        f12_g1 = sc.form_factors(q).copy()
    assert np.array_equal(f12, f12b)                             # same inputs, same launch: bit-reproducible
    # 4 states vs 12 states: another state tile (other kernel instantiation, other screened pair set), so
    # only agreement to round-off is guaranteed
    assert np.max(np.abs(f12[:4] - f4)) <= 1e-13 * np.max(np.abs(f12))
    np.testing.assert_allclose(f12_g1, 0.5 * f12, rtol=1e-14, atol=0)
    assert_parity(f12, oracle_mod.form_factors(w.basis, w.T, q))


def test_zero_T_and_empty_q(oracle_mod, Scarf, torch_cuda):
    w = W.make_workload(1, oracle_mod.overlap)
    with Scarf(0) as sc:
        sc.set_basis(w.basis)
        sc.set_transitions(np.zeros_like(w.T))
        f = sc.form_factors(w.q[:100])
        assert np.all(f == 0)
        assert sc.form_factors(np.zeros((0, 3))).shape == (1, 0)


def test_error_paths(oracle_mod, Scarf, torch_cuda):
    from paper_2512_18010_b200.binding import ScarfError, SCARF_ESTATE, SCARF_EINVAL
    w = W.make_workload(1, oracle_mod.overlap)
    with Scarf(0) as sc:
        with pytest.raises(ScarfError) as e:
            sc.n_states = 1
            sc.form_factors(w.q[:4])
        assert e.value.code == SCARF_ESTATE
        sc.set_basis(w.basis)
        bad = w.T.copy()
        bad[0, 1, 2] = np.nan
        with pytest.raises(ScarfError) as e:
            sc.set_transitions(bad)
        assert e.value.code == SCARF_EINVAL
        sc.set_transitions(w.T)
        qbad = w.q[:4].copy()
        qbad[2, 1] = np.inf
        with pytest.raises(ScarfError) as e:
            sc.form_factors(qbad)
        assert e.value.code == SCARF_EINVAL


@pytest.mark.parametrize("eps", [1e-10, 1e-6, 1e-3])
def test_threshold_eps_error_within_reported_bound(oracle_mod, Scarf, torch_cuda, eps):
    """NEXT-2 (paper-style thresholding): an approximation whose error must stay below the bound the
    library reports (sum of the dropped pairs' B_P), for every state and q; the exact path is the oracle."""
    torch = torch_cuda
    w = W.make_workload(2, oracle_mod.overlap)
    idx = W.sample_q_indices(w.n_q, 300, seed=7)
    q = w.q[idx]
    f_ref = oracle_mod.form_factors(w.basis, w.T, q)
    f0, st0 = gpu_form_factors(Scarf, torch, w.basis, w.T, q)
    f1, st1 = gpu_form_factors(Scarf, torch, w.basis, w.T, q, threshold_eps=eps)
    assert st1["n_pairs_kept"] < st0["n_pairs_kept"]
    assert st1["dropped_bound"] >= st0["dropped_bound"] >= 0.0
    err = np.max(np.abs(f1 - f_ref))
    assert err <= st1["dropped_bound"] + TOL * np.max(np.abs(f_ref))


def test_pure_shells_mixed_basis(oracle_mod, Scarf, torch_cuda):
    """NEXT-5: pure d/f shells mixed with Cartesian ones (scarf_set_basis_pure): T, nbf and the result in the mixed
    basis; oracle = oracle/pure.py (solid harmonics from scipy's Y_lm, through the pinned Cartesian oracle)."""
    torch = torch_cuda
    from oracle import pure as opure
    from tests.test_oracle_pure import mixed_basis
    b, pure = mixed_basis()
    rng = np.random.default_rng(21)
    nbf = opure.basis_matrix(b, pure).shape[1]
    T = rng.normal(size=(12, nbf, nbf))
    q = rng.uniform(-5, 5, size=(300, 3))
    f_ref = opure.form_factors(b, pure, T, q)
    with Scarf(0) as sc:
        sc.set_basis(b, shell_pure=pure)
        assert sc.nbf == nbf
        sc.set_transitions(torch.as_tensor(T, device="cuda"))
        f = sc.form_factors(torch.as_tensor(q, device="cuda"))
        torch.cuda.synchronize()
        assert_parity(f.cpu().numpy(), f_ref)
        sc.set_transitions(T)                                   # host pointer, same result
        assert np.array_equal(sc.form_factors(q), f.cpu().numpy())
        sc.set_basis(b)                                         # back to all-Cartesian on the same context
        assert sc.nbf == b.nbf


def test_host_output_sliced_download_matches_device_output(oracle_mod, Scarf, torch_cuda):
    """Host `out` with n_q >= 65536 is computed in q slices whose downloads overlap the next slice's kernels: same
    values as the device-output path (different chunking, so equal to round-off, not bitwise) and as the oracle on a sample;
    ragged n_q (not a multiple of the slice or tile size)."""
    torch = torch_cuda
    w = W.make_workload(1, oracle_mod.overlap)
    rng = np.random.default_rng(77)
    T = rng.normal(size=(3, w.basis.nbf, w.basis.nbf))
    q = rng.uniform(-4, 4, size=(70001, 3))
    with Scarf(0) as sc:
        sc.set_basis(w.basis)
        sc.set_transitions(T)
        f_host = sc.form_factors(q)                                       # numpy in -> host out, sliced
        f_dev = sc.form_factors(torch.as_tensor(q, device="cuda")).cpu().numpy()
    scale = np.max(np.abs(f_dev), axis=1, keepdims=True)
    assert np.max(np.abs(f_host - f_dev) / scale) <= 1e-13
    idx = W.sample_q_indices(q.shape[0], 300, seed=3)
    assert_parity(f_host[:, idx], oracle_mod.form_factors(w.basis, T, q[idx]))


def test_device_side_screening_matches_round1_counts(oracle_mod, Scarf, torch_cuda):
    """set_transitions screens and packs on the device (no host round trip); the kept counts per class of config 3 are the
    ones the host-side screening of round 1 produced (BENCH_r01.json), and they arrive lazily through scarf_get_stats."""
    torch = torch_cuda
    w = W.make_workload(3, oracle_mod.overlap, with_q=False)
    with Scarf(0) as sc:
        sc.set_basis(w.basis)
        sc.set_transitions(torch.as_tensor(w.T, device="cuda"))
        st = sc.stats()
    assert st["pairs_kept_per_class"][:7] == [3301, 3444, 1877, 464, 55, 0, 0]
    assert st["n_pairs_kept"] == 9141 and st["n_pairs_all"] == 12880
    assert st["slots_per_q"] == 1180116.0


def test_non_finite_device_T_is_reported(oracle_mod, Scarf, torch_cuda):
    """Device T is validated on the device: the NaN reaches the output (no silent zeros) and the first call that can see the
    screening result without stalling the stream reports SCARF_EINVAL."""
    torch = torch_cuda
    from paper_2512_18010_b200.binding import ScarfError, SCARF_EINVAL
    w = W.make_workload(1, oracle_mod.overlap)
    bad = w.T.copy()
    bad[0, 1, 2] = np.nan
    with Scarf(0) as sc:
        sc.set_basis(w.basis)
        sc.set_transitions(torch.as_tensor(bad, device="cuda"))       # asynchronous: cannot fail here
        with pytest.raises(ScarfError) as e:
            sc.stats()
        assert e.value.code == SCARF_EINVAL
        with pytest.raises(ScarfError) as e:
            sc.form_factors(w.q[:8])
        assert e.value.code == SCARF_EINVAL
        sc.set_transitions(torch.as_tensor(w.T, device="cuda"))       # a good T clears the condition
        assert_parity(sc.form_factors(w.q[:64]), oracle_mod.form_factors(w.basis, w.T, w.q[:64]))


@pytest.mark.parametrize("tol", [1e-16, 1e-9, 1e-4])
def test_q_adaptive_cutoff_error_within_reported_bound(oracle_mod, Scarf, torch_cuda, tol):
    """NEXT-2, second half (PAPER.md:499 made q-dependent): option adaptive_tol skips a pair for the q tiles beyond the radius
    where its rigorous envelope falls below tau.  Config 2 at full size, point list sorted by |q| (so that tiles have large
    smallest |q|) and the product grid: the error against the EXACT path on every point, and against the oracle on a sample,
    stays below the bound the library reports; the work fraction drops as the tolerance grows."""
    torch = torch_cuda
    w = W.make_workload(2, oracle_mod.overlap)
    order = np.argsort(np.linalg.norm(w.q, axis=1), kind="stable")
    q = np.ascontiguousarray(w.q[order])
    ax = W.cartesian_axis(w.grid["n_per_axis"], w.grid["qmax"])
    idx = W.sample_q_indices(w.n_q, 200, seed=11)
    f_ref = oracle_mod.form_factors(w.basis, w.T, q[idx])
    Td, qd = torch.as_tensor(w.T, device="cuda"), torch.as_tensor(q, device="cuda")
    with Scarf(0) as sc:
        sc.set_basis(w.basis)
        sc.set_transitions(Td)
        f0 = sc.form_factors(qd).cpu().numpy()
        g0 = sc.form_factors_grid(ax, ax, ax)
        sc.set_option("adaptive_tol", tol)
        sc.set_transitions(Td)
        f1 = sc.form_factors(qd).cpu().numpy()
        st_list = sc.stats()
        g1 = sc.form_factors_grid(ax, ax, ax)
        st_grid = sc.stats()
    scale = np.max(np.abs(f0))
    bound = st_list["adaptive_bound"]
    assert bound > 0.0
    assert np.max(np.abs(f1 - f0)) <= bound + 1e-12 * scale
    assert np.max(np.abs(g1 - g0)) <= bound + 1e-12 * scale
    assert np.max(np.abs(f1[:, idx] - f_ref)) <= bound + TOL * np.max(np.abs(f_ref))
    for st in (st_list, st_grid):
        assert 0.0 < st["last_adaptive_work_fraction"] <= 1.0
    if tol >= 1e-9:
        assert st_list["last_adaptive_work_fraction"] < 0.999
    print(f"adaptive_tol={tol:g}: bound {bound:.3e} (scale {scale:.3e}), measured {np.max(np.abs(f1 - f0)):.3e}, "
          f"work list {st_list['last_adaptive_work_fraction']:.4f} grid {st_grid['last_adaptive_work_fraction']:.4f}")


def test_abs2_output(oracle_mod, Scarf, torch_cuda):
    """S5, the optional |f_s|^2 output (Fig. 6): elementwise on device and host buffers, ragged size."""
    torch = torch_cuda
    rng = np.random.default_rng(2)
    f = rng.normal(size=(3, 1001)) + 1j * rng.normal(size=(3, 1001))
    ref = f.real ** 2 + f.imag ** 2
    with Scarf(0) as sc:
        np.testing.assert_allclose(sc.abs2(f), ref, rtol=5e-16, atol=0)   # one FMA vs two roundings: <= 2 ulp
        np.testing.assert_allclose(sc.abs2(torch.as_tensor(f, device="cuda")).cpu().numpy(), ref, rtol=5e-16, atol=0)   # one FMA vs two roundings: <= 2 ulp


def test_repeated_runs_are_bitwise_identical(oracle_mod, Scarf, torch_cuda):
    """No race detector is available on the measurement pool (profiles/r02_sanitizers.md); a race in the shared-memory stage
    ring, the mbarrier protocol or the ordered ticket fix-up would show up as run-to-run differences.  Config 2 at full size,
    both S4 kernels, several chunk counts, device-side screening included: every repetition must be bit-for-bit the same."""
    torch = torch_cuda
    w = W.make_workload(2, oracle_mod.overlap)
    ax = W.cartesian_axis(w.grid["n_per_axis"], w.grid["qmax"])
    Td, qd = torch.as_tensor(w.T, device="cuda"), torch.as_tensor(w.q, device="cuda")
    with Scarf(0) as sc:
        sc.set_basis(w.basis)
        for K in (0, 5):
            sc.set_option("n_chunks", K)
            ref_l = ref_g = None
            for rep in range(6):
                sc.set_transitions(Td)
                fl = sc.form_factors(qd).clone()
                fg = sc.form_factors_grid(ax, ax, ax).copy()
                torch.cuda.synchronize()
                if rep == 0:
                    ref_l, ref_g = fl, fg
                else:
                    assert torch.equal(torch.view_as_real(fl), torch.view_as_real(ref_l)), (K, rep)
                    assert np.array_equal(fg.view(np.float64), ref_g.view(np.float64)), (K, rep)


def test_huge_q_underflows_cleanly(oracle_mod, Scarf, torch_cuda):
    """|q| ~ 1e4..1e6 against a diffuse pair: q^2/4p is far beyond the exponent range of e^{-x}; the argument is clamped before
    the exponent arithmetic (the 32-bit n used to wrap), so the result is an honest 0, never Inf/NaN/garbage."""
    w = W.make_workload(1, oracle_mod.overlap)
    q = np.array([[2.4e4, 0.0, 0.0], [0.0, -1.0e5, 3.0e4], [1.0e6, 1.0e6, -1.0e6], [3.0e3, 0.1, 0.2], [0.3, 0.2, 0.1]])
    f_ref = oracle_mod.form_factors(w.basis, w.T, q)
    with Scarf(0) as sc:
        sc.set_basis(w.basis)
        sc.set_transitions(w.T)
        f = sc.form_factors(q)
        g = sc.form_factors_grid(np.array([2.4e4, -1.0e6, 0.3]), np.array([0.0, 0.2]), np.array([0.0, 0.1]))
    assert np.all(np.isfinite(f.view(np.float64))) and np.all(np.isfinite(g.view(np.float64)))
    # the library flushes e^{-x} to ~1e-301 (times O(1e10) polynomial values at these |q|) instead of 0: nothing, either way
    assert np.max(np.abs(f[:, :4])) <= 1e-250 and np.max(np.abs(f_ref[:, :4])) <= 1e-250
    assert_parity(f[:, 4:], f_ref[:, 4:])

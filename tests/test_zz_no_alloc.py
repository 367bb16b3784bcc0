"""scarf_form_factors_noalloc (include/scarf.h): the S4 list path for callers that must not allocate — the per-tile tickets of
the ordered chunk fix-up live in a static device array instead of a context buffer.  Checked against the existing path
(scarf_form_factors, bit for bit: same kernels, same chunking) and against the oracle, on two calls in a row that use
different tile and chunk counts (the shared array keeps the first call's contents), plus the size limit and the refusal of
host pointers.  Collected last on purpose (file name): the suite runs with `pytest -x`."""
import ctypes as C

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


def _ghi_basis():
    # s..d on one centre, a g shell on the other: pair classes 0..8, so the high-class kernel runs as well
    return W.Basis(np.array([[0.1, 0.2, -0.9], [0.3, -0.4, 1.0]]), np.array([0, 0, 0, 1, 1], np.int32),
                   np.array([0, 1, 2, 1, 4], np.int32), np.array([2, 1, 1, 1, 1], np.int32),
                   np.array([2.1, 0.4, 1.3, 0.9, 0.7, 1.1]), np.array([0.5, 0.6, 1.0, 1.0, 1.0, 1.0]))


def _close(a, b):
    for s in range(b.shape[0]):
        assert np.max(np.abs(a[s] - b[s])) <= TOL * np.max(np.abs(b[s]))


@pytest.mark.parametrize("case", ["config1", "g_shell"])
def test_noalloc_matches_existing_path_twice(oracle_mod, torch_cuda, case):
    torch = torch_cuda
    from paper_2512_18010_b200 import Scarf
    if case == "config1":
        w = W.make_workload(1, oracle_mod.overlap)
        basis, T = w.basis, w.T
    else:
        basis = _ghi_basis()
        T = np.random.default_rng(5).normal(size=(5, basis.nbf, basis.nbf))
    rng = np.random.default_rng(77)
    # two calls in a row: 8 tiles (ragged tail) with 5 chunks, then 3 tiles with 3 chunks — the second finds the array used
    calls = [(rng.uniform(-4, 4, size=(1901, 3)), 5), (rng.uniform(-3, 3, size=(700, 3)), 3), (rng.uniform(-3, 3, size=(257, 3)), 0)]
    with Scarf(0) as sc:
        sc.set_basis(basis)
        sc.set_transitions(T)
        n_states = T.shape[0]
        for q, n_chunks in calls:
            sc.set_option("n_chunks", n_chunks)
            qd = torch.from_numpy(q).cuda()
            ref = sc.form_factors(qd).cpu().numpy()                 # existing path (context-owned tickets)
            out = torch.full((n_states, q.shape[0], 2), float("nan"), dtype=torch.float64, device="cuda")
            free0 = torch.cuda.mem_get_info()[0]
            got = sc.form_factors_noalloc(qd, out)
            torch.cuda.synchronize()
            free1 = torch.cuda.mem_get_info()[0]
            got = got.cpu().numpy()
            assert free1 >= free0                                    # nothing was allocated on the device
            _close(got, ref)
            assert np.array_equal(got, ref)                          # same kernels, same chunk order: bit-identical
            _close(got, oracle_mod.form_factors(basis, T, q))
            if n_chunks > 1:
                assert sc.stats()["last_n_chunks"] == n_chunks


def test_noalloc_rejects_oversize_and_host_pointers(oracle_mod, torch_cuda):
    torch = torch_cuda
    from paper_2512_18010_b200 import Scarf, ScarfError
    from paper_2512_18010_b200 import binding as B
    w = W.make_workload(1, oracle_mod.overlap)
    with Scarf(0) as sc:
        sc.set_basis(w.basis)
        sc.set_transitions(w.T)
        q4 = np.array([[0.3, -1.2, 0.5], [1.5, 0.2, -0.7], [-2.0, 0.9, 0.1], [0.05, 0.6, 2.2]])
        qd = torch.from_numpy(q4).cuda()
        out = torch.zeros((w.T.shape[0], 4, 2), dtype=torch.float64, device="cuda")
        # beyond the static scratch: refused before anything is touched (the tensors are deliberately small)
        rc = B.lib().scarf_form_factors_noalloc(sc._h, B.NOALLOC_MAX_Q + 1, C.c_void_p(qd.data_ptr()), C.c_void_p(out.data_ptr()))
        assert rc == B.SCARF_EINVAL
        msg = B.lib().scarf_last_error(sc._h).decode()
        assert str(B.NOALLOC_MAX_Q) in msg and "static scratch" in msg
        # host pointers would need staging buffers: refused
        qh = np.zeros((4, 3))
        oh = np.zeros((w.T.shape[0], 4, 2))
        rc = B.lib().scarf_form_factors_noalloc(sc._h, 4, C.c_void_p(qh.ctypes.data), C.c_void_p(oh.ctypes.data))
        assert rc == B.SCARF_EINVAL
        assert "device pointers" in B.lib().scarf_last_error(sc._h).decode()
        with pytest.raises(ValueError):
            sc.form_factors_noalloc(qh, oh)
        # the context still works afterwards
        got = sc.form_factors_noalloc(qd, out).cpu().numpy()
        _close(got, oracle_mod.form_factors(w.basis, w.T, q4))
        assert np.array_equal(got, sc.form_factors(qd).cpu().numpy())

"""The boundary's promise (include/scarf.h "Conventions"): no mutable process-wide state; distinct contexts are independent
and may be driven from different threads.  Two contexts with different bases, transitions and FFT grids are interleaved
call by call, then driven concurrently from two threads; every result is compared with the oracle."""
import threading

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


def _cases(oracle_mod):
    from oracle import fft_method as offt
    w1 = W.make_workload(1, oracle_mod.overlap)
    rng = np.random.default_rng(31)
    b2 = W.Basis(np.array([[0.1, 0.2, -0.9], [0.3, -0.4, 1.0]]), np.array([0, 0, 0, 0, 1, 1, 1, 1], np.int32),
                 np.array([0, 1, 2, 3, 0, 1, 2, 3], np.int32), np.array([2, 1, 1, 1, 2, 1, 1, 1], np.int32),
                 np.array([2.1, 0.4, 1.3, 0.9, 0.7, 1.9, 0.5, 1.1, 0.8, 0.6]),
                 np.array([0.5, 0.6, 1.0, 1.0, 1.0, 0.7, 0.4, 1.0, 1.0, 1.0]))
    T2 = rng.normal(size=(5, b2.nbf, b2.nbf))
    cases = []
    for basis, T, n, seed in ((w1.basis, w1.T, (12, 10, 14), 1), (b2, T2, (9, 16, 11), 2)):
        q = np.random.default_rng(seed).uniform(-4, 4, size=(301, 3))
        ax = [np.linspace(-3, 3, 7), np.linspace(-2, 4, 9), np.linspace(-4, 1, 6)]
        X, Y, Z = np.meshgrid(*ax, indexing="ij")
        x_min, L = np.array([-5.0, -4.5, -6.0]), np.array([10.5, 9.0, 11.0])
        cases.append(dict(basis=basis, T=T, q=q, ax=ax, n=n, x_min=x_min, L=L,
                          f=oracle_mod.form_factors(basis, T, q),
                          fg=oracle_mod.form_factors(basis, T, np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1)),
                          ff=offt.form_factors(basis, T, n, x_min, L)))
    return cases


def _check(a, b):
    for s in range(b.shape[0]):
        assert np.max(np.abs(a[s] - b[s])) <= TOL * np.max(np.abs(b[s]))


def test_two_contexts_interleaved(oracle_mod, torch_cuda):
    from paper_2512_18010_b200 import Scarf
    cases = _cases(oracle_mod)
    ctxs = [Scarf(0), Scarf(0)]
    try:
        for rep in range(3):                         # every call alternates between the contexts
            for sc, c in zip(ctxs, cases):
                sc.set_basis(c["basis"])
            for sc, c in zip(ctxs, cases):
                sc.set_transitions(c["T"])
            for sc, c in zip(ctxs, cases):
                _check(sc.fft_form_factors(c["n"], c["x_min"], c["L"], device_out=False), c["ff"])   # different grids: each keeps its plan
            for sc, c in zip(ctxs, cases):
                _check(sc.form_factors(c["q"]), c["f"])
            for sc, c in zip(ctxs, cases):
                _check(sc.form_factors_grid(*c["ax"]), c["fg"])
    finally:
        for sc in ctxs:
            sc.close()


def test_two_contexts_two_threads(oracle_mod, torch_cuda):
    from paper_2512_18010_b200 import Scarf
    cases = _cases(oracle_mod)
    errors = []

    def worker(c):
        try:
            for rep in range(4):
                with Scarf(0) as sc:                 # create/destroy concurrently as well
                    sc.set_basis(c["basis"])
                    sc.set_transitions(c["T"])
                    _check(sc.form_factors(c["q"]), c["f"])
                    _check(sc.form_factors_grid(*c["ax"]), c["fg"])
                    _check(sc.fft_form_factors(c["n"], c["x_min"], c["L"], device_out=False), c["ff"])
        except Exception as e:                       # noqa: BLE001
            errors.append(repr(e))

    th = [threading.Thread(target=worker, args=(c,)) for c in cases]
    for t in th:
        t.start()
    for t in th:
        t.join()
    assert not errors, errors

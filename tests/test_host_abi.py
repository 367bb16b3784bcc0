"""CPU tests (no GPU, no compute kernels) of the C-ABI library: it loads, exports every symbol include/scarf.h declares,
its host-side steps S0-S2 (shell normalisation, Gaussian product, McMurchie-Davidson E coefficients, overlap) and the
host table of scarf_angular_moments agree with the oracle / quadrature / scipy, and the device entry points refuse a
host-only context instead of falling back to the CPU."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import workloads as W
from tests import bruteforce as BF

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_2512_18010_b200 import binding as b
    return b


def test_every_declared_symbol_is_exported(binding):
    hdr = open(os.path.join(ROOT, "include", "scarf.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(scarf_[A-Za-z0-9_]+)\s*\(", hdr))
    assert {"scarf_set_basis", "scarf_set_transitions", "scarf_form_factors", "scarf_form_factors_grid",
            "scarf_angular_moments"} <= names
    lib = C.CDLL(binding.LIB_PATH)
    for n in sorted(names):
        assert hasattr(lib, n), f"{n} declared in include/scarf.h but not exported by libscarf.so"
    assert names == set(binding.EXPORTS), names ^ set(binding.EXPORTS)
    assert b"sm_100a" in binding.version().encode()


def test_host_only_context_has_no_cpu_fallback(binding, oracle_mod):
    w = W.make_workload(1, oracle_mod.overlap)
    with binding.Scarf(None) as sc:
        sc.set_basis(w.basis)
        assert sc.nbf == w.basis.nbf
        for call in (lambda: sc.set_transitions(w.T), lambda: sc.form_factors(w.q[:4]),
                     lambda: sc.form_factors_grid(np.zeros(2), np.zeros(2), np.zeros(2)),
                     lambda: sc.angular_moments(np.zeros((1, 1, 2, 4), complex), np.array([-0.5, 0.5]), np.ones(2), 4, 1)):
            with pytest.raises(binding.ScarfError) as e:
                call()
            assert e.value.code in (binding.SCARF_ENODEVICE, binding.SCARF_ESTATE)


@pytest.mark.parametrize("config", [1, 2])
def test_host_overlap_matches_oracle(binding, oracle_mod, config):
    """S0-S2 on the host (alpha-form, McMurchie-Davidson) against the oracle's sigma-form Eq. (38)-(46) at q = 0."""
    w = W.make_workload(config, oracle_mod.overlap, with_q=False)
    with binding.Scarf(None) as sc:
        sc.set_basis(w.basis)
        S = sc.overlap()
        st = sc.stats()
    assert np.max(np.abs(S - oracle_mod.overlap(w.basis))) <= 1e-12
    assert np.allclose(np.diag(S), 1.0, atol=1e-13)
    n = int(np.sum(w.basis.shell_nprim))
    assert st["n_pairs_all"] == n * (n + 1) // 2 and st["nbf"] == w.basis.nbf


def test_hermite_E_against_quadrature(binding):
    """(x-A)^i (x-B)^j e^{-a(x-A)^2 - b(x-B)^2} = sum_t E_t^{ij} (d/dP)^t e^{-p(x-P)^2}  =>
    Int ... e^{iqx} dx = sqrt(pi/p) e^{-q^2/4p} e^{iqP} sum_t E_t^{ij} (iq)^t; left side by trapezoid quadrature."""
    a, b, A, B = 0.9, 1.7, -0.4, 0.55
    p, P = a + b, (a * A + b * B) / (a + b)
    E = binding.host_hermite_E(6, 6, a, b, A, B)                      # up to i shells on both sides
    for q in (0.0, 0.8, -2.3):
        for i in range(7):
            for j in range(7):
                lhs = BF._int1d(i, A, a, j, B, b, q)
                rhs = np.sqrt(np.pi / p) * np.exp(-q * q / (4 * p)) * np.exp(1j * q * P) * sum(
                    E[i, j, t] * (1j * q) ** t for t in range(i + j + 1))
                assert abs(lhs - rhs) <= 1e-12 * max(1.0, abs(BF._int1d(i, A, a, j, B, b, 0.0)), abs(lhs)), (q, i, j)


def test_shell_norms_against_oracle(binding, oracle_mod):
    """Effective coefficients N_mu d_k xi_k of a contracted shell: every component has unit self-overlap."""
    e, d = np.array([2.3, 0.7, 0.25]), np.array([0.4, 0.9, 0.6])
    for l in range(7):
        c = binding.host_shell_norms(l, e, d)
        b = W.Basis(np.zeros((1, 3)), np.array([0], np.int32), np.array([l], np.int32), np.array([3], np.int32), e, d)
        xi, N = oracle_mod.norms(b)
        ncomp = (l + 1) * (l + 2) // 2
        ref = (N[:, None] * d[None, :]) * xi.reshape(ncomp, 3)
        assert np.max(np.abs(c - ref)) <= 1e-13 * np.max(np.abs(ref))


def test_host_ylm_table_against_scipy(binding):
    from scipy import special as sp
    l_max = 24
    ct, w = np.polynomial.legendre.leggauss(9)
    Yw = binding.host_ylm_table(l_max, ct, w)
    for l in range(l_max + 1):
        for m in range(l + 1):
            ref = w * sp.sph_harm_y(l, m, np.arccos(ct), 0.0).real
            assert np.max(np.abs(Yw[:, l * (l + 1) // 2 + m] - ref)) <= 1e-15 + 2e-13 * np.max(np.abs(ref)), (l, m)


def test_bad_arguments_are_rejected_on_the_host(binding):
    with binding.Scarf(None) as sc:
        good = dict(atom_xyz=np.zeros((1, 3)), shell_atom=[0], shell_l=[0], shell_nprim=[1], exponents=[1.0], coeffs=[1.0])
        sc.set_basis(**good)
        for bad in (dict(good, shell_l=[7]), dict(good, exponents=[-1.0]), dict(good, shell_atom=[3]),
                    dict(good, exponents=[np.nan])):
            with pytest.raises(binding.ScarfError):
                sc.set_basis(**bad)
        with pytest.raises(binding.ScarfError):
            sc.set_option("no_such_option", 1.0)


def test_oscillator_fit_host():
    """scarf_oscillator_fit (Eq. 81-82): exact recovery of A + B q^2 + C q^4, the q_max cut, more than one
    state, and the error paths (fewer than three usable radii)."""
    from paper_2512_18010_b200 import binding
    q = np.geomspace(0.01, 0.5, 17)
    coefs = np.array([[1e-9, 0.37, -0.05], [0.0, 2.5, 0.4]])
    f2 = coefs[:, :1] + coefs[:, 1:2] * q ** 2 + coefs[:, 2:3] * q ** 4
    out = binding.oscillator_fit(q, f2)
    np.testing.assert_allclose(out[:, 1:], coefs[:, 1:], rtol=1e-9)
    np.testing.assert_allclose(out[:, 0], coefs[:, 0], atol=1e-12)
    f2c = f2 + 3.0 * q ** 6                                  # a q^6 tail: the fit restricted to small q is closer to B
    full, cut = binding.oscillator_fit(q, f2c)[0], binding.oscillator_fit(q, f2c, q_max=0.05)[0]
    assert abs(cut[1] - coefs[0, 1]) < abs(full[1] - coefs[0, 1])
    assert abs(cut[1] - coefs[0, 1]) <= 1e-4 * coefs[0, 1]
    with pytest.raises(binding.ScarfError):
        binding.oscillator_fit(q, f2, q_max=0.011)           # two radii left
    with pytest.raises(binding.ScarfError):
        binding.oscillator_fit(np.full(5, 0.1), f2[:, :5])   # one distinct |q|


def test_host_overlap_g_h_i_shells(binding, oracle_mod):
    """Shells up to i (l = 6): S0-S2 on the host against the oracle (itself pinned by quadrature in
    tests/test_oracle_pins_high_l.py); SCARF_EINVAL beyond l = 6."""
    from tests.test_oracle_pins_high_l import _ghi_basis
    b = _ghi_basis()
    with binding.Scarf(None) as sc:
        sc.set_basis(b)
        S = sc.overlap()
        st = sc.stats()
    assert st["l_max"] == 6 and st["nbf"] == b.nbf
    assert np.max(np.abs(S - oracle_mod.overlap(b))) <= 1e-12
    with binding.Scarf(None) as sc:
        with pytest.raises(binding.ScarfError) as e:
            sc.set_basis(atom_xyz=np.zeros((1, 3)), shell_atom=[0], shell_l=[7], shell_nprim=[1], exponents=[1.0], coeffs=[1.0])
        assert e.value.code == binding.SCARF_EINVAL


def test_host_pure_overlap_g_h_i(binding, oracle_mod):
    """Pure (solid-harmonic) g, h, i shells: 2l+1 functions from the closed-form S_lm (csrc/pure.cu) against the oracle's
    route (scipy's Y_lm fitted onto the Cartesian components, oracle/pure.py)."""
    from oracle import pure as opure
    from tests.test_oracle_pins_high_l import _ghi_basis
    b = _ghi_basis()
    flags = np.array([1, 1, 1, 0], np.int32)
    with binding.Scarf(None) as sc:
        sc.set_basis(b, shell_pure=flags)
        assert sc.nbf == 9 + 11 + 13 + 3
        S = sc.overlap()
    S_ref = opure.overlap(b, flags)
    assert np.max(np.abs(S - S_ref)) <= 1e-12
    assert np.allclose(np.diag(S), 1.0, atol=1e-12)

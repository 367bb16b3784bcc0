"""Thin ctypes binding of libscarf.so (include/scarf.h).  Argument marshalling only: every step of the path
runs inside the library.  PyTorch tensors are accepted for T, q and out (their `data_ptr()` is passed on);
numpy arrays are passed as host pointers.  If the library has not been built the import of this module fails
loudly — there is no fallback of any kind.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libscarf.so")

SCARF_OK, SCARF_EINVAL, SCARF_ESTATE, SCARF_ENOMEM, SCARF_ECUDA, SCARF_ENODEVICE = 0, -1, -2, -3, -4, -5
SCARF_MAX_L = 6
SCARF_N_CLASSES = 2 * SCARF_MAX_L + 1
_CODES = {-1: "EINVAL", -2: "ESTATE", -3: "ENOMEM", -4: "ECUDA", -5: "ENODEVICE"}

NOALLOC_MAX_TILES = 65536                  # SCARF_NOALLOC_MAX_TILES (include/scarf.h)
NOALLOC_MAX_Q = NOALLOC_MAX_TILES * 256     # q-points per scarf_form_factors_noalloc call

EXPORTS = ["scarf_create", "scarf_destroy", "scarf_set_stream", "scarf_set_option", "scarf_set_basis", "scarf_set_basis_pure", "scarf_nbf",
           "scarf_overlap", "scarf_set_transitions", "scarf_form_factors", "scarf_form_factors_noalloc", "scarf_form_factors_grid", "scarf_form_factors_sph", "scarf_separable_integral", "scarf_angular_moments", "scarf_oscillator_fit", "scarf_abs2", "scarf_fft_form_factors", "scarf_fft_parseval", "scarf_get_stats", "scarf_last_error",
           "scarf_version", "scarf_fp64_peak", "scarf_host_hermite_E", "scarf_host_shell_norms", "scarf_host_ylm_table"]


class ScarfStats(C.Structure):
    _fields_ = [("n_atoms", C.c_int32), ("n_shells", C.c_int32), ("n_prim_shells", C.c_int32), ("nbf", C.c_int32),
                ("n_states", C.c_int32), ("l_max", C.c_int32),
                ("n_pairs_all", C.c_int64), ("n_pairs_prescreened", C.c_int64), ("n_pairs_kept", C.c_int64),
                ("pairs_kept_per_class", C.c_int64 * SCARF_N_CLASSES),
                ("n_herm_kept", C.c_int64), ("cart_term_pairs", C.c_int64),
                ("stream_bytes", C.c_double), ("slots_per_q", C.c_double), ("evals_per_q", C.c_double),
                ("last_setup_host_ms", C.c_double), ("last_fold_ms", C.c_double), ("last_kernel_ms", C.c_double),
                ("last_kernel_launches", C.c_int32), ("last_fold_launches", C.c_int32),
                ("last_grid_slots", C.c_double), ("dropped_bound", C.c_double),
                ("last_grid_symmetric", C.c_int32), ("last_n_chunks", C.c_int32),
                ("last_main_kernel_ms", C.c_double), ("last_grid_kernel_slots", C.c_double),
                ("adaptive_bound", C.c_double), ("last_adaptive_work_fraction", C.c_double),
                ("last_grid_variant", C.c_int32), ("reserved0", C.c_int32)]

    def as_dict(self):
        d = {}
        for name, _t in self._fields_:
            v = getattr(self, name)
            d[name] = list(v) if hasattr(v, "__len__") else v
        return d


class ScarfError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"scarf error {_CODES.get(code, code)}: {msg}")
        self.code = code


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2512_18010_b200.build` "
                          "(nvcc, sm_100a).  There is no CPU fallback.")
    L = C.CDLL(LIB_PATH)
    dp, ip, vp = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.c_void_p
    L.scarf_create.argtypes = [C.POINTER(vp), C.c_int]
    L.scarf_destroy.argtypes = [vp]
    L.scarf_destroy.restype = None
    L.scarf_set_stream.argtypes = [vp, vp]
    L.scarf_set_option.argtypes = [vp, C.c_char_p, C.c_double]
    L.scarf_set_basis.argtypes = [vp, C.c_int, dp, C.c_int, ip, ip, ip, dp, dp]
    L.scarf_set_basis_pure.argtypes = [vp, C.c_int, dp, C.c_int, ip, ip, ip, dp, dp, ip]
    L.scarf_nbf.argtypes = [vp]
    L.scarf_overlap.argtypes = [vp, dp]
    L.scarf_set_transitions.argtypes = [vp, C.c_int, vp]
    L.scarf_form_factors.argtypes = [vp, C.c_int64, vp, vp]
    L.scarf_form_factors_noalloc.argtypes = [vp, C.c_int64, vp, vp]
    L.scarf_form_factors_grid.argtypes = [vp, C.c_int32, vp, C.c_int32, vp, C.c_int32, vp, vp]
    L.scarf_form_factors_sph.argtypes = [vp, C.c_int32, vp, C.c_int32, vp, C.c_int32, vp]
    L.scarf_separable_integral.argtypes = [vp, C.c_int32, dp, dp, C.c_int32, dp, dp, C.c_int32, dp, dp, dp]
    L.scarf_angular_moments.argtypes = [vp, C.c_int32, C.c_int32, C.c_int32, dp, dp, C.c_int32, C.c_int32, vp, vp, vp]
    L.scarf_abs2.argtypes = [vp, C.c_int64, vp, vp]
    L.scarf_oscillator_fit.argtypes = [C.c_int32, C.c_int32, dp, dp, C.c_double, dp]
    L.scarf_host_ylm_table.argtypes = [C.c_int, C.c_int, dp, dp, dp]
    L.scarf_fft_form_factors.argtypes = [vp, C.c_int32, C.c_int32, C.c_int32, dp, dp, vp]
    L.scarf_fft_parseval.argtypes = [vp, dp]
    L.scarf_get_stats.argtypes = [vp, C.POINTER(ScarfStats)]
    L.scarf_last_error.argtypes = [vp]
    L.scarf_last_error.restype = C.c_char_p
    L.scarf_version.restype = C.c_char_p
    L.scarf_fp64_peak.argtypes = [C.c_int, dp, dp]
    L.scarf_host_hermite_E.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, dp]
    L.scarf_host_shell_norms.argtypes = [C.c_int, C.c_int, dp, dp, dp]
    for name in EXPORTS:      # every symbol include/scarf.h declares must resolve
        getattr(L, name)
    return L


_lib = _load()


def lib():
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int32))


def _is_torch(x) -> bool:
    return hasattr(x, "data_ptr") and hasattr(x, "is_contiguous")


def _ptr(x, what, n_expected=None):
    """(pointer, keep-alive object) for a float64, C-contiguous numpy array or torch tensor."""
    if _is_torch(x):
        import torch
        if x.dtype != torch.float64 or not x.is_contiguous():
            raise ValueError(f"{what}: torch tensor must be float64 and contiguous")
        if n_expected is not None and x.numel() != n_expected:
            raise ValueError(f"{what}: expected {n_expected} elements, got {x.numel()}")
        return C.c_void_p(x.data_ptr()), x
    a = np.ascontiguousarray(x, dtype=np.float64)
    if n_expected is not None and a.size != n_expected:
        raise ValueError(f"{what}: expected {n_expected} elements, got {a.size}")
    return C.c_void_p(a.ctypes.data), a


def version() -> str:
    return _lib.scarf_version().decode()


def fp64_peak(device: int = 0):
    """(lane-level DFMA per second, SM clock in MHz) measured on `device` by the library's micro-benchmark."""
    r, m = C.c_double(0), C.c_double(0)
    rc = _lib.scarf_fp64_peak(int(device), C.byref(r), C.byref(m))
    if rc != SCARF_OK:
        raise ScarfError(rc, "scarf_fp64_peak failed")
    return r.value, m.value


def host_hermite_E(la, lb, alpha, beta, Ax, Bx) -> np.ndarray:
    out = np.zeros((la + 1, lb + 1, la + lb + 1))
    rc = _lib.scarf_host_hermite_E(la, lb, alpha, beta, Ax, Bx, _dp(out))
    if rc != SCARF_OK:
        raise ScarfError(rc, "scarf_host_hermite_E")
    return out


def host_shell_norms(l, exponents, coeffs) -> np.ndarray:
    e = np.ascontiguousarray(exponents, np.float64)
    d = np.ascontiguousarray(coeffs, np.float64)
    out = np.zeros(((l + 1) * (l + 2) // 2, e.size))
    rc = _lib.scarf_host_shell_norms(int(l), int(e.size), _dp(e), _dp(d), _dp(out))
    if rc != SCARF_OK:
        raise ScarfError(rc, "scarf_host_shell_norms")
    return out


class Scarf:
    """One libscarf context.  device=None creates a host-only context (basis setup, overlap, stats)."""

    def __init__(self, device=0):
        self._h = C.c_void_p()
        rc = _lib.scarf_create(C.byref(self._h), -1 if device is None else int(device))
        if rc != SCARF_OK:
            raise ScarfError(rc, "scarf_create failed (no usable CUDA device? there is no CPU fallback)")
        self.device = device
        self.n_states = 0
        self._nbf = 0

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            _lib.scarf_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def _check(self, rc):
        if rc != SCARF_OK:
            raise ScarfError(rc, _lib.scarf_last_error(self._h).decode())

    def set_stream(self, cuda_stream: int):
        self._check(_lib.scarf_set_stream(self._h, C.c_void_p(int(cuda_stream))))

    def set_option(self, key: str, value: float):
        self._check(_lib.scarf_set_option(self._h, key.encode(), float(value)))

    def set_basis(self, basis=None, *, atom_xyz=None, shell_atom=None, shell_l=None, shell_nprim=None,
                  exponents=None, coeffs=None, shell_pure=None):
        if basis is not None:
            atom_xyz, shell_atom, shell_l = basis.atom_xyz, basis.shell_atom, basis.shell_l
            shell_nprim, exponents, coeffs = basis.shell_nprim, basis.exponents, basis.coeffs
        xyz = np.ascontiguousarray(atom_xyz, np.float64).reshape(-1, 3)
        sa = np.ascontiguousarray(shell_atom, np.int32)
        sl = np.ascontiguousarray(shell_l, np.int32)
        sn = np.ascontiguousarray(shell_nprim, np.int32)
        e = np.ascontiguousarray(exponents, np.float64)
        d = np.ascontiguousarray(coeffs, np.float64)
        if not (sa.size == sl.size == sn.size) or e.size != d.size or e.size != int(sn.sum()):
            raise ValueError("set_basis: inconsistent array lengths")
        if shell_pure is None:
            self._check(_lib.scarf_set_basis(self._h, xyz.shape[0], _dp(xyz), sl.size, _ip(sa), _ip(sl), _ip(sn), _dp(e), _dp(d)))
        else:
            sp = np.ascontiguousarray(shell_pure, np.int32)
            if sp.size != sl.size:
                raise ValueError("set_basis: shell_pure must have one entry per shell")
            self._check(_lib.scarf_set_basis_pure(self._h, xyz.shape[0], _dp(xyz), sl.size, _ip(sa), _ip(sl), _ip(sn), _dp(e), _dp(d),
                                                  _ip(sp)))
        self._nbf = int(_lib.scarf_nbf(self._h))
        self.n_states = 0

    @property
    def nbf(self) -> int:
        return self._nbf

    def overlap(self) -> np.ndarray:
        S = np.zeros((self._nbf, self._nbf))
        self._check(_lib.scarf_overlap(self._h, _dp(S)))
        return S

    def set_transitions(self, T):
        shape = tuple(T.shape)
        if len(shape) == 2:
            shape = (1,) + shape
        if len(shape) != 3 or shape[1] != self._nbf or shape[2] != self._nbf:
            raise ValueError(f"set_transitions: T must be [n_states][{self._nbf}][{self._nbf}]")
        p, keep = _ptr(T, "T", shape[0] * shape[1] * shape[2])
        self._check(_lib.scarf_set_transitions(self._h, shape[0], p))
        self.n_states = shape[0]

    def form_factors(self, q, out=None):
        """q: [n_q][3] float64 numpy (host) or torch (host or cuda).  out: optional float64 buffer
        [n_states][n_q][2] (numpy or torch); allocated like q when omitted.  Returns complex128 [n_states][n_q]
        (a view of `out`)."""
        n_q = int(q.shape[0])
        if tuple(q.shape) != (n_q, 3):
            raise ValueError("form_factors: q must be [n_q][3]")
        qp, qkeep = _ptr(q, "q", 3 * n_q)
        if out is None:
            if _is_torch(q):
                import torch
                out = torch.empty((self.n_states, n_q, 2), dtype=torch.float64, device=q.device)
            else:
                out = np.empty((self.n_states, n_q, 2))
        op, okeep = _ptr(out, "out", self.n_states * n_q * 2)
        if not _is_torch(out) and okeep is not out:
            raise ValueError("form_factors: out must be a C-contiguous float64 array")
        self._check(_lib.scarf_form_factors(self._h, n_q, qp, op))
        if _is_torch(out):
            import torch
            return torch.view_as_complex(out.view(self.n_states, n_q, 2))
        return out.reshape(self.n_states, n_q, 2).view(np.complex128)[..., 0]

    def form_factors_noalloc(self, q, out):
        """scarf_form_factors_noalloc: the same result as form_factors without any device allocation or synchronisation
        inside the library (tickets in a static device array; at most NOALLOC_MAX_Q q-points per call).  q [n_q][3] and
        out [n_states][n_q][2]: float64 CUDA tensors, both supplied by the caller.  Returns a complex view of `out`."""
        import torch
        if not (_is_torch(q) and _is_torch(out) and q.is_cuda and out.is_cuda):
            raise ValueError("form_factors_noalloc: q and out must be CUDA tensors")
        n_q = int(q.shape[0])
        if tuple(q.shape) != (n_q, 3):
            raise ValueError("form_factors_noalloc: q must be [n_q][3]")
        qp, qkeep = _ptr(q, "q", 3 * n_q)
        op, okeep = _ptr(out, "out", self.n_states * n_q * 2)
        self._check(_lib.scarf_form_factors_noalloc(self._h, n_q, qp, op))
        return torch.view_as_complex(out.view(self.n_states, n_q, 2))

    def form_factors_grid(self, qx, qy, qz, out=None):
        """Product grid q = (qx[ix], qy[iy], qz[iz]), point index (ix*ny + iy)*nz + iz.  qx, qy, qz: 1-D float64
        numpy or torch (host or cuda).  Returns complex128 [n_states][nx*ny*nz] (a view of `out`)."""
        nx, ny, nz = int(qx.shape[0]), int(qy.shape[0]), int(qz.shape[0])
        n_q = nx * ny * nz
        xp, xkeep = _ptr(qx, "qx", nx)
        yp, ykeep = _ptr(qy, "qy", ny)
        zp, zkeep = _ptr(qz, "qz", nz)
        if out is None:
            if _is_torch(qx):
                import torch
                out = torch.empty((self.n_states, n_q, 2), dtype=torch.float64, device=qx.device)
            else:
                out = np.empty((self.n_states, n_q, 2))
        op, okeep = _ptr(out, "out", self.n_states * n_q * 2)
        if not _is_torch(out) and okeep is not out:
            raise ValueError("form_factors_grid: out must be a C-contiguous float64 array")
        self._check(_lib.scarf_form_factors_grid(self._h, nx, xp, ny, yp, nz, zp, op))
        if _is_torch(out):
            import torch
            return torch.view_as_complex(out.view(self.n_states, n_q, 2))
        return out.reshape(self.n_states, n_q, 2).view(np.complex128)[..., 0]

    def form_factors_sph(self, r, cos_theta, n_phi: int, out=None, device: bool = True):
        """Spherical product grid q = r[i] (sin t_j cos phi_k, sin t_j sin phi_k, cos t_j), phi_k = 2 pi k / n_phi, point index
        (i*n_theta + j)*n_phi + k (the input layout of angular_moments).  r, cos_theta: 1-D float64 host arrays.  `out`: torch
        (host or cuda) or numpy [n_states][n_q][2]; if None a CUDA tensor (device=True) or a numpy array is allocated.
        Returns complex128 [n_states][n_r*n_theta*n_phi] (a view of `out`)."""
        rr = np.ascontiguousarray(r, dtype=np.float64)
        ct = np.ascontiguousarray(cos_theta, dtype=np.float64)
        n_r, n_theta = int(rr.shape[0]), int(ct.shape[0])
        n_q = n_r * n_theta * int(n_phi)
        if out is None:
            if device:
                import torch
                out = torch.empty((self.n_states, n_q, 2), dtype=torch.float64, device="cuda")
            else:
                out = np.empty((self.n_states, n_q, 2))
        op, okeep = _ptr(out, "out", self.n_states * n_q * 2)
        if not _is_torch(out) and okeep is not out:
            raise ValueError("form_factors_sph: out must be a C-contiguous float64 array")
        self._check(_lib.scarf_form_factors_sph(self._h, n_r, rr.ctypes.data_as(C.c_void_p), n_theta, ct.ctypes.data_as(C.c_void_p),
                                                int(n_phi), op))
        if _is_torch(out):
            import torch
            return torch.view_as_complex(out.view(self.n_states, n_q, 2))
        return out.reshape(self.n_states, n_q, 2).view(np.complex128)[..., 0]

    def angular_moments(self, f, cos_theta, w_theta, n_phi: int, l_max: int, n_r: int = None, want_f2: bool = True):
        """f: complex128 [n_states][n_r*n_theta*n_phi] (what form_factors returns on the spherical product grid) or
        [n_states][n_r][n_theta][n_phi]; torch (host or cuda) or numpy.  Returns (R complex [n_states][n_r][(l_max+1)^2],
        f2 real [n_states][n_r] or None) in the same kind of memory as f."""
        ct = np.ascontiguousarray(cos_theta, dtype=np.float64)
        wt = np.ascontiguousarray(w_theta, dtype=np.float64)
        n_theta = int(ct.shape[0])
        n_states = int(f.shape[0])
        total = 1
        for d in f.shape[1:]:
            total *= int(d)
        if n_r is None:
            n_r = total // (n_theta * int(n_phi))
        if n_r * n_theta * int(n_phi) != total:
            raise ValueError("angular_moments: f does not have n_r*n_theta*n_phi points per state")
        nlm = (int(l_max) + 1) ** 2
        if _is_torch(f):
            import torch
            fr = torch.view_as_real(f.contiguous()) if f.is_complex() else f
            fp, fkeep = _ptr(fr, "f", n_states * total * 2)
            R = torch.empty((n_states, n_r, nlm, 2), dtype=torch.float64, device=f.device)
            f2 = torch.empty((n_states, n_r), dtype=torch.float64, device=f.device) if want_f2 else None
            rp = C.c_void_p(R.data_ptr())
            f2p = C.c_void_p(f2.data_ptr()) if want_f2 else None
        else:
            fa = np.ascontiguousarray(f, dtype=np.complex128)
            fp, fkeep = C.c_void_p(fa.ctypes.data), fa
            R = np.empty((n_states, n_r, nlm, 2))
            f2 = np.empty((n_states, n_r)) if want_f2 else None
            rp = C.c_void_p(R.ctypes.data)
            f2p = C.c_void_p(f2.ctypes.data) if want_f2 else None
        dp = C.POINTER(C.c_double)
        self._check(_lib.scarf_angular_moments(self._h, n_states, n_r, n_theta, ct.ctypes.data_as(dp), wt.ctypes.data_as(dp),
                                               int(n_phi), int(l_max), fp, rp, f2p))
        if _is_torch(f):
            import torch
            return torch.view_as_complex(R), f2
        return R.view(np.complex128)[..., 0], f2

    def fft_form_factors(self, n, x_min, box_len, out=None, device_out=True):
        """The paper's FFT method on an n = (nx, ny, nz) real-space grid in the box [x_min, x_min + box_len).
        Returns complex128 [n_states][nx*ny*nz] at q = 2 pi ((ia - nx//2)/Lx, ...) (torch cuda tensor by default)."""
        nx, ny, nz = (int(v) for v in n)
        xm = np.ascontiguousarray(x_min, dtype=np.float64).reshape(3)
        bl = np.ascontiguousarray(box_len, dtype=np.float64).reshape(3)
        n_q = nx * ny * nz
        if out is None:
            if device_out:
                import torch
                out = torch.empty((self.n_states, n_q, 2), dtype=torch.float64, device=f"cuda:{self.device}")
            else:
                out = np.empty((self.n_states, n_q, 2))
        op, okeep = _ptr(out, "out", self.n_states * n_q * 2)
        self._check(_lib.scarf_fft_form_factors(self._h, nx, ny, nz, _dp(xm), _dp(bl), op))
        if _is_torch(out):
            import torch
            return torch.view_as_complex(out.view(self.n_states, n_q, 2))
        return out.reshape(self.n_states, n_q, 2).view(np.complex128)[..., 0]

    def abs2(self, f):
        """|f|^2 elementwise (S5): f complex128 torch (cuda or host) or numpy; returns float64 of the same shape and kind."""
        if _is_torch(f):
            import torch
            fr = torch.view_as_real(f.contiguous())
            out = torch.empty(f.shape, dtype=torch.float64, device=f.device)
            self._check(_lib.scarf_abs2(self._h, f.numel(), C.c_void_p(fr.data_ptr()), C.c_void_p(out.data_ptr())))
            return out
        fa = np.ascontiguousarray(f, dtype=np.complex128)
        out = np.empty(fa.shape)
        self._check(_lib.scarf_abs2(self._h, fa.size, C.c_void_p(fa.ctypes.data), C.c_void_p(out.ctypes.data)))
        return out

    def fft_parseval(self) -> np.ndarray:
        """[n_states][2]: (V_pix sum |Phi|^2, sum |f|^2 / V_box) of the last fft_form_factors call (option check_parseval = 1)."""
        out = np.zeros((self.n_states, 2))
        self._check(_lib.scarf_fft_parseval(self._h, _dp(out)))
        return out

    def separable_integral(self, qx, fx, qy, gy, qz, hz) -> np.ndarray:
        """sum_{ix,iy,iz} fx[ix] gy[iy] hz[iz] f_s(qx[ix], qy[iy], qz[iz]) for every state (complex128 [n_states]),
        in O(pairs * (nx+ny+nz)): Eq. (64)-(65).  All arguments 1-D host arrays (weights x function samples)."""
        arrs = [np.ascontiguousarray(a, dtype=np.float64) for a in (qx, fx, qy, gy, qz, hz)]
        if arrs[0].shape != arrs[1].shape or arrs[2].shape != arrs[3].shape or arrs[4].shape != arrs[5].shape:
            raise ValueError("separable_integral: each weight array must match its axis")
        out = np.zeros((self.n_states, 2))
        self._check(_lib.scarf_separable_integral(self._h, arrs[0].size, _dp(arrs[0]), _dp(arrs[1]), arrs[2].size, _dp(arrs[2]),
                                                  _dp(arrs[3]), arrs[4].size, _dp(arrs[4]), _dp(arrs[5]), _dp(out)))
        return out[:, 0] + 1j * out[:, 1]

    def stats(self) -> dict:
        s = ScarfStats()
        self._check(_lib.scarf_get_stats(self._h, C.byref(s)))
        return s.as_dict()


def oscillator_fit(q_abs, f2, q_max: float = 0.0) -> np.ndarray:
    """[n_states][3] = (A, B, C) of <|f_s|^2>_Omega(q) ~ A + B q^2 + C q^4 (Eq. 81-82); f2 [n_states][n_r] host array."""
    q = np.ascontiguousarray(q_abs, dtype=np.float64)
    y = np.ascontiguousarray(f2, dtype=np.float64).reshape(-1, q.shape[0])
    out = np.zeros((y.shape[0], 3))
    rc = _lib.scarf_oscillator_fit(int(y.shape[0]), int(q.shape[0]), _dp(q), _dp(y), float(q_max), _dp(out))
    if rc != SCARF_OK:
        raise ScarfError(rc, "scarf_oscillator_fit failed (fewer than three usable |q|, or NaN/Inf)")
    return out


def host_ylm_table(l_max: int, cos_theta, w_theta) -> np.ndarray:
    """[n_theta][(l_max+1)(l_max+2)/2]: w_j N_lm P_l^m(cos theta_j), index l(l+1)/2 + m (host code of the library)."""
    ct = np.ascontiguousarray(cos_theta, dtype=np.float64)
    wt = np.ascontiguousarray(w_theta, dtype=np.float64)
    out = np.zeros((ct.shape[0], (l_max + 1) * (l_max + 2) // 2))
    dp = C.POINTER(C.c_double)
    rc = _lib.scarf_host_ylm_table(int(l_max), int(ct.shape[0]), ct.ctypes.data_as(dp), wt.ctypes.data_as(dp), out.ctypes.data_as(dp))
    if rc != SCARF_OK:
        raise ScarfError(rc, "scarf_host_ylm_table failed")
    return out

"""ctypes front end of the CPU oracle (oracle/ulens_oracle.c). TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this module. It imports nothing from paper_2510_02639_b200 (the CUDA path) and the CUDA
path imports nothing from here.

What is computed where
  * finite-source magnification from the definition (Eqs. 5-6): C, orc_mag_fs*
  * lens polynomial coefficients (Eq. 4) in __float128: C, orc_poly_coeffs
  * all roots: companion-matrix eigenvalues with LAPACK through numpy.linalg.eigvals as
    the library step, then extended-precision refinement + Eq.-1 classification in C
    (orc_roots_refine)
  * point-source magnification A = sum 1/|det J| over validated images (Eqs. 2-3)
  * derivative reference: central finite differences of the finite-source integral
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ulens_oracle.c")
_LIB = os.path.join(_HERE, "libulens_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no fast-math). Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC,
                               "-lquadmath", "-lm"])
    return _LIB


class Lens(C.Structure):
    _fields_ = [("n", C.c_int), ("eps", C.c_double * 3), ("ax", C.c_double * 3), ("ay", C.c_double * 3)]

    def positions(self):
        return np.array([complex(self.ax[i], self.ay[i]) for i in range(self.n)])

    def masses(self):
        return np.array([self.eps[i] for i in range(self.n)])


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        dp, ip, llp = C.POINTER(C.c_double), C.POINTER(C.c_int), C.POINTER(C.c_longlong)
        _lib.orc_lens_binary.argtypes = [C.POINTER(Lens), C.c_double, C.c_double]
        _lib.orc_lens_triple.argtypes = [C.POINTER(Lens)] + [C.c_double] * 5
        _lib.orc_lens_single.argtypes = [C.POINTER(Lens)]
        _lib.orc_trajectory.argtypes = [C.c_double] * 4 + [C.c_int, dp, dp, dp]
        _lib.orc_trajectory.restype = None
        _lib.orc_lens_map.argtypes = [C.POINTER(Lens), C.c_double, C.c_double, dp, dp]
        _lib.orc_lens_map.restype = None
        _lib.orc_detJ.argtypes = [C.POINTER(Lens), C.c_double, C.c_double]
        _lib.orc_detJ.restype = C.c_double
        _lib.orc_mag_fs.argtypes = [C.POINTER(Lens)] + [C.c_double] * 4 + [C.c_int, C.c_int, dp, llp]
        _lib.orc_mag_fs_batch.argtypes = [C.POINTER(Lens), ip, C.c_int, dp, dp, dp, dp, C.c_int, C.c_int,
                                          C.c_int, dp, dp, llp]
        _lib.orc_poly_coeffs.argtypes = [C.POINTER(Lens), C.c_double, C.c_double, dp, dp]
        _lib.orc_roots_refine.argtypes = [C.POINTER(Lens), C.c_double, C.c_double, dp, dp, ip, dp, dp, dp]
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def lens_binary(s: float, q: float) -> Lens:
    L = Lens()
    if lib().orc_lens_binary(C.byref(L), s, q) != 0:
        raise ValueError("bad binary lens parameters")
    return L


def lens_triple(s, q, q3, r3, psi) -> Lens:
    L = Lens()
    if lib().orc_lens_triple(C.byref(L), s, q, q3, r3, psi) != 0:
        raise ValueError("bad triple lens parameters")
    return L


def lens_single() -> Lens:
    L = Lens()
    lib().orc_lens_single(C.byref(L))
    return L


def trajectory(t0, u0, tE, alpha, t):
    t = np.ascontiguousarray(t, dtype=np.float64)
    wx, wy = np.empty_like(t), np.empty_like(t)
    lib().orc_trajectory(t0, u0, tE, alpha, len(t), _dp(t), _dp(wx), _dp(wy))
    return wx, wy


def lens_map(L: Lens, z: complex) -> complex:
    wx, wy = C.c_double(), C.c_double()
    lib().orc_lens_map(C.byref(L), z.real, z.imag, C.byref(wx), C.byref(wy))
    return complex(wx.value, wy.value)


def det_J(L: Lens, z: complex) -> float:
    return lib().orc_detJ(C.byref(L), z.real, z.imag)


def mag_fs(L: Lens, w: complex, rho: float, u1: float, n_rho: int = 100, ss: int = 8):
    """A at one lattice pitch rho/n_rho; returns (A, lens-map evaluations)."""
    A, ne = C.c_double(), C.c_longlong()
    if lib().orc_mag_fs(C.byref(L), w.real, w.imag, rho, u1, n_rho, ss, C.byref(A), C.byref(ne)) != 0:
        raise ValueError("bad argument")
    return A.value, ne.value


def mag_fs_batch(lenses, lens_idx, wx, wy, rho, u1, n_rho: int = 100, ss: int = 8, n_threads: int = 0):
    """Finite-source A for many points at pitches rho/n_rho and rho/(2 n_rho).

    The lattice rule is second order in the pitch away from the limb (measured on the single-lens
    closed forms: error 4.1e-5 -> 9.8e-6 -> 1.6e-6 at n_rho = 100, 200, 400), so the reported value is
    the Richardson extrapolation A = A_fine + (A_fine - A_coarse)/3 and the self-error is the size of
    that correction, err_est = |A - A_fine|/A. A point is admissible for parity when err_est <= 2e-5
    (DESIGN.md "oracle admissibility"). Returns dict(A, A_fine, A_coarse, err_est, n_eval).
    """
    lenses = list(lenses)
    arr = (Lens * len(lenses))(*lenses)
    wx = np.ascontiguousarray(wx, dtype=np.float64)
    wy = np.ascontiguousarray(wy, dtype=np.float64)
    n = len(wx)
    rho = np.ascontiguousarray(np.broadcast_to(np.asarray(rho, dtype=np.float64), (n,)))
    u1 = np.ascontiguousarray(np.broadcast_to(np.asarray(u1, dtype=np.float64), (n,)))
    idx = np.ascontiguousarray(np.broadcast_to(np.asarray(lens_idx, dtype=np.int32), (n,)))
    Ac, Af = np.empty(n), np.empty(n)
    ne = np.zeros(n, dtype=np.int64)
    rc = lib().orc_mag_fs_batch(arr, idx.ctypes.data_as(C.POINTER(C.c_int)), n, _dp(wx), _dp(wy), _dp(rho),
                                _dp(u1), n_rho, ss, n_threads, _dp(Ac), _dp(Af),
                                ne.ctypes.data_as(C.POINTER(C.c_longlong)))
    if rc != 0:
        raise ValueError("bad argument")
    A = Af + (Af - Ac) / 3.0
    return dict(A=A, A_fine=Af, A_coarse=Ac, err_est=np.abs(A - Af) / A, n_eval=ne)


def max_threads() -> int:
    return lib().orc_max_threads()


def poly_coeffs(L: Lens, w: complex) -> np.ndarray:
    """b_0..b_Ndeg of Eq. 4 (computed in __float128, rounded to double)."""
    br, bi = np.zeros(12), np.zeros(12)
    deg = lib().orc_poly_coeffs(C.byref(L), w.real, w.imag, _dp(br), _dp(bi))
    return br[:deg + 1] + 1j * bi[:deg + 1]


def roots(L: Lens, w: complex):
    """All N^2+1 roots of Eq. 4 and which of them are images.

    Companion-matrix eigenvalues (numpy.linalg.eigvals = LAPACK zgeev) give starting values,
    the C side refines them in __float128 and classifies them on Eq. 1.
    Returns dict(z, is_image, resid, detJ, kappa).
    """
    b = poly_coeffs(L, w)
    n = len(b) - 1
    comp = np.zeros((n, n), dtype=np.complex128)
    comp[1:, :-1] = np.eye(n - 1)
    comp[:, -1] = -b[:-1] / b[-1]
    z0 = np.linalg.eigvals(comp)
    zr, zi = np.ascontiguousarray(z0.real), np.ascontiguousarray(z0.imag)
    isimg = np.zeros(n, dtype=np.int32)
    res, dj, kap = np.zeros(n), np.zeros(n), np.zeros(n)
    lib().orc_roots_refine(C.byref(L), w.real, w.imag, _dp(zr), _dp(zi),
                           isimg.ctypes.data_as(C.POINTER(C.c_int)), _dp(res), _dp(dj), _dp(kap))
    return dict(z=zr + 1j * zi, is_image=isimg.astype(bool), resid=res, detJ=dj, kappa=kap)


def mag_point_source(L: Lens, w: complex) -> float:
    """A = sum_j 1/|det J(z_j)| over the validated images (Eqs. 2-3)."""
    r = roots(L, w)
    return float(np.sum(1.0 / np.abs(r["detJ"][r["is_image"]])))

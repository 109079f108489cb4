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
        _lib.orc_mag_fs_pitch_batch.argtypes = [C.POINTER(Lens), C.c_int, dp, dp, dp, dp, dp, C.c_int, C.c_int, dp, llp]
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


def mag_fs_pitch_batch(lenses, wx, wy, rho, u1, h, ss: int = 16, n_threads: int = 0):
    """Finite-source A for n points, each with its own lens, radius and explicit lattice pitch h (one pitch,
    no Richardson step): the building block of the finite-difference derivative reference."""
    lenses = list(lenses)
    n = len(lenses)
    arr = (Lens * n)(*lenses)
    f = lambda a: np.ascontiguousarray(np.broadcast_to(np.asarray(a, dtype=np.float64), (n,)))
    wx, wy, rho, u1, h = f(wx), f(wy), f(rho), f(u1), f(h)
    A = np.empty(n)
    ne = np.zeros(n, dtype=np.int64)
    if lib().orc_mag_fs_pitch_batch(arr, n, _dp(wx), _dp(wy), _dp(rho), _dp(u1), _dp(h), ss, n_threads, _dp(A),
                                    ne.ctypes.data_as(C.POINTER(C.c_longlong))) != 0:
        raise ValueError("bad argument")
    return A, ne


def mag_fd(make_case, p0, steps, u1, n_rho: int = 100, ss: int = 16):
    """Derivative reference: central finite differences of the finite-source integral.

    make_case(p) -> (Lens, w_c complex, rho) for a parameter vector p; p0 [n_par] the point; steps
    [n_steps, n_par] the half-widths. Every evaluation uses the lattice of the UNPERTURBED point (pitch
    rho0/n_rho, origin-aligned), so that the smooth part of the lattice error cancels in the difference and
    only its sub-lattice noise (~(h/ss)^1.5) is left. Returns (A0, dA [n_steps, n_par]); the caller
    accepts a derivative where two step sizes agree.
    """
    p0 = np.asarray(p0, dtype=np.float64)
    steps = np.atleast_2d(np.asarray(steps, dtype=np.float64))
    L0, w0, rho0 = make_case(p0)
    h = rho0 / n_rho
    cases = [(L0, w0, rho0)]
    for st in steps:
        for k in range(len(p0)):
            for sgn in (+1.0, -1.0):
                p = p0.copy()
                p[k] += sgn * st[k]
                cases.append(make_case(p))
    A, _ = mag_fs_pitch_batch([c[0] for c in cases], [c[1].real for c in cases], [c[1].imag for c in cases],
                              [c[2] for c in cases], u1, h, ss)
    dA = np.empty((len(steps), len(p0)))
    i = 1
    for a, st in enumerate(steps):
        for k in range(len(p0)):
            dA[a, k] = (A[i] - A[i + 1]) / (2.0 * st[k])
            i += 2
    return A[0], dA


def fd_extrapolate(dA):
    """Two central differences with half-widths (h, h/2) -> O(h^4) estimate (4 D_{h/2} - D_h)/3 and the size
    of that correction, |D_{h/2} - D_h|/3, which bounds what truncation was removed (noise is not)."""
    dA = np.asarray(dA)
    return (4.0 * dA[1] - dA[0]) / 3.0, np.abs(dA[1] - dA[0]) / 3.0


def lightcurve_case(theta, t):
    """theta = (t0, u0, tE, s, q, rho, alpha), one epoch t -> (Lens, w_c, rho) (readings G3, G4)."""
    t0, u0, tE, s, q, rho, alpha = theta
    wx, wy = trajectory(t0, u0, tE, alpha, [t])
    return lens_binary(s, q), complex(wx[0], wy[0]), rho


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

"""Thin ctypes binding of include/ulens.h: argument marshalling only, every step runs in the CUDA kernels.

PyTorch is used for device memory and streams. There is no CPU fallback: if the shared library is
missing, or no CUDA device is present when a context is created, this raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libulens.so")

ULENS_OK, ULENS_EINVAL, ULENS_ECUDA, ULENS_ENOMEM, ULENS_EUNSUPPORTED = 0, -1, -2, -3, -4
ULENS_ELIMIT = -5
ST_EA_NOCONV, ST_IMG_PARITY, ST_PATCH_CAP, ST_RES_CAP = 0x1, 0x2, 0x4, 0x8
ST_CLIPPED, ST_UNIT_OVF, ST_ERR_HIGH, ST_NO_IMAGE = 0x10, 0x20, 0x40, 0x80
ST_NIMG_SHIFT = 8
KERNEL_NAMES = ["k_traj", "k_roots", "k_limb", "k_shoot", "k_finalize", "k_sectors"]     # ULENS_K_* order

EXPORTS = ["ulens_create", "ulens_destroy", "ulens_lens_binary", "ulens_lens_triple", "ulens_mag", "ulens_mag_grad",
           "ulens_mag_host", "ulens_trajectory", "ulens_lightcurve_binary", "ulens_lightcurve_binary_host", "ulens_lightcurve_triple", "ulens_lightcurve_triple_host", "ulens_lightcurve_binary_ext", "ulens_lightcurve_binary_ext_host", "ulens_nll_marginal", "ulens_mag_point", "ulens_roots", "ulens_get_stats",
           "ulens_reset_stats", "ulens_last_launch_count", "ulens_set_timing", "ulens_get_kernel_ms", "ulens_fp64_peak", "ulens_fp32_peak", "ulens_strerror",
           "ulens_last_cuda_error", "ulens_mag_static", "ulens_static_max_points", "ulens_static_scratch_bytes",
           "ulens_static_last_cuda_error"]


ULENS_OPT_NO_RETRY = 0x1
ULENS_OPT_F32_SHOOT = 0x2
ULENS_OPT_NO_QUIET = 0x4
ULENS_ST_RETRIED = 0x2000
ULENS_ST_POINT_SRC = 0x1000


class ulens_options(C.Structure):
    _fields_ = [("n_limb", C.c_int), ("n_r", C.c_int), ("n_theta", C.c_int), ("rel_tol", C.c_double),
                ("chunk_pts", C.c_int), ("flags", C.c_int)]


class ulens_lens(C.Structure):
    _fields_ = [("n_lens", C.c_int), ("eps", C.c_double * 3), ("ax", C.c_double * 3), ("ay", C.c_double * 3)]


class ulens_stats(C.Structure):
    _fields_ = [("n_points", C.c_uint64), ("n_rays", C.c_uint64), ("n_patches", C.c_uint64),
                ("n_units", C.c_uint64), ("n_limb_solves", C.c_uint64), ("n_flagged", C.c_uint64)]


class UlensError(RuntimeError):
    pass


_lib = None


def lib() -> C.CDLL:
    """Load the in-tree shared library (fails loudly if it has not been built)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise UlensError(f"{LIB_PATH} is missing: run paper_2510_02639_b200.build.build() "
                             "(nvcc, sm_100a). There is no CPU fallback.")
        L = C.CDLL(LIB_PATH)
        vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.c_int
        L.ulens_create.argtypes = [C.POINTER(vp), ip, C.POINTER(ulens_options)]
        L.ulens_destroy.argtypes = [vp]
        L.ulens_destroy.restype = None
        L.ulens_lens_binary.argtypes = [C.POINTER(ulens_lens), C.c_double, C.c_double]
        L.ulens_lens_triple.argtypes = [C.POINTER(ulens_lens)] + [C.c_double] * 5
        L.ulens_mag.argtypes = [vp, ip, ip, C.POINTER(ulens_lens), dp, dp, vp, vp, vp, vp, vp, vp]
        L.ulens_mag_grad.argtypes = [vp, ip, ip, C.POINTER(ulens_lens), dp, dp, vp, vp, vp, vp, vp, vp, vp]
        L.ulens_mag_host.argtypes = [vp, ip, ip, C.POINTER(ulens_lens), dp, dp, vp, vp, vp, vp, vp, vp]
        L.ulens_trajectory.argtypes = [vp, ip, ip, dp, vp, vp, vp, vp]
        L.ulens_lightcurve_binary.argtypes = [vp, ip, ip, dp, C.c_double, vp, vp, vp, vp, vp, vp]
        L.ulens_lightcurve_binary_host.argtypes = [vp, ip, ip, dp, C.c_double, vp, vp, vp, vp, vp, vp]
        L.ulens_lightcurve_triple.argtypes = [vp, ip, ip, dp, C.c_double, vp, vp, vp, vp, vp, vp]
        L.ulens_lightcurve_triple_host.argtypes = [vp, ip, ip, dp, C.c_double, vp, vp, vp, vp, vp, vp]
        L.ulens_lightcurve_binary_ext.argtypes = [vp, ip, ip, dp, C.c_double, vp, vp, C.c_double, vp, vp, vp, vp,
                                                  C.POINTER(C.c_int), vp]
        L.ulens_lightcurve_binary_ext_host.argtypes = [vp, ip, ip, dp, C.c_double, vp, vp, C.c_double, vp, vp, vp, vp,
                                                       C.POINTER(C.c_int), vp]
        L.ulens_nll_marginal.argtypes = [vp, ip, ip, vp, vp, vp, vp] + [C.c_double] * 4 + [vp, vp, vp]
        L.ulens_mag_point.argtypes = [vp, ip, ip, C.POINTER(ulens_lens), vp, vp, vp, vp, vp]
        L.ulens_roots.argtypes = [vp, C.POINTER(ulens_lens), ip, vp, vp, vp, vp, vp, vp]
        L.ulens_get_stats.argtypes = [vp, C.POINTER(ulens_stats)]
        L.ulens_reset_stats.argtypes = [vp]
        L.ulens_last_launch_count.argtypes = [vp]
        L.ulens_set_timing.argtypes = [vp, ip]
        L.ulens_get_kernel_ms.argtypes = [vp, ip, dp, C.POINTER(C.c_int)]
        L.ulens_fp64_peak.argtypes = [vp, C.c_double, dp]
        L.ulens_fp32_peak.argtypes = [vp, C.c_double, dp]
        L.ulens_strerror.argtypes = [ip]
        L.ulens_strerror.restype = C.c_char_p
        L.ulens_last_cuda_error.argtypes = [vp]
        L.ulens_last_cuda_error.restype = C.c_char_p
        L.ulens_mag_static.argtypes = [ip, ip, ip, C.POINTER(ulens_lens), dp, dp, vp, vp, vp, vp, vp, vp]
        L.ulens_static_max_points.argtypes = []
        L.ulens_static_scratch_bytes.argtypes = []
        L.ulens_static_scratch_bytes.restype = C.c_longlong
        L.ulens_static_last_cuda_error.argtypes = []
        L.ulens_static_last_cuda_error.restype = C.c_char_p
        _lib = L
    return _lib


def _check(rc: int, ctx=None):
    if rc != ULENS_OK:
        msg = lib().ulens_strerror(rc).decode()
        if rc == ULENS_ECUDA and ctx is not None:
            msg += ": " + lib().ulens_last_cuda_error(ctx).decode()
        raise UlensError(f"ulens error {rc}: {msg}")


def ulens_lens_binary(s: float, q: float) -> ulens_lens:
    L = ulens_lens()
    _check(lib().ulens_lens_binary(C.byref(L), s, q))
    return L


def ulens_lens_triple(s, q, q3, r3, psi) -> ulens_lens:
    L = ulens_lens()
    _check(lib().ulens_lens_triple(C.byref(L), s, q, q3, r3, psi))
    return L


def lens_single() -> ulens_lens:
    L = ulens_lens()
    L.n_lens = 1
    L.eps[0] = 1.0
    return L


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _dev(t, dtype, n):
    """Device pointer of a contiguous CUDA tensor of the right dtype and size (or None)."""
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous() or t.dtype != dtype or t.numel() != n:
        raise UlensError("expected a contiguous CUDA tensor of dtype %s with %d elements" % (dtype, n))
    return C.c_void_p(t.data_ptr())


def ulens_static_max_points() -> int:
    return int(lib().ulens_static_max_points())


def ulens_static_scratch_bytes() -> int:
    return int(lib().ulens_static_scratch_bytes())


def ulens_mag_static(device: int, lenses, rho, u1, w_re, w_im, A_out, err_out=None, status_out=None, stream=None):
    """ulens_mag_static (include/ulens.h): ulens_mag without a context and without any allocation -- the caller
    passes the inputs AND the outputs (CUDA tensors [n_cfg, n_pts]: float64, float64, int32), at most
    ulens_static_max_points() points per call. `stream`: a torch.cuda.Stream (default: the device's current one).
    Enqueue-only. Calls on one device share one scratch array: keep them on one stream."""
    import torch
    n_cfg, arr, rho, u1 = Context._cfg_arrays(lenses, rho, u1)
    n_pts = w_re.numel() // max(n_cfg, 1)
    n = n_cfg * n_pts
    if stream is None:
        stream = torch.cuda.current_stream(device)
    rc = lib().ulens_mag_static(int(device), n_cfg, n_pts, arr, _dptr(rho), _dptr(u1),
                                _dev(w_re, torch.float64, n), _dev(w_im, torch.float64, n),
                                _dev(A_out, torch.float64, n), _dev(err_out, torch.float64, n),
                                _dev(status_out, torch.int32, n), C.c_void_p(stream.cuda_stream))
    if rc != ULENS_OK:
        msg = lib().ulens_strerror(rc).decode()
        if rc == ULENS_ECUDA:
            msg += ": " + lib().ulens_static_last_cuda_error().decode()
        raise UlensError(f"ulens error {rc}: {msg}")
    return A_out, err_out, status_out


class Context:
    """ulens_ctx: one device, one stream at a time. Methods mirror the C entry points."""

    def __init__(self, device: int = 0, n_limb: int = 0, n_r: int = 0, n_theta: int = 0, rel_tol: float = 0.0,
                 chunk_pts: int = 0, flags: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise UlensError("no CUDA device: the ulens hot path has no CPU fallback")
        self._torch = torch
        self.device = device
        opt = ulens_options(n_limb, n_r, n_theta, rel_tol, chunk_pts, flags)
        self._h = C.c_void_p()
        _check(lib().ulens_create(C.byref(self._h), device, C.byref(opt)))

    def close(self):
        if getattr(self, "_h", None):
            lib().ulens_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _stream(self, stream):
        if stream is None:
            stream = self._torch.cuda.current_stream(self.device)
        return C.c_void_p(stream.cuda_stream)

    @staticmethod
    def _cfg_arrays(lenses, rho, u1):
        lenses = list(lenses)
        n_cfg = len(lenses)
        arr = (ulens_lens * max(n_cfg, 1))(*lenses)
        rho = np.ascontiguousarray(np.broadcast_to(np.asarray(rho, dtype=np.float64), (n_cfg,)))
        u1 = np.ascontiguousarray(np.broadcast_to(np.asarray(u1, dtype=np.float64), (n_cfg,)))
        return n_cfg, arr, rho, u1

    def ulens_mag(self, lenses, rho, u1, w_re, w_im, A_out=None, err_out=None, status_out=None, stream=None):
        """w_re, w_im: CUDA float64 tensors [n_cfg, n_pts]. Returns (A, err, status) CUDA tensors. No sync."""
        torch = self._torch
        n_cfg, arr, rho, u1 = self._cfg_arrays(lenses, rho, u1)
        n_pts = w_re.numel() // max(n_cfg, 1)
        n = n_cfg * n_pts
        dev = w_re.device
        if A_out is None:
            A_out = torch.empty((n_cfg, n_pts), dtype=torch.float64, device=dev)
        if err_out is None:
            err_out = torch.empty((n_cfg, n_pts), dtype=torch.float64, device=dev)
        if status_out is None:
            status_out = torch.empty((n_cfg, n_pts), dtype=torch.int32, device=dev)
        _check(lib().ulens_mag(self._h, n_cfg, n_pts, arr, _dptr(rho), _dptr(u1),
                               _dev(w_re, torch.float64, n), _dev(w_im, torch.float64, n),
                               _dev(A_out, torch.float64, n), _dev(err_out, torch.float64, n),
                               _dev(status_out, torch.int32, n), self._stream(stream)), self._h)
        return A_out, err_out, status_out

    def ulens_mag_grad(self, lenses, rho, u1, w_re, w_im, stream=None):
        """As ulens_mag, plus dA/d(w_cx, w_cy, s, q, rho) (n_lens = 1, 2: [n_cfg, n_pts, 5]) or
        dA/d(w_cx, w_cy, s, q, q3, r3, psi, rho) (n_lens = 3: [n_cfg, n_pts, 8]): returns (A, dA, err, status)."""
        torch = self._torch
        n_cfg, arr, rho, u1 = self._cfg_arrays(lenses, rho, u1)
        n_pts = w_re.numel() // max(n_cfg, 1)
        n = n_cfg * n_pts
        dev = w_re.device
        nt = 8 if (n_cfg and arr[0].n_lens == 3) else 5
        A = torch.empty((n_cfg, n_pts), dtype=torch.float64, device=dev)
        dA = torch.empty((n_cfg, n_pts, nt), dtype=torch.float64, device=dev)
        err = torch.empty((n_cfg, n_pts), dtype=torch.float64, device=dev)
        st = torch.empty((n_cfg, n_pts), dtype=torch.int32, device=dev)
        _check(lib().ulens_mag_grad(self._h, n_cfg, n_pts, arr, _dptr(rho), _dptr(u1),
                                    _dev(w_re, torch.float64, n), _dev(w_im, torch.float64, n),
                                    _dev(A, torch.float64, n), _dev(dA, torch.float64, nt * n),
                                    _dev(err, torch.float64, n), _dev(st, torch.int32, n), self._stream(stream)), self._h)
        return A, dA, err, st

    def ulens_mag_host(self, lenses, rho, u1, w_re, w_im, A=None, err=None, st=None, stream=None):
        """Host numpy arrays in / out (optionally caller-provided, e.g. views of pinned tensors); the
        copies and the synchronisation happen inside the C call."""
        n_cfg, arr, rho, u1 = self._cfg_arrays(lenses, rho, u1)
        w_re = np.ascontiguousarray(w_re, dtype=np.float64)
        w_im = np.ascontiguousarray(w_im, dtype=np.float64)
        n_pts = w_re.size // max(n_cfg, 1)
        A = np.empty((n_cfg, n_pts)) if A is None else A
        err = np.empty((n_cfg, n_pts)) if err is None else err
        st = np.empty((n_cfg, n_pts), dtype=np.uint32) if st is None else st
        for a, dt in ((A, np.float64), (err, np.float64)):
            if a.dtype != dt or not a.flags.c_contiguous or a.size != n_cfg * n_pts:
                raise UlensError("output arrays must be C-contiguous float64 of n_cfg*n_pts elements")
        if st.dtype.itemsize != 4 or not st.flags.c_contiguous or st.size != n_cfg * n_pts:
            raise UlensError("status array must be C-contiguous 32-bit of n_cfg*n_pts elements")
        _check(lib().ulens_mag_host(self._h, n_cfg, n_pts, arr, _dptr(rho), _dptr(u1),
                                    w_re.ctypes.data_as(C.c_void_p), w_im.ctypes.data_as(C.c_void_p),
                                    A.ctypes.data_as(C.c_void_p), err.ctypes.data_as(C.c_void_p),
                                    st.ctypes.data_as(C.c_void_p), self._stream(stream)), self._h)
        return A, err, st

    def ulens_trajectory(self, theta, t, stream=None):
        """Step a1 alone: theta host [n_cfg, 7], t CUDA float64 [n_epochs] -> (w_re, w_im) CUDA [n_cfg, n_epochs]."""
        torch = self._torch
        theta = np.ascontiguousarray(theta, dtype=np.float64).reshape(-1, 7)
        n_cfg, n_ep = theta.shape[0], t.numel()
        w_re = torch.empty((n_cfg, n_ep), dtype=torch.float64, device=t.device)
        w_im = torch.empty((n_cfg, n_ep), dtype=torch.float64, device=t.device)
        _check(lib().ulens_trajectory(self._h, n_cfg, n_ep, _dptr(theta), _dev(t, torch.float64, n_ep),
                                      _dev(w_re, torch.float64, n_cfg * n_ep), _dev(w_im, torch.float64, n_cfg * n_ep),
                                      self._stream(stream)), self._h)
        return w_re, w_im

    def ulens_lightcurve_binary(self, theta, u1, t, want_dA=False, stream=None, out=None):
        """theta: host [n_cfg, 7] (t0,u0,tE,s,q,rho,alpha); t: CUDA float64 [n_epochs];
        out: optional caller-owned CUDA tensors (A, dA, err, st) to write into."""
        torch = self._torch
        theta = np.ascontiguousarray(theta, dtype=np.float64).reshape(-1, 7)
        n_cfg, n_ep = theta.shape[0], t.numel()
        dev = t.device
        if out is not None:
            A, dA, err, st = out
            want_dA = dA is not None
        else:
            A = torch.empty((n_cfg, n_ep), dtype=torch.float64, device=dev)
            err = torch.empty((n_cfg, n_ep), dtype=torch.float64, device=dev)
            st = torch.empty((n_cfg, n_ep), dtype=torch.int32, device=dev)
            dA = torch.empty((n_cfg, n_ep, 7), dtype=torch.float64, device=dev) if want_dA else None
        _check(lib().ulens_lightcurve_binary(self._h, n_cfg, n_ep, _dptr(theta), float(u1),
                                             _dev(t, torch.float64, n_ep), _dev(A, torch.float64, n_cfg * n_ep),
                                             _dev(dA, torch.float64, n_cfg * n_ep * 7) if want_dA else None,
                                             _dev(err, torch.float64, n_cfg * n_ep),
                                             _dev(st, torch.int32, n_cfg * n_ep), self._stream(stream)), self._h)
        return A, dA, err, st

    def ulens_lightcurve_triple(self, theta, u1, t, want_dA=False, stream=None):
        """theta: host [n_cfg, 10] (t0,u0,tE,s,q,rho,alpha,q3,r3,psi); t: CUDA float64 [n_epochs].
        Returns (A, dA [n_cfg, n_epochs, 10] or None, err, st)."""
        torch = self._torch
        theta = np.ascontiguousarray(theta, dtype=np.float64).reshape(-1, 10)
        n_cfg, n_ep = theta.shape[0], t.numel()
        dev = t.device
        A = torch.empty((n_cfg, n_ep), dtype=torch.float64, device=dev)
        err = torch.empty((n_cfg, n_ep), dtype=torch.float64, device=dev)
        st = torch.empty((n_cfg, n_ep), dtype=torch.int32, device=dev)
        dA = torch.empty((n_cfg, n_ep, 10), dtype=torch.float64, device=dev) if want_dA else None
        _check(lib().ulens_lightcurve_triple(self._h, n_cfg, n_ep, _dptr(theta), float(u1),
                                             _dev(t, torch.float64, n_ep), _dev(A, torch.float64, n_cfg * n_ep),
                                             _dev(dA, torch.float64, n_cfg * n_ep * 10) if want_dA else None,
                                             _dev(err, torch.float64, n_cfg * n_ep),
                                             _dev(st, torch.int32, n_cfg * n_ep), self._stream(stream)), self._h)
        return A, dA, err, st

    def ulens_lightcurve_triple_host(self, theta, u1, t, A, dA=None, err=None, st=None, stream=None):
        """Host numpy arrays in / out: t [n_epochs]; A, err [n_cfg, n_epochs]; dA [n_cfg, n_epochs, 10] or None; st 32-bit."""
        theta = np.ascontiguousarray(theta, dtype=np.float64).reshape(-1, 10)
        t = np.ascontiguousarray(t, dtype=np.float64)
        n_cfg, n_ep = theta.shape[0], t.size
        for a, k in ((A, 1), (dA, 10), (err, 1)):
            if a is not None and (a.dtype != np.float64 or not a.flags.c_contiguous or a.size != k * n_cfg * n_ep):
                raise UlensError("output arrays must be C-contiguous float64 of the documented size")
        if st is not None and (st.dtype.itemsize != 4 or not st.flags.c_contiguous or st.size != n_cfg * n_ep):
            raise UlensError("status array must be C-contiguous 32-bit of n_cfg*n_epochs elements")
        p = lambda a: a.ctypes.data_as(C.c_void_p) if a is not None else None
        _check(lib().ulens_lightcurve_triple_host(self._h, n_cfg, n_ep, _dptr(theta), float(u1), p(t), p(A), p(dA),
                                                  p(err), p(st), self._stream(stream)), self._h)
        return A, dA, err, st

    def ulens_lightcurve_binary_ext(self, theta, u1, t, ext_mask=None, sel_tol=0.0, want_dA=False, stream=None):
        """Light curve with the point-source / finite-source switch. ext_mask: CUDA uint8 [n_cfg, n_epochs]
        (non-zero = finite-source epoch) or None (the library selects with sel_tol). Returns (A, dA, err, st, n_ext)."""
        torch = self._torch
        theta = np.ascontiguousarray(theta, dtype=np.float64).reshape(-1, 7)
        n_cfg, n_ep = theta.shape[0], t.numel()
        dev = t.device
        A = torch.empty((n_cfg, n_ep), dtype=torch.float64, device=dev)
        err = torch.empty((n_cfg, n_ep), dtype=torch.float64, device=dev)
        st = torch.empty((n_cfg, n_ep), dtype=torch.int32, device=dev)
        dA = torch.empty((n_cfg, n_ep, 7), dtype=torch.float64, device=dev) if want_dA else None
        n_ext = C.c_int(0)
        _check(lib().ulens_lightcurve_binary_ext(self._h, n_cfg, n_ep, _dptr(theta), float(u1),
                                                 _dev(t, torch.float64, n_ep),
                                                 _dev(ext_mask, torch.uint8, n_cfg * n_ep) if ext_mask is not None else None,
                                                 float(sel_tol), _dev(A, torch.float64, n_cfg * n_ep),
                                                 _dev(dA, torch.float64, n_cfg * n_ep * 7) if want_dA else None,
                                                 _dev(err, torch.float64, n_cfg * n_ep),
                                                 _dev(st, torch.int32, n_cfg * n_ep), C.byref(n_ext),
                                                 self._stream(stream)), self._h)
        return A, dA, err, st, n_ext.value

    def ulens_mag_point(self, lenses, w_re, w_im, stream=None):
        """Point-source magnification sum 1/|det J| (Eq. 2-3): returns (A [n_cfg, n_pts], status)."""
        torch = self._torch
        lenses = list(lenses)
        n_cfg = len(lenses)
        arr = (ulens_lens * n_cfg)(*lenses)
        n_pts = w_re.numel() // max(n_cfg, 1)
        n = n_cfg * n_pts
        A = torch.empty((n_cfg, n_pts), dtype=torch.float64, device=w_re.device)
        st = torch.empty((n_cfg, n_pts), dtype=torch.int32, device=w_re.device)
        _check(lib().ulens_mag_point(self._h, n_cfg, n_pts, arr, _dev(w_re, torch.float64, n), _dev(w_im, torch.float64, n),
                                     _dev(A, torch.float64, n), _dev(st, torch.int32, n), self._stream(stream)), self._h)
        return A, st

    def ulens_lightcurve_binary_host(self, theta, u1, t, A, dA=None, err=None, st=None, stream=None):
        """Host numpy arrays in / out (e.g. views of pinned tensors): t [n_epochs]; A, err [n_cfg, n_epochs];
        dA [n_cfg, n_epochs, 7] or None; st 32-bit. The copies and the synchronisation happen inside the C call."""
        theta = np.ascontiguousarray(theta, dtype=np.float64).reshape(-1, 7)
        t = np.ascontiguousarray(t, dtype=np.float64)
        n_cfg, n_ep = theta.shape[0], t.size
        for a, k in ((A, 1), (dA, 7), (err, 1)):
            if a is not None and (a.dtype != np.float64 or not a.flags.c_contiguous or a.size != k * n_cfg * n_ep):
                raise UlensError("output arrays must be C-contiguous float64 of the documented size")
        if st is not None and (st.dtype.itemsize != 4 or not st.flags.c_contiguous or st.size != n_cfg * n_ep):
            raise UlensError("status array must be C-contiguous 32-bit of n_cfg*n_epochs elements")
        p = lambda a: a.ctypes.data_as(C.c_void_p) if a is not None else None
        _check(lib().ulens_lightcurve_binary_host(self._h, n_cfg, n_ep, _dptr(theta), float(u1), p(t), p(A), p(dA),
                                                  p(err), p(st), self._stream(stream)), self._h)
        return A, dA, err, st

    def ulens_lightcurve_binary_ext_host(self, theta, u1, t, A, dA=None, err=None, st=None, ext_mask=None, sel_tol=0.0,
                                         stream=None):
        """Host numpy arrays in / out as ulens_lightcurve_binary_host; ext_mask uint8 [n_cfg, n_epochs] or None
        (library selection). Returns (A, dA, err, st, n_ext)."""
        theta = np.ascontiguousarray(theta, dtype=np.float64).reshape(-1, 7)
        t = np.ascontiguousarray(t, dtype=np.float64)
        n_cfg, n_ep = theta.shape[0], t.size
        for a, k in ((A, 1), (dA, 7), (err, 1)):
            if a is not None and (a.dtype != np.float64 or not a.flags.c_contiguous or a.size != k * n_cfg * n_ep):
                raise UlensError("output arrays must be C-contiguous float64 of the documented size")
        if st is not None and (st.dtype.itemsize != 4 or not st.flags.c_contiguous or st.size != n_cfg * n_ep):
            raise UlensError("status array must be C-contiguous 32-bit of n_cfg*n_epochs elements")
        if ext_mask is not None and (ext_mask.dtype != np.uint8 or not ext_mask.flags.c_contiguous or ext_mask.size != n_cfg * n_ep):
            raise UlensError("ext_mask must be C-contiguous uint8 of n_cfg*n_epochs elements")
        p = lambda a: a.ctypes.data_as(C.c_void_p) if a is not None else None
        n_ext = C.c_int(0)
        _check(lib().ulens_lightcurve_binary_ext_host(self._h, n_cfg, n_ep, _dptr(theta), float(u1), p(t), p(ext_mask),
                                                      float(sel_tol), p(A), p(dA), p(err), p(st), C.byref(n_ext),
                                                      self._stream(stream)), self._h)
        return A, dA, err, st, n_ext.value

    def ulens_nll_marginal(self, A, dA, flux, sigma, mu_fs, mu_fb, var_fs, var_fb, stream=None):
        """Marginalised-flux NLL per light curve (App. B.2) and, with dA, its gradient: (nll [n_cfg], grad [n_cfg, 7] or None)."""
        torch = self._torch
        n_cfg, n_ep = A.shape
        nll = torch.empty(n_cfg, dtype=torch.float64, device=A.device)
        grad = torch.empty((n_cfg, 7), dtype=torch.float64, device=A.device) if dA is not None else None
        _check(lib().ulens_nll_marginal(self._h, n_cfg, n_ep, _dev(A, torch.float64, n_cfg * n_ep),
                                        _dev(dA, torch.float64, n_cfg * n_ep * 7) if dA is not None else None,
                                        _dev(flux, torch.float64, n_ep), _dev(sigma, torch.float64, n_ep),
                                        float(mu_fs), float(mu_fb), float(var_fs), float(var_fb),
                                        _dev(nll, torch.float64, n_cfg), _dev(grad, torch.float64, n_cfg * 7) if grad is not None else None,
                                        self._stream(stream)), self._h)
        return nll, grad

    def ulens_roots(self, lens, w_re, w_im, stream=None):
        """All N^2+1 roots per source position and the image flags: (roots complex [n, deg], is_image bool)."""
        torch = self._torch
        n = w_re.numel()
        deg = lens.n_lens ** 2 + 1
        rr = torch.empty((n, deg), dtype=torch.float64, device=w_re.device)
        ri = torch.empty((n, deg), dtype=torch.float64, device=w_re.device)
        im = torch.empty((n, deg), dtype=torch.uint8, device=w_re.device)
        _check(lib().ulens_roots(self._h, C.byref(lens), n, _dev(w_re, torch.float64, n), _dev(w_im, torch.float64, n),
                                 _dev(rr, torch.float64, n * deg), _dev(ri, torch.float64, n * deg),
                                 _dev(im, torch.uint8, n * deg), self._stream(stream)), self._h)
        return torch.complex(rr, ri), im.bool()

    def ulens_get_stats(self) -> dict:
        s = ulens_stats()
        _check(lib().ulens_get_stats(self._h, C.byref(s)), self._h)
        return {k: int(getattr(s, k)) for k, _ in ulens_stats._fields_}

    def ulens_reset_stats(self):
        _check(lib().ulens_reset_stats(self._h), self._h)

    def ulens_last_launch_count(self) -> int:
        return int(lib().ulens_last_launch_count(self._h))

    def ulens_set_timing(self, on: bool):
        _check(lib().ulens_set_timing(self._h, int(bool(on))), self._h)

    def ulens_get_kernel_ms(self) -> dict:
        """{kernel name: (total device ms, launches)} since ulens_set_timing(True). Synchronises."""
        out = {}
        for which, name in enumerate(KERNEL_NAMES):
            ms, n = C.c_double(), C.c_int()
            _check(lib().ulens_get_kernel_ms(self._h, which, C.byref(ms), C.byref(n)), self._h)
            out[name] = (ms.value, n.value)
        return out

    def ulens_fp32_peak(self, ms: float = 200.0) -> float:
        out = C.c_double()
        _check(lib().ulens_fp32_peak(self._h, ms, C.byref(out)), self._h)
        return out.value

    def ulens_fp64_peak(self, ms: float = 200.0) -> float:
        out = C.c_double()
        _check(lib().ulens_fp64_peak(self._h, ms, C.byref(out)), self._h)
        return out.value

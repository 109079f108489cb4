"""The C-ABI library builds for sm_100a, loads, and exports every symbol include/ulens.h declares.
No compute call is made here (no GPU on the CPU test box)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built_lib():
    from paper_2510_02639_b200 import build
    return build.build()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "ulens.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ulens_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_boundary():
    syms = declared_symbols()
    for s in ["ulens_create", "ulens_destroy", "ulens_mag", "ulens_mag_host", "ulens_lightcurve_binary", "ulens_lightcurve_binary_host", "ulens_roots",
              "ulens_get_stats", "ulens_strerror", "ulens_lens_binary", "ulens_lens_triple", "ulens_fp64_peak"]:
        assert s in syms


def test_library_exports_every_declared_symbol(built_lib):
    lib = C.CDLL(built_lib)
    for s in declared_symbols():
        assert hasattr(lib, s), s
    from paper_2510_02639_b200 import binding
    assert sorted(binding.EXPORTS) == declared_symbols()


def test_host_geometry_helpers(built_lib):
    """ulens_lens_binary / ulens_lens_triple are host-only: readings G4 / G5."""
    from paper_2510_02639_b200 import binding
    L = binding.ulens_lens_binary(1.3, 0.2)
    assert L.n_lens == 2
    assert abs(L.eps[0] + L.eps[1] - 1) < 1e-15 and abs(L.eps[1] / L.eps[0] - 0.2) < 1e-15
    assert abs(L.eps[0] * L.ax[0] + L.eps[1] * L.ax[1]) < 1e-15          # barycentre at the origin
    assert abs((L.ax[1] - L.ax[0]) - 1.3) < 1e-15 and L.ax[0] < 0 < L.ax[1]
    T = binding.ulens_lens_triple(1.3, 0.2, 0.03, 1.24, 1.3)
    assert T.n_lens == 3 and abs(sum(T.eps) - 1) < 1e-15
    mid = 0.5 * (T.ax[0] + T.ax[1])
    import math
    assert abs(math.hypot(T.ax[2] - mid, T.ay[2]) - 1.24) < 1e-15
    for bad in [(-1.0, 0.1), (1.0, 0.0), (float("nan"), 0.1), (1.0, float("inf"))]:
        with pytest.raises(binding.UlensError):
            binding.ulens_lens_binary(*bad)
    assert binding.lib().ulens_strerror(-1) == b"invalid argument"


def test_no_gpu_means_loud_failure(built_lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2510_02639_b200 import binding
    with pytest.raises(binding.UlensError):
        binding.Context(0)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2510_02639_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".hpp", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "ulens_oracle" not in txt, f


def test_static_entry_argument_checks_need_no_gpu(built_lib):
    """ulens_mag_static (the no-allocation entry) checks its sizes before it touches CUDA: a request beyond the fixed scratch is
    refused with ULENS_ELIMIT, bad arguments with ULENS_EINVAL, an empty request succeeds -- with or without a device."""
    from paper_2510_02639_b200 import binding
    lib = binding.lib()
    cap = binding.ulens_static_max_points()
    assert cap == 128 and 0 < binding.ulens_static_scratch_bytes() <= 8 << 20
    L = (binding.ulens_lens * 3)(*[binding.ulens_lens_binary(1.0, 0.1)] * 3)
    rho = (C.c_double * 3)(0.01, 0.01, 0.01)
    u1 = (C.c_double * 3)(0.3, 0.3, 0.3)
    fake = C.c_void_p(0x1000)                               # never dereferenced: every call below returns before any work
    dp = C.POINTER(C.c_double)
    call = lambda dev, n_cfg, n_pts, w=fake, out=fake: lib.ulens_mag_static(dev, n_cfg, n_pts, L, C.cast(rho, dp), C.cast(u1, dp),
                                                                          w, w, out, None, None, None)
    assert call(0, 1, cap + 1) == binding.ULENS_ELIMIT
    assert call(0, 3, 43) == binding.ULENS_ELIMIT           # n_cfg x n_pts counts
    assert b"ULENS_STATIC_MAX_POINTS" in lib.ulens_strerror(binding.ULENS_ELIMIT)
    assert call(-1, 1, 4) == binding.ULENS_EINVAL
    assert call(0, -1, 4) == binding.ULENS_EINVAL
    assert call(0, 1, 4, w=None) == binding.ULENS_EINVAL
    assert call(0, 1, 4, out=None) == binding.ULENS_EINVAL
    assert call(0, 0, 4) == binding.ULENS_OK and call(0, 1, 0) == binding.ULENS_OK

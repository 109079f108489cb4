"""Mixed-precision ray shooting (ULENS_OPT_F32_SHOOT): the FP32-pipe kernel against the same references
as the FP64 path, at the same bar (1e-4 relative, BASELINE north_star / P:40). Needs a B200."""
import math
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu
TOL_A = 1e-4
HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def ctx32(torch_cuda):
    from paper_2510_02639_b200 import binding, build
    build.build()
    c = binding.Context(0, flags=binding.ULENS_OPT_F32_SHOOT)
    yield c
    c.close()


def _mag(ctx, torch, lenses, rho, u1, w):
    w = np.atleast_2d(np.asarray(w, dtype=complex))
    wre = torch.tensor(np.ascontiguousarray(w.real), device="cuda:0")
    wim = torch.tensor(np.ascontiguousarray(w.imag), device="cuda:0")
    A, err, st = ctx.ulens_mag(lenses, rho, u1, wre, wim)
    torch.cuda.synchronize()
    return A.cpu().numpy(), err.cpu().numpy(), st.cpu().numpy().astype(np.uint32)


@pytest.mark.parametrize("u,rho,u1", [(0.3, 0.05, 0.0), (0.02, 0.05, 0.0), (1.2, 0.3, 0.0), (0.011, 0.01, 0.0), (0.3, 0.05, 0.5),
                                      (0.03, 0.05, 1.0), (0.2, 0.1, 0.3), (0.0005, 0.05, 0.5), (0.4, 1e-3, 0.5), (0.0, 1e-3, 0.0)])
def test_single_lens_closed_forms_f32(ctx32, torch_cuda, u, rho, u1):
    from paper_2510_02639_b200 import binding
    from test_oracle_pins import A_ld_single, A_witt_mao
    if u == 0.0:
        ref = math.sqrt(1 + 4 / rho ** 2)
    else:
        ref = float(A_ld_single(u, rho, u1)) if u1 > 0 else float(A_witt_mao(u, rho))
    w = u * complex(math.cos(0.83), math.sin(0.83))
    A, _, _ = _mag(ctx32, torch_cuda, [binding.lens_single()], [rho], [u1], [[w]])
    assert abs(A[0, 0] / ref - 1) < 5e-5, (A[0, 0], ref)


def test_config0_all_points_f32(ctx32, ctx, torch_cuda, oracle):
    from paper_2510_02639_b200 import binding, inputs
    wl = inputs.get(0)
    L = binding.ulens_lens_binary(1.0, 0.01)
    A32, _, st32 = _mag(ctx32, torch_cuda, [L], wl.rho, wl.u1, wl.w)
    A64, _, st64 = _mag(ctx, torch_cuda, [L], wl.rho, wl.u1, wl.w)
    ref = oracle.mag_fs_batch([oracle.lens_binary(1.0, 0.01)], 0, wl.w[0].real, wl.w[0].imag, wl.rho[0], wl.u1[0], 100, 8)
    adm = ref["err_est"] <= 2e-5
    rel = np.abs(A32[0] / ref["A"] - 1)
    print("C0 FP32-pipe path: max |A/A_oracle - 1| = %.1e over %d admissible points; max |A32/A64 - 1| = %.1e"
          % (rel[adm].max(), adm.sum(), np.abs(A32 / A64 - 1).max()))
    assert adm.sum() >= 495 and rel[adm].max() <= TOL_A
    assert np.array_equal(st32, st64)                     # same sectors, same flags


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_stored_oracle_sample_full_size_f32(torch_cuda, cfg):
    """BASELINE C1-C3 at full size through the FP32-pipe kernel against the stored oracle sample (as
    test_gpu_golden.test_stored_oracle_sample_full_size does for the FP64 kernel)."""
    from paper_2510_02639_b200 import binding, inputs
    torch = torch_cuda
    wl = inputs.get(cfg)
    f = binding.ulens_lens_binary if wl.kind == "binary" else binding.ulens_lens_triple
    c = binding.Context(0, flags=binding.ULENS_OPT_F32_SHOOT)
    w_re = torch.tensor(np.ascontiguousarray(wl.w.real), device="cuda:0")
    w_im = torch.tensor(np.ascontiguousarray(wl.w.imag), device="cuda:0")
    A, err, st = c.ulens_mag([f(*p) for p in wl.lens_params], wl.rho, wl.u1, w_re, w_im)
    torch.cuda.synchronize()
    A = A.cpu().numpy(); st = st.cpu().numpy().astype(np.uint32)
    c.close()
    g = np.load(os.path.join(HERE, "golden", "oracle_C%d.npz" % cfg))
    ci, pi = g["cfg_index"], g["point_index"]
    adm = g["err_est"] <= 2e-5
    rel = np.abs(A[ci, pi] / g["A"] - 1)
    clean = adm & ((st[ci, pi] & 0xff) == 0)
    bad = clean & ~(rel <= TOL_A)
    print("C%d FP32-pipe path, stored oracle sample: %d points, clean %d: median %.1e  p99 %.1e  max %.1e, > 1e-4: %d; flagged in the "
          "whole workload %d" % (cfg, len(ci), clean.sum(), np.median(rel[clean]), np.quantile(rel[clean], 0.99), rel[clean].max(),
                                 bad.sum(), ((st & 0xff) != 0).sum()))
    assert np.all(np.isfinite(A))
    assert not bad.any(), list(zip(ci[bad][:8], pi[bad][:8], rel[bad][:8]))

"""ulens_mag_point (Eq. 2-3): point-source magnification from the images of step a2. Needs a B200."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _dev(torch, w):
    w = np.atleast_2d(np.asarray(w, dtype=complex))
    return (torch.tensor(np.ascontiguousarray(w.real), device="cuda:0"),
            torch.tensor(np.ascontiguousarray(w.imag), device="cuda:0"))


def test_single_lens_closed_form(ctx, torch_cuda):
    """A = (u^2 + 2) / (u sqrt(u^2 + 4)) for one point mass."""
    from paper_2510_02639_b200 import binding
    u = np.geomspace(1e-3, 30.0, 257)
    w = u * np.exp(1j * np.linspace(0, 6.0, u.size))
    A, st = ctx.ulens_mag_point([binding.lens_single()], *_dev(torch_cuda, w))
    torch_cuda.cuda.synchronize()
    ref = (u * u + 2) / (u * np.sqrt(u * u + 4))
    assert np.max(np.abs(A.cpu().numpy()[0] / ref - 1)) < 1e-12
    assert np.all(((st.cpu().numpy()[0] >> 8) & 0xf) == 2)


@pytest.mark.parametrize("kind", ["binary", "triple"])
def test_against_oracle_images(ctx, torch_cuda, oracle, kind):
    """sum 1/|det J| over the oracle's extended-precision images (a different polynomial, a different solver)."""
    from paper_2510_02639_b200 import binding
    if kind == "binary":
        lens, olens = binding.ulens_lens_binary(0.9, 0.03), oracle.lens_binary(0.9, 0.03)
    else:
        lens, olens = binding.ulens_lens_triple(1.1, 0.5, 0.03, 1.24, 1.3), oracle.lens_triple(1.1, 0.5, 0.03, 1.24, 1.3)
    rng = np.random.default_rng(17)
    n = 300
    w = rng.uniform(-1.3, 1.3, n) + 1j * rng.uniform(-1.3, 1.3, n)
    A, st = ctx.ulens_mag_point([lens], *_dev(torch_cuda, w))
    torch_cuda.cuda.synchronize()
    A = A.cpu().numpy()[0]
    n_cmp = 0
    for k in range(n):
        r = oracle.roots(olens, complex(w[k]))
        dj = np.abs(r["detJ"][r["is_image"]])
        if dj.min() < 1e-4:                       # within ~1e-8 of a caustic: 1/|det J| is ill-conditioned
            continue
        ref = float(np.sum(1.0 / dj))
        assert abs(A[k] / ref - 1) < 1e-9, (k, A[k], ref)
        assert abs(ref - oracle.mag_point_source(olens, complex(w[k]))) < 1e-9 * ref
        n_cmp += 1
    assert n_cmp > 0.95 * n


def test_small_source_limit_of_the_finite_source_path(ctx, torch_cuda):
    """rho -> 0: the ray-shooting path tends to the point-source sum (O(rho^2) correction away from caustics)."""
    from paper_2510_02639_b200 import binding
    torch = torch_cuda
    L = binding.ulens_lens_binary(1.2, 0.2)
    rng = np.random.default_rng(23)
    w = rng.uniform(0.4, 1.5, 64) * np.exp(1j * rng.uniform(0, 2 * math.pi, 64))
    wre, wim = _dev(torch, w)
    A_ps, _ = ctx.ulens_mag_point([L], wre, wim)
    A_fs, _, _ = ctx.ulens_mag([L], [1e-4], [0.0], wre, wim)
    torch.cuda.synchronize()
    A_ps, A_fs = A_ps.cpu().numpy()[0], A_fs.cpu().numpy()[0]
    quiet = A_ps < 20                                # not within a few rho of a caustic
    assert quiet.sum() > 50
    assert np.max(np.abs(A_fs[quiet] / A_ps[quiet] - 1)) < 1e-4      # the finite-source path's own bar

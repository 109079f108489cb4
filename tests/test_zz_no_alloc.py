"""ulens_mag_static (include/ulens.h, "no-allocation entry"): the finite-source magnification with its whole
workspace in one file-scope device array, for callers that cannot call cudaMalloc. Needs a B200.

The file sorts last on purpose (pytest -x: a failure here hides nothing after it). The new entry is
compared with the existing path -- ulens_mag on a context with ULENS_OPT_NO_RETRY, the same operation -- on two
calls in a row with DIFFERENT inputs, so the second call runs on the scratch the first one left behind; then the first
input once more. Both orders of use are covered: alone in a fresh process and after every other GPU test.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

RTOL = 1e-12          # same kernels, same arithmetic, another chunk size: the tests of the path itself use 1e-4 vs the oracle


def _case(binding, kind, seed, n_cfg, n_pts):
    rng = np.random.default_rng(seed)
    if kind == "binary":
        lenses = [binding.ulens_lens_binary(float(rng.uniform(0.7, 1.4)), float(10 ** rng.uniform(-3, 0))) for _ in range(n_cfg)]
    elif kind == "triple":
        lenses = [binding.ulens_lens_triple(float(rng.uniform(0.8, 1.3)), float(10 ** rng.uniform(-3, -1)),
                                            float(10 ** rng.uniform(-3, -1)), float(rng.uniform(0.5, 1.5)),
                                            float(rng.uniform(0, 2 * np.pi))) for _ in range(n_cfg)]
    else:
        lenses = [binding.lens_single() for _ in range(n_cfg)]
    rho = 10 ** rng.uniform(-3, -1.3, n_cfg)
    u1 = rng.uniform(0.0, 0.8, n_cfg)
    if seed % 2:
        u1[:] = 0.0                                       # the uniform-source kernels too
    # source centres on and around the caustic region: several images, sectors and work units per point
    w = rng.uniform(-0.6, 0.6, (n_cfg, n_pts)) + 1j * rng.uniform(-0.4, 0.4, (n_cfg, n_pts))
    return lenses, rho, u1, w


def _run_both(torch, binding, ctx, case):
    lenses, rho, u1, w = case
    n_cfg, n_pts = w.shape
    w_re = torch.tensor(np.ascontiguousarray(w.real), device="cuda:0")
    w_im = torch.tensor(np.ascontiguousarray(w.imag), device="cuda:0")
    A0, e0, s0 = ctx.ulens_mag(lenses, rho, u1, w_re, w_im)
    A1 = torch.full((n_cfg, n_pts), -7.0, dtype=torch.float64, device="cuda:0")
    e1 = torch.full((n_cfg, n_pts), -7.0, dtype=torch.float64, device="cuda:0")
    s1 = torch.full((n_cfg, n_pts), -7, dtype=torch.int32, device="cuda:0")
    binding.ulens_mag_static(0, lenses, rho, u1, w_re, w_im, A1, e1, s1)
    torch.cuda.synchronize()
    return (A0.cpu().numpy(), e0.cpu().numpy(), s0.cpu().numpy()), (A1.cpu().numpy(), e1.cpu().numpy(), s1.cpu().numpy())


def _compare(ref, got, what):
    (A0, e0, s0), (A1, e1, s1) = ref, got
    assert np.array_equal(s0, s1), what
    fin = np.isfinite(A0)
    assert np.array_equal(fin, np.isfinite(A1)), what
    assert fin.mean() > 0.9, what
    assert np.all(A1[fin] >= 1.0 - 1e-3), what
    rel = np.abs(A1[fin] / A0[fin] - 1)
    assert rel.max() <= RTOL, (what, rel.max())
    assert np.allclose(e1[fin], e0[fin], rtol=0, atol=1e-9), what
    return rel.max(), bool(np.array_equal(A0[fin], A1[fin]))


@pytest.mark.parametrize("kind", ["binary", "triple", "single"])
def test_static_entry_matches_existing_path_two_calls_in_a_row(torch_cuda, kind):
    torch = torch_cuda
    from paper_2510_02639_b200 import binding
    cap = binding.ulens_static_max_points()
    assert cap == 128 and binding.ulens_static_scratch_bytes() <= 8 << 20
    ctx = binding.Context(0, flags=binding.ULENS_OPT_NO_RETRY)
    try:
        first = _case(binding, kind, 11, 4, cap // 4)     # the full 128 points
        second = _case(binding, kind, 12, 3, 17)          # fewer points, other lenses, uniform sources: stale scratch around
        out = []
        for what, case in (("first call", first), ("second call", second), ("first input again", first)):
            ref, got = _run_both(torch, binding, ctx, case)
            out.append((what,) + _compare(ref, got, "%s, %s" % (kind, what)))
        print("%s: " % kind + "; ".join("%s max rel diff %.1e%s" % (w, r, " (bit-equal)" if b else "") for w, r, b in out))
    finally:
        ctx.close()


def test_static_entry_without_optional_outputs_and_on_a_side_stream(torch_cuda):
    torch = torch_cuda
    from paper_2510_02639_b200 import binding
    lenses, rho, u1, w = _case(binding, "binary", 21, 2, 40)
    w_re = torch.tensor(np.ascontiguousarray(w.real), device="cuda:0")
    w_im = torch.tensor(np.ascontiguousarray(w.imag), device="cuda:0")
    A_full = torch.empty((2, 40), dtype=torch.float64, device="cuda:0")
    e_full = torch.empty_like(A_full)
    s_full = torch.empty((2, 40), dtype=torch.int32, device="cuda:0")
    binding.ulens_mag_static(0, lenses, rho, u1, w_re, w_im, A_full, e_full, s_full)
    A_only = torch.empty_like(A_full)
    side = torch.cuda.Stream(device=0)
    torch.cuda.synchronize()
    binding.ulens_mag_static(0, lenses, rho, u1, w_re, w_im, A_only, None, None, stream=side)
    side.synchronize()
    assert torch.equal(A_full, A_only)


def test_static_entry_rejects_sizes_beyond_the_scratch(torch_cuda):
    torch = torch_cuda
    from paper_2510_02639_b200 import binding
    cap = binding.ulens_static_max_points()
    L = binding.ulens_lens_binary(1.0, 0.1)
    n = cap + 1
    w_re = torch.full((1, n), 0.3, dtype=torch.float64, device="cuda:0")
    w_im = torch.zeros((1, n), dtype=torch.float64, device="cuda:0")
    A = torch.full((1, n), -7.0, dtype=torch.float64, device="cuda:0")
    with pytest.raises(binding.UlensError, match="ULENS_STATIC_MAX_POINTS"):
        binding.ulens_mag_static(0, [L], 0.01, 0.3, w_re, w_im, A)
    torch.cuda.synchronize()
    assert bool((A == -7.0).all())                        # refused: nothing was enqueued
    # n_cfg x n_pts counts, not n_pts alone
    w3 = torch.full((3, 43), 0.3, dtype=torch.float64, device="cuda:0")
    with pytest.raises(binding.UlensError, match="ULENS_STATIC_MAX_POINTS"):
        binding.ulens_mag_static(0, [L] * 3, 0.01, 0.3, w3, torch.zeros_like(w3), torch.empty_like(w3))
    # empty requests are fine and do nothing
    e = torch.empty((0,), dtype=torch.float64, device="cuda:0")
    binding.ulens_mag_static(0, [], np.zeros(0), np.zeros(0), e, e, e)


def test_static_entry_allocates_no_device_memory(torch_cuda):
    """Device memory in use (cudaMemGetInfo, which sees every allocation of the process) does not move over calls."""
    torch = torch_cuda
    from paper_2510_02639_b200 import binding
    lenses, rho, u1, w = _case(binding, "binary", 31, 4, 32)
    w_re = torch.tensor(np.ascontiguousarray(w.real), device="cuda:0")
    w_im = torch.tensor(np.ascontiguousarray(w.imag), device="cuda:0")
    A = torch.empty((4, 32), dtype=torch.float64, device="cuda:0")
    e = torch.empty_like(A)
    s = torch.empty((4, 32), dtype=torch.int32, device="cuda:0")
    binding.ulens_mag_static(0, lenses, rho, u1, w_re, w_im, A, e, s)       # set-up, module load, kernel images
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info(0)
    for _ in range(5):
        binding.ulens_mag_static(0, lenses, rho, u1, w_re, w_im, A, e, s)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info(0)
    assert free1 == free0, (free0, free1)

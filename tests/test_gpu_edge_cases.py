"""Edge cases of the CUDA path beyond tests/test_gpu_parity.py: chunk boundaries, many tiny configurations,
the degenerate geometries of the method (equal masses, source covering the lenses, u1 = 1, source on the third
lens of a triple), symmetries, and the size limit. Needs a B200."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu
TOL_A = 1e-4


def _mag(ctx, torch, lenses, rho, u1, w):
    w = np.atleast_2d(np.asarray(w, dtype=complex))
    wre = torch.tensor(np.ascontiguousarray(w.real), device="cuda:0")
    wim = torch.tensor(np.ascontiguousarray(w.imag), device="cuda:0")
    A, err, st = ctx.ulens_mag(lenses, rho, u1, wre, wim)
    torch.cuda.synchronize()
    return A.cpu().numpy(), err.cpu().numpy(), st.cpu().numpy().astype(np.uint32)


def test_chunk_boundary_and_small_chunks(torch_cuda):
    """A call that spans several workspace chunks with a ragged last one gives, point by point, the bits of a
    single-chunk call (chunk_pts = 1000 against the default 65,536; 2,531 points)."""
    from paper_2510_02639_b200 import binding
    rng = np.random.default_rng(31)
    w = rng.uniform(-0.8, 0.8, 2531) + 1j * rng.uniform(-0.8, 0.8, 2531)
    L = binding.ulens_lens_binary(1.1, 0.05)
    big, small = binding.Context(0), binding.Context(0, chunk_pts=1000)
    A1, _, s1 = _mag(big, torch_cuda, [L], [5e-3], [0.3], w)
    A2, _, s2 = _mag(small, torch_cuda, [L], [5e-3], [0.3], w)
    big.close(); small.close()
    assert np.array_equal(A1, A2) and np.array_equal(s1, s2)


def test_many_configurations_of_one_point(ctx, torch_cuda, oracle):
    """n_cfg = 300 lenses x 1 point each (the per-configuration tables are the long axis)."""
    from paper_2510_02639_b200 import binding
    rng = np.random.default_rng(37)
    n = 300
    s = 10 ** rng.uniform(-0.4, 0.4, n); q = 10 ** rng.uniform(-3, 0, n)
    rho = 10 ** rng.uniform(-2.5, -1.5, n); u1 = rng.uniform(0, 1, n)
    w = rng.uniform(-0.5, 0.5, n) + 1j * rng.uniform(-0.5, 0.5, n)
    A, err, st = _mag(ctx, torch_cuda, [binding.ulens_lens_binary(a, b) for a, b in zip(s, q)], rho, u1, w[:, None])
    assert A.shape == (n, 1) and np.all(np.isfinite(A)) and A.min() >= 1 - 1e-4
    pick = rng.choice(n, 24, replace=False)
    n_adm = 0
    for k in pick:
        ref = oracle.mag_fs_batch([oracle.lens_binary(s[k], q[k])], 0, [w[k].real], [w[k].imag], rho[k], u1[k], 100, 8)
        if ref["err_est"][0] <= 2e-5:
            n_adm += 1
            assert abs(A[k, 0] / ref["A"][0] - 1) <= TOL_A, (k, A[k, 0], ref["A"][0])
    assert n_adm >= 20


@pytest.mark.parametrize("s,q,rho,u1,w", [
    (1.0, 1.0, 0.05, 0.5, 0.0 + 0.0j),          # equal masses, source at the centre of symmetry
    (0.6, 1.0, 0.8, 0.0, 0.1 + 0.05j),          # source disk covers both lenses: ring image with holes
    (0.9, 0.3, 0.3, 1.0, 0.2 - 0.1j),           # u1 = 1: the profile vanishes at the limb
    (2.5, 1e-4, 0.02, 0.4, 2.4996 + 0.001j),    # source over a far, light companion (planetary caustic)
    (0.35, 0.7, 0.01, 0.2, 0.003 + 0.004j),     # close binary, tiny central caustic
])
def test_degenerate_binary_geometries(ctx, torch_cuda, oracle, s, q, rho, u1, w):
    from paper_2510_02639_b200 import binding
    A, err, st = _mag(ctx, torch_cuda, [binding.ulens_lens_binary(s, q)], [rho], [u1], [[w]])
    ref = oracle.mag_fs_batch([oracle.lens_binary(s, q)], 0, [w.real], [w.imag], rho, u1, 100, 8)
    assert ref["err_est"][0] <= 2e-5
    assert abs(A[0, 0] / ref["A"][0] - 1) <= TOL_A, (A[0, 0], ref["A"][0], hex(int(st[0, 0])))


def test_triple_source_on_third_lens_and_q3_to_zero(ctx, torch_cuda, oracle):
    from paper_2510_02639_b200 import binding
    p = (1.1, 0.5, 0.03, 1.24, 1.3)
    L, OL = binding.ulens_lens_triple(*p), oracle.lens_triple(*p)
    w3 = complex(L.ax[2], L.ay[2])
    w = np.array([w3, w3 + 0.002, 0.1 + 0.2j])
    A, _, _ = _mag(ctx, torch_cuda, [L], [0.01], [0.5], [w])
    ref = oracle.mag_fs_batch([OL], 0, w.real, w.imag, 0.01, 0.5, 100, 8)
    adm = ref["err_est"] <= 2e-5
    assert adm.sum() >= 2 and np.all(np.isfinite(A))
    assert np.abs(A[0] / ref["A"] - 1)[adm].max() <= TOL_A
    # a third body of vanishing mass: the triple-lens kernels reproduce the binary-lens kernels
    Lt = binding.ulens_lens_triple(0.9, 0.2, 1e-12, 1.5, 0.7)
    Lb = binding.ulens_lens_binary(0.9, 0.2)
    wq = np.array([0.05 + 0.02j, 0.3 - 0.2j, -0.4 + 0.1j])
    At, _, _ = _mag(ctx, torch_cuda, [Lt], [0.02], [0.3], [wq])
    Ab, _, _ = _mag(ctx, torch_cuda, [Lb], [0.02], [0.3], [wq])
    assert np.abs(At / Ab - 1).max() < 2e-5


def test_symmetries(ctx, torch_cuda):
    """Binary on the real axis: A(conj w) = A(w); q -> 1/q with x -> -x."""
    from paper_2510_02639_b200 import binding
    rng = np.random.default_rng(41)
    w = rng.uniform(-0.7, 0.7, 40) + 1j * rng.uniform(0.01, 0.7, 40)
    L = binding.ulens_lens_binary(0.95, 0.25)
    A1, _, _ = _mag(ctx, torch_cuda, [L], [0.01], [0.5], [w])
    A2, _, _ = _mag(ctx, torch_cuda, [L], [0.01], [0.5], [np.conj(w)])
    assert np.abs(A1 / A2 - 1).max() < 2e-5
    Lm = binding.ulens_lens_binary(0.95, 1 / 0.25)
    A3, _, _ = _mag(ctx, torch_cuda, [Lm], [0.01], [0.5], [-w.real + 1j * w.imag])
    # ulens_lens_binary keeps the barycentre at the origin for both labellings, so the mirror image is exact
    assert np.abs(A1 / A3 - 1).max() < 2e-5


def test_size_limit_and_lightcurve_edge_inputs(ctx, torch_cuda):
    from paper_2510_02639_b200 import binding
    torch = torch_cuda
    L = binding.ulens_lens_binary(1.0, 0.1)
    w = torch.zeros(4, dtype=torch.float64, device="cuda:0")
    # n_cfg * n_pts beyond 2^31 - 1: refused before any device buffer is touched
    lib = binding.lib()
    import ctypes as C
    arr = (binding.ulens_lens * 2)(L, L)
    rho = np.array([1e-2, 1e-2]); u1 = np.array([0.0, 0.0])
    rc = lib.ulens_mag(ctx._h, 2, 2 ** 31 - 1, arr, rho.ctypes.data_as(C.POINTER(C.c_double)),
                       u1.ctypes.data_as(C.POINTER(C.c_double)), w.data_ptr(), w.data_ptr(), w.data_ptr(), None, None, None)
    assert rc < 0                      # the point index is a 32-bit int: 2 x (2^31 - 1) points are refused, nothing is read
    assert b"unsupported" in lib.ulens_strerror(rc).lower() or rc == -4 or rc < 0
    # light-curve entry: zero epochs is a no-op; tE <= 0 and non-finite parameters are rejected
    t0 = torch.empty(0, dtype=torch.float64, device="cuda:0")
    A, _, _, _ = ctx.ulens_lightcurve_binary(np.array([[0, 0.1, 1.0, 1.0, 0.1, 0.01, 0.3]]), 0.5, t0)
    assert A.numel() == 0
    t1 = torch.zeros(3, dtype=torch.float64, device="cuda:0")
    for bad in ([0, 0.1, 0.0, 1.0, 0.1, 0.01, 0.3], [0, 0.1, 1.0, -1.0, 0.1, 0.01, 0.3], [0, float("nan"), 1.0, 1.0, 0.1, 0.01, 0.3],
                [0, 0.1, 1.0, 1.0, 0.1, 0.0, 0.3]):
        with pytest.raises(binding.UlensError):
            ctx.ulens_lightcurve_binary(np.array([bad]), 0.5, t1)


def test_device_entries_do_not_synchronise(ctx, torch_cuda):
    """include/ulens.h: 'all device work is enqueued on the caller's stream and the call does NOT synchronise'.
    The stream is kept busy (a spin kernel of ~0.3 s) before the calls; each call must return while that work is
    still running, i.e. without waiting for the stream (pinned staging of the host tables, no cudaStreamSynchronize)."""
    from paper_2510_02639_b200 import binding, inputs
    torch = torch_cuda
    wl = inputs.get(0)
    L = binding.ulens_lens_binary(1.0, 0.01)
    wre = torch.tensor(np.ascontiguousarray(wl.w.real), device="cuda:0")
    wim = torch.tensor(np.ascontiguousarray(wl.w.imag), device="cuda:0")
    t = torch.tensor(wl.t.copy(), device="cuda:0")
    # warm-up: the first calls grow the workspace (cudaMalloc / cudaFree wait for the device)
    ctx.ulens_mag([L], wl.rho, wl.u1, wre, wim)
    ctx.ulens_mag_grad([L], wl.rho, wl.u1, wre, wim)
    ctx.ulens_lightcurve_binary(wl.theta, 0.0, t, want_dA=True)
    ctx.ulens_trajectory(wl.theta, t)
    ctx.ulens_mag_point([L], wre, wim)
    torch.cuda.synchronize()
    stream = torch.cuda.current_stream()
    for name, call in [("ulens_mag", lambda: ctx.ulens_mag([L], wl.rho * 1.01, wl.u1, wre, wim)),
                       ("ulens_mag_grad", lambda: ctx.ulens_mag_grad([L], wl.rho * 1.02, wl.u1, wre, wim)),
                       ("ulens_lightcurve_binary", lambda: ctx.ulens_lightcurve_binary(wl.theta * 1.001, 0.0, t, want_dA=True)),
                       ("ulens_trajectory", lambda: ctx.ulens_trajectory(wl.theta * 1.002, t)),
                       ("ulens_mag_point", lambda: ctx.ulens_mag_point([binding.ulens_lens_binary(1.0, 0.02)], wre, wim))]:
        torch.cuda._sleep(int(0.3 * 1.9e9))               # ~0.3 s of spinning on the stream
        done = torch.cuda.Event()
        call()
        done.record()
        assert not stream.query(), name + " returned only after the stream had drained"
        assert not done.query(), name
        torch.cuda.synchronize()


def test_trajectory_entry_matches_oracle(ctx, torch_cuda, oracle):
    """Step a1 directly: k_traj's source centres against oracle.trajectory (pinned in test_oracle_pins.py), to the
    last bits (the two sides may contract multiply-adds differently: 4 ulp of the largest term)."""
    from paper_2510_02639_b200 import inputs
    torch = torch_cuda
    wl = inputs.get(4)
    cs = [0, 17, 1023]
    t = torch.tensor(wl.t.copy(), device="cuda:0")
    w_re, w_im = ctx.ulens_trajectory(wl.theta[cs], t)
    torch.cuda.synchronize()
    w_re, w_im = w_re.cpu().numpy(), w_im.cpu().numpy()
    for k, c in enumerate(cs):
        t0, u0, tE, _, _, _, al = wl.theta[c]
        ox, oy = oracle.trajectory(t0, u0, tE, al, wl.t)
        scale = np.abs((wl.t - t0) / tE) + abs(u0)
        assert np.all(np.abs(w_re[k] - ox) <= 1e-15 * scale) and np.all(np.abs(w_im[k] - oy) <= 1e-15 * scale)
    with pytest.raises(Exception):
        bad = wl.theta[:1].copy(); bad[0, 2] = 0.0
        ctx.ulens_trajectory(bad, t)


def test_large_sources_fill_the_unit_queue_without_overflow(torch_cuda):
    """Sources of rho = 0.3 ... 2 need hundreds of 32-line work units per point (the old queue of
    192 units per point overflowed and left NaNs). The queue now holds chunk_pts x the per-point cap, and units are
    claimed with a compare-and-swap that refuses rather than overshoots. Single lens, so the reference is the
    Witt-Mao closed form (test_oracle_pins.A_witt_mao, mpmath); a small chunk makes the call span many chunks."""
    from paper_2510_02639_b200 import binding
    from test_oracle_pins import A_witt_mao
    torch = torch_cuda
    c = binding.Context(0, chunk_pts=64)
    rng = np.random.default_rng(5)
    for rho in (0.3, 0.5, 1.0, 2.0):
        u = rng.uniform(0.05, 2.5, 150)
        ph = rng.uniform(0, 2 * np.pi, 150)
        w = u * np.exp(1j * ph)
        A, err, st = _mag(c, torch, [binding.lens_single()], [rho], [0.0], [w])
        assert np.all(np.isfinite(A)), rho
        assert not np.any(st & binding.ST_UNIT_OVF), rho
        ref = np.array([float(A_witt_mao(float(x), rho)) for x in u[:40]])
        assert np.abs(A[0, :40] / ref - 1).max() <= TOL_A, (rho, np.abs(A[0, :40] / ref - 1).max())
    units = c.ulens_get_stats()["n_units"] / (4 * 150)
    assert units > 100                                    # the case really is unit-hungry
    c.close()

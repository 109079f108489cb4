"""Light-curve driver with the point-source / finite-source switch ("(iii) ... only a
preselected set of N_ext epochs (e.g., near caustics) are modeled"). Needs a B200.

References (never the CUDA path itself):
  * point-source epochs: oracle.mag_point_source (companion-matrix roots refined in __float128, Eq. 2-3) and its
    central finite differences through oracle.lightcurve_case for the 7 derivatives;
  * finite-source epochs: oracle.mag_fs_batch (brute-force inverse ray shooting), value bar 1e-4.
Gather / scatter: integer work, compared bit for bit with the unswitched entry on the same epochs.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

ST_POINT_SRC = 0x1000
TOL_A = 1e-4


@pytest.fixture(scope="module")
def oracle():
    from oracle import oracle as O
    O.build()
    return O


def _case(n_cfg=3, n_ep=700):
    """C4-shaped light curves (inputs.config4: the paper's injected vector, jittered 1 %)."""
    from paper_2510_02639_b200 import inputs
    wl = inputs.config4(n_cfg=n_cfg, n_epochs=n_ep)
    return wl.theta, wl.t


def _np(x):
    return x.cpu().numpy()


def test_all_selected_equals_unswitched_entry(ctx, torch_cuda):
    """mask = 1 everywhere: the identity gather map must reproduce ulens_lightcurve_binary bit for bit."""
    torch = torch_cuda
    theta, t = _case(2, 300)
    td = torch.tensor(t, device="cuda:0")
    A0, dA0, err0, st0 = ctx.ulens_lightcurve_binary(theta, 0.5, td, want_dA=True)
    mask = torch.ones((2, 300), dtype=torch.uint8, device="cuda:0")
    A1, dA1, err1, st1, n_ext = ctx.ulens_lightcurve_binary_ext(theta, 0.5, td, ext_mask=mask, want_dA=True)
    torch.cuda.synchronize()
    assert n_ext == 600
    assert np.array_equal(_np(A0), _np(A1)) and np.array_equal(_np(dA0), _np(dA1), equal_nan=True)
    assert np.array_equal(_np(err0), _np(err1)) and np.array_equal(_np(st0), _np(st1))


def test_random_mask_gather_scatter(ctx, torch_cuda):
    """Selected epochs carry the finite-source result of the unswitched entry bit for bit (ragged counts per
    light curve, chunk-crossing map); the others carry the point-source result, the status bit and err = 0."""
    torch = torch_cuda
    theta, t = _case(3, 700)
    td = torch.tensor(t, device="cuda:0")
    rng = np.random.default_rng(11)
    m = (rng.random((3, 700)) < np.array([0.05, 0.5, 0.9])[:, None])
    m[0, :40] = False
    m[2, -33:] = True
    mask = torch.tensor(m.astype(np.uint8), device="cuda:0")
    A0, dA0, err0, st0 = ctx.ulens_lightcurve_binary(theta, 0.5, td, want_dA=True)
    zero = torch.zeros_like(mask)
    Ap, dAp, _, stp, n0 = ctx.ulens_lightcurve_binary_ext(theta, 0.5, td, ext_mask=zero, want_dA=True)
    A1, dA1, err1, st1, n_ext = ctx.ulens_lightcurve_binary_ext(theta, 0.5, td, ext_mask=mask, want_dA=True)
    torch.cuda.synchronize()
    assert n0 == 0 and n_ext == int(m.sum())
    A0, dA0, err0, st0, Ap, dAp, stp, A1, dA1, err1, st1 = map(_np, (A0, dA0, err0, st0, Ap, dAp, stp, A1, dA1, err1, st1))
    assert np.array_equal(A1[m], A0[m]) and np.array_equal(dA1[m], dA0[m], equal_nan=True)
    assert np.array_equal(err1[m], err0[m]) and np.array_equal(st1[m], st0[m])
    assert np.array_equal(A1[~m], Ap[~m]) and np.array_equal(dA1[~m], dAp[~m])
    assert np.all(st1[~m] & ST_POINT_SRC) and not np.any(st1[m] & ST_POINT_SRC)
    assert np.all(stp & ST_POINT_SRC) and np.all(err1[~m] == 0.0)


def test_point_source_epochs_vs_oracle(ctx, torch_cuda, oracle):
    """mask = 0 everywhere: A and dA/d(t0,u0,tE,s,q,rho,alpha) of Eq. 2-3 against the oracle's point-source
    magnification and its central finite differences (two half-widths, Richardson)."""
    torch = torch_cuda
    O = oracle
    theta, t = _case(2, 500)
    td = torch.tensor(t, device="cuda:0")
    zero = torch.zeros((2, 500), dtype=torch.uint8, device="cuda:0")
    A, dA, _, st, _ = ctx.ulens_lightcurve_binary_ext(theta, 0.5, td, ext_mask=zero, want_dA=True)
    torch.cuda.synchronize()
    A, dA = _np(A), _np(dA)
    rng = np.random.default_rng(5)
    # epochs spread over the whole curve plus the ones around the peak (the caustic region of this geometry)
    picks = [(c, int(e)) for c in range(2) for e in np.concatenate([rng.choice(500, 10, replace=False),
                                                                    np.argsort(-A[c])[:6]])]
    n_checked = 0
    for c, e in picks:
        def f(p):
            L, w, _ = O.lightcurve_case(p, t[e])
            return O.mag_point_source(L, w)
        ref = f(theta[c])
        assert abs(A[c, e] / ref - 1) < 1e-9, (c, e, A[c, e], ref)
        scale = np.array([1.0, 1.0, theta[c, 2], 1.0, theta[c, 4], 1.0, 1.0])
        for k in range(7):
            d = []
            for h in (2e-5 * scale[k], 1e-5 * scale[k]):
                pp, pm = theta[c].copy(), theta[c].copy()
                pp[k] += h
                pm[k] -= h
                d.append((f(pp) - f(pm)) / (2 * h))
            fd, corr = (4 * d[1] - d[0]) / 3, abs(d[1] - d[0]) / 3
            if corr > 1e-4 * abs(fd) + 1e-9:
                continue                     # a caustic within the stencil: the difference is not a derivative
            assert abs(dA[c, e, k] - fd) <= 1e-5 * abs(fd) + 1e-6 * ref / scale[k], (c, e, k, dA[c, e, k], fd)
            n_checked += 1
    assert n_checked >= 150
    assert np.all(dA[..., 5] == 0.0)         # a point source has no rho


def test_library_selection_vs_oracle(ctx, torch_cuda, oracle):
    """ext_mask = NULL: the library's multipole probe decides. The switched light curve must still meet the value
    bar against the finite-source oracle on BOTH kinds of epoch, and the switch must actually switch."""
    torch = torch_cuda
    O = oracle
    theta, t = _case(4, 2000)
    td = torch.tensor(t, device="cuda:0")
    A, _, _, st, n_ext = ctx.ulens_lightcurve_binary_ext(theta, 0.5, td, ext_mask=None, sel_tol=0.0)
    A0, _, _, st0 = ctx.ulens_lightcurve_binary(theta, 0.5, td)
    torch.cuda.synchronize()
    A, st, A0 = _np(A), _np(st), _np(A0)
    ps = (st & ST_POINT_SRC) != 0
    assert n_ext == int((~ps).sum())
    assert 0 < n_ext < 0.5 * ps.size, n_ext          # far epochs (most of the curve) take the point-source value
    # property at full size: nowhere does the switched curve leave the unswitched one by more than the bar
    assert np.max(np.abs(A / A0 - 1)) < TOL_A
    assert np.array_equal(A[~ps], A0[~ps])
    # parity on samples: the point-source epochs closest to being selected (largest finite-source effect) and random ones
    rng = np.random.default_rng(3)
    for c in range(4):
        idx_ps = np.flatnonzero(ps[c])
        worst = idx_ps[np.argsort(-np.abs(A[c, idx_ps] / A0[c, idx_ps] - 1))[:6]]
        some = rng.choice(idx_ps, 6, replace=False)
        ext = rng.choice(np.flatnonzero(~ps[c]), 4, replace=False)
        ep = np.concatenate([worst, some, ext])
        L = O.lens_binary(theta[c, 3], theta[c, 4])
        wx, wy = O.trajectory(theta[c, 0], theta[c, 1], theta[c, 2], theta[c, 6], t[ep])
        ref = O.mag_fs_batch([L], 0, wx, wy, theta[c, 5], 0.5)
        ok = ref["err_est"] <= 2e-5
        assert ok.sum() >= 12
        assert np.max(np.abs(A[c, ep][ok] / ref["A"][ok] - 1)) < TOL_A


def test_ext_edge_cases(ctx, torch_cuda):
    torch = torch_cuda
    theta, t = _case(1, 64)
    td = torch.tensor(t, device="cuda:0")
    # empty inputs
    A, _, _, _, n_ext = ctx.ulens_lightcurve_binary_ext(theta[:0], 0.5, td)
    assert n_ext == 0 and A.numel() == 0
    # one selected epoch at the very end, and at the very start
    for pos in (0, 63):
        m = torch.zeros((1, 64), dtype=torch.uint8, device="cuda:0")
        m[0, pos] = 1
        A1, _, _, st1, n_ext = ctx.ulens_lightcurve_binary_ext(theta, 0.5, td, ext_mask=m)
        torch.cuda.synchronize()
        st1 = _np(st1)
        assert n_ext == 1 and not (st1[0, pos] & ST_POINT_SRC) and ((st1[0] & ST_POINT_SRC) != 0).sum() == 63


def test_ext_host_entry_matches_device_entry(ctx, torch_cuda):
    """ulens_lightcurve_binary_ext_host (host arrays, mask copied in) against the device entry, bit for bit."""
    torch = torch_cuda
    theta, t = _case(2, 400)
    rng = np.random.default_rng(17)
    m = (rng.random((2, 400)) < 0.3).astype(np.uint8)
    td = torch.tensor(t, device="cuda:0")
    for mask_h in (m, None):
        mask_d = torch.tensor(m, device="cuda:0") if mask_h is not None else None
        A0, dA0, err0, st0, n0 = ctx.ulens_lightcurve_binary_ext(theta, 0.5, td, ext_mask=mask_d, want_dA=True)
        torch.cuda.synchronize()
        A = np.empty((2, 400)); dA = np.empty((2, 400, 7)); err = np.empty((2, 400)); st = np.empty((2, 400), dtype=np.int32)
        _, _, _, _, n1 = ctx.ulens_lightcurve_binary_ext_host(theta, 0.5, t, A, dA, err, st, ext_mask=mask_h)
        assert n0 == n1 and (mask_h is None or n1 == int(m.sum()))
        assert np.array_equal(A, _np(A0)) and np.array_equal(dA, _np(dA0), equal_nan=True)
        assert np.array_equal(err, _np(err0)) and np.array_equal(st, _np(st0))

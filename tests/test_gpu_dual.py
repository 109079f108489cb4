"""Forward-mode (dual-number) variant of the CUDA path, SURVEY 8.a row a8 / BASELINE.json configs[4]. Needs a B200.

References (never the CUDA path itself):
  * single lens: mpmath derivatives of the closed forms pinned in test_oracle_pins (Witt-Mao, annulus form);
  * binary lens: the oracle's central finite differences (oracle.mag_fd, pinned on the same closed forms),
    two step sizes, Richardson-combined; a component takes part only where the two step sizes agree.

Tolerance: |dA_gpu - dA_ref| <= 1e-3 |dA_ref| + 1e-4 A / scale_p. The first term is
BASELINE.json's "1e-3 relative"; the second is the resolution of the value bar itself (A is certified to
1e-4 relative, so a change of A over one natural scale of the parameter -- the source radius in the source
plane, the finite-difference half-width for the oracle reference -- is not known better than 1e-4 A).
"""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

REL = 1e-3
ABS_A = 1e-4


def _grad(ctx, torch, lenses, rho, u1, w):
    w = np.atleast_2d(np.asarray(w, dtype=complex))
    wre = torch.tensor(np.ascontiguousarray(w.real), device="cuda:0")
    wim = torch.tensor(np.ascontiguousarray(w.imag), device="cuda:0")
    A, dA, err, st = ctx.ulens_mag_grad(lenses, rho, u1, wre, wim)
    torch.cuda.synchronize()
    return A.cpu().numpy(), dA.cpu().numpy(), st.cpu().numpy().astype(np.uint32)


@pytest.mark.parametrize("u,rho,u1", [(0.3, 0.05, 0.0), (0.03, 0.05, 0.0), (0.3, 0.05, 0.5), (0.06, 0.05, 0.5),
                                      (1.2, 0.3, 0.3), (0.011, 0.01, 0.0)])
def test_single_lens_derivatives_closed_form(ctx, torch_cuda, u, rho, u1):
    """dA/du (along the source offset), dA/d(perpendicular) = 0 and dA/drho against mpmath derivatives."""
    import mpmath as mp
    from paper_2510_02639_b200 import binding
    from test_oracle_pins import A_ld_single, A_witt_mao
    f = (lambda uu, rr: A_ld_single(uu, rr, u1)) if u1 > 0 else A_witt_mao
    ang = 0.83
    w = u * complex(math.cos(ang), math.sin(ang))
    A, dA, _ = _grad(ctx, torch_cuda, [binding.lens_single()], [rho], [u1], [[w]])
    ref = float(f(u, rho))
    du = float(mp.diff(lambda x: f(x, mp.mpf(rho)), u))
    dr = float(mp.diff(lambda x: f(mp.mpf(u), x), rho))
    g = dA[0, 0]
    assert abs(A[0, 0] / ref - 1) < 5e-5
    du_gpu = g[0] * math.cos(ang) + g[1] * math.sin(ang)
    dperp = -g[0] * math.sin(ang) + g[1] * math.cos(ang)
    floor = ABS_A * ref / rho
    assert abs(du_gpu - du) <= REL * abs(du) + floor, (du_gpu, du)
    assert abs(dperp) <= REL * abs(du) + floor, dperp
    assert abs(g[4] - dr) <= REL * abs(dr) + floor, (g[4], dr)
    assert g[2] == 0.0 and g[3] == 0.0                      # a single lens has no (s, q)


def test_dual_value_equals_primal_value(ctx, torch_cuda):
    """The dual kernels shoot the same grid as the primal ones: A from ulens_mag_grad == A from ulens_mag."""
    from paper_2510_02639_b200 import binding, inputs
    torch = torch_cuda
    wl = inputs.get(0)
    L = binding.ulens_lens_binary(1.0, 0.01)
    w = wl.w[:, ::7]
    A2, _, _ = _grad(ctx, torch, [L], wl.rho, wl.u1, w)
    wre = torch.tensor(np.ascontiguousarray(w.real), device="cuda:0")
    wim = torch.tensor(np.ascontiguousarray(w.imag), device="cuda:0")
    A1, _, _ = ctx.ulens_mag([L], wl.rho, wl.u1, wre, wim)
    torch.cuda.synchronize()
    assert np.allclose(A1.cpu().numpy(), A2, rtol=1e-9, atol=0)


def test_lightcurve_chain_rule(ctx, torch_cuda, oracle):
    """dA/d(t0,u0,tE,alpha) from ulens_lightcurve_binary == the chain rule through the trajectory (reading G3)
    applied in numpy to dA/d(w_cx, w_cy) from ulens_mag_grad; (s, q, rho) pass through unchanged."""
    from paper_2510_02639_b200 import binding, inputs
    torch = torch_cuda
    wl = inputs.get(4, n_cfg=2, n_epochs=2000)
    th = wl.theta[1]
    t0, u0, tE, s, q, rho, al = th
    tt = wl.t[700:1300:40]
    t = torch.tensor(tt.copy(), device="cuda:0")
    A, dA, _, _ = ctx.ulens_lightcurve_binary(th[None, :], 0.5, t, want_dA=True)
    torch.cuda.synchronize()
    dA = dA.cpu().numpy()[0]
    wx, wy = oracle.trajectory(t0, u0, tE, al, tt)
    A2, g, _ = _grad(ctx, torch, [binding.ulens_lens_binary(s, q)], [rho], [0.5], [wx + 1j * wy])
    g = g[0]
    tau = (tt - t0) / tE
    ca, sa = math.cos(al), math.sin(al)
    dtau_dt0, dtau_dtE = -1.0 / tE, -tau / tE
    d_t0 = (g[:, 0] * ca + g[:, 1] * sa) * dtau_dt0
    d_tE = (g[:, 0] * ca + g[:, 1] * sa) * dtau_dtE
    d_u0 = -g[:, 0] * sa + g[:, 1] * ca
    d_al = g[:, 0] * (-tau * sa - u0 * ca) + g[:, 1] * (tau * ca - u0 * sa)
    ref = np.stack([d_t0, d_u0, d_tE, g[:, 2], g[:, 3], g[:, 4], d_al], axis=1)
    # k_traj's w_c may differ from the host trajectory in the last bit -> a sector border may move by one cell
    scale = np.abs(ref).max(axis=0, keepdims=True)
    assert np.all(np.abs(dA - ref) <= 2e-4 * np.abs(ref) + 2e-5 * scale), np.abs(dA - ref).max(axis=0) / scale


def test_config4_derivatives_vs_oracle_fd(ctx, torch_cuda, oracle):
    """BASELINE configs[4]: dA/d(t0,u0,tE,s,q,rho,alpha) against the oracle's central finite differences on a
    seeded subsample (2 parameter vectors x 7 epochs spanning the peak)."""
    from paper_2510_02639_b200 import inputs
    torch = torch_cuda
    wl = inputs.get(4)                                     # the full C4 workload; vectors 0 and 3 of its 1,024
    sel = np.array([600, 800, 900, 950, 1050, 1100, 1300])
    t = torch.tensor(wl.t[sel].copy(), device="cuda:0")
    n_used = n_ok = 0
    worst = 0.0
    for c in (0, 3):
        th = wl.theta[c]
        A, dA, _, st = ctx.ulens_lightcurve_binary(th[None, :], 0.5, t, want_dA=True)
        torch.cuda.synchronize()
        A = A.cpu().numpy()[0]; dA = dA.cpu().numpy()[0]
        rho = th[5]
        for j, e in enumerate(sel):
            tau = (wl.t[e] - th[0]) / th[2]
            wabs = abs(wl.w[c][e])
            # half-widths that move the source (or the caustics) by about one source radius
            steps = np.array([rho * th[2], rho, rho * th[2] / max(abs(tau), 0.1), rho, 0.3 * th[4], 0.3 * rho,
                              rho / max(wabs, 0.1)])
            A0, D = oracle.mag_fd(lambda p: oracle.lightcurve_case(p, wl.t[e]), th, [steps, 0.5 * steps], 0.5, 200, 16)
            Dx, corr = oracle.fd_extrapolate(D)
            assert abs(A[j] / A0 - 1) < 1e-4
            tol = REL * np.abs(Dx) + ABS_A * A0 / steps
            ok_ref = corr <= 0.3 * tol                    # the two step sizes agree: the reference is usable
            bad = (np.abs(dA[j] - Dx) > tol) & ok_ref
            worst = max(worst, float((np.abs(dA[j] - Dx) / tol)[ok_ref].max(initial=0.0)))
            n_used += int(ok_ref.sum()); n_ok += int((ok_ref & ~bad).sum())
            assert not bad.any(), (c, e, dA[j], Dx, corr, tol)
    print("C4 derivative components compared: %d (of %d), worst |err|/tol = %.2f" % (n_used, 2 * len(sel) * 7, worst))
    assert n_used >= 0.8 * 2 * len(sel) * 7

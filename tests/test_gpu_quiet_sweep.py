"""The quiet-point shortcut on lenses the BASELINE configs do not contain. Needs a B200.

Seeded random families -- binaries with s in [0.32, 3.2] and q in [1e-5, 1], planetary binaries (q down to 3e-6), triples
(q in [1e-4, 1], q3 in [1e-6, 1e-1]) and the single lens; rho in [1e-4, 0.32], u1 in [0, 1]; source positions uniform in
[-2, 2]^2, half of them drawn towards the lens -- are run with the shortcut (production) and with ULENS_OPT_NO_QUIET.
The shortcut only changes how densely quiet points are sampled and shot, so the two runs must agree: no point that is
clean in both may differ by more than 1e-4, and the flagged sets must (nearly) coincide. The worst clean points are then
sent to the oracle. Measured (1.4 M points): largest difference 3.3e-5; the worst points are within 3.4e-5 of the oracle
(before the quiet points' sectors ended at the true extremes of their images: 6.3e-5 and 6.1e-5).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _family(binding, name, seed, n_cfg, n_pts):
    rng = np.random.default_rng(seed)
    if name == "binary":
        par = [(float(10 ** rng.uniform(-0.5, 0.5)), float(10 ** rng.uniform(-5, 0))) for _ in range(n_cfg)]
    elif name == "binary_planet":
        par = [(float(rng.uniform(0.7, 1.5)), float(10 ** rng.uniform(-5.5, -2.5))) for _ in range(n_cfg)]
    elif name == "triple":
        par = [(float(rng.uniform(0.6, 1.8)), float(10 ** rng.uniform(-4, 0)), float(10 ** rng.uniform(-6, -1)),
                float(rng.uniform(0.4, 2.0)), float(rng.uniform(0, 2 * np.pi))) for _ in range(n_cfg)]
    else:
        par = [() for _ in range(n_cfg)]
    rho = 10 ** rng.uniform(-4, -0.5, n_cfg)
    u1 = rng.uniform(0, 1, n_cfg)
    w = rng.uniform(-2, 2, (n_cfg, n_pts)) + 1j * rng.uniform(-2, 2, (n_cfg, n_pts))
    w[:, ::2] *= 0.35
    return par, rho, u1, w


def _make(mod, name, par):
    if name == "triple":
        return [mod.lens_triple(*p) if hasattr(mod, "lens_triple") else mod.ulens_lens_triple(*p) for p in par]
    if name == "single":
        return [mod.lens_single() for _ in par]
    return [mod.lens_binary(*p) if hasattr(mod, "lens_binary") else mod.ulens_lens_binary(*p) for p in par]


@pytest.mark.parametrize("name,seed,n_cfg", [("binary", 1, 192), ("binary_planet", 2, 192), ("triple", 3, 96), ("single", 4, 192)])
def test_quiet_shortcut_on_random_lenses(torch_cuda, oracle, name, seed, n_cfg):
    torch = torch_cuda
    from paper_2510_02639_b200 import binding
    par, rho, u1, w = _family(binding, name, seed, n_cfg, 2048)
    lenses = _make(binding, name, par)
    w_re = torch.tensor(np.ascontiguousarray(w.real), device="cuda:0")
    w_im = torch.tensor(np.ascontiguousarray(w.imag), device="cuda:0")
    out = {}
    for tag, fl in (("full", binding.ULENS_OPT_NO_QUIET), ("prod", 0)):
        c = binding.Context(0, flags=fl)
        A, e, s = c.ulens_mag(lenses, rho, u1, w_re, w_im)
        torch.cuda.synchronize()
        out[tag] = (A.cpu().numpy(), s.cpu().numpy().astype(np.uint32), c.ulens_get_stats()["n_limb_solves"] / A.numel())
        c.close()
    A0, s0, n0 = out["full"]; A1, s1, n1 = out["prod"]
    assert np.array_equal(np.isnan(A0), np.isnan(A1))
    f0 = (s0 & 0xff) != 0; f1 = (s1 & 0xff) != 0
    rel = np.abs(A1 / A0 - 1)
    rel[f0 | f1 | np.isnan(rel)] = 0.0
    assert n1 < 0.8 * n0                                   # the shortcut did engage
    assert abs(int(f0.sum()) - int(f1.sum())) <= 0.01 * max(int(f0.sum()), 100)
    assert rel.max() <= 6e-5, np.argwhere(rel > 6e-5)[:8]
    # the worst clean points against the oracle (magnification < 30 keeps the oracle affordable)
    cand = np.where(A0 < 30, rel, 0.0)
    order = np.argsort(cand.ravel())[::-1][:12]
    ci, pi = np.unravel_index(order, rel.shape)
    ol = _make(oracle, name, par)
    ref = oracle.mag_fs_batch(ol, ci.astype(np.int32), w[ci, pi].real.copy(), w[ci, pi].imag.copy(), rho[ci], u1[ci], 100, 8)
    adm = ref["err_est"] <= 2e-5
    r1 = np.abs(A1[ci, pi] / ref["A"] - 1)[adm]
    print("%s: %d points, limb solves per point %.0f -> %.0f, flagged %d -> %d; largest difference between the runs %.1e (%d above 5e-5); "
          "the 12 worst points against the oracle: max %.1e" % (name, A0.size, n0, n1, int(f0.sum()), int(f1.sum()), rel.max(),
                                                                 int((rel > 5e-5).sum()), r1.max() if len(r1) else 0.0))
    assert adm.sum() >= 8 and r1.max() <= 6e-5

"""Marginalised-flux NLL and gradient on the GPU (ulens_nll_marginal, App. B.2 / SURVEY 8.f-3) against oracle/nll.py
(dense B17, no Woodbury) on seeded synthetic data shaped like the paper's injection (one data set, many
parameter vectors). Needs a B200."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _data(n_cfg, n_ep, seed):
    """Light-curve-like A (a peak on a baseline), dA random but smooth in scale, noisy fluxes of the first curve."""
    rng = np.random.default_rng(seed)
    t = np.linspace(-2, 2, n_ep)
    A = 1.0 + np.stack([(2.0 + 0.2 * rng.random()) / np.sqrt(t ** 2 + (0.1 + 0.02 * rng.random()) ** 2) * 0.1 for _ in range(n_cfg)])
    dA = rng.standard_normal((n_cfg, n_ep, 7)) * (A - 1.0)[..., None]
    sigma = rng.uniform(0.01, 0.03, n_ep)
    flux = (A[0] - 1.0) * 1.5 + 0.3 + sigma * rng.standard_normal(n_ep)
    return A, dA, flux, sigma


@pytest.mark.parametrize("n_cfg,n_ep,mu,var", [(5, 700, (0.0, 0.0), (4.0, 1.0)),        # the paper's "mu = 0" case
                                               (3, 257, (1.4, 0.25), (0.3, 0.05)),      # ragged against the 256-thread block
                                               (2, 1, (1.0, 0.2), (0.5, 0.5)),          # one epoch
                                               (1, 2000, (0.0, 0.0), (1e2, 1e2))])      # C4-sized curve, wide priors (std 10 against fluxes ~ 1)
def test_nll_and_gradient_vs_dense_oracle(ctx, torch_cuda, n_cfg, n_ep, mu, var):
    torch = torch_cuda
    from oracle import nll as N
    A, dA, flux, sigma = _data(n_cfg, n_ep, 100 + n_ep)
    dev = lambda x: torch.tensor(np.ascontiguousarray(x), device="cuda:0")
    nll, grad = ctx.ulens_nll_marginal(dev(A), dev(dA), dev(flux), dev(sigma), mu[0], mu[1], var[0], var[1])
    nll_only, none = ctx.ulens_nll_marginal(dev(A), None, dev(flux), dev(sigma), mu[0], mu[1], var[0], var[1])
    torch.cuda.synchronize()
    nll, grad = nll.cpu().numpy(), grad.cpu().numpy()
    assert none is None and np.array_equal(nll, nll_only.cpu().numpy())
    for c in range(n_cfg):
        ref = N.nll_dense(A[c], flux, sigma, mu, var)
        # Tolerance 1e-9 relative: fp64 sums on both sides, and the oracle's dense solve loses eps * cond(B) ~
        # eps * n var / sigma^2 (2e9 * 2.2e-16 in the widest case here; with var = 1e4 that term alone was 4e-5 absolute).
        assert abs(nll[c] - ref) <= 1e-9 * max(1.0, abs(ref)), (c, nll[c], ref)
        # Reference gradient: Richardson-combined central differences of the DENSE oracle with half-widths (1e-2, 5e-3) of
        # the largest dA. The dense solve's rounding noise (eps * cond(B), up to 4e-7 absolute here) over 2h must stay
        # below the bar, which rules out small steps (measured on the n = 2000 case against the same formula in numpy:
        # h = 1e-6 -> 1e-2 relative, 1e-4 -> 4e-5, 1e-2 -> 9e-7); the h^2 truncation term is what the Richardson step removes.
        g, corr = N.nll_grad_fd(A[c], dA[c], flux, sigma, mu, var, h=1e-2)
        assert np.all(np.abs(grad[c] - g) <= 1e-5 * np.abs(g) + 1e-6 * np.max(np.abs(g))), (c, grad[c], g, corr)


def test_nll_invalid_arguments(ctx, torch_cuda):
    torch = torch_cuda
    from paper_2510_02639_b200 import binding
    A = torch.ones((1, 4), dtype=torch.float64, device="cuda:0")
    f = torch.ones(4, dtype=torch.float64, device="cuda:0")
    with pytest.raises(binding.UlensError):
        ctx.ulens_nll_marginal(A, None, f, f, 0.0, 0.0, 0.0, 1.0)            # variance must be positive
    with pytest.raises(binding.UlensError):
        ctx.ulens_nll_marginal(A, None, f, f, float("nan"), 0.0, 1.0, 1.0)

"""Pins of oracle/nll.py (App. B) on what the mathematics fixes -- none of the expected values comes from the oracle
itself or from the CUDA path."""
import math

import numpy as np

from oracle import nll as N


def _case(n=4, seed=0):
    rng = np.random.default_rng(seed)
    A = 1.0 + rng.uniform(0.2, 3.0, n)
    sigma = rng.uniform(0.05, 0.2, n)
    flux = (A - 1.0) * 1.3 + 0.4 + sigma * rng.standard_normal(n)
    return A, flux, sigma


def test_brute_force_marginalisation_over_beta():
    """B15: p(y|theta) = Int N(y|M beta, C) N(beta|mu, Lambda) d beta, by a tensor-product Gauss-Hermite rule in the two
    linear parameters (exact for the Gaussian weight up to the polynomial degree; 120 nodes per axis)."""
    A, flux, sigma = _case(4, 1)
    sigma = sigma * 8.0                 # likelihood as wide as the prior: the rule's nodes (prior scale) resolve it
    mu, var = np.array([1.0, 0.3]), np.array([0.5, 0.2])
    x, w = np.polynomial.hermite.hermgauss(120)
    b1 = mu[0] + math.sqrt(2 * var[0]) * x
    b2 = mu[1] + math.sqrt(2 * var[1]) * x
    M = np.stack([A - 1.0, np.ones_like(A)], axis=1)
    tot = 0.0
    for i in range(len(x)):
        pred = M[:, 0][None, :] * b1[i] + b2[:, None]                      # [n2, n]
        like = np.exp(-0.5 * np.sum(((flux[None, :] - pred) / sigma[None, :]) ** 2, axis=1)) / np.prod(np.sqrt(2 * np.pi) * sigma)
        tot += w[i] * np.sum(w * like)
    p = tot / np.pi                                                         # the two 1/sqrt(pi) of the Hermite weights
    ref = -math.log(p) - 0.5 * len(A) * math.log(2 * math.pi)               # B17 drops n/2 ln 2 pi
    assert abs(N.nll_dense(A, flux, sigma, mu, var) - ref) < 1e-9 * max(1.0, abs(ref))


def test_sharp_prior_limit_is_chi_square():
    """Lambda -> 0: the linear parameters are known, NLL -> 1/2 chi^2 + sum ln sigma_i."""
    A, flux, sigma = _case(7, 2)
    mu = np.array([1.2, 0.5])
    ref = 0.5 * np.sum(((flux - (A - 1.0) * mu[0] - mu[1]) / sigma) ** 2) + np.sum(np.log(sigma))
    assert abs(N.nll_dense(A, flux, sigma, mu, [1e-14, 1e-14]) - ref) < 1e-8


def test_no_magnification_column_reduces_to_a_constant_offset():
    """A = 1 everywhere: only F_base acts; one-parameter closed form (Sherman-Morrison by hand)."""
    n = 6
    A = np.ones(n)
    rng = np.random.default_rng(3)
    sigma = rng.uniform(0.1, 0.3, n)
    flux = 0.7 + sigma * rng.standard_normal(n)
    mu, var = np.array([5.0, 0.6]), np.array([2.0, 0.3])
    w = 1.0 / sigma ** 2
    r = flux - mu[1]
    s = 1.0 / var[1] + w.sum()
    ref = 0.5 * (np.sum(w * r * r) - np.sum(w * r) ** 2 / s) + 0.5 * (np.sum(np.log(sigma ** 2)) + math.log(var[1]) + math.log(s))
    assert abs(N.nll_dense(A, flux, sigma, mu, var) - ref) < 1e-10


def test_scaling_invariance():
    """Units of flux: F, sigma, mu -> c F, c sigma, c mu and Lambda -> c^2 Lambda shift the NLL by n ln c."""
    A, flux, sigma = _case(9, 4)
    mu, var = np.array([0.9, 0.2]), np.array([0.4, 0.1])
    c = 3.7
    d = N.nll_dense(A, c * flux, c * sigma, c * mu, c * c * var) - N.nll_dense(A, flux, sigma, mu, var)
    assert abs(d - len(A) * math.log(c)) < 1e-9


def test_fd_gradient_on_a_quadratic_direction():
    """nll_grad_fd on the sharp-prior limit, where d NLL/dA_i = -mu_1 r_i / sigma_i^2 in closed form."""
    A, flux, sigma = _case(5, 5)
    mu = np.array([1.1, 0.4])
    dA = np.random.default_rng(6).standard_normal((5, 7))
    r = flux - (A - 1.0) * mu[0] - mu[1]
    ref = (-mu[0] * r / sigma ** 2) @ dA
    g, corr = N.nll_grad_fd(A, dA, flux, sigma, mu, [1e-14, 1e-14])
    assert np.allclose(g, ref, rtol=1e-6, atol=1e-8)

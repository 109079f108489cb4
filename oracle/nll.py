"""Oracle for the marginalised-flux negative log-likelihood (App. B of arXiv 2510.02639). TEST INFRASTRUCTURE ONLY:
imported by tests/ (and nothing in the product path); shares no code with the CUDA path.

The definition written out, dense and slow, in numpy float64 (P = line of /root/reference/PAPER.md):

    NLL(theta) = 1/2 (F - M mu)^T B^-1 (F - M mu) + 1/2 ln|B|,   B = C + M Lambda M^T           (B17)
    M = [A(t_i; theta) - 1, 1]  (n x 2),  mu = (F_S, F_base),  Lambda = diag(var_FS, var_Fbase)   (B21-B23)
    C = diag(sigma_i^2)                                                                          ("Lambda and C_j are diagonal")

B is built as an n x n matrix and handed to numpy.linalg (solve, slogdet): no Woodbury identity (B18-B19), which is
what the CUDA path uses. As in B17 the constant n/2 ln(2 pi) of the Gaussian is left out.
Pins: tests/test_oracle_nll_pins.py (brute-force marginalisation over beta, the Lambda -> 0 limit, B14's factorisation).
"""
import numpy as np


def design(A):
    A = np.asarray(A, dtype=np.float64)
    return np.stack([A - 1.0, np.ones_like(A)], axis=1)                       # B21


def nll_dense(A, flux, sigma, mu, var):
    """B17 for one light curve. A, flux, sigma [n]; mu = (F_S, F_base); var = (var_FS, var_Fbase)."""
    M = design(A)
    B = np.diag(np.asarray(sigma, dtype=np.float64) ** 2) + M @ np.diag(np.asarray(var, dtype=np.float64)) @ M.T
    r = np.asarray(flux, dtype=np.float64) - M @ np.asarray(mu, dtype=np.float64)
    sign, logdet = np.linalg.slogdet(B)
    if sign <= 0:
        raise ValueError("B is not positive definite")
    return 0.5 * r @ np.linalg.solve(B, r) + 0.5 * logdet


def nll_grad_fd(A, dA, flux, sigma, mu, var, h=1e-6):
    """Directional central differences of nll_dense along the columns of dA [n, 7] (dA/dtheta_k): two half-widths
    (h, h/2) Richardson-combined. Returns (grad [7], size of the Richardson correction [7])."""
    A = np.asarray(A, dtype=np.float64)
    dA = np.asarray(dA, dtype=np.float64)
    out, corr = np.empty(dA.shape[1]), np.empty(dA.shape[1])
    for k in range(dA.shape[1]):
        d = dA[:, k]
        sc = max(np.max(np.abs(d)), 1e-300)
        e = []
        for hh in (h / sc, 0.5 * h / sc):
            e.append((nll_dense(A + hh * d, flux, sigma, mu, var) - nll_dense(A - hh * d, flux, sigma, mu, var)) / (2 * hh))
        out[k] = (4 * e[1] - e[0]) / 3
        corr[k] = abs(e[1] - e[0]) / 3
    return out, corr

"""Seeded synthetic inputs for the five BASELINE.json configs C0..C4.

This module serves BOTH the CUDA path's tests/bench and the oracle's tests. It holds none of the
method's arithmetic (no root solver, no quadrature, no magnification): it only draws lens
parameters, source radii and source positions. The one piece of lens algebra here is the recipe
that places points near a caustic ("each test point is sampled within a circular
region ... centered at a randomly selected point along the caustic curve"), which needs caustic
points: critical-curve points from numpy.roots mapped through Eq. 1. Neither the oracle nor
the CUDA path calls it.

All inputs are synthetic stand-ins for the paper's own workloads (random draws near a caustic,
P:205; light curves); no public dataset is involved.

Lens geometry conventions (readings G4/G5 in DESIGN.md) are repeated here only to locate caustics.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

SEED_ROOT = 251002639


@dataclass
class Workload:
    """One config: n_cfg lens/source configurations x n_pts source positions each."""
    name: str
    kind: str                      # "binary" | "triple"
    lens_params: np.ndarray        # [n_cfg, 2] (s, q)  or  [n_cfg, 5] (s, q, q3, r3, psi)
    rho: np.ndarray                # [n_cfg]
    u1: np.ndarray                 # [n_cfg]
    w: np.ndarray                  # [n_cfg, n_pts] complex128 source-centre positions
    near_caustic: np.ndarray       # [n_cfg, n_pts] bool, True for the near-caustic half
    traj: np.ndarray | None = None  # [n_cfg, 4] (t0, u0, tE, alpha) where the points came from a line
    t: np.ndarray | None = None     # [n_pts] epochs (C0, C4)
    theta: np.ndarray | None = None  # C4: [n_cfg, 7] (t0, u0, tE, s, q, rho, alpha)
    meta: dict = field(default_factory=dict)

    @property
    def n_cfg(self):
        return self.w.shape[0]

    @property
    def n_pts(self):
        return self.w.shape[1]


def _rng(cfg: int) -> np.random.Generator:
    return np.random.default_rng(np.random.SeedSequence([SEED_ROOT, cfg]))


def lens_geometry(kind: str, p) -> tuple[np.ndarray, np.ndarray]:
    """(eps, a) for a parameter row; only used to locate caustics for the input recipe."""
    if kind == "binary":
        s, q = p[:2]
        eps = np.array([1.0, q]) / (1.0 + q)
        a = np.array([-s * q / (1.0 + q), s / (1.0 + q)], dtype=complex)
    else:
        s, q, q3, r3, psi = p
        eps = np.array([1.0, q, q3]) / (1.0 + q + q3)
        a1, a2 = -s * q / (1.0 + q), s / (1.0 + q)
        a = np.array([a1, a2, 0.5 * (a1 + a2) + r3 * np.exp(1j * psi)], dtype=complex)
    return eps, a


def caustic_points(eps: np.ndarray, a: np.ndarray, n_phi: int = 512) -> np.ndarray:
    """Points on the caustics: solve sum_i eps_i/(z-a_i)^2 = e^{-i phi} (degree 2N in z) on a uniform
    phi grid, map the critical-curve points through Eq. 1."""
    n = len(a)
    full = np.poly(np.repeat(a, 2))                       # prod_k (z-a_k)^2
    parts = [eps[i] * np.poly(np.repeat(np.delete(a, i), 2)) for i in range(n)]
    lhs = np.zeros(2 * n + 1, dtype=complex)
    for p_ in parts:
        lhs[-len(p_):] += p_
    out = []
    for phi in 2 * np.pi * (np.arange(n_phi) + 0.5) / n_phi:
        z = np.roots(lhs - np.exp(-1j * phi) * full)
        w = z - np.sum(eps[None, :] / np.conj(z[:, None] - a[None, :]), axis=1)
        out.append(w)
    return np.concatenate(out)


def line_points(t0, u0, tE, alpha, t):
    """Source positions on a straight trajectory (reading G3; input recipe only)."""
    tau = (np.asarray(t) - t0) / tE
    return (tau * np.cos(alpha) - u0 * np.sin(alpha)) + 1j * (tau * np.sin(alpha) + u0 * np.cos(alpha))


def _mixed_points(rng, kind, p, rho, n_pts, tau_half):
    """Half the points on a random line, half within 3 rho of a random caustic point (C1..C3)."""
    u0 = rng.uniform(-0.1, 0.1)
    alpha = rng.uniform(0.0, 2 * np.pi)
    n_line = n_pts // 2
    tau = np.sort(rng.uniform(-tau_half, tau_half, n_line))
    w_line = line_points(0.0, u0, 1.0, alpha, tau)
    eps, a = lens_geometry(kind, p)
    cau = caustic_points(eps, a)
    n_near = n_pts - n_line
    pick = cau[rng.integers(0, len(cau), n_near)]
    rad = 3.0 * rho * np.sqrt(rng.uniform(0.0, 1.0, n_near))
    ang = rng.uniform(0.0, 2 * np.pi, n_near)
    w_near = pick + rad * np.exp(1j * ang)
    w = np.concatenate([w_line, w_near])
    flag = np.concatenate([np.zeros(n_line, bool), np.ones(n_near, bool)])
    return w, flag, np.array([0.0, u0, 1.0, alpha])


def config0() -> Workload:
    """C0: binary s=1, q=0.01, rho=1e-2, u1=0; 500 points tau=-1.5..1.5, u0=0.05, alpha=0.7."""
    t = -1.5 + 3.0 * np.arange(500) / 499.0
    traj = np.array([[0.0, 0.05, 1.0, 0.7]])
    w = line_points(0.0, 0.05, 1.0, 0.7, t)[None, :]
    return Workload("C0", "binary", np.array([[1.0, 0.01]]), np.array([1e-2]), np.array([0.0]), w,
                    np.zeros_like(w, dtype=bool), traj=traj, t=t,
                    theta=np.array([[0.0, 0.05, 1.0, 1.0, 0.01, 1e-2, 0.7]]))


def config1(n_cfg: int = 64, n_pts: int = 2048) -> Workload:
    """C1: binary, u1=0.5, rho=1e-3; s log-U[0.3,3], q log-U[1e-5,1]."""
    rng = _rng(1)
    P, W, F, T = [], [], [], []
    for _ in range(n_cfg):
        s = 10 ** rng.uniform(np.log10(0.3), np.log10(3.0))
        q = 10 ** rng.uniform(-5.0, 0.0)
        w, f, tr = _mixed_points(rng, "binary", (s, q), 1e-3, n_pts, 2.0)
        P.append((s, q)); W.append(w); F.append(f); T.append(tr)
    return Workload("C1", "binary", np.array(P), np.full(n_cfg, 1e-3), np.full(n_cfg, 0.5), np.array(W),
                    np.array(F), traj=np.array(T))


def config2(n_cfg: int = 64, n_pts: int = 4096) -> Workload:
    """C2: binary, large source: rho log-U[1e-2,1e-1], u1 U[0.3,0.7]; points as C1."""
    rng = _rng(2)
    P, W, F, T, R, U = [], [], [], [], [], []
    for _ in range(n_cfg):
        s = 10 ** rng.uniform(np.log10(0.3), np.log10(3.0))
        q = 10 ** rng.uniform(-5.0, 0.0)
        rho = 10 ** rng.uniform(-2.0, -1.0)
        u1 = rng.uniform(0.3, 0.7)
        w, f, tr = _mixed_points(rng, "binary", (s, q), rho, n_pts, 2.0)
        P.append((s, q)); W.append(w); F.append(f); T.append(tr); R.append(rho); U.append(u1)
    return Workload("C2", "binary", np.array(P), np.array(R), np.array(U), np.array(W), np.array(F),
                    traj=np.array(T))


def config3(n_cfg: int = 32, n_pts: int = 4096) -> Workload:
    """C3: triple, u1=0.5, rho=1e-3 (parameter mapping: reading G5)."""
    rng = _rng(3)
    P, W, F, T = [], [], [], []
    for _ in range(n_cfg):
        s = 10 ** rng.uniform(np.log10(0.5), np.log10(2.0))
        q = 10 ** rng.uniform(-4.0, -1.0)
        r3 = 10 ** rng.uniform(np.log10(0.3), np.log10(3.0))
        q3 = 10 ** rng.uniform(-5.0, -2.0)
        psi = rng.uniform(0.0, 2 * np.pi)
        p = (s, q, q3, r3, psi)
        w, f, tr = _mixed_points(rng, "triple", p, 1e-3, n_pts, 2.0)
        P.append(p); W.append(w); F.append(f); T.append(tr)
    return Workload("C3", "triple", np.array(P), np.full(n_cfg, 1e-3), np.full(n_cfg, 0.5), np.array(W),
                    np.array(F), traj=np.array(T))


def config4(n_cfg: int = 1024, n_epochs: int = 2000) -> Workload:
    """C4: inference-style batch; theta = (t0,u0,tE,s,q,rho,alpha) jittered +-1% around a seeded
    centre taken from the paper's injected vector, u1=0.5, rho=5e-3."""
    rng = _rng(4)
    tE = 10 ** 1.21
    q_c = 10 ** rng.uniform(-4.0, -2.0)
    centre = np.array([0.0, 0.06, tE, 10 ** 0.012, q_c, 5e-3, 4.156])
    theta = centre[None, :] * (1.0 + 0.01 * rng.uniform(-1.0, 1.0, (n_cfg, 7)))
    theta[:, 0] = 0.01 * tE * rng.uniform(-1.0, 1.0, n_cfg)
    t = np.linspace(-1.5 * tE, 1.5 * tE, n_epochs)
    w = np.stack([line_points(th[0], th[1], th[2], th[6], t) for th in theta])
    return Workload("C4", "binary", theta[:, 3:5].copy(), theta[:, 5].copy(), np.full(n_cfg, 0.5), w,
                    np.zeros_like(w, dtype=bool), traj=theta[:, [0, 1, 2, 6]].copy(), t=t, theta=theta,
                    meta={"centre": centre})


def get(cfg: int, **kw) -> Workload:
    return [config0, config1, config2, config3, config4][cfg](**kw)


def subsample(wl: Workload, n_per_cfg: int, seed: int = 0) -> np.ndarray:
    """Seeded stratified sample of point indices per config: half from the near-caustic half.
    Returns int array [n_cfg, n_per_cfg] (sorted)."""
    rng = np.random.default_rng(np.random.SeedSequence([SEED_ROOT, 99, seed]))
    out = []
    for c in range(wl.n_cfg):
        near = np.flatnonzero(wl.near_caustic[c])
        far = np.flatnonzero(~wl.near_caustic[c])
        k_near = min(len(near), n_per_cfg // 2)
        k_far = n_per_cfg - k_near
        pick = np.concatenate([rng.choice(near, k_near, replace=False) if k_near else np.array([], int),
                               rng.choice(far, k_far, replace=False)])
        out.append(np.sort(pick))
    return np.array(out)


def light_body_zone(wl: Workload, c: int, eps_max: float = 1e-3) -> np.ndarray:
    """Workload points of config c that lie within 8 sqrt(eps_a) + 2 rho of the planetary-caustic centre
    w_a = a_a - sum_{b != a} eps_b / conj(a_a - a_b) of a light body (eps_a < eps_max): the geometry in which a
    faint image pair hides next to the light lens. Input selection only; returns a bool mask [n_pts]."""
    eps, a = lens_geometry(wl.kind, wl.lens_params[c])
    mask = np.zeros(wl.n_pts, dtype=bool)
    for i in range(len(a)):
        if not eps[i] < eps_max:
            continue
        others = [b for b in range(len(a)) if b != i]
        w_a = a[i] - np.sum(eps[others] / np.conj(a[i] - a[others]))
        mask |= np.abs(wl.w[c] - w_a) < 8.0 * np.sqrt(eps[i]) + 2.0 * wl.rho[c]
    return mask


def golden_sample(wl: Workload, cfg: int, n_total: int = 2048, n_zone: int = 12):
    """The seeded sample behind tests/golden/oracle_C<cfg>.npz: n_total / n_cfg stratified points of every
    configuration (subsample(), seed 500 + cfg) plus up to n_zone further points per configuration from
    light_body_zone(). Returns (cfg_index [m], point_index [m], in_zone [m])."""
    idx = subsample(wl, n_total // wl.n_cfg, seed=500 + cfg)
    rng = np.random.default_rng(np.random.SeedSequence([SEED_ROOT, 98, cfg]))
    cs, ps, zs = [], [], []
    for c in range(wl.n_cfg):
        zone = light_body_zone(wl, c)
        base = idx[c]
        cand = np.setdiff1d(np.flatnonzero(zone), base)
        extra = np.sort(rng.choice(cand, min(n_zone, len(cand)), replace=False)) if len(cand) else np.array([], int)
        p = np.concatenate([base, extra])
        cs.append(np.full(len(p), c)); ps.append(p); zs.append(zone[p])
    return np.concatenate(cs), np.concatenate(ps), np.concatenate(zs)


def golden_c4_sample(wl: Workload, n_vec: int = 16, n_ep: int = 16):
    """The seeded (vector, epoch) sample behind tests/golden/oracle_C4_fd.npz: n_vec parameter vectors, and per
    vector n_ep epochs, half of them from |tau| < 0.15 (the caustic crossing and the peak), half from the rest."""
    rng = np.random.default_rng(np.random.SeedSequence([SEED_ROOT, 97, 4]))
    vec = np.sort(rng.choice(wl.n_cfg, n_vec, replace=False))
    eps_ = []
    for c in vec:
        tau = (wl.t - wl.theta[c, 0]) / wl.theta[c, 2]
        near = np.flatnonzero(np.abs(tau) < 0.15)
        far = np.flatnonzero(np.abs(tau) >= 0.15)
        eps_.append(np.sort(np.concatenate([rng.choice(near, n_ep // 2, replace=False),
                                            rng.choice(far, n_ep - n_ep // 2, replace=False)])))
    return vec, np.array(eps_)

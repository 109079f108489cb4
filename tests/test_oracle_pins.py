"""Pins for the CPU oracle: what the paper and the mathematics fix, independent of oracle code.

Every expected value here comes from a closed form, an invariant, a textbook special case or a
brute-force evaluation written in this file (mpmath / numpy) -- never from the CUDA path and never
from the oracle itself.
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest


# ---------------------------------------------------------------- closed forms (single lens)

def A_ps_single(u):
    """Point-source magnification of one point lens (textbook; Eq. 2-3 with N=1)."""
    return (u * u + 2) / (u * mp.sqrt(u * u + 4))


def A_uniform_single_sourceplane(u, rho):
    """Uniform disk behind a single lens by integrating the point-source magnification over the
    source disk in polar coordinates about the lens (plain definition, source-plane side):
    A = 1/(pi rho^2) Int A_ps(r) * r * dphi(r) dr, dphi(r) = angular extent of the disk at radius r."""
    u, rho = mp.mpf(u), mp.mpf(rho)

    def width(r):
        if u <= rho and r <= rho - u:
            return 2 * mp.pi
        c = (r * r + u * u - rho * rho) / (2 * r * u)
        c = max(-1, min(1, c))
        return 2 * mp.acos(c)

    f = lambda r: (r * r + 2) / mp.sqrt(r * r + 4) * width(r)
    lo, hi = abs(u - rho), u + rho
    pts = [0, rho - u, hi] if u < rho else [lo, hi]
    return mp.quad(f, pts) / (mp.pi * rho * rho)


def A_witt_mao(u, rho):
    """Witt & Mao (1994) elliptic-integral form named by BASELINE.json north_star (u != rho)."""
    u, rho = mp.mpf(u), mp.mpf(rho)
    n = 4 * u * rho / (u + rho) ** 2
    S = mp.sqrt(4 + (u - rho) ** 2)
    k2 = 4 * n / (4 + (u - rho) ** 2)
    K, E, Pi = mp.ellipk(k2), mp.ellipe(k2), mp.ellippi(n, k2)
    return (1 / (2 * mp.pi)) * ((u + rho) / rho ** 2 * S * E
                                - (u - rho) / rho ** 2 * (8 + u * u - rho * rho) / S * K
                                + 4 * (u - rho) ** 2 / (rho ** 2 * (u + rho)) * (1 + rho * rho) / S * Pi)


def A_ld_single(u, rho, u1):
    """Linear limb darkening by decomposing sqrt(1-x^2) into uniform disks of radius rho sin(phi):
    A_LD = [(1-u1) A_U(u,rho) + u1 Int_0^{pi/2} sin^3(phi) A_U(u, rho sin phi) dphi] / (1 - u1/3)."""
    AU = lambda r: A_witt_mao(u, r) if u > 0 else mp.sqrt(1 + 4 / mp.mpf(r) ** 2)
    integ = mp.quad(lambda p: mp.sin(p) ** 3 * AU(rho * mp.sin(p)), [0, mp.pi / 4, mp.pi / 2])
    return ((1 - u1) * AU(rho) + u1 * integ) / (1 - mp.mpf(u1) / 3)


def test_closed_forms_agree_with_each_other():
    # the two independent single-lens forms (elliptic vs source-plane quadrature) pin each other
    for u, rho in [(0.3, 0.05), (0.02, 0.05), (1.2, 0.3)]:
        assert abs(A_witt_mao(u, rho) / A_uniform_single_sourceplane(u, rho) - 1) < 1e-10


@pytest.mark.parametrize("rho", [0.1, 0.01, 1e-3])
def test_uniform_single_lens_centre(oracle, rho):
    """A = sqrt(1 + 4/rho^2) at u = 0 (north_star)."""
    L = oracle.lens_single()
    A, _ = oracle.mag_fs(L, 0j, rho, 0.0, 100, 8)
    assert abs(A / math.sqrt(1 + 4 / rho ** 2) - 1) < 5e-6


@pytest.mark.parametrize("u,rho", [(0.3, 0.05), (0.02, 0.05), (0.05, 0.05), (1.2, 0.3), (0.011, 0.01)])
def test_uniform_single_lens_witt_mao(oracle, u, rho):
    L = oracle.lens_single()
    ref = float(A_witt_mao(u, rho)) if u != rho else float(A_uniform_single_sourceplane(u, rho))
    # source off-axis in a generic direction so no lattice symmetry helps
    w = u * complex(math.cos(0.83), math.sin(0.83))
    r = oracle.mag_fs_batch([L], 0, [w.real], [w.imag], rho, 0.0, 100, 8)
    assert abs(r["A"][0] / ref - 1) < 5e-6
    assert r["err_est"][0] < 2e-5


@pytest.mark.parametrize("u,rho,u1", [(0.0, 0.05, 0.5), (0.3, 0.05, 0.5), (0.03, 0.05, 1.0), (0.2, 0.1, 0.3)])
def test_limb_darkened_single_lens(oracle, u, rho, u1):
    L = oracle.lens_single()
    ref = float(A_ld_single(u, rho, u1))
    w = u * complex(math.cos(2.1), math.sin(2.1))
    r = oracle.mag_fs_batch([L], 0, [w.real], [w.imag], rho, u1, 100, 8)
    assert abs(r["A"][0] / ref - 1) < 1e-5
    assert r["err_est"][0] < 2e-5


def test_F0_normalisation():
    """I0 = 3/(pi(3-u1)) normalises Eq. A6 to unit flux <=> F0 = pi rho^2 (1-u1/3)."""
    for u1 in (0.0, 0.3, 1.0):
        flux = mp.quad(lambda x: (1 - u1 * (1 - mp.sqrt(1 - x * x))) * 2 * mp.pi * x, [0, 1])
        assert abs(flux - mp.pi * (1 - mp.mpf(u1) / 3)) < 1e-12
        assert abs(flux * 3 / (mp.pi * (3 - u1)) - 1) < 1e-12


# ---------------------------------------------------------------- exact cover: brute force on a dense lattice

def test_quadtree_equals_dense_lattice(oracle):
    """For a uniform source the oracle's sum is exactly the count of inside sub-lattice points: a
    dense numpy evaluation over the whole bounding box (no culling, no tree) must give the same A."""
    L = oracle.lens_binary(0.9, 0.3)
    w, rho, n_rho, ss = complex(0.05, 0.02), 0.1, 8, 2
    A, _ = oracle.mag_fs(L, w, rho, 0.0, n_rho, ss)
    p = rho / n_rho / ss
    half = int(math.ceil(4.0 / p))
    g = (np.arange(-half, half) + 0.5) * p
    Z = g[None, :] + 1j * g[:, None]
    a, eps = L.positions(), L.masses()
    W = Z - sum(e / np.conj(Z - ai) for e, ai in zip(eps, a))
    inside = np.abs(W - w) < rho
    A_dense = inside.sum() * p * p / (math.pi * rho * rho)
    assert abs(A / A_dense - 1) < 1e-12


def test_quadtree_equals_dense_lattice_limb_darkened(oracle):
    """Same with limb darkening at ss=1 in the near-limb band ... the interior midpoint rule is on the
    coarse cells, so compare against a dense lattice at the coarse pitch with ss=1 everywhere."""
    L = oracle.lens_binary(1.3, 0.05)
    w, rho, n_rho, u1 = complex(-0.2, 0.1), 0.1, 16, 0.6
    A, _ = oracle.mag_fs(L, w, rho, u1, n_rho, 1)
    p = rho / n_rho
    half = int(math.ceil(4.5 / p))
    g = (np.arange(-half, half) + 0.5) * p
    Z = g[None, :] + 1j * g[:, None]
    a, eps = L.positions(), L.masses()
    W = Z - sum(e / np.conj(Z - ai) for e, ai in zip(eps, a))
    x2 = np.abs(W - w) ** 2 / rho ** 2
    I = np.where(x2 < 1, 1 - u1 * (1 - np.sqrt(np.clip(1 - x2, 0, None))), 0.0)
    A_dense = I.sum() * p * p / (math.pi * rho * rho * (1 - u1 / 3))
    assert abs(A / A_dense - 1) < 1e-12


# ---------------------------------------------------------------- limits and symmetries (binary / triple)

def test_point_source_limit(oracle):
    """A(w_c, rho) -> sum 1/|det J| as rho -> 0 away from caustics (O(rho^2) correction)."""
    L = oracle.lens_binary(1.0, 0.01)
    for w in (complex(0.3, 0.2), complex(-0.5, 0.05)):
        Aps = oracle.mag_point_source(L, w)
        r = oracle.mag_fs_batch([L], 0, [w.real], [w.imag], 1e-4, 0.0, 100, 8)
        assert abs(r["A"][0] / Aps - 1) < 2e-5


def test_far_field(oracle):
    """A -> 1 far from the lenses (north_star). Leading term: the primary image sees shear 1/|w|^2
    (total mass 1, dipole zero about the barycentre) -> 1/(1-|w|^-4) ~ 1 + |w|^-4, and each lens i
    keeps one faint image of magnification eps_i^2/|w|^4:  A - 1 -> (1 + sum eps_i^2)/|w|^4
    (= 2/|w|^4 for a single lens, the textbook value)."""
    L = oracle.lens_binary(0.8, 0.5)
    lead = 1 + sum(e * e for e in L.masses())
    for w in (complex(12.0, 5.0), complex(-3.0, 20.0)):
        Aps = oracle.mag_point_source(L, w)
        assert abs((Aps - 1) / (lead / abs(w) ** 4) - 1) < 2e-2
        r = oracle.mag_fs_batch([L], 0, [w.real], [w.imag], 0.05, 0.3, 100, 8)
        assert abs(r["A"][0] - 1) < 3 / abs(w) ** 4 + 2e-5
    S = oracle.lens_single()
    assert abs((oracle.mag_point_source(S, 15 + 0j) - 1) / (2 / 15.0 ** 4) - 1) < 2e-2


def test_binary_mirror_symmetry(oracle):
    L = oracle.lens_binary(1.1, 0.2)
    w = complex(0.13, 0.07)
    r = oracle.mag_fs_batch([L], 0, [w.real, w.real], [w.imag, -w.imag], 0.02, 0.4, 100, 8)
    assert abs(r["A"][0] / r["A"][1] - 1) < 1e-9     # the lattice is mirror symmetric too


def test_q_inversion_symmetry(oracle):
    """q -> 1/q with x -> -x is the same lens (reading G4 puts the barycentre at the origin)."""
    L1, L2 = oracle.lens_binary(0.9, 0.25), oracle.lens_binary(0.9, 4.0)
    w = complex(0.11, -0.06)
    a = oracle.mag_fs_batch([L1], 0, [w.real], [w.imag], 0.03, 0.0, 100, 8)["A"][0]
    b = oracle.mag_fs_batch([L2], 0, [-w.real], [w.imag], 0.03, 0.0, 100, 8)["A"][0]
    assert abs(a / b - 1) < 1e-9


def test_triple_reduces_to_binary(oracle):
    Lb = oracle.lens_binary(1.2, 0.1)
    Lt = oracle.lens_triple(1.2, 0.1, 1e-14, 0.7, 1.0)
    w = complex(0.2, 0.1)
    a = oracle.mag_fs_batch([Lb], 0, [w.real], [w.imag], 0.02, 0.5, 100, 8)["A"][0]
    b = oracle.mag_fs_batch([Lt], 0, [w.real], [w.imag], 0.02, 0.5, 100, 8)["A"][0]
    assert abs(a / b - 1) < 1e-8
    assert abs(oracle.mag_point_source(Lb, w) / oracle.mag_point_source(Lt, w) - 1) < 1e-8


def test_wide_binary_reduces_to_single(oracle):
    """Binary with a remote, light companion -> single lens (Witt-Mao) within the tidal perturbation."""
    L = oracle.lens_binary(50.0, 1e-6)
    u, rho = 0.3, 0.05
    w = complex(L.ax[0], 0) + u * complex(math.cos(1.0), math.sin(1.0))   # measured from the primary
    A = oracle.mag_fs_batch([L], 0, [w.real], [w.imag], rho, 0.0, 100, 8)["A"][0]
    assert abs(A / float(A_witt_mao(u, rho)) - 1) < 1e-5


# ---------------------------------------------------------------- geometry, trajectory, Jacobian

def test_lens_geometry(oracle):
    s, q = 1.3, 0.2
    L = oracle.lens_binary(s, q)
    assert abs(L.eps[0] + L.eps[1] - 1) < 1e-15 and abs(L.eps[1] / L.eps[0] - q) < 1e-15
    assert abs(L.eps[0] * L.ax[0] + L.eps[1] * L.ax[1]) < 1e-15      # barycentre at the origin
    assert abs((L.ax[1] - L.ax[0]) - s) < 1e-15 and L.ax[0] < 0 < L.ax[1]  # reading G4
    # Fig. 2 values, read from the fixture
    fig2 = dict(l.split() for l in open(os.path.join(os.path.dirname(__file__), "golden", "fig2_triple_lens.txt"))
                if l.strip() and not l.startswith("#"))
    q3, r3, psi = float(fig2["q3"]), float(fig2["r3"]), math.radians(float(fig2["psi"]))
    assert (q3, r3) == (0.03, 1.24)
    T = oracle.lens_triple(s, q, q3, r3, psi)
    assert abs(sum(T.eps[:3]) - 1) < 1e-15 and abs(T.eps[2] / T.eps[0] - q3) < 1e-15
    mid = 0.5 * (T.ax[0] + T.ax[1])
    d = complex(T.ax[2] - mid, T.ay[2])
    assert abs(abs(d) - r3) < 1e-15 and abs(math.atan2(d.imag, d.real) - psi) < 1e-15
    assert abs((T.ax[1] - T.ax[0]) - s) < 1e-15


def test_trajectory(oracle):
    t = np.linspace(-2, 3, 11)
    wx, wy = oracle.trajectory(0.5, 0.1, 2.0, 0.0, t)                 # alpha = 0: along +x at height u0
    assert np.allclose(wx, (t - 0.5) / 2.0) and np.allclose(wy, 0.1)
    wx, wy = oracle.trajectory(0.5, 0.1, 2.0, math.pi / 2, t)          # alpha = 90 deg
    assert np.allclose(wx, -0.1) and np.allclose(wy, (t - 0.5) / 2.0)
    wx, wy = oracle.trajectory(0.5, 0.1, 2.0, 0.7, t)                  # |w|^2 = tau^2 + u0^2, closest at t0
    assert np.allclose(wx ** 2 + wy ** 2, ((t - 0.5) / 2.0) ** 2 + 0.01)


def test_detJ_matches_finite_difference_jacobian(oracle):
    L = oracle.lens_triple(1.1, 0.5, 0.03, 1.24, 1.3)
    z, h = complex(0.4, -0.7), 1e-6
    fx = (oracle.lens_map(L, z + h) - oracle.lens_map(L, z - h)) / (2 * h)
    fy = (oracle.lens_map(L, z + 1j * h) - oracle.lens_map(L, z - 1j * h)) / (2 * h)
    det = fx.real * fy.imag - fx.imag * fy.real
    assert abs(det - oracle.det_J(L, z)) < 1e-8


# ---------------------------------------------------------------- polynomial and roots

def test_polynomial_vanishes_on_images(oracle):
    """Brute force: pick z, set w = f_map(z); then z must be a root of Eq. 4 built for that w."""
    rng = np.random.default_rng(5)
    for L in (oracle.lens_single(), oracle.lens_binary(0.8, 0.3), oracle.lens_triple(1.1, 0.5, 0.03, 1.24, 1.3)):
        for _ in range(20):
            z = complex(*rng.uniform(-1.5, 1.5, 2))
            w = oracle.lens_map(L, z)
            b = oracle.poly_coeffs(L, w)
            assert len(b) - 1 == L.n ** 2 + 1
            val = sum(bl * z ** l for l, bl in enumerate(b))
            scale = sum(abs(bl) * abs(z) ** l for l, bl in enumerate(b))
            assert abs(val) < 1e-13 * scale
            # leading coefficient prod (conj w - conj a_i)
            lead = np.prod([np.conj(w) - np.conj(a) for a in L.positions()])
            assert abs(b[-1] - lead) < 1e-14 * abs(lead)


def test_roots_vieta_residual_count_parity(oracle):
    rng = np.random.default_rng(7)
    cases = [(oracle.lens_binary(10 ** rng.uniform(-0.5, 0.5), 10 ** rng.uniform(-3, 0)), (3, 5)) for _ in range(30)]
    cases += [(oracle.lens_triple(10 ** rng.uniform(-0.3, 0.3), 10 ** rng.uniform(-2, 0), 10 ** rng.uniform(-2, 0),
                                  10 ** rng.uniform(-0.5, 0.5), rng.uniform(0, 6.28)), (4, 6, 8, 10)) for _ in range(30)]
    for L, counts in cases:
        w = complex(*rng.uniform(-1, 1, 2))
        b = oracle.poly_coeffs(L, w)
        r = oracle.roots(L, w)
        n = len(b) - 1
        assert abs(np.sum(r["z"]) + b[n - 1] / b[n]) < 1e-9 * max(1, abs(b[n - 1] / b[n]))      # Vieta sum
        assert abs(np.prod(r["z"]) - (-1) ** n * b[0] / b[n]) < 1e-8 * max(1, abs(b[0] / b[n]))  # Vieta product
        img = r["is_image"]
        assert img.sum() in counts                                          # N+1 .. 5(N-1) images
        assert np.all(r["resid"][img] < 1e-21) and np.all(r["resid"][~img] > 1e-8)
        for z in r["z"][img]:
            assert abs(oracle.lens_map(L, complex(z)) - w) < 1e-12
        assert int(np.sum(np.sign(r["detJ"][img]))) == 1 - L.n              # parity sum 1 - N


def test_signed_magnification_sum_inside_binary_caustic(oracle):
    """Binary lens with 5 images: sum 1/det J = 1 exactly (Witt & Mao 1995 theorem)."""
    L = oracle.lens_binary(1.0, 0.01)
    r = oracle.roots(L, complex(-0.00161720, 0.06401082))
    assert r["is_image"].sum() == 5
    assert abs(np.sum(1 / r["detJ"][r["is_image"]]) - 1) < 1e-11


def test_single_lens_roots_closed_form(oracle):
    L = oracle.lens_single()
    u = 0.37
    r = oracle.roots(L, complex(u, 0))
    zs = np.sort(r["z"][r["is_image"]].real)
    assert np.allclose(zs, [(u - math.sqrt(u * u + 4)) / 2, (u + math.sqrt(u * u + 4)) / 2], atol=1e-15)
    assert abs(oracle.mag_point_source(L, complex(u, 0)) - float(A_ps_single(mp.mpf(u)))) < 1e-13


# ---------------------------------------------------------------- derivative reference (finite differences)

@pytest.mark.parametrize("u,rho,u1", [(0.3, 0.05, 0.0), (0.03, 0.05, 0.0), (0.0, 0.05, 0.0), (0.3, 0.05, 0.5)])
def test_fd_derivative_reference_single_lens(oracle, u, rho, u1):
    """oracle.mag_fd against closed forms: dA/drho = -4/(rho^3 sqrt(1+4/rho^2)) at u = 0 and
    mpmath derivatives of the Witt-Mao / limb-darkened closed forms elsewhere."""
    S = oracle.lens_single()

    def case(p):
        return S, complex(p[0] * math.cos(0.83), p[0] * math.sin(0.83)), p[1]

    ss = 16 if u1 == 0 else 8
    steps = [[0.2 * rho, 0.1 * rho], [0.1 * rho, 0.05 * rho]]
    A0, dA = oracle.mag_fd(case, [u, rho], steps, u1, 100, ss)
    D, corr = oracle.fd_extrapolate(dA)
    if u == 0.0:
        exact_rho = -4.0 / (rho ** 3 * math.sqrt(1 + 4 / rho ** 2))
        assert abs(D[1] / exact_rho - 1) < 2e-4
        assert abs(D[0]) < 2e-4 * abs(exact_rho)            # symmetric in u
        return
    f = (lambda uu, rr: A_ld_single(uu, rr, u1)) if u1 > 0 else A_witt_mao
    du = float(mp.diff(lambda x: f(x, mp.mpf(rho)), u))
    dr = float(mp.diff(lambda x: f(mp.mpf(u), x), rho))
    scale = A0 / rho                                       # natural size of a derivative in source-plane units
    assert abs(D[0] - du) < 1e-3 * max(abs(du), 0.02 * scale)
    assert abs(D[1] - dr) < 1e-3 * max(abs(dr), 0.02 * scale)

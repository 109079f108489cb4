"""Host-compiled logic of the device headers (no GPU needed): tests/host_logic.cpp runs, for one source point,
the code of k_roots, k_regions (three phases, lane by lane), k_shoot (every scan line) and k_finalize on the
CPU. This checks the builder's host-testable logic -- polynomial, root solver, sector construction (cover,
disjointness), line rule -- against numpy, closed forms and the oracle. It is test infrastructure: the
product path has no CPU route (tests/test_abi.py::test_no_gpu_means_loud_failure)."""
import math
import os
import subprocess

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def exe(tmp_path_factory):
    out = str(tmp_path_factory.mktemp("host_logic") / "host_logic")
    subprocess.check_call(["g++", "-O2", "-std=c++17", "-o", out, os.path.join(HERE, "host_logic.cpp")])
    return out


def run(exe, eps, a, rho, u1, w, n_limb=512, n_r=96, n_theta=48):
    a = np.asarray(a, dtype=complex)
    args = [exe, str(len(eps))] + [repr(float(e)) for e in eps] + [repr(float(z.real)) for z in a] + \
           [repr(float(z.imag)) for z in a] + [repr(float(rho)), repr(float(u1)), repr(float(w.real)), repr(float(w.imag)),
                                              str(n_limb), str(n_r), str(n_theta)]
    txt = subprocess.run(args, capture_output=True, text=True, check=True).stdout
    out = {"coef": [], "roots": [], "img": [], "patches": []}
    for line in txt.splitlines():
        f = line.split()
        if f[0] == "coef":
            out["coef"].append(complex(float(f[2]), float(f[3])))
        elif f[0] == "root":
            out["roots"].append(complex(float(f[2]), float(f[3]))); out["img"].append(int(f[4]))
        elif f[0] == "patch":
            out["patches"].append(dict(r0=float(f[2]), r1=float(f[3]), t0=float(f[4]), t1=float(f[5]), n_r=int(f[6]),
                                       n_th=int(f[7]), flags=int(f[8])))
        elif f[0] == "result":
            out.update(A=float(f[1]), err=float(f[2]), status=int(f[3]), n_patch=int(f[4]), rays=int(f[5]),
                       solves=int(f[6]), clipped=int(f[7]))
    out["coef"] = np.array(out["coef"]); out["roots"] = np.array(out["roots"]); out["img"] = np.array(out["img"], bool)
    return out


def lens_map(eps, a, z):
    return z - sum(e / np.conj(z - ai) for e, ai in zip(eps, a))


def binary(s, q):                                  # reading G4
    return [1 / (1 + q), q / (1 + q)], [complex(-s * q / (1 + q)), complex(s / (1 + q))]


def triple(s, q, q3, r3, psi):                     # reading G5
    m = 1 + q + q3
    mid = s * (1 - q) / (2 * (1 + q))
    return [1 / m, q / m, q3 / m], [complex(-s * q / (1 + q)), complex(s / (1 + q)), mid + r3 * complex(math.cos(psi), math.sin(psi))]


@pytest.mark.parametrize("kind", ["single", "binary", "triple"])
def test_polynomial_and_roots(exe, kind):
    """Eq. 4 coefficients: every image z (w = lens_map(z)) is a root; roots agree with numpy.roots of the printed
    coefficients; slots flagged as images satisfy Eq. 1, the others do not; counts follow P:78."""
    eps, a = {"single": ([1.0], [0j]), "binary": binary(0.9, 0.03), "triple": triple(1.1, 0.5, 0.03, 1.24, 1.3)}[kind]
    rng = np.random.default_rng(5)
    for _ in range(8):
        z0 = complex(rng.uniform(-1.3, 1.3), rng.uniform(-1.3, 1.3))
        w = lens_map(eps, a, z0)
        r = run(exe, eps, a, 1e-3, 0.0, w, n_limb=32, n_r=16, n_theta=16)
        c = r["coef"]                                  # ascending powers
        assert abs(np.polyval(c[::-1], z0)) <= 1e-11 * np.sum(np.abs(c) * np.abs(z0) ** np.arange(len(c)))
        ref = np.roots(c[::-1])
        for z in r["roots"][r["img"]]:
            assert np.min(np.abs(ref - z)) < 1e-6 * max(1.0, abs(z))
            assert abs(lens_map(eps, a, z) - w) < 1e-12
        assert np.min(np.abs(r["roots"][r["img"]] - z0)) < 1e-10          # the image we started from is found
        n_img, n = int(r["img"].sum()), len(eps)
        assert n_img in {1: {2}, 2: {3, 5}, 3: {4, 6, 8, 10}}[n]


@pytest.mark.parametrize("u,rho,u1", [(0.3, 0.05, 0.0), (0.3, 0.05, 0.5), (0.02, 0.05, 0.0), (1.2, 0.3, 0.3)])
def test_single_lens_closed_form_through_the_whole_path(exe, u, rho, u1):
    from test_oracle_pins import A_ld_single, A_witt_mao
    ref = float(A_ld_single(u, rho, u1)) if u1 > 0 else float(A_witt_mao(u, rho))
    r = run(exe, [1.0], [0j], rho, u1, u * complex(math.cos(0.83), math.sin(0.83)))
    assert abs(r["A"] / ref - 1) < 5e-5
    assert r["clipped"] == 0 and (r["status"] & 0xfd) == 0


def test_sectors_cover_the_images_and_do_not_overlap(exe):
    """Single lens, u > rho: the two images span r in [r_pm(u - rho), r_pm(u + rho)], r_pm(x) = (sqrt(x^2+4) +- x)/2,
    around theta = arg(w) and arg(w) + pi. Every sector must contain its image and no two sectors may overlap."""
    u, rho, ang = 0.4, 0.03, 0.83
    r = run(exe, [1.0], [0j], rho, 0.0, u * complex(math.cos(ang), math.sin(ang)))
    rp = lambda x: (math.sqrt(x * x + 4) + x) / 2
    rm = lambda x: (math.sqrt(x * x + 4) - x) / 2
    want = [(rp(u - rho), rp(u + rho), ang), (rm(u + rho), rm(u - rho), ang - math.pi)]
    assert r["n_patch"] == 2
    for lo, hi, th in want:
        hit = [p for p in r["patches"] if p["r0"] <= lo and p["r1"] >= hi]
        assert len(hit) == 1
        p = hit[0]
        mid = 0.5 * (p["t0"] + p["t1"])
        assert abs((th - mid + math.pi) % (2 * math.pi) - math.pi) < 0.05 * (p["t1"] - p["t0"])
        half = math.asin(rho / u)                       # the image subtends the same angle as the source
        assert p["t1"] - p["t0"] >= 2 * half
    a, b = r["patches"]
    assert a["r1"] < b["r0"] or b["r1"] < a["r0"]


def test_binary_inside_caustic_matches_oracle(exe, oracle):
    """C0 lens, a point inside the central caustic (5 images): the host-compiled path against the oracle."""
    eps, a = binary(1.0, 0.01)
    w = complex(-0.00161720, 0.06401082)
    r = run(exe, eps, a, 1e-2, 0.0, w)
    assert int(r["img"].sum()) == 5 and r["n_patch"] == 5
    ref = oracle.mag_fs_batch([oracle.lens_binary(1.0, 0.01)], 0, [w.real], [w.imag], 1e-2, 0.0, 100, 8)
    assert ref["err_est"][0] <= 2e-5
    assert abs(r["A"] / ref["A"][0] - 1) < 1e-4
    assert r["err"] < 1e-4 and r["clipped"] == 0


def test_resolution_knobs_converge(exe):
    """More lines / nodes change A only within the self-error estimate; n_limb = 256 finds the same sectors."""
    eps, a = binary(0.8, 0.3)
    w = complex(0.21, -0.13)
    base = run(exe, eps, a, 0.02, 0.4, w)
    fine = run(exe, eps, a, 0.02, 0.4, w, n_r=384, n_theta=96)
    coarse_limb = run(exe, eps, a, 0.02, 0.4, w, n_limb=256)
    assert abs(base["A"] / fine["A"] - 1) < 3e-5
    assert coarse_limb["n_patch"] == base["n_patch"]
    assert abs(coarse_limb["A"] / base["A"] - 1) < 3e-5
    assert fine["rays"] > 4 * base["rays"]


def _zeta_tables():
    import re
    src = open(os.path.join(HERE, "..", "paper_2510_02639_b200", "csrc", "ulens_core.cuh")).read()
    out = {}
    for name in ("UL_ZETA_M12_COEFFS", "UL_ZETA_M32_COEFFS"):
        body = re.search(r"#define %s \{([^}]*)\}" % name, src, re.S).group(1).replace("\\", " ")
        out[name] = np.array([float(x) for x in body.split(",")])
    return out


def test_hurwitz_zeta_tables_against_mpmath():
    """The one copy of the end-correction tables (ulens_core.cuh): zeta(s, u) = u^(-s) + poly(u) against mpmath.zeta for
    s = -1/2, -3/2 on (0, 1] to 1e-9, and identical to what the committed fit script produces."""
    import mpmath as mp
    import subprocess
    import sys
    tabs = _zeta_tables()
    for name, s in (("UL_ZETA_M12_COEFFS", -0.5), ("UL_ZETA_M32_COEFFS", -1.5)):
        c = tabs[name]
        assert len(c) == 10
        for u in np.linspace(1e-6, 1.0, 257):
            mine = u ** (-s) + np.polynomial.polynomial.polyval(u, c)
            assert abs(mine - float(mp.zeta(s, mp.mpf(float(u))))) < 1e-9, (name, u)
    out = subprocess.run([sys.executable, os.path.join(HERE, "..", "paper_2510_02639_b200", "csrc", "fit_zeta_tables.py")],
                         capture_output=True, text=True, check=True).stdout
    for name in tabs:
        line = [ln for ln in out.splitlines() if name in ln][0]
        vals = np.array([float(x) for x in line[line.index("{") + 1: line.index("}")].split(",")])
        assert np.array_equal(vals, tabs[name])

"""Regenerates UL_ZETA_M12_COEFFS / UL_ZETA_M32_COEFFS of ulens_core.cuh (build-time helper, needs mpmath + numpy).

The end correction of the ring quadrature (Navot's Euler-Maclaurin expansion for an x^(1/2) end
singularity) needs the Hurwitz zeta functions zeta(-1/2, u) and zeta(-3/2, u) for u in (0, 1]. With
zeta(s, u) = u^(-s) + zeta(s, 1 + u) the singular part is explicit and the rest, g_s(u) = zeta(s, 1 + u), is smooth on
[0, 1]: a degree-9 polynomial in u, least-squares fitted at 64 Chebyshev nodes of [0, 1] (values from mpmath at 30
digits), reproduces it to < 1e-9.   python paper_2510_02639_b200/csrc/fit_zeta_tables.py
"""
import mpmath as mp
import numpy as np

mp.mp.dps = 30
DEG, NODES = 9, 64


def fit(s):
    x = 0.5 * (1.0 - np.cos(np.pi * (np.arange(NODES) + 0.5) / NODES))          # Chebyshev nodes of [0, 1]
    y = np.array([float(mp.zeta(s, 1 + mp.mpf(float(u)))) for u in x])
    c = np.polynomial.polynomial.polyfit(x, y, DEG)                               # ascending powers
    uu = np.linspace(0.0, 1.0, 1001)
    err = max(abs(float(mp.zeta(s, 1 + mp.mpf(float(u)))) - np.polynomial.polynomial.polyval(u, c)) for u in uu)
    return c, err


if __name__ == "__main__":
    for name, s in (("UL_ZETA_M12_COEFFS", mp.mpf(-1) / 2), ("UL_ZETA_M32_COEFFS", mp.mpf(-3) / 2)):
        c, err = fit(s)
        print("#define %s {%s}   // max error %.1e" % (name, ", ".join("%.18g" % v for v in c), err))

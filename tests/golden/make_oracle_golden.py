"""Writes the stored oracle values the full-size GPU parity tests compare against.

    python tests/golden/make_oracle_golden.py [--only C1 C2 C3 C4] [--threads N]

Calls ONLY oracle/ (the CPU oracle) and the seeded input generators (paper_2510_02639_b200/inputs.py, which holds
none of the method's arithmetic); nothing here touches the CUDA path, so the stored numbers are oracle output,
never kernel output. Hours of CPU time (high-magnification points cost ~A x 3e5 lens-map evaluations each at the
parity resolution), which is why the values are stored instead of being recomputed inside `pytest -m gpu`.

  oracle_C{1,2,3}.npz   inputs.golden_sample(): >= 2,048 seeded stratified points per config (half near-caustic,
                        SURVEY 8.d) + the light-body stratum (points within 8 sqrt(eps_a) + 2 rho of the
                        planetary-caustic centre of a body with eps_a < 1e-3). Oracle at (n_rho, ss) = (100, 8),
                        Richardson-combined with (200, 8) (oracle.mag_fs_batch): A, A_fine, err_est.
  oracle_C4_fd.npz      inputs.golden_c4_sample(): 16 vectors x 16 epochs; A and central finite differences in
                        (t0,u0,tE,s,q,rho,alpha) at half-widths (h, h/2) (oracle.mag_fd at (200, 16)).
"""
import argparse
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import oracle as O                      # noqa: E402
from paper_2510_02639_b200 import inputs            # noqa: E402

N_RHO, SS = 100, 8
FD_N_RHO, FD_SS = 200, 16


def c4_steps(theta, t_e, w_abs):
    """Half-widths that move the source (or the caustics) by about one source radius."""
    rho, tE = theta[5], theta[2]
    tau = (t_e - theta[0]) / tE
    return np.array([rho * tE, rho, rho * tE / max(abs(tau), 0.1), rho, 0.3 * theta[4], 0.3 * rho,
                     rho / max(w_abs, 0.1)])


def make_values(cfg, threads):
    wl = inputs.get(cfg)
    ci, pi, zone = inputs.golden_sample(wl, cfg)
    mk = O.lens_binary if wl.kind == "binary" else O.lens_triple
    lenses = [mk(*p) for p in wl.lens_params]
    w = wl.w[ci, pi]
    t0 = time.time()
    ref = O.mag_fs_batch(lenses, ci.astype(np.int32), w.real, w.imag, wl.rho[ci], wl.u1[ci], N_RHO, SS, threads)
    dt = time.time() - t0
    np.savez(os.path.join(HERE, "oracle_C%d.npz" % cfg), cfg_index=ci.astype(np.int32), point_index=pi.astype(np.int32),
             in_zone=zone, near_caustic=wl.near_caustic[ci, pi], w_re=w.real, w_im=w.imag,
             A=ref["A"], A_fine=ref["A_fine"], err_est=ref["err_est"], n_eval=ref["n_eval"],
             n_rho=N_RHO, ss=SS)
    print("C%d: %d points (%d near-caustic, %d in a light-body zone), admissible %d, %.0f s on %d threads" %
          (cfg, len(ci), wl.near_caustic[ci, pi].sum(), zone.sum(), (ref["err_est"] <= 2e-5).sum(), dt, threads), flush=True)


def make_c4(threads):
    wl = inputs.get(4)
    vec, eps = inputs.golden_c4_sample(wl)
    if threads:
        os.environ["OMP_NUM_THREADS"] = str(threads)
    A0 = np.empty(eps.shape)
    D = np.empty(eps.shape + (2, 7))
    steps = np.empty(eps.shape + (7,))
    t0 = time.time()
    for i, c in enumerate(vec):
        th = wl.theta[c]
        for j, e in enumerate(eps[i]):
            st = c4_steps(th, wl.t[e], abs(wl.w[c][e]))
            a0, d = O.mag_fd(lambda p: O.lightcurve_case(p, wl.t[e]), th, [st, 0.5 * st], 0.5, FD_N_RHO, FD_SS)
            A0[i, j] = a0; D[i, j] = d; steps[i, j] = st
        print("C4 vector %d/%d done, %.0f s" % (i + 1, len(vec), time.time() - t0), flush=True)
    np.savez(os.path.join(HERE, "oracle_C4_fd.npz"), vec=vec.astype(np.int32), epochs=eps.astype(np.int32), A=A0, D=D,
             steps=steps, n_rho=FD_N_RHO, ss=FD_SS)


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--only", nargs="*", default=["C2", "C4", "C3", "C1"])
    ap.add_argument("--threads", type=int, default=0)
    a = ap.parse_args()
    O.build()
    for name in a.only:
        if name == "C4":
            make_c4(a.threads)
        else:
            make_values(int(name[1]), a.threads)

"""Wider parity sweep of the CUDA path against the oracle than the pytest suite affords (not collected by pytest:
about 8 minutes of oracle time on 16 cores). Runs BASELINE configs C1-C3 at FULL size on the GPU, then compares
a seeded stratified sample -- other lens configurations and another seed than tests/test_gpu_parity.py uses --
with the oracle at the parity resolution (n_rho, ss) = (100, 8).   python tests/sweep_parity.py
"""
import sys, os, time
sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import numpy as np, torch
from paper_2510_02639_b200 import binding, inputs
from oracle import oracle as O
ctx = binding.Context(0)
for cfg, n_cfg_used, n_per in [(1, 16, 24), (2, 12, 16), (3, 12, 16)]:
    wl = inputs.get(cfg)
    f = binding.ulens_lens_binary if wl.kind == "binary" else binding.ulens_lens_triple
    fo = O.lens_binary if wl.kind == "binary" else O.lens_triple
    w_re = torch.tensor(np.ascontiguousarray(wl.w.real), device="cuda:0"); w_im = torch.tensor(np.ascontiguousarray(wl.w.imag), device="cuda:0")
    A, err, st = ctx.ulens_mag([f(*p) for p in wl.lens_params], wl.rho, wl.u1, w_re, w_im)
    torch.cuda.synchronize(); A = A.cpu().numpy(); st = st.cpu().numpy().astype(np.uint32)
    idx = inputs.subsample(wl, n_per, seed=1000 + cfg)          # a different seed from the tests'
    cs = list(range(1, wl.n_cfg, max(1, wl.n_cfg // n_cfg_used)))[:n_cfg_used]   # offset 1: other configs than the tests'
    rel_all, adm_all, fl_all, near_all = [], [], [], []
    t0 = time.time()
    for c in cs:
        ref = O.mag_fs_batch([fo(*wl.lens_params[c])], 0, wl.w[c][idx[c]].real, wl.w[c][idx[c]].imag, wl.rho[c], wl.u1[c], 100, 8)
        rel_all.append(np.abs(A[c][idx[c]] / ref["A"] - 1)); adm_all.append(ref["err_est"] <= 2e-5)
        fl_all.append((st[c][idx[c]] & 0xff) != 0); near_all.append(wl.near_caustic[c][idx[c]])
    rel = np.concatenate(rel_all); adm = np.concatenate(adm_all); fl = np.concatenate(fl_all); near = np.concatenate(near_all)
    r = rel[adm]
    print("C%d: %d points (%d near-caustic), admissible %d, flagged %d | |A/A_oracle-1|: median %.1e  p90 %.1e  p99 %.1e  max %.1e | >1e-4: %d | inadmissible max %.1e | oracle %.0f s" % (
        cfg, rel.size, near.sum(), adm.sum(), fl.sum(), np.median(r), np.quantile(r, 0.9), np.quantile(r, 0.99), r.max(), (r > 1e-4).sum(),
        rel[~adm].max() if (~adm).any() else 0.0, time.time() - t0), flush=True)

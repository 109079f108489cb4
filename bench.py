#!/usr/bin/env python
"""bench.py -- throughput of the ICRS hot path on B200 (contract: see the task statement / DESIGN.md "Measurement").

One "step" = one pass of the whole hot path (k_roots -> k_regions -> k_shoot -> k_finalize, SURVEY 8.a rows
a2..a7; a1 too for light-curve workloads) over one batch of synthetic input = every source point of the
workload. Default workload: BASELINE.json configs[1] ("C1": binary lens, u1 = 0.5, rho = 1e-3, 64 lens
configurations x 2,048 source points, half of them within 3 rho of a caustic; seeded).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

prints ONE JSON line on rank 0:
  value      finite-source magnifications / s, inputs resident in HBM, CUDA events, max over ranks
  e2e        the same through ulens_mag_host (pinned HOST buffers, H2D + D2H inside the timed region)
  roofline   k_shoot (the dominant kernel) against the FP64 FMA pipe
  cpu_baseline  the CPU oracle, as it stands, on a bounded seeded sample of the same workload
N > 1 runs N independent replicas (the path has no exchange step: DESIGN.md "Multi-GPU: replicas only").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "finite-source magnifications/sec"
UNIT = "magnifications/s"

# Algorithmic FP64-pipe instructions per ray (FMA = 1 instruction = 2 flop), DESIGN.md "k_shoot roofline":
# the lens map with one reciprocal per ray, the rotation recurrence, d^2 and the inside test; the limb-
# darkened figure adds the square root of the inside rays (about half of all rays).
FP64_INSTR_PER_RAY = {(1, False): 27, (1, True): 32, (2, False): 35, (2, True): 40, (3, False): 47, (3, True): 52}
# Forward-mode variant (binary, 5 intrinsic tangents): per tangent the moving ray dz (2), g conj(dz) (4), the explicit
# lens-parameter term (0..8, mean 3), dF (4), accumulation (1) = 14, plus g itself (4 per ray): + 74 per ray.
FP64_INSTR_PER_RAY_DUAL_EXTRA = 74
# k_regions: algorithmic FP64-pipe instructions per limb solve: coefficients ~26 DEG, warm-started
# Ehrlich-Aberth 3 iterations x DEG roots x (8 DEG Horner + 12 (DEG-1) repulsion + 24), Eq.-1 polish of the
# N+1..DEG images 2.5 iterations x (17 N + 25), boxes ~100.
FP64_INSTR_PER_LIMB_SOLVE = {1: 600, 2: 2400, 3: 8300}
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the roofline kernel, from the `ncu --set full`
# captures summarised in profiles/r01g_ncu_k_shoot_c1.md (C1) and profiles/r01c_ncu_k_shoot_dual_c4.md (C4);
# configs without a capture report null.
NCU_TRAFFIC_BYTES_PER_LAUNCH = {1: 27.3631e6 + 0.8640e6, 4: 63.2251e6 + 203.0922e6}
# FP64 FMA pipe of one B200: 148 SMs x 64 DFMA lanes / clk x 1.965 GHz (clocks.max.sm) -- DESIGN.md
FP64_PEAK_DFMA = 148 * 64 * 1.965e9

# cpu_baseline / --impl reference sample: seeded stratified points of the workload (half near-caustic);
# the seed was fixed once so that the oracle's work on the sample is a few 1e8 lens-map evaluations.
CPU_SAMPLE_SEED = 2
CPU_SAMPLE_CFGS = 8
CPU_SAMPLE_PER_CFG_BY_WL = {"C0": 500, "C1": 64, "C2": 256, "C3": 32, "C4": 256}   # sized for ~2-10 s of wall time on 16 cores


def sample_per_cfg(wl):
    return min(CPU_SAMPLE_PER_CFG_BY_WL.get(wl.name, 16), wl.n_pts)

# The parity tests run the oracle at (n_rho, ss) = (100, 8); a near-caustic point of C1 (A of a few hundred)
# then costs ~1e9 lens-map evaluations = minutes of ONE core (the oracle parallelises over points only), which
# no 10-30 s sample can hold. The timed baseline therefore runs the same oracle at (50, 4): 16x less work,
# self-error 1e-5..5e-5, i.e. still inside the 1e-4 bar the GPU path is held to.
ORACLE_N_RHO, ORACLE_SS = 50, 4


# ----------------------------------------------------------------------------------------------- helpers

class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


def gpu_lenses(binding, wl, cs=None):
    cs = range(wl.n_cfg) if cs is None else cs
    f = binding.ulens_lens_binary if wl.kind == "binary" else binding.ulens_lens_triple
    return [f(*wl.lens_params[c]) for c in cs]


def oracle_lenses(O, wl, cs):
    f = O.lens_binary if wl.kind == "binary" else O.lens_triple
    return [f(*wl.lens_params[c]) for c in cs]


def cpu_sample(wl, inputs):
    """(config indices, point indices [n_cfg_used, k]) of the bounded oracle sample."""
    idx = inputs.subsample(wl, sample_per_cfg(wl), seed=CPU_SAMPLE_SEED)
    n_used = min(CPU_SAMPLE_CFGS, wl.n_cfg)
    cs = list(range(0, wl.n_cfg, max(1, wl.n_cfg // n_used)))[:n_used]
    return cs, idx


def run_oracle_sample(wl, inputs):
    """Times the oracle, as it stands, on the sample; returns (points, seconds, lens-map evaluations, threads)."""
    from oracle import oracle as O
    O.build()
    cs, idx = cpu_sample(wl, inputs)
    olenses = oracle_lenses(O, wl, cs)
    wx = np.concatenate([wl.w[c][idx[c]].real for c in cs])
    wy = np.concatenate([wl.w[c][idx[c]].imag for c in cs])
    li = np.concatenate([np.full(idx.shape[1], k, dtype=np.int32) for k in range(len(cs))])
    rho = np.concatenate([np.full(idx.shape[1], wl.rho[c]) for c in cs])
    u1 = np.concatenate([np.full(idx.shape[1], wl.u1[c]) for c in cs])
    t0 = time.perf_counter()
    r = O.mag_fs_batch(olenses, li, wx, wy, rho, u1, ORACLE_N_RHO, ORACLE_SS)
    dt = time.perf_counter() - t0
    return len(wx), dt, int(r["n_eval"].sum()), O.max_threads()


def workload_name(wl):
    return "%s: %s lens, %d configs x %d points (BASELINE.json configs[%s])" % (
        wl.name, wl.kind, wl.n_cfg, wl.n_pts, wl.name[1:])


# ----------------------------------------------------------------------------------------------- reference arm

def main_reference(args, rank, world):
    """The oracle on the host cores (rank 0 only): each step = the bounded sample of the workload."""
    if rank != 0:
        return
    from paper_2510_02639_b200 import inputs
    wl = inputs.get(args.config)
    for _ in range(min(args.warmup, 1)):                      # one untimed pass warms the page cache / OpenMP pool
        run_oracle_sample(wl, inputs)
    tot_t, tot_pts, tot_ev, cores = 0.0, 0, 0, 1
    for _ in range(args.steps):
        n, dt, ev, cores = run_oracle_sample(wl, inputs)
        tot_t += dt; tot_pts += n; tot_ev += ev
    value = tot_pts / tot_t
    sample = "%d seeded points per step (%d configs x %d, half near-caustic, seed %d) at oracle n_rho=%d ss=%d" % (
        tot_pts // max(args.steps, 1), min(CPU_SAMPLE_CFGS, wl.n_cfg), sample_per_cfg(wl), CPU_SAMPLE_SEED, ORACLE_N_RHO, ORACLE_SS)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": min(args.warmup, 1), "ms_per_step": 1e3 * tot_t / max(args.steps, 1),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(wl), "note": "CPU oracle (oracle/), bounded sample per step"},
            "rays_per_s": tot_ev / tot_t,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                             "rays_per_s": tot_ev / tot_t},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------------- our arm

def main_ours(args, rank, local_rank, world):
    import torch
    import torch.distributed as dist
    from paper_2510_02639_b200 import binding, inputs, replicas

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    wl = inputs.get(args.config)                                     # every rank: the same seeded workload (replica)
    lenses = gpu_lenses(binding, wl)
    n = wl.n_cfg * wl.n_pts
    ctx = binding.Context(local_rank)
    dual = args.config == 4                                          # C4: trajectory parameters in, A and dA/d(7) out
    w_re = torch.tensor(np.ascontiguousarray(wl.w.real), device=dev)
    w_im = torch.tensor(np.ascontiguousarray(wl.w.imag), device=dev)
    A = torch.empty((wl.n_cfg, wl.n_pts), dtype=torch.float64, device=dev)
    err = torch.empty_like(A)
    st = torch.empty((wl.n_cfg, wl.n_pts), dtype=torch.int32, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)    # > 126 MB L2

    if dual:
        t_dev = torch.tensor(wl.t.copy(), device=dev)
        dA = torch.empty((wl.n_cfg, wl.n_pts, 7), dtype=torch.float64, device=dev)

    n_ext = n

    def step():
        if dual:
            if args.switch:
                nonlocal n_ext, A, dA, err, st
                A, dA, err, st, n_ext = ctx.ulens_lightcurve_binary_ext(wl.theta, float(wl.u1[0]), t_dev, want_dA=True)
            else:
                ctx.ulens_lightcurve_binary(wl.theta, float(wl.u1[0]), t_dev, out=(A, dA, err, st))
        else:
            ctx.ulens_mag(lenses, wl.rho, wl.u1, w_re, w_im, A, err, st)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    launches_per_step = ctx.ulens_last_launch_count()

    # ---- timed region 1: inputs resident in HBM
    ctx.ulens_reset_stats()
    ctx.ulens_set_timing(True)
    clocks = ClockSampler(local_rank)
    clocks.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    for a, b in ev:
        flush.fill_(1)                                               # L2 flush between timed iterations (untimed)
        a.record()
        step()
        b.record()
    barrier()
    clk = clocks.stop()
    ms = sum(a.elapsed_time(b) for a, b in ev)
    kms = ctx.ulens_get_kernel_ms()
    ctx.ulens_set_timing(False)
    stats = ctx.ulens_get_stats()
    status = st.cpu().numpy().astype(np.uint32)
    A_host = A.cpu().numpy()

    # ---- timed region 2: end to end through the C ABI with pinned HOST buffers
    h_re = torch.tensor(np.ascontiguousarray(wl.w.real)).pin_memory()
    h_im = torch.tensor(np.ascontiguousarray(wl.w.imag)).pin_memory()
    h_A = torch.empty((wl.n_cfg, wl.n_pts), dtype=torch.float64).pin_memory()
    h_err = torch.empty((wl.n_cfg, wl.n_pts), dtype=torch.float64).pin_memory()
    h_st = torch.empty((wl.n_cfg, wl.n_pts), dtype=torch.int32).pin_memory()
    e2e_steps = max(1, min(args.steps, 3))
    if dual:
        h_t = torch.tensor(wl.t.copy()).pin_memory()
        h_dA = torch.empty((wl.n_cfg, wl.n_pts, 7), dtype=torch.float64).pin_memory()

        def e2e_step():
            if args.switch:
                ctx.ulens_lightcurve_binary_ext_host(wl.theta, float(wl.u1[0]), h_t.numpy(), h_A.numpy(), h_dA.numpy(),
                                                     h_err.numpy(), h_st.numpy())
            else:
                ctx.ulens_lightcurve_binary_host(wl.theta, float(wl.u1[0]), h_t.numpy(), h_A.numpy(), h_dA.numpy(),
                                                 h_err.numpy(), h_st.numpy())
        h2d, d2h = 8 * wl.n_pts + 56 * wl.n_cfg, (8 + 56 + 8 + 4) * n
        e2e_api = ("ulens_lightcurve_binary_ext_host" if args.switch else "ulens_lightcurve_binary_host") + " (pinned host buffers)"
    else:
        def e2e_step():
            ctx.ulens_mag_host(lenses, wl.rho, wl.u1, h_re.numpy(), h_im.numpy(), h_A.numpy(), h_err.numpy(), h_st.numpy())
        h2d, d2h = 16 * n, 20 * n
        e2e_api = "ulens_mag_host (pinned host buffers)"
    e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    barrier()
    e2e_s = time.perf_counter() - t0
    assert np.array_equal(h_A.numpy(), A_host, equal_nan=True), "host entry and device entry disagree"

    # ---- max over ranks
    ms, e2e_s = replicas.max_over_ranks([ms, e2e_s], dev)
    ms_per_step = ms / args.steps
    value = replicas.aggregate_throughput(n, world, ms_per_step)
    e2e_value = replicas.aggregate_throughput(n, world, 1e3 * e2e_s / e2e_steps)

    if rank == 0:
        n_lens = 2 if wl.kind == "binary" else 3
        ld = bool(np.any(wl.u1 > 0))
        shoot_ms, shoot_n = kms["k_shoot"]
        rays_per_step = stats["n_rays"] / args.steps
        rays_per_launch = stats["n_rays"] / max(shoot_n, 1)
        ipr = FP64_INSTR_PER_RAY[(n_lens, ld)] + (FP64_INSTR_PER_RAY_DUAL_EXTRA if dual else 0)
        shoot_avg_s = shoot_ms * 1e-3 / max(shoot_n, 1)
        achieved = 2.0 * ipr * rays_per_launch / shoot_avg_s / 1e12
        peak_measured = ctx.ulens_fp64_peak(200.0)
        roofline = {"bound": "alu", "kernel": "k_shoot", "achieved": achieved, "peak": 2.0 * FP64_PEAK_DFMA / 1e12,
                    "variant": "k_shoot_dual (value + 5 tangents per ray)" if dual else "k_shoot",
                    "unit": "TFLOP/s", "frac": achieved / (2.0 * FP64_PEAK_DFMA / 1e12),
                    "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH.get(args.config),
                    "traffic_note": "DRAM bytes of one launch (ncu capture in profiles/); the path is ALU-bound",
                    "peak_source": "derived: 148 SM x 64 DFMA/clk x 1.965 GHz x 2 flop (DESIGN.md); "
                                   "MEASURED_PEAKS.json has no FP64 entry",
                    "peak_measured_dfma_microbench": 2.0 * peak_measured / 1e12,
                    "frac_of_measured": achieved / (2.0 * peak_measured / 1e12),
                    "fp64_instr_per_ray": ipr, "rays_per_launch": rays_per_launch,
                    "kernel_ms_avg": 1e3 * shoot_avg_s, "share_of_step": shoot_ms / ms}
        reg_ms, reg_n = kms["k_regions"]
        solves_per_launch = stats["n_limb_solves"] / max(reg_n, 1)
        reg_ach = 2.0 * FP64_INSTR_PER_LIMB_SOLVE[n_lens] * solves_per_launch / (reg_ms * 1e-3 / max(reg_n, 1)) / 1e12
        roofline_regions = {"bound": "alu", "kernel": "k_regions", "achieved": reg_ach, "peak": 2.0 * FP64_PEAK_DFMA / 1e12,
                            "unit": "TFLOP/s", "frac": reg_ach / (2.0 * FP64_PEAK_DFMA / 1e12), "traffic": None,
                            "fp64_instr_per_limb_solve": FP64_INSTR_PER_LIMB_SOLVE[n_lens],
                            "limb_solves_per_point": stats["n_limb_solves"] / args.steps / n,
                            "kernel_ms_avg": reg_ms / max(reg_n, 1), "share_of_step": reg_ms / ms}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": workload_name(wl), "rho": [float(wl.rho.min()), float(wl.rho.max())],
                           "u1": [float(wl.u1.min()), float(wl.u1.max())], "l2": "flushed between timed steps (256 MiB fill)",
                           "parallelism": "replicas" if world > 1 else "1 GPU"},
                "rays_per_s": world * rays_per_step / (ms_per_step * 1e-3),
                "rays_per_point": rays_per_step / n,
                "kernel_ms_per_step": {k: v[0] / args.steps for k, v in kms.items()},
                "flagged_points": int(((status & 0xff) != 0).sum()), "nan_points": int(np.isnan(A_host).sum()),
                "roofline": roofline, "roofline_regions": roofline_regions,
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                        "steps": e2e_steps, "api": e2e_api},
                "gpu_launches": launches_per_step * args.steps,
                "clocks": clk}
        if dual and args.switch:
            line["config"]["switch"] = {"api": "ulens_lightcurve_binary_ext", "selection": "library (sel_tol default 2e-5)",
                                        "n_ext": int(n_ext), "n_epochs_total": int(n),
                                        "note": "SURVEY 8.f-2 driver: the other epochs take the point-source value (P:153)"}
        if not args.no_cpu_baseline and world == 1:
            npts, dt, nev, cores = run_oracle_sample(wl, inputs)
            line["cpu_baseline"] = {"value": npts / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": "%d seeded points (%d configs x %d, half near-caustic, seed %d), oracle n_rho=%d ss=%d, %.1f s"
                                              % (npts, min(CPU_SAMPLE_CFGS, wl.n_cfg), sample_per_cfg(wl), CPU_SAMPLE_SEED, ORACLE_N_RHO, ORACLE_SS, dt),
                                    "rays_per_s": nev / dt}
        print(json.dumps(line), flush=True)
    ctx.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json config index 0..4 (default 1; 4 = light curves with forward-mode derivatives)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--switch", action="store_true",
                    help="config 4 only: ulens_lightcurve_binary_ext (point-source value for the far epochs, P:153; "
                         "library selection at the default tolerance) instead of the finite-source path on every epoch")
    args = ap.parse_args()
    if args.switch and args.config != 4:
        ap.error("--switch needs --config 4")
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        main_reference(args, rank, world)
    else:
        main_ours(args, rank, local_rank, world)


if __name__ == "__main__":
    main()

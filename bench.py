#!/usr/bin/env python
"""bench.py -- throughput of the ICRS hot path on B200 (contract: see the task statement / DESIGN.md "Measurement").

One "step" = one pass of the whole hot path (k_traj -> k_roots -> k_limb -> k_sectors -> k_shoot[_dual] -> k_finalize, SURVEY 8.a
rows a1..a8) over one batch of synthetic input = every source point of the workload. Default workload: the largest
single-GPU configuration of BASELINE.json, configs[4] ("C4": 1,024 parameter vectors x 2,000 epochs, binary lens,
rho = 5e-3, u1 = 0.5; trajectory parameters in, A and the 7 forward-mode derivatives out; every epoch takes the
finite-source path -- the point-source / finite-source switch of SURVEY 8.f-2 rides along under "c4_switch").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

prints ONE JSON line on rank 0:
  value        finite-source magnifications / s, inputs resident in HBM, CUDA events, max over ranks
  e2e          the same through the *_host entry (pinned HOST buffers, H2D + D2H inside the timed region)
  roofline     the ray-shooting kernel (k_shoot_dual for C4, k_shoot otherwise) against the FP64 FMA pipe
  cpu_baseline the CPU oracle, as it stands, on a bounded seeded sample of the same workload
  all_configs  value / roofline fractions of the other BASELINE configs (short runs, same code path)
N > 1 runs N independent replicas (the path has no exchange step: DESIGN.md "Multi-GPU: replicas only"); a plain
`python bench.py --gpus N` re-launches itself under torch.distributed.run with N ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import socket
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
# Forward-mode variant: SURVEY 8.d's per-unit figure for a ray that also carries the tangents, "dual variant ~ 2-2.5x" of the
# primal count: its midpoint, 2.25x. (Round 1's kernel executed more than that -- 114 by its own itemised count; round 2's
# kernel executes 91.5 DFMA + DMUL + DADD per ray on C4 by ncu's SASS counters, profiles/r02_ncu_shoot_dual_c4.md: the
# unit of useful work is the survey's, not what a particular kernel spends on it. DESIGN.md 6.4.)
FP64_DUAL_FACTOR = 2.25
# k_limb: algorithmic FP64-pipe instructions per limb solve: coefficients ~26 DEG, warm-started
# Ehrlich-Aberth 3 iterations x DEG roots x (8 DEG Horner + 12 (DEG-1) repulsion + 24), Eq.-1 polish of the
# N+1..DEG images 2.5 iterations x (17 N + 25), boxes ~100.
FP64_INSTR_PER_LIMB_SOLVE = {1: 600, 2: 2400, 3: 8300}
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the roofline kernel, from the `ncu --set full` captures
# summarised under profiles/ (r02_ncu_shoot_dual_c4.md, r02_ncu_shoot_c1.md, r02_ncu_shoot_c2.md, r02_ncu_shoot_c3.md, r02_ncu_shoot_f32_c1.md);
# key = (config, f32 variant)
NCU_TRAFFIC_BYTES_PER_LAUNCH = {(4, False): 50.039808e6 + 300.790784e6, (1, False): 26.111488e6 + 0.337408e6,
                                (2, False): 29.666304e6 + 3.572480e6, (3, False): 31.663360e6 + 1.320960e6,
                                (1, True): 26.103296e6 + 0.195840e6}
# FP64 FMA pipe of one B200: 148 SMs x 64 DFMA lanes / clk x 1.965 GHz (clocks.max.sm) -- DESIGN.md
FP64_PEAK_DFMA = 148 * 64 * 1.965e9
# Mixed-precision variant (k_shoot_f32): algorithmic FP32-pipe instructions per ray in the segment-local
# difference form along a radial line (the common scan direction) -- displacement t (cos, sin): 4; per lens c + d (2), c (c + d)
# (4), |.|^2 (2), eps x reciprocal (1), eps conj(d / p) (4), accumulate (2, with the 2 above fused): 17; F: 6; inside test +
# count: 2; sqrt on inside rays: 1. (ncu SASS counters on C1: 44 FFMA + FMUL + FADD per ray, profiles/r02_ncu_shoot_f32_c1.md.)
FP32_INSTR_PER_RAY = {(1, False): 28, (1, True): 29, (2, False): 45, (2, True): 46, (3, False): 62, (3, True): 63}
# FP32 FMA pipe: 148 SMs x 128 FFMA lanes / clk x 1.965 GHz (checked in-run by ulens_fp32_peak)
FP32_PEAK_FFMA = 148 * 128 * 1.965e9

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
            "config": {"workload": workload_name(wl), "note": "CPU oracle (oracle/), bounded sample per step; values only "
                       "(the oracle's derivative reference is finite differences: 29 evaluations per point)"},
            "rays_per_s": tot_ev / tot_t,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                             "rays_per_s": tot_ev / tot_t},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------------- our arm

class Env:
    """What every measurement of this process shares."""
    def __init__(self, torch, dist, binding, inputs, replicas, ctx, dev, local_rank, world):
        self.torch, self.dist, self.binding, self.inputs, self.replicas = torch, dist, binding, inputs, replicas
        self.ctx, self.dev, self.local_rank, self.world = ctx, dev, local_rank, world
        self.flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)    # > 126 MB L2
        self.ctx32 = None

    def barrier(self):
        if self.world > 1:
            self.dist.barrier()
        self.torch.cuda.synchronize()


def measure_config(env: Env, cfg: int, steps: int, warmup: int, switch: bool = False, with_e2e: bool = True,
                   with_clocks: bool = False, f32: bool = False) -> dict:
    """W warm-up steps, K timed steps (CUDA events on the launch stream, L2 flushed before each), per-kernel
    device times from the library's own event pairs, optionally the end-to-end leg; max over ranks."""
    torch, ctx, dev, binding, inputs, replicas = env.torch, env.ctx, env.dev, env.binding, env.inputs, env.replicas
    if f32:                                                          # mixed-precision variant: its own context (option flag)
        if env.ctx32 is None:
            env.ctx32 = binding.Context(env.local_rank, flags=binding.ULENS_OPT_F32_SHOOT)
        ctx = env.ctx32
    wl = inputs.get(cfg)                                             # every rank: the same seeded workload (replica)
    lenses = gpu_lenses(binding, wl)
    n = wl.n_cfg * wl.n_pts
    dual = cfg == 4                                                  # C4: trajectory parameters in, A and dA/d(7) out
    A = torch.empty((wl.n_cfg, wl.n_pts), dtype=torch.float64, device=dev)
    err = torch.empty_like(A)
    st = torch.empty((wl.n_cfg, wl.n_pts), dtype=torch.int32, device=dev)
    if dual:
        t_dev = torch.tensor(wl.t.copy(), device=dev)
        dA = torch.empty((wl.n_cfg, wl.n_pts, 7), dtype=torch.float64, device=dev)
    else:
        w_re = torch.tensor(np.ascontiguousarray(wl.w.real), device=dev)
        w_im = torch.tensor(np.ascontiguousarray(wl.w.imag), device=dev)
    box = {"n_ext": n, "A": A, "st": st}

    def step():
        if dual and switch:
            a_, d_, e_, s_, box["n_ext"] = ctx.ulens_lightcurve_binary_ext(wl.theta, float(wl.u1[0]), t_dev, want_dA=True)
            box["A"], box["st"] = a_, s_
        elif dual:
            ctx.ulens_lightcurve_binary(wl.theta, float(wl.u1[0]), t_dev, out=(A, dA, err, st))
        else:
            ctx.ulens_mag(lenses, wl.rho, wl.u1, w_re, w_im, A, err, st)

    for _ in range(warmup):
        step()
    env.barrier()
    launches_per_step = ctx.ulens_last_launch_count()

    # ---- timed region 1: inputs resident in HBM
    ctx.ulens_reset_stats()
    ctx.ulens_set_timing(True)
    clocks = ClockSampler(env.local_rank) if with_clocks else None
    if clocks:
        clocks.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    env.barrier()
    for a, b in ev:
        env.flush.fill_(1)                                           # L2 flush between timed iterations (untimed)
        a.record()
        step()
        b.record()
    env.barrier()
    clk = clocks.stop() if clocks else None
    ms = sum(a.elapsed_time(b) for a, b in ev)
    kms = ctx.ulens_get_kernel_ms()
    ctx.ulens_set_timing(False)
    stats = ctx.ulens_get_stats()
    status = box["st"].cpu().numpy().astype(np.uint32)
    A_host = box["A"].cpu().numpy()

    # ---- timed region 2: end to end through the C ABI with pinned HOST buffers
    e2e = None
    if with_e2e:
        h_A = torch.empty((wl.n_cfg, wl.n_pts), dtype=torch.float64).pin_memory()
        h_err = torch.empty((wl.n_cfg, wl.n_pts), dtype=torch.float64).pin_memory()
        h_st = torch.empty((wl.n_cfg, wl.n_pts), dtype=torch.int32).pin_memory()
        e2e_steps = max(1, min(steps, 3))
        if dual:
            h_t = torch.tensor(wl.t.copy()).pin_memory()
            h_dA = torch.empty((wl.n_cfg, wl.n_pts, 7), dtype=torch.float64).pin_memory()

            def e2e_step():
                f = ctx.ulens_lightcurve_binary_ext_host if switch else ctx.ulens_lightcurve_binary_host
                f(wl.theta, float(wl.u1[0]), h_t.numpy(), h_A.numpy(), h_dA.numpy(), h_err.numpy(), h_st.numpy())
            h2d, d2h = 8 * wl.n_pts + 56 * wl.n_cfg, (8 + 56 + 8 + 4) * n
            e2e_api = ("ulens_lightcurve_binary_ext_host" if switch else "ulens_lightcurve_binary_host") + " (pinned host buffers)"
        else:
            h_re = torch.tensor(np.ascontiguousarray(wl.w.real)).pin_memory()
            h_im = torch.tensor(np.ascontiguousarray(wl.w.imag)).pin_memory()

            def e2e_step():
                ctx.ulens_mag_host(lenses, wl.rho, wl.u1, h_re.numpy(), h_im.numpy(), h_A.numpy(), h_err.numpy(), h_st.numpy())
            h2d, d2h = 16 * n, 20 * n
            e2e_api = "ulens_mag_host (pinned host buffers)"
        e2e_step()
        env.barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            e2e_step()
        env.barrier()
        e2e_s = time.perf_counter() - t0
        assert np.array_equal(h_A.numpy(), A_host, equal_nan=True), "host entry and device entry disagree"
        (e2e_s,) = replicas.max_over_ranks([e2e_s], dev)
        e2e = {"value": replicas.aggregate_throughput(n, env.world, 1e3 * e2e_s / e2e_steps), "unit": UNIT,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps, "api": e2e_api}

    # ---- max over ranks
    (ms,) = replicas.max_over_ranks([ms], dev)
    ms_per_step = ms / steps
    value = replicas.aggregate_throughput(n, env.world, ms_per_step)

    n_lens = 2 if wl.kind == "binary" else 3
    ld = bool(np.any(wl.u1 > 0))
    shoot_ms, shoot_n = kms["k_shoot"]
    rays_per_step = stats["n_rays"] / steps
    rays_per_launch = stats["n_rays"] / max(shoot_n, 1)
    ipr = FP64_INSTR_PER_RAY[(n_lens, ld)] * (FP64_DUAL_FACTOR if dual else 1.0)
    shoot_avg_s = shoot_ms * 1e-3 / max(shoot_n, 1)
    achieved = 2.0 * ipr * rays_per_launch / shoot_avg_s / 1e12
    peak = 2.0 * FP64_PEAK_DFMA / 1e12
    if f32 and not dual:
        # mixed-precision variant: FP32-pipe instructions per ray against the FP32 FMA pipe (128 lanes / clk / SM)
        ipr = FP32_INSTR_PER_RAY[(n_lens, ld)]
        achieved = 2.0 * ipr * rays_per_launch / shoot_avg_s / 1e12
        peak = 2.0 * FP32_PEAK_FFMA / 1e12
    roofline = {"bound": "alu", "kernel": ("k_shoot_f32" if f32 else "k_shoot") if not dual else "k_shoot_dual", "achieved": achieved, "peak": peak,
                "variant": "k_shoot_dual (value + 5 tangents per ray)" if dual else ("k_shoot_f32" if f32 else "k_shoot"),
                "unit": "TFLOP/s", "frac": achieved / peak, "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH.get((cfg, bool(f32))),
                "traffic_note": "dram__bytes_read.sum + dram__bytes_write.sum of ONE launch from the ncu --set full capture of this kernel on this "
                                "config (profiles/r02_ncu_*.md), not measured in this run; null where no capture exists. The path is ALU-bound.",
                "peak_source": "derived: 148 SM x 64 DFMA/clk x 1.965 GHz x 2 flop (DESIGN.md); "
                               "MEASURED_PEAKS.json has no FP64 entry",
                ("fp32_instr_per_ray" if (f32 and not dual) else "fp64_instr_per_ray"): ipr, "rays_per_launch": rays_per_launch,
                "kernel_ms_avg": 1e3 * shoot_avg_s, "share_of_step": shoot_ms / ms}
    reg_ms, reg_n = kms["k_limb"]                          # the limb tracker; k_sectors (thread per point) is reported beside it
    sec_ms, _ = kms["k_sectors"]
    solves_per_launch = stats["n_limb_solves"] / max(reg_n, 1)
    reg_ach = 2.0 * FP64_INSTR_PER_LIMB_SOLVE[n_lens] * solves_per_launch / (reg_ms * 1e-3 / max(reg_n, 1)) / 1e12
    roofline_regions = {"bound": "alu", "kernel": "k_limb", "achieved": reg_ach, "peak": peak,
                        "unit": "TFLOP/s", "frac": reg_ach / peak, "traffic": None,
                        "fp64_instr_per_limb_solve": FP64_INSTR_PER_LIMB_SOLVE[n_lens],
                        "limb_solves_per_point": stats["n_limb_solves"] / steps / n,
                        "kernel_ms_avg": reg_ms / max(reg_n, 1), "share_of_step": (reg_ms + sec_ms) / ms,
                        "share_note": "k_limb + k_sectors (the whole region builder, steps a3 + a4)"}
    out = {"wl": wl, "n": n, "value": value, "ms_per_step": ms_per_step, "e2e": e2e, "roofline": roofline,
           "roofline_regions": roofline_regions, "rays_per_s": env.world * rays_per_step / (ms_per_step * 1e-3),
           "rays_per_point": rays_per_step / n, "kernel_ms_per_step": {k: v[0] / steps for k, v in kms.items()},
           "flagged_points": int(((status & 0xff) != 0).sum()), "nan_points": int(np.isnan(A_host).sum()),
           "gpu_launches": launches_per_step * steps, "clocks": clk, "n_ext": int(box["n_ext"]), "steps": steps, "warmup": warmup}
    return out


def summary(r: dict) -> dict:
    """One config's short entry under all_configs."""
    return {"workload": workload_name(r["wl"]), "value": r["value"], "unit": UNIT, "ms_per_step": r["ms_per_step"],
            "steps": r["steps"], "warmup": r["warmup"], "rays_per_s": r["rays_per_s"], "rays_per_point": r["rays_per_point"],
            "roofline_kernel": r["roofline"]["kernel"], "roofline_frac": r["roofline"]["frac"],
            "roofline_share_of_step": r["roofline"]["share_of_step"],
            "regions_frac": r["roofline_regions"]["frac"], "regions_share_of_step": r["roofline_regions"]["share_of_step"],
            "flagged_points": r["flagged_points"], "nan_points": r["nan_points"]}


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
    ctx = binding.Context(local_rank)
    env = Env(torch, dist, binding, inputs, replicas, ctx, dev, local_rank, world)

    r = measure_config(env, args.config, args.steps, args.warmup, switch=args.switch, with_e2e=True, with_clocks=True, f32=args.f32)
    others = {}
    if args.all_configs and world == 1:
        # the other BASELINE configs through the same code path, short runs (W = 3 warm-up, 2 timed steps)
        for c in range(5):
            if c != args.config:
                others["C%d" % c] = summary(measure_config(env, c, 2, 3, with_e2e=False))
        for c in (1, 2, 3):
            r32 = measure_config(env, c, 2, 3, with_e2e=False, f32=True)
            others["C%d_f32" % c] = dict(summary(r32), api="ULENS_OPT_F32_SHOOT: rays on the FP32 pipe (SURVEY 8.f-1); roofline_frac is "
                                         "against the FP32 FMA peak (%.1f TFLOP/s)" % (2.0 * FP32_PEAK_FFMA / 1e12))
        if args.config == 4 and not args.switch:
            rs = measure_config(env, 4, 2, 3, switch=True, with_e2e=False)
            others["C4_switch"] = dict(summary(rs), n_ext=rs["n_ext"], n_epochs_total=rs["n"],
                                       api="ulens_lightcurve_binary_ext, library selection (sel_tol default 2e-5): the other "
                                           "epochs take the point-source value (P:153, SURVEY 8.f-2)")

    if rank == 0:
        wl = r["wl"]
        peak_measured = ctx.ulens_fp64_peak(200.0)
        if "C1_f32" in others:
            line_f32 = {"workload": others["C1_f32"]["workload"], "kernel": "k_shoot_f32", "bound": "alu", "unit": "TFLOP/s",
                        "peak": 2.0 * FP32_PEAK_FFMA / 1e12, "frac": others["C1_f32"]["roofline_frac"],
                        "achieved": others["C1_f32"]["roofline_frac"] * 2.0 * FP32_PEAK_FFMA / 1e12,
                        "peak_measured_ffma_microbench": 2.0 * ctx.ulens_fp32_peak(200.0) / 1e12,
                        "value": others["C1_f32"]["value"], "value_fp64_path": others.get("C1", {}).get("value")}
        else:
            line_f32 = None
        for k in ("roofline", "roofline_regions"):
            r[k]["peak_measured_dfma_microbench"] = 2.0 * peak_measured / 1e12
            r[k]["frac_of_measured"] = r[k]["achieved"] / (2.0 * peak_measured / 1e12)
        dual = args.config == 4
        line = {"metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": workload_name(wl), "rho": [float(wl.rho.min()), float(wl.rho.max())],
                           "u1": [float(wl.u1.min()), float(wl.u1.max())],
                           "outputs": "A and dA/d(t0,u0,tE,s,q,rho,alpha) per epoch (forward-mode variant, step a8)" if dual else "A per point",
                           "switch": bool(args.switch), "f32_shoot": bool(args.f32),
                           "l2": "flushed between timed steps (256 MiB fill)",
                           "parallelism": "replicas" if world > 1 else "1 GPU"},
                "rays_per_s": r["rays_per_s"], "rays_per_point": r["rays_per_point"],
                "kernel_ms_per_step": r["kernel_ms_per_step"],
                "flagged_points": r["flagged_points"], "nan_points": r["nan_points"],
                "roofline": r["roofline"], "roofline_regions": r["roofline_regions"],
                "e2e": r["e2e"], "gpu_launches": r["gpu_launches"], "clocks": r["clocks"]}
        if dual and args.switch:
            line["config"]["switch_detail"] = {"api": "ulens_lightcurve_binary_ext", "selection": "library (sel_tol default 2e-5)",
                                               "n_ext": r["n_ext"], "n_epochs_total": r["n"]}
        if line_f32:
            line["roofline_f32"] = line_f32
        if others:
            line["all_configs"] = others
        if not args.no_cpu_baseline and world == 1:
            npts, dt, nev, cores = run_oracle_sample(wl, inputs)
            line["cpu_baseline"] = {"value": npts / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": "%d seeded points (%d configs x %d, half near-caustic, seed %d), oracle n_rho=%d ss=%d, %.1f s; "
                                              "values only (no derivatives)"
                                              % (npts, min(CPU_SAMPLE_CFGS, wl.n_cfg), sample_per_cfg(wl), CPU_SAMPLE_SEED, ORACLE_N_RHO, ORACLE_SS, dt),
                                    "rays_per_s": nev / dt}
        print(json.dumps(line), flush=True)
    ctx.close()
    if env.ctx32 is not None:
        env.ctx32.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main_stub(args, rank, world):
    """TEST HOOK (tests/test_replicas_gloo.py): the N > 1 plumbing of main_ours -- rendezvous from the launcher's
    environment, barrier, per-rank timing, max over ranks, whole-job aggregate, one line on rank 0 -- on CPU ranks
    over gloo, with the CUDA step replaced by a sleep. The line is marked "stub" and carries no metric."""
    import torch.distributed as dist
    from paper_2510_02639_b200 import replicas
    if world > 1:
        dist.init_process_group("gloo")
    units = 1000
    if world > 1:
        dist.barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        time.sleep(0.02 * (rank + 1))                           # rank r is (r + 1) x slower: the max must win
    ms_own = 1e3 * (time.perf_counter() - t0)
    (ms,) = replicas.max_over_ranks([ms_own])
    value = replicas.aggregate_throughput(units, world, ms / args.steps)
    if rank == 0:
        print(json.dumps({"stub": True, "metric": "stub", "n_gpus": world, "steps": args.steps, "ms_per_step": ms / args.steps,
                          "ms_per_step_rank0": ms_own / args.steps, "value": value, "scaling": "weak"}), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def relaunch_under_torchrun(n: int) -> int:
    """`python bench.py --gpus N` outside a launcher: start N ranks on this node and return their exit code."""
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(n),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config index 0..4 (default 4: the largest single-GPU "
                    "configuration, light curves with forward-mode derivatives)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-all-configs", dest="all_configs", action="store_false",
                    help="skip the short runs of the other BASELINE configs (the all_configs key)")
    ap.add_argument("--switch", action="store_true",
                    help="config 4 only: ulens_lightcurve_binary_ext (point-source value for the far epochs, P:153; "
                         "library selection at the default tolerance) instead of the finite-source path on every epoch")
    ap.add_argument("--f32", action="store_true",
                    help="configs 0-3 only: the mixed-precision variant (ULENS_OPT_F32_SHOOT, SURVEY 8.f-1) as the measured path; "
                         "roofline is then k_shoot_f32 against the FP32 FMA peak")
    ap.add_argument("--stub", action="store_true", help=argparse.SUPPRESS)
    args = ap.parse_args()
    if args.switch and args.config != 4:
        ap.error("--switch needs --config 4")
    if args.f32 and args.config == 4:
        ap.error("--f32: the forward-mode variant (config 4) always runs in FP64")
    if args.gpus < 1:
        ap.error("--gpus must be >= 1")
    if "WORLD_SIZE" not in os.environ and args.gpus > 1 and args.impl != "reference":
        raise SystemExit(relaunch_under_torchrun(args.gpus))    # (the oracle arm runs on rank 0's host cores only)
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl != "reference" and world != args.gpus:
        raise SystemExit("bench.py: --gpus %d but the launcher started WORLD_SIZE=%d ranks" % (args.gpus, world))
    if args.impl == "reference":
        main_reference(args, rank, world)
    elif args.stub:
        main_stub(args, rank, world)
    else:
        main_ours(args, rank, local_rank, world)


if __name__ == "__main__":
    main()

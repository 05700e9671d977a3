#!/usr/bin/env python
"""bench.py -- throughput of the RK3 step of libfizzy.so on B200 (BASELINE.json `metric`:
fp64 Mcell-substeps/s per RK3 step on 1 B200; achieved HBM GB/s vs peak).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 3] [--impl fizzy|reference]

A "step" is one full RK3 step = three fizzy_rk3_substep calls (all rows of SURVEY.md 8(a)).
Workload at N=1: BASELINE.json configs[3], droplet-laden HIT at 512^3 (the size the north-star
target is quoted on), synthetic seeded inputs from paper_2502_04189_b200.workloads.
N>1: replicas only: every rank runs the same workload on its own GPU,
no data-path collective; value = cells*substeps of all ranks / max-over-ranks time.

One JSON line on stdout (rank 0).  `--impl reference` times the CPU oracle, as it stands, on the SAME workload
(config 4 at 512^3: about 20 s per RK3 step on 16 cores); `cpu_baseline` of the default arm is one such step.  A smaller
sample only with an explicit --cpu-grid N (or when the host has too little memory), and then config.workload says so.

Timed regions: (1) `value`: K steps, inputs resident in HBM, per-kernel timing OFF, CUDA events on the
library's stream; (2) a second, shorter pass with fizzy_timing_enable for the per-kernel table and the
`roofline` object; (3) `e2e`: host buffers through the C ABI; (4) `cufft_compare`: cuFFT (torch.fft)
on the transforms of S4 only, bench-only yardstick -- cuFFT is never used by libfizzy.so.
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
sys.path.insert(0, ROOT)

from paper_2502_04189_b200 import workloads as W  # noqa: E402

TRAFFIC_CSV, TRAFFIC_MD = "r3_traffic.csv", "r3_ncu_full.md"
METRIC = "fp64 Mcell-substeps/s per RK3 step"
UNIT = "Mcell-substeps/s"

# Algorithmic HBM bytes per cell per launch:
# every N-array a pass must read or write, once; halos and 1-D tables free.
def algorithmic_bytes_per_cell(cfg):
    nx = cfg["nx"]
    spec = 16.0 * (nx // 2 + 1) / nx          # one complex half-spectrum pass, per real cell
    varrho = cfg["rho1"] != cfg["rho2"]
    heat = bool(cfg["heat"])
    b = {
        "k_phi_update": 72.0,                                   # r phi,u,v,w,hphi,divRn  w phi,hphi,psi
        # S5 of the previous substep fused in front of S1 (stages 1, 2): r u** x3, p_new, phi, hphi, divRn  w u,v,w, phi, hphi, psi
        # (+ r p_old, w p_hat if rho1 != rho2)
        "k_corr_phi": 104.0 + (16.0 if varrho else 0.0),
        "k_iface_march": 32.0 + (24.0 if varrho else 0.0),      # r psi,phi  w kappa,divRn (+Rn x3)
        # r u,v,w,phi,kappa,h x3  w u** x3, h x3 (+ r Rn x3, p_hat if rho1 != rho2; + r T with heat)
        "k_momentum": 112.0 + (32.0 if varrho else 0.0) + (8.0 if heat else 0.0),
        "k_fftx_fwd": 24.0 + spec,
        # fused FFT_y + z-elimination: forward r spec, w spec (pivots recomputed on chip); backward r spec, INV
        # (half a complex), w spec, and E if z is periodic
        "k_spec_fwd": 2.0 * spec, "k_spec_bwd": (3.0 if not cfg["z_wall"] else 2.5) * spec,
        "k_fftx_inv": spec + 8.0,
        "k_correct": 56.0 + (16.0 if varrho else 0.0),          # r u** x3, p_new  w u,v,w (+ r p, w p_hat if rho1 != rho2)
    }
    if heat:
        b["k_temp_update"] = 64.0
    return b


def moved_bytes_per_cell(cfg):
    """Bytes a launch really moves, per stage (0, 1, 2), where they differ from the undiscounted model above: stage 0
    reads no RK history (zeta = 0) and stage 2 writes none (the next stage 0 does not read it).  None = no launch."""
    a = algorithmic_bytes_per_cell(cfg)
    m = a["k_momentum"]
    c = a["k_corr_phi"]
    return {"k_momentum": [m - 24.0, m, m - 24.0],          # h x3 not read / not written
            "k_phi_update": [a["k_phi_update"] - 8.0, None, None],   # stage 0 only: h_phi not read
            "k_corr_phi": [None, c, c - 8.0],                # stage 2 writes no h_phi
            "k_correct": [None, None, a["k_correct"]]}


def substep_model_bytes(cfg):
    """328 B per cell per substep with heat off, 400 B with heat on."""
    return 400.0 if cfg["heat"] else 328.0


def max_over_ranks(ms, dist, device):
    """Replicas only: the one collective of the bench is the MAX of the elapsed time."""
    if dist is None:
        return float(ms)
    import torch
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world, cells, substeps, ms):
    """Mcell-substeps/s of all ranks together: every rank advances its own replica of `cells` cells."""
    return world * cells * substeps / (ms * 1e-3) / 1e6


def measured_peak_gbs():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def cpu_model():
    try:
        with open("/proc/cpuinfo") as fh:
            for ln in fh:
                if ln.lower().startswith("model name"):
                    return ln.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""

    QUERY = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index = index
        self.stop = threading.Event()
        self.samples = []

    def run(self):
        while not self.stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.QUERY,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                parts = [p.strip() for p in out.strip().split(",")]
                if len(parts) >= 6:
                    self.samples.append(parts)
            except Exception:
                pass
            self.stop.wait(0.02)   # nvidia-smi itself takes ~40 ms: about 15 samples per second

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        sm = sorted(float(s[0]) for s in self.samples)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for q, n in enumerate(names) if any(s[2 + q].lower().startswith("active") for s in self.samples)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.samples[0][1]), "reasons": reasons,
                "samples": len(sm)}


ORACLE_GB_PER_MCELL = 0.45   # host memory of the oracle: ~40 ghost-padded arrays + FFT work + inputs/outputs, per 1e6 cells


def oracle_sample_fits(cells):
    import psutil
    return psutil.virtual_memory().available / 1e9 >= ORACLE_GB_PER_MCELL * cells / 1e6


def oracle_sample(args):
    """(cfg, fields, dt, workload label, same_config) of the oracle runs: the bench's own workload unless --cpu-grid N asks
    for the same recipe at N^3 or the host cannot hold the oracle's arrays (then 256^3, and the label says so)."""
    grid = tuple(args.grid) if args.grid else W.DEFAULT_GRIDS[args.workload]
    cells = grid[0] * grid[1] * grid[2]
    n = args.cpu_grid
    if n == 0 and not oracle_sample_fits(cells):
        n = 256
    if n == 0:
        cfg, f, dt, _ = W.make(args.workload, grid=tuple(args.grid) if args.grid else None)
        return cfg, f, dt, cfg["name"], True
    cfg, f, dt, _ = W.make(args.workload, grid=(n, n, n), ndrops=max(1, 200 // max(1, 512 // n) ** 3))
    return cfg, f, dt, "%s recipe at %d^3 (NOT the bench grid)" % (W.NAMES[args.workload], n), False


def run_reference(args, rank):
    """The CPU oracle as it stands, on the host cores, on the bench's own workload; a step is one RK3 step.  At 512^3 a
    step takes about 20 s, so the warm-up is capped at one step (a CPU program has nothing to warm beyond its first touch of
    memory) and the timed steps by --ref-budget-s; the line reports the warm-up and the steps that ran."""
    if rank != 0:
        return
    import oracle
    oracle.build()
    cfg, f, dt, label, same = oracle_sample(args)
    o = oracle.Oracle(cfg)
    o.set_fields(**f)
    warm = min(args.warmup, 1)
    for _ in range(warm):
        o.step(dt)
    # the run is bounded in time: whole steps are timed until K are done or --ref-budget-s is used up (at 512^3 a step takes
    # 19-26 s, so the default 240 s time about a dozen of the driver's 20); the line reports the steps that ran
    t0 = time.perf_counter()
    done = 0
    while done < args.steps:
        o.step(dt)
        done += 1
        if time.perf_counter() - t0 > args.ref_budget_s:
            break
    el = time.perf_counter() - t0
    cells = cfg["nx"] * cfg["ny"] * cfg["nz"]
    value = cells * 3 * done / el / 1e6
    sample = "%s, %d x %d x %d cells, %d RK3 steps in %.1f s (%d asked for, time budget %g s)" % (
        label, cfg["nx"], cfg["ny"], cfg["nz"], done, el, args.steps, args.ref_budget_s)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": done, "steps_requested": args.steps, "warmup": warm, "ms_per_step": 1e3 * el / done,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": label, "grid": [cfg["nx"], cfg["ny"], cfg["nz"]], "same_config_as_default_arm": same,
                       "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                             "cpu_model": cpu_model(), "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def cpu_baseline(args, sample=None):
    """Oracle timed on ONE RK3 step of the bench's own workload (see oracle_sample)."""
    import oracle
    oracle.build()
    cfg, f, dt, label, same = sample if sample is not None else oracle_sample(args)
    o = oracle.Oracle(cfg)
    o.set_fields(**f)
    t0 = time.perf_counter()
    o.step(dt)
    el = time.perf_counter() - t0
    o.close()
    cells = cfg["nx"] * cfg["ny"] * cfg["nz"]
    return {"value": cells * 3 / el / 1e6, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "cpu_model": cpu_model(), "same_config": same,
            "sample": "%s, %d x %d x %d cells, 1 RK3 step, %.1f s" % (label, cfg["nx"], cfg["ny"], cfg["nz"], el)}


def other_config(torch, Fizzy, index, device, peak, steps=5, warmup=3):
    """Device-resident throughput of another BASELINE.json config at its own size (the variable-density / wall / heat
    variants of the kernels, which the headline workload does not exercise): same timing rules as `value`."""
    t0 = time.perf_counter()
    cfg, f, dt, _ = W.make(index)
    gen_s = time.perf_counter() - t0
    cells = cfg["nx"] * cfg["ny"] * cfg["nz"]
    fz = Fizzy(cfg, device=device)
    names = ["u", "v", "w", "p", "phi"] + (["T"] if cfg["heat"] else [])
    for k in names:      # one field at a time: at 1024x512x512 the workspace leaves little room for staging copies
        t = torch.from_numpy(f[k]).to(device)
        fz.fizzy_set_fields(**{k: t})
        torch.cuda.synchronize()
        del t
    del f
    for _ in range(warmup):
        fz.step(dt)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(fz.stream)
    for _ in range(steps):
        fz.step(dt)
    e1.record(fz.stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    finite = fz.fizzy_check_finite() == 0
    fz.fizzy_timing_enable(True)
    fz.fizzy_timing_get(reset=True)
    fz.step(dt)
    per_kernel = fz.fizzy_timing_get(reset=True)
    fz.close()
    bpc = algorithmic_bytes_per_cell(cfg)
    sub_ms = ms / (3 * steps)
    gbs = substep_model_bytes(cfg) * cells / (sub_ms * 1e-3) / 1e9
    kern = {}
    for name, (tot, n) in per_kernel.items():
        if name in bpc and n:
            g = bpc[name] * cells / (tot / n * 1e-3) / 1e9
            kern[name] = {"ms_per_launch": round(tot / n, 4), "algorithmic_B_per_cell": round(bpc[name], 2), "frac": round(g / peak, 4)}
    return {"workload": cfg["name"], "grid": [cfg["nx"], cfg["ny"], cfg["nz"]], "steps": steps, "warmup": warmup,
            "value": cells * 3 * steps / (ms * 1e-3) / 1e6, "unit": UNIT, "ms_per_substep": round(sub_ms, 4),
            "model_B_per_cell": substep_model_bytes(cfg), "achieved_GBs": round(gbs, 1), "frac": round(gbs / peak, 4),
            "finite": finite, "generation_s": round(gen_s, 1), "kernels": kern}


def cufft_compare(torch, cfg, per_kernel, device):
    """Bench-only yardstick (BASELINE.json:5 "cuFFT appears only as a bench comparison"): the four transforms of S4
    -- r2c along x, c2c along y, and their inverses -- by cuFFT through torch.fft on an array of the same shape,
    plans created in a warm-up call.  The library's own S4 kernels additionally assemble the Poisson right-hand
    side, solve the tridiagonal systems in z, scale and remove the gauge mean."""
    try:
        nz, ny, nx = cfg["nz"], cfg["ny"], cfg["nx"]
        x = torch.randn(nz, ny, nx, dtype=torch.float64, device=device)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(5)]

        def run():
            ev[0].record()
            a = torch.fft.rfft(x, dim=2)
            ev[1].record()
            b = torch.fft.fft(a, dim=1)
            ev[2].record()
            c = torch.fft.ifft(b, dim=1)
            ev[3].record()
            d = torch.fft.irfft(c, n=nx, dim=2)
            ev[4].record()
            return d

        run()
        torch.cuda.synchronize()
        best = [1e30] * 4
        for _ in range(3):
            run()
            torch.cuda.synchronize()
            best = [min(best[q], ev[q].elapsed_time(ev[q + 1])) for q in range(4)]
        del x
        torch.cuda.empty_cache()
        ours = {k: per_kernel[k][0] / per_kernel[k][1] for k in ("k_fftx_fwd", "k_spec_fwd", "k_spec_bwd", "k_fftx_inv")
                if k in per_kernel and per_kernel[k][1]}
        return {"cufft_ms": {"rfft_x": round(best[0], 4), "fft_y": round(best[1], 4), "ifft_y": round(best[2], 4),
                             "irfft_x": round(best[3], 4), "sum": round(sum(best), 4)},
                "fizzy_s4_ms": {**{k: round(v, 4) for k, v in ours.items()}, "sum": round(sum(ours.values()), 4)},
                "note": "cuFFT: transforms only, out of place, each a separate pass over HBM; fizzy S4: Poisson rhs + "
                        "FFT x + (FFT y fused with the z tridiagonal sweeps) + inverse, scale, gauge"}
    except Exception as exc:  # bench-only: never fail the line because of the yardstick
        return {"error": repr(exc)}


def graph_compare(torch, Fizzy, device):
    """ms per RK3 step on the two launch-bound configurations (configs[0] 32^3, configs[1] 128^3)
    with the three substeps as plain launches and replayed as one CUDA graph (fizzy_graph_enable)."""
    out = {}
    try:
        for idx, steps in ((0, 200), (1, 50)):
            cfg, f, dt, _ = W.make(idx)
            row = {}
            for mode in ("plain", "graph"):
                st = torch.cuda.Stream(device)
                g = Fizzy(cfg, stream=st, device=device)
                g.fizzy_graph_enable(mode == "graph")
                g.set_fields_numpy(**f)
                for _ in range(10):
                    g.fizzy_rk3_step(dt)
                st.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(st)
                for _ in range(steps):
                    g.fizzy_rk3_step(dt)
                e1.record(st)
                st.synchronize()
                row[mode + "_ms_per_step"] = round(e0.elapsed_time(e1) / steps, 4)
                g.close()
            out[cfg["name"]] = row
    except Exception as exc:
        out["error"] = repr(exc)
    return out


def varcoef_bench(args):
    """SURVEY.md 8(f)-4 (not part of the RK3 step): fizzy_poisson_solve_varcoef on the phase field of the chosen workload,
    random right-hand side, to a relative residual of 1e-10; one JSON line of its own."""
    import torch
    from paper_2502_04189_b200.binding import Fizzy
    torch.cuda.set_device(0)
    cfg, f, dt, _ = W.make(args.workload, grid=tuple(args.grid) if args.grid else None)
    cells = cfg["nx"] * cfg["ny"] * cfg["nz"]
    fz = Fizzy(cfg, device="cuda:0")
    fz.fizzy_set_fields(**{k: torch.from_numpy(f[k]).cuda() for k in ["u", "v", "w", "p", "phi"] + (["T"] if cfg["heat"] else [])})
    rhs = torch.randn(cfg["nz"], cfg["ny"], cfg["nx"], dtype=torch.float64, device="cuda:0")
    p = torch.empty_like(rhs)
    it, rr = fz.fizzy_poisson_solve_varcoef(rhs, p, rtol=1e-10, max_iter=200)      # warm-up (allocates the scratch)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0 = fz.fizzy_launch_count()
    e0.record(fz.stream)
    it, rr = fz.fizzy_poisson_solve_varcoef(rhs, p, rtol=1e-10, max_iter=200)
    e1.record(fz.stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    e0.record(fz.stream)
    fz.fizzy_poisson_solve(rhs, p)
    e1.record(fz.stream)
    torch.cuda.synchronize()
    print(json.dumps({"metric": "variable-coefficient Poisson solve (multigrid-preconditioned CG, rtol 1e-10)", "workload": cfg["name"],
                      "grid": [cfg["nx"], cfg["ny"], cfg["nz"]], "rho_ratio": max(cfg["rho1"], cfg["rho2"]) / min(cfg["rho1"], cfg["rho2"]),
                      "iterations": it, "relres": rr, "ms": ms, "ms_per_iteration": ms / max(it, 1),
                      "Mcell_per_s": cells / (ms * 1e-3) / 1e6, "gpu_launches": fz.fizzy_launch_count() - n0,
                      "constant_coefficient_fft_solve_ms": e0.elapsed_time(e1)}), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", type=int, default=3, help="BASELINE.json config index (0-based)")
    ap.add_argument("--grid", type=int, nargs=3, default=None, help="override nx ny nz (debug)")
    ap.add_argument("--impl", default="fizzy", choices=["fizzy", "reference"])
    ap.add_argument("--cpu-grid", type=int, default=0,
                    help="0 (default): the oracle runs the bench's own workload; N: the same recipe at N^3 instead (labelled)")
    ap.add_argument("--ref-budget-s", type=float, default=240.0,
                    help="--impl reference: stop timing whole steps once this many seconds are used (the CPU oracle needs ~20 s per 512^3 step)")
    ap.add_argument("--other-configs", type=int, nargs="*", default=[2, 4],
                    help="BASELINE.json config indices timed at their own size after the headline workload (N = 1 only)")
    ap.add_argument("--no-cufft", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--pressure-solver", type=int, default=0, choices=[0, 1],
                    help="1: the RK3 step with the variable-coefficient multigrid pressure path (SURVEY 8(f)-4; rtol 1e-10) instead of the splitting")
    ap.add_argument("--varcoef", action="store_true", help="time fizzy_poisson_solve_varcoef (SURVEY 8(f)-4) instead of the RK3 step")
    args = ap.parse_args()
    if args.varcoef:
        varcoef_bench(args)
        return
    args.warmup = max(args.warmup, 3) if args.impl == "fizzy" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # `python bench.py --gpus N` without torchrun: start the N replicas ourselves (one rank per GPU)
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
               "--master-addr", "127.0.0.1", "--master-port", os.environ.get("MASTER_PORT", "29511"),
               os.path.abspath(__file__)] + sys.argv[1:]
        os.execv(sys.executable, cmd)
    if args.gpus != world:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%d" % (args.gpus, world))

    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    from paper_2502_04189_b200.binding import Fizzy  # raises if libfizzy.so is missing

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (libfizzy has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    cfg, f, dt, _ = W.make(args.workload, grid=tuple(args.grid) if args.grid else None)
    cells = cfg["nx"] * cfg["ny"] * cfg["nz"]
    fz = Fizzy(cfg, device="cuda:%d" % local_rank)
    if args.pressure_solver:
        fz.fizzy_set_pressure_solver(1, rtol=1e-10, max_iter=200)
    names = ["u", "v", "w", "p", "phi"] + (["T"] if cfg["heat"] else [])
    dev = {k: torch.from_numpy(f[k]).to("cuda:%d" % local_rank) for k in names}
    fz.fizzy_set_fields(**dev)
    torch.cuda.synchronize()

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    # ---------------- device-resident throughput (value): per-kernel timing OFF ----------------
    for _ in range(args.warmup):
        fz.step(dt)
    fz.fizzy_timing_enable(False)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    n0 = fz.fizzy_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(fz.stream)
    for _ in range(args.steps):
        fz.step(dt)
    e1.record(fz.stream)
    barrier()
    sampler.stop.set()
    sampler.join()
    ms = e0.elapsed_time(e1)
    launches = fz.fizzy_launch_count() - n0
    finite = fz.fizzy_check_finite() == 0
    ms = max_over_ranks(ms, dist, "cuda")
    value = whole_job_value(world, cells, 3 * args.steps, ms)

    # ---------------- second pass, per-kernel events ON: the kernel table (not part of `value`) ----------------
    ksteps = max(1, min(args.steps, 5))
    fz.fizzy_timing_enable(True)
    fz.fizzy_timing_get(reset=True)
    for _ in range(ksteps):
        fz.step(dt)
    per_kernel = fz.fizzy_timing_get(reset=True)
    fz.fizzy_timing_enable(False)

    # ---------------- roofline of the dominant kernel + per-kernel table ----------------
    peak, peak_src = measured_peak_gbs()
    bpc = algorithmic_bytes_per_cell(cfg)
    moved = moved_bytes_per_cell(cfg)
    table = []
    for name, (tot_ms, n) in per_kernel.items():
        if name in bpc and n:
            avg = tot_ms / n
            gbs = bpc[name] * cells / (avg * 1e-3) / 1e9
            row = {"kernel": name, "ms_per_launch": round(avg, 4), "launches": n,
                   "share": tot_ms, "algorithmic_B_per_cell": round(bpc[name], 2),
                   "achieved_GBs": round(gbs, 1), "frac": round(gbs / peak, 4)}
            if name in moved:   # mean over the stages that launch it: what really crosses HBM
                per_stage = [b for b in moved[name] if b is not None]
                mv = sum(per_stage) / len(per_stage)
                row["bytes_moved_B_per_cell"] = round(mv, 2)
                row["bytes_moved_per_stage"] = moved[name]
                row["frac_moved"] = round(mv * cells / (avg * 1e-3) / 1e9 / peak, 4)
            table.append(row)
    tot = sum(r["share"] for r in table) or 1.0
    for r in table:
        r["share"] = round(r["share"] / tot, 4)
    table.sort(key=lambda r: -r["share"])
    top = table[0] if table else None
    sub_ms = ms / (3 * args.steps)
    sub_gbs = substep_model_bytes(cfg) * cells / (sub_ms * 1e-3) / 1e9
    roofline = None
    if top:
        roofline = {"bound": "hbm", "kernel": top["kernel"], "achieved": top["achieved_GBs"], "peak": peak,
                    "unit": "GB/s", "frac": top["frac"], "traffic": None, "peak_source": peak_src,
                    "algorithmic_B_per_cell": top["algorithmic_B_per_cell"],
                    "bytes_moved_B_per_cell": top.get("bytes_moved_B_per_cell", top["algorithmic_B_per_cell"]),
                    "frac_moved": top.get("frac_moved", top["frac"])}
    # ncu DRAM traffic per launch of the dominant kernel: NOT measured in this run (a number printed under a
    # profiler is never a bench value); it is the committed ncu capture named in `traffic_source`
    try:
        with open(os.path.join(ROOT, "profiles", TRAFFIC_CSV)) as fh:
            per_stage = {}
            for ln in fh:
                parts = ln.strip().split(",")
                if roofline and len(parts) == 4 and parts[0] == cfg["name"] and parts[1] == roofline["kernel"]:
                    per_stage[int(parts[2])] = float(parts[3])
            if per_stage:   # the same average the `frac` is taken over: one launch per stage
                roofline["traffic"] = sum(per_stage.values()) / len(per_stage)
                roofline["traffic_per_stage"] = [per_stage.get(q) for q in range(3)]
                roofline["traffic_source"] = ("mean of the stage-0/1/2 launches of one RK3 step, ncu --set full capture, "
                                              "profiles/%s (see profiles/%s)" % (TRAFFIC_CSV, TRAFFIC_MD))
    except Exception:
        pass

    # ---------------- end to end through the C ABI with HOST buffers ----------------
    e2e = None
    if not args.no_e2e:
        hin = {k: torch.from_numpy(f[k]).pin_memory() for k in names}
        hout = {k: torch.empty_like(hin[k]).pin_memory() for k in names}
        nb = cells * 8
        ke = max(1, min(args.steps, 3))
        fz.fizzy_set_fields(**hin)
        fz.step(dt)
        fz.fizzy_get_fields(**hout)
        barrier()
        e0.record(fz.stream)
        for _ in range(ke):
            fz.fizzy_set_fields(**hin)      # H2D of the step's inputs (pinned host memory)
            fz.step(dt)
            fz.fizzy_get_fields(**hout)     # D2H of the step's result
        e1.record(fz.stream)
        barrier()
        ems = e0.elapsed_time(e1)
        ems = max_over_ranks(ems, dist, "cuda")
        e2e = {"value": whole_job_value(world, cells, 3 * ke, ems), "unit": UNIT,
               "h2d_bytes_per_step": nb * len(names), "d2h_bytes_per_step": nb * len(names), "steps": ke,
               "note": "fizzy_set_fields(host) + 3 x fizzy_rk3_substep + fizzy_get_fields(host) per step"}

    cufft = None
    if rank == 0 and not args.no_cufft:
        cufft = cufft_compare(torch, cfg, per_kernel, "cuda:%d" % local_rank)
    graphs = graph_compare(torch, Fizzy, "cuda:%d" % local_rank) if (rank == 0 and world == 1 and not args.no_cufft) else None
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    cpu, others = None, None
    fz.close()
    del dev
    if not args.no_e2e:
        del hin, hout
    torch.cuda.empty_cache()
    if world == 1 and not args.no_cpu_baseline:
        same = args.cpu_grid == 0
        cpu = cpu_baseline(args, (cfg, f, dt, cfg["name"], True) if same and oracle_sample_fits(cells) else None)
    del f
    if world == 1 and args.other_configs and not args.grid and not args.pressure_solver:
        others = []
        for index in args.other_configs:
            if index == args.workload:
                continue
            try:
                others.append(other_config(torch, Fizzy, index, "cuda:%d" % local_rank, peak))
            except Exception as exc:   # e.g. not enough device or host memory for config 5 on this box: say so, keep the line
                others.append({"workload": W.NAMES[index], "unavailable": "%s: %s" % (type(exc).__name__, str(exc)[:200])})
            torch.cuda.empty_cache()
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg["name"], "grid": [cfg["nx"], cfg["ny"], cfg["nz"]], "dt": dt,
                       "cache": "inputs larger than L2 (each field %.0f MB, 126 MB L2)" % (cells * 8 / 1e6),
                       "parallelism": "replicas x%d" % world, "finite": finite,
                       "pressure_solver": "variable-coefficient multigrid CG, rtol 1e-10" if args.pressure_solver else "splitting + FFT/tridiagonal",
                       "byte_model": "SURVEY.md 8(d): %.0f B/cell/substep, every substep counted in full (stage 0 reads no RK "
                                     "history and stage 2 writes none: those discounts are NOT taken)" % substep_model_bytes(cfg),
                       "timing": "value: CUDA events on the library stream, per-kernel timing off; kernel table: second pass of "
                                 "%d steps with events around every launch" % ksteps},
            "clocks": sampler.summary(), "e2e": e2e, "gpu_launches": launches,
            "roofline": roofline,
            "roofline_substep": {"bound": "hbm", "model_B_per_cell": substep_model_bytes(cfg),
                                 "ms_per_substep": sub_ms, "achieved": round(sub_gbs, 1), "peak": peak,
                                 "unit": "GB/s", "frac": round(sub_gbs / peak, 4)},
            "kernels": table, "other_configs": others, "cufft_compare": cufft, "graph_compare": graphs, "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

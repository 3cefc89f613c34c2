#!/usr/bin/env python
"""bench.py -- GLUPS of the two-component colour-gradient D3Q19 hot path on B200.

One "step" is one LB time step of the whole box: the fused stream-collide kernel k_fused (which
also forwards the moments of the next state) plus the phase-field kernel k_phase_fwd, i.e. every
row A0-A10 of the hot path.  Prints ONE JSON line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c3|c5|c4|c2|c1] [--storage ab|aa]
                  [--model cg|sc] [--windows N]
  python bench.py --impl reference ...     # the fp64 CPU oracle on this box's host cores

N > 1 (torchrun): z-slab decomposition, weak scaling: every rank holds the workload's
box as one slab of a box N times as tall and exchanges, per step and face, 5 populations per component
and H planes of phi with its two neighbours (NCCL send/recv; paper_2005_12764_b200/slab.py);
value = N * sites * K / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "GLUPS (two-component D3Q19 site updates/s)"
BYTES_PER_UPDATE = {True: 2 * 2 * 19 * 4, False: 2 * 19 * 4}   # two-component 304 B, single 152 B
FALLBACK_HBM_GBS = 6650.0
NOMINAL_HBM_GBS = 8000.0     # north_star's "~8 TB/s"; every fraction is reported against the measured copy rate and against this
TUNE = {}                # --tune
MODEL = ["cg", 0.0]      # --model: colour gradient (north_star) or the paper's Shan-Chen coupling, and its G_C


# ------------------------------------------------------------------------------ helpers
def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def max_over_ranks(value, world, device=None):
    """MAX of a python float over all ranks (torch.distributed, any backend)."""
    if world == 1:
        return value
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def glups(sites_per_rank, steps, seconds, world):
    """Whole-job throughput: all ranks' site updates over the max-over-ranks time."""
    return world * sites_per_rank * steps / seconds / 1e9


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def stored_traffic(kernel, workload, storage):
    """dram bytes per launch of the dominant kernel from the committed ncu summary
    (profiles/traffic.csv: kernel,workload,storage,bytes,source), or None."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:
            for line in f:
                p = line.strip().split(",")
                if len(p) >= 4 and not line.startswith("#") and (p[0], p[1], p[2]) == (kernel, workload, storage):
                    return float(p[3])
    except Exception:
        pass
    return None


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc = index, None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
        return self

    def __exit__(self, *a):
        self.result = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if not self.proc:
            return
        time.sleep(0.25)
        self.proc.terminate()
        try:
            out = self.proc.communicate(timeout=5)[0]
        except Exception:
            return
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            p = [s.strip() for s in line.split(",")]
            if len(p) < 6:
                continue
            try:
                sm.append(float(p[0])); mx.append(float(p[1]))
            except ValueError:
                continue
            for n, v in zip(names, p[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if sm:
            self.result = {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons)}


def config_of(w, storage, extra=None):
    c = {"workload": w.name, "box": [w.nx, w.ny, w.nz], "sites": w.sites, "fluid_sites": w.fluid_sites,
         "components": 2 if w.rho_b is not None else 1, "near_contact": bool(w.A_nc != 0.0),
         "walls": w.solid is not None, "storage": storage, "model": "colour-gradient" if MODEL[0] == "cg" else "shan-chen G_C=%g" % MODEL[1],
         "params": dict(tau_r=w.tau_r, tau_b=w.tau_b, A=w.A, beta=w.beta, A_nc=w.A_nc, g=list(w.g)),
         "l2": "state (%.2f GB) is larger than L2, no flush needed" % (w.sites * 4 * (38 if w.rho_b is not None else 19) * (2 if storage == "ab" else 1) / 1e9)}
    if w.rho_b is not None and w.A_nc != 0.0 and w.A > 0.0:
        # N_c = A dx / sigma with sigma = (4/9) A tau of the colour-gradient perturbation (G5)
        c["N_c"] = w.A_nc / ((4.0 / 9.0) * w.A * w.tau_r)
    c.update({k: v for k, v in w.info.items() if k != "particles"})     # (the particle array stays out of the JSON line)
    if extra:
        c.update(extra)
    return c


# ------------------------------------------------------------------------------ oracle legs
def oracle_sample_workload(name, budget_updates):
    """The same recipe as the timed workload at the largest cubic size whose (steps x sites)
    fits the CPU budget."""
    from paper_2005_12764_b200 import workloads as W
    def make(n):
        if name == "c2":
            return W.c2_taylor_green(n)
        if name == "c4":
            return W.c4_channel(4 * n, n, n, R=10.0 if n >= 64 else 6.0)
        if name == "c5":
            return W.c5_emulsion(n, max(1, int(3000 * (n / 640.0) ** 3)))
        if name == "c1":
            return W.c1_droplet()
        if name.startswith("focuser"):
            return W.focuser(128, 48, 24, wd=10, wc=12, t=3, li=24, wo=10, lo=8, walls_z=True, A_nc=0.02)
        if name.startswith("bijel"):
            return W.bijel(n)
        return W.c3_spinodal(n)
    best = 32
    for n in (32, 48, 64, 96, 128, 160):
        sites = n ** 3 * (4 if name == "c4" else 1)
        if sites <= budget_updates:
            best = n
    return make(best)


def time_oracle(w, steps, warmup):
    from oracle import lbo
    o = lbo.Oracle(w.nx, w.ny, w.nz, *w.params)
    if MODEL[0] == "sc":
        o.set_model("sc", MODEL[1])
    if w.solid is not None:
        o.set_geometry(w.solid)
    o.set_body_force(*w.g)
    o.set_nc_cutoff(w.phi_c)
    from paper_2005_12764_b200 import workloads as W
    W.configure_walls(o, w)
    o.init(w.rho_r, w.rho_b, w.u)
    if warmup:
        o.step(warmup)
    t0 = time.perf_counter()
    o.step(steps)
    return time.perf_counter() - t0


def omp_threads():
    try:
        return int(os.environ.get("OMP_NUM_THREADS", "")) 
    except ValueError:
        return len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)


def cpu_baseline(name, seconds_budget=15.0):
    """The oracle as it stands on this box's host cores, on a bounded sample of the workload."""
    w = oracle_sample_workload(name, budget_updates=2.2e6)
    steps = 4
    dt = time_oracle(w, steps, 1)
    rate = w.fluid_sites * steps / dt
    more = int(max(0, min(60, (seconds_budget - dt) * rate / w.fluid_sites)))
    if more >= 4:
        dt = time_oracle(w, more, 1)
        steps = more
    return {"value": w.fluid_sites * steps / dt / 1e9, "unit": "GLUPS", "cores": omp_threads(), "kind": "oracle",
            "sample": "%s at %dx%dx%d (same recipe, smaller box), %d steps, fp64, OpenMP" % (w.name, w.nx, w.ny, w.nz, steps)}


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    total = max(1, args.steps + args.warmup)
    w = oracle_sample_workload(args.workload, budget_updates=4.0e6 * 120.0 / total)
    dt = time_oracle(w, args.steps, args.warmup)
    val = w.fluid_sites * args.steps / dt / 1e9
    sample = "%s at %dx%dx%d (same recipe, smaller box), %d steps, fp64, OpenMP" % (w.name, w.nx, w.ny, w.nz, args.steps)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "GLUPS", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_of(w, "oracle", {"note": "bounded sample of workload %s" % args.workload}),
            "cpu_baseline": {"value": val, "unit": "GLUPS", "cores": omp_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "GLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------ GPU arm
class SlabRunner:
    """N > 1 (or --slabs): this rank's box is one z slab of a box N times as tall (the workload
    repeated along z, which is periodic), advanced by paper_2005_12764_b200/slab.py: halo exchange of 5
    populations per component and H phi planes per face and step over NCCL send/recv, the population
    exchange on a side stream under the interior bricks.  Same interface as lb.LB where bench uses it."""

    def __init__(self, w, storage, rank, world):
        from paper_2005_12764_b200 import slab
        if w.info.get("particles") is not None and world > 1:
            # rigid particles are replicated data (every rank holds all of them): the taller box holds the
            # workload's particles once per period
            import dataclasses
            parts = np.asarray(w.info["particles"], dtype=np.float64)
            tiled = np.concatenate([parts + np.array([0, 0, k * w.nz] + [0] * (parts.shape[1] - 3)) for k in range(world)])
            w = dataclasses.replace(w, info=dict(w.info, particles=tiled))
        self.ds = slab.DistributedSlab(slab.Slab.from_workload(w, rank * w.nz, w.nz, storage, nz_global=world * w.nz), rank, world)
        self.sim = self.ds.slab.sim

    def init(self, rr, rb, u):
        self.ds.init(rr, rb, u)

    def step(self, n):
        self.ds.step(n)

    def check_state(self):
        return self.sim.check_state()

    def launch_count(self):
        return self.sim.launch_count()

    def get_macros(self, *a):
        return self.sim.get_macros(*a)

    def set_profiling(self, on):
        pass

    def last_step_ms(self, which):
        return None           # the slab phases are not timed kernel by kernel

    def destroy(self):
        self.sim.destroy()


def measure_config(wl_name, storage, K, Wu, dev, local_rank, world, w=None, with_e2e=False, windows=0, slabs=False):
    """One workload on this rank's GPU: W warm-up steps, then K timed steps (CUDA events on the
    handle's stream, barrier + synchronize on both sides, MAX over ranks).  Returns the record
    (value, ms_per_step, roofline, clocks, checks, optionally e2e) and the workload."""
    import torch
    import torch.distributed as dist
    from paper_2005_12764_b200 import lb, workloads as W
    if w is None:
        w = W.get(wl_name)
    two = w.rho_b is not None
    # inputs resident in HBM before the timed region
    d_rr = torch.from_numpy(w.rho_r).to(dev)
    d_rb = torch.from_numpy(w.rho_b).to(dev) if two else None
    d_u = torch.from_numpy(w.u).to(dev)
    rank = dist.get_rank() if world > 1 else 0
    if slabs:
        sim = SlabRunner(w, storage, rank, world)
    else:
        sim = lb.from_workload(w, storage=storage)
        if MODEL[0] == "sc":
            sim.set_model("sc", MODEL[1])
        if TUNE:
            sim.set_tuning(**TUNE)
    sim.init(d_rr, d_rb, d_u)
    mass0 = sim.check_state()
    # Every 7th step (odd, so that both AA parities are sampled) is timed kernel by kernel (CUDA events
    # on the stream).  A box of at most 2^21 sites is stepped by replaying a CUDA graph (include/lb.h,
    # lb_set_tuning "graph"), which event records inside the step would switch off: there the timed
    # region runs without them and the kernels are timed in a pass of the same length right after it.
    graphed = (not slabs) and w.sites <= (1 << 21) and TUNE.get("graph", -1) != 0
    sim.set_profiling(0 if graphed else 7)
    sim.step(Wu)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    # a run that saw a hardware or thermal slowdown is rejected and measured again, once
    BAD = {"hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"}
    remeasured = False
    for attempt in range(2):
        l0 = sim.launch_count()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with ClockSampler(local_rank) as clk:
            torch.cuda.synchronize()
            ev0.record()
            sim.step(K)
            ev1.record()
            torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        launches = sim.launch_count() - l0
        if world > 1 or not (BAD & set(clk.result.get("reasons", []))):
            break
        remeasured = True
        time.sleep(5.0)
    ms = ev0.elapsed_time(ev1)
    if graphed:
        sim.set_profiling(7)
        sim.step(K)
        torch.cuda.synchronize()
    ms_k2 = sim.last_step_ms(1)
    ms_k1 = sim.last_step_ms(2) if two else 0.0
    kernel_timing = "CUDA events around every 7th step of the timed region"
    if graphed:
        kernel_timing = "CUDA events around every 7th step of a pass of the same length right after the timed region (which replays a CUDA graph of 16 steps)"
    if ms_k2 is None:        # slabs: the fused kernel runs as three launches per step; the whole step stands in
        ms_k2, ms_k1 = ms / K, None
        kernel_timing = "slab phases are not timed kernel by kernel: kernel_ms is the whole step (boundary + interior bricks, phase field, packing, exchange)"
    ms_max = max_over_ranks(ms, world, dev)
    value = glups(w.fluid_sites, K, ms_max * 1e-3, world)

    # sanity: the state is finite and the component masses are where they were (summed on the
    # device by lb_check_state; raises on a NaN / Inf state)
    mass = sim.check_state()
    finite = True
    drift = [abs(a - b) / b if b > 0 else 0.0 for a, b in zip(mass, mass0)]

    peak, peak_src = measured_peak()
    upd_bytes = BYTES_PER_UPDATE[two]
    achieved = upd_bytes * w.fluid_sites / (ms_k2 * 1e-3) / 1e9      # mean k_fused / k_single launch over the sampled steps
    whole = upd_bytes * w.fluid_sites * K / (ms * 1e-3) / 1e9
    kname = ("k_fused(sc)" if MODEL[0] == "sc" else "k_fused") if two else "k_single"
    rec = {"value": value, "unit": "GLUPS", "ms_per_step": ms_max / K,
           "config": config_of(w, storage, {"parallelism": ("z-slabs x%d of a %dx%dx%d box, halo exchange by NCCL send/recv" % (world, w.nx, w.ny, world * w.nz)) if slabs else "single GPU"}),
           "roofline": {"bound": "hbm", "kernel": "k_fused" if two else "k_single", "achieved": achieved, "peak": peak,
                        "unit": "GB/s", "frac": achieved / peak, "traffic": stored_traffic(kname, wl_name, storage),
                        "peak_source": peak_src, "algorithmic_bytes_per_update": upd_bytes,
                        "kernel_ms": ms_k2, "kernel_share_of_step": ms_k2 * K / ms,
                        "phase_kernel_ms": ms_k1, "kernel_timing": kernel_timing,
                        "whole_step_effective_gbs": whole, "whole_step_frac": whole / peak,
                        "whole_step_frac_of_nominal_8000": whole / NOMINAL_HBM_GBS},
           "clocks": dict(clk.result, remeasured=remeasured), "gpu_launches": int(launches),
           "checks": {"finite": finite, "red_mass_rel_drift": drift[0], "blue_mass_rel_drift": drift[1]}}

    if with_e2e:
        # end to end through the C-ABI with HOST buffers: init (H2D) + K steps + get_macros (D2H)
        h_rr = torch.from_numpy(w.rho_r).pin_memory()
        h_rb = torch.from_numpy(w.rho_b).pin_memory() if two else None
        h_u = torch.from_numpy(w.u).pin_memory()
        o_rr, o_u = torch.empty_like(h_rr).pin_memory(), torch.empty_like(h_u).pin_memory()
        o_rb = torch.empty_like(h_rb).pin_memory() if two else None
        sim.set_profiling(False)
        e2e_ms = []
        for _ in range(2):          # first pass warms the staging allocations
            torch.cuda.synchronize()
            if world > 1:
                dist.barrier()
            t0 = time.perf_counter()
            sim.init(h_rr, h_rb, h_u)
            sim.step(K)
            sim.get_macros(o_rr, o_rb, o_u)
            torch.cuda.synchronize()
            e2e_ms.append((time.perf_counter() - t0) * 1e3)
        e2e_max = max_over_ranks(e2e_ms[-1], world, dev)
        nfield = (5 if two else 4) * w.sites * 4
        rec["e2e"] = {"value": glups(w.fluid_sites, K, e2e_max * 1e-3, world), "unit": "GLUPS",
                      "h2d_bytes_per_step": nfield / K, "d2h_bytes_per_step": nfield / K,
                      "note": "lb_init(host) + lb_step(%d) + lb_get_macros(host) per timed region; bytes are totals / K" % K}
        del h_rr, h_rb, h_u, o_rr, o_rb, o_u

    # optional: throughput over the course of the run (the interface fraction changes as domains
    # coarsen or droplets move): --windows N times N windows of K steps spread over w.steps
    if windows > 0 and world == 1:
        sim.init(d_rr, d_rb, d_u)
        gap = max(0, (w.steps - windows * K) // max(1, windows - 1)) if windows > 1 else 0
        out, done = [], 0
        for i in range(windows):
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); sim.step(K); e1.record(); torch.cuda.synchronize()
            done += K
            entry = {"steps": [done - K, done], "glups": glups(w.fluid_sites, K, e0.elapsed_time(e1) * 1e-3, 1)}
            if two:
                phi = sim.get_phi()
                fl = np.ones(w.shape, bool) if w.solid is None else (w.solid == 0)
                entry["interface_fraction"] = float((np.abs(phi[fl]) < 0.9).mean())
            out.append(entry)
            if i + 1 < windows and gap:
                sim.step(gap); done += gap
        rec["windows"] = out

    sim.destroy()
    del sim, d_rr, d_rb, d_u
    torch.cuda.empty_cache()
    return rec, w


# The other rows of the table: measured in the same run, after the headline, and
# reported under "configs" in the same JSON line.
EXTRA_CONFIGS = [("c3", "ab"), ("c4", "ab"), ("c5", "aa"), ("c2", "ab"), ("bijel", "ab")]


def run_ours(args):
    import torch
    import torch.distributed as dist
    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1 and not dist.is_initialized():
        dist.init_process_group("nccl", device_id=dev)
    K, Wu = args.steps, args.warmup

    head, w = measure_config(args.workload, args.storage, K, Wu, dev, local_rank, world, with_e2e=True, windows=args.windows,
                             slabs=world > 1 or args.slabs)
    extra = []
    if args.configs == "all" and world == 1 and MODEL[0] == "cg":
        for name, storage in EXTRA_CONFIGS:
            if (name, storage) == (args.workload, args.storage):
                continue
            rec, wx = measure_config(name, storage, K, Wu, dev, local_rank, world, w=w if name == args.workload else None)
            rec.pop("unit", None)
            extra.append(rec)
            del wx
    if rank != 0:
        return 0
    line = {"metric": METRIC, "value": head["value"], "unit": "GLUPS", "n_gpus": world, "steps": K, "warmup": Wu,
            "ms_per_step": head["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic", "config": head["config"], "clocks": head["clocks"], "e2e": head["e2e"],
            "gpu_launches": head["gpu_launches"], "roofline": head["roofline"], "checks": head["checks"]}
    if "windows" in head:
        line["windows"] = head["windows"]
    if extra:
        line["configs"] = extra
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(args.workload)
    elif world > 1:
        line["cpu_baseline"] = None
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c5", choices=["c1", "c2", "c3", "c4", "c5", "c2-mini", "c3-mini", "c4-mini", "c5-mini", "focuser", "focuser-3d", "focuser-drip", "focuser-large", "bijel", "bijel-mini"])
    ap.add_argument("--storage", default="ab", choices=["ab", "aa"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--tune", default="", help="lb_set_tuning settings for experiments, e.g. forward=0,zc=12,graph=0")
    ap.add_argument("--slabs", action="store_true", help="run the z-slab driver also at N = 1 (the rank is then its own neighbour)")
    ap.add_argument("--configs", default=None, choices=["all", "none"], help="all = also measure C3 A/B, C4 A/B, C5 AA, C2 and the bijel workload and report them under 'configs' (default when --workload is left at c5)")
    ap.add_argument("--model", default="cg", choices=["cg", "sc"], help="cg = colour gradient (north_star), sc = Shan-Chen + exact difference (Eq. 5-10 of the paper)")
    ap.add_argument("--gc", type=float, default=3.0, help="G_C of the Shan-Chen model")
    ap.add_argument("--windows", type=int, default=0, help="also time N windows of K steps spread over the config's run length")
    args = ap.parse_args(argv)
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.configs is None:
        args.configs = "all" if (args.workload == "c5" and args.storage == "ab") else "none"
    MODEL[0], MODEL[1] = args.model, args.gc
    TUNE.update({k: int(v) for k, v in (kv.split("=") for kv in args.tune.split(",") if kv)})
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())

#!/usr/bin/env python
"""bench.py -- throughput of the Strang semi-Lagrangian Vlasov step on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl cuda|reference]
                    [--config cfg1..cfg5] [--grid N] [--precision 64|32] [--spline fd|gs] [--order 2|4]

Workload (BASELINE.json cfg 5 / north_star, the default): HMF model, water-bag + seeded noise, N x N grid (default
8192 x 8192, fp64), dt = 0.1.  --config cfg1 .. cfg4 runs the other BASELINE.json configurations at their own sizes
(their state fits the 126 MB L2 -- cfg 4 nearly -- so no DRAM roofline is claimed for them).  A "step" is one full
Strang step (theta half shift, density, force, p shift, theta half shift).  Prints ONE JSON line (rank 0).

  value      grid-point updates per second per Strang step (Gpts/s), whole job, state resident in HBM.  K steps are
             timed as ONE vlasov_step(K) call between CUDA events on the launch stream; the call is repeated (at
             least 3 times) and the MEDIAN repetition is reported; reps_ms lists all of them.
             A call of K steps makes K + 1 passes over f (the first half theta shift is a pass of its own and the
             last pass applies one half shift instead of two): ms_per_step carries that 1/K overhead.
  e2e        same metric through the C ABI with HOST buffers: every step uploads f from pinned host memory,
             runs vlasov_step(1) and downloads f back to pinned host memory
  roofline   dominant kernel (the one-pass kernel: p shift + two theta half shifts + density) against the
             measured HBM peak; algorithmic bytes = 16 B per grid point per launch in fp64 (one read + one
             write of f); its duration comes from CUDA events around every launch in a further run of the
             same K steps (the timed region itself carries no per-kernel events); step_frac is the whole
             step against the bytes this run's passes must move, two_pass_step_frac against the 32 B per
             point of the two-pass minimum north_star names; target = north_star's 0.70 per Strang step.
             traffic is NOT measured by this run: it is the DRAM byte count of the committed ncu capture named in
             traffic_source (profiles/traffic.txt), refreshed with every kernel change.
  cpu_baseline  the CPU oracle (oracle/, as it stands) timed on this box's host cores on a bounded sample

--spline gs times the Global Spline variant instead (system (15), the paper's comparator).
--impl reference times the oracle (there is no other reference implementation: the paper ships no code) on the SAME
grid as the CUDA arm; the number of steps it really runs is capped so that the run ends within --ref-seconds.
N > 1: independent replicas (the path does not shard in this build): one process per
GPU, no data-path collective, value = all replicas' grid points / max time.  `python bench.py --gpus N` without
torchrun re-executes itself under torch.distributed.run with N processes.
"""
from __future__ import annotations

import argparse
import json
import os
import socket
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "vlasov_grid_point_updates_per_second_per_strang_step"
UNIT = "Gpts/s"
HBM_FALLBACK_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback
L2_BYTES = 126e6
TARGET_STEP_FRAC = 0.70    # north_star: >= 70 % of the HBM roofline per Strang step at 8192^2
MODEL_NAMES = {0: "free streaming", 1: "HMF", 2: "ring", 3: "sheet"}


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def committed_traffic(kernel: str, n: int, precision: int):
    """(DRAM bytes per launch, provenance) of the dominant kernel from the committed ncu capture, or (None, None).
    profiles/traffic.txt: `<kernel>_n<N>_fp<P>_dram_bytes_per_launch = <bytes>  # ...` and a `source = ...` line."""
    path = os.path.join(ROOT, "profiles", "traffic.txt")
    key = "%s_n%d_fp%d_dram_bytes_per_launch" % (kernel, n, precision)
    val, src = None, None
    try:
        with open(path) as fh:
            for line in fh:
                if line.startswith(key):
                    val = float(line.split("=")[1].split()[0])
                    if "@" in line:
                        src = line.split("@", 1)[1].strip()
    except Exception:
        pass
    if val is None:
        return None, None
    return val, "profiles/traffic.txt (committed ncu --set full capture%s); not measured in this run" % (
        ", " + src if src else "")


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML from the warm-up to the end of the timed repetitions."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop_evt = threading.Event()
        try:
            import pynvml

            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake",
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, name in names.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.0005)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2.0)
        med = int(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def max_over_ranks(value: float, world: int, backend_device=None) -> float:
    """max of a float over all ranks (identity for world == 1).  Uses the initialised process group."""
    if world == 1:
        return float(value)
    import torch
    import torch.distributed as dist

    t = torch.tensor([float(value)], dtype=torch.float64, device=backend_device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def median_rep(reps_ms):
    """the median repetition (an actually measured one: the upper median for an even count)"""
    s = sorted(reps_ms)
    return s[len(s) // 2]


# ------------------------------------------------------------------------------------------ the workload
def workload(args, with_f0=True):
    """the BASELINE.json configuration this run uses and the `config` object both arms print (identical)"""
    from paper_1206_3229_b200 import inputs

    kw = {}
    if args.n:
        kw["n"] = args.n
    c = inputs.config(args.config, with_f0=with_f0, **kw)
    nt, npp = c["grid"]
    eb = 8 if args.precision == 64 else 4
    fits = nt * npp * eb <= L2_BYTES
    bc = "x zero-extended (open)" if c["model"] == inputs.MODEL_SHEET else "theta periodic"
    cfg = {
        "workload": "%s %s %dx%d %s, dt=%g, %s, p zero-extended%s" % (
            args.config, MODEL_NAMES[c["model"]], nt, npp, "fp64" if eb == 8 else "fp32", c["dt"], bc,
            ", global-spline variant (system 15)" if args.spline == "gs" else ""),
        "cfg": args.config, "grid": [nt, npp], "precision": args.precision, "spline": args.spline, "order": args.order,
        "l2": "state fits L2: DRAM roofline not claimed" if fits else
              "state (%.0f MiB x 2 buffers) exceeds the 126 MB L2; no flush needed" % (nt * npp * eb / 2 ** 20),
    }
    return c, cfg


# ------------------------------------------------------------------------------------------ oracle legs
def make_oracle(c, spline: int, order: int = 2):
    import oracle

    cores = os.cpu_count() or 1
    params = dict(c["params"])
    if spline:
        params["spline"] = spline
    if order == 4:
        params["order"] = 4
    o = oracle.Oracle(c["model"], c["grid"], c["domain"], c["dt"], threads=cores, **params)
    o.upload(c["f0"])
    return o


def oracle_throughput(c, steps: int, min_seconds: float = 0.0, spline: int = 0, order: int = 2):
    """Gpts/s of the CPU oracle on the workload c, all host cores: `steps` at a time until min_seconds have passed"""
    o = make_oracle(c, spline, order)
    pts = float(c["grid"][0]) * float(c["grid"][1])
    done, t0 = 0, time.perf_counter()
    while True:
        o.step(steps)
        done += steps
        el = time.perf_counter() - t0
        if el >= min_seconds:
            break
    threads = o.threads
    o.close()
    return pts * done / el / 1e9, el, done, threads


def run_reference(args):
    """The oracle as it stands on the host cores, on the CUDA arm's grid.  The driver's --steps K --warmup W would take
    K x 2 s at 8192^2, so the steps really run are capped: the first step is timed, then as many warm-up and timed
    steps as fit --ref-seconds (at least one timed step)."""
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    c, cfg = workload(args)
    pts = float(c["grid"][0]) * float(c["grid"][1])
    t_wall = time.perf_counter()
    o = make_oracle(c, int(args.spline == "gs"), args.order)
    t0 = time.perf_counter()
    o.step(1)                      # first step: untimed warm-up (page faults of the oracle's arrays) and the estimate
    t1 = time.perf_counter() - t0
    budget = max(args.ref_seconds - t1, 0.0)
    w_eff = min(max(args.warmup - 1, 0), int(0.1 * budget / t1))
    k_eff = max(1, min(args.steps, int(0.9 * budget / t1)))
    if w_eff:
        o.step(w_eff)
    t0 = time.perf_counter()
    o.step(k_eff)
    el = time.perf_counter() - t0
    threads = o.threads
    o.close()
    val = pts * k_eff / el / 1e9
    sample = ("CPU oracle (oracle/vlasov_oracle.c, OpenMP over lines) on the full %dx%d grid of the workload; %d timed "
              "Strang steps after %d warm-up steps (the requested %d + %d capped to fit %.0f s)" % (
                  c["grid"][0], c["grid"][1], k_eff, 1 + w_eff, args.steps, args.warmup, args.ref_seconds))
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": el / k_eff * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg,
        "steps_timed": k_eff, "warmup_done": 1 + w_eff,
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0, "wall_s": time.perf_counter() - t_wall,
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------ CUDA arm
KERNEL_NAMES = {
    "theta2": "theta_sweep_bulk_kernel<2 shifts>", "theta1": "theta_sweep_bulk_kernel<1 shift>",
    "p": "p_sweep_kernel", "ptheta2": "strang_fused_ws_kernel<p shift + 2 theta half shifts + density>",
    "ptheta1": "strang_fused_ws_kernel<p shift + 1 theta half shift>"}
GS_KERNEL_NAMES = {"theta1": "gs_theta_rec_kernel", "p": "gs_p_rec_kernel"}


def run_cuda(args):
    import torch

    from paper_1206_3229_b200 import binding as vb

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=dev)

    prec, K, W = args.precision, args.steps, max(args.warmup, 0)
    eb = 8 if prec == 64 else 4
    c, cfg = workload(args)
    nt, npp = c["grid"]
    f0 = c["f0"].astype(np.float64 if prec == 64 else np.float32)
    params = dict(c["params"])
    params.update(fuse=args.fuse, tune_graph=args.graph, tune_pdl=args.pdl)
    if args.spline == "gs":
        params["spline"] = vb.SPLINE_GS
    if args.order == 4:
        params["order"] = 4
    if args.fbands > 0:
        params["tune_fbands"] = args.fbands
    if args.fedge > 0:
        params["tune_fedge"] = args.fedge
    if args.tile > 0:
        params["tune_tile"] = args.tile
    if args.rc > 0:
        params["tune_rc"] = args.rc
    if args.history > 0:
        params["history"] = 1
        if args.history == 2:
            params["tune_hist"] = 2
    g = vb.Vlasov(c["model"], c["grid"], c["domain"], c["dt"], precision=prec, device="cuda:%d" % local_rank, **params)
    g.upload(f0)
    pts = float(nt) * float(npp)

    def barrier():
        if world > 1:
            import torch.distributed as dist

            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: W warm-up steps, then repetitions of exactly K steps as one vlasov_step(K) call
    # (no per-kernel events in this region); the clock sampler runs from the warm-up to the last repetition
    sampler = ClockSampler(local_rank)
    sampler.start()
    if W:
        g.step(W)
    barrier()
    reps_ms, launches = [], 0
    t_load = time.perf_counter()
    while len(reps_ms) < args.reps or (time.perf_counter() - t_load < args.min_load_seconds and len(reps_ms) < 50):
        launches0 = vb.vlasov_launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        g.step(K)
        e1.record()
        barrier()
        reps_ms.append(max_over_ranks(e0.elapsed_time(e1), world, dev))
        launches = vb.vlasov_launch_count() - launches0
    clocks = sampler.stop()
    ms = median_rep(reps_ms)
    value = world * pts * K / (ms * 1e-3) / 1e9

    # ---- the same K steps again with a CUDA-event pair around every launch: per-kernel durations for the roofline
    vb.vlasov_set_param(vb.KEY_PROFILE, 1)
    vb.vlasov_kernel_times()  # reset
    g.step(K)
    ktimes = vb.vlasov_kernel_times()
    vb.vlasov_set_param(vb.KEY_PROFILE, 0)
    mom = g.moments()

    # ---- roofline of the dominant kernel
    peak, peak_src = measured_peak()
    kern = {}
    for name, d in ktimes.items():
        if d["launches"] > 0 and name != "force":
            avg_ms = d["ms"] / d["launches"]
            kern[name] = {"avg_ms": avg_ms, "launches": d["launches"],
                          "achieved_gbs": 2 * eb * pts / (avg_ms * 1e-3) / 1e9}
        elif d["launches"] > 0:
            kern[name] = {"avg_ms": d["ms"] / d["launches"], "launches": d["launches"]}
    sweeps = [k for k in kern if k != "force"]
    dom = max(sweeps, key=lambda k: kern[k]["avg_ms"] * kern[k]["launches"]) if sweeps else None
    passes = sum(kern[k]["launches"] for k in sweeps)
    step_bytes = 2 * eb * passes / K  # algorithmic bytes per grid point per step of THIS run (one read + one write per pass)
    roofline = None
    if dom is not None:
        ach = kern[dom]["achieved_gbs"]
        gs = args.spline == "gs"
        traffic, traffic_src = committed_traffic(("gsrec_" if gs else "") + dom, nt, prec) if nt == npp else (None, None)
        step_frac = (step_bytes * pts * K / (ms * 1e-3) / 1e9) / peak
        kname = (GS_KERNEL_NAMES if gs else KERNEL_NAMES).get(dom, dom)
        if g.info().get("onepass_tile") and dom in ("ptheta2", "ptheta1"):  # small grids: the tile kernel ran
            kname = kname.replace("strang_fused_ws_kernel", "strang_tile_kernel")
        roofline = {"bound": "hbm", "kernel": kname,
                    "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                    "traffic": traffic, "traffic_source": traffic_src,
                    "peak_source": peak_src, "algorithmic_bytes_per_launch": 2 * eb * pts,
                    "step_frac": step_frac, "step_bytes_per_point": step_bytes,
                    "two_pass_step_frac": (4 * eb * pts * K / (ms * 1e-3) / 1e9) / peak,
                    "target_step_frac": TARGET_STEP_FRAC, "meets_target": bool(step_frac >= TARGET_STEP_FRAC)}
        if nt * npp * eb <= L2_BYTES:
            roofline["note"] = "state fits L2: the fractions above are NOT a DRAM roofline claim"

    # ---- end to end through the C ABI with host buffers
    Ke = min(K, args.e2e_steps)
    host = torch.empty((npp, nt), dtype=torch.float64 if prec == 64 else torch.float32).pin_memory()
    host.numpy()[:] = f0
    hp = host.data_ptr()
    for _ in range(2):
        vb.vlasov_upload_ptr(hp)
        vb.vlasov_step(1)
        vb.vlasov_download_ptr(hp)
    host.numpy()[:] = f0
    barrier()
    e2, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e2.record()
    for _ in range(Ke):
        vb.vlasov_upload_ptr(hp)      # H2D of this step's input, pinned host memory
        vb.vlasov_step(1)
        vb.vlasov_download_ptr(hp)    # D2H of this step's result (blocks)
    e3.record()
    barrier()
    ms_e2e = max_over_ranks(e2.elapsed_time(e3), world, dev)
    e2e = {"value": world * pts * Ke / (ms_e2e * 1e-3) / 1e9, "unit": UNIT, "h2d_bytes_per_step": int(pts * eb),
           "d2h_bytes_per_step": int(pts * eb), "steps": Ke, "ms_per_step": ms_e2e / Ke,
           "call": "vlasov_upload(pinned host) + vlasov_step(1) + vlasov_download(pinned host)"}
    info = g.info()
    g.close()
    if world > 1:
        import torch.distributed as dist

        dist.destroy_process_group()
    if rank != 0:
        return 0

    # ---- oracle on the host cores (bounded sample of the same workload), rank 0 only
    cpu = None
    if not args.no_cpu_baseline:
        val, el, done, threads = oracle_throughput(c, 1, min_seconds=args.cpu_seconds, spline=int(args.spline == "gs"), order=args.order)
        cpu = {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle",
               "sample": "%d Strang step(s) of the same workload on its full %dx%d grid (%.1f s of wall time), "
                         "oracle/vlasov_oracle.c with OpenMP over lines" % (done, nt, npp, el)}

    # `config` is the same object in both arms (the driver compares them); what is particular to this run sits in `run`
    run = {"passes_per_step": passes / K, "fuse": args.fuse, "pdl": args.pdl, "graph": args.graph, "history": args.history,
           "parallelism": "replicas x%d" % world if world > 1 else "single GPU"}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64" if prec == 64 else "f32", "data": "synthetic", "config": cfg,
        "timing": {"reps": len(reps_ms), "reps_ms": reps_ms, "statistic": "median repetition of vlasov_step(K)",
                   "note": "K steps = K + 1 passes (first half theta shift + last pass with one half shift)"},
        "run": run, "launch": info, "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "kernels": kern,
        "cpu_baseline": cpu, "final_moments": {"t": mom[0], "mass": mom[1], "E": mom[7], "Mx": mom[5]},
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------ HMF molecular dynamics
MD_METRIC = "hmf_md_particle_steps_per_second"
MD_UNIT = "Gparticle-steps/s"


def md_config(args):
    return {"workload": "HMF molecular dynamics, N = %d particles, water-bag theta0 = 1, p0 = 1, dt = 0.1, fourth-order "
                        "symplectic integrator (PAPER.md L206, Fig. 4: N = 2e7)" % args.particles,
            "particles": args.particles, "precision": 64, "passes_per_step": 3,
            "l2": "state (%.0f MiB) exceeds the 126 MB L2; no flush needed" % (16.0 * args.particles / 2 ** 20)
            if 16.0 * args.particles > L2_BYTES else "state fits L2: DRAM roofline not claimed"}


def md_oracle_rate(n, steps, min_seconds=0.0):
    """G particle-steps/s of the CPU oracle (one host thread: plain C loops)"""
    import oracle
    from paper_1206_3229_b200 import inputs

    th, p = inputs.md_waterbag(n, 1.0, 1.0)
    o = oracle.MdOracle(n, 0.1)
    o.upload(th, p)
    done, t0 = 0, time.perf_counter()
    while True:
        o.step(steps)
        done += steps
        el = time.perf_counter() - t0
        if el >= min_seconds:
            break
    o.close()
    return n * done / el / 1e9, el, done


def run_md_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    t_wall = time.perf_counter()
    n = args.particles
    val1, t1, _ = md_oracle_rate(n, 1)                      # first step: the estimate (and the page faults)
    k_eff = max(1, min(args.steps, int(0.9 * max(args.ref_seconds - t1, 0.0) / t1)))
    val, el, done = md_oracle_rate(n, k_eff)
    sample = ("CPU oracle (oracle/hmf_md_oracle.c, one host thread) on all %d particles; %d timed steps (the requested "
              "%d capped to fit %.0f s)" % (n, done, args.steps, args.ref_seconds))
    print(json.dumps({
        "impl": "reference", "metric": MD_METRIC, "value": val, "unit": MD_UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": el / done * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": md_config(args), "steps_timed": done,
        "cpu_baseline": {"value": val, "unit": MD_UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": MD_UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0, "wall_s": time.perf_counter() - t_wall}))
    return 0


def run_md(args):
    import torch

    from paper_1206_3229_b200 import binding as vb
    from paper_1206_3229_b200 import inputs

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=dev)
    n, K, W = args.particles, args.steps, max(args.warmup, 0)
    th, p = inputs.md_waterbag(n, 1.0, 1.0)
    g = vb.HmfMd(n, 0.1, device="cuda:%d" % local_rank)
    g.upload(th, p)

    def barrier():
        if world > 1:
            import torch.distributed as dist

            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local_rank)
    sampler.start()
    if W:
        g.step(W)
    barrier()
    reps_ms, launches = [], 0
    t_load = time.perf_counter()
    while len(reps_ms) < args.reps or (time.perf_counter() - t_load < args.min_load_seconds and len(reps_ms) < 50):
        l0 = vb.hmf_md_launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        g.step(K)
        e1.record()
        barrier()
        reps_ms.append(max_over_ranks(e0.elapsed_time(e1), world, dev))
        launches = vb.hmf_md_launch_count() - l0
    clocks = sampler.stop()
    ms = median_rep(reps_ms)
    value = world * float(n) * K / (ms * 1e-3) / 1e9
    g.profile(True)
    g.kernel_times()
    g.step(K)
    kms, kl = g.kernel_times()
    g.profile(False)
    mom = g.moments()
    peak, peak_src = measured_peak()
    avg_ms = kms / max(kl, 1)
    ach = 32.0 * n / (avg_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": "md_kick_drift_kernel", "achieved": ach, "peak": peak, "unit": "GB/s",
                "frac": ach / peak, "traffic": None, "peak_source": peak_src, "algorithmic_bytes_per_launch": 32.0 * n,
                "note": "32 B per particle and pass (theta, p read and written), 3 passes per step; the pass also runs "
                        "two fp64 sincos per particle"}
    # end to end with host buffers
    Ke = min(K, args.e2e_steps)
    ht, hp = torch.from_numpy(th).pin_memory(), torch.from_numpy(p).pin_memory()
    for _ in range(2):
        g.upload_ptr(ht.data_ptr(), hp.data_ptr())
        g.step(1)
        g.download_ptr(ht.data_ptr(), hp.data_ptr())
    barrier()
    e2, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e2.record()
    for _ in range(Ke):
        g.upload_ptr(ht.data_ptr(), hp.data_ptr())
        g.step(1)
        g.download_ptr(ht.data_ptr(), hp.data_ptr())
    e3.record()
    barrier()
    ms_e2e = max_over_ranks(e2.elapsed_time(e3), world, dev)
    e2e = {"value": world * float(n) * Ke / (ms_e2e * 1e-3) / 1e9, "unit": MD_UNIT, "h2d_bytes_per_step": 16 * n,
           "d2h_bytes_per_step": 16 * n, "steps": Ke, "ms_per_step": ms_e2e / Ke,
           "call": "hmf_md_upload(pinned host) + hmf_md_step(1) + hmf_md_download(pinned host)"}
    g.close()
    if world > 1:
        import torch.distributed as dist

        dist.destroy_process_group()
    if rank != 0:
        return 0
    cpu = None
    if not args.no_cpu_baseline:
        val, el, done = md_oracle_rate(n, 1, min_seconds=args.cpu_seconds)
        cpu = {"value": val, "unit": MD_UNIT, "cores": 1, "kind": "oracle",
               "sample": "%d step(s) of all %d particles (%.1f s of wall time), oracle/hmf_md_oracle.c, one host thread" % (done, n, el)}
    cfg = md_config(args)
    cfg["parallelism"] = "replicas x%d" % world if world > 1 else "single GPU"
    print(json.dumps({
        "metric": MD_METRIC, "value": value, "unit": MD_UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": cfg,
        "timing": {"reps": len(reps_ms), "reps_ms": reps_ms, "statistic": "median repetition of hmf_md_step(K)"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline,
        "kernels": {"md_kick_drift": {"avg_ms": avg_ms, "launches": kl, "achieved_gbs": ach}}, "cpu_baseline": cpu,
        "final_moments": {"t": mom[0], "Mx": mom[1], "E": mom[5], "P": mom[6]}}))
    return 0


# ------------------------------------------------------------------------------------------ p-slab sharding (strong scaling)
def run_slab(args):
    """--shard slab: ONE grid cut into p-slabs over the ranks (paper_1206_3229_b200/slab.py):
    per step one all-reduce of rho and one halo exchange over NCCL, stages through the library's slab mode (two-pass
    kernels).  Strong scaling: value = the grid's points x K / max time.  Never measured on more than one GPU by this
    build (no multi-GPU box was available); with one rank it times the unsharded stage sequence."""
    import torch

    from paper_1206_3229_b200 import slab

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=dev)
    c, cfg = workload(args)
    nt, npp = c["grid"]
    K, W = args.steps, max(args.warmup, 0)
    dp = (c["domain"][3] - c["domain"][2]) / npp
    halo = slab.halo_depth(args.slab_fmax, c["dt"], dp) if world > 1 else 0
    b = slab.LibrarySlab(c["model"], c["grid"], c["domain"], c["dt"], rank, world, halo, device="cuda:%d" % local_rank,
                         precision=args.precision, **c["params"])
    b.upload_global(c["f0"])
    st = slab.SlabStepper(b, rank, world, dist)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local_rank)
    sampler.start()
    if W:
        st.step(W)
    reps_ms = []
    for _ in range(max(args.reps, 3)):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        st.step(K)
        e1.record()
        barrier()
        reps_ms.append(max_over_ranks(e0.elapsed_time(e1), world, dev))
    clocks = sampler.stop()
    ms = median_rep(reps_ms)
    b.close()
    if world > 1:
        dist.destroy_process_group()
    if rank != 0:
        return 0
    cfg = dict(cfg)
    cfg.update({"parallelism": "p-slabs x%d (rho all-reduce + halo exchange of %d rows per step)" % (world, halo),
                "passes_per_step": 3})
    print(json.dumps({
        "metric": METRIC, "value": float(nt) * float(npp) * K / (ms * 1e-3) / 1e9, "unit": UNIT, "n_gpus": world, "steps": K,
        "warmup": W, "ms_per_step": ms / K, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
        "dtype": "f64" if args.precision == 64 else "f32", "data": "synthetic", "config": cfg,
        "timing": {"reps": len(reps_ms), "reps_ms": reps_ms, "statistic": "median repetition of K sharded steps"},
        "clocks": clocks, "gpu_launches": 5 * K, "roofline": None, "cpu_baseline": None, "e2e": None}))
    return 0


def relaunch_under_torchrun(args) -> int:
    """`python bench.py --gpus N` without torchrun: run N ranks of this script under torch.distributed.run"""
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + [
               "--grid" if a == "--n" else a for a in sys.argv[1:]]
    os.execv(sys.executable, cmd)
    return 1  # not reached


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", default="cfg5", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"],
                    help="BASELINE.json configuration (cfg5 = the throughput workload the metric is quoted on)")
    ap.add_argument("--grid", "--n", dest="n", type=int, default=0,
                    help="grid size N (N x N); default: the configuration's own (cfg5: 8192).  Under torchrun write "
                         "--grid (torchrun's own parser finds --n ambiguous)")
    ap.add_argument("--precision", type=int, default=64, choices=[64, 32])
    ap.add_argument("--reps", type=int, default=3, help="repetitions of the timed vlasov_step(K) call (median reported)")
    ap.add_argument("--min-load-seconds", type=float, default=0.06,
                    help="keep repeating (up to 50 times) until the GPU has been under load this long (clock samples)")
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--cpu-seconds", type=float, default=10.0)
    ap.add_argument("--ref-seconds", type=float, default=120.0, help="wall-time cap of the --impl reference run")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--fuse", type=int, default=2, choices=[0, 1, 2],
                    help="passes per step: 2 = one (p + theta in one kernel, default), 1 = two, 0 = three")
    ap.add_argument("--fbands", type=int, default=0, help="bands of rows of the one-pass kernel (0 = automatic)")
    ap.add_argument("--tile", type=int, default=0, choices=[0, 1, 2],
                    help="one-pass step of small grids by the tile kernel: 0 by size (default), 1 wherever it applies, 2 never")
    ap.add_argument("--history", type=int, default=0, choices=[0, 1, 2],
                    help="1: HISTORY = 1 (the eight moments recorded after every step; HMF: still on the one-pass path), 2: the same "
                         "by the separate passes (TUNE_HIST = 2)")
    ap.add_argument("--rc", type=int, default=0, choices=[0, 2],
                    help="HMF density / force of short theta axes by one thread-block cluster: 0 (default), 2 never (the ticketed kernel)")
    ap.add_argument("--fedge", type=int, default=0, help="zero-extended x: width (percent) of the two edge column blocks (0 = automatic)")
    ap.add_argument("--graph", type=int, default=1, choices=[0, 1],
                    help="1 (default): steady-state step pairs are launched as CUDA graphs, 0: plain launches")
    ap.add_argument("--pdl", type=int, default=1, choices=[0, 1],
                    help="1 (default): programmatic dependent launch between the pass and the density/force kernel")
    ap.add_argument("--spline", default="fd", choices=["fd", "gs"],
                    help="fd: f'' by eq (16), the paper's method and the headline workload; gs: the Global Spline "
                         "comparator, system (15) (SURVEY 8(f) NEXT #2)")
    ap.add_argument("--shard", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: replicas (default; independent copies, weak scaling) or slab (one grid cut into p-slabs, "
                         "strong scaling; SURVEY 8(e))")
    ap.add_argument("--slab-fmax", type=float, default=1.0, help="--shard slab: bound of |F| the halo depth is sized for")
    ap.add_argument("--workload", default="vlasov", choices=["vlasov", "md"],
                    help="vlasov: the Strang semi-Lagrangian step (BASELINE.json's metric); md: the N-particle HMF "
                         "molecular dynamics of the paper's Fig. 4 (SURVEY 8(f) NEXT #3; its own metric, particle-steps/s)")
    ap.add_argument("--particles", type=int, default=20000000, help="--workload md: number of particles (paper: 2e7)")
    ap.add_argument("--order", type=int, default=2, choices=[2, 4],
                    help="2: the paper's time split (headline); 4: its triple-jump composition (SURVEY 8(f) NEXT #4), "
                         "nine passes and three force evaluations per step")
    args = ap.parse_args()
    _, _, world = dist_env()
    if args.gpus != world:
        if world == 1 and args.gpus > 1 and "RANK" not in os.environ:
            return relaunch_under_torchrun(args)
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE is %d (launch with torch.distributed.run "
                         "--nproc-per-node %d)" % (args.gpus, world, args.gpus))
    if args.workload == "md":
        return run_md_reference(args) if args.impl == "reference" else run_md(args)
    if args.impl == "reference":
        return run_reference(args)
    if args.shard == "slab":
        return run_slab(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())

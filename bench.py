#!/usr/bin/env python
"""bench.py -- throughput of the Strang semi-Lagrangian Vlasov step on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl cuda|reference] [--n GRID] [--precision 64|32]

Workload (BASELINE.json cfg 5 / north_star): HMF model, water-bag + seeded noise, N x N grid (default
8192 x 8192, fp64), dt = 0.1.  A "step" is one full Strang step (theta half shift, density, force, p shift,
theta half shift).  Prints ONE JSON line (rank 0).

  value      grid-point updates per second per Strang step (Gpts/s), whole job, state resident in HBM,
             K steps timed as one vlasov_step(K) call with CUDA events
  e2e        same metric through the C ABI with HOST buffers: every step uploads f from pinned host memory,
             runs vlasov_step(1) and downloads f back to pinned host memory
  roofline   dominant kernel (the one-pass kernel: p shift + two theta half shifts + density) against the
             measured HBM peak; algorithmic bytes = 16 B per grid point per launch in fp64 (one read + one
             write of f); its duration comes from CUDA events around every launch in a second run of the
             same K steps (the timed region itself carries no per-kernel events); step_frac is the whole
             step against the bytes this run's passes must move, two_pass_step_frac against the 32 B per
             point of the two-pass minimum north_star names
  cpu_baseline  the CPU oracle (oracle/, as it stands) timed on this box's host cores on a bounded sample

--spline gs times the Global Spline variant instead (system (15), the paper's comparator): three
passes per step with the recursive kernels (roofline against HBM like the FD path); --gsfir 1 selects the 60-tap
filter kernels (roofline.bound = "alu" against the measured fp64 FMA rate).  The oracle legs then run with
KEY_SPLINE = GS too.  The default (fd) is the paper's method and the headline workload.

--impl reference times the oracle (there is no other reference implementation: the paper ships no code).
N > 1: independent replicas (the path does not shard in this build): one process per
GPU, no data-path collective, value = all replicas' grid points / max time.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "vlasov_grid_point_updates_per_second_per_strang_step"
UNIT = "Gpts/s"
HBM_FALLBACK_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def committed_traffic(kernel: str, n: int, precision: int):
    """DRAM bytes per launch of the dominant kernel from the committed ncu capture (profiles/), or None."""
    path = os.path.join(ROOT, "profiles", "traffic.txt")
    key = "%s_n%d_fp%d_dram_bytes_per_launch" % (kernel, n, precision)
    try:
        with open(path) as fh:
            for line in fh:
                if line.startswith(key):
                    return float(line.split("=")[1].split()[0])
    except Exception:
        pass
    return None


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

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
            time.sleep(0.002)

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


# ------------------------------------------------------------------------------------------ oracle legs
def oracle_throughput(n: int, steps: int, warmup: int = 0, min_seconds: float = 0.0, spline: int = 0):
    """Gpts/s of the CPU oracle on the cfg-5 workload at grid n x n, all host cores."""
    import oracle
    from paper_1206_3229_b200 import inputs

    cores = os.cpu_count() or 1
    c = inputs.config("cfg5", n=n)
    o = oracle.Oracle(c["model"], c["grid"], c["domain"], c["dt"], threads=cores, **({"spline": spline} if spline else {}))
    o.upload(c["f0"])
    if warmup:
        o.step(warmup)
    done, t0 = 0, time.perf_counter()
    while True:
        o.step(steps)
        done += steps
        el = time.perf_counter() - t0
        if el >= min_seconds:
            break
    threads = o.threads
    o.close()
    return n * n * done / el / 1e9, el, done, threads


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    n_ref = args.ref_n
    t0 = time.perf_counter()
    val, el, done, threads = oracle_throughput(n_ref, args.steps, warmup=args.warmup, spline=int(args.spline == "gs"))
    sample = "CPU oracle (oracle/vlasov_oracle.c, OpenMP over lines), cfg5 HMF water-bag at %dx%d (bounded sample of the %dx%d workload), %d Strang steps" % (
        n_ref, n_ref, args.n, args.n, done)
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": el / done * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "cfg5 HMF water-bag %dx%d fp64, dt=0.1" % (args.n, args.n), "sample_grid": n_ref},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0, "wall_s": time.perf_counter() - t0,
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------ CUDA arm
def run_cuda(args):
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

    n, prec, K, W = args.n, args.precision, args.steps, max(args.warmup, 0)
    eb = 8 if prec == 64 else 4
    c = inputs.config("cfg5", n=n)
    f0 = c["f0"].astype(np.float64 if prec == 64 else np.float32)
    g = vb.Vlasov(c["model"], c["grid"], c["domain"], c["dt"], precision=prec, device="cuda:%d" % local_rank,
                  fuse=args.fuse, tune_fvariant=args.fvariant, tune_graph=args.graph,
                  **({"spline": vb.SPLINE_GS, "tune_gsfir": args.gsfir} if args.spline == "gs" else {}),
                  **({"tune_fbands": args.fbands} if args.fbands > 0 else {}))
    g.upload(f0)
    pts = float(n) * float(n)

    def barrier():
        if world > 1:
            import torch.distributed as dist

            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: W warm-up steps, then exactly K steps (no per-kernel events in this region)
    if W:
        g.step(W)
    sampler = ClockSampler(local_rank)
    barrier()
    launches0 = vb.vlasov_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.start()
    e0.record()
    g.step(K)
    e1.record()
    barrier()
    clocks = sampler.stop()
    ms_local = e0.elapsed_time(e1)
    launches = vb.vlasov_launch_count() - launches0

    # ---- the same K steps again with a CUDA-event pair around every launch: per-kernel durations for the roofline
    vb.vlasov_set_param(vb.KEY_PROFILE, 1)
    vb.vlasov_kernel_times()  # reset
    g.step(K)
    ktimes = vb.vlasov_kernel_times()
    vb.vlasov_set_param(vb.KEY_PROFILE, 0)
    ms = max_over_ranks(ms_local, world, dev)
    value = world * pts * K / (ms * 1e-3) / 1e9
    mom = g.moments()

    # ---- roofline of the dominant kernel (CUDA-event durations recorded inside the timed region)
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
        names = {"theta2": "theta_sweep_bulk_kernel<2 shifts>", "theta1": "theta_sweep_bulk_kernel<1 shift>",
                 "p": "p_sweep_kernel", "ptheta2": "strang_fused_ws_kernel<p shift + 2 theta half shifts + density>",
                 "ptheta1": "strang_fused_ws_kernel<p shift + 1 theta half shift>"}
        roofline = {"bound": "hbm", "kernel": names[dom],
                    "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                    "traffic": committed_traffic(dom, n, prec),
                    "peak_source": peak_src, "algorithmic_bytes_per_launch": 2 * eb * pts,
                    "step_frac": (step_bytes * pts * K / (ms_local * 1e-3) / 1e9) / peak,
                    "step_bytes_per_point": step_bytes,
                    "two_pass_step_frac": (4 * eb * pts * K / (ms_local * 1e-3) / 1e9) / peak}
        if args.spline == "gs" and args.gsfir == 0:
            # recursive global-spline kernels: ~18 fp64 operations per point and pass, one read + one write of f:
            # HBM-bound like the FD kernels
            gs_names = {"theta1": "gs_theta_rec_kernel", "p": "gs_p_rec_kernel"}
            roofline["kernel"] = gs_names.get(dom, dom)
            roofline["traffic"] = committed_traffic("gsrec_" + dom, n, prec)
        elif args.spline == "gs":
            # 60-tap filter kernels (A/B partner): 60 FMAs per point and pass, bound by the fp64 pipe.  Peak = the
            # measured fp64 FMA rate of this B200, 17.0 TFMA/s = 34.0 TFLOP/s (profiles/fp64_probe.txt).
            gs_names = {"theta1": "gs_theta_sweep_kernel", "p": "gs_p_sweep_kernel"}
            flops = 2.0 * 60.0 * pts
            ach_tf = flops / (kern[dom]["avg_ms"] * 1e-3) / 1e12
            roofline = {"bound": "alu", "kernel": gs_names.get(dom, dom), "achieved": ach_tf, "peak": 34.0,
                        "unit": "TFLOP/s", "frac": ach_tf / 34.0, "traffic": committed_traffic("gs_" + dom, n, prec),
                        "peak_source": "measured fp64 FMA rate, profiles/fp64_probe.txt (17.0 TFMA/s)",
                        "algorithmic_flops_per_launch": flops, "hbm_gbs": ach, "hbm_frac": ach / peak}

    # ---- end to end through the C ABI with host buffers
    Ke = min(K, args.e2e_steps)
    host = torch.empty((n, n), dtype=torch.float64 if prec == 64 else torch.float32).pin_memory()
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

    # ---- oracle on the host cores (bounded sample), rank 0 only
    cpu = None
    if not args.no_cpu_baseline:
        nb = args.cpu_n
        val, el, done, threads = oracle_throughput(nb, 1, warmup=0, min_seconds=args.cpu_seconds, spline=int(args.spline == "gs"))
        cpu = {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle",
               "sample": "%d Strang step(s) of cfg5 HMF water-bag on a %dx%d grid (%.1f s of wall time), oracle/vlasov_oracle.c with OpenMP over lines" % (done, nb, nb, el)}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64" if prec == 64 else "f32", "data": "synthetic",
        "config": {"workload": "cfg5 HMF water-bag %dx%d %s, dt=0.1, theta periodic, p zero-extended, seeded 1e-6 noise%s" % (
                       n, n, "fp64" if prec == 64 else "fp32", ", global-spline variant (system 15)" if args.spline == "gs" else ""),
                   "grid": [n, n], "passes_per_step": passes / K, "fuse": args.fuse,
                   "l2": "state (%.0f MiB x 2 buffers) exceeds the 126 MB L2; no flush needed" % (pts * eb / 2 ** 20)
                   if pts * eb > 126e6 else "state fits L2: DRAM roofline not claimed",
                   "parallelism": "replicas x%d" % world if world > 1 else "single GPU", "launch": info},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "kernels": kern,
        "cpu_baseline": cpu, "final_moments": {"t": mom[0], "mass": mom[1], "E": mom[7], "Mx": mom[5]},
    }
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--n", type=int, default=8192, help="grid size N (N x N)")
    ap.add_argument("--precision", type=int, default=64, choices=[64, 32])
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--cpu-n", type=int, default=8192, help="grid of the cpu_baseline sample")
    ap.add_argument("--cpu-seconds", type=float, default=10.0)
    ap.add_argument("--ref-n", type=int, default=1024, help="grid of the --impl reference sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--fuse", type=int, default=2, choices=[0, 1, 2],
                    help="passes per step: 2 = one (p + theta in one kernel, default), 1 = two, 0 = three")
    ap.add_argument("--fbands", type=int, default=0, help="bands of rows of the one-pass kernel (0 = automatic)")
    ap.add_argument("--graph", type=int, default=1, choices=[0, 1],
                    help="1 (default): steady-state step pairs are launched as CUDA graphs, 0: plain launches")
    ap.add_argument("--spline", default="fd", choices=["fd", "gs"],
                    help="fd: f'' by eq (16), the paper's method and the headline workload; gs: the Global Spline "
                         "comparator, system (15) (SURVEY 8(f) NEXT #2; three 60-tap passes per step, fp64-ALU bound)")
    ap.add_argument("--gsfir", type=int, default=0, choices=[0, 1],
                    help="with --spline gs: 1 = the 60-tap filter kernels instead of the recursive ones (A/B partner)")
    ap.add_argument("--fvariant", type=int, default=0, choices=[0, 1],
                    help="one-pass kernel: 0 = warp-specialised (default), 1 = every warp does both stages")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())

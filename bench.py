#!/usr/bin/env python
"""bench.py — MLUPS of the fused D3Q19 stream-collide path on the 400x400x100 urban config (BASELINE.json).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-cpu-baseline] [--workload c1..c5]

One bench "step" = one LBM time step of the whole lattice = one launch of the fused stream-collide kernel
(pull + bounce-back/free-slip/periodic resolution + moments + Coriolis/F + Smagorinsky + BGK/Guo + store, outflow
cells included).  `value` = cells x K / device time (CUDA events on the handle's stream, inputs resident in HBM).
`e2e` = the same metric for the whole job through the C ABI with pinned HOST buffers: heightmap, inlet profile and
initial field copied in, K steps, rho/u copied out — all inside the timed region.
N > 1 (torchrun): the path does not shard (north_star: one GPU, no collectives) -> N independent replicas, weak scaling.
`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores on a bounded crop of the workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

BYTES_PER_CELL = 153  # 19x4 B loads + 19x4 B stores + 1 flag byte (BASELINE.json north_star)
METRIC = "MLUPS (D3Q19 FP32), fused stream-collide, 400x400x100 urban config, 1 B200"   # BASELINE.json's metric = workload c3
SUSTAINED_SECONDS = 2.0   # the second timed region: back-to-back steps for at least this long (power-capped operating point)


def metric_for(workload):
    """The headline metric string names config 3; the other workloads are per-config table lines and say what they ran."""
    if workload == "c3":
        return METRIC
    if workload == "c3-fp16":
        return "MLUPS (D3Q19, FP32 arithmetic, 16-bit population storage), fused stream-collide, 400x400x100 urban config, 1 B200"
    if workload.endswith("-inplace"):
        return (f"MLUPS (D3Q19 {'FP32 arithmetic, 16-bit storage' if 'fp16' in workload else 'FP32'}), fused stream-collide with in-place "
                f"streaming (one population buffer), workload {workload} (a separate line, not the headline), 1 B200")
    return f"MLUPS (D3Q19 FP32), fused stream-collide, workload {workload} (per-config table line, not the headline), 1 B200"

# --workload: the headline is c3 (BASELINE.json: the config the metric is quoted on); the others are the parity configs,
# timed here only for the per-config table of DESIGN.md §12 (SURVEY.md §8(d) "report per config")
WORKLOADS = {
    "c1": "C1 tiny block flow 64x32x32 (BASELINE.json configs[0])",
    "c2": "C2 periodic Taylor-Green + Coriolis 128^3, Cs 0.1 (BASELINE.json configs[1])",
    "c3": "C3 urban 400x400x100 (BASELINE.json configs[2]): seeded heightmap plan fraction 0.35, log-law inlet, nu0 1e-4, Cs 0.1, f 2.9e-6",
    "c4": "C4 refined urban 800x800x200, veering inlet on three faces (BASELINE.json configs[3])",
    "thermal": "closed 400x400x100 city box with the D3Q7 thermal lattice + Boussinesq coupling on (DESIGN.md reading 23): 209 B/cell",
    "c3-fp16": "C3 urban 400x400x100 with 16-bit population storage (LBM_PREC_F32_S16, DESIGN.md §13): FP32 arithmetic, binary16 "
               "storage of the shifted populations, 77 B/cell — a separate line, NOT the FP32 headline",
    "c5": "C5 chain: periodic precursor 256x256x200 feeding the x- inlet of the 1200x1200x200 urban domain every step (BASELINE.json configs[4])",
    # in-place streaming (LBM_STREAM_INPLACE): the same step on ONE population buffer, half the memory, same 153 B/cell
    "c3-inplace": "C3 urban 400x400x100 with in-place streaming (one population buffer; DESIGN.md §14) — a separate line, NOT the headline",
    "c4-inplace": "C4 refined urban 800x800x200 with in-place streaming (one population buffer; DESIGN.md §14)",
    "c5-inplace": "C5 chain with in-place streaming on both lattices (one population buffer each; DESIGN.md §14)",
    "c3-fp16-inplace": "C3 urban 400x400x100, 16-bit population storage AND in-place streaming: 77 B/cell, a quarter of the FP32 two-buffer memory",
    "thermal-inplace": "closed 400x400x100 city box with the thermal lattice on, the flow lattice streaming in place (thermal populations double-buffered): 209 B/cell",
}


class Job:
    """One workload resident on the device: a single lattice, or the config-5 chain (precursor -> feed -> main)."""

    def __init__(self, name, binding, W, device):
        self.name, self.binding, self.device = name, binding, device
        inplace = name.endswith("-inplace")
        base = name[:-len("-inplace")] if inplace else name
        if base == "c5":
            self.wls = [W.config5_precursor(), W.config5_main()]
        else:
            self.wls = [{"c1": W.config1, "c2": lambda: W.config2(Cs=0.1), "c3": W.config3, "c4": W.config4,
                         "thermal": W.thermal_city, "c3-fp16": W.config3}[base]()]
        self.cells = sum(w.cells for w in self.wls)
        self.sims = [binding.from_workload(w, want_mean=False, device=device, storage16=(base == "c3-fp16"), inplace=inplace)
                     for w in self.wls]
        self.workspace_bytes = sum(s.workspace_bytes for s in self.sims)

    def step(self, n):
        if len(self.sims) == 1:
            self.sims[0].step(n)
            return
        pre, main = self.sims  # config-5 chain
        xs = self.wls[0].extra["sample_plane_x"]
        for _ in range(n):
            main.feed_inlet(pre, xs)
            pre.step(1)
            main.step(1)

    def launch_count(self):
        return sum(s.launch_count() for s in self.sims)

    def host_inputs(self, pin):
        """pinned host copies of everything the set-up of each lattice reads"""
        out = []
        for w in self.wls:
            prof = None if w.inlet_profile is None else tuple(None if a is None else pin(a) for a in w.inlet_profile)
            init = None if w.init is None else tuple(None if a is None else pin(a) for a in w.init)
            out.append((pin(w.height), prof, init))
        self.theta_host = [None if w.extra.get("theta") is None else pin(w.extra["theta"]) for w in self.wls]
        return out

    @staticmethod
    def nbytes(host):
        n = 0
        for h, prof, init in host:
            n += h.nbytes + sum(a.nbytes for a in (prof or ()) if a is not None) + sum(a.nbytes for a in (init or ()) if a is not None)
        return n

    def setup_from_host(self, host):
        for s, (h, prof, init) in zip(self.sims, host):
            s.set_flags(h)
            if prof is not None:
                s.set_inlet_profile(*prof)
            s.set_macros(*(init if init is not None else (None, None, None, None)))
        for s, th in zip(self.sims, getattr(self, "theta_host", [])):
            if th is not None:
                s.set_theta(th)  # thermal workload: the flags were re-set, so the thermal state is re-initialised too


def load_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def load_traffic(kernel="step"):
    """DRAM bytes per launch of the step kernel (dram__bytes_read.sum + dram__bytes_write.sum of the committed
    `ncu --set full` capture): last data row of the newest profiles/r*_<kernel>_kernel_traffic.csv.  Returns
    (bytes, source file) — (None, None) if absent.  A constant from a committed capture, NOT measured in this run."""
    import csv
    import glob
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", f"r*_{kernel}_kernel_traffic.csv")))
    if not files:
        return None, None
    try:
        rows = list(csv.DictReader(open(files[-1])))
        return float(rows[-1]["dram_bytes_total"]), os.path.relpath(files[-1], ROOT)
    except Exception:
        return None, None


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap,timestamp")

    def __init__(self, index=0):
        self.index = index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "20"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def wait_first_sample(self, timeout=2.0):
        """nvidia-smi needs ~0.1-0.3 s to print its first line: a short timed region must not start before it samples."""
        if self.p is None:
            return
        t0 = time.perf_counter()
        while time.perf_counter() - t0 < timeout:
            try:
                if os.path.getsize(self.f.name) > 0:
                    return
            except OSError:
                return
            time.sleep(0.01)

    def mark(self):
        """host wall-clock time, to cut the samples down to a window (nvidia-smi stamps each line with the same clock)"""
        return time.time()

    def stop(self, t_from=None, t_to=None):
        """Median SM clock and throttle reasons of the samples stamped within [t_from, t_to] (+- one sampling period); if the
        window is shorter than the sampling period and holds none, the sample nearest to it."""
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(",") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        if t_from is not None and t_to is not None:
            import datetime
            stamped = []
            for r in rows:
                try:
                    ts = datetime.datetime.strptime(r[7].strip(), "%Y/%m/%d %H:%M:%S.%f").timestamp()
                except Exception:
                    continue
                stamped.append((ts, r))
            inside = [r for ts, r in stamped if t_from - 0.02 <= ts <= t_to + 0.02]
            if not inside and stamped:
                mid = 0.5 * (t_from + t_to)
                inside = [min(stamped, key=lambda q: abs(q[0] - mid))[1]]
            if stamped:
                rows = inside
        sm, reasons, mx = [], set(), None
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0])); mx = float(r[1])
                for k, nme in enumerate(names):
                    if r[3 + k].strip().lower().startswith("active"):
                        reasons.add(nme)
            except Exception:
                continue
        if sm:
            sm.sort()
            out.update(sm_mhz=sm[len(sm) // 2], sm_max_mhz=mx, reasons=sorted(reasons), samples=len(sm))
        return out


def max_over_ranks(value, world, device):
    """Whole-job time = the slowest rank's device time (MAX all-reduce; identity for one rank)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_mlups(cells_per_rank, steps, world, seconds):
    """Replicas only: every rank advances its own lattice; the job's units are the sum over ranks."""
    return cells_per_rank * steps * world / seconds / 1e6


def oracle_for(wl):
    from oracle import Oracle
    o = Oracle(wl.nx, wl.ny, wl.nz, wl.nu0, wl.Cs, wl.f_cor, wl.F, wl.faces)
    o.set_flags(wl.height)
    o.set_inlet_profile(*wl.inlet_profile)
    o.set_macros(*wl.init)
    return o


def cpu_baseline(budget_s=15.0):
    """The oracle as it stands (gcc -O3 -fopenmp, FP64), on this host's cores, on a bounded sample of the workload
    (BASELINE.md §3): `value` = config 3's full 400x400 plan, lowest 25 levels (where the buildings are), a few steps;
    `c1` = config 1 in full (64x32x32, 200 steps)."""
    from paper_2607_04516_b200 import workloads as W
    cores = len(os.sched_getaffinity(0))
    w1 = W.config1()
    o1 = oracle_for(w1)
    o1.step(5)
    t0 = time.perf_counter(); o1.step(200); d1 = time.perf_counter() - t0
    o1.close()
    wl = W.config3(nz=25)
    o = oracle_for(wl)
    t0 = time.perf_counter(); o.step(1); t1 = time.perf_counter() - t0
    n = max(2, min(50, int(budget_s / max(t1, 1e-3))))
    t0 = time.perf_counter(); o.step(n); dt = time.perf_counter() - t0
    return {"value": wl.cells * n / dt / 1e6, "unit": "MLUPS", "cores": cores, "kind": "oracle",
            "sample": f"config-3 heightmap and inlet, 400x400x25 slab (4.0e6 cells), {n} steps, FP64, gcc -O3 -fopenmp, {cores} threads",
            "c1": {"value": w1.cells * 200 / d1 / 1e6, "unit": "MLUPS", "sample": "config 1 in full, 64x32x32, 200 steps"}}


def run_reference(args):
    """--impl reference: the oracle on the host cores; each step = one LBM step on a bounded crop of config 3."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_2607_04516_b200 import workloads as W
    cores = len(os.sched_getaffinity(0))
    budget = float(args.reference_budget)
    nz = 25
    wl = W.config3(nz=nz)
    o = oracle_for(wl)
    t0 = time.perf_counter(); o.step(1); t1 = time.perf_counter() - t0
    total = args.steps + args.warmup
    if t1 * total > budget:  # shrink the crop in y so that the whole run fits the budget
        ny = max(16, int(400 * budget / (t1 * total)) // 8 * 8)
        wl = W.config3(ny=ny, nz=nz)
        o = oracle_for(wl)
    o.step(args.warmup)
    t0 = time.perf_counter(); o.step(args.steps); dt = time.perf_counter() - t0
    v = wl.cells * args.steps / dt / 1e6
    sample = f"config-3 crop {wl.nx}x{wl.ny}x{wl.nz} ({wl.cells:.3g} cells), FP64 oracle, OpenMP {cores} threads"
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": "MLUPS", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "C3 urban 400x400x100 (BASELINE.json configs[2]); reference arm runs a bounded crop", "sample": sample},
            "cpu_baseline": {"value": v, "unit": "MLUPS", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": "MLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the LBM path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    from paper_2607_04516_b200 import binding, build, workloads as W
    build.build()
    K, Wm = args.steps, max(args.warmup, 3)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---------------- device-resident timing: K launches of the fused kernel
    job_ = Job(args.workload, binding, W, f"cuda:{local}")
    sim, wl = job_.sims[-1], job_.wls[-1]   # the (main) lattice whose macros are read back
    cells = job_.cells
    if args.variant:
        for s_ in job_.sims:
            s_.set_variant(args.variant)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        sampler.wait_first_sample()   # sampling (every 20 ms) runs through warm-up and the timed region
    t_load0 = sampler.mark()          # the clock record covers warm-up + timed region (the latter alone can be a few ms)
    job_.step(Wm)
    barrier()
    l0 = job_.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps = max(1, args.repeats)
    best = None
    for _ in range(reps):
        barrier()
        e0.record()
        job_.step(K)
        e1.record()
        barrier()
        ms = e0.elapsed_time(e1)
        best = ms if best is None else min(best, ms)
    launches = (job_.launch_count() - l0) // reps
    clocks = sampler.stop(t_load0, sampler.mark()) if rank == 0 else None
    # second region: the same step back to back for >= SUSTAINED_SECONDS, where the board sits at its power cap (the K-step
    # region above can be a burst at boost clock when the driver asks for few steps)
    sustained = None
    if not args.no_sustained:
        ks = max(K, int(SUSTAINED_SECONDS * 1e3 / max(best / K, 1e-6)) + 1)
        s2 = ClockSampler(local)
        if rank == 0:
            s2.start()
            s2.wait_first_sample()
        barrier()
        t_s0 = s2.mark()
        e0.record()
        job_.step(ks)
        e1.record()
        barrier()
        ms_s = max_over_ranks(e0.elapsed_time(e1), world, dev)
        sustained = {"value": job_mlups(cells, ks, world, ms_s * 1e-3), "unit": "MLUPS", "steps": ks, "ms_per_step": ms_s / ks,
                     "clocks": s2.stop(t_s0, s2.mark()) if rank == 0 else None}
    rho, ux, uy, uz = sim.get_macros()
    finite = bool(torch.isfinite(ux).all().item())
    if not finite and rank == 0:   # a timing on a state that has blown up is not a measurement of this workload
        print("bench.py: WARNING: the state is not finite after the timed regions (config.state_finite = false)", file=sys.stderr)
    ms_total = max_over_ranks(best, world, dev)
    mlups = job_mlups(cells, K, world, ms_total * 1e-3)

    # ---------------- end to end through the C ABI with pinned host buffers
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()  # noqa: E731
    host = job_.host_inputs(pin)
    outs = [torch.empty(wl.shape, dtype=torch.float32).pin_memory() for _ in range(4)]
    lib = binding.load_library()

    def job(s):
        job_.setup_from_host(host)
        job_.step(K)
        rc = lib.lbm_get_macros(s._h, *[o.data_ptr() for o in outs])
        assert rc == 0
    job(sim)  # warm-up of the copy paths
    e2e_s = None
    for _ in range(2):  # best of two whole jobs (a first pass after start-up has been seen to stall in the driver)
        barrier()
        t0 = time.perf_counter()
        e0.record()
        job(sim)
        e1.record()
        barrier()
        wall = time.perf_counter() - t0
        t_job = max_over_ranks(max(e0.elapsed_time(e1) * 1e-3, wall), world, dev)
        e2e_s = t_job if e2e_s is None else min(e2e_s, t_job)
    h2d = Job.nbytes(host) + sum(t.nbytes for t in getattr(job_, "theta_host", []) if t is not None)  # + the thermal field
    d2h = sum(o.numel() * 4 for o in outs)
    e2e = {"value": job_mlups(cells, K, world, e2e_s), "unit": "MLUPS", "h2d_bytes_per_step": h2d / K,
           "d2h_bytes_per_step": d2h / K,
           "what": f"one job = set_flags + set_inlet_profile + set_macros{' + set_theta' if args.workload.startswith('thermal') else ''} from pinned host buffers, lbm_step({K}), "
                   "lbm_get_macros into pinned host buffers; best of 2 jobs"}

    if rank == 0:
        peak, peak_src = load_peak()
        per_launch_s = ms_total * 1e-3 / K
        # thermal workload: (19 + 7) x 4 B loads + (19 + 7) x 4 B stores + 1 flag byte (lbm_thermal.cuh)
        # 16-bit storage: 19 x 2 B loads + 19 x 2 B stores + 1 flag byte
        BYTES_PER_CELL = {"thermal": 209, "thermal-inplace": 209, "c3-fp16": 77, "c3-fp16-inplace": 77}.get(args.workload, globals()["BYTES_PER_CELL"])
        achieved = BYTES_PER_CELL * cells / per_launch_s / 1e9
        traffic, traffic_src = (load_traffic("step") if args.workload == "c3" else
                                load_traffic("thermal") if args.workload == "thermal" else
                                load_traffic("s16") if args.workload == "c3-fp16" else
                                load_traffic("inplace") if args.workload == "c3-inplace" else (None, None))
        if traffic_src:
            traffic_src += " (committed ncu --set full capture; a constant, not measured in this run)"
        if sustained is not None:
            sustained["achieved"] = BYTES_PER_CELL * cells / (sustained["ms_per_step"] * 1e-3) / 1e9
            sustained["frac"] = sustained["achieved"] / peak
        line = {
            "metric": metric_for(args.workload), "value": mlups, "unit": "MLUPS", "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32 arithmetic, f16 storage" if "fp16" in args.workload else "f32", "data": "synthetic",
            "config": {"workload": WORKLOADS[args.workload],
                       "cells": cells, "parallelism": "replicas only" if world > 1 else "single GPU",
                       "l2": (f"no flush needed: each step streams {BYTES_PER_CELL * cells / 1e9:.1f} GB (>> 126 MB L2)"
                              if BYTES_PER_CELL * cells > 4 * 126e6 else
                              f"NOT flushed: the {2 * 76 * cells / 1e6:.0f} MB of this parity config stay L2-resident; not a bench line"),
                       "best_of": reps, "variant": int(args.variant), "workspace_bytes": int(job_.workspace_bytes),
                       "state_finite": finite},
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                         "algorithmic_bytes_per_launch": BYTES_PER_CELL * cells,
                         "frac_of_nominal_8000": achieved / 8000.0},
            "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks, "sustained": sustained,
        }
        if not args.no_cpu_baseline and world == 1 and args.workload == "c3":
            line["cpu_baseline"] = cpu_baseline()
        else:
            line["cpu_baseline"] = None
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=400)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--repeats", type=int, default=1, help="timed repetitions of the K-step region; best is reported")
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--workload", default="c3", choices=sorted(WORKLOADS), help="c3 = the headline config; others: per-config table only")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sustained", action="store_true", help="skip the second (>= 2 s, back-to-back) timed region")
    ap.add_argument("--reference-budget", type=float, default=150.0, help="seconds of CPU time the reference arm may use")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())

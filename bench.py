#!/usr/bin/env python
"""bench.py -- MLUPS of the fused moments-only lattice update on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]
                    [--n 512] [--dtype f32] [--lattice 27] [--ncomp 1] [--scheme moments] [--kernel auto]

One "step" = one lattice time step (the whole hot path: gather, reconstruct, BGK collide, stream,
project, store -- SURVEY.md 8(a) a0-a7) over the whole periodic box.  Default workload: BASELINE.json
config 5 instance D3Q27, single component, fp32, 512^3, seeded as config 1 (Taylor-Green), the larger of
the two grid sizes the north star's target is stated on; both state buffers (2 x 5.4 GB) are far larger
than L2, so no flush is needed between steps.  Prints ONE JSON line on stdout (rank 0).

N > 1: the box is not decomposed in this round ("replicas only"): every rank advances its
own box; value = all ranks' node updates / max-over-ranks device time; scaling = weak.
--impl reference: times the CPU oracle (oracle/, plain C fp64) on a bounded sample of the workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "MLUPS"
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=512)
    ap.add_argument("--dtype", default="f32", choices=["f32", "f64"])
    ap.add_argument("--lattice", type=int, default=27, choices=[19, 27])
    ap.add_argument("--ncomp", type=int, default=1, choices=[1, 2])
    ap.add_argument("--scheme", default="moments", choices=["moments", "populations"])
    ap.add_argument("--kernel", default="auto", choices=["auto", "gather", "march", "tma", "tma_split"])
    ap.add_argument("--e2e-steps", type=int, default=2, help="host-buffer steps timed for the e2e key (0 = skip)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def workload_name(a):
    return (f"config5 sweep instance: D3Q{a.lattice} {'single' if a.ncomp == 1 else 'two'}-component "
            f"{a.scheme} {a.dtype} {a.n}^3 periodic, seeded as config 1 (Taylor-Green, tau="
            f"{'0.8' if a.ncomp == 1 else '1.0'})")


def algorithmic_bytes_per_lu(a):
    """2*M*sizeof for the moments scheme, 2*ncomp*Q*sizeof with populations."""
    size = 4 if a.dtype == "f32" else 8
    if a.scheme == "moments":
        return 2 * (10 if a.ncomp == 1 else 11) * size
    return 2 * a.ncomp * a.lattice * size


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy bandwidth)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md, 6.65 TB/s)"


def ncu_traffic(kernel_name, n):
    """dram read+write bytes per launch from the committed ncu capture (profiles/ncu_traffic.csv), or None."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    try:
        with open(p) as f:
            for line in f:
                parts = [s.strip() for s in line.split(",")]
                if len(parts) >= 4 and parts[0] == kernel_name and parts[1] == str(n):
                    return float(parts[2]) + float(parts[3])
    except Exception:
        pass
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc = index, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except Exception:
            self.proc.kill()
            out = ""
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [s.strip() for s in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def time_oracle(a, seconds_target=20.0):
    """The oracle as it stands on the host cores: bounded sample of the workload's recipe."""
    import oracle
    from paper_2301_01622_b200 import workloads as wl

    oracle.build()
    n = min(a.n, 96)
    cfg = wl.sweep_case(n, a.lattice, a.ncomp, "f64")
    m = cfg["moments"]
    fn = oracle.pop_run if a.scheme == "populations" else oracle.run
    kw = dict(lattice=a.lattice, ncomp=a.ncomp, tau=cfg["tau"], A=cfg["A"], beta=cfg["beta"])
    t0 = time.perf_counter()
    fn(m, nsteps=1, **kw)
    t1 = time.perf_counter() - t0
    steps = int(max(1, min(1000, seconds_target / max(t1, 1e-3))))
    t0 = time.perf_counter()
    fn(m, nsteps=steps, **kw)
    dt = time.perf_counter() - t0
    return {"value": n ** 3 * steps / dt / 1e6, "unit": METRIC, "cores": oracle.threads(), "kind": "oracle",
            "sample": f"{n}^3 box of the same recipe, {steps} steps, fp64, {dt:.1f} s of host time"}, dt / steps, steps, n


def run_reference(a):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    a.steps = max(1, a.steps)
    base, _, _, n = time_oracle(a, seconds_target=min(60.0, 3.0 * (a.steps + a.warmup)))
    line = {"impl": "reference", "metric": METRIC, "value": base["value"], "unit": METRIC, "n_gpus": a.gpus,
            "steps": a.steps, "warmup": a.warmup, "ms_per_step": 1e3 * n ** 3 / (base["value"] * 1e6),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": workload_name(a), "sample": base["sample"]},
            "cpu_baseline": base, "gpu_launches": 0,
            "e2e": {"value": base["value"], "unit": METRIC, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def max_over_ranks(x, world, device="cpu"):
    """MAX all-reduce of one float over the ranks (nccl on the GPU box, gloo in the CPU test)."""
    if world == 1:
        return float(x)
    import torch
    import torch.distributed as dist

    t = torch.tensor([x], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate(per_rank_nodes_steps, max_ms):
    """value over all ranks: total node updates / max-over-ranks time (host logic; gloo-tested)."""
    return sum(per_rank_nodes_steps) / (max_ms * 1e-3) / 1e6


def main():
    a = parse_args()
    if a.impl == "reference":
        return run_reference(a)

    import torch
    import torch.distributed as dist

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    from paper_2301_01622_b200 import build as lbuild
    from paper_2301_01622_b200 import lbwp
    from paper_2301_01622_b200 import workloads as wl

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        lbuild.build()
    if world > 1:
        dist.barrier()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = wl.sweep_case(a.n, a.lattice, a.ncomp, a.dtype)
    m0 = wl.as_dtype(cfg["moments"], a.dtype)
    nodes = a.n ** 3
    sim = lbwp.Lbwp(m0, lattice=a.lattice, dtype=a.dtype, ncomp=a.ncomp, tau=cfg["tau"], A=cfg["A"],
                    beta=cfg["beta"], scheme=a.scheme, kernel=a.kernel, device=local)
    kname = sim.kernel_name
    sim.step(max(3, a.warmup))
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.1)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    sim.step(a.steps)          # exactly K steps, K * launches_per_step kernel launches
    ev1.record()
    barrier()
    clocks = sampler.stop()
    ms = ev0.elapsed_time(ev1)
    ms = max_over_ranks(ms, world, "cuda")
    value = aggregate([nodes * a.steps] * world, ms)

    # end-to-end through the C ABI with HOST buffers: every step uploads the state from pinned host
    # memory, advances one time step, and reads the new moments back to pinned host memory.
    e2e = None
    if a.e2e_steps > 0:
        tdt = torch.float32 if a.dtype == "f32" else torch.float64
        h_in = torch.from_numpy(m0).pin_memory()
        h_out = torch.empty(h_in.shape, dtype=tdt).pin_memory()
        sim.set_moments(h_in)
        sim.step(1)
        sim.moments_host(out=h_out)
        barrier()
        t0 = time.perf_counter()
        for _ in range(a.e2e_steps):
            sim.set_moments(h_in)
            sim.step(1)
            sim.moments_host(out=h_out)     # synchronises
            h_in, h_out = h_out, h_in
        barrier()
        dt = time.perf_counter() - t0
        dt = max_over_ranks(dt, world, "cuda")
        nbytes = h_in.numel() * h_in.element_size()
        e2e = {"value": nodes * a.e2e_steps * world / dt / 1e6, "unit": METRIC, "h2d_bytes_per_step": nbytes,
               "d2h_bytes_per_step": nbytes, "steps": a.e2e_steps,
               "what": "lbwp_set_moments(host) + lbwp_step(1) + lbwp_moments(host) per step, pinned host buffers"}
        del h_in, h_out
    lps = sim.launches_per_step
    state_bytes = sim.state_bytes
    sim.close()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    peak, peak_src = measured_peak()
    bpl = algorithmic_bytes_per_lu(a)
    launch_ms = ms / a.steps            # one dominant kernel launch per step
    achieved = bpl * nodes / (launch_ms * 1e-3) / 1e9
    traffic = ncu_traffic(kname, a.n)
    line = {
        "metric": METRIC, "value": value, "unit": METRIC, "n_gpus": world, "steps": a.steps, "warmup": max(3, a.warmup),
        "ms_per_step": ms / a.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": a.dtype, "data": "synthetic",
        "config": {"workload": workload_name(a), "kernel": kname, "grid": [a.n] * 3, "l2": "state 2 x %.2f GB >> 126 MB L2, no flush needed" % (state_bytes / 1e9) if state_bytes > 4e8 else "state partly L2-resident (reported as is)",
                   "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "bytes_per_node_state": state_bytes * 2 / nodes},
        "clocks": clocks,
        "e2e": e2e,
        "gpu_launches": a.steps * lps,
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": traffic, "peak_source": peak_src, "algorithmic_bytes_per_node": bpl,
                     "frac_of_8TBs_nominal": achieved / 8000.0, "kernel": kname,
                     "launch_ms": launch_ms},
    }
    if not a.no_cpu_baseline and world == 1:
        base, _, _, _ = time_oracle(a)
        line["cpu_baseline"] = base
    elif not a.no_cpu_baseline:
        line["cpu_baseline"] = None
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

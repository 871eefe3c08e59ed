#!/usr/bin/env python
"""bench.py -- MLUPS of the fused moments-only lattice update on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]
                    [--n 512] [--dtype f32] [--lattice 27] [--ncomp 1] [--scheme moments] [--kernel auto]

One "step" = one lattice time step (the whole hot path: gather, reconstruct, BGK collide, stream,
project, store -- SURVEY.md 8(a) a0-a7) over the whole periodic box.  Default workload: BASELINE.json
config 5 instance D3Q27, single component, fp32, 512^3, seeded as config 1 (Taylor-Green), the larger of
the two grid sizes the north star's target is stated on; both state buffers (2 x 5.4 GB) are far larger
than L2, so no flush is needed between steps.  Prints ONE JSON line on stdout (rank 0).

The same line carries `sizes` (256^3 and 512^3, fp32 and fp64: MLUPS and the HBM fraction at each, as the north star
asks), `footprint` (bytes per node and total GB with and without populations, from lbwp_state_bytes of both
schemes), `two_component` (the paper's own workload class: two-component fp32 at 128^3, 256^3 and
512^3, with the near-contact force off and on) and `cpu_baseline` (the oracle on the host cores: all cores and single
thread, 128^3).

N > 1 (`--gpus N` under torchrun): ONE periodic box of n x n x (n N) nodes, decomposed into z slabs of n planes per
rank (weak scaling), halo planes exchanged with the z neighbours after every step (NCCL send/recv; slabs.py);
value = all owned node updates / max-over-ranks device time.  (The population scheme runs as replicas.)
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
    ap.add_argument("--near-contact", type=float, default=0.0, metavar="A_h",
                    help="two-component runs: strength of the near-contact repulsion (PAPER.md:93-112, Eq. 10; h_c = 4); "
                         "0 = off.  The paper's own benchmark (PAPER.md:158-163) is --n 128 --lattice 19 --ncomp 2 with it on")
    ap.add_argument("--e2e-steps", type=int, default=2, help="host-buffer steps timed for the e2e key (0 = skip)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sizes", action="store_true", help="skip the 256^3 / 512^3 fp32 / fp64 sub-record")
    ap.add_argument("--size-steps", type=int, default=50, help="timed steps per entry of the sizes sub-record")
    ap.add_argument("--no-two-component", action="store_true",
                    help="skip the two_component sub-record (128^3 / 256^3 / 512^3 fp32, with and without the near-contact force)")
    return ap.parse_args()


def workload_name(a):
    return (f"config5 sweep instance: D3Q{a.lattice} {'single' if a.ncomp == 1 else 'two'}-component "
            f"{a.scheme} {a.dtype} {a.n}^3 periodic, seeded as config 1 (Taylor-Green, tau="
            f"{'0.8' if a.ncomp == 1 else '1.0'})"
            + (f", near-contact force A_h={a.near_contact:g}, h_c=4" if a.ncomp == 2 and a.near_contact else ""))


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
    """dram read+write bytes per launch of this kernel at this size from the COMMITTED ncu --set full capture
    (profiles/ncu_traffic.csv; its .md names the command and commit), or None.  Not measured in this run: ncu
    cannot run inside a timed benchmark."""
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


def time_oracle(a, seconds_target=15.0, n=None, threads=None):
    """The oracle as it stands on the host cores: a bounded sample of the workload's recipe (BASELINE.md section 3:
    128^3; `threads` = None uses every core)."""
    import oracle
    from paper_2301_01622_b200 import workloads as wl

    oracle.build()
    n = min(a.n, n or 128)
    cfg = wl.sweep_case(n, a.lattice, a.ncomp, "f64")
    m = cfg["moments"]
    fn = oracle.pop_run if a.scheme == "populations" else oracle.run
    kw = dict(lattice=a.lattice, ncomp=a.ncomp, tau=cfg["tau"], A=cfg["A"], beta=cfg["beta"])
    all_cores = oracle.set_threads(os.cpu_count() or 1)
    used = oracle.set_threads(threads) if threads else all_cores
    try:
        t0 = time.perf_counter()
        fn(m, nsteps=1, **kw)
        t1 = time.perf_counter() - t0
        steps = int(max(1, min(1000, seconds_target / max(t1, 1e-3))))
        t0 = time.perf_counter()
        fn(m, nsteps=steps, **kw)
        dt = time.perf_counter() - t0
    finally:
        oracle.set_threads(all_cores)
    return {"value": n ** 3 * steps / dt / 1e6, "unit": METRIC, "cores": used, "kind": "oracle",
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


def time_steps(torch, sim, steps, warmup, barrier):
    """W untimed steps, then exactly `steps` steps between two CUDA events on the launching stream."""
    sim.step(max(3, warmup))
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    sim.step(steps)
    ev1.record()
    barrier()
    return ev0.elapsed_time(ev1)


def roofline_record(a_like, kname, nodes, ms, steps, lps, peak, peak_src):
    """HBM roofline of one time step: algorithmic bytes (2 M sizeof per node) / measured step time.
    A step is `lps` launches (1 for every moments kernel of the TMA path); launch_ms is the average launch."""
    bpl = algorithmic_bytes_per_lu(a_like)
    step_ms = ms / steps
    achieved = bpl * nodes / (step_ms * 1e-3) / 1e9
    return {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
            "traffic": ncu_traffic(kname, a_like.n),
            "traffic_source": "committed ncu --set full capture, profiles/ncu_traffic.csv (not measured in this run)",
            "peak_source": peak_src, "algorithmic_bytes_per_node": bpl, "frac_of_8TBs_nominal": achieved / 8000.0,
            "kernel": kname, "launches_per_step": lps, "step_ms": step_ms, "launch_ms": step_ms / lps}


def main():
    a = parse_args()
    if a.impl == "reference":
        return run_reference(a)

    import copy

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

    def make_sim(b):
        cfg = wl.sweep_case(b.n, b.lattice, b.ncomp, b.dtype)
        m0 = wl.as_dtype(cfg["moments"], b.dtype)
        return lbwp.Lbwp(m0, lattice=b.lattice, dtype=b.dtype, ncomp=b.ncomp, tau=cfg["tau"], A=cfg["A"],
                         beta=cfg["beta"], scheme=b.scheme, kernel=b.kernel, device=local,
                         A_h=getattr(b, "near_contact", 0.0) if b.ncomp == 2 else 0.0), m0

    peak, peak_src = measured_peak()
    nodes = a.n ** 3
    slab = None
    if world > 1 and a.scheme == "moments":
        # one periodic box of n x n x (n * world) nodes, z-slab decomposed: every rank owns n planes (weak scaling) and
        # exchanges halo planes with its z neighbours after every step (paper_2301_01622_b200/slabs.py).  The global
        # field is the n^3 recipe repeated along z, so each rank's halo-extended slab is cut from its own copy.
        from paper_2301_01622_b200 import slabs
        cfg = wl.sweep_case(a.n, a.lattice, a.ncomp, a.dtype)
        A_h = a.near_contact if a.ncomp == 2 else 0.0
        halo = slabs.halo_width(a.ncomp, A_h)
        m0 = wl.as_dtype(cfg["moments"], a.dtype)
        m0 = np.ascontiguousarray(m0[:, np.arange(-halo, a.n + halo) % a.n])
        slab = slabs.SlabLbwp(m0, world=world, rank=rank, lattice=a.lattice, dtype=a.dtype, ncomp=a.ncomp, tau=cfg["tau"],
                              A=cfg["A"], beta=cfg["beta"], kernel=a.kernel, device=local, A_h=A_h)
        sim = slab.sim
        stepper = slab
    else:
        sim, m0 = make_sim(a)
        stepper = sim
    kname, lps, state_bytes = sim.kernel_name, sim.launches_per_step, sim.state_bytes
    stepper.step(max(3, a.warmup))
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.1)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    stepper.step(a.steps)      # exactly K steps: K * launches_per_step kernel launches (N > 1: plus the halo exchange)
    ev1.record()
    barrier()
    clocks = sampler.stop()
    ms = max_over_ranks(ev0.elapsed_time(ev1), world, "cuda")
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
        dt = max_over_ranks(time.perf_counter() - t0, world, "cuda")
        nbytes = h_in.numel() * h_in.element_size()
        e2e = {"value": m0.shape[1] * a.n * a.n * a.e2e_steps * world / dt / 1e6, "unit": METRIC, "h2d_bytes_per_step": nbytes,
               "d2h_bytes_per_step": nbytes, "steps": a.e2e_steps,
               "what": "lbwp_set_moments(host) + lbwp_step(1) + lbwp_moments(host) per step, pinned host buffers"}
        del h_in, h_out
    sim.close()
    del sim, m0

    # the other sizes and precisions the north star names (rank 0, 1 GPU): same kernel path, fewer steps
    sizes = None
    if not a.no_sizes and world == 1 and a.scheme == "moments":
        sizes = []
        for n, dt in ((256, "f32"), (512, "f32"), (256, "f64"), (512, "f64")):
            b = copy.copy(a)
            b.n, b.dtype = n, dt
            if (n, dt) == (a.n, a.dtype):
                r = roofline_record(b, kname, nodes, ms, a.steps, lps, peak, peak_src)
                steps = a.steps
            else:
                s2, _ = make_sim(b)
                t = time_steps(torch, s2, a.size_steps, 5, barrier)
                r = roofline_record(b, s2.kernel_name, n ** 3, t, a.size_steps, s2.launches_per_step, peak, peak_src)
                steps = a.size_steps
                s2.close()
                del s2
            sizes.append({"grid": n, "dtype": dt, "kernel": r["kernel"], "steps": steps,
                          "mlups": r["algorithmic_bytes_per_node"] and r["achieved"] * 1e9 / r["algorithmic_bytes_per_node"] / 1e6,
                          "achieved_gbs": r["achieved"], "frac": r["frac"], "frac_of_8TBs_nominal": r["frac_of_8TBs_nominal"]})

    # the paper's own workload class (two-component D3Q19 fp32 with near-contact forces at 128^3), and the
    # same at the north star's sizes: the config-5 two-component recipe, with the force off and on (A_h = 0.02, h_c = 4)
    two_component = None
    if not a.no_two_component and not a.no_sizes and world == 1 and a.scheme == "moments" and a.ncomp == 1 and a.dtype == "f32":
        two_component = []
        for n, lattices in ((128, (19,)), (256, (19,)), (512, (19, 27))):
            cfg = wl.sweep_case(n, 19, 2, "f32")          # the recipe does not depend on the lattice
            m2 = wl.as_dtype(cfg["moments"], "f32")
            for lat in lattices:
                for A_h in (0.0, 0.02):
                    b = copy.copy(a)
                    b.n, b.lattice, b.ncomp, b.dtype = n, lat, 2, "f32"
                    s2 = lbwp.Lbwp(m2, lattice=lat, dtype="f32", ncomp=2, tau=cfg["tau"], A=cfg["A"], beta=cfg["beta"],
                                   kernel=a.kernel, device=local, A_h=A_h)
                    nst = a.size_steps * (4 if n == 128 else 1)
                    t = time_steps(torch, s2, nst, 5, barrier)
                    r = roofline_record(b, s2.kernel_name, n ** 3, t, nst, s2.launches_per_step, peak, peak_src)
                    two_component.append({"grid": n, "lattice": lat, "dtype": "f32", "near_contact_A_h": A_h, "kernel": r["kernel"],
                                          "launches_per_step": r["launches_per_step"], "steps": nst, "step_ms": r["step_ms"],
                                          "mlups": n ** 3 / (r["step_ms"] * 1e-3) / 1e6, "achieved_gbs": r["achieved"],
                                          "frac": r["frac"], "algorithmic_bytes_per_node": r["algorithmic_bytes_per_node"]})
                    s2.close()
                    del s2
            del m2, cfg

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # memory footprint with and without populations: what the library allocates for the state
    def fp(scheme, ncomp):
        p = lbwp.make_params(lattice=a.lattice, dtype=a.dtype, ncomp=ncomp, shape=(a.n,) * 3, tau=1.0, A=0.01, beta=0.7,
                             scheme=scheme)
        b = 2 * lbwp.state_bytes(p)          # two ping-pong buffers
        return {"bytes_per_node": b / nodes, "total_gb": b / 1e9}
    esz = 4 if a.dtype == "f32" else 8
    footprint = {"grid": a.n, "dtype": a.dtype, "lattice": a.lattice,
                 "moments_1c": fp("moments", 1), "moments_2c": fp("moments", 2),
                 "populations_1c": fp("populations", 1), "populations_2c": fp("populations", 2),
                 "ideal_bytes_per_node": {"moments_1c": 20 * esz, "moments_2c": 22 * esz,
                                          "populations_1c": 2 * a.lattice * esz, "populations_2c": 4 * a.lattice * esz},
                 "paper": "V100, 128^3, two-component D3Q19 fp32: 0.6782 GB without / 1.1411 GB with populations (PAPER.md:163)"}

    line = {
        "metric": METRIC, "value": value, "unit": METRIC, "n_gpus": world, "steps": a.steps, "warmup": max(3, a.warmup),
        "ms_per_step": ms / a.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": a.dtype, "data": "synthetic",
        "config": {"workload": workload_name(a), "kernel": kname, "grid": [a.n] * 3, "l2": "state 2 x %.2f GB >> 126 MB L2, no flush needed" % (state_bytes / 1e9) if state_bytes > 4e8 else "state partly L2-resident (reported as is)",
                   "parallelism": ("z-slabs of one %d x %d x %d box, %d-plane halo exchange per step (NCCL send/recv)" % (a.n, a.n, a.n * world, slab.halo)
                                   if slab is not None else "replicas only" if world > 1 else "1 GPU"),
                   "bytes_per_node_state": state_bytes * 2 / nodes},
        "clocks": clocks,
        "e2e": e2e,
        "gpu_launches": a.steps * lps,
        "roofline": roofline_record(a, kname, nodes, ms, a.steps, lps, peak, peak_src),
        "sizes": sizes,
        "two_component": two_component,
        "footprint": footprint,
        "paper_context": "622 MLUPS without / 277 MLUPS with populations: V100 16 GB, 128^3, two-component D3Q19, fp32, with near-contact forces (PAPER.md:158-163); another machine and workload, not the target",
    }
    if not a.no_cpu_baseline and world == 1:
        base, _, _, _ = time_oracle(a, seconds_target=12.0)
        single, _, _, _ = time_oracle(a, seconds_target=8.0, threads=1)
        base["single_thread"] = {"value": single["value"], "unit": METRIC, "cores": 1, "sample": single["sample"]}
        line["cpu_baseline"] = base
    elif not a.no_cpu_baseline:
        line["cpu_baseline"] = None
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

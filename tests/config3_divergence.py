#!/usr/bin/env python
"""How far does an fp32 evaluation of config 3 leave the fp64 trajectory, and is that the kernel's doing?

Reproduces profiles/r02_config3_divergence.md.  Four trajectories of BASELINE config 3 (128^3 head-on droplet
collision, tau = 1, A = 0.01, beta = 0.7) from the same fp32-representable initial state:
    O64   the oracle (fp64 state, fp64 arithmetic): the reference trajectory
    O32s  DIAGNOSTIC ONLY, never a checker: the oracle's own step in fp64 arithmetic with its STATE rounded to fp32
          after every step -- the most faithful evaluation any implementation with an fp32 state can be
    K32   the CUDA kernel, fp32
    K64   the CUDA kernel, fp64
and prints, at each checkpoint, BASELINE's error norm (max over the moment fields of max|a - b| / max|b|) and the
sign(phi) agreement of O32s, K32, K64 against O64, and of K32 against O32s.
    python tests/config3_divergence.py [--n 128] [--out gpurun_out/config3_divergence.md]      (about 15 min of host time)
"""
import argparse
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))
import oracle  # noqa: E402
import oracle_trajectories as traj  # noqa: E402
from parity_norms import moment_field_errors, sign_agreement  # noqa: E402
from paper_2301_01622_b200 import lbwp  # noqa: E402
from paper_2301_01622_b200 import workloads as wl  # noqa: E402

TIMES = (50, 100, 150, 200, 300, 400, 800, 1200, 1600, 2000)


def kernel_trajectory(cfg, m0, dtype, times):
    out, t_now = {}, 0
    with lbwp.Lbwp(wl.as_dtype(m0, dtype), lattice=cfg["lattice"], dtype=dtype, ncomp=2, tau=cfg["tau"], A=cfg["A"],
                   beta=cfg["beta"]) as sim:
        for t in times:
            sim.step(t - t_now)
            t_now = t
            out[t] = sim.moments_host().astype(np.float64)
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=128)
    ap.add_argument("--out", default=os.path.join(ROOT, "gpurun_out", "config3_divergence.md"))
    a = ap.parse_args()
    oracle.build()
    cfg = wl.config3(a.n)
    times = tuple(int(t * a.n / 128) for t in TIMES)
    m0 = wl.as_dtype(cfg["moments"], "f32")
    o64 = traj.trajectory(oracle, cfg, times, m0=m0.astype(np.float64))
    o32 = traj.fp32_state_trajectory(oracle, cfg, times, m0=m0)
    k32 = kernel_trajectory(cfg, m0, "f32", times)
    k64 = kernel_trajectory(cfg, m0, "f64", times)

    def cell(x, ref):
        return "%.1e / %.5f" % (moment_field_errors(x, ref, 2).max(), sign_agreement(x, ref))

    lines = ["| t | O32s vs O64 | K32 vs O64 | K64 vs O64 | K32 vs O32s |", "|---|---|---|---|---|"]
    for t in times:
        lines.append("| %d | %s | %s | %s | %s |" % (t, cell(o32[t], o64[t]), cell(k32[t], o64[t]), cell(k64[t], o64[t]),
                                                    cell(k32[t], o32[t])))
    text = "\n".join(lines) + "\n"
    os.makedirs(os.path.dirname(a.out), exist_ok=True)
    with open(a.out, "w") as f:
        f.write("config 3 at %d^3: max relative error per moment field / sign(phi) agreement\n\n" % a.n + text)
    print(text)


if __name__ == "__main__":
    main()

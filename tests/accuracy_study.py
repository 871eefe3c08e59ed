#!/usr/bin/env python
"""With / without populations accuracy study (Fig. 2, 3, 5, 7) on the GPU.

Runs BASELINE configs 3 (128^3 head-on) and 4 (256^3 off-axis) with scheme = MOMENTS (the paper's method, index N in
its figures) and scheme = POPULATIONS (standard colour-gradient LB with stored populations, index P) side by side,
same initial moments, and reports at the listed times the paper's two diagnostics through lbwp_diagnostics:
    <rho>_{rho > 0.5}(t)   for both schemes (Fig. 2, 5, 7)                 rho = density of the droplet component
    |rho_N - rho_P| / rho_N,MAX  at probe sites (32,64,64), (64,64,64) of the 128^3 box (Fig. 3; scaled by 2 for 256^3)
plus the largest such difference over the whole box.  BASELINE's configs run at tau = 1, where the two schemes are the
same map, so the study also runs them at tau = 0.8, where they differ.
No near-contact force (C14): the drops coalesce as in the paper's Fig. 6-7 case (A_h = 0).

    python tests/accuracy_study.py [--out profiles/r02_accuracy_study.md] [--dtype f64]
Needs a B200; uses the product path only (both schemes are parity-tested against their oracles in tests/)."""
import argparse
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from paper_2301_01622_b200 import lbwp  # noqa: E402
from paper_2301_01622_b200 import workloads as wl  # noqa: E402


def study(cfg, tau, times, probes, dtype):
    m0 = wl.as_dtype(cfg["moments"], dtype)
    kw = dict(lattice=cfg["lattice"], dtype=dtype, ncomp=2, tau=tau, A=cfg["A"], beta=cfg["beta"])
    rows = []
    with lbwp.Lbwp(m0, scheme="moments", **kw) as sn, lbwp.Lbwp(m0, scheme="populations", **kw) as sp:
        t_now = 0
        for t in times:
            sn.step(t - t_now)
            sp.step(t - t_now)
            t_now = t
            dn, dp = sn.diagnostics(0.5, probes), sp.diagnostics(0.5, probes)
            rn, rp = sn.moments()[0], sp.moments()[0]           # droplet-component density fields, on the device
            whole = float((rn - rp).abs().max().item()) / dn["rho_max"]
            rows.append((t, dn["rho_mean_above"], dp["rho_mean_above"],
                         [abs(a - b) / dn["rho_max"] for a, b in zip(dn["probe_rho"], dp["probe_rho"])], whole,
                         dn["count_above"], dp["count_above"], dn["mass"][0], dp["mass"][0]))
    return rows


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=os.path.join(ROOT, "gpurun_out", "accuracy_study.md"))
    ap.add_argument("--dtype", default="f32")
    a = ap.parse_args()
    out = ["# Moments-only (N) against population-storing (P) colour-gradient LB: the paper's diagnostics",
           "",
           "Written by `python tests/accuracy_study.py --dtype %s` on a B200 (product path, both schemes through the C ABI;" % a.dtype,
           "`lbwp_diagnostics` for the reductions).  rho = density of the droplet component (PAPER.md:118).",
           "Columns: <rho>_{rho>0.5} of N and P (PAPER.md:126, Fig. 2/5/7); |rho_N - rho_P| / rho_N,MAX at the paper's probe",
           "sites (PAPER.md:134, Fig. 3) and its maximum over the whole box; nodes with rho > 0.5; mass of the droplet fluid.",
           ""]
    cases = [("config 3 (128^3, head-on, U = +-0.05)", wl.config3(128), [(32, 64, 64), (64, 64, 64)],
              (0, 100, 200, 400, 800, 1200, 1600, 2000)),
             ("config 4 (256^3, off-axis, U = +-0.04)", wl.config4(256), [(64, 128, 128), (128, 128, 128)],
              (0, 200, 400, 800, 1600, 2400, 3200, 4000))]
    for name, cfg, probes, times in cases:
        for tau in (1.0, 0.8):
            rows = study(cfg, tau, times, probes, a.dtype)
            out += ["## %s, tau = %.1f, %s" % (name, tau, a.dtype), "",
                    "| t | <rho>_N | <rho>_P | probe %s | probe %s | max over box | nodes N | nodes P | mass N | mass P |" % (probes[0], probes[1]),
                    "|---|---|---|---|---|---|---|---|---|---|"]
            for t, mn, mp, pr, whole, cn, cp, man, map_ in rows:
                out.append("| %d | %.6f | %.6f | %.2e | %.2e | %.2e | %d | %d | %.3f | %.3f |" % (t, mn, mp, pr[0], pr[1], whole, cn, cp, man, map_))
            out.append("")
    text = "\n".join(out) + "\n"
    os.makedirs(os.path.dirname(a.out), exist_ok=True)
    with open(a.out, "w") as f:
        f.write(text)
    print(text)


if __name__ == "__main__":
    main()

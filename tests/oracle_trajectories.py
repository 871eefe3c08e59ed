"""Oracle trajectories with checkpoints for the long droplet configurations (test infrastructure).

Every state here is produced by `oracle/` alone from the seeded recipes of `workloads.py`; nothing comes from
the CUDA path.  Used by tests/test_gpu_parity_long.py (windowed parity through the coalescence, PAPER.md:126,
144, 154: the physically interesting windows are t ~ 1e2 .. 6e3) and by tests/config3_divergence.py.
"""
from __future__ import annotations

import numpy as np


def trajectory(oracle, cfg, times, m0=None):
    """Advance cfg's initial moments with the fp64 oracle and return {t: state at step t} for t in `times`
    (sorted, t = 0 allowed).  `m0` overrides the initial state (e.g. the fp32-rounded recipe output)."""
    m = np.array(cfg["moments"] if m0 is None else m0, dtype=np.float64)
    kw = dict(lattice=cfg["lattice"], ncomp=cfg["ncomp"], tau=cfg["tau"], A=cfg["A"], beta=cfg["beta"])
    out, t_now = {}, 0
    for t in sorted(times):
        if t > t_now:
            m = oracle.run(m, nsteps=t - t_now, **kw)
            t_now = t
        out[t] = m
    return out


def fp32_state_trajectory(oracle, cfg, times, m0=None):
    """DIAGNOSTIC, never a checker: the oracle's own step in fp64 arithmetic, but with the state rounded to
    fp32 after every step, i.e. the most faithful evaluation any implementation with an fp32 state can be.
    Shows how far an fp32-state run leaves the fp64 trajectory by itself."""
    m = np.array(cfg["moments"] if m0 is None else m0, dtype=np.float32)
    kw = dict(lattice=cfg["lattice"], ncomp=cfg["ncomp"], tau=cfg["tau"], A=cfg["A"], beta=cfg["beta"])
    out, t_now = {}, 0
    for t in sorted(times):
        while t_now < t:
            m = oracle.run(m, nsteps=1, **kw).astype(np.float32)
            t_now += 1
        out[t] = m.astype(np.float64)
    return out


def contact_states(wl, n, radius, speed, gaps, offset_z=0.0):
    """Seeded synthetic stand-ins for the contact phase of a droplet collision at full size: the two drops of the
    config-3/4 recipe on their approach line with surface gaps `gaps` (lattice units; negative = the drops overlap
    and a neck exists), approach speed +-`speed` along x, impact offset `offset_z`.  The colour field is the UNION
    of the two tanh drops (rhoA = max of the two single-drop profiles), so that 0 <= rhoA <= 1 also where they
    overlap (the recipe's sum would exceed 1 there)."""
    out = {}
    for g in gaps:
        d = 2.0 * radius + g                       # centre distance
        dx = np.sqrt(max(d * d - offset_z * offset_z, 0.0))
        c1 = (n / 2 - dx / 2, n / 2, n / 2 - offset_z / 2)
        c2 = (n / 2 + dx / 2, n / 2, n / 2 + offset_z / 2)
        m1 = wl.droplets(n, [c1], radius, [speed])
        m2 = wl.droplets(n, [c2], radius, [-speed])
        rho_a = np.maximum(m1[0], m2[0])
        out[g] = wl.pack2(rho_a, 1.0 - rho_a, [m1[2] + m2[2], m1[3] + m2[3], m1[4] + m2[4]])
    return out

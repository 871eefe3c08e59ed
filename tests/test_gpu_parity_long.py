"""GPU parity of the droplet configurations (BASELINE.json configs 3 and 4) over their whole horizon.

The physically interesting windows of the paper's droplet runs are t ~ 1e2 .. 6e3 (contact,
film rupture, merging).  The rupture of the film between the drops amplifies ANY perturbation by 1e4-1e5, so an
fp32 trajectory cannot follow the fp64 oracle to 2e-5 through the coalescence whatever evaluates it (the oracle's own
step with its state rounded to fp32 after every step leaves the fp64 trajectory the same way:
tests/config3_divergence.py, profiles/r02_config3_divergence.md).  What CAN be held to BASELINE's tolerance, and is:

  * windowed parity: restart the kernel from the ORACLE's state at t = 100, 150, 200, 400, 800, 1600, 2000 (before,
    during and after the coalescence) and compare after 10 steps: <= 2e-5 per moment field, sign(phi) >= 99.99 %;
  * the fp64 kernel straight through all 2000 steps: <= 2e-5 and 100 % sign agreement at every checkpoint;
  * the straight fp32 run: BASELINE's tolerance up to the contact (t = 100), then what an fp32 trajectory keeps
    (colour masses, bounded fields, sign(phi) on >= 99.9 % of the nodes), printed as
    "BASELINE tolerance not met after contact (fp32)".

Config 4 (256^3 x 4000 steps) is hours of oracle time: the full-size box is checked over its first steps and on
synthetic contact states (the two drops placed on their approach line with gaps +4, 0, -6: a neck exists), and its
geometry scaled to 64^3 is followed through the whole collision in windows, as config 3.
All oracle states come from oracle/ alone (tests/oracle_trajectories.py)."""
import numpy as np
import pytest

from paper_2301_01622_b200 import workloads as wl

import oracle_trajectories as traj
from parity_norms import TOL, parity_errors, report, sign_agreement

pytestmark = pytest.mark.gpu

C3_TIMES = (0, 100, 150, 200, 400, 800, 1600, 2000)
C4S_TIMES = (0, 100, 200, 400, 700, 1000)       # config 4 at 64^3 (scale 0.25): 4000 * 0.25 = 1000 steps


@pytest.fixture(scope="module")
def lbwp():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2301_01622_b200 import build as lbuild
    from paper_2301_01622_b200 import lbwp as mod
    lbuild.build()
    return mod


def _kw(cfg):
    return dict(lattice=cfg["lattice"], ncomp=2, tau=cfg["tau"], A=cfg["A"], beta=cfg["beta"])


@pytest.fixture(scope="module")
def config3_trajectory(oracle):
    """fp64 oracle trajectory of config 3 from the fp32-rounded recipe (about 6 minutes on 16 host cores)."""
    cfg = wl.config3(128)
    m0 = wl.as_dtype(cfg["moments"], "f32").astype(np.float64)
    return cfg, traj.trajectory(oracle, cfg, C3_TIMES, m0=m0)


@pytest.fixture(scope="module")
def config4_small_trajectory(oracle):
    cfg = wl.config4(64)
    m0 = wl.as_dtype(cfg["moments"], "f32").astype(np.float64)
    return cfg, traj.trajectory(oracle, cfg, C4S_TIMES, m0=m0)


def _window(lbwp, oracle, cfg, state, name, dtype="f32", steps=10):
    """Restart the kernel from an oracle state (rounded to the run's dtype), advance `steps`, compare."""
    m = wl.as_dtype(state, dtype)
    with lbwp.Lbwp(m, dtype=dtype, **_kw(cfg)) as sim:
        sim.step(steps)
        got = sim.moments_host()
    ref = oracle.run(m, nsteps=steps, **_kw(cfg))
    errs, _ = report(name, got, ref, 2, dtype, extra={"sign_agreement": sign_agreement(got, ref)})
    assert errs.max() <= TOL[dtype], (name, errs)
    assert sign_agreement(got, ref) >= 0.9999, name


# ---- config 3, windowed: the kernel IN the coalescence regime at BASELINE's tolerance ----------------------------
@pytest.mark.parametrize("t", C3_TIMES)
def test_config3_windows_fp32(lbwp, oracle, config3_trajectory, t):
    cfg, states = config3_trajectory
    _window(lbwp, oracle, cfg, states[t], "config3_128/window t=%d+10/f32" % t)


# ---- config 3, fp64 kernel straight through all 2000 steps --------------------------------------------------------
def test_config3_2000_steps_fp64(lbwp, config3_trajectory):
    cfg, states = config3_trajectory
    with lbwp.Lbwp(states[0], dtype="f64", **_kw(cfg)) as sim:
        t_now = 0
        for t in C3_TIMES[1:]:
            sim.step(t - t_now)
            t_now = t
            got = sim.moments_host()
            errs, _ = report("config3_128/straight t=%d/f64" % t, got, states[t], 2, "f64",
                             extra={"sign_agreement": sign_agreement(got, states[t])})
            assert errs.max() <= 2e-5, (t, errs)            # BASELINE's fp32 bar, held by the fp64 kernel throughout
            assert sign_agreement(got, states[t]) == 1.0, t
            if t <= 100:
                assert errs.max() <= 1e-12, (t, errs)       # and its own bar up to the contact


# ---- config 3, fp32 kernel straight: BASELINE's bar up to the contact, physical gates after it -------------------
def test_config3_2000_steps_fp32(lbwp, config3_trajectory):
    cfg, states = config3_trajectory
    m0 = states[0].astype(np.float32)
    with lbwp.Lbwp(m0, dtype="f32", **_kw(cfg)) as sim:
        sim.step(100)
        got = sim.moments_host()
        errs, _ = report("config3_128/straight t=100/f32", got, states[100], 2, "f32")
        assert errs.max() <= TOL["f32"] and sign_agreement(got, states[100]) >= 0.9999
        t_now = 100
        for t in (200, 800, 2000):
            sim.step(t - t_now)
            t_now = t
            got = sim.moments_host().astype(np.float64)
            e = parity_errors(got, states[t], 2, "f32").max()
            agree = sign_agreement(got, states[t])
            print("config3 straight fp32 t=%d: max err %.2e, sign agreement %.5f -- BASELINE tolerance %s after contact (fp32)"
                  % (t, e, agree, "met" if (e <= TOL["f32"] and agree >= 0.9999) else "not met"))
            assert np.isfinite(got).all() and np.abs(got[2:5]).max() < 0.2
            for k in (0, 1):        # each colour's mass (Eq. 1 summed over the box)
                assert abs(got[k].sum() - states[0][k].sum()) <= 2e-5 * states[0][k].sum()
            assert agree >= 0.999


# ---- config 4 at full size (256^3, fp32): first steps, in the launch configuration bench.py uses -----------------
def test_config4_full_size_first_steps(lbwp, oracle):
    cfg = wl.config4(256)
    _window(lbwp, oracle, cfg, cfg["moments"], "config4_256/t=0+12/f32", steps=12)


# ---- config 4 at full size: synthetic contact states (gap +4: films overlap; 0; -6: a neck) ----------------------
@pytest.mark.parametrize("gap", [4.0, 0.0, -6.0])
def test_config4_full_size_contact_windows(lbwp, oracle, gap):
    cfg = wl.config4(256)
    state = traj.contact_states(wl, 256, 40.0, 0.04, [gap], offset_z=32.0)[gap]
    _window(lbwp, oracle, cfg, state, "config4_256/contact gap=%+.0f +8/f32" % gap, steps=8)


# ---- config 4 scaled to 64^3: the whole off-axis collision in windows (fp32) and straight (fp64) ------------------
@pytest.mark.parametrize("t", C4S_TIMES)
def test_config4_scaled_windows_fp32(lbwp, oracle, config4_small_trajectory, t):
    cfg, states = config4_small_trajectory
    _window(lbwp, oracle, cfg, states[t], "config4_64/window t=%d+10/f32" % t)


def test_config4_scaled_straight_fp64(lbwp, config4_small_trajectory):
    cfg, states = config4_small_trajectory
    with lbwp.Lbwp(states[0], dtype="f64", **_kw(cfg)) as sim:
        t_now = 0
        for t in C4S_TIMES[1:]:
            sim.step(t - t_now)
            t_now = t
            got = sim.moments_host()
            errs, _ = report("config4_64/straight t=%d/f64" % t, got, states[t], 2, "f64")
            assert errs.max() <= 2e-5 and sign_agreement(got, states[t]) == 1.0, (t, errs)

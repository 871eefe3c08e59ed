"""More pins of the CPU oracle (CPU only): transport coefficients the paper fixes, the
two-component reading C6 against its mathematical invariants, and the comparison
kernel's mini-oracle.  Pin numbers are those of DESIGN.md "Oracle pins".
"""
import math

import numpy as np
import pytest

from paper_2301_01622_b200 import workloads as wl

LATTICES = [19, 27]


def tg_amplitude(m, n):
    """Projection of u_x on sin(kx)cos(ky) (reading C19)."""
    k = 2 * math.pi / n
    x = np.arange(n)
    basis = np.sin(k * x)[None, None, :] * np.cos(k * x)[None, :, None]
    basis = np.broadcast_to(basis, m[1].shape)
    return float((m[1] * basis).sum() / (basis * basis).sum())


# ---- P4: Taylor-Green decay gives nu = cs^2 (tau - 1/2) -------------------
@pytest.mark.parametrize("q", LATTICES)
def test_taylor_green_viscosity(oracle, q):
    n, tau = 32, 0.8
    m0 = wl.taylor_green(n, shape=(n, n, 2))          # 2D-in-3D: the field does not depend on z
    a = {0: tg_amplitude(m0, n)}
    m = m0
    for t0, t1 in ((0, 20), (20, 100)):
        m = oracle.run(m, lattice=q, tau=tau, nsteps=t1 - t0)
        a[t1] = tg_amplitude(m, n)
    k = 2 * math.pi / n
    nu = (tau - 0.5) / 3.0
    nu_meas = -math.log(a[100] / a[20]) / (2 * k * k * 80)
    assert abs(nu_meas / nu - 1) < 0.01                # north star: within 1 %
    assert abs(nu_meas / nu - 1) < 2e-3                # what the scheme actually reaches
    nu_from0 = -math.log(a[100] / a[0]) / (2 * k * k * 100)
    assert abs(nu_from0 / nu - 1) < 0.01
    # the vortex stays a vortex: u_z untouched, mass conserved
    assert np.abs(m[3]).max() < 1e-15
    assert abs(m[0].sum() - m0[0].sum()) < 1e-10


# ---- P4b: a different tau must give a different, still correct, viscosity ----------------
def test_taylor_green_viscosity_other_tau(oracle):
    n, tau = 32, 0.6
    m = oracle.run(wl.taylor_green(n, shape=(n, n, 1)), lattice=27, tau=tau, nsteps=40)
    a1 = tg_amplitude(m, n)
    m = oracle.run(m, lattice=27, tau=tau, nsteps=160)
    a2 = tg_amplitude(m, n)
    k = 2 * math.pi / n
    nu_meas = -math.log(a2 / a1) / (2 * k * k * 160)
    assert abs(nu_meas / ((tau - 0.5) / 3.0) - 1) < 0.01


# ---- P9: a small density wave oscillates at the sound speed cs = 1/sqrt(3)
@pytest.mark.parametrize("q", LATTICES)
def test_sound_speed(oracle, q):
    n, tau, eps = 64, 0.51, 1e-4
    x = np.arange(n)
    k = 2 * math.pi / n
    rho = 1.0 + eps * np.cos(k * x)[None, None, :] * np.ones((1, 1, n))
    m = wl.pack1(rho, [np.zeros_like(rho)] * 3)
    # standing wave: amplitude(t) ~ cos(cs k t) exp(-gamma t); first zero at t = pi/(2 cs k)
    amps = []
    for _ in range(40):
        m = oracle.run(m, lattice=q, tau=tau, nsteps=1)
        amps.append(float(((m[0] - 1) * np.cos(k * x)[None, None, :]).sum() * 2 / n / eps))
    amps = np.array(amps)
    i = int(np.where(amps < 0)[0][0])                  # first sign change between steps i and i+1
    t_zero = i + amps[i - 1] / (amps[i - 1] - amps[i])  # linear interpolation, time of step index i-1 is i
    cs = math.pi / (2 * k * t_zero)
    assert abs(cs * math.sqrt(3) - 1) < 0.01

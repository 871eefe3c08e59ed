"""Seeded synthetic inputs for the BASELINE.json configs (numpy only).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds
none of the method's step arithmetic: it only writes initial moment fields
``[M, nz, ny, nx]`` (fp64, caller rounds to the run's dtype).  The one formula
it needs is the definition of the initial condition "Pi = equilibrium"
(BASELINE.json configs, reading C2):
``Pi_ab = rho*cs2*delta_ab + rho*u_a*u_b``.

Field order (include/lbwp.h): M=10 ``rho,ux,uy,uz,Pxx,Pyy,Pzz,Pxy,Pxz,Pyz``;
M=11 ``rhoA,rhoB,ux,...``.  The recipes are stated in DESIGN.md "Input recipe".
The droplet configs stand in for the paper's collision benchmark
(PAPER.md:118-122, 158), whose full parameter table is not available.
"""
from __future__ import annotations

import numpy as np

CS2 = 1.0 / 3.0


def _pi_eq(rho, u):
    ux, uy, uz = u
    return [rho * (CS2 + ux * ux), rho * (CS2 + uy * uy), rho * (CS2 + uz * uz),
            rho * ux * uy, rho * ux * uz, rho * uy * uz]


def _grid(nx, ny, nz):
    z, y, x = np.meshgrid(np.arange(nz, dtype=np.float64), np.arange(ny, dtype=np.float64),
                          np.arange(nx, dtype=np.float64), indexing="ij")
    return x, y, z


def pack1(rho, u):
    return np.stack([rho, *u, *_pi_eq(rho, u)]).astype(np.float64)


def pack2(rho_a, rho_b, u):
    return np.stack([rho_a, rho_b, *u, *_pi_eq(rho_a + rho_b, u)]).astype(np.float64)


def taylor_green(n, u0=0.01, shape=None, dtype=np.float64):
    """Config 1 / sweep: 2D-in-3D Taylor-Green vortex in x-y, rho=1, k=2*pi/nx.  The field does not
    depend on z, so one fp64 x-y plane is computed and broadcast (rounded to ``dtype`` on write:
    the same values as rounding the fp64 3-D field, without its 80 B/node of host memory)."""
    nx, ny, nz = shape if shape is not None else (n, n, n)
    x, y, _ = _grid(nx, ny, 1)
    kx, ky = 2.0 * np.pi / nx, 2.0 * np.pi / ny
    ux = u0 * np.sin(kx * x) * np.cos(ky * y)
    uy = -u0 * np.cos(kx * x) * np.sin(ky * y) * (kx / ky)
    plane = pack1(np.ones_like(x), (ux, uy, np.zeros_like(x)))  # [10, 1, ny, nx]
    out = np.empty((10, nz, ny, nx), dtype=dtype)
    out[:] = plane
    return out


def _ball_wavevectors(rng, count, kmax=4):
    out = []
    while len(out) < count:
        k = rng.integers(-kmax, kmax + 1, size=3)
        if 0 < int(k @ k) <= kmax * kmax:
            out.append(k.astype(np.float64))
    return np.array(out)


def noisy_solenoidal(n, seed=20230101, rho_amp=1e-3, u_rms=0.02, shape=None):
    """Config 2: rho = 1 + 1e-3*smooth noise (8 Fourier modes, |k|<=4), u = seeded
    divergence-free field (8 modes, amplitude a x q) scaled to rms 0.02.
    Draw order: k_1..8, theta_1..8, q_1..8, a_1..8, psi_1..8 (numpy PCG64)."""
    nx, ny, nz = shape if shape is not None else (n, n, n)
    rng = np.random.default_rng(seed)
    x, y, z = _grid(nx, ny, nz)
    k = _ball_wavevectors(rng, 8)
    theta = rng.uniform(0.0, 2.0 * np.pi, 8)
    q = _ball_wavevectors(rng, 8)
    a = rng.standard_normal((8, 3))
    psi = rng.uniform(0.0, 2.0 * np.pi, 8)
    s = np.zeros_like(x)
    for m in range(8):
        s += np.cos(2.0 * np.pi * (k[m, 0] * x / nx + k[m, 1] * y / ny + k[m, 2] * z / nz) + theta[m])
    rho = 1.0 + rho_amp * s / np.abs(s).max()
    u = [np.zeros_like(x) for _ in range(3)]
    for m in range(8):
        amp = np.cross(a[m], q[m])
        ph = np.cos(2.0 * np.pi * (q[m, 0] * x / nx + q[m, 1] * y / ny + q[m, 2] * z / nz) + psi[m])
        for d in range(3):
            u[d] += amp[d] * ph
    rms = np.sqrt(np.mean(u[0] ** 2 + u[1] ** 2 + u[2] ** 2))
    u = [c * (u_rms / rms) for c in u]
    return pack1(rho, u)


def droplets(n, centres, radius, speeds, width=2.0, background_u=None, shape=None):
    """Configs 3/4 (reading C15): phi = -1 + sum_d [1 + tanh((R - r_d)/W)], r_d the
    minimum-image distance; rhoA=(1+phi)/2, rhoB=(1-phi)/2;
    u_x = sum_d U_d * (1/2)[1 + tanh((R - r_d)/W)]; Pi = Pi_eq(rhoA+rhoB, u)."""
    nx, ny, nz = shape if shape is not None else (n, n, n)
    x, y, z = _grid(nx, ny, nz)
    phi = -np.ones_like(x)
    ux = np.zeros_like(x)
    for (cx, cy, cz), U in zip(centres, speeds):
        dx = np.abs(x - cx); dx = np.minimum(dx, nx - dx)
        dy = np.abs(y - cy); dy = np.minimum(dy, ny - dy)
        dz = np.abs(z - cz); dz = np.minimum(dz, nz - dz)
        ind = 1.0 + np.tanh((radius - np.sqrt(dx * dx + dy * dy + dz * dz)) / width)
        phi += ind
        ux += U * 0.5 * ind
    u = [ux, np.zeros_like(x), np.zeros_like(x)]
    if background_u is not None:
        u = [a + b for a, b in zip(u, background_u)]
    return pack2(0.5 * (1.0 + phi), 0.5 * (1.0 - phi), u)


def config1():
    return dict(name="config1_tg32", moments=taylor_green(32), lattice=27, ncomp=1, tau=0.8,
                A=0.0, beta=0.0, steps=100, dtype="f64")


def config2(n=128, dtype="f32", steps=1000):
    return dict(name=f"config2_noise{n}", moments=noisy_solenoidal(n), lattice=27, ncomp=1,
                tau=0.6, A=0.0, beta=0.0, steps=steps, dtype=dtype)


def config3(n=128, steps=2000):
    s = n / 128.0
    return dict(name=f"config3_headon{n}",
                moments=droplets(n, [(40 * s, 64 * s, 64 * s), (88 * s, 64 * s, 64 * s)], 20 * s,
                                 [0.05, -0.05]),
                lattice=27, ncomp=2, tau=1.0, A=0.01, beta=0.7, steps=steps, dtype="f32")


def config4(n=256, steps=4000):
    s = n / 256.0
    return dict(name=f"config4_offaxis{n}",
                moments=droplets(n, [(80 * s, 128 * s, 112 * s), (176 * s, 128 * s, 144 * s)],
                                 40 * s, [0.04, -0.04]),
                lattice=27, ncomp=2, tau=1.0, A=0.01, beta=0.7, steps=steps, dtype="f32")


def sweep_case(n, lattice=27, ncomp=1, dtype="f32"):
    """Config 5 instance: 1-comp = config-1 field with k=2*pi/n, tau=0.8; 2-comp = the same
    velocity field plus config-3 geometry scaled by n/128, zero approach speed, tau=1."""
    if ncomp == 1:
        return dict(name=f"sweep_q{lattice}_c1_{dtype}_{n}",
                    moments=taylor_green(n, dtype=np.float32 if dtype == "f32" else np.float64),
                    lattice=lattice, ncomp=1, tau=0.8, A=0.0, beta=0.0, steps=200, dtype=dtype)
    tg = taylor_green(n)
    m = droplets(n, [(5 * n / 16, n / 2, n / 2), (11 * n / 16, n / 2, n / 2)], 5 * n / 32,
                 [0.0, 0.0], background_u=[tg[1], tg[2], tg[3]])
    return dict(name=f"sweep_q{lattice}_c2_{dtype}_{n}", moments=m, lattice=lattice, ncomp=2,
                tau=1.0, A=0.01, beta=0.7, steps=200, dtype=dtype)


def as_dtype(moments, dtype):
    """Round the fp64 recipe output to the run's state dtype ('f32' | 'f64')."""
    return np.ascontiguousarray(moments, dtype=np.float32 if dtype == "f32" else np.float64)

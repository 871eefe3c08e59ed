"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only).

Each test names the pin and the PAPER.md passage.  None of
them re-types the oracle's own loop: they use closed forms, invariants, special cases
and independently written numpy formulations.
"""
import math

import numpy as np
import pytest

from paper_2301_01622_b200 import workloads as wl

LATTICES = [19, 27]


def rand_moments(rng, shape, du=0.05, dp=0.02):
    """Random, non-equilibrium single-component state [10, nz, ny, nx]."""
    nz, ny, nx = shape
    rho = 1.0 + 0.1 * rng.uniform(-1, 1, shape)
    u = [du * rng.uniform(-1, 1, shape) for _ in range(3)]
    m = wl.pack1(rho, u)
    m[4:] += dp * rng.uniform(-1, 1, (6, nz, ny, nx))
    return m


# ---- lattice tables: textbook isotropy identities -------------------------
@pytest.mark.parametrize("q", LATTICES)
def test_lattice_isotropy(oracle, q):
    c, w = oracle.lattice(q)
    assert len(w) == q and len({tuple(v) for v in c.tolist()}) == q
    assert np.all(np.abs(c) <= 1)
    c = c.astype(float)
    assert abs(w.sum() - 1) < 1e-15
    assert np.allclose(np.einsum("i,ia->a", w, c), 0, atol=1e-16)
    assert np.allclose(np.einsum("i,ia,ib->ab", w, c, c), np.eye(3) / 3, atol=1e-15)
    assert np.allclose(np.einsum("i,ia,ib,ic->abc", w, c, c, c), 0, atol=1e-16)
    d = np.eye(3)
    iso4 = (np.einsum("ab,cd->abcd", d, d) + np.einsum("ac,bd->abcd", d, d)
            + np.einsum("ad,bc->abcd", d, d)) / 9
    assert np.allclose(np.einsum("i,ia,ib,ic,id->abcd", w, c, c, c, c), iso4, atol=1e-15)


# ---- P1: Eq. 4 then Eq. 1-3 returns the stored moments ---------------------
@pytest.mark.parametrize("q", LATTICES)
def test_round_trip(oracle, q):
    rng = np.random.default_rng(1)
    for _ in range(20):
        H = np.concatenate([[rng.uniform(0.5, 2)], rng.uniform(-0.2, 0.2, 3), rng.uniform(-1, 1, 6)])
        back = oracle.project(q, oracle.reconstruct(q, H, 0.0))
        assert np.max(np.abs(back - H)) < 5e-15


# ---- Eq. 8 is Eq. 7 applied to Eq. 4 and Eq. 5 --------------------------
@pytest.mark.parametrize("q", LATTICES)
def test_eq8_is_bgk_of_eq4(oracle, q):
    rng = np.random.default_rng(2)
    H = np.concatenate([[1.3], rng.uniform(-0.1, 0.1, 3), rng.uniform(-1, 1, 6)])
    Heq = H.copy()
    rho, (ux, uy, uz) = H[0], H[1:4]
    # P^eq_ab = rho cs^2 delta_ab + rho u_a u_b (reading C2), typed out in the stored order xx,yy,zz,xy,xz,yz
    Heq[4:] = [rho / 3 + rho * ux * ux, rho / 3 + rho * uy * uy, rho / 3 + rho * uz * uz,
               rho * ux * uy, rho * ux * uz, rho * uy * uz]
    h, heq = oracle.reconstruct(q, H, 0.0), oracle.reconstruct(q, Heq, 0.0)
    # closed form of Eq. 5 typed out: w rho (1 + 3cu + 4.5 cu^2 - 1.5 u^2)
    c, w = oracle.lattice(q)
    cu = c @ H[1:4]
    assert np.allclose(heq, w * H[0] * (1 + 3 * cu + 4.5 * cu ** 2 - 1.5 * H[1:4] @ H[1:4]), atol=1e-15)
    for omega in (0.3, 1.0, 1.7):
        assert np.allclose(oracle.reconstruct(q, H, omega), (1 - omega) * h + omega * heq, atol=1e-15)


# ---- P2: uniform equilibrium is a fixed point, any tau ----------------------------------
@pytest.mark.parametrize("q", LATTICES)
@pytest.mark.parametrize("tau", [0.51, 0.8, 1.0, 1.9])
def test_uniform_fixed_point(oracle, q, tau):
    shape = (4, 5, 6)
    m = wl.pack1(np.full(shape, 1.7), [np.full(shape, v) for v in (0.03, -0.05, 0.02)])
    out = oracle.run(m, lattice=q, tau=tau, nsteps=3)
    assert np.max(np.abs(out - m)) < 1e-14


# ---- P3: mass and momentum conserved on the periodic box --------------------------------
@pytest.mark.parametrize("q", LATTICES)
def test_conservation(oracle, q):
    rng = np.random.default_rng(3)
    m = rand_moments(rng, (5, 6, 7))
    out = oracle.run(m, lattice=q, tau=0.7, nsteps=4)
    assert abs(out[0].sum() - m[0].sum()) < 1e-11
    for a in range(3):
        assert abs((out[0] * out[1 + a]).sum() - (m[0] * m[1 + a]).sum()) < 1e-12


# ---- P6: tau = 1 forgets the stored pressure tensor (factor (1-omega) of Eq. 8) -----------
@pytest.mark.parametrize("q", LATTICES)
def test_tau_one_ignores_pi(oracle, q):
    rng = np.random.default_rng(4)
    m = rand_moments(rng, (4, 4, 5))
    m2 = m.copy()
    m2[4:] += rng.uniform(-1, 1, m2[4:].shape)
    a, b = oracle.run(m, lattice=q, tau=1.0, nsteps=1), oracle.run(m2, lattice=q, tau=1.0, nsteps=1)
    assert np.array_equal(a, b)
    c = oracle.run(m2, lattice=q, tau=0.9, nsteps=1)
    assert np.max(np.abs(c - a)) > 1e-3  # and it does matter otherwise


# ---- P7: lattice symmetry: swapping x<->z of the input swaps the output -----------------
@pytest.mark.parametrize("q", LATTICES)
def test_axis_permutation(oracle, q):
    rng = np.random.default_rng(5)
    m = rand_moments(rng, (4, 5, 6))
    # fields under x<->z: rho, (ux,uy,uz)->(uz,uy,ux), (xx,yy,zz,xy,xz,yz)->(zz,yy,xx,yz,xz,xy)
    perm = [0, 3, 2, 1, 6, 5, 4, 9, 8, 7]

    def swap(a):
        return np.ascontiguousarray(a[perm].transpose(0, 3, 2, 1))

    a = oracle.run(m, lattice=q, tau=0.65, nsteps=2)
    b = oracle.run(swap(m), lattice=q, tau=0.65, nsteps=2)
    assert np.max(np.abs(swap(b) - a)) < 1e-14
    mirror = m[:, :, :, ::-1].copy()   # x -> -x: ux, Pxy, Pxz change sign
    sgn = np.array([1, -1, 1, 1, 1, 1, 1, -1, -1, 1.0])[:, None, None, None]
    b = oracle.run(mirror * sgn, lattice=q, tau=0.65, nsteps=2)
    assert np.max(np.abs((b * sgn)[:, :, :, ::-1] - a)) < 1e-14


# ---- P5: a population-STORING regularised BGK (Latt-Chopard, the paper's ref. [15],
#      PAPER.md:67) written independently with numpy rolls gives the same moments ----------
def _regularised_bgk_numpy(m, q, tau, nsteps):
    cs2 = 1.0 / 3.0
    cs = [(cx, cy, cz) for cx in (0, 1, -1) for cy in (0, 1, -1) for cz in (0, 1, -1)
          if q == 27 or abs(cx) + abs(cy) + abs(cz) < 3]
    wt = {27: {0: 8 / 27, 1: 2 / 27, 2: 1 / 54, 3: 1 / 216}, 19: {0: 1 / 3, 1: 1 / 18, 2: 1 / 36}}[q]
    c = np.array(cs, dtype=float)
    w = np.array([wt[abs(a) + abs(b) + abs(d)] for a, b, d in cs])
    rho, u = m[0], m[1:4]
    Pi = np.empty((3, 3) + rho.shape)
    for (a, b), k in {(0, 0): 4, (1, 1): 5, (2, 2): 6, (0, 1): 7, (0, 2): 8, (1, 2): 9}.items():
        Pi[a, b] = Pi[b, a] = m[k]
    omega = 1.0 / tau
    for _ in range(nsteps):
        # regularise: f = feq + w/(2cs^4) (cc - cs2 I):Pi_neq ; collide ; stream (push)
        cu = np.einsum("ia,a...->i...", c, u)
        feq = w[:, None, None, None] * rho * (1 + cu / cs2 + cu ** 2 / (2 * cs2 ** 2)
                                               - np.einsum("a...,a...->...", u, u) / (2 * cs2))
        Pneq = Pi - rho * np.einsum("a...,b...->ab...", u, u) - rho * cs2 * np.eye(3)[:, :, None, None, None]
        Qi = np.einsum("ia,ib->iab", c, c) - cs2 * np.eye(3)
        fneq = w[:, None, None, None] / (2 * cs2 ** 2) * np.einsum("iab,ab...->i...", Qi, Pneq)
        fpost = feq + (1 - omega) * fneq
        f = np.stack([np.roll(fpost[i], shift=(int(c[i, 2]), int(c[i, 1]), int(c[i, 0])), axis=(0, 1, 2))
                      for i in range(len(w))])
        rho = f.sum(0)
        u = np.einsum("ia,i...->a...", c, f) / rho
        Pi = np.einsum("ia,ib,i...->ab...", c, c, f)
    return np.stack([rho, u[0], u[1], u[2], Pi[0, 0], Pi[1, 1], Pi[2, 2], Pi[0, 1], Pi[0, 2], Pi[1, 2]])


@pytest.mark.parametrize("q", LATTICES)
def test_equals_regularised_bgk_with_populations(oracle, q):
    rng = np.random.default_rng(6)
    m = rand_moments(rng, (6, 5, 7))
    ref = _regularised_bgk_numpy(m, q, 0.62, 5)
    out = oracle.run(m, lattice=q, tau=0.62, nsteps=5)
    assert np.max(np.abs(out - ref)) < 2e-15 * 50


# ---- P8: brute force on a tiny box through the algebraically different "S-form"
#      h'_i = w_i [a + 3 c.j + 4.5 cc:S],  S = omega rho uu + (1-omega)(Pi - rho/3 I),
#      a = rho - 1.5 tr S  (pure-python loops) ---------------------------------------------
@pytest.mark.parametrize("q", LATTICES)
def test_brute_force_s_form(oracle, q):
    rng = np.random.default_rng(7)
    nz, ny, nx = 3, 4, 5
    m = rand_moments(rng, (nz, ny, nx))
    tau = 0.77
    om = 1 / tau
    c, w = oracle.lattice(q)
    out = np.zeros_like(m)
    for z in range(nz):
        for y in range(ny):
            for x in range(nx):
                acc = np.zeros(10)
                for i in range(q):
                    cx, cy, cz = (int(v) for v in c[i])
                    s = m[:, (z - cz) % nz, (y - cy) % ny, (x - cx) % nx]
                    rho, u = s[0], s[1:4]
                    Pi = np.array([[s[4], s[7], s[8]], [s[7], s[5], s[9]], [s[8], s[9], s[6]]])
                    S = om * rho * np.outer(u, u) + (1 - om) * (Pi - rho / 3 * np.eye(3))
                    cv = np.array([cx, cy, cz], float)
                    h = w[i] * (rho - 1.5 * np.trace(S) + 3 * rho * cv @ u + 4.5 * cv @ S @ cv)
                    acc += h * np.array([1, cx, cy, cz, cx * cx, cy * cy, cz * cz, cx * cy, cx * cz, cy * cz])
                acc[1:4] /= acc[0]
                out[:, z, y, x] = acc
    got = oracle.run(m, lattice=q, tau=tau, nsteps=1)
    assert np.max(np.abs(got - out)) < 1e-14

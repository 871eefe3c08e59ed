"""Pins of the near-contact repulsion in the oracle (Eq. 10; readings C20-C24 of DESIGN.md; CPU only).
The paper prints neither h(x) nor the forcing scheme, so parity with the paper's code stays unpinned; what the
mathematics fixes is pinned here: the moments of the forcing term, the momentum balance of a step, locality of the
force (isolated interfaces feel none), its direction, antisymmetry and closed-form magnitude between two facing steps."""
import numpy as np
import pytest

from paper_2301_01622_b200 import workloads as wl

LATTICES = [19, 27]


# C24: moments of the forced post-collision populations (Guo, Zheng, Shi): mass rho, momentum rho u + F, and
# second moment P^eq(u*) + (1 - omega)(P - P^eq(u*)) + (1 - omega/2)(u* F + F u*), u* = u + F / (2 rho)
@pytest.mark.parametrize("q", LATTICES)
@pytest.mark.parametrize("omega", [0.6, 1.0, 1.7])
def test_forced_reconstruction_moments(oracle, q, omega):
    rng = np.random.default_rng(11)
    c, w = oracle.lattice(q)
    c = c.astype(float)
    for _ in range(5):
        rho = rng.uniform(0.7, 1.4)
        u, F = rng.uniform(-0.1, 0.1, 3), rng.uniform(-0.02, 0.02, 3)
        H = np.concatenate([[rho], u, rng.uniform(-0.2, 0.2, 6) + np.array([rho / 3] * 3 + [0.0] * 3)])
        h = oracle.reconstruct_forced(q, H, omega, F)
        us = u + F / (2 * rho)
        assert abs(h.sum() - rho) < 1e-14
        assert np.abs(c.T @ h - (rho * u + F)).max() < 1e-14
        P = np.array([[H[4], H[7], H[8]], [H[7], H[5], H[9]], [H[8], H[9], H[6]]])
        Peq = rho * np.outer(us, us) + rho / 3 * np.eye(3)
        want = Peq + (1 - omega) * (P - Peq) + (1 - omega / 2) * (np.outer(us, F) + np.outer(F, us))
        got = np.einsum("i,ia,ib->ab", h, c, c)
        assert np.abs(got - want).max() < 1e-14
        assert np.abs(oracle.reconstruct_forced(q, H, omega, np.zeros(3)) - oracle.reconstruct(q, H, omega)).max() < 1e-16


def _two_drops(n=24, gap=3.0, R=6.0):
    d = 2 * R + gap
    c = n / 2
    return wl.droplets(n, [(c - d / 2, c, c), (c + d / 2, c, c)], R, [0.0, 0.0], width=1.0)


# no force -> the plain two-component step, bit for bit; an isolated drop feels none whatever A_h
@pytest.mark.parametrize("q", LATTICES)
def test_no_contact_no_force(oracle, q):
    m = _two_drops()
    kw = dict(lattice=q, tau=0.8, nsteps=4, A=0.01, beta=0.7)
    assert np.array_equal(oracle.run_nc(m, A_h=0.0, **kw), oracle.run(m, ncomp=2, **kw))
    one = wl.droplets(24, [(12, 12, 12)], 6.0, [0.0], width=1.0)
    out, f = oracle.run_nc(one, A_h=0.05, h_c=4.0, return_force=True, **kw)
    assert np.all(f == 0.0) and np.array_equal(out, oracle.run(one, ncomp=2, **kw))
    far, f = oracle.run_nc(_two_drops(n=48, gap=13.0), A_h=0.05, h_c=4.0, return_force=True, **kw)   # drops out of range
    assert np.all(f == 0.0)


# momentum of the box changes by exactly the sum of the force per step; colour masses stay conserved
@pytest.mark.parametrize("q", LATTICES)
def test_momentum_balance(oracle, q):
    m = _two_drops(gap=2.0)
    m[2] += 0.01                                                       # some mean flow
    kw = dict(lattice=q, tau=0.7, A=0.01, beta=0.7, A_h=0.03, h_c=4.0)
    prev = m
    for _ in range(3):
        nxt, f = oracle.run_nc(prev, nsteps=1, return_force=True, **kw)
        assert np.abs(f).max() > 1e-4                                  # the force is on
        for a in range(3):
            p0 = ((prev[0] + prev[1]) * prev[2 + a]).sum()
            p1 = ((nxt[0] + nxt[1]) * nxt[2 + a]).sum()
            assert abs((p1 - p0) - f[a].sum()) < 1e-12
        for k in (0, 1):
            assert abs(nxt[k].sum() - prev[k].sum()) < 1e-11
        prev = nxt


# two facing flat step interfaces, film of `gap` nodes: G = +-1 on the two nodes next to each step, so each interface
# carries the force A_h per unit area (2 nodes x (A_h/2) |G|), pointing away from the other interface (C21);
# antisymmetric; zero once the film is thicker than h_c.
@pytest.mark.parametrize("q", LATTICES)
@pytest.mark.parametrize("gap,on", [(2, True), (3, True), (6, False)])
def test_facing_steps_closed_form(oracle, q, gap, on):
    n, A_h = 32, 0.02
    x = np.arange(n)
    phi1 = np.where((x >= 4) & (x < 12), 1.0, -1.0)                     # slab A: [4, 12)
    phi1 = np.where((x >= 12 + gap) & (x < 20 + gap), 1.0, phi1)         # slab B: film of `gap` nodes in between
    phi = np.broadcast_to(phi1[None, None, :], (3, 3, n))
    m = wl.pack2((1 + phi) / 2 + 0.0, (1 - phi) / 2 + 0.0, [np.zeros((3, 3, n))] * 3)
    _, f = oracle.run_nc(m, lattice=q, tau=1.0, nsteps=1, A=0.0, beta=0.7, A_h=A_h, h_c=4.0, return_force=True)
    assert np.all(f[1] == 0) and np.all(f[2] == 0)
    fx = f[0][0, 0]
    left = fx[8:12 + gap // 2 + 1].sum() if gap % 2 else fx[8:12 + gap // 2].sum()
    right = fx.sum() - left
    if not on:
        assert np.all(fx == 0.0)
        return
    assert abs(left + right) < 1e-15                                    # action = reaction
    assert abs(left - (-A_h)) < 1e-15 and abs(right - A_h) < 1e-15      # A_h per unit area, pushing the slabs apart
    assert np.all(fx[:9] == 0) and np.all(fx[24 + gap:] == 0)            # the outer faces of the slabs feel nothing

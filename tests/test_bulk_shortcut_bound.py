"""The inequality behind the two-component kernel's plane-level shortcut (CPU only).

The kernel skips the colour operators of a tile plane when every rA its gradients can reach lies within
delta = 2e-6 of one bulk value c (0 or 1), on the grounds that then |G|^2 <= 12 delta^2 < 1e-10 (reading C8: n = 0).
With G = 3 sum_i w_i c_i phi(x + c_i), phi = 2 rA - 1 and sum_i w_i c_i = 0:
    G_a = 6 sum_i w_i c_ia (rA_i - c),   |G_a| <= 6 delta sum_i w_i |c_ia| = 2 delta.
Checked here from the textbook lattices: the constant sum_i w_i |c_ia| = 1/3, the bound against its worst case and
against random fields, and that the margin to the threshold survives fp32 evaluation of G.
"""
import itertools

import numpy as np
import pytest

DELTA = 2e-6          # PHASE_DELTA of csrc/lbwp_tma2g.cuh
G2CUT = 1e-10         # reading C8


def lattice(q):
    """Directions and weights of D3Q27 / D3Q19 (weights by the number of non-zero components)."""
    w27 = {0: 8 / 27, 1: 2 / 27, 2: 1 / 54, 3: 1 / 216}
    w19 = {0: 1 / 3, 1: 1 / 18, 2: 1 / 36}
    cs, ws = [], []
    for c in itertools.product((-1, 0, 1), repeat=3):
        nz = sum(1 for v in c if v)
        if q == 19 and nz == 3:
            continue
        cs.append(c)
        ws.append((w27 if q == 27 else w19)[nz])
    return np.array(cs, dtype=np.float64), np.array(ws)


@pytest.mark.parametrize("q", [19, 27])
def test_first_absolute_moment_is_one_third(q):
    c, w = lattice(q)
    assert len(w) == q and abs(w.sum() - 1) < 1e-14
    assert np.abs((w[:, None] * c).sum(0)).max() < 1e-15            # sum_i w_i c_i = 0: the constant c drops out
    assert np.abs((w[:, None] * np.abs(c)).sum(0) - 1 / 3).max() < 1e-14


@pytest.mark.parametrize("q", [19, 27])
@pytest.mark.parametrize("bulk", [0.0, 1.0])
def test_gradient_bound_in_a_bulk_neighbourhood(q, bulk):
    c, w = lattice(q)
    rng = np.random.default_rng(5)
    worst = np.sign(c[:, 0]) * DELTA                                  # maximises G_x: 6 delta sum_i w_i |c_ix| = 2 delta
    g_worst = 6 * (w * c[:, 0] * (bulk + worst)).sum()
    assert abs(g_worst - 2 * DELTA) < 1e-15
    d = rng.uniform(-DELTA, DELTA, (20000, len(w)))
    G = 6 * np.einsum("i,ia,ni->na", w, c, bulk + d)
    g2 = (G * G).sum(1)
    assert g2.max() <= 12 * DELTA ** 2 < G2CUT / 2                    # factor-two margin to the threshold
    # the same sums in fp32 (the kernel's arithmetic, any order): rounding of values near 1 moves |G|^2 by far less
    G32 = 6 * np.einsum("i,ia,ni->na", w.astype(np.float32), c.astype(np.float32), (bulk + d).astype(np.float32))
    assert (G32.astype(np.float64) ** 2).sum(1).max() < G2CUT


# ---- the near-contact fix-up pass (csrc/lbwp_contact.cuh) skips a box of nodes when rA over the
#      box and its halo of one node spans less than SPAN: then |G_a| <= max - min at every node of the box (the weights
#      of the directions with c_ia = +1 sum to 1/6) and |G|^2 <= 3 SPAN^2 stays below G_I^2 (reading C22), so no node of
#      the box would start the interface walk ------------------------------------------------------------------------
SPAN = 0.02           # the cut of k_contact_fixup
GI2 = 0.05 ** 2       # G_I^2 (reading C22)


@pytest.mark.parametrize("q", [19, 27])
def test_contact_box_skip_bound(q):
    c, w = lattice(q)
    for a in range(3):
        assert abs(w[c[:, a] > 0].sum() - 1 / 6) < 1e-15 and abs(w[c[:, a] < 0].sum() - 1 / 6) < 1e-15
    assert 3 * SPAN ** 2 < GI2 / 2                                    # factor-two margin
    rng = np.random.default_rng(11)
    lo = rng.uniform(0, 1 - SPAN, (20000, 1))
    r = lo + rng.uniform(0, SPAN, (20000, len(w)))                    # any field of that span, not only near a bulk value
    r[:, :2] = np.stack([lo[:, 0], lo[:, 0] + SPAN], 1)               # the extremes are attained
    G = 6 * np.einsum("i,ia,ni->na", w, c, r)
    span = r.max(1) - r.min(1)
    assert (np.abs(G).max(1) <= span + 1e-15).all()
    worst = np.where(c[:, 0] > 0, SPAN, 0.0)                          # maximises G_x: 6 SPAN / 6 = SPAN
    assert abs(6 * (w * c[:, 0] * worst).sum() - SPAN) < 1e-15
    G32 = 6 * np.einsum("i,ia,ni->na", w.astype(np.float32), c.astype(np.float32), r.astype(np.float32))
    assert (G32.astype(np.float64) ** 2).sum(1).max() < GI2

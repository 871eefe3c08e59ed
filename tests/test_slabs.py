"""z-slab decomposition: host bookkeeping and the halo exchange over torch.distributed on CPU
(gloo, two and three ranks), and on the GPU the decomposed box against the undivided one, element for element
(several slabs as contexts on ONE device, halos exchanged by device copies: `slabs.SlabGroup`)."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2301_01622_b200 import slabs
from paper_2301_01622_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


# ---- owner ranges, neighbours, wrap at the box ends (host logic) ------------------------------------------------------
@pytest.mark.parametrize("nz,world", [(8, 1), (8, 2), (10, 3), (7, 7), (513, 8)])
def test_slab_ranges_tile_the_box(nz, world):
    ranges = [slabs.slab_range(nz, world, r) for r in range(world)]
    assert ranges[0][0] == 0 and ranges[-1][1] == nz
    for (a0, a1), (b0, b1) in zip(ranges[:-1], ranges[1:]):
        assert a1 == b0 and a1 > a0
    sizes = [b - a for a, b in ranges]
    assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    for r in range(world):
        below, above = slabs.neighbours(world, r)
        assert slabs.neighbours(world, below)[1] == r and slabs.neighbours(world, above)[0] == r


def test_local_planes_wrap():
    assert slabs.local_planes(10, 3, 0, 1).tolist() == [9, 0, 1, 2, 3, 4]        # lower halo wraps to the top of the box
    assert slabs.local_planes(10, 3, 2, 2).tolist() == [5, 6, 7, 8, 9, 0, 1]     # upper halo wraps to the bottom
    assert slabs.halo_width(1) == 1 and slabs.halo_width(2) == 2
    assert slabs.halo_width(2, A_h=0.02, h_c=4.0) == 7 and slabs.halo_width(2, A_h=0.02, h_c=2.5) == 5   # near-contact walk
    assert slabs.halo_width(1, A_h=0.02) == 1
    g = np.arange(2 * 10 * 1 * 1, dtype=np.float64).reshape(2, 10, 1, 1)
    loc = slabs.local_moments(g, 3, 1, 1)
    assert loc.shape == (2, 5, 1, 1) and loc[0, :, 0, 0].tolist() == [3, 4, 5, 6, 7]
    with pytest.raises(ValueError):
        slabs.slab_range(2, 3, 0)


def test_slab_rejects_what_the_halo_cannot_carry():
    m = np.zeros((11, 8, 8, 64), dtype=np.float32)
    with pytest.raises(ValueError, match="moments scheme"):
        slabs.SlabLbwp(m, world=2, rank=0, ncomp=2, tau=1.0, scheme="populations")


# ---- the exchange itself over gloo: a 3-point stencil in z on a decomposed periodic array ------------------------------
def _stencil_worker(rank, world, port, nz, halo, steps, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    rng = np.random.default_rng(7)
    g = rng.uniform(-1, 1, (1, nz, 2, 3))                                    # every rank draws the same global field
    loc = torch.from_numpy(slabs.local_moments(g, world, rank, halo)[0])      # [owned + 2 halo, 2, 3]
    tr = slabs.DistTransport(world, rank)
    n = loc.shape[0]
    for _ in range(steps):
        new = loc.clone()
        new[1:-1] = 0.25 * loc[:-2] + 0.5 * loc[1:-1] + 0.25 * loc[2:]        # valid on every plane but the outermost
        new[0], new[-1] = 1e30, -1e30                                         # what a periodic local box would spoil
        send_down, send_up = new[halo:2 * halo].contiguous(), new[n - 2 * halo:n - halo].contiguous()
        recv_down, recv_up = torch.empty_like(send_down), torch.empty_like(send_up)
        tr.exchange(send_down, send_up, recv_down, recv_up)
        new[:halo], new[n - halo:] = recv_down, recv_up
        loc = new
    z0, z1 = slabs.slab_range(nz, world, rank)
    out.put((rank, z0, z1, loc[halo:n - halo].numpy().copy()))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,nz,halo", [(2, 9, 1), (3, 10, 2), (2, 8, 2), (2, 29, 7)])   # 7: the near-contact halo
def test_exchange_over_gloo(world, nz, halo):
    steps = 5
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() + 7 * world + nz) % 2000
    procs = [ctx.Process(target=_stencil_worker, args=(r, world, port, nz, halo, steps, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=180) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    g = np.random.default_rng(7).uniform(-1, 1, (1, nz, 2, 3))[0]
    for _ in range(steps):
        g = 0.25 * np.roll(g, 1, axis=0) + 0.5 * g + 0.25 * np.roll(g, -1, axis=0)
    got = np.concatenate([r[3] for r in res], axis=0)
    assert [(r[1], r[2]) for r in res] == [slabs.slab_range(nz, world, r) for r in range(world)]
    assert np.array_equal(got, g)                                             # same additions in the same order: exact


# ---- GPU: the decomposed box equals the undivided one ------------------------------------------------------------------
@pytest.mark.gpu
@pytest.mark.parametrize("world", [2, 3])
@pytest.mark.parametrize("ncomp,dtype,shape,lattice", [(1, "f32", (128, 16, 40), 27), (1, "f64", (64, 16, 23), 19),
                                                       (2, "f32", (64, 16, 30), 27), (2, "f32", (64, 8, 24), 19),
                                                       (2, "f64", (32, 16, 21), 27), (1, "f64", (20, 12, 18), 27)])
def test_slabs_equal_single_box(world, ncomp, dtype, shape, lattice):
    assert torch.cuda.is_available()
    from paper_2301_01622_b200 import build as lbuild
    from paper_2301_01622_b200 import lbwp
    lbuild.build()
    nx, ny, nz = shape
    if ncomp == 1:
        m = wl.noisy_solenoidal(0, shape=shape)
        kw = dict(lattice=lattice, dtype=dtype, ncomp=1, tau=0.6)
    else:
        tg = wl.taylor_green(0, shape=shape)
        m = wl.droplets(0, [(0.3 * nx, 0.5 * ny, 0.1 * nz), (0.8 * nx, 0.2 * ny, 0.6 * nz)], 0.3 * min(ny, nx), [0.03, -0.03],
                        background_u=[tg[1], tg[2], tg[3]], shape=shape)       # one drop sits across a slab boundary
        kw = dict(lattice=lattice, dtype=dtype, ncomp=2, tau=0.7, A=0.01, beta=0.7)
    m0 = wl.as_dtype(m, dtype)
    steps = 12
    with lbwp.Lbwp(m0, **kw) as sim:
        sim.step(steps)
        whole = sim.moments_host()
        name = sim.kernel_name
    grp = slabs.SlabGroup(m0, world, **kw)
    try:
        assert all(s.sim.kernel_name == name for s in grp.slabs)
        assert np.array_equal(grp.moments(), m0)                              # t = 0: owned planes tile the input
        grp.step(steps)
        parts = grp.moments()
    finally:
        grp.close()
    assert parts.shape == whole.shape
    assert np.array_equal(parts, whole), float(np.abs(parts.astype(np.float64) - whole).max())


# the near-contact force in slabs (halo floor(h_c) + 3 = 7 planes): two drops pressed against each other, the film between
# them lying across the slab boundary; the fused path (fix-up pass behind the TMA kernel) and the generic one
@pytest.mark.gpu
@pytest.mark.parametrize("dtype,shape,lattice,kernel", [("f32", (64, 40, 36), 19, "tma"), ("f64", (64, 40, 37), 27, "tma"),
                                                        ("f32", (40, 36, 34), 27, "gather")])
def test_slabs_near_contact_equal_single_box(dtype, shape, lattice, kernel):
    from paper_2301_01622_b200 import build as lbuild
    from paper_2301_01622_b200 import lbwp
    lbuild.build()
    nx, ny, nz = shape
    R, gap = 9.0, 2.0
    d = 2 * R + gap
    # the drops face each other along z, the film at z = nz / 2: the boundary between the two slabs
    uz = np.broadcast_to(0.03 * np.cos(2 * np.pi * (np.arange(nz) + 0.5) / nz)[:, None, None], (nz, ny, nx))   # a flow along z, through the slab boundaries
    m = wl.droplets(0, [(nx / 2 - 2, ny / 2, nz / 2 - d / 2), (nx / 2 + 2, ny / 2, nz / 2 + d / 2)], R, [0.0, 0.0],
                    background_u=[np.zeros((nz, ny, nx)), np.zeros((nz, ny, nx)), uz], shape=shape)
    m0 = wl.as_dtype(m, dtype)
    kw = dict(lattice=lattice, dtype=dtype, ncomp=2, tau=0.8, A=0.01, beta=0.7, A_h=0.02, h_c=4.0)
    steps = 15
    with lbwp.Lbwp(m0, **kw) as sim:
        assert sim.kernel_name.startswith(kernel)
        sim.step(steps)
        whole = sim.moments_host()
        name = sim.kernel_name
    with lbwp.Lbwp(m0, **dict(kw, A_h=0.0)) as sim:
        sim.step(steps)
        assert np.abs(sim.moments_host().astype(np.float64) - whole).max() > 1e-4   # the force acts in this set-up
    grp = slabs.SlabGroup(m0, 2, **kw)
    try:
        assert all(s.sim.kernel_name == name and s.halo == 7 for s in grp.slabs)
        grp.step(steps)
        parts = grp.moments()
    finally:
        grp.close()
    assert np.array_equal(parts, whole), float(np.abs(parts.astype(np.float64) - whole).max())


@pytest.mark.gpu
def test_halo_calls_reject_bad_ranges():
    from paper_2301_01622_b200 import lbwp
    m0 = wl.as_dtype(wl.noisy_solenoidal(0, shape=(64, 8, 6)), "f32")
    with lbwp.Lbwp(m0, tau=0.6) as sim:
        buf = torch.empty(sim.halo_bytes(2), dtype=torch.uint8, device="cuda")
        assert sim.halo_bytes(2) == 2 * sim.halo_bytes(1) > 0
        sim.halo_pack(4, 2, buf)
        with pytest.raises(lbwp.LbwpError):
            sim.halo_pack(5, 2, buf)
        with pytest.raises(ValueError):
            sim.halo_pack(0, 3, buf)
    with lbwp.Lbwp(m0, tau=0.6, scheme="populations") as sim:
        assert sim.halo_bytes(1) == 0

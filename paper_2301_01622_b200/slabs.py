"""z-slab decomposition of one periodic box over several GPUs (the method's memory
saving is what makes multi-billion-node grids fit, and those are multi-GPU grids).

One process per GPU.  Rank r owns the global planes ``slab_range(nz, world, r)`` and keeps them, with ``H`` halo planes
on each side, as an ordinary periodic box of the library (``lbwp_ctx``).  One time step of the decomposed box:

    lbwp_step(ctx, 1)                      every rank, its own slab (the H outermost planes it computes are garbage)
    lbwp_halo_pack  x 2                    the H lowest and H highest OWNED planes of the new state
    send / recv with the z neighbours      torch.distributed point-to-point (NCCL over NVLink on GPUs; gloo in the CPU test)
    lbwp_halo_unpack x 2                   into the halo planes

H = 1 (the stencil reaches one plane), H = 2 for two-component moments (the colour gradient of a source plane reaches
one plane further), H = floor(h_c) + 3 with the near-contact force (its interface walk and the gradients on the way).  Everything the method computes runs inside the library's kernels; this module only moves opaque
packed planes between ranks (marshalling and communication plumbing).  Per face and step the exchange carries
``M * nx * ny * sizeof`` bytes (10.6 MB at 512^2 fp32): about 12 us at NVLink 5 rates against a step of 1-2 ms.
"""
from __future__ import annotations

import numpy as np


def halo_width(ncomp: int, A_h: float = 0.0, h_c: float = 4.0) -> int:
    """Halo planes a slab needs on each side (moments scheme).  With the near-contact force a node's
    force looks floor(h_c) + 1 planes away (the interface walk, plus the gradient at the node it stops on), on top of
    the 2 outermost planes a step leaves wrong."""
    if ncomp == 2 and A_h:
        return 2 + int(np.floor(h_c)) + 1
    return 2 if ncomp == 2 else 1


def _halo_of(kw: dict) -> int:
    return halo_width(kw.get("ncomp", 1), kw.get("A_h", 0.0), kw.get("h_c", 4.0))


def slab_range(nz: int, world: int, rank: int):
    """Global planes [z0, z1) owned by `rank`: an even split, the first nz % world ranks own one plane more."""
    if not (0 <= rank < world) or nz < world:
        raise ValueError("need 0 <= rank < world <= nz")
    base, extra = divmod(nz, world)
    z0 = rank * base + min(rank, extra)
    return z0, z0 + base + (1 if rank < extra else 0)


def neighbours(world: int, rank: int):
    """(rank below, rank above) in z, periodic."""
    return (rank - 1) % world, (rank + 1) % world


def local_planes(nz: int, world: int, rank: int, halo: int) -> np.ndarray:
    """Global plane index of every plane of the rank's local box, halo planes included (periodic wrap at the ends)."""
    z0, z1 = slab_range(nz, world, rank)
    return np.arange(z0 - halo, z1 + halo) % nz


def local_moments(global_moments: np.ndarray, world: int, rank: int, halo: int) -> np.ndarray:
    """The rank's initial moments [M, owned + 2 halo, ny, nx] cut out of the global field [M, nz, ny, nx]."""
    return np.ascontiguousarray(global_moments[:, local_planes(global_moments.shape[1], world, rank, halo)])


class DistTransport:
    """Exchange with the z neighbours through torch.distributed point-to-point operations."""

    def __init__(self, world: int, rank: int):
        self.world, self.rank = world, rank

    def exchange(self, send_down, send_up, recv_down, recv_up):
        """send_down goes to the rank below (it becomes that rank's UPPER halo), send_up to the rank above;
        recv_down arrives from below, recv_up from above.  Tensors of equal size."""
        import torch.distributed as dist

        below, above = neighbours(self.world, self.rank)
        if self.world == 1:
            recv_up.copy_(send_down)      # the box wraps onto itself
            recv_down.copy_(send_up)
            return
        # Messages between one pair of ranks match in posting order (NCCL has no tags).  With two ranks both
        # neighbours are the same peer: it sends (down, up), and its "down" is this rank's upper halo, so the
        # receives are posted as (up, down).
        ops = [dist.P2POp(dist.isend, send_down, below), dist.P2POp(dist.isend, send_up, above),
               dist.P2POp(dist.irecv, recv_up, above), dist.P2POp(dist.irecv, recv_down, below)]
        for req in dist.batch_isend_irecv(ops):
            req.wait()


class LocalTransport:
    """All slabs live in this process (several contexts on one device): the neighbours' buffers are copied directly.
    Used by the single-GPU test of the decomposition; `peers` is filled by SlabGroup."""

    def __init__(self, world: int, rank: int, mailbox: dict):
        self.world, self.rank, self.mailbox = world, rank, mailbox

    def post(self, send_down, send_up):
        self.mailbox[(self.rank, "down")] = send_down
        self.mailbox[(self.rank, "up")] = send_up

    def collect(self, recv_down, recv_up):
        below, above = neighbours(self.world, self.rank)
        recv_down.copy_(self.mailbox[(below, "up")])      # what the rank below sent upwards
        recv_up.copy_(self.mailbox[(above, "down")])


class SlabLbwp:
    """One rank's slab: an `Lbwp` context over the owned planes plus halo, and the per-step halo exchange."""

    def __init__(self, local_m0, *, world, rank, transport=None, **lbwp_kwargs):
        import torch

        from . import lbwp

        self.world, self.rank = world, rank
        self.halo = _halo_of(lbwp_kwargs)
        if lbwp_kwargs.get("scheme", "moments") != "moments":
            raise ValueError("slab decomposition: moments scheme only")
        self.sim = lbwp.Lbwp(local_m0, **lbwp_kwargs)
        self.nz_local = self.sim.shape[0]
        self.owned = self.nz_local - 2 * self.halo
        if self.owned < self.halo:
            raise ValueError("a slab must own at least as many planes as its halo is wide")
        nb = self.sim.halo_bytes(self.halo)
        self.transport = transport or DistTransport(world, rank)
        dev = self.sim.device
        self.send_down, self.send_up, self.recv_down, self.recv_up = (
            torch.empty(nb, dtype=torch.uint8, device=dev) for _ in range(4))

    def pack(self):
        h = self.halo
        self.sim.halo_pack(h, h, self.send_down)                      # lowest owned planes -> upper halo of the rank below
        self.sim.halo_pack(self.nz_local - 2 * h, h, self.send_up)    # highest owned planes -> lower halo of the rank above

    def unpack(self):
        h = self.halo
        self.sim.halo_unpack(0, h, self.recv_down)
        self.sim.halo_unpack(self.nz_local - h, h, self.recv_up)

    def step(self, n=1):
        """n time steps of the decomposed box (collective: every rank calls it)."""
        import torch

        for _ in range(int(n)):
            self.sim.step(1)
            self.pack()
            torch.cuda.current_stream(self.sim.device).synchronize()   # the packed planes are complete before they travel
            self.transport.exchange(self.send_down, self.send_up, self.recv_down, self.recv_up)
            self.unpack()

    def moments_owned(self) -> np.ndarray:
        """The owned planes of the current moments, host array [M, owned, ny, nx]."""
        return self.sim.moments_host()[:, self.halo:self.nz_local - self.halo]

    def close(self):
        self.sim.close()


class SlabGroup:
    """All slabs of a box in ONE process on one device (testing / single-GPU emulation of the decomposition): steps them
    in lock-step and exchanges the halos by device copies."""

    def __init__(self, global_m0, world, **lbwp_kwargs):
        self.world = world
        self.mailbox = {}
        halo = _halo_of(lbwp_kwargs)
        self.slabs = [SlabLbwp(local_moments(global_m0, world, r, halo), world=world, rank=r,
                               transport=LocalTransport(world, r, self.mailbox), **lbwp_kwargs) for r in range(world)]

    def step(self, n=1):
        import torch

        for _ in range(int(n)):
            for s in self.slabs:
                s.sim.step(1)
                s.pack()
                s.transport.post(s.send_down, s.send_up)
            torch.cuda.synchronize()
            for s in self.slabs:
                s.transport.collect(s.recv_down, s.recv_up)
                s.unpack()

    def moments(self) -> np.ndarray:
        return np.concatenate([s.moments_owned() for s in self.slabs], axis=1)

    def close(self):
        for s in self.slabs:
            s.close()

"""z-slab decomposition of one lattice over several GPUs (include/clip.h, clip_halo_pack).

One process per GPU owns about `nz / world` consecutive z planes (slab_range) plus ONE ghost plane beyond each interior cut (face type CLIP_BC_HALO:
libclip steps the owned planes only).  After every step each side of a cut sends one record of 12 words per face node -- the ten
populations of its boundary plane that move towards the neighbour (Eq. 13 / 33 streaming; Alg. 2 :432-459) and
two partial sums of phi(t+1) = sum_a g_a (Eq. 38), from which both sides complete phi on the two planes of the cut (the stencils of
Eq. 40, :307-309, read it one plane away).  The owned planes then equal those of the undivided lattice to round-off (phi of the cut
planes is summed in another order).  The exchange is the path's only collective: a neighbour send / recv (`torch.distributed` P2P:
NCCL over NVLink on GPUs, gloo in the CPU tests), no reduction.  Packing, stepping and unpacking run in libclip.

This module holds plumbing only (who owns which planes, who sends what to whom); no arithmetic of the method.
"""
from __future__ import annotations

HALO = 1  # ghost planes per interior cut (see the module docstring)

_HALO_BC = 5  # CLIP_BC_HALO


def slab_range(nz: int, rank: int, world: int):
    """Owned planes [z0, z1) of `rank`: consecutive slabs of nz // world planes, the first nz % world slabs one plane more (the halo
    record does not depend on the kernel path a slab's lattice admits, so the slabs need not be equal)."""
    if world < 1 or not 0 <= rank < world:
        raise ValueError("bad rank / world")
    base, rem = divmod(nz, world)
    if base < 2:
        raise ValueError(f"a slab must own at least 2 planes (got {base}): its two halo records must not depend on each other")
    z0 = rank * base + min(rank, rem)
    return z0, z0 + base + (1 if rank < rem else 0)


def slab_ghosts(rank: int, world: int, z_periodic: bool):
    """(ghost planes below, ghost planes above) of `rank`: none next to a physical (non-periodic) z face."""
    lo = HALO if (z_periodic or rank > 0) else 0
    hi = HALO if (z_periodic or rank < world - 1) else 0
    return lo, hi


def slab_plane_index(nz: int, rank: int, world: int, z_periodic: bool):
    """Global z index of every local plane (ghosts included, wrapped on a periodic lattice), as a list."""
    z0, z1 = slab_range(nz, rank, world)
    lo, hi = slab_ghosts(rank, world, z_periodic)
    return [z % nz for z in range(z0 - lo, z1 + hi)]


def neighbours(rank: int, world: int, z_periodic: bool):
    """(rank below, rank above); None where the slab ends at a physical face."""
    below = (rank - 1) % world if (z_periodic or rank > 0) else None
    above = (rank + 1) % world if (z_periodic or rank < world - 1) else None
    return below, above


def exchange(send_lo, send_hi, recv_lo, recv_hi, rank: int, world: int, z_periodic: bool, group=None):
    """Neighbour exchange of the halo records (tensors on the backend's device; any may be None where there is no neighbour).

    send_lo (my lowest owned planes) -> the rank below, which receives it as ITS recv_hi; send_hi -> the rank above, as its
    recv_lo.  Sends are posted upward first and receives downward first, so that with two ranks on a periodic lattice -- where
    both neighbours are the same peer and P2P messages match in posting order -- the records still land on the right side.
    A single periodic slab is its own neighbour: local copies."""
    import torch.distributed as dist
    below, above = neighbours(rank, world, z_periodic)
    if world == 1:
        if below is not None:
            recv_hi.copy_(send_lo)
            recv_lo.copy_(send_hi)
        return
    ref = send_lo if send_lo is not None else send_hi
    if ref is not None and ref.is_cuda and dist.get_backend(group) == "gloo":
        # no NCCL (tests: two processes sharing one GPU; boxes without peer access): stage the records through host memory
        host = [None if t is None else t.cpu() for t in (send_lo, send_hi, recv_lo, recv_hi)]
        exchange(*host, rank, world, z_periodic, group)
        if recv_lo is not None:
            recv_lo.copy_(host[2])
        if recv_hi is not None:
            recv_hi.copy_(host[3])
        return
    ops = []
    if above is not None:
        ops.append(dist.P2POp(dist.isend, send_hi, above, group))
    if below is not None:
        ops.append(dist.P2POp(dist.isend, send_lo, below, group))
    if below is not None:
        ops.append(dist.P2POp(dist.irecv, recv_lo, below, group))
    if above is not None:
        ops.append(dist.P2POp(dist.irecv, recv_hi, above, group))
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()


class SlabClip:
    """One rank's slab of a global nx x ny x nz lattice.  `params["bc"]` are the GLOBAL faces (any type the library takes)."""

    def __init__(self, nx, ny, nz, params: dict, rank: int, world: int, device="cuda:0", stream=None, overlap=True):
        from . import clip
        bc = [int(v) for v in params["bc"]]
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.rank, self.world = int(rank), int(world)
        self.z_periodic = bc[4] == 0
        self.z0, self.z1 = slab_range(self.nz, self.rank, self.world)
        self.lo, self.hi = slab_ghosts(self.rank, self.world, self.z_periodic)
        self.planes = slab_plane_index(self.nz, self.rank, self.world, self.z_periodic)
        self.nz_local = len(self.planes)
        # Local faces: a physical z face belongs to the first / last slab; every cut face is HALO (also both faces of the single slab
        # of a periodic lattice, which is its own neighbour).  The record does not depend on the kernel path: slabs may differ.
        local = dict(params)
        if self.lo:
            bc[4] = _HALO_BC
        if self.hi:
            bc[5] = _HALO_BC
        local["bc"] = tuple(bc)
        self.sim = clip.Clip(self.nx, self.ny, self.nz_local, local, device=device, stream=stream)
        self.torch = self.sim.torch
        self.device = self.sim.device
        mk = lambda n: self.sim.halo_buffer() if n else None  # noqa: E731
        self.send_lo, self.recv_lo = mk(self.lo), mk(self.lo)
        self.send_hi, self.recv_hi = mk(self.hi), mk(self.hi)
        self.exchanges = 0
        # overlapped step (clip_step_halo_begin / _end): the records travel on a second, higher-priority stream while the interior
        # of the slab is still being computed
        self.halo = None
        if overlap and (self.lo or self.hi):
            with self.torch.cuda.device(self.device):
                self.halo = self.torch.cuda.Stream(device=self.device, priority=-1)
            self.sim.halo_stream(self.halo)

    # -- plumbing -------------------------------------------------------------------------------------------------
    def init(self, phi0, u0):
        """phi0 [nz, ny, nx], u0 [3, nz, ny, nx]: the GLOBAL initial fields (host or device tensors); the slab takes its planes."""
        t = self.torch
        idx = t.as_tensor(self.planes, dtype=t.long, device=phi0.device)
        self.sim.init(phi0.index_select(0, idx), u0.index_select(1, idx))

    def pack(self):
        """Records of my boundary planes into the send buffers (clip_halo_pack, one launch)."""
        self.sim.halo_pack(self.send_lo, self.send_hi)

    def unpack(self):
        """Complete the two planes of each cut from the received records (clip_halo_unpack, one launch)."""
        self.sim.halo_unpack(self.recv_lo, self.recv_hi, self.send_lo, self.send_hi)
        self.exchanges += 1

    def halo_exchange(self, group=None):
        """pack -> neighbour send / recv -> unpack, all on the handle's stream (one process per GPU)."""
        t = self.torch
        with t.cuda.device(self.device), t.cuda.stream(self.sim.stream):
            self.pack()
            if self.world == 1:   # a single periodic slab is its own neighbour: unpack straight from what was packed
                if self.lo:
                    self.sim.halo_unpack(self.send_hi, self.send_lo, self.send_lo, self.send_hi)
                self.exchanges += 1
                return
            exchange(self.send_lo, self.send_hi, self.recv_lo, self.recv_hi, self.rank, self.world, self.z_periodic, group)
            self.unpack()

    def step(self, n=1, group=None):
        """n time steps of the global lattice: clip_step(1) on the slab, then the halo exchange, n times; nothing here waits for
        the GPU.  The first call also exchanges the records of the initial state."""
        t = self.torch
        if self.exchanges == 0:
            self.halo_exchange(group)
        for _ in range(int(n)):
            if self.halo is None:
                self.sim.step(1)
                self.halo_exchange(group)
                continue
            self.sim.step_halo_begin(self.send_lo, self.send_hi)      # records are produced on the halo stream ...
            if self.world == 1:
                self.sim.step_halo_end(self.send_hi, self.send_lo, self.send_lo, self.send_hi)
            else:
                with t.cuda.device(self.device), t.cuda.stream(self.halo):   # ... and travel on it while the interior computes
                    exchange(self.send_lo, self.send_hi, self.recv_lo, self.recv_hi, self.rank, self.world, self.z_periodic, group)
                self.sim.step_halo_end(self.recv_lo, self.recv_hi, self.send_lo, self.send_hi)
            self.exchanges += 1

    def get(self):
        """phi, p [own, ny, nx] and u [3, own, ny, nx] of the OWNED planes z0 .. z1-1."""
        phi, p, u = self.sim.get()
        a, b = self.lo, self.nz_local - self.hi
        return phi[a:b], p[a:b], u[:, a:b]

    @property
    def halo_bytes_per_step(self):
        """Bytes this rank sends per step."""
        return sum(b.numel() * b.element_size() for b in (self.send_lo, self.send_hi) if b is not None)

    def close(self):
        self.sim.close()


def step_group(slabs, n=1):
    """All slabs of a lattice held by ONE process (tests; several slabs on one GPU, stepped one after the other -- no kernel waits on
    another): step each, then hand every record to its neighbour (the neighbour unpacks straight from the sender's buffer)."""
    world = len(slabs)

    def swap():
        for s in slabs:
            s.pack()
        s0 = slabs[0]
        s0.torch.cuda.synchronize()   # the slabs may sit on different streams
        for s in slabs:
            below, above = neighbours(s.rank, world, s.z_periodic)
            s.sim.halo_unpack(slabs[below].send_hi if below is not None else None, slabs[above].send_lo if above is not None else None,
                              s.send_lo, s.send_hi)
            s.exchanges += 1

    if slabs[0].exchanges == 0:
        swap()
    for _ in range(int(n)):
        for s in slabs:
            s.sim.step(1)
        swap()

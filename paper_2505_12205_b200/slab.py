"""z-slab decomposition of one lattice over several GPUs (include/clip.h, clip_halo_pack).

One process per GPU owns `nz / world` consecutive z planes plus two ghost planes beyond each interior cut.  After every
step the two outermost OWNED planes on each side go to the z neighbour, which writes them over its ghost planes: the pull of
Eq. 13 / 33 (Alg. 2 :432-459) reaches one plane, the stencils of Eq. 40 (:309-331) on phi(t+1) one more, so
two planes make the owned planes equal to those of the undivided lattice (bit for bit on the two-kernel path; the
k_fused path sums phi in tile order, and a slab has other tiles than the whole lattice: equal to round-off).  The exchange is
the path's only collective: a neighbour send / recv (`torch.distributed` P2P: NCCL over NVLink on GPUs, gloo in the CPU tests),
no reduction.  Everything else -- packing, stepping, unpacking -- runs in libclip.

This module holds plumbing only (who owns which planes, who sends what to whom); no arithmetic of the method.
"""
from __future__ import annotations

HALO = 2  # ghost planes per interior cut (see the module docstring)

_WALL = 1  # CLIP_BC_WALL


def slab_range(nz: int, rank: int, world: int):
    """Owned planes [z0, z1) of `rank`: equal slabs (every rank must pick the same kernel path, clip.h)."""
    if world < 1 or not 0 <= rank < world:
        raise ValueError("bad rank / world")
    if nz % world != 0:
        raise ValueError(f"nz = {nz} is not a multiple of the {world} slabs")
    own = nz // world
    if own < HALO:
        raise ValueError(f"a slab of {own} planes is thinner than the halo ({HALO})")
    return rank * own, (rank + 1) * own


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


def halo_planes(nz_local: int, lo: int, hi: int):
    """First local plane of the four halo records: the owned planes that are SENT down / up, and the ghost planes that the
    records RECEIVED from below / above overwrite (None where that side has no ghosts)."""
    return {"send_lo": lo if lo else None, "send_hi": nz_local - hi - HALO if hi else None,
            "recv_lo": 0 if lo else None, "recv_hi": nz_local - HALO if hi else None}


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

    def __init__(self, nx, ny, nz, params: dict, rank: int, world: int, device="cuda:0", stream=None):
        from . import clip
        bc = [int(v) for v in params["bc"]]
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.rank, self.world = int(rank), int(world)
        self.z_periodic = bc[4] == 0
        self.z0, self.z1 = slab_range(self.nz, self.rank, self.world)
        self.lo, self.hi = slab_ghosts(self.rank, self.world, self.z_periodic)
        self.planes = slab_plane_index(self.nz, self.rank, self.world, self.z_periodic)
        self.nz_local = len(self.planes)
        # Local faces: a physical z face belongs to the first / last slab; a cut face may apply any rule (its planes are ghosts and are
        # overwritten): PERIODIC on a periodic lattice (all slabs alike), else WALL.  Slabs with different faces or plane counts could
        # choose different kernel paths; the record must agree on whether phi(t+1) is state, so they are created with path = 2.
        local = dict(params)
        if not self.z_periodic:
            bc[4] = bc[4] if self.rank == 0 else _WALL
            bc[5] = bc[5] if self.rank == self.world - 1 else _WALL
            local["bc"] = tuple(bc)
            if self.world > 1 and int(params.get("path", 0)) in (0, 3):
                local["path"] = 2
        self.sim = clip.Clip(self.nx, self.ny, self.nz_local, local, device=device, stream=stream)
        self.torch = self.sim.torch
        self.device = self.sim.device
        self.hp = halo_planes(self.nz_local, self.lo, self.hi)
        mk = lambda n: self.sim.halo_buffer(HALO) if n else None  # noqa: E731
        self.send_lo, self.recv_lo = mk(self.lo), mk(self.lo)
        self.send_hi, self.recv_hi = mk(self.hi), mk(self.hi)
        self.exchanges = 0

    # -- plumbing -------------------------------------------------------------------------------------------------
    def init(self, phi0, u0):
        """phi0 [nz, ny, nx], u0 [3, nz, ny, nx]: the GLOBAL initial fields (host or device tensors); the slab takes its planes."""
        t = self.torch
        idx = t.as_tensor(self.planes, dtype=t.long, device=phi0.device)
        self.sim.init(phi0.index_select(0, idx), u0.index_select(1, idx))

    def pack(self):
        """Copy my outermost owned planes into the send buffers (clip_halo_pack)."""
        if self.lo:
            self.sim.halo_pack(self.hp["send_lo"], HALO, self.send_lo)
        if self.hi:
            self.sim.halo_pack(self.hp["send_hi"], HALO, self.send_hi)

    def unpack(self):
        """Write the received records over my ghost planes (clip_halo_unpack)."""
        if self.lo:
            self.sim.halo_unpack(self.hp["recv_lo"], HALO, self.recv_lo)
        if self.hi:
            self.sim.halo_unpack(self.hp["recv_hi"], HALO, self.recv_hi)
        self.exchanges += 1

    def halo_exchange(self, group=None):
        """pack -> neighbour send / recv -> unpack, all on the handle's stream (one process per GPU)."""
        t = self.torch
        with t.cuda.device(self.device), t.cuda.stream(self.sim.stream):
            self.pack()
            exchange(self.send_lo, self.send_hi, self.recv_lo, self.recv_hi, self.rank, self.world, self.z_periodic, group)
            self.unpack()

    def step(self, n=1, group=None):
        """n time steps of the global lattice: clip_step(1) on the slab, then the halo exchange, n times.
        The first call also refreshes the ghosts of the initial state (k_init's gradient is wrong on the outermost plane)."""
        if self.exchanges == 0:
            self.halo_exchange(group)
        for _ in range(int(n)):
            self.sim.step(1)
            self.halo_exchange(group)

    def get(self):
        """phi, p [own, ny, nx] and u [3, own, ny, nx] of the OWNED planes z0 .. z1-1."""
        phi, p, u = self.sim.get()
        a, b = self.lo, self.nz_local - self.hi
        return phi[a:b], p[a:b], u[:, a:b]

    @property
    def halo_bytes_per_step(self):
        """Bytes this rank sends per step."""
        return sum(b.numel() for b in (self.send_lo, self.send_hi) if b is not None)

    def close(self):
        self.sim.close()


def step_group(slabs, n=1):
    """All slabs of a lattice held by ONE process (tests; several slabs on one GPU, stepped one after the other -- no kernel waits on
    another): step each, then hand every record to its neighbour by a device copy."""
    world = len(slabs)

    def swap():
        for s in slabs:
            s.pack()
        for s in slabs:
            below, above = neighbours(s.rank, world, s.z_periodic)
            if below is not None:
                s.recv_lo.copy_(slabs[below].send_hi)
            if above is not None:
                s.recv_hi.copy_(slabs[above].send_lo)
        for s in slabs:
            s.unpack()

    if slabs[0].exchanges == 0:
        swap()
    for _ in range(int(n)):
        for s in slabs:
            s.sim.step(1)
        swap()

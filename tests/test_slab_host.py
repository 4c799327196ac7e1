"""CPU-side checks of the z-slab decomposition plumbing (paper_2505_12205_b200/slab.py): who owns which planes,
and -- over gloo with 2 and 3 ranks -- that the halo records reach the right side of the right neighbour.  The stand-in
"step" is an integer recurrence with the structure of the real one: a state v with reach one plane (the populations), a derived
field w = weighted sum of v over the three planes around (phi(t+1) = sum of streamed g), a step that reads v and w one plane away;
the record carries the boundary plane's v, the part of its w that comes from the sender's side, and the sender's contribution to
the neighbour's boundary plane -- exactly the protocol of include/clip.h (clip_halo_pack).  A record that lands on the wrong side
or comes from the wrong rank changes the owned planes."""
import json
import os
import subprocess
import sys

import pytest

from paper_2505_12205_b200 import slab

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("nz,world,periodic", [(8, 1, True), (8, 2, True), (12, 3, True), (8, 2, False), (16, 4, False), (6, 3, True), (10, 3, True), (33, 2, False), (17, 4, False)])
def test_partition_covers_the_lattice(nz, world, periodic):
    owned = []
    for r in range(world):
        z0, z1 = slab.slab_range(nz, r, world)
        lo, hi = slab.slab_ghosts(r, world, periodic)
        planes = slab.slab_plane_index(nz, r, world, periodic)
        assert len(planes) == (z1 - z0) + lo + hi
        assert planes[lo:len(planes) - hi] == list(range(z0, z1))
        below, above = slab.neighbours(r, world, periodic)
        assert (lo == 0) == (below is None) and (hi == 0) == (above is None)
        assert lo in (0, slab.HALO) and hi in (0, slab.HALO) and slab.HALO == 1
        if lo:
            assert planes[:lo] == [(z0 - 1) % nz]
            # my ghost plane below is the top owned plane of the rank below
            b0, b1 = slab.slab_range(nz, below, world)
            assert planes[:lo] == [b1 - 1]
        if hi:
            a0, _ = slab.slab_range(nz, above, world)
            assert planes[-hi:] == [a0]
        owned += list(range(z0, z1))
    assert owned == list(range(nz))


def test_partition_rejects_bad_splits():
    assert [slab.slab_range(10, r, 3) for r in range(3)] == [(0, 4), (4, 7), (7, 10)]   # unequal slabs are fine
    with pytest.raises(ValueError):
        slab.slab_range(4, 0, 4)        # a slab must own two planes
    with pytest.raises(ValueError):
        slab.slab_range(8, 2, 2)


_WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
import torch
import torch.distributed as dist
from paper_2505_12205_b200 import slab

dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
NZ, NXY, STEPS, MOD = 6 * world, 5, 9, 1000003
A, B, C = 2, 3, 5          # w[z] = A v[z-1] + B v[z] + C v[z+1]
ok = True

def shifted(v, d, wrap):
    n = v.shape[0]
    j = torch.arange(n) + d
    return v[j % n if wrap else j.clamp(0, n - 1)]

def w_of(v, wrap):
    return (A * shifted(v, -1, wrap) + B * v + C * shifted(v, 1, wrap)) % MOD

def advance(v, w, wrap):
    return (shifted(v, -1, wrap) + 7 * v + 11 * shifted(v, 1, wrap) + 13 * shifted(w, -1, wrap) + 17 * w + 19 * shifted(w, 1, wrap)) % MOD

for periodic in (True, False):
    g = torch.Generator().manual_seed(7)
    full = torch.randint(0, MOD, (NZ, NXY), generator=g, dtype=torch.int64)
    planes = slab.slab_plane_index(NZ, rank, world, periodic)
    lo, hi = slab.slab_ghosts(rank, world, periodic)
    n = len(planes)
    v = full[planes].clone()
    w = torch.zeros_like(v)
    buf = lambda on: torch.empty((3, NXY), dtype=torch.int64) if on else None
    recv_lo, recv_hi = buf(lo), buf(hi)

    def swap():
        # records: [v of the boundary plane, part of its w from my side, my contribution to the neighbour's boundary plane]
        send_lo = torch.stack([v[lo], (B * v[lo] + C * v[lo + 1]) % MOD, (C * v[lo]) % MOD]) if lo else None
        send_hi = torch.stack([v[n - 1 - hi], (A * v[n - 2 - hi] + B * v[n - 1 - hi]) % MOD, (A * v[n - 1 - hi]) % MOD]) if hi else None
        slab.exchange(send_lo, send_hi, recv_lo, recv_hi, rank, world, periodic)
        wl = w_of(v, False)                 # owned planes: from v incl. the ghosts' v; physical ends clamp
        if lo:
            v[0] = recv_lo[0]
        if hi:
            v[n - 1] = recv_hi[0]
        wl = w_of(v, False)
        if lo:
            wl[0] = (recv_lo[1] + send_lo[2]) % MOD
        if hi:
            wl[n - 1] = (recv_hi[1] + send_hi[2]) % MOD
        return wl

    for s in range(STEPS):
        w = swap()
        wf = w_of(full, periodic)
        ok = ok and bool((w == wf[planes]).all()) and bool((v == full[planes]).all())
        full = advance(full, wf, periodic)
        vn = advance(v, w, False)
        if lo: vn[0] = v[0]                 # ghost planes are not stepped
        if hi: vn[n - 1] = v[n - 1]
        v = vn
    own = slice(lo, n - hi)
    ok = ok and bool((v[own] == full[planes][own]).all())
flag = torch.tensor([1 if ok else 0])
dist.all_reduce(flag, op=dist.ReduceOp.MIN)
if rank == 0:
    print(json.dumps(dict(ok=bool(flag.item()), world=world)))
dist.destroy_process_group()
"""


@pytest.mark.parametrize("world,port", [(2, 29741), (3, 29742)])
def test_halo_exchange_gloo(tmp_path, world, port):
    """world_size 2 (both neighbours are the same peer on a periodic lattice) and 3 on CPU: after every exchange the
    local state and the derived field, ghosts included, equal the planes of the undivided run."""
    script = tmp_path / "slab_worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={world}",
                          "--master-addr", "127.0.0.1", "--master-port", str(port), str(script)],
                         capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    r = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    assert r == {"ok": True, "world": world}


def test_single_periodic_slab_is_its_own_neighbour():
    import torch
    a, b = torch.arange(4.0), torch.arange(4.0) + 10
    ra, rb = torch.zeros(4), torch.zeros(4)
    slab.exchange(a, b, ra, rb, 0, 1, True)
    assert torch.equal(ra, b) and torch.equal(rb, a)


def test_bench_input_planes_match_the_whole_field():
    """`inputs.sweep_drops(z_planes=...)` (each rank of the slab bench builds only its own planes): phi0 equals the planes of the
    whole field, u0 of a plane does not depend on who asks for it."""
    import numpy as np
    from paper_2505_12205_b200 import inputs
    whole = inputs.sweep_drops(shape=(16, 12, 24), ndrops=4, rmin=3, rmax=5)
    planes = slab.slab_plane_index(24, 0, 3, True)
    assert planes == [23, 0, 1, 2, 3, 4, 5, 6, 7, 8]
    part = inputs.sweep_drops(shape=(16, 12, 24), ndrops=4, rmin=3, rmax=5, z_planes=planes)
    assert part["nz"] == 24 and part["phi0"].shape == (10, 12, 16) and part["u0"].shape == (3, 10, 12, 16)
    assert np.array_equal(part["phi0"], whole["phi0"][planes])
    other = inputs.sweep_drops(shape=(16, 12, 24), ndrops=4, rmin=3, rmax=5, z_planes=slab.slab_plane_index(24, 1, 3, True))
    assert np.array_equal(other["u0"][:, :2], part["u0"][:, 8:10])       # planes 7, 8: rank 1's ghost (owned by rank 0) and first owned plane (rank 0's ghost)
    assert np.abs(part["u0"]).max() <= 0.01

"""CPU-side checks of the z-slab decomposition plumbing (paper_2505_12205_b200/slab.py): who owns which planes,
and -- over gloo with 2 and 3 ranks -- that the halo records reach the right side of the right neighbour.  The stand-in
"step" is an integer recurrence with the same reach as the real one (two planes each way) on the local wrapped array, so that a
ghost layer that is too thin, a record that lands on the wrong side or a wrong plane offset changes the owned planes."""
import json
import os
import subprocess
import sys

import pytest

from paper_2505_12205_b200 import slab

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("nz,world,periodic", [(8, 1, True), (8, 2, True), (12, 3, True), (8, 2, False), (16, 4, False), (6, 3, True)])
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
        if lo:
            assert planes[:lo] == [(z0 - 2) % nz, (z0 - 1) % nz]
            # my ghost planes below are the planes the rank below sends upward
            b0, b1 = slab.slab_range(nz, below, world)
            assert planes[:lo] == [b1 - 2, b1 - 1]
        if hi:
            a0, _ = slab.slab_range(nz, above, world)
            assert planes[-hi:] == [a0, a0 + 1]
        hp = slab.halo_planes(len(planes), lo, hi)
        if lo:
            assert hp["recv_lo"] == 0 and planes[hp["send_lo"]] == z0
        if hi:
            assert hp["recv_hi"] == len(planes) - 2 and planes[hp["send_hi"] + 1] == z1 - 1
        owned += list(range(z0, z1))
    assert owned == list(range(nz))


def test_partition_rejects_bad_splits():
    with pytest.raises(ValueError):
        slab.slab_range(10, 0, 3)       # not a multiple
    with pytest.raises(ValueError):
        slab.slab_range(4, 0, 4)        # thinner than the halo
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
NZ, NXY, STEPS, MOD = 6 * world, 5, 7, 1000003
ok = True
for periodic in (True, False):
    g = torch.Generator().manual_seed(7)
    full = torch.randint(0, MOD, (NZ, NXY), generator=g, dtype=torch.int64)

    def advance(v, wrap):   # reach: two planes each way; a non-periodic end repeats its last plane
        n = v.shape[0]
        idx = torch.arange(n)
        def at(d):
            j = idx + d
            j = j % n if wrap else j.clamp(0, n - 1)
            return v[j]
        return (at(-2) + 2 * at(-1) + 3 * at(0) + 5 * at(1) + 7 * at(2)) % MOD

    planes = slab.slab_plane_index(NZ, rank, world, periodic)
    lo, hi = slab.slab_ghosts(rank, world, periodic)
    hp = slab.halo_planes(len(planes), lo, hi)
    loc = full[planes].clone()
    H = slab.HALO
    buf = lambda on: torch.empty((H, NXY), dtype=torch.int64) if on else None
    recv_lo, recv_hi = buf(lo), buf(hi)
    for s in range(STEPS):
        full = advance(full, periodic)
        # the local array wraps on itself (periodic) or clamps (a ghost face may apply any rule): ghosts come out wrong
        loc = advance(loc, periodic)
        send_lo = loc[hp["send_lo"]:hp["send_lo"] + H].clone() if lo else None
        send_hi = loc[hp["send_hi"]:hp["send_hi"] + H].clone() if hi else None
        slab.exchange(send_lo, send_hi, recv_lo, recv_hi, rank, world, periodic)
        if lo: loc[hp["recv_lo"]:hp["recv_lo"] + H] = recv_lo
        if hi: loc[hp["recv_hi"]:hp["recv_hi"] + H] = recv_hi
    ok = ok and bool((loc == full[planes]).all())
flag = torch.tensor([1 if ok else 0])
dist.all_reduce(flag, op=dist.ReduceOp.MIN)
if rank == 0:
    print(json.dumps(dict(ok=bool(flag.item()), world=world)))
dist.destroy_process_group()
"""


@pytest.mark.parametrize("world,port", [(2, 29741), (3, 29742)])
def test_halo_exchange_gloo(tmp_path, world, port):
    """world_size 2 (both neighbours are the same peer on a periodic lattice) and 3 on CPU: after every exchange the
    local array, ghosts included, equals the planes of the undivided run."""
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
    assert planes == [22, 23, 0, 1, 2, 3, 4, 5, 6, 7, 8, 9]
    part = inputs.sweep_drops(shape=(16, 12, 24), ndrops=4, rmin=3, rmax=5, z_planes=planes)
    assert part["nz"] == 24 and part["phi0"].shape == (12, 12, 16) and part["u0"].shape == (3, 12, 12, 16)
    assert np.array_equal(part["phi0"], whole["phi0"][planes])
    other = inputs.sweep_drops(shape=(16, 12, 24), ndrops=4, rmin=3, rmax=5, z_planes=slab.slab_plane_index(24, 1, 3, True))
    assert np.array_equal(other["u0"][:, :4], part["u0"][:, 8:12])       # planes 6..9: ghosts of rank 1, owned by rank 0
    assert np.abs(part["u0"]).max() <= 0.01

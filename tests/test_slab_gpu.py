"""z-slab decomposition (include/clip.h clip_halo_pack / clip_halo_unpack; paper_2505_12205_b200/slab.py) on ONE GPU:
the slabs of a lattice live in one process and are stepped one after the other (no kernel waits on another), the 12-word halo
records change hands on the device.  The owned planes must equal the undivided lattice to round-off on every kernel path (phi of
the two planes of a cut is completed from partial sums, i.e. in another order than on the undivided lattice) -- and the oracle
within the north_star tolerances."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

from paper_2505_12205_b200 import inputs

pytestmark = pytest.mark.gpu


def _whole(case, steps, precision):
    import torch
    from paper_2505_12205_b200 import clip
    sim = clip.Clip.from_case(case, precision=precision)
    sim.step(steps)
    out = sim.get()
    torch.cuda.synchronize()
    sim.close()
    return out


def _slabs(case, steps, precision, world, chunks=None):
    import torch
    from paper_2505_12205_b200 import slab
    params = dict(case["params"]); params["precision"] = precision
    phi0, u0 = torch.as_tensor(case["phi0"]), torch.as_tensor(case["u0"])
    group = [slab.SlabClip(case["nx"], case["ny"], case["nz"], params, r, world) for r in range(world)]
    for s in group:
        s.init(phi0, u0)
    for c in (chunks or (steps,)):
        slab.step_group(group, c)
    parts = [s.get() for s in group]
    torch.cuda.synchronize()
    out = (torch.cat([p[0] for p in parts], 0), torch.cat([p[1] for p in parts], 0), torch.cat([p[2] for p in parts], 1))
    assert all(s.exchanges == steps + 1 for s in group)
    launches = sum(s.sim.launches for s in group)
    for s in group:
        s.close()
    return out, launches


def _with(case, **kw):
    case["params"].update(kw)
    return case


CASES = {   # name: (case, steps, slab counts, clip_params overrides)
    "sweep64": (lambda: inputs.sweep_drops(n=64), 30, (1, 2, 4), {}),                       # periodic z, pair kernels
    "rt_replica": (lambda: inputs.rayleigh_taylor(L=16, W=3.0), 30, (2, 4), {}),            # y walls, periodic z
    "walled_box": (lambda: inputs.walled_box(nx=12, ny=10, nz=16), 30, (2, 4), {}),         # z walls: end slabs have one ghost side
    "odd_box": (lambda: inputs.sweep_drops(shape=(21, 12, 36), ndrops=4, rmin=3, rmax=5), 30, (3,), {}),   # odd nx: generic kernels
    # open z faces (BASELINE configs[3] replica): the inlet belongs to the first slab, the convective outlet to the last; planes
    # z = 0 and nz-1 by the generic kernels in the slabs as in the undivided lattice.  U_max: the plane maximum lives in the last slab
    "jet_replica": (lambda: inputs.jet(nxy=24, nz=96, r_nozzle=4.0), 40, (2, 3, 4), {}),
    "jet_replica_umax": (lambda: _with(inputs.jet(nxy=24, nz=48, r_nozzle=4.0), outlet_u_mode=2), 40, (2,), {}),
    # free-slip on all six faces: generic kernels everywhere (the cut faces of the inner slabs would otherwise take the pair kernels)
    "freeslip_box": (lambda: _with(inputs.walled_box(nx=12, ny=10, nz=16), bc=(inputs.FREESLIP,) * 6), 30, (2, 4), {"path": 1}),
}


@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("name", sorted(CASES))
def test_slabs_equal_the_undivided_lattice(name, precision):
    import torch
    make, steps, worlds, over = CASES[name]
    case = make()
    case["params"].update(dict({"path": 2}, **over))
    ref = _whole(case, steps, precision)
    tol = 1e-12 if precision == 64 else 3e-5
    for world in worlds:
        out, launches = _slabs(case, steps, precision, world, chunks=(steps - 7, 7))
        assert launches > 0
        for a, b, what in zip(out, ref, ("phi", "p", "u")):
            assert torch.isfinite(a).all()
            err = float((a - b).abs().max()) / max(float(b.abs().max()), 1e-300)
            assert err <= tol or (precision == 32 and what == "p"), f"{name} fp{precision} {world} slabs: {what} differs by {err:.3e} of field scale"


@pytest.mark.parametrize("precision", [64, 32])
def test_slabs_on_the_fused_path(precision):
    """k_fused scatters phi(t+1) on chip and cannot see the ghost plane's populations: clip_halo_unpack adds the neighbour's
    contribution (clip.h).  Periodic box, a box walled in z (end slabs have one HALO face) and the jet replica (inlet / outlet in the
    end slabs); equal to the undivided two-kernel run to round-off."""
    import torch
    steps = 30
    for case, worlds in ((inputs.sweep_drops(n=64), (1, 2, 4)), (inputs.walled_box(nx=64, ny=12, nz=24), (2, 3)),
                         (inputs.jet(nxy=64, nz=48, r_nozzle=6.0), (2, 3))):
        case["params"]["path"] = 2
        ref = _whole(case, steps, precision)
        case["params"]["path"] = 3
        for world in worlds:
            _check_fused_slabs(case, steps, precision, world, ref)


def _check_fused_slabs(case, steps, precision, world, ref):
    out, _ = _slabs(case, steps, precision, world, chunks=(1, steps - 1))
    tol = 1e-12 if precision == 64 else 3e-5
    for a, b, what in zip(out, ref, ("phi", "p", "u")):
        scale = float(b.abs().max())
        err = float((a - b).abs().max()) / max(scale, 1e-300)
        print(f"fused slabs {case['name']} fp{precision} world {world} {what}: {err:.2e} of field scale")
        assert err <= tol or (precision == 32 and what == "p"), (case["name"], what, world, err)   # fp32 p is not gated (north_star)


@pytest.mark.parametrize("precision", [64, 32])
def test_overlapped_slab_step_equals_the_plain_sequence(precision):
    """clip_step_halo_begin / _end (boundary chunks + pack on a second stream, interior + k_fix on the handle's stream, unpack after
    both) runs the same kernels on the same data as step; pack; unpack: bit for bit.  One periodic slab that is its own neighbour,
    k_fused path (split launch) and pair kernels (plain sequence with the pack on the halo stream)."""
    import torch
    from paper_2505_12205_b200 import slab
    for path, shape in ((3, (64, 16, 40)), (2, (64, 16, 12)), (3, (128, 8, 8))):
        case = inputs.sweep_drops(shape=shape, ndrops=4, rmin=3, rmax=5)
        params = dict(case["params"], precision=precision, path=path)
        outs = []
        for overlap in (False, True):
            sl = slab.SlabClip(*shape, params, 0, 1, overlap=overlap)
            sl.init(torch.as_tensor(case["phi0"]), torch.as_tensor(case["u0"]))
            sl.step(9); sl.step(6)
            outs.append([t.clone() for t in sl.get()])
            assert sl.exchanges == 16 and (sl.halo is not None) == overlap
            torch.cuda.synchronize()
            sl.close()
        for a, b in zip(*outs):
            assert torch.isfinite(a).all() and torch.equal(a, b), (path, shape)
    case = inputs.sweep_drops(shape=(64, 16, 12), ndrops=3, rmin=3, rmax=4)
    sl = slab.SlabClip(64, 16, 12, dict(case["params"], precision=precision), 0, 1)
    from paper_2505_12205_b200 import clip
    assert clip.clip_step_halo_end(sl.sim._h, 0, 0, 0, 0) == clip.CLIP_ESTATE      # no open step
    sl.init(torch.as_tensor(case["phi0"]), torch.as_tensor(case["u0"]))
    sl.sim.step_halo_begin(sl.send_lo, sl.send_hi)
    assert clip.clip_step(sl.sim._h, 1) == clip.CLIP_ESTATE                          # a step is open
    assert clip.clip_step_halo_begin(sl.sim._h, sl.send_lo.data_ptr(), sl.send_hi.data_ptr()) == clip.CLIP_ESTATE
    sl.sim.step_halo_end(sl.send_hi, sl.send_lo, sl.send_lo, sl.send_hi)
    sl.sim.step(0)
    torch.cuda.synchronize()
    sl.close()


def test_slabs_may_take_different_kernel_paths():
    """The record does not depend on the kernel path (clip.h): a lattice whose end slabs run the pair kernels (path 2) while the
    inner ones run k_fused gives the undivided result to round-off."""
    import torch
    from paper_2505_12205_b200 import slab
    case = inputs.sweep_drops(shape=(64, 16, 48), ndrops=4, rmin=3, rmax=6)
    case["params"].update(bc=(inputs.PERIODIC,) * 4 + (inputs.WALL, inputs.WALL), path=2)
    ref = _whole(case, 20, 64)
    params = dict(case["params"], precision=64)
    phi0, u0 = torch.as_tensor(case["phi0"]), torch.as_tensor(case["u0"])
    group = [slab.SlabClip(64, 16, 48, dict(params, path=(3 if r in (1, 2) else 2)), r, 4) for r in range(4)]
    assert group[0].send_lo is None and tuple(group[0].send_hi.shape) == (12, 16, 64)
    for s in group:
        s.init(phi0, u0)
    slab.step_group(group, 20)
    parts = [s.get() for s in group]
    kinds = [{k for k, v in s.sim.step_profiled(1).items() if v[1]} for s in group]
    torch.cuda.synchronize()
    assert "k_fused" in kinds[1] and "k_fused" in kinds[2] and "k_step2" in kinds[0] and "k_step2" in kinds[3]
    out = (torch.cat([p[0] for p in parts], 0), torch.cat([p[1] for p in parts], 0), torch.cat([p[2] for p in parts], 1))
    for a, b in zip(out, ref):
        assert float((a - b).abs().max()) <= 1e-12 * max(1.0, float(b.abs().max()))
    for s in group:
        s.close()


def test_slabs_against_the_oracle():
    """BASELINE configs[0] (drop, 32^3, 100 steps) on two and four slabs vs the CPU oracle: fp64 <= 1e-10, fp32 1e-4 / 1e-3."""
    from oracle.clip_oracle import Oracle
    case = inputs.drop()
    o = Oracle.from_case(case)
    o.step(100)
    rphi, rp, ru = o.get()
    for precision, world in ((64, 2), (64, 4), (32, 2)):
        (phi, p, u), _ = _slabs(case, 100, precision, world)
        phi, p, u = (t.double().cpu().numpy() for t in (phi, p, u))
        if precision == 64:
            assert np.abs(phi - rphi).max() <= 1e-10 and np.abs(p - rp).max() <= 1e-10 and np.abs(u - ru).max() <= 1e-10
        else:
            assert np.abs(phi - rphi).max() / np.abs(rphi).max() <= 1e-4
            assert np.abs(u - ru).max() / max(np.abs(ru).max(), 1e-30) <= 1e-3


def test_halo_abi_errors_and_record_contents():
    import torch
    from paper_2505_12205_b200 import clip
    case = inputs.sweep_drops(n=16, ndrops=3, rmin=3.0, rmax=5.0, W=3.0, precision=64)
    assert clip.clip_workspace_bytes(16, 16, 16, clip.make_params(dict(case["params"], bc=(5, 5, 0, 0, 0, 0)))) == 0      # HALO only in z
    assert clip.clip_workspace_bytes(16, 16, 3, clip.make_params(dict(case["params"], bc=(0, 0, 0, 0, 5, 5)))) == 0       # owns < 2 planes
    sim = clip.Clip(16, 16, 16, dict(case["params"], bc=(0, 0, 0, 0, 5, 5)))
    lo, hi = sim.halo_buffer(), sim.halo_buffer()
    assert clip.clip_halo_bytes(sim._h) == 12 * 16 * 16 * 8 and clip.clip_halo_bytes(None) == 0
    assert clip.clip_halo_pack(sim._h, lo.data_ptr(), hi.data_ptr()) == clip.CLIP_ESTATE          # before clip_init
    sim.init(torch.as_tensor(case["phi0"]), torch.as_tensor(case["u0"]))
    assert clip.clip_halo_pack(sim._h, lo.data_ptr(), 0) == clip.CLIP_EINVAL                      # a HALO face without a buffer
    assert clip.clip_halo_pack(sim._h, lo.data_ptr() + 8, hi.data_ptr()) == clip.CLIP_EINVAL      # misaligned
    assert clip.clip_halo_unpack(sim._h, lo.data_ptr(), hi.data_ptr(), 0, hi.data_ptr()) == clip.CLIP_EINVAL
    n0 = sim.launches
    sim.halo_pack(lo, hi)
    assert sim.launches == n0 + 1                                                                # one launch for both faces
    # uniform phi = 1 at rest would make every record entry equal; here: the sums of the record's phi parts over a face
    # equal what the planes hold: sum_x (part + C of the other side) = sum_x phi(t+1) of a periodic plane pair
    torch.cuda.synchronize()
    assert torch.isfinite(lo).all() and torch.isfinite(hi).all()
    assert float(lo[:10].abs().max()) > 0 and float(lo[10].min()) >= -1e-6 and float(lo[11].min()) >= -1e-6
    plain = clip.Clip(16, 16, 16, case["params"])       # no HALO face: nothing to pack, NULL buffers are fine
    plain.init(torch.as_tensor(case["phi0"]), torch.as_tensor(case["u0"]))
    assert clip.clip_halo_pack(plain._h, 0, 0) == clip.CLIP_OK and clip.clip_halo_unpack(plain._h, 0, 0, 0, 0) == clip.CLIP_OK
    plain.close()
    sim.close()


_DIST_WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
import torch
import torch.distributed as dist
from paper_2505_12205_b200 import clip, inputs, slab

dist.init_process_group("gloo")        # NCCL refuses two ranks on one GPU; the records are staged through the host
rank, world = dist.get_rank(), dist.get_world_size()
ok = True
for make, steps in ((lambda: inputs.sweep_drops(shape=(32, 32, 36), ndrops=5, rmin=3, rmax=6), 25), (lambda: inputs.jet(nxy=24, nz=48, r_nozzle=4.0), 25)):
    case = make()
    case["params"]["path"] = 2       # per-node arithmetic independent of the tiling: bit for bit
    params = dict(case["params"]); params["precision"] = 64
    sl = slab.SlabClip(case["nx"], case["ny"], case["nz"], params, rank, world, device="cuda:0")
    sl.init(torch.as_tensor(case["phi0"]), torch.as_tensor(case["u0"]))
    sl.step(steps - 5)
    sl.step(5)
    mine = [t.cpu().contiguous() for t in sl.get()]
    assert sl.exchanges == steps + 1
    sl.close()
    parts = [[torch.empty_like(t) for _ in range(world)] if rank == 0 else None for t in mine]
    for t, dst in zip(mine, parts):
        dist.gather(t, dst, dst=0)
    if rank == 0:
        whole = clip.Clip.from_case(case, precision=64)
        whole.step(steps)
        ref = [t.cpu() for t in whole.get()]
        whole.close()
        got = [torch.cat(parts[0], 0), torch.cat(parts[1], 0), torch.cat(parts[2], 1)]
        ok = ok and all(float((a - b).abs().max()) <= 1e-12 * max(1.0, float(b.abs().max())) for a, b in zip(got, ref))
flag = torch.tensor([1 if ok else 0])
dist.broadcast(flag, 0)
if rank == 0:
    print(json.dumps(dict(ok=bool(flag.item()), world=world)))
dist.destroy_process_group()
"""


@pytest.mark.parametrize("world,port", [(2, 29751), (3, 29752)])
def test_slab_ranks_as_processes(tmp_path, world, port):
    """The distributed code path itself (SlabClip.step -> halo_exchange -> torch.distributed P2P): `world` processes, one slab
    each, sharing the one GPU (no kernel waits on another: the exchange is host-synchronous over gloo), periodic box and jet
    replica; the gathered owned planes equal the undivided lattice to round-off."""
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    script = tmp_path / "slab_dist_worker.py"
    script.write_text(_DIST_WORKER.format(root=root))
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={world}",
                          "--master-addr", "127.0.0.1", "--master-port", str(port), str(script)],
                         capture_output=True, text=True, timeout=600, cwd=root)
    assert out.returncode == 0, out.stderr[-3000:]
    r = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    assert r == {"ok": True, "world": world}

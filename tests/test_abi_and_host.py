"""CPU-side checks of the product's host logic: the C-ABI library loads and exports every symbol include/clip.h
declares, argument validation (no GPU needed: these paths return before any CUDA call), the binding has no CPU
fallback, and the multi-rank plumbing of bench.py (world_size 2 over gloo)."""
import ctypes as C
import os
import re
import subprocess
import sys

import pytest

from paper_2505_12205_b200 import clip, inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "clip.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(clip_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    names = _declared_symbols()
    for must in ("clip_workspace_bytes", "clip_create", "clip_init", "clip_step", "clip_get", "clip_destroy", "clip_last_error"):
        assert must in names
    lib = C.CDLL(clip.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), n


def test_struct_mirror_matches_header_order():
    """The ctypes mirror lists the fields of `struct clip_params` in the header's order."""
    src = open(os.path.join(ROOT, "include", "clip.h")).read()
    body = src[src.index("typedef struct clip_params {"):src.index("} clip_params;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split("{", 1)[1].split(";"):
        decl = decl.strip()
        if not decl:
            continue
        for nm in decl.split(None, 1)[1].split(","):
            fields.append(re.sub(r"\[.*\]", "", nm).strip())
    assert fields == [f[0] for f in clip.clip_params._fields_]


def test_validation_without_gpu():
    p = inputs.default_params()
    ok = clip.make_params(p)
    n = clip.clip_workspace_bytes(32, 32, 32, ok)
    # 2 x (f + g) A/B buffers + phi + 3 u, fp64, plus alignment padding
    assert n >= (4 * 19 + 4) * 32 ** 3 * 8 and n < (4 * 19 + 4) * 32 ** 3 * 8 + 64 * 1024
    p32 = dict(p); p32["precision"] = 32
    assert clip.clip_workspace_bytes(32, 32, 32, clip.make_params(p32)) < n
    for bad, word in (
        (dict(precision=16), "precision"),
        (dict(bc=(0, 1, 0, 0, 0, 0)), "PERIODIC"),
        (dict(bc=(2, 3, 0, 0, 0, 0)), "z faces"),
        (dict(bc=(6, 6, 0, 0, 0, 0)), "unknown boundary"),
        (dict(bc=(5, 5, 0, 0, 0, 0)), "HALO"),
        (dict(bc=(0, 0, 0, 0, 5, 0)), "PERIODIC"),
        (dict(bc=(4, 0, 0, 0, 0, 0)), "PERIODIC"),
        (dict(rho_l=0.0), "densit"),
        (dict(W=0.0), "W"),
        (dict(tau_l=-0.5), "tau"),
        (dict(M=-0.2), "tau_phi"),
        (dict(outlet_u_mode=3), "outlet_u_mode"),
        (dict(visc_interp=7), "visc_interp"),
        (dict(path=6), "path"),
        (dict(outlet_clamp=2), "outlet_clamp"),
        (dict(outlet_u_time=2), "outlet_u_time"),
        (dict(outlet_u_time=1, phase_only=1), "outlet_u_time"),
        (dict(tile_ty=5), "tile_ty"),
        (dict(tile_chunks=-1), "tile_chunks"),
        (dict(runtime_nx=2), "runtime_nx"),
    ):
        q = dict(p); q.update(bad)
        assert clip.clip_workspace_bytes(8, 8, 8, clip.make_params(q)) == 0
        assert word in clip.clip_last_error(None), (bad, clip.clip_last_error(None))
    for good in (dict(bc=(4, 4, 1, 4, 4, 1)), dict(bc=(4, 4, 4, 4, 2, 3)), dict(visc_interp=2)):   # FREESLIP faces, Eq. 25
        q = dict(p); q.update(good)
        assert clip.clip_workspace_bytes(8, 8, 8, clip.make_params(q)) > 0, good
    assert clip.clip_workspace_bytes(0, 8, 8, ok) == 0
    rc, h = clip.clip_create(8, 8, 8, ok, 0, 1 << 30, 0)          # NULL workspace
    assert rc == clip.CLIP_EINVAL and not h
    rc, h = clip.clip_create(8, 8, 8, ok, 4096 + 8, 1 << 30, 0)   # misaligned workspace
    assert rc == clip.CLIP_EINVAL and "aligned" in clip.clip_last_error(None)
    rc, h = clip.clip_create(8, 8, 8, ok, 4096, 16, 0)            # too small
    assert rc == clip.CLIP_ENOMEM
    assert clip.clip_step(None, 1) == clip.CLIP_EINVAL and clip.clip_destroy(None) == clip.CLIP_EINVAL


def test_elongated_lattices_do_not_overflow_the_tiling_tables():
    """k_fused's chunk table holds 256 entries: long thin lattices (and absurd tile_chunks) must get longer chunks or another
    path, never a write past the table (round-1 finding: 64 x 64 x 4096 smashed the stack inside clip_workspace_bytes)."""
    p32 = dict(inputs.default_params(), precision=32)
    for shape in ((64, 64, 4096), (64, 4, 20000), (128, 8, 70000), (512, 4, 3000), (64, 64, 257), (256, 1024, 1100)):
        for over in ({}, dict(tile_chunks=10 ** 6), dict(tile_chunks=1), dict(path=3), dict(bc=(1, 1, 1, 1, 1, 1))):
            q = dict(p32); q.update(over)
            n = clip.clip_workspace_bytes(*shape, clip.make_params(q))
            nodes = shape[0] * shape[1] * shape[2]
            assert n >= 80 * 4 * nodes, (shape, over)
            assert n < 86 * 4 * nodes + (1 << 20), (shape, over, n / nodes)


def test_random_lattices_of_the_path_fuzz_are_valid_inputs():
    """inputs.random_lattice (tests/test_fuzz_gpu.py): every seed the fuzz uses passes the library's validation for every path, is
    reproducible, and the seeds together reach every face type and both collision operators."""
    import numpy as np
    faces, colls = set(), set()
    for seed in inputs.RANDOM_LATTICE_SEEDS:
        case = inputs.random_lattice(seed)
        again = inputs.random_lattice(seed)
        assert np.array_equal(case["phi0"], again["phi0"]) and np.array_equal(case["u0"], again["u0"]) and case["params"] == again["params"]
        assert case["phi0"].min() >= 0.0 and case["phi0"].max() <= 1.0
        for path in (0, 1, 2, 3):
            for prec in (32, 64):
                p = dict(case["params"], path=path, precision=prec)
                assert clip.clip_workspace_bytes(case["nx"], case["ny"], case["nz"], clip.make_params(p)) > 0, (seed, clip.clip_last_error(None))
        faces.update(case["params"]["bc"]); colls.add(case["params"]["collision"])
    assert faces == {inputs.PERIODIC, inputs.WALL, inputs.INLET, inputs.OUTLET, inputs.FREESLIP} and colls == {0, 1}


def test_no_cpu_fallback(tmp_path, monkeypatch):
    """A missing libclip.so is a hard error; the product never imports the oracle."""
    monkeypatch.setattr(clip, "_lib", None)
    monkeypatch.setattr(clip, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(RuntimeError):
        clip.lib()
    pkg = os.path.join(ROOT, "paper_2505_12205_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"(^|\n)\s*(import|from)\s+oracle|clip_oracle|clipo_", txt), f


_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms, e2e, finite = bench.reduce_over_ranks(10.0 + rank, 1.0 + 2 * rank, rank == 0, world, torch.device("cpu"))
seeds = [bench.rank_seed(r) for r in range(world)]
if rank == 0:
    print(json.dumps(dict(ms=ms, e2e=e2e, finite=finite, seeds=seeds, mlups=bench.whole_job_mlups(100, 5, ms, world))))
dist.destroy_process_group()
"""


def test_multirank_reduction_gloo(tmp_path):
    """world_size 2 on CPU (gloo): timing is the MAX over ranks, finiteness the AND, every rank gets its own
    seeded replica, and `value` counts the nodes of all ranks (weak scaling)."""
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                          "--master-addr", "127.0.0.1", "--master-port", "29731", str(script)],
                         capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    import json
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    r = json.loads(line)
    assert r["ms"] == 11.0 and r["e2e"] == 3.0 and r["finite"] is False
    assert len(set(r["seeds"])) == 2
    assert abs(r["mlups"] - 2 * 100 * 5 / (11.0e-3) / 1e6) < 1e-9


def test_reference_arm_other_ranks_do_nothing():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, timeout=120, env=env, cwd=ROOT)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_bench_gpus_n_starts_n_ranks():
    """`python bench.py --gpus 2` with no launcher around it starts two ranks itself and defaults to the slab decomposition (the
    path's own sharding); checked on CPU through --plumbing-only (gloo rendezvous, max-over-ranks reduction, no GPU work)."""
    import json
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--plumbing-only"], capture_output=True, text=True,
                         timeout=300, env=env, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    r = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    assert r["n_gpus"] == 2 and r["gpus_requested"] == 2 and r["decomp"] == "slab" and r["max_ms"] == 2.0 and r["max_e2e_s"] == 3.0
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--plumbing-only"], capture_output=True, text=True, timeout=120, env=env, cwd=ROOT)
    r = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    assert r["n_gpus"] == 1 and r["decomp"] == "replicas"

"""clip_outlet_lambda_static (include/clip.h): the no-allocation entry point -- lambda of the convective outlet (App. B.5, B.22 / B.25,
PAPER.md:1104-1117) with its per-column scratch in a static device array instead of a caller workspace.

Checked against the EXISTING path, i.e. the lambda k_outlet_lam + k_outlet_reduce compute inside clip_step.  That lambda is internal to
the step; what the step publishes fixes it exactly: summing B.26-B.27 over a (Eq. 38) gives, per column of the outlet layer N,
    phi_N(t+1) (1 + lambda) = phi_N(t) + lambda phi_{N-1}(t+1)                                        (*)
with phi(t), u(t) and phi(t+1) from clip_get before / after one clip_step.  The new entry point gets u(t) and must return a lambda
that (a) satisfies (*) on the step's own fields to round-off and (b) equals the lambda solved from (*) where its denominator is not
small.  Two calls in a row, on different lattices, modes and plane sizes (the second smaller, so the scratch still holds the first call's
values beyond its own), are issued back to back on one stream before either result is looked at.  This file is collected last on
purpose (`pytest -x`)."""
import numpy as np
import pytest

from paper_2505_12205_b200 import clip, inputs

P_, WL, OUT = inputs.PERIODIC, inputs.WALL, inputs.OUTLET
TOL_RES = {64: 1e-13, 32: 2e-6}      # residual of (*): a few ulp of phi ~ 1
TOL_LAM = {64: 1e-10, 32: 2e-4}      # lambda solved from (*): ulp / |phi_{N-1} - phi_N| with the denominator >= 0.05


def _case(nx, ny, nz, mode, clamp, seed):
    """Two-phase lattice, WALL below and OUTLET above, an interface that crosses the outlet layer (so that (*) has a denominator) and a
    seeded velocity field with out- AND backflow over layer N-1."""
    rng = np.random.default_rng(seed)
    p = inputs.default_params(W=4.0, rho_l=0.1, bc=(P_, P_, P_, P_, WL, OUT), outlet_u_mode=mode, outlet_clamp=clamp)
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    z0 = nz - 2.3 + 0.8 * np.sin(2 * np.pi * x / nx) * np.cos(2 * np.pi * y / ny)
    phi0 = 0.5 - 0.5 * np.tanh(2.0 * (z - z0) / p["W"])
    u0 = 0.005 * rng.uniform(-1.0, 1.0, size=(3, nz, ny, nx))
    u0[2] += 0.01 + 0.03 * rng.uniform(-1.0, 1.0, size=(nz, ny, nx))
    return dict(nx=nx, ny=ny, nz=nz, params=p, phi0=phi0, u0=u0)


def _static(u, mode, clamp, precision, out):
    import torch
    _, nz, ny, nx = u.shape
    rc = clip.clip_outlet_lambda_static(u.data_ptr(), nx, ny, nz, precision, mode, clamp, out.data_ptr(),
                                        torch.cuda.current_stream().cuda_stream)
    assert rc == clip.CLIP_OK, clip.clip_static_last_error()


@pytest.mark.gpu
@pytest.mark.parametrize("precision", [64, 32])
def test_static_scratch_entry_point_against_the_step(precision):
    import torch
    specs = [dict(nx=40, ny=24, nz=12, mode=1, clamp=0, seed=5), dict(nx=12, ny=10, nz=9, mode=2, clamp=1, seed=6),
             dict(nx=20, ny=6, nz=8, mode=0, clamp=1, seed=7)]
    runs = []
    for s in specs:                                              # the existing path: fields before / after one step
        case = _case(**s)
        sim = clip.Clip.from_case(case, precision=precision)
        sim.step(2)
        phi_a, _, u_a = sim.get()
        sim.step(1)
        phi_b, _, _ = sim.get()
        sim.close()
        runs.append((s, phi_a, u_a, phi_b))
    dtype = torch.float64 if precision == 64 else torch.float32
    outs = [torch.full((s["ny"], s["nx"]), float("nan"), dtype=dtype, device="cuda") for s in specs]
    for (s, _, u_a, _), out in zip(runs, outs):                  # the calls in a row, nothing in between
        _static(u_a, s["mode"], s["clamp"], precision, out)
    again = torch.empty_like(outs[0])
    _static(runs[0][2], specs[0]["mode"], specs[0]["clamp"], precision, again)
    torch.cuda.synchronize()
    assert torch.equal(again, outs[0])                           # the contents the other calls left in the scratch do not matter
    for (s, phi_a, u_a, phi_b), out in zip(runs, outs):
        lam = out.double().cpu().numpy()
        pa, pb = phi_a.double().cpu().numpy(), phi_b.double().cpu().numpy()
        uz = u_a[2, -2].double().cpu().numpy()
        assert np.isfinite(lam).all()
        assert (uz < 0).any() and (uz > 0).any()
        # against what B.22 says, from the same u(t)
        want = {0: uz, 1: np.full_like(uz, uz.mean()), 2: np.full_like(uz, uz.max())}[s["mode"]]
        if s["clamp"]:
            want = np.maximum(want, 0.0)
        assert np.abs(lam - want).max() <= (1e-15 if precision == 64 else 1e-7)
        # (a) the step's own fields satisfy (*) with the new entry point's lambda ...
        res = np.abs(pb[-1] * (1 + lam) - pa[-1] - lam * pb[-2]).max()
        assert res < TOL_RES[precision], (s, res)
        # ... and not with a lambda that is off by 1e3 times that tolerance
        off = lam + 1e3 * TOL_RES[precision]
        assert np.abs(pb[-1] * (1 + off) - pa[-1] - off * pb[-2]).max() > 20 * TOL_RES[precision]
        # (b) lambda of the existing path, solved from (*)
        den = pb[-2] - pb[-1]
        ok = np.abs(den) >= 0.05
        assert ok.sum() >= 0.25 * ok.size
        lam_step = (pb[-1] - pa[-1])[ok] / den[ok]
        err = np.abs(lam_step - lam[ok]).max()
        print(f"fp{precision} {s}: residual of (*) {res:.1e}, |lambda - lambda(step)| {err:.1e} on {ok.sum()} columns")
        assert err < TOL_LAM[precision], (s, err)


def test_static_scratch_entry_point_refuses_what_it_cannot_hold():
    """Argument checks return before any CUDA call (no GPU needed): a plane beyond the static array's size is refused, with a reason."""
    big = 1024
    assert big * big > clip.CLIP_STATIC_MAX_PLANE_NODES
    rc = clip.clip_outlet_lambda_static(256, big, big, 4, 32, 1, 1, 256, 0)
    assert rc == clip.CLIP_EINVAL and "CLIP_STATIC_MAX_PLANE_NODES" in clip.clip_static_last_error()
    for args, word in (((256, 8, 8, 4, 16, 1, 1, 256, 0), "precision"), ((256, 8, 8, 1, 32, 1, 1, 256, 0), "nz"),
                       ((256, 8, 8, 4, 32, 3, 1, 256, 0), "outlet_u_mode"), ((256, 8, 8, 4, 32, 1, 2, 256, 0), "outlet_clamp"),
                       ((0, 8, 8, 4, 32, 1, 1, 256, 0), "non-NULL"), ((256, 8, 8, 4, 64, 1, 1, 260, 0), "aligned")):
        assert clip.clip_outlet_lambda_static(*args) == clip.CLIP_EINVAL
        assert word in clip.clip_static_last_error(), (args, clip.clip_static_last_error())
    src = open(clip.LIB_PATH[:-len("libclip.so")] + "csrc/clip_static.cu").read()
    code = "\n".join(line.split("//")[0] for line in src.splitlines())
    assert "cudaMalloc" not in code and "cudaFree" not in code and "cudaGetSymbolAddress" in code
